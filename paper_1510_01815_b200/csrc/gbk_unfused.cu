// Unfused comparison path of libgbk (north_star item 3; gbk_eval_batch_unfused of include/gbk.h).
//
// One kernel per step of the paper's pipeline, in the paper's order, with the FP32 model cube
// written to device memory between steps -- the structure of PAPER.md:197-251 (cube evaluation
// kernel :199-210, convolution :212-218 done here as direct sums like the paper's 2-D + 1-D
// decomposition :568-571 instead of cuFFT, down-sampling :220-224, moments kernel :234, residual
// kernel :238, chi^2 sum :246).  It exists to be compared with the fused kernel: it is bound by
// HBM traffic (the cube is written and re-read by every step) where the fused kernel is bound by
// the SM arithmetic pipes.  It uses the accurate math library (expf, atanf, sqrtf), not the
// approximate intrinsics of the fused kernel, so agreement between the two is also a check of those.
//
// Layout of a chunk of rows: cube[row][channel][y][x], x fastest (the paper's slice-major cube,
// PAPER.md:234), over the extended grid (u nx + 2R) x (u ny + 2R) x (nv + 2 R_v) with R the
// largest PSF radius of the problem.
#include <math.h>

#include <algorithm>

#include "gbk_internal.h"

namespace gbk {

namespace {

struct URow {          // constants of one parameter row (a1)
  float xo, yo, sp, cp, si, inv_ci, vsys, vt, inv_rt, inv_r0, i0, sigma0, ea, eg;
  int gal, psf_set, r_p, valid;
};

__device__ URow uf_row(const DevProblem& dp, const float* params, const int32_t* gal_index, long long k) {
  const float* p = params + k * dp.row_stride;
  URow r;
  bool finite = true;
  for (int j = 0; j < dp.row_stride; ++j) finite = finite && isfinite(p[j]);
  r.ea = r.eg = 1.0f;
  if (dp.rc_model == GBK_RC_EPINAT) r.ea = p[10], r.eg = p[11];
  sincospif(p[2] * (1.0f / 180.0f), &r.sp, &r.cp);
  float ci;
  sincospif(p[3] * (1.0f / 180.0f), &r.si, &ci);
  r.xo = p[0], r.yo = p[1], r.vsys = p[4], r.vt = p[5], r.sigma0 = p[7], r.i0 = p[9];
  r.inv_ci = 1.0f / ci, r.inv_rt = 1.0f / p[6], r.inv_r0 = 1.0f / p[8];
  int gal = gal_index ? gal_index[k] : 0;
  const bool gal_ok = gal >= 0 && gal < dp.n_gal;
  if (!gal_ok) gal = 0;
  r.gal = gal;
  r.psf_set = dp.psf_per_gal ? gal : 0;
  r.r_p = dp.psf_r[r.psf_set];
  r.valid = finite && gal_ok && p[7] > 0.f && p[8] > 0.f && p[6] > 0.f && p[9] > 0.f && !(fabsf(ci) < 1e-6f) &&
            r.ea > 0.f && r.eg > 0.f;
  return r;
}

// Which PSF set a row uses (the convolution kernels need nothing else of the row).
__device__ __forceinline__ URow uf_row_psf(const DevProblem& dp, const int32_t* gal_index, long long k) {
  URow r;
  int gal = gal_index ? gal_index[k] : 0;
  if (gal < 0 || gal >= dp.n_gal) gal = 0;
  r.gal = gal;
  r.psf_set = dp.psf_per_gal ? gal : 0;
  r.r_p = dp.psf_r[r.psf_set];
  r.valid = 1;
  return r;
}

struct UGeom {         // extended grid of the unfused path
  int R, EW, EH, nvx;
  size_t plane, cube;  // EW*EH, plane*nvx
};

__host__ __device__ inline UGeom uf_geom(const DevProblem& dp) {
  UGeom g;
  g.R = dp.r_p_max, g.EW = dp.fw + 2 * g.R, g.EH = dp.fh + 2 * g.R, g.nvx = dp.nvx;
  g.plane = (size_t)g.EW * g.EH, g.cube = g.plane * g.nvx;
  return g;
}

// Step 1: one thread per extended spatial sample evaluates its whole spectrum;
// consecutive threads <-> consecutive x, so every channel slice is written coalesced.
__global__ void uf_cube_kernel(const __grid_constant__ DevProblem dp, const float* __restrict__ params,
                               const int32_t* __restrict__ gal_index, long long k0, int nrows,
                               float* __restrict__ cube) {
  const UGeom g = uf_geom(dp);
  const long long n = (long long)nrows * g.plane;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / g.plane);
    const int pix = (int)(idx - row * (long long)g.plane);
    const int ey = pix / g.EW, ex = pix - ey * g.EW;
    const URow r = uf_row(dp, params, gal_index, k0 + row);
    float* out = cube + (size_t)row * g.cube + pix;
    if (!r.valid) {
      for (int c = 0; c < g.nvx; ++c) out[(size_t)c * g.plane] = 0.0f;
      continue;
    }
    const float x = ((float)(ex - g.R) + 0.5f) * dp.inv_u - 0.5f - r.xo;   // A1
    const float y = ((float)(ey - g.R) + 0.5f) * dp.inv_u - 0.5f - r.yo;
    const float xe = -x * r.sp + y * r.cp;                                  // eq. 1
    const float ye = (-x * r.cp - y * r.sp) * r.inv_ci;                     // eq. 2 / cos i
    const float rad = sqrtf(xe * xe + ye * ye);                             // eq. 3
    const float cos_t = rad > 0.0f ? xe / rad : 0.0f;                       // eq. 4, A8
    float bright;
    if (dp.tab_n > 0) {                                                     // tabulated T(r / r0)
      const float tc = fminf(rad * r.inv_r0 * dp.tab_inv_dx, (float)(dp.tab_n - 1));
      const int j = min((int)tc, dp.tab_n - 2);
      bright = r.i0 * (dp.tab[j] + (tc - (float)j) * (dp.tab[j + 1] - dp.tab[j]));
    } else {
      bright = r.i0 * expf(-rad * r.inv_r0);                                // eq. 5
    }
    const float q = rad * r.inv_rt;
    float vrot;
    if (dp.rc_model == GBK_RC_ARCTAN) vrot = 0.63661977236758134f * r.vt * atanf(q);            // eq. 6
    else if (dp.rc_model == GBK_RC_RAMP) vrot = r.vt * fminf(q, 1.0f);                          // A7
    else vrot = q > 0.0f ? r.vt * powf(q, r.eg) / (1.0f + powf(q, r.ea)) : 0.0f;                // eq. 7
    const float vlos = (r.vsys - dp.v_center) + vrot * r.si * cos_t;        // eq. 8, from v_center
    const float amp = bright * dp.dv / (r.sigma0 * 2.5066282746310002f) ; // A3
    const float inv_s = 1.0f / r.sigma0;
    for (int c = 0; c < g.nvx; ++c) {
      const float t = (dp.vrel_first + (float)c * dp.dv - vlos) * inv_s;
      out[(size_t)c * g.plane] = amp * expf(-0.5f * t * t);
    }
  }
}

// Step 2a: LSF along v (direct sum, "valid": nvx -> nv channels).  lsf[j], j = 0..2 r_v.
__global__ void uf_lsf_kernel(const __grid_constant__ DevProblem dp, const float* __restrict__ lsf,
                              int nrows, const float* __restrict__ in, float* __restrict__ out) {
  const UGeom g = uf_geom(dp);
  const size_t per_row = g.plane * dp.nv;
  const long long n = (long long)nrows * per_row;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / per_row);
    const size_t rem = idx - row * (long long)per_row;
    const int c = (int)(rem / g.plane);
    const size_t pix = rem - c * g.plane;
    const float* src = in + (size_t)row * g.cube + pix;
    float s = 0.0f;
    for (int j = -dp.r_v; j <= dp.r_v; ++j)            // out[c] = sum_j L[j] in[c - j]
      s = fmaf(lsf[j + dp.r_v], src[(size_t)(c + dp.r_v - j) * g.plane], s);
    out[(size_t)row * g.cube + rem] = s;
  }
}

// Step 2b: one 1-D pass of the separable Gaussian PSF along x (axis = 0) or y (axis = 1), in the
// extended layout.  The x pass produces columns [R, R + fw); the y pass rows [R, R + fh).
__global__ void uf_psf1d_kernel(const __grid_constant__ DevProblem dp, const float* __restrict__ params,
                                const int32_t* __restrict__ gal_index, long long k0, int nrows, int axis,
                                const float* __restrict__ in, float* __restrict__ out) {
  const UGeom g = uf_geom(dp);
  const int W = dp.fw, H = axis == 0 ? g.EH : dp.fh;
  const size_t per_chan = (size_t)W * H, per_row = per_chan * dp.nv;
  const long long n = (long long)nrows * per_row;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / per_row);
    size_t rem = idx - row * (long long)per_row;
    const int c = (int)(rem / per_chan);
    rem -= c * per_chan;
    const int yy = (int)(rem / W), xx = (int)(rem - (size_t)yy * W);
    const URow r = uf_row_psf(dp, gal_index, k0 + row);
    const float* taps = dp.psf_taps + (size_t)r.psf_set * dp.psf_stride;
    const int ex = xx + g.R, ey = axis == 0 ? yy : yy + g.R;
    const float* src = in + (size_t)row * g.cube + (size_t)c * g.plane + (size_t)ey * g.EW + ex;
    const int stride = axis == 0 ? 1 : g.EW;
    float s = 0.0f;
    for (int j = -r.r_p; j <= r.r_p; ++j) s = fmaf(taps[j + r.r_p], src[-j * stride], s);
    out[(size_t)row * g.cube + (size_t)c * g.plane + (size_t)ey * g.EW + ex] = s;
  }
}

// Step 2b for a general PSF image: direct 2-D sum per voxel.  The image is stored flipped at
// create, so this correlation is the true convolution (A11).
__global__ void uf_psf2d_kernel(const __grid_constant__ DevProblem dp, const float* __restrict__ params,
                                const int32_t* __restrict__ gal_index, long long k0, int nrows,
                                const float* __restrict__ in, float* __restrict__ out) {
  const UGeom g = uf_geom(dp);
  const size_t per_chan = (size_t)dp.fw * dp.fh, per_row = per_chan * dp.nv;
  const long long n = (long long)nrows * per_row;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / per_row);
    size_t rem = idx - row * (long long)per_row;
    const int c = (int)(rem / per_chan);
    rem -= c * per_chan;
    const int yy = (int)(rem / dp.fw), xx = (int)(rem - (size_t)yy * dp.fw);
    const URow r = uf_row_psf(dp, gal_index, k0 + row);
    const int nn = 2 * r.r_p + 1;
    const float* taps = dp.psf_taps + (size_t)r.psf_set * dp.psf_stride;
    const float* src = in + (size_t)row * g.cube + (size_t)c * g.plane + (size_t)(yy + g.R - r.r_p) * g.EW +
                       xx + g.R - r.r_p;
    float s = 0.0f;
    for (int ky = 0; ky < nn; ++ky)
      for (int kx = 0; kx < nn; ++kx) s = fmaf(taps[ky * nn + kx], src[(size_t)ky * g.EW + kx], s);
    out[(size_t)row * g.cube + (size_t)c * g.plane + (size_t)(yy + g.R) * g.EW + xx + g.R] = s;
  }
}

// Steps 3-5: per spaxel, down-sample every channel (mean over the u x u block),
// moments (two passes over the spectrum, like a plain implementation), residuals against the packed
// observation, and the spaxel's chi^2 contribution.
__global__ void uf_moments_kernel(const __grid_constant__ DevProblem dp, const float* __restrict__ params,
                                  const int32_t* __restrict__ gal_index, long long k0, int nrows,
                                  const float* __restrict__ cube, float* __restrict__ contrib,
                                  const EvalArgs a) {
  const UGeom g = uf_geom(dp);
  const int npix = dp.nx * dp.ny;
  const long long n = (long long)nrows * npix;
  const float inf = __int_as_float(0x7f800000), nan = __int_as_float(0x7fc00000);
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / npix);
    const int pix = (int)(idx - (long long)row * npix);
    const int Y = pix / dp.nx, X = pix - Y * dp.nx;
    const long long k = k0 + row;
    const URow r = uf_row(dp, params, gal_index, k);
    const float4 ob = dp.obs[(size_t)r.gal * npix + pix];
    const bool unmasked = ob.y > 0.0f;
    float m0 = nan, m1 = nan, m2 = nan, t = nan, s = nan, c2 = inf;
    if (r.valid) {
      const float* src = cube + (size_t)row * g.cube + (size_t)(Y * dp.u + g.R) * g.EW + X * dp.u + g.R;
      const float v_first = -0.5f * (float)(dp.nv - 1) * dp.dv;
      float s0 = 0.0f, s1 = 0.0f;
      for (int c = 0; c < dp.nv; ++c) {
        float blk = 0.0f;
        for (int dy = 0; dy < dp.u; ++dy)
          for (int dx = 0; dx < dp.u; ++dx) blk += src[(size_t)c * g.plane + (size_t)dy * g.EW + dx];
        blk *= dp.inv_u2;
        s0 += blk;
        s1 = fmaf(blk, v_first + (float)c * dp.dv, s1);
      }
      m0 = s0;
      m1 = s1 / s0;
      float s2 = 0.0f;
      for (int c = 0; c < dp.nv; ++c) {
        float blk = 0.0f;
        for (int dy = 0; dy < dp.u; ++dy)
          for (int dx = 0; dx < dp.u; ++dx) blk += src[(size_t)c * g.plane + (size_t)dy * g.EW + dx];
        blk *= dp.inv_u2;
        const float d = v_first + (float)c * dp.dv - m1;
        s2 = fmaf(blk * d, d, s2);
      }
      const float var = s2 / s0;
      m2 = var > 0.0f ? sqrtf(var) : (var == var ? 0.0f : var);            // A5
      const bool dark = !(m0 >= 1e-30f * r.i0);                             // A15
      t = (m1 - ob.x) * ob.y;
      s = (m2 - ob.z) * ob.w;
      c2 = fmaf(t, t, s * s);
      const bool bad = dark || !(c2 < inf);
      if (dark) m1 = m2 = nan;
      if (!unmasked) t = s = 0.0f, c2 = 0.0f;
      else if (bad) t = s = nan, c2 = inf;
      m1 += dp.v_center;
    } else if (!unmasked) {
      c2 = inf;   // an out-of-domain row is +INF whatever the mask
    }
    contrib[idx] = c2;
    const size_t o = (size_t)k * npix + pix;
    if (a.m0) a.m0[o] = m0;
    if (a.m1) a.m1[o] = m1;
    if (a.m2) a.m2[o] = m2;
    if (a.resid) {
      a.resid[2 * (size_t)k * npix + pix] = t;
      a.resid[(2 * (size_t)k + 1) * npix + pix] = s;
    }
  }
}

// chi^2 of a row = fixed-order sum of its spaxel contributions: one block per row.
__global__ void uf_chi2_kernel(const float* __restrict__ contrib, int npix, long long k0,
                               float* __restrict__ chi2) {
  __shared__ float red[32];
  const float* c = contrib + (size_t)blockIdx.x * npix;
  float s = 0.0f;
  for (int i = threadIdx.x; i < npix; i += blockDim.x) s += c[i];
  for (int off = 16; off > 0; off >>= 1) s += __shfl_down_sync(0xffffffffu, s, off);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    float tot = 0.0f;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) tot += red[w];
    if (!(tot < __int_as_float(0x7f800000))) tot = __int_as_float(0x7f800000);
    chi2[k0 + blockIdx.x] = tot;
  }
}

inline unsigned grid_for(long long n, int threads, int sm_count) {
  const long long want = (n + threads - 1) / threads;
  const long long cap = (long long)sm_count * 32;     // grid-stride: a few waves per SM
  return (unsigned)std::max(1LL, std::min(want, cap));
}

}  // namespace

size_t unfused_bytes_per_row(const DevProblem& dp) {
  const UGeom g = uf_geom(dp);
  return sizeof(float) * (2 * g.cube + (size_t)dp.nx * dp.ny);
}

// Algorithmic HBM bytes of the unfused pipeline per row (every array written once, read once per
// consumer).
double unfused_algorithmic_bytes_per_row(const DevProblem& dp) {
  const UGeom g = uf_geom(dp);
  const double ext = (double)g.cube, lsf = (double)g.plane * dp.nv;
  const double px = (double)dp.fw * g.EH * dp.nv, fine = (double)dp.fw * dp.fh * dp.nv;
  double b = ext /*w*/ + ext /*r*/ + lsf /*w*/;
  if (dp.psf_kind == GBK_PSF_GAUSSIAN) b += lsf + px + px + fine;   // x pass r/w, y pass r/w
  else b += lsf + fine;
  b += 2.0 * fine;                                                    // moments: two passes
  return 4.0 * b;
}

cudaError_t launch_unfused(const DevProblem& dp, const EvalArgs& a, const float* lsf_taps, float* scratch,
                           long long chunk_rows, int sm_count, cudaStream_t st) {
  const UGeom g = uf_geom(dp);
  const int T = 256, npix = dp.nx * dp.ny;
  float* A = scratch;
  float* B = A + (size_t)chunk_rows * g.cube;
  float* contrib = B + (size_t)chunk_rows * g.cube;
  for (long long k0 = 0; k0 < a.K; k0 += chunk_rows) {
    const int n = (int)std::min(chunk_rows, a.K - k0);
    uf_cube_kernel<<<grid_for((long long)n * g.plane, T, sm_count), T, 0, st>>>(dp, a.params, a.gal_index, k0, n, A);
    uf_lsf_kernel<<<grid_for((long long)n * g.plane * dp.nv, T, sm_count), T, 0, st>>>(dp, lsf_taps, n, A, B);
    const float* conv;
    if (dp.psf_kind == GBK_PSF_GAUSSIAN) {
      uf_psf1d_kernel<<<grid_for((long long)n * dp.fw * g.EH * dp.nv, T, sm_count), T, 0, st>>>(
          dp, a.params, a.gal_index, k0, n, 0, B, A);
      uf_psf1d_kernel<<<grid_for((long long)n * dp.fw * dp.fh * dp.nv, T, sm_count), T, 0, st>>>(
          dp, a.params, a.gal_index, k0, n, 1, A, B);
      conv = B;
    } else {
      uf_psf2d_kernel<<<grid_for((long long)n * dp.fw * dp.fh * dp.nv, T, sm_count), T, 0, st>>>(
          dp, a.params, a.gal_index, k0, n, B, A);
      conv = A;
    }
    uf_moments_kernel<<<grid_for((long long)n * npix, 128, sm_count), 128, 0, st>>>(dp, a.params, a.gal_index,
                                                                                  k0, n, conv, contrib, a);
    uf_chi2_kernel<<<n, 256, 0, st>>>(contrib, npix, k0, a.chi2);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace gbk
