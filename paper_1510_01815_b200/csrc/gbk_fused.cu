// Fused hot path of libgbk for sm_100a: one thread block = (parameter row k, spatial tile).
//
// What one block does (steps a1..a9 of SURVEY.md section 8(a); PAPER.md = arXiv:1510.01815):
//   a1  row constants from the 10 parameters (eq. 1-8)
//   a2  per fine spatial sample of the tile + PSF halo: deprojection (eq. 1-4),
//       exponential brightness (eq. 5, :110), rotation curve (eq. 6, :120, or ramp), line-of-sight
//       velocity (eq. 8, :143)
//   a3  Gaussian line at every extended channel, one MUFU.EX2 per voxel
//   a4  LSF along v: folded into per-channel weights (see below)
//   a5  PSF in (x, y) from shared memory: separable Gaussian passes or a general 2-D image
//   a6  down-sampling by u
//   a7  moments       a8  residual, mask, chi^2 (eq. 11, :246)
//   a9  chi^2 (and optional maps / residuals) to global memory
//
// The cube never exists, not even in shared memory.  The un-normalised moments
//   S_q(x, y) = sum_k v_k^q C_k(x, y),  q = 0, 1, 2
// are linear in the cube, and LSF, PSF and down-sampling are linear and act on different axes,
// so  S_q = downsample( PSF (*) sum_c w_q[c] line(x, y, c) )  with the per-problem weights
//   w_q[c] = sum_{k in band} L[k - c] v_k^q
// (LSF taps L and band edges folded in exactly; built in gbk_api.cu).  Only three 2-D maps per
// tile are convolved.  m1 = S1/S0, m2 = sqrt(S2/S0 - m1^2).  Velocities are measured from
// v_center so the FP32 cancellation in m2 stays ~1e-4 km/s.
#include <math.h>

#include "gbk_internal.h"

namespace gbk {

namespace {

constexpr int kMaxThreads = 384;
constexpr int kMinBlocks = 2;

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__host__ __device__ __forceinline__ int round_up4(int v) { return (v + 3) & ~3; }

struct Smem {
  float* maps;      // 3 x ehs x ews
  float4* chan;     // nvx
  float* taps;      // round_up4(psf_stride)
  RowConst* rc;
  float* red;       // 32
};

__device__ __forceinline__ Smem carve(const DevProblem& dp, unsigned char* raw) {
  Smem s;
  s.maps = reinterpret_cast<float*>(raw);
  s.chan = reinterpret_cast<float4*>(s.maps + 3 * dp.ehs * dp.ews);
  s.taps = reinterpret_cast<float*>(s.chan + dp.nvx);
  s.rc = reinterpret_cast<RowConst*>(s.taps + round_up4(dp.psf_stride));
  s.red = reinterpret_cast<float*>(s.rc + 1);
  return s;
}

// ---------------------------------------------------------------------------------- a1 ------
__device__ void row_constants(const DevProblem& dp, const EvalArgs& a, long long k, RowConst* rc) {
  const float* p = a.params + k * GBK_P;
  float v[GBK_P];
  bool finite = true;
#pragma unroll
  for (int j = 0; j < GBK_P; ++j) {
    v[j] = p[j];
    finite = finite && isfinite(v[j]);
  }
  float sp, cp, si, ci;
  sincospif(v[2] * (1.0f / 180.0f), &sp, &cp);
  sincospif(v[3] * (1.0f / 180.0f), &si, &ci);
  const float sigma0 = v[7], r0 = v[8], rt = v[6], i0 = v[9];
  const bool ok = finite && sigma0 > 0.f && r0 > 0.f && rt > 0.f && i0 > 0.f && !(fabsf(ci) < 1e-6f);
  int gal = a.gal_index ? a.gal_index[k] : 0;
  const bool gal_ok = gal >= 0 && gal < dp.n_gal;
  if (!gal_ok) gal = 0;
  rc->gal = gal;
  rc->psf_set = dp.psf_per_gal ? gal : 0;
  rc->r_p = dp.psf_r[rc->psf_set];
  rc->valid = (ok && gal_ok) ? 1 : 0;
  rc->xo = v[0];
  rc->yo = v[1];
  rc->sp = sp;
  rc->cp = cp;
  rc->inv_ci = 1.0f / ci;
  rc->vrot_scale = (dp.rc_model == GBK_RC_ARCTAN ? 0.63661977236758134f : 1.0f) * v[5] * si;
  rc->inv_rt = 1.0f / rt;
  rc->nl2e_inv_r0 = -1.4426950408889634f / r0;
  rc->vsys_rel = v[4] - dp.v_center;
  rc->s = 1.0f / (sigma0 * 1.1774100225154747f);  // sqrt(2 ln 2)
  rc->step = rc->s * dp.dv;
  rc->d_first = rc->s * dp.vrel_first;
  const float line_amp = dp.dv / (sigma0 * 2.5066282746310002f) * dp.inv_u2;  // sqrt(2 pi)
  rc->amp = i0 * line_amp;
  rc->dark_s0 = 1e-30f / line_amp;
}

// ---------------------------------------------------------------------------- a7, a8, a9 ----
// One spaxel: moments from the block sums, residuals, chi^2 contribution, optional outputs.
__device__ __forceinline__ float spaxel_finish(const DevProblem& dp, const EvalArgs& a,
                                               const RowConst& rc, long long k, int X, int Y,
                                               float S0, float S1, float S2) {
  const int npix = dp.nx * dp.ny;
  const int pix = Y * dp.nx + X;
  const float4 ob = __ldg(&dp.obs[(size_t)rc.gal * npix + pix]);
  const float inv = 1.0f / S0;
  float m1r = S1 * inv;
  const float var = fmaf(-m1r, m1r, S2 * inv);
  float m2 = sqrtf(fmaxf(var, 0.0f));
  if (var != var) m2 = var;                       // fmaxf drops NaN
  const bool dark = !(S0 >= rc.dark_s0);
  if (dark) m1r = m2 = __int_as_float(0x7fc00000);
  const bool bad = dark || !isfinite(m1r) || !isfinite(m2);
  const bool unmasked = ob.y > 0.0f;
  float t = 0.0f, s = 0.0f, contrib = 0.0f;
  if (unmasked) {
    if (bad) {
      t = s = __int_as_float(0x7fc00000);
      contrib = __int_as_float(0x7f800000);
    } else {
      t = (m1r - ob.x) * ob.y;
      s = dp.has_disp ? (m2 - ob.z) * ob.w : 0.0f;
      contrib = fmaf(t, t, s * s);
    }
  }
  const size_t o = (size_t)k * npix + pix;
  if (a.m0) a.m0[o] = rc.amp * S0;
  if (a.m1) a.m1[o] = m1r + dp.v_center;
  if (a.m2) a.m2[o] = m2;
  if (a.resid) {
    a.resid[2 * (size_t)k * npix + pix] = t;
    a.resid[(2 * (size_t)k + 1) * npix + pix] = s;
  }
  return contrib;
}

// ---------------------------------------------------------------------------------- a5 ------
// Horizontal pass of the separable PSF, in place: a row is owned by one group of lanes, which
// loads everything it needs before it stores (true convolution: out[x] = sum_k T[k] in[x+2R-k]).
template <int R>
__device__ __forceinline__ void hpass(float* maps, int map_stride, int ews, int EH, int tw,
                                      const float* taps, int tid, int nthreads) {
  constexpr int NT = 2 * R + 1, NV4 = (4 + 2 * R + 3) / 4;
  float t[R + 1];   // Gaussian taps are symmetric: tap(k) = t[|k - R|]
#pragma unroll
  for (int j = 0; j <= R; ++j) t[j] = taps[R + j];
  const int lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
  const int nx4 = (tw + 3) >> 2;
  int lpr_log = 0;
  while ((1 << lpr_log) < nx4 && lpr_log < 5) ++lpr_log;
  const int lpr = 1 << lpr_log;                 // lanes per row
  const int rpp = 32 >> lpr_log;                // rows per pass
  const int l = lane & (lpr - 1), rsub = lane >> lpr_log;
  const int nchunks = (nx4 + lpr - 1) >> lpr_log;
  const int npass = (EH + rpp - 1) / rpp;
  for (int job = warp; job < 3 * npass; job += nwarps) {
    const int q = job / npass, pass = job - q * npass;
    const int row = pass * rpp + rsub;
    float* rowp = maps + q * map_stride + row * ews;
    for (int chunk = 0; chunk < nchunks; ++chunk) {
      const int x0 = ((chunk << lpr_log) + l) << 2;
      const bool active = row < EH && x0 < tw;
      float v[NV4 * 4];
      if (active) {
#pragma unroll
        for (int i = 0; i < NV4; ++i) {
          const float4 f = *reinterpret_cast<const float4*>(rowp + x0 + 4 * i);
          v[4 * i] = f.x, v[4 * i + 1] = f.y, v[4 * i + 2] = f.z, v[4 * i + 3] = f.w;
        }
      }
      __syncwarp();
      if (active) {
        float o[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int kk = 0; kk < NT; ++kk)
#pragma unroll
          for (int i = 0; i < 4; ++i) o[i] = fmaf(t[kk < R ? R - kk : kk - R], v[i + 2 * R - kk], o[i]);
        *reinterpret_cast<float4*>(rowp + x0) = make_float4(o[0], o[1], o[2], o[3]);
      }
      __syncwarp();
    }
  }
}

// Vertical pass fused with moments and chi^2 (u == 1): a thread owns kVBlock consecutive rows of
// one column; lanes run along x, so shared-memory reads are conflict-free and global accesses
// coalesced.
template <int R>
__device__ __forceinline__ float vpass_moments(const DevProblem& dp, const EvalArgs& a,
                                               const RowConst& rc, long long k, const float* maps,
                                               int map_stride, int ews, int EH, int tw, int th,
                                               int tx0, int ty0, const float* taps, int tid,
                                               int nthreads) {
  constexpr int NT = 2 * R + 1, BY = kVBlock;
  float t[R + 1];
#pragma unroll
  for (int j = 0; j <= R; ++j) t[j] = taps[R + j];
  const int nyb = (th + BY - 1) / BY;
  float chi = 0.0f;
  for (int item = tid; item < tw * nyb; item += nthreads) {
    const int yb = item / tw, x = item - yb * tw, y0 = yb * BY;
    float res[3][BY];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const float* col = maps + q * map_stride + y0 * ews + x;
      float acc[BY];
#pragma unroll
      for (int o = 0; o < BY; ++o) acc[o] = 0.0f;
#pragma unroll
      for (int i = 0; i < BY + 2 * R; ++i) {
        const float v = (y0 + i < EH) ? col[i * ews] : 0.0f;
#pragma unroll
        for (int o = 0; o < BY; ++o) {
          const int kk = 2 * R - (i - o);
          if (kk >= 0 && kk < NT) acc[o] = fmaf(t[kk < R ? R - kk : kk - R], v, acc[o]);
        }
      }
#pragma unroll
      for (int o = 0; o < BY; ++o) res[q][o] = acc[o];
    }
#pragma unroll
    for (int o = 0; o < BY; ++o)
      if (y0 + o < th)
        chi += spaxel_finish(dp, a, rc, k, tx0 + x, ty0 + y0 + o, res[0][o], res[1][o], res[2][o]);
  }
  return chi;
}

// Vertical pass in place (u > 1): a thread owns one column of one map and walks it top to bottom
// in chunks, so the rows it overwrites are never read again.
template <int R>
__device__ __forceinline__ void vpass_inplace(float* maps, int map_stride, int ews, int EH, int tw,
                                              int th, const float* taps, int tid, int nthreads) {
  constexpr int NT = 2 * R + 1, BY = kVBlock;
  float t[R + 1];
#pragma unroll
  for (int j = 0; j <= R; ++j) t[j] = taps[R + j];
  for (int item = tid; item < 3 * tw; item += nthreads) {
    const int q = item / tw, x = item - q * tw;
    float* col = maps + q * map_stride + x;
    for (int y0 = 0; y0 < th; y0 += BY) {
      float acc[BY];
#pragma unroll
      for (int o = 0; o < BY; ++o) acc[o] = 0.0f;
#pragma unroll
      for (int i = 0; i < BY + 2 * R; ++i) {
        const float v = (y0 + i < EH) ? col[(y0 + i) * ews] : 0.0f;
#pragma unroll
        for (int o = 0; o < BY; ++o) {
          const int kk = 2 * R - (i - o);
          if (kk >= 0 && kk < NT) acc[o] = fmaf(t[kk < R ? R - kk : kk - R], v, acc[o]);
        }
      }
#pragma unroll
      for (int o = 0; o < BY; ++o)
        if (y0 + o < th) col[(y0 + o) * ews] = acc[o];
    }
  }
}

// a6 + a7/a8 for u > 1 after both in-place passes: block sums over u x u fine pixels.
__device__ __forceinline__ float moments_blocks(const DevProblem& dp, const EvalArgs& a,
                                                const RowConst& rc, long long k, const float* maps,
                                                int map_stride, int ews, int tw, int th, int tx0,
                                                int ty0, int tid, int nthreads) {
  const int u = dp.u, sw = tw / u, sh = th / u;
  float chi = 0.0f;
  for (int item = tid; item < sw * sh; item += nthreads) {
    const int Y = item / sw, X = item - Y * sw;
    float s[3] = {0.f, 0.f, 0.f};
    for (int q = 0; q < 3; ++q)
      for (int dy = 0; dy < u; ++dy)
        for (int dx = 0; dx < u; ++dx) s[q] += maps[q * map_stride + (Y * u + dy) * ews + X * u + dx];
    chi += spaxel_finish(dp, a, rc, k, tx0 / u + X, ty0 / u + Y, s[0], s[1], s[2]);
  }
  return chi;
}

// General 2-D PSF image (any u): direct sum per spaxel from shared memory.  The image is stored
// flipped at create, so this correlation is the true convolution.
__device__ __noinline__ float conv2d_moments(const DevProblem& dp, const EvalArgs& a,
                                                const RowConst& rc, long long k, const float* maps,
                                                int map_stride, int ews, int tw, int th, int tx0,
                                                int ty0, const float* taps, int tid, int nthreads) {
  const int u = dp.u, sw = tw / u, sh = th / u, n = 2 * rc.r_p + 1;
  float chi = 0.0f;
  for (int item = tid; item < sw * sh; item += nthreads) {
    const int Y = item / sw, X = item - Y * sw;
    float s0 = 0.f, s1 = 0.f, s2 = 0.f;
    for (int dy = 0; dy < u; ++dy)
      for (int dx = 0; dx < u; ++dx) {
        const float* base = maps + (Y * u + dy) * ews + X * u + dx;
        for (int ky = 0; ky < n; ++ky)
          for (int kx = 0; kx < n; ++kx) {
            const float w = taps[ky * n + kx];
            const float* pp = base + ky * ews + kx;
            s0 = fmaf(w, pp[0], s0);
            s1 = fmaf(w, pp[map_stride], s1);
            s2 = fmaf(w, pp[2 * map_stride], s2);
          }
      }
    chi += spaxel_finish(dp, a, rc, k, tx0 / u + X, ty0 / u + Y, s0, s1, s2);
  }
  return chi;
}

template <int R>
__device__ __noinline__ float separable_phase(const DevProblem& dp, const EvalArgs& a,
                                                 const RowConst& rc, long long k, float* maps,
                                                 int map_stride, int EH, int tw, int th, int tx0,
                                                 int ty0, const float* taps, int tid, int nthreads) {
  hpass<R>(maps, map_stride, dp.ews, EH, tw, taps, tid, nthreads);
  __syncthreads();
  if (dp.u == 1)
    return vpass_moments<R>(dp, a, rc, k, maps, map_stride, dp.ews, EH, tw, th, tx0, ty0, taps, tid,
                            nthreads);
  vpass_inplace<R>(maps, map_stride, dp.ews, EH, tw, th, taps, tid, nthreads);
  __syncthreads();
  return moments_blocks(dp, a, rc, k, maps, map_stride, dp.ews, tw, th, tx0, ty0, tid, nthreads);
}

// ------------------------------------------------------------------------------ the kernel ---
template <int P>
__global__ void __launch_bounds__(kMaxThreads, kMinBlocks)
    fused_kernel(const __grid_constant__ DevProblem dp, const __grid_constant__ EvalArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const Smem sm = carve(dp, smem_raw);
  const int tid = threadIdx.x, nthreads = blockDim.x;
  const long long bid = blockIdx.x;
  const long long k = bid / dp.ntiles;
  const int tile = (int)(bid - k * dp.ntiles);
  const int tyi = tile / dp.tiles_x, txi = tile - tyi * dp.tiles_x;
  const int tx0 = txi * dp.tile_w, ty0 = tyi * dp.tile_h;
  const int tw = min(dp.tile_w, dp.fw - tx0), th = min(dp.tile_h, dp.fh - ty0);
  const int map_stride = dp.ehs * dp.ews;

  if (tid == 0) row_constants(dp, a, k, sm.rc);
  for (int c = tid; c < dp.nvx; c += nthreads) sm.chan[c] = dp.chan_tab[c];
  __syncthreads();
  const RowConst rc = *sm.rc;   // by value: registers, no aliasing with the map stores
  for (int j = tid; j < dp.psf_stride; j += nthreads)
    sm.taps[j] = dp.psf_taps[(size_t)rc.psf_set * dp.psf_stride + j];

  float chi = 0.0f;
  if (!rc.valid) {
    // out-of-domain row: chi^2 = +INF, NaN maps and residuals for this tile's spaxels
    const int u = dp.u, sw = tw / u, sh = th / u, npix = dp.nx * dp.ny;
    const float qnan = __int_as_float(0x7fc00000);
    for (int item = tid; item < sw * sh; item += nthreads) {
      const int Y = item / sw, X = item - Y * sw;
      const size_t pix = (size_t)(ty0 / u + Y) * dp.nx + tx0 / u + X;
      if (a.m0) a.m0[k * npix + pix] = qnan;
      if (a.m1) a.m1[k * npix + pix] = qnan;
      if (a.m2) a.m2[k * npix + pix] = qnan;
      if (a.resid) a.resid[2 * k * npix + pix] = a.resid[(2 * k + 1) * npix + pix] = qnan;
    }
    chi = __int_as_float(0x7f800000);
  } else {
    // ------------------------------------------------------------------ a2, a3, a4 -------
    const int R = rc.r_p;
    const int EW = tw + 2 * R, EH = th + 2 * R, n_ext = EW * EH;
    const float step = rc.step, inv_u = dp.inv_u;
    const int nvx = dp.nvx;
    for (int base = 0; base < n_ext; base += nthreads * P) {
      float d0[P], In[P];
      int sidx[P];
#pragma unroll
      for (int p = 0; p < P; ++p) {
        const int idx = base + p * nthreads + tid;
        const int idc = min(idx, n_ext - 1);
        const int ey = idc / EW, ex = idc - ey * EW;
        sidx[p] = idx < n_ext ? ey * dp.ews + ex : -1;
        const float x = ((float)(tx0 + ex - R) + 0.5f) * inv_u - 0.5f;
        const float y = ((float)(ty0 + ey - R) + 0.5f) * inv_u - 0.5f;
        const float dx = x - rc.xo, dy = y - rc.yo;
        const float xe = fmaf(dy, rc.cp, -dx * rc.sp);            // eq. 1
        const float ye = -fmaf(dx, rc.cp, dy * rc.sp);            // eq. 2
        const float yd = ye * rc.inv_ci;
        const float r2 = fmaf(xe, xe, yd * yd);                   // eq. 3
        const float rs = r2 > 0.0f ? rsqrt_approx(r2) : 0.0f;
        const float r = r2 * rs;
        const float cos_t = xe * rs;                              // eq. 4 (0 at r = 0)
        In[p] = ex2_approx(r * rc.nl2e_inv_r0);                   // eq. 5 / I0
        const float q = r * rc.inv_rt;
        const float vrot = rc.vrot_scale * (dp.rc_model == GBK_RC_ARCTAN ? atanf(q) : fminf(q, 1.0f));
        const float vlos_rel = fmaf(vrot, cos_t, rc.vsys_rel);    // eq. 8 (minus v_center)
        d0[p] = fmaf(-rc.s, vlos_rel, rc.d_first);
      }
      float s0[P], s1[P], s2[P];
#pragma unroll
      for (int p = 0; p < P; ++p) s0[p] = s1[p] = s2[p] = 0.0f;
#pragma unroll 4
      for (int c = 0; c < nvx; ++c) {
        const float4 w = sm.chan[c];
#pragma unroll
        for (int p = 0; p < P; ++p) {
          const float d = fmaf(w.x, step, d0[p]);
          const float g = ex2_approx(-d * d);                     // Gaussian line
          s0[p] = fmaf(w.y, g, s0[p]);
          s1[p] = fmaf(w.z, g, s1[p]);
          s2[p] = fmaf(w.w, g, s2[p]);
        }
      }
#pragma unroll
      for (int p = 0; p < P; ++p)
        if (sidx[p] >= 0) {
          sm.maps[sidx[p]] = s0[p] * In[p];
          sm.maps[map_stride + sidx[p]] = s1[p] * In[p];
          sm.maps[2 * map_stride + sidx[p]] = s2[p] * In[p];
        }
    }
    // zero the pad columns the vectorised horizontal pass may read
    const int padw = dp.ews - EW;
    for (int i = tid; i < 3 * EH * padw; i += nthreads) {
      const int q = i / (EH * padw), rem = i - q * (EH * padw);
      const int row = rem / padw, col = EW + rem - row * padw;
      sm.maps[q * map_stride + row * dp.ews + col] = 0.0f;
    }
    __syncthreads();

    // ------------------------------------------------------------------ a5 .. a9 ---------
    if (dp.psf_kind == GBK_PSF_IMAGE) {
      chi = conv2d_moments(dp, a, rc, k, sm.maps, map_stride, dp.ews, tw, th, tx0, ty0, sm.taps, tid,
                           nthreads);
    } else {
#define GBK_SEP_CASE(RR)                                                                        \
  case RR:                                                                                      \
    chi = separable_phase<RR>(dp, a, rc, k, sm.maps, map_stride, EH, tw, th, tx0, ty0, sm.taps, \
                              tid, nthreads);                                                   \
    break;
      switch (R) {
        GBK_SEP_CASE(0) GBK_SEP_CASE(1) GBK_SEP_CASE(2) GBK_SEP_CASE(3) GBK_SEP_CASE(4)
        GBK_SEP_CASE(5) GBK_SEP_CASE(6) GBK_SEP_CASE(7) GBK_SEP_CASE(8) GBK_SEP_CASE(9)
        GBK_SEP_CASE(10) GBK_SEP_CASE(11) GBK_SEP_CASE(12) GBK_SEP_CASE(13) GBK_SEP_CASE(14)
        GBK_SEP_CASE(15) GBK_SEP_CASE(16)
        default: break;
      }
#undef GBK_SEP_CASE
    }
  }

  // ------------------------------------------------ block reduction, fixed order ----------
#pragma unroll
  for (int off = 16; off > 0; off >>= 1) chi += __shfl_down_sync(0xffffffffu, chi, off);
  __syncthreads();  // all reads of the maps are done; red[] does not alias them, but keep order
  if ((tid & 31) == 0) sm.red[tid >> 5] = chi;
  __syncthreads();
  if (tid == 0) {
    float tot = 0.0f;
    for (int w = 0; w < (nthreads >> 5); ++w) tot += sm.red[w];
    if (!(tot < __int_as_float(0x7f800000))) tot = __int_as_float(0x7f800000);
    if (dp.ntiles == 1)
      a.chi2[k] = tot;
    else
      a.partial[bid] = tot;
  }
}

__global__ void finish_kernel(const float* __restrict__ partial, int ntiles, long long K,
                              float* __restrict__ chi2) {
  const long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= K) return;
  float tot = 0.0f;
  for (int t = 0; t < ntiles; ++t) tot += partial[k * ntiles + t];   // fixed order
  if (!(tot < __int_as_float(0x7f800000))) tot = __int_as_float(0x7f800000);
  chi2[k] = tot;
}

template <int P>
cudaError_t launch_p(const DevProblem& dp, const EvalArgs& a, const FusedLaunch& fl,
                     cudaStream_t st) {
  const long long nblocks = a.K * dp.ntiles;
  fused_kernel<P><<<(unsigned)nblocks, fl.threads, fl.smem_bytes, st>>>(dp, a);
  return cudaGetLastError();
}

template <int P>
cudaError_t prepare_p(const FusedLaunch& fl) {
  return cudaFuncSetAttribute(fused_kernel<P>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              fl.smem_bytes);
}

template <int P>
cudaError_t occupancy_p(const FusedLaunch& fl, int* n) {
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(n, fused_kernel<P>, fl.threads,
                                                       fl.smem_bytes);
}

}  // namespace

size_t fused_smem_bytes(const DevProblem& dp) {
  return sizeof(float) * 3 * (size_t)dp.ehs * dp.ews + sizeof(float4) * dp.nvx +
         sizeof(float) * round_up4(dp.psf_stride) + sizeof(RowConst) + sizeof(float) * 32;
}

cudaError_t fused_prepare(const FusedLaunch& fl) {
  return prepare_p<4>(fl);
}

cudaError_t fused_occupancy(const FusedLaunch& fl, int* n) {
  return occupancy_p<4>(fl, n);
}

cudaError_t launch_fused(const DevProblem& dp, const EvalArgs& a, const FusedLaunch& fl,
                         cudaStream_t st) {
  cudaError_t e = launch_p<4>(dp, a, fl, st);
  if (e != cudaSuccess) return e;
  if (dp.ntiles > 1) {
    const int th = 128;
    finish_kernel<<<(unsigned)((a.K + th - 1) / th), th, 0, st>>>(a.partial, dp.ntiles, a.K, a.chi2);
    e = cudaGetLastError();
  }
  return e;
}

// ------------------------------------------------------------------- pipe probes ------------
namespace {
__global__ void probe_mufu(long long iters, float* sink) {
  float x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = -1.0f - 0.001f * (threadIdx.x + i);
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int rep = 0; rep < 2; ++rep)
#pragma unroll
      for (int i = 0; i < 8; ++i) asm volatile("ex2.approx.ftz.f32 %0, %0;" : "+f"(x[i]));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  if (s == 12345.678f) sink[0] = s;
}
__global__ void probe_ffma(long long iters, float* sink) {
  float x[8];
  const float a = 0.999f, b = 0.001f;
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = 0.001f * (threadIdx.x + i);
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int rep = 0; rep < 2; ++rep)
#pragma unroll
      for (int i = 0; i < 8; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  if (s == 12345.678f) sink[0] = s;
}
}  // namespace

cudaError_t launch_probe(int which, long long iters, int blocks, int threads, float* sink,
                         cudaStream_t st) {
  if (which == 0)
    probe_mufu<<<blocks, threads, 0, st>>>(iters, sink);
  else
    probe_ffma<<<blocks, threads, 0, st>>>(iters, sink);
  return cudaGetLastError();
}

}  // namespace gbk
