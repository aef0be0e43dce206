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

#include "gbk_device.cuh"
#include "gbk_internal.h"

namespace gbk {

namespace {

struct URow {          // constants of one parameter row (a1)
  float xo, yo, sp, cp, si, inv_ci, vsys, vt, inv_rt, inv_r0, i0, sigma0, ea, eg;
  int gal, psf_set, r_p, valid;
  int precise;         // a line may be centred well outside the band: FP64 geometry (as in the fused kernel)
  double dsp, dcp, dsi, dinv_ci, drt;
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
  // the fused kernel's criterion: only the far wing of such a line is in the band, where
  // the voxel values need the line offset to ~1e-6 sigma_0
  const float s = 1.0f / (p[7] * 1.1774100225154747f);
  const float k1 = -s * (dp.rc_model == GBK_RC_ARCTAN ? 0.63661977236758134f : 1.0f) * p[5] * r.si;
  const float k0 = s * dp.vrel_first - s * (p[4] - dp.v_center);
  r.precise = r.valid && line_leaves_band(dp, k0, k1, curve_sup(dp, p, r.inv_ci), s * dp.dv, kPreciseMargin);
  r.dsp = r.dcp = r.dsi = r.dinv_ci = 0.0, r.drt = (double)p[6];
  if (r.precise) {
    double dci;
    sincospi((double)p[2] * (1.0 / 180.0), &r.dsp, &r.dcp);
    sincospi((double)p[3] * (1.0 / 180.0), &r.dsi, &dci);
    r.dinv_ci = 1.0 / dci;
  }
  return r;
}

// a1 once per row of the chunk (the step kernels read the constants instead of re-deriving them)
__global__ void uf_rows_kernel(const __grid_constant__ DevProblem dp, const float* __restrict__ params,
                               const int32_t* __restrict__ gal_index, long long k0, int nrows,
                               URow* __restrict__ rows) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nrows) rows[i] = uf_row(dp, params, gal_index, k0 + i);
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
__global__ void uf_cube_kernel(const __grid_constant__ DevProblem dp, const URow* __restrict__ rows, int nrows,
                               float* __restrict__ cube) {
  const UGeom g = uf_geom(dp);
  const long long n = (long long)nrows * g.plane;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / g.plane);
    const int pix = (int)(idx - row * (long long)g.plane);
    const int ey = pix / g.EW, ex = pix - ey * g.EW;
    const URow r = rows[row];
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
    if (r.precise) {   // the same formulas with the line offset in FP64 (rare rows)
      const double dx = ((double)(ex - g.R) + 0.5) / (double)dp.u - 0.5 - (double)r.xo;
      const double dy = ((double)(ey - g.R) + 0.5) / (double)dp.u - 0.5 - (double)r.yo;
      const double dxe = -dx * r.dsp + dy * r.dcp, dye = (-dx * r.dcp - dy * r.dsp) * r.dinv_ci;
      const double drad = sqrt(dxe * dxe + dye * dye);
      const double dcos = drad > 0.0 ? dxe / drad : 0.0;
      const double dq = drad / r.drt;
      double dvrot;
      if (dp.rc_model == GBK_RC_ARCTAN) dvrot = 0.63661977236758134 * (double)r.vt * atan(dq);
      else if (dp.rc_model == GBK_RC_RAMP) dvrot = (double)r.vt * fmin(dq, 1.0);
      else dvrot = dq > 0.0 ? (double)r.vt * pow(dq, (double)r.eg) / (1.0 + pow(dq, (double)r.ea)) : 0.0;
      const double dvlos = ((double)r.vsys - (double)dp.v_center) + dvrot * r.dsi * dcos;
      const double first = (-(double)dp.r_v - 0.5 * (double)(dp.nv - 1)) * (double)dp.dv - dvlos;
      const double dinv_s = 1.0 / (double)r.sigma0;
      for (int c = 0; c < g.nvx; ++c) {
        const float t = (float)(((double)c * (double)dp.dv + first) * dinv_s);
        out[(size_t)c * g.plane] = amp * expf(-0.5f * t * t);
      }
      continue;
    }
    for (int c = 0; c < g.nvx; ++c) {
      const float t = (dp.vrel_first + (float)c * dp.dv - vlos) * inv_s;
      out[(size_t)c * g.plane] = amp * expf(-0.5f * t * t);
    }
  }
}

// Step 2a: LSF along v (direct sum, "valid": nvx -> nv channels), lsf[j], j = 0..2 r_v.  A block
// takes 32 consecutive pixels of one row's plane and walks the channels in pieces of kLsfPiece: the
// slab [piece + 2 r_v][32] goes through shared memory, so every input value is read from device
// memory once (128-byte coalesced lines) however many taps use it.
constexpr int kLsfPiece = 64, kLsfPix = 64;       // channels per piece, pixels per block pass (2 per lane)
__global__ void __launch_bounds__(256) uf_lsf_kernel(const __grid_constant__ DevProblem dp,
                                                     const float* __restrict__ lsf, int nrows,
                                                     const float* __restrict__ in, float* __restrict__ out) {
  extern __shared__ float slab[];                 // [kLsfPiece + 2 r_v][kLsfPix]
  __shared__ float taps[2 * kMaxLsfR + 1];
  const UGeom g = uf_geom(dp);
  const int ntap = 2 * dp.r_v + 1;
  for (int j = threadIdx.x; j < ntap; j += blockDim.x) taps[j] = lsf[j];
  const int lane = threadIdx.x & 31, grp = threadIdx.x >> 5, ngrp = blockDim.x >> 5;
  const long long nseg = ((long long)g.plane + kLsfPix - 1) / kLsfPix;
  for (long long job = blockIdx.x; job < (long long)nrows * nseg; job += gridDim.x) {
    const int row = (int)(job / nseg);
    const size_t pix = (size_t)(job - (long long)row * nseg) * kLsfPix + lane;
    const bool live0 = pix < g.plane, live1 = pix + 32 < g.plane;
    const float* src = in + (size_t)row * g.cube + pix;
    float* dst = out + (size_t)row * g.cube + pix;
    for (int c0 = 0; c0 < dp.nv; c0 += kLsfPiece) {
      const int nc = min(kLsfPiece, dp.nv - c0);
      __syncthreads();
#pragma unroll 4
      for (int c = grp; c < nc + ntap - 1; c += ngrp) {
        const float* q = src + (size_t)(c0 + c) * g.plane;
        slab[c * kLsfPix + lane] = live0 ? q[0] : 0.0f;
        slab[c * kLsfPix + lane + 32] = live1 ? q[32] : 0.0f;
      }
      __syncthreads();
      for (int c = grp; c < nc; c += ngrp) {      // out[c] = sum_j L[j] in[c - j]  (extended index c + r_v - j)
        float sa = 0.0f, sb = 0.0f;
        for (int j = 0; j < ntap; ++j) {
          const float t = taps[j];
          sa = fmaf(t, slab[(c + ntap - 1 - j) * kLsfPix + lane], sa);
          sb = fmaf(t, slab[(c + ntap - 1 - j) * kLsfPix + lane + 32], sb);
        }
        float* q = dst + (size_t)(c0 + c) * g.plane;
        if (live0) q[0] = sa;
        if (live1) q[32] = sb;
      }
    }
  }
}

// Step 2a for the usual small LSF radii (RV <= kLsfRegMaxR): no shared memory at all.  A thread owns one pixel and
// walks its channels with the last 2 RV + 1 inputs in a register ring (static indices: the loop is unrolled by
// the ring length), so every input is loaded from device memory exactly once, 128-byte coalesced across the
// warp, with a whole group of 2 RV + 1 loads in flight per thread; 2 RV + 1 FMAs per output and nothing else.
constexpr int kLsfRegMaxR = 6;
template <int RV>
__global__ void __launch_bounds__(256, 4) uf_lsf_reg_kernel(const __grid_constant__ DevProblem dp,
                                                         const float* __restrict__ lsf, int nrows,
                                                         const float* __restrict__ in, float* __restrict__ out) {
  constexpr int NT = 2 * RV + 1;
  float L[NT];
#pragma unroll
  for (int j = 0; j < NT; ++j) L[j] = lsf[j];
  const UGeom g = uf_geom(dp);
  const long long n = (long long)nrows * (long long)g.plane;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / (long long)g.plane);
    const size_t pix = (size_t)(idx - (long long)row * (long long)g.plane);
    const float* src = in + (size_t)row * g.cube + pix;
    float* dst = out + (size_t)row * g.cube + pix;
    // a group of NT outputs c .. c + NT - 1 needs the inputs c .. c + 2 NT - 2: NT - 1 carried over from the
    // group before, NT new ones, which are requested one group ahead (`nxt`) so that their latency hides
    // behind the arithmetic of the current group
    float v[2 * NT - 1], nxt[NT];
#pragma unroll
    for (int e = 0; e < NT - 1; ++e) v[e] = src[(size_t)e * g.plane];
#pragma unroll
    for (int e = 0; e < NT; ++e) nxt[e] = e < dp.nv ? src[(size_t)(NT - 1 + e) * g.plane] : 0.0f;
    for (int c = 0; c < dp.nv; c += NT) {
#pragma unroll
      for (int e = 0; e < NT; ++e) v[NT - 1 + e] = nxt[e];
#pragma unroll
      for (int e = 0; e < NT; ++e)                 // inputs of the next group (output c + NT + e exists)
        nxt[e] = c + NT + e < dp.nv ? src[(size_t)(c + 2 * NT - 1 + e) * g.plane] : 0.0f;
#pragma unroll
      for (int k = 0; k < NT; ++k)
        if (c + k < dp.nv) {
          float sum = 0.0f;
#pragma unroll
          for (int j = 0; j < NT; ++j) sum = fmaf(L[j], v[k + NT - 1 - j], sum);   // out[c] = sum_j L[j] in[c - j]
          dst[(size_t)(c + k) * g.plane] = sum;
        }
#pragma unroll
      for (int e = 0; e < NT - 1; ++e) v[e] = v[NT + e];
    }
  }
}

constexpr int kPsfTileW = 64;
constexpr int kPsfMidW = kPsfTileW + 4;   // row stride of the intermediate: 16-byte rows
// The two passes of one tile from shared memory (shared by the two kernels below): x pass tin -> tmid, y pass
// tmid -> device memory.
template <int R, int IW, int IH>
__device__ __forceinline__ void psf_tile_passes(const float (*tin)[IW], float (*tmid)[kPsfMidW], const float* taps,
                                                int tw, int th, float* dst, int fw) {
  // Tap pairs for packed FP32 (FFMA2): an output pair (o[x], o[x+1]) receives from input v[i],
  // i = 0..2R+1, the pair (f[i], f[i-1]) of flipped taps f[j] = taps[2R - j] (f[-1] = f[2R+1] = 0)
  // times the broadcast input, i.e. 2R + 2 instructions per two outputs instead of 2 (2R + 1).
  u64 tp[2 * R + 2];
#pragma unroll
  for (int i = 0; i < 2 * R + 2; ++i)
    tp[i] = pk(i <= 2 * R ? taps[2 * R - i] : 0.0f, i >= 1 ? taps[2 * R - (i - 1)] : 0.0f);
  constexpr int NX4 = kPsfTileW / 4;
  for (int i = threadIdx.x; i < (th + 2 * R) * NX4; i += blockDim.x) {      // x pass
    const int yy = i / NX4, xx = (i - yy * NX4) * 4;
    float v[4 + 2 * R + 3];
#pragma unroll
    for (int q = 0; q < (4 + 2 * R + 3) / 4; ++q) {
      const float4 f = *reinterpret_cast<const float4*>(&tin[yy][xx + 4 * q]);
      v[4 * q] = f.x, v[4 * q + 1] = f.y, v[4 * q + 2] = f.z, v[4 * q + 3] = f.w;
    }
    u64 o01 = pk(0.f, 0.f), o23 = o01;
#pragma unroll
    for (int j = 0; j < 2 * R + 2; ++j) {
      o01 = fma2(tp[j], pk1(v[j]), o01);
      o23 = fma2(tp[j], pk1(v[j + 2]), o23);
    }
    float4 o;
    upk(o01, o.x, o.y);
    upk(o23, o.z, o.w);
    *reinterpret_cast<float4*>(&tmid[yy][xx]) = o;
  }
  __syncthreads();
  // y pass: a thread owns a column PAIR (one 8-byte read per row, both columns in one FFMA2 with the tap as the
  // broadcast scalar operand) and 4 output rows: 4 (2R + 1) FFMA2 and 4 + 2R reads for 8 outputs
  float f[2 * R + 1];                    // out[y] = sum_t f[t] in[y + t], f[t] = taps[2R - t] as in the x pass
#pragma unroll
  for (int t = 0; t < 2 * R + 1; ++t) f[t] = taps[2 * R - t];
  const int ny4 = (th + 3) / 4, nxp = (tw + 1) >> 1;
  const bool pair_store = (fw & 1) == 0 && (reinterpret_cast<size_t>(dst) & 7) == 0;
  for (int i = threadIdx.x; i < ny4 * nxp; i += blockDim.x) {
    const int yb = i / nxp, xx = (i - yb * nxp) << 1, yy = yb * 4;
    u64 acc[4];
#pragma unroll
    for (int m = 0; m < 4; ++m) acc[m] = pk(0.f, 0.f);
    const bool inside = yy + 4 + 2 * R <= IH;   // all 4 + 2R rows lie inside tmid (always, for a full tile): no checks;
                                                // rows past th + 2R hold older values and only feed outputs not stored
#pragma unroll
    for (int j = 0; j < 4 + 2 * R; ++j) {
      u64 v = pk(0.f, 0.f);
      if (inside || yy + j < th + 2 * R) v = *reinterpret_cast<const u64*>(&tmid[yy + j][xx]);
#pragma unroll
      for (int m = 0; m < 4; ++m)
        if (j - m >= 0 && j - m <= 2 * R) acc[m] = fma2(pk1(f[j - m]), v, acc[m]);
    }
#pragma unroll
    for (int m = 0; m < 4; ++m)
      if (yy + m < th) {
        float* q = dst + (size_t)(yy + m) * fw + xx;
        float oa, ob;
        upk(acc[m], oa, ob);
        if (pair_store && xx + 1 < tw) {
          *reinterpret_cast<float2*>(q) = make_float2(oa, ob);
        } else {
          q[0] = oa;
          if (xx + 1 < tw) q[1] = ob;
        }
      }
  }
}

// Step 2b, separable Gaussian PSF: both 1-D passes in one kernel.  A block takes one tile of one
// channel of one row: the extended tile (tile + 2R each way) is read once into shared memory, the x
// pass writes an intermediate (tile width x extended height) there, the y pass writes the fine-grid
// result to device memory; a thread produces 4 consecutive outputs per pass from 4 + 2R inputs held
// in registers.  R is the problem's largest tap radius; a data set with a narrower PSF has its taps
// centred and zero-padded to that radius (the same sums).
// in: extended layout [row][c][EH][EW]; out: compact [row][c][fh][fw].
template <int R>
__global__ void __launch_bounds__(256) uf_psf_sep_kernel(const __grid_constant__ DevProblem dp,
                                                         const URow* __restrict__ rows, int nrows,
                                                         const float* __restrict__ in, float* __restrict__ out) {
  constexpr int kPsfTileH = R <= 8 ? 64 : 32;     // the taller tile has less halo; R > 8 would not fit 48 KB
  constexpr int IW = (kPsfTileW + 2 * R + 3) & ~3, IH = kPsfTileH + 2 * R;
  __shared__ __align__(16) float tin[IH][IW];
  __shared__ __align__(16) float tmid[IH][kPsfMidW];
  __shared__ float taps[2 * R + 1];
  const UGeom g = uf_geom(dp);
  const int ntx = (dp.fw + kPsfTileW - 1) / kPsfTileW, nty = (dp.fh + kPsfTileH - 1) / kPsfTileH;
  const long long per_row = (long long)dp.nv * ntx * nty;
  for (long long job = blockIdx.x; job < (long long)nrows * per_row; job += gridDim.x) {
    const int row = (int)(job / per_row);
    long long rem = job - (long long)row * per_row;
    const int c = (int)(rem / (ntx * nty));
    rem -= (long long)c * ntx * nty;
    const int ty = (int)(rem / ntx), tx = (int)(rem - (long long)ty * ntx);
    const URow r = rows[row];
    __syncthreads();
    if (threadIdx.x < 2 * R + 1) {
      const int idx = (int)threadIdx.x - (R - r.r_p);
      taps[threadIdx.x] = idx >= 0 && idx <= 2 * r.r_p ? dp.psf_taps[(size_t)r.psf_set * dp.psf_stride + idx] : 0.0f;
    }
    const int x0 = tx * kPsfTileW, y0 = ty * kPsfTileH;
    const int tw = min(kPsfTileW, dp.fw - x0), th = min(kPsfTileH, dp.fh - y0);
    const float* src = in + (size_t)row * g.cube + (size_t)c * g.plane + (size_t)y0 * g.EW + x0;
    if ((g.EW & 3) == 0 && (reinterpret_cast<size_t>(src) & 15) == 0 && tw == kPsfTileW) {
      for (int i = threadIdx.x; i < (th + 2 * R) * (IW / 4); i += blockDim.x) {   // 16-byte loads
        const int yy = i / (IW / 4), xx = (i - yy * (IW / 4)) * 4;
        float4 f = make_float4(0.f, 0.f, 0.f, 0.f);
        if (xx + 3 < tw + 2 * R) {
          f = *reinterpret_cast<const float4*>(src + (size_t)yy * g.EW + xx);
        } else {
          if (xx < tw + 2 * R) f.x = src[(size_t)yy * g.EW + xx];
          if (xx + 1 < tw + 2 * R) f.y = src[(size_t)yy * g.EW + xx + 1];
          if (xx + 2 < tw + 2 * R) f.z = src[(size_t)yy * g.EW + xx + 2];
        }
        *reinterpret_cast<float4*>(&tin[yy][xx]) = f;
      }
    } else {
      for (int i = threadIdx.x; i < (th + 2 * R) * IW; i += blockDim.x) {
        const int yy = i / IW, xx = i - yy * IW;
        tin[yy][xx] = xx < tw + 2 * R ? src[(size_t)yy * g.EW + xx] : 0.0f;
      }
    }
    __syncthreads();
    float* dst = out + (size_t)row * g.cube + (size_t)c * dp.fw * dp.fh + (size_t)y0 * dp.fw + x0;
    psf_tile_passes<R, IW, IH>(tin, tmid, taps, tw, th, dst, dp.fw);
  }
}

// The same step with the tile loads taken off the critical path: the block walks its jobs with TWO input
// buffers and requests the tile of its next job with cp.async (16-byte copies straight into shared memory)
// before it computes the current one, so a block always has a tile in flight.  For the aligned case only
// (extended rows a multiple of 16 bytes, full-width tiles): the launcher falls back to the kernel above otherwise.
template <int R>
__global__ void __launch_bounds__(256) uf_psf_sep_pipe_kernel(const __grid_constant__ DevProblem dp,
                                                              const URow* __restrict__ rows, int nrows,
                                                              const float* __restrict__ in, float* __restrict__ out) {
  constexpr int kPsfTileH = R <= 8 ? 64 : 32;
  constexpr int IW = (kPsfTileW + 2 * R + 3) & ~3, IH = kPsfTileH + 2 * R;
  extern __shared__ __align__(16) unsigned char psf_smem[];
  float (*tin0)[IW] = reinterpret_cast<float (*)[IW]>(psf_smem);
  float (*tin1)[IW] = reinterpret_cast<float (*)[IW]>(psf_smem + sizeof(float) * IH * IW);
  float (*tmid)[kPsfMidW] = reinterpret_cast<float (*)[kPsfMidW]>(psf_smem + 2 * sizeof(float) * IH * IW);
  __shared__ float taps[2 * R + 1];
  const UGeom g = uf_geom(dp);
  const int ntx = dp.fw / kPsfTileW, nty = (dp.fh + kPsfTileH - 1) / kPsfTileH;
  const long long per_row = (long long)dp.nv * ntx * nty, njobs = (long long)nrows * per_row;
  struct Job {
    int row, c, x0, y0, th;
  };
  auto decode = [&](long long job) {
    Job j;
    j.row = (int)(job / per_row);
    long long rem = job - (long long)j.row * per_row;
    j.c = (int)(rem / (ntx * nty));
    rem -= (long long)j.c * ntx * nty;
    const int ty = (int)(rem / ntx), tx = (int)(rem - (long long)ty * ntx);
    j.x0 = tx * kPsfTileW, j.y0 = ty * kPsfTileH;
    j.th = min(kPsfTileH, dp.fh - j.y0);
    return j;
  };
  auto request = [&](const Job& j, float (*buf)[IW]) {      // all IW columns lie inside the extended row
    const float* src = in + (size_t)j.row * g.cube + (size_t)j.c * g.plane + (size_t)j.y0 * g.EW + j.x0;
    for (int i = threadIdx.x; i < (j.th + 2 * R) * (IW / 4); i += blockDim.x) {
      const int yy = i / (IW / 4), xx = (i - yy * (IW / 4)) * 4;
      const unsigned dst = (unsigned)__cvta_generic_to_shared(&buf[yy][xx]);
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src + (size_t)yy * g.EW + xx) : "memory");
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  long long job = blockIdx.x;
  if (job < njobs) request(decode(job), tin0);
  int cur = 0;
  for (; job < njobs; job += gridDim.x, cur ^= 1) {
    const Job j = decode(job);
    const long long next = job + gridDim.x;
    // the other buffer was last read by the x pass of the job before this one, which every thread has left
    // (barrier after that pass), so it is free
    if (next < njobs) {
      request(decode(next), cur ? tin0 : tin1);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    const URow r = rows[j.row];
    if (threadIdx.x < 2 * R + 1) {     // nobody reads `taps` or `tmid` of the previous job any more: see the last barrier
      const int idx = (int)threadIdx.x - (R - r.r_p);
      taps[threadIdx.x] = idx >= 0 && idx <= 2 * r.r_p ? dp.psf_taps[(size_t)r.psf_set * dp.psf_stride + idx] : 0.0f;
    }
    __syncthreads();                   // this job's tile (everybody's copies) and taps are visible
    float* dst = out + (size_t)j.row * g.cube + (size_t)j.c * dp.fw * dp.fh + (size_t)j.y0 * dp.fw + j.x0;
    psf_tile_passes<R, IW, IH>(cur ? tin1 : tin0, tmid, taps, kPsfTileW, j.th, dst, dp.fw);
    __syncthreads();                   // the y pass is done with tmid and taps before the next job rewrites them
  }
}

// Step 2b for a general PSF image: direct 2-D sum from a shared-memory tile.  The image is stored
// flipped at create, so this correlation is the true convolution (A11).
constexpr int kImgTile = 32;
__global__ void __launch_bounds__(256) uf_psf2d_kernel(const __grid_constant__ DevProblem dp,
                                                       const URow* __restrict__ rows, int nrows,
                                                       const float* __restrict__ in, float* __restrict__ out) {
  extern __shared__ float sh[];                   // [(kImgTile + 2R)^2] tile, then [n^2] taps
  const UGeom g = uf_geom(dp);
  const int Rm = g.R;
  const int ntx = (dp.fw + kImgTile - 1) / kImgTile, nty = (dp.fh + kImgTile - 1) / kImgTile;
  const long long per_row = (long long)dp.nv * ntx * nty;
  for (long long job = blockIdx.x; job < (long long)nrows * per_row; job += gridDim.x) {
    const int row = (int)(job / per_row);
    long long rem = job - (long long)row * per_row;
    const int c = (int)(rem / (ntx * nty));
    rem -= (long long)c * ntx * nty;
    const int ty = (int)(rem / ntx), tx = (int)(rem - (long long)ty * ntx);
    const URow r = rows[row];
    const int R = r.r_p, n = 2 * R + 1, iw = kImgTile + 2 * Rm;
    float* tile = sh;
    float* taps = sh + iw * iw;
    const int x0 = tx * kImgTile, y0 = ty * kImgTile;
    const int tw = min(kImgTile, dp.fw - x0), th = min(kImgTile, dp.fh - y0);
    __syncthreads();
    for (int i = threadIdx.x; i < n * n; i += blockDim.x) taps[i] = dp.psf_taps[(size_t)r.psf_set * dp.psf_stride + i];
    const float* src = in + (size_t)row * g.cube + (size_t)c * g.plane + (size_t)(y0 + Rm - R) * g.EW + x0 + Rm - R;
    for (int i = threadIdx.x; i < (th + 2 * R) * (tw + 2 * R); i += blockDim.x) {
      const int yy = i / (tw + 2 * R), xx = i - yy * (tw + 2 * R);
      tile[yy * iw + xx] = src[(size_t)yy * g.EW + xx];
    }
    __syncthreads();
    float* dst = out + (size_t)row * g.cube + (size_t)c * dp.fw * dp.fh + (size_t)y0 * dp.fw + x0;
    for (int i = threadIdx.x; i < th * tw; i += blockDim.x) {
      const int yy = i / tw, xx = i - yy * tw;
      float sum = 0.0f;
      for (int ky = 0; ky < n; ++ky)
        for (int kx = 0; kx < n; ++kx) sum = fmaf(taps[ky * n + kx], tile[(yy + ky) * iw + xx + kx], sum);
      dst[(size_t)yy * dp.fw + xx] = sum;
    }
  }
}

// Steps 3-5: per spaxel, down-sample every channel (mean over the u x u block),
// moments, residuals against the packed observation, and the spaxel's chi^2 contribution.  One pass
// over the spectrum with the weighted running-mean update (W' = W + w; mean += (w / W')(v - mean);
// M2 += (v - mean_old)^2 W w / W'), velocities from a reference close to the line (V_sys clamped
// to the band, as in the fused kernel): m1 = mean, m2^2 = M2 / W.  Unlike S2/S0 - m1^2 this does not
// cancel where a line centred far outside the band leaves m2 << dv.
__global__ void uf_moments_kernel(const __grid_constant__ DevProblem dp, const URow* __restrict__ rows,
                                  long long k0, int nrows, const float* __restrict__ cube,
                                  float* __restrict__ contrib, const EvalArgs a) {
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
    const URow r = rows[row];
    const float4 ob = dp.obs[(size_t)r.gal * npix + pix];
    const bool unmasked = ob.y > 0.0f;
    float m0 = nan, m1 = nan, m2 = nan, t = nan, s = nan, c2 = inf;
    if (r.valid) {
      // the convolved cube is compact: [row][c][fh][fw]
      const size_t cplane = (size_t)dp.fw * dp.fh;
      const float* src = cube + (size_t)row * g.cube + (size_t)(Y * dp.u) * dp.fw + X * dp.u;
      const float v_ref = fminf(fmaxf(r.vsys - dp.v_center, -dp.vhalf), dp.vhalf);
      const float v_first = -dp.vhalf - v_ref;                               // channel 0 from the reference
      float s0 = 0.0f, mean = 0.0f, s2 = 0.0f;
      if (dp.u == 1) {
#pragma unroll 8
        for (int c = 0; c < dp.nv; ++c) {
          const float blk = src[(size_t)c * cplane];
          const float v = fmaf((float)c, dp.dv, v_first);
          const float w_old = s0;
          s0 += blk;
          const float dl = v - mean, rw = s0 > 0.0f ? __fdividef(blk, s0) : 0.0f;
          mean = fmaf(rw, dl, mean);
          s2 = fmaf(dl * dl, w_old * rw, s2);
        }
      } else {
        for (int c = 0; c < dp.nv; ++c) {
          float blk = 0.0f;
          for (int dy = 0; dy < dp.u; ++dy)
            for (int dx = 0; dx < dp.u; ++dx) blk += src[(size_t)c * cplane + (size_t)dy * dp.fw + dx];
          blk *= dp.inv_u2;
          const float v = fmaf((float)c, dp.dv, v_first);
          const float w_old = s0;
          s0 += blk;
          const float dl = v - mean, rw = s0 > 0.0f ? __fdividef(blk, s0) : 0.0f;
          mean = fmaf(rw, dl, mean);
          s2 = fmaf(dl * dl, w_old * rw, s2);
        }
      }
      m0 = s0;
      m1 = s0 > 0.0f ? mean : nan;
      const float var = s2 / s0;
      m2 = var > 0.0f ? sqrtf(var) : (var == var ? 0.0f : var);            // A5
      const bool dark = !(m0 >= 1e-30f * r.i0);                             // A15
      t = (m1 + (v_ref - ob.x)) * ob.y;
      s = (m2 - ob.z) * ob.w;
      c2 = fmaf(t, t, s * s);
      const bool bad = dark || !(c2 < inf);
      if (dark) m1 = m2 = nan;
      if (!unmasked) t = s = 0.0f, c2 = 0.0f;
      else if (bad) t = s = nan, c2 = inf;
      m1 += v_ref + dp.v_center;
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

// Steps 3-5 with the Gaussian-profile extraction the paper describes as the alternative to moments
// (reading A23 of DESIGN.md): per spaxel, down-sample every
// channel, fit A exp(-(v - mu)^2 / (2 s^2)) to the spectrum by unweighted least squares (Levenberg-
// Marquardt started from the moments; the 3 x 3 normal equations in FP64), velocity = mu,
// dispersion = s, m0 = the plain sum; then residuals and the chi^2 contribution as usual.  The fit
// needs the whole convolved spectrum of a spaxel, so it cannot use the moment-first identity of the
// fused kernel: it runs on this pipeline only.  A fit that does not converge gives NaN maps and, at an
// unmasked spaxel, chi^2 = +INF ("may occasionally fail to converge").
__device__ __forceinline__ float uf_spaxel_channel(const DevProblem& dp, const float* src, size_t cplane, int c) {
  float blk = 0.0f;
  for (int dy = 0; dy < dp.u; ++dy)
    for (int dx = 0; dx < dp.u; ++dx) blk += src[(size_t)c * cplane + (size_t)dy * dp.fw + dx];
  return blk * dp.inv_u2;
}

__global__ void uf_gaussfit_kernel(const __grid_constant__ DevProblem dp, const URow* __restrict__ rows,
                                   long long k0, int nrows, const float* __restrict__ cube,
                                   float* __restrict__ contrib, const EvalArgs a) {
  const UGeom g = uf_geom(dp);
  const int npix = dp.nx * dp.ny, nv = dp.nv;
  const long long n = (long long)nrows * npix;
  const float inf = __int_as_float(0x7f800000), nan = __int_as_float(0x7fc00000);
  const double dv = dp.dv, v_first = -0.5 * (double)(nv - 1) * dv;            // velocities from v_center
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < n;
       idx += (long long)gridDim.x * blockDim.x) {
    const int row = (int)(idx / npix);
    const int pix = (int)(idx - (long long)row * npix);
    const int Y = pix / dp.nx, X = pix - Y * dp.nx;
    const long long k = k0 + row;
    const URow r = rows[row];
    const float4 ob = dp.obs[(size_t)r.gal * npix + pix];
    const bool unmasked = ob.y > 0.0f;
    float m0 = nan, m1 = nan, m2 = nan, t = nan, s = nan, c2 = inf;
    if (r.valid) {
      const size_t cplane = (size_t)dp.fw * dp.fh;
      const float* src = cube + (size_t)row * g.cube + (size_t)(Y * dp.u) * dp.fw + X * dp.u;
      double s0 = 0.0, s1 = 0.0;
      for (int c = 0; c < nv; ++c) {
        const double v = uf_spaxel_channel(dp, src, cplane, c);
        s0 += v;
        s1 += v * (v_first + c * dv);
      }
      const double mean = s1 / s0;
      double s2 = 0.0;
      for (int c = 0; c < nv; ++c) {
        const double d = v_first + c * dv - mean;
        s2 += (double)uf_spaxel_channel(dp, src, cplane, c) * d * d;
      }
      const double var = s2 / s0;
      m0 = (float)s0;
      bool done = false;
      double mu = mean, sg = fmax(sqrt(fmax(var, 0.0)), 0.5 * dv);
      if (s0 > 0.0 && isfinite(mean) && isfinite(var)) {
        double A = s0 * dv / (sg * 2.5066282746310002);
        double lambda = 1e-3;
        for (int it = 0; it < 200 && !done; ++it) {
          double j00 = 0, j01 = 0, j02 = 0, j11 = 0, j12 = 0, j22 = 0, r0 = 0, r1 = 0, r2 = 0, sse = 0;
          const double is2 = 1.0 / (sg * sg);
          for (int c = 0; c < nv; ++c) {
            const double d = v_first + c * dv - mu;
            const double e = exp(-0.5 * d * d * is2);
            const double res = (double)uf_spaxel_channel(dp, src, cplane, c) - A * e;
            const double J0 = e, J1 = A * e * d * is2, J2 = J1 * d / sg;
            j00 += J0 * J0, j01 += J0 * J1, j02 += J0 * J2, j11 += J1 * J1, j12 += J1 * J2, j22 += J2 * J2;
            r0 += J0 * res, r1 += J1 * res, r2 += J2 * res;
            sse += res * res;
          }
          if (sse <= 1e-28 * s0 * s0) {
            done = true;
            break;
          }
          // (J^T J + lambda diag) delta = J^T r by Cramer's rule
          const double a00 = j00 * (1.0 + lambda), a11 = j11 * (1.0 + lambda), a22 = j22 * (1.0 + lambda);
          const double det = a00 * (a11 * a22 - j12 * j12) - j01 * (j01 * a22 - j12 * j02) + j02 * (j01 * j12 - a11 * j02);
          const double d0 = (r0 * (a11 * a22 - j12 * j12) - j01 * (r1 * a22 - j12 * r2) + j02 * (r1 * j12 - a11 * r2)) / det;
          const double d1 = (a00 * (r1 * a22 - j12 * r2) - r0 * (j01 * a22 - j12 * j02) + j02 * (j01 * r2 - r1 * j02)) / det;
          const double d2 = (a00 * (a11 * r2 - r1 * j12) - j01 * (j01 * r2 - r1 * j02) + r0 * (j01 * j12 - a11 * j02)) / det;
          const double A1 = A + d0, mu1 = mu + d1, sg1 = sg + d2;
          double sse1 = INFINITY;
          if (isfinite(A1) && isfinite(mu1) && sg1 > 0.0 && sg1 < 1e3 * nv * dv) {
            sse1 = 0.0;
            const double is21 = 1.0 / (sg1 * sg1);
            for (int c = 0; c < nv; ++c) {
              const double d = v_first + c * dv - mu1;
              const double res = (double)uf_spaxel_channel(dp, src, cplane, c) - A1 * exp(-0.5 * d * d * is21);
              sse1 += res * res;
            }
          }
          if (sse1 < sse) {
            A = A1, mu = mu1, sg = sg1;
            lambda = fmax(lambda / 10.0, 1e-12);
            if (fabs(d1) < 1e-6 * dv && fabs(d2) < 1e-6 * dv) done = true;
          } else {
            lambda *= 10.0;
            if (!(lambda <= 1e12)) break;
          }
        }
      }
      if (done) m1 = (float)mu, m2 = (float)sg;
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
  return sizeof(float) * (2 * g.cube + (size_t)dp.nx * dp.ny) + sizeof(URow) + 16;   // + 16: URow alignment
}

// Algorithmic HBM bytes of the unfused pipeline per row: every array written once and read once by
// the step that consumes it (cube: written, read by the LSF; LSF output: written, read by the PSF
// kernel; convolved cube: written, read by the extraction kernel, whose second pass over a spectrum
// comes from cache).
double unfused_algorithmic_bytes_per_row(const DevProblem& dp) {
  const UGeom g = uf_geom(dp);
  const double ext = (double)g.cube, lsf = (double)g.plane * dp.nv, fine = (double)dp.fw * dp.fh * dp.nv;
  return 4.0 * (2.0 * ext + 2.0 * lsf + 2.0 * fine);
}

namespace {
template <int R>
void launch_psf_sep(const DevProblem& dp, const URow* rows, int n, unsigned cap, const float* in, float* out,
                    cudaStream_t st) {
  constexpr int th = R <= 8 ? 64 : 32;
  const long long jobs = (long long)n * dp.nv * ((dp.fw + kPsfTileW - 1) / kPsfTileW) * ((dp.fh + th - 1) / th);
  const UGeom g = uf_geom(dp);
  constexpr int IW = (kPsfTileW + 2 * R + 3) & ~3, IH = th + 2 * R;
  // cp.async pipeline: every 16-byte copy must be aligned and inside the extended row (IW <= EW)
  const bool aligned = (g.EW & 3) == 0 && dp.fw % kPsfTileW == 0 && IW <= g.EW && (reinterpret_cast<uintptr_t>(in) & 15) == 0 &&
                       (g.plane & 3) == 0 && (g.cube & 3) == 0;
  if (aligned) {
    const size_t smem = sizeof(float) * (2 * (size_t)IH * IW + (size_t)IH * kPsfMidW);
    // per device and cheap: set on every launch rather than remembered (the library serves several devices)
    cudaFuncSetAttribute(uf_psf_sep_pipe_kernel<R>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    const unsigned blocks = (unsigned)std::min<long long>(jobs, cap);
    uf_psf_sep_pipe_kernel<R><<<blocks, 256, smem, st>>>(dp, rows, n, in, out);
    return;
  }
  uf_psf_sep_kernel<R><<<(unsigned)std::min<long long>(jobs, cap), 256, 0, st>>>(dp, rows, n, in, out);
}
}  // namespace

cudaError_t launch_unfused(const DevProblem& dp, const EvalArgs& a, const float* lsf_taps, float* scratch,
                           long long chunk_rows, int sm_count, int extraction, cudaStream_t st) {
  const UGeom g = uf_geom(dp);
  const int T = 256, npix = dp.nx * dp.ny;
  float* A = scratch;
  float* B = A + (size_t)chunk_rows * g.cube;
  float* contrib = B + (size_t)chunk_rows * g.cube;
  const uintptr_t rows_at = reinterpret_cast<uintptr_t>(contrib + (size_t)chunk_rows * npix);
  URow* rows = reinterpret_cast<URow*>((rows_at + 15) & ~(uintptr_t)15);   // URow holds doubles
  const unsigned wide = (unsigned)sm_count * 16;      // block-per-job kernels: grid-stride over the jobs
  for (long long k0 = 0; k0 < a.K; k0 += chunk_rows) {
    const int n = (int)std::min(chunk_rows, a.K - k0);
    uf_rows_kernel<<<(n + 127) / 128, 128, 0, st>>>(dp, a.params, a.gal_index, k0, n, rows);
    uf_cube_kernel<<<grid_for((long long)n * g.plane, T, sm_count), T, 0, st>>>(dp, rows, n, A);
    {
      const long long jobs = (long long)n * (((long long)g.plane + kLsfPix - 1) / kLsfPix);
      const size_t smem = sizeof(float) * kLsfPix * (kLsfPiece + 2 * dp.r_v);
      const unsigned rgrid = grid_for((long long)n * g.plane, 256, sm_count);
#define GBK_LSF_CASE(RR) case RR: uf_lsf_reg_kernel<RR><<<rgrid, 256, 0, st>>>(dp, lsf_taps, n, A, B); break;
      switch (dp.r_v) {
        GBK_LSF_CASE(0) GBK_LSF_CASE(1) GBK_LSF_CASE(2) GBK_LSF_CASE(3) GBK_LSF_CASE(4) GBK_LSF_CASE(5) GBK_LSF_CASE(6)
        default:
          uf_lsf_kernel<<<(unsigned)std::min<long long>(jobs, wide), 256, smem, st>>>(dp, lsf_taps, n, A, B);
      }
#undef GBK_LSF_CASE
      static_assert(kLsfRegMaxR == 6, "the switch above lists the register-ring instantiations");
    }
    // PSF: B (extended layout) -> A (compact fine-grid layout)
    if (dp.psf_kind == GBK_PSF_GAUSSIAN) {
#define GBK_UF_CASE(RR) case RR: launch_psf_sep<RR>(dp, rows, n, wide, B, A, st); break;
      switch (dp.r_p_max) {
        GBK_UF_CASE(0) GBK_UF_CASE(1) GBK_UF_CASE(2) GBK_UF_CASE(3) GBK_UF_CASE(4) GBK_UF_CASE(5)
        GBK_UF_CASE(6) GBK_UF_CASE(7) GBK_UF_CASE(8) GBK_UF_CASE(9) GBK_UF_CASE(10) GBK_UF_CASE(11)
        GBK_UF_CASE(12) GBK_UF_CASE(13) GBK_UF_CASE(14) GBK_UF_CASE(15) GBK_UF_CASE(16)
        default: return cudaErrorInvalidValue;
      }
#undef GBK_UF_CASE
    } else {
      const long long jobs = (long long)n * dp.nv * ((dp.fw + kImgTile - 1) / kImgTile) *
                             ((dp.fh + kImgTile - 1) / kImgTile);
      const int iw = kImgTile + 2 * g.R, nn = 2 * g.R + 1;
      const size_t smem = sizeof(float) * ((size_t)iw * iw + (size_t)nn * nn);
      uf_psf2d_kernel<<<(unsigned)std::min<long long>(jobs, wide), 256, smem, st>>>(dp, rows, n, B, A);
    }
    if (extraction == GBK_EXTRACT_GAUSSFIT)
      uf_gaussfit_kernel<<<grid_for((long long)n * npix, 128, sm_count), 128, 0, st>>>(dp, rows, k0, n, A, contrib, a);
    else
      uf_moments_kernel<<<grid_for((long long)n * npix, 128, sm_count), 128, 0, st>>>(dp, rows, k0, n, A, contrib, a);
    uf_chi2_kernel<<<n, 256, 0, st>>>(contrib, npix, k0, a.chi2);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace gbk
