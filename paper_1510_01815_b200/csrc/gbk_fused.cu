// Fused hot path of libgbk for sm_100a: one thread block = (parameter row k, spatial tile); one launch per batch.
//
// What one block does (steps a1..a9 of SURVEY.md section 8(a); PAPER.md = arXiv:1510.01815):
//   a1  row constants from the parameters (eq. 1-8)
//   a2  per fine spatial sample of the tile + PSF halo: deprojection (eq. 1-4),
//       brightness (eq. 5, :110, or a tabulated profile, :106), rotation curve (eq. 6, :120, the ramp,
//       or eq. 7, :124-129), line-of-sight velocity (eq. 8, :143)
//   a3  Gaussian line over the extended channels: summed per block of 8 channels as a
//       polynomial in the line ratio (two MUFU.EX2 per pixel and block), or voxel by voxel for narrow lines
//   a4  LSF along v: folded into per-channel weights (see below)
//   a5  PSF in (x, y) from shared memory: separable Gaussian passes or a general 2-D image
//   a6  down-sampling by u
//   a7  moments       a8  residual, mask, chi^2 (eq. 11, :246)
//   a9  chi^2 (and optional maps / residuals) to global memory
//
// The cube never exists, not even in shared memory.  The un-normalised moments
//   S_q(x, y) = sum_k (v_k - v_ref)^q C_k(x, y),  q = 0, 1, 2
// are linear in the cube, and LSF, PSF and down-sampling are linear and act on different axes,
// so  S_q = downsample( PSF (*) sum_c w_q[c] line(x, y, c) )  with the weights
//   w_q[c] = sum_{k in band} L[k - c] (v_k - v_ref)^q
// (LSF taps L and band edges folded in exactly; built in FP64 in gbk_api.cu about v_center and shifted
// to the row's reference velocity v_ref in the prologue).  Only three 2-D maps per tile are convolved.
// m1 = v_ref + S1/S0, m2 = sqrt(S2/S0 - (S1/S0)^2).
//
// Instruction economy: the kernel is bound by the FP32 FMA pipe, so the FP32
// arithmetic is written for Blackwell's packed FFMA2/FMUL2 (two FP32 lanes per issued instruction, which
// saves issue slots, not pipe time): pixels are processed in horizontally adjacent pairs in the voxel
// loop, and the PSF passes combine pixel pairs with broadcast taps or tap pairs with broadcast inputs.
#include <math.h>

#include "gbk_device.cuh"
#include "gbk_internal.h"

namespace gbk {

namespace {

constexpr int kMaxThreads = 256;
constexpr int kMinBlocks = 3;
constexpr int kVBlockX = 4;      // output rows per thread in the x-packed vertical pass (divides kVBlock)
constexpr int kPairs = 2;        // pixel pairs per lane in the voxel loop (4 pixels per thread)
constexpr int kStripPairs = 8;    // width of a strip of the voxel loop in pixel pairs (a power of two; 4 and 16
                                  // measure the same on config 3)
constexpr int kSqueezed = 2;               // RowConst::precise of such rows
constexpr float kSqueezedMargin = 3.5f;   // like kPreciseMargin: rows that also keep per-pixel central moments
constexpr float kTruncD = 6.5f;   // lines centred in the band are summed out to |d| < this (6.0: -1.4 %, 5.5:
                                  // -2.2 % of config 3's time; 6.5 keeps the left-out tail below 2^-42)

// floats of the PSF tap area: image taps of the register-tiled pass are stored as (w, w) pairs
__host__ __device__ __forceinline__ int taps_floats(const DevProblem& dp) {
  const int n = 2 * dp.r_p_max + 1;
  return dp.img_fast ? round_up4(2 * n * (n + 1)) : round_up4(dp.psf_stride) + 2 * (n + 1);   // + (w[i], w[i-1]) pairs
}

// Velocity (from v_center) of the centre of channel block b of the extended band (precise rows).
__device__ __forceinline__ float block_centre_velocity(const DevProblem& dp, int b) {
  return dp.vrel_first + ((float)(b * kChanBlock) + 0.5f * (float)(kChanBlock - 1)) * dp.dv;
}

struct Smem {
  float* maps;      // 3 x ehs x ews
  float* spare;     // tile_h x ews (register-tiled image-PSF pass only)
  float4* chan;     // nvx_pad
  float* coef;      // nvx_pad / 8 blocks x 3 moments x 8 coefficients of the block polynomial
  float* coefb;     // the same for the polynomial anchored at the block's last channel
  RowConstD* rcd;   // FP64 row constants (precise rows only)
  float* taps;      // round_up4(psf_stride)
  RowConst* rc;
  float* red;       // 32
};

__device__ __forceinline__ Smem carve(const DevProblem& dp, unsigned char* raw) {
  Smem s;
  s.maps = reinterpret_cast<float*>(raw);
  s.spare = s.maps + 3 * dp.ehs * dp.ews;
  s.chan = reinterpret_cast<float4*>(s.spare + dp.spare_plane);
  s.coef = reinterpret_cast<float*>(s.chan + dp.nvx_pad);
  s.coefb = s.coef + 3 * dp.nvx_pad;
  s.rcd = reinterpret_cast<RowConstD*>(s.coefb + 3 * dp.nvx_pad);
  s.taps = reinterpret_cast<float*>(s.rcd + 1);
  s.rc = reinterpret_cast<RowConst*>(s.taps + taps_floats(dp));
  s.red = reinterpret_cast<float*>(s.rc + 1);
  return s;
}

// ---------------------------------------------------------------------------------- a1 ------
__device__ void row_constants(const DevProblem& dp, const EvalArgs& a, long long k, RowConst* rc,
                              RowConstD* rd) {
  const float* p = a.params + k * dp.row_stride;
  float v[GBK_P_MAX];
  bool finite = true;
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j) {
    v[j] = j < dp.row_stride ? p[j] : 1.0f;
    finite = finite && isfinite(v[j]);
  }
  float sp, cp, si, ci;
  sincospif(v[2] * (1.0f / 180.0f), &sp, &cp);
  sincospif(v[3] * (1.0f / 180.0f), &si, &ci);
  const float sigma0 = v[7], r0 = v[8], rt = v[6], i0 = v[9];
  const bool ok = finite && sigma0 > 0.f && r0 > 0.f && rt > 0.f && i0 > 0.f && !(fabsf(ci) < 1e-6f) &&
                  (dp.rc_model != GBK_RC_EPINAT || (v[10] > 0.f && v[11] > 0.f));
  rc->ea = v[10], rc->eg = v[11];
  int gal = a.gal_index ? a.gal_index[k] : 0;
  const bool gal_ok = gal >= 0 && gal < dp.n_gal;
  if (!gal_ok) gal = 0;
  rc->gal = gal;
  rc->psf_set = dp.psf_per_gal ? gal : 0;
  rc->r_p = dp.psf_r[rc->psf_set];
  rc->valid = (ok && gal_ok) ? 1 : 0;
  const float inv_ci = 1.0f / ci;
  const float s = 1.0f / (sigma0 * 1.1774100225154747f);  // sqrt(2 ln 2): 2^-(s dv)^2 = exp(-dv^2/2sigma0^2)
  const float vrot_scale = (dp.rc_model == GBK_RC_ARCTAN ? 0.63661977236758134f : 1.0f) * v[5] * si;
  rc->xo = v[0];
  rc->yo = v[1];
  rc->sp = sp;
  rc->cp = cp;
  rc->nsp = -sp;
  rc->ncp_ci = -cp * inv_ci;
  rc->nsp_ci = -sp * inv_ci;
  rc->inv_rt = 1.0f / rt;
  rc->rt = rt;
  rc->nl2e_inv_r0 = -1.4426950408889634f / r0;
  rc->tab_scale = dp.tab_inv_dx / r0;
  rc->step = s * dp.dv;
  rc->m2step = -2.0f * rc->step;
  rc->mstep2 = -rc->step * rc->step;
  rc->use_poly = rc->step <= kPolyMaxStep ? 1 : 0;
  rc->inv_bstep = 1.0f / ((float)kChanBlock * rc->step);
  rc->k1 = -s * vrot_scale;                                  // d0 = k1 * f(r) * cos(theta) + k0
  rc->k0 = s * dp.vrel_first - s * (v[4] - dp.v_center);
  rc->v_ref = fminf(fmaxf(v[4] - dp.v_center, -dp.vhalf), dp.vhalf);
  rc->anchor_margin = fminf(10.5f, 7.3f / rc->step);
  rc->cen_lo = (float)dp.r_v * rc->step;                      // line centres inside the band proper:
  rc->cen_hi = (float)(dp.r_v + dp.nv - 1) * rc->step;        // -d0 in [cen_lo, cen_hi]
  const float line_amp = dp.dv / (sigma0 * 2.5066282746310002f) * dp.inv_u2;  // sqrt(2 pi)
  rc->amp = i0 * line_amp;
  rc->dark_s0 = 1e-30f / line_amp;
  // Precise rows: d0 ranges over k0 -+ |k1| sup f; the line of a sample is centred
  // at offset -d0 from extended channel 0, the extended band ends at (nvx - 1) step.  A line centred
  // further than kPreciseMargin outside the band shows only its far wing, where the voxel values need
  // d to ~1e-6: those rows take the FP64 geometry.  (A non-finite test value is a row that is out of
  // domain anyway.)
  const float fsup = curve_sup(dp, v, inv_ci);
  rc->precise = line_leaves_band(dp, rc->k0, rc->k1, fsup, rc->step, kPreciseMargin) ? 1 : 0;
  // ... and further out than kSqueezedMargin a spaxel may see its line squeezed into the band's edge channel:
  // those rows also keep per-pixel central moments (precise_finish)
  if (rc->precise && line_leaves_band(dp, rc->k0, rc->k1, fsup, rc->step, kSqueezedMargin)) rc->precise = kSqueezed;
  rc->step_lo = 0.0f;
  if (rc->precise && rc->valid) {
    double dsp, dcp, dsi, dci;
    sincospi((double)v[2] * (1.0 / 180.0), &dsp, &dcp);
    sincospi((double)v[3] * (1.0 / 180.0), &dsi, &dci);
    const double sd = 1.0 / ((double)sigma0 * 1.1774100225154747);
    const double stepd = sd * (double)dp.dv;
    rc->step_lo = (float)(stepd - (double)rc->step);
    rd->xo = v[0], rd->yo = v[1];
    rd->nsp = -dsp, rd->cp = dcp;
    rd->ncp_ci = -dcp / dci, rd->nsp_ci = -dsp / dci;
    rd->inv_rt = 1.0 / (double)rt, rd->rt = rt;
    rd->k1 = -sd * (dp.rc_model == GBK_RC_ARCTAN ? 0.63661977236758134 : 1.0) * (double)v[5] * dsi;
    rd->ea = v[10], rd->eg = v[11];
    rd->tab_scale = (double)dp.tab_inv_dx / (double)r0;
    const double vrel_first = (-(double)dp.r_v - 0.5 * (double)(dp.nv - 1)) * (double)dp.dv;
    rd->k0 = sd * (vrel_first - ((double)v[4] - (double)dp.v_center));
  }
}

// ---------------------------------------------------------------------------- a7, a8, a9 ----
// One spaxel: moments from the block sums, residuals, chi^2 contribution, optional outputs.
// The packed observation has 1/E = 0 where masked and {0, 0} for a missing dispersion map, so
// neither needs a branch.  OUT = false is the chi^2-only instantiation (no output predicates).
// The tail of one spaxel from its moments: m1r = velocity about the row's v_ref, var = central variance
// (NaN m1r marks a model-dark spaxel).
template <bool OUT>
__device__ __forceinline__ float spaxel_finish_moments(const DevProblem& dp, const EvalArgs& a,
                                                       const RowConst& rc, long long k, int pix, const float4 ob,
                                                       float S0, float m1r, float var, bool dark) {
  float m2 = sqrt_approx(fmaxf(var, 0.0f));                     // fmaxf drops a NaN var: m1r carries it
  const bool unmasked = ob.y > 0.0f;
  float t = (m1r + (rc.v_ref - ob.x)) * ob.y;
  float s = (m2 - ob.z) * ob.w;
  float contrib = fmaf(t, t, s * s);
  const bool bad = !(contrib < f_inf());                        // NaN or Inf moments
  contrib = fminf(contrib, f_inf());                            // ... count +INF (fminf drops the NaN): no branch
  contrib = unmasked ? contrib : 0.0f;
  if (OUT) {
    if (dark) m1r = m2 = f_nan();
    if (!unmasked) t = s = 0.0f;
    else if (bad) t = s = f_nan();
    const size_t npix = (size_t)dp.nx * dp.ny;
    const size_t o = (size_t)k * npix + pix;
    if (a.m0) a.m0[o] = rc.amp * S0;
    if (a.m1) a.m1[o] = m1r + (rc.v_ref + dp.v_center);
    if (a.m2) a.m2[o] = m2;
    if (a.resid) {
      a.resid[2 * (size_t)k * npix + pix] = t;
      a.resid[(2 * (size_t)k + 1) * npix + pix] = s;
    }
  }
  return contrib;
}

template <bool OUT>
__device__ __forceinline__ float spaxel_finish(const DevProblem& dp, const EvalArgs& a,
                                               const RowConst& rc, long long k, int pix,
                                               const float4 ob, float S0, float S1, float S2) {
  // A model-dark spaxel (S0 below the threshold, or not a number) poisons the moments with NaN,
  // so the one test "contrib < inf" in the tail catches dark, NaN and overflowing spaxels alike.
  const bool dark = !(S0 >= rc.dark_s0);
  const float inv = dark ? f_nan() : rcp_approx(S0);
  const float m1r = S1 * inv;
  return spaxel_finish_moments<OUT>(dp, a, rc, k, pix, ob, S0, m1r, fmaf(-m1r, m1r, S2 * inv), dark);
}

__device__ __forceinline__ float4 load_obs(const DevProblem& dp, const RowConst& rc, int pix) {
  return __ldg(&dp.obs[(size_t)rc.gal * ((size_t)dp.nx * dp.ny) + pix]);
}

// ---------------------------------------------------------------------------------- a5 ------
// Separable Gaussian PSF.  Taps are symmetric, so out[x] = sum_{j=0..2R} t[j] in[x + j].
// An output PAIR (out[x], out[x+1]) receives from input in[x + i], i = 0..2R+1, the tap pair
// tp[i] = (t[i], t[i-1]) (t[-1] = t[2R+1] = 0): one FFMA2 with a broadcast input per pair and
// input, i.e. (R + 1) instructions per output instead of (2R + 1).
template <int R>
__device__ __forceinline__ void load_tap_pairs(const float* taps, u64 (&tp)[2 * R + 2]) {
#pragma unroll
  for (int i = 0; i < 2 * R + 2; ++i)
    tp[i] = pk(i <= 2 * R ? taps[i] : 0.0f, i >= 1 ? taps[i - 1] : 0.0f);
}

// Horizontal pass, in place: a row is owned by one group of lanes of one warp, which loads
// everything it needs before it stores.  A lane produces 4 consecutive outputs.
template <int R>
__device__ __forceinline__ void hpass(float* maps, int map_stride, int ews, int EH, int tw,
                                      const u64 (&tp)[2 * R + 2], int tid, int nthreads) {
  constexpr int NV4 = (4 + 2 * R + 3) / 4;
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
    const int q = job >= 2 * npass ? 2 : (job >= npass ? 1 : 0);
    const int row = (job - q * npass) * rpp + rsub;
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
        u64 o0 = pk(0.f, 0.f), o1 = o0;
#pragma unroll
        for (int i = 0; i < 2 * R + 2; ++i) {
          o0 = fma2(pk1(v[i]), tp[i], o0);
          o1 = fma2(pk1(v[i + 2]), tp[i], o1);
        }
        float4 f;
        upk(o0, f.x, f.y);
        upk(o1, f.z, f.w);
        *reinterpret_cast<float4*>(rowp + x0) = f;
      }
      __syncwarp();
    }
  }
}

// Vertical pass of kVBlock output rows of one column of one map into registers.
template <int R>
__device__ __forceinline__ void vcolumn(const float* col, int ews, const u64 (&tp)[2 * R + 2],
                                        float (&res)[kVBlock]) {
  constexpr int BY = kVBlock;
  u64 acc[BY / 2];
#pragma unroll
  for (int m = 0; m < BY / 2; ++m) acc[m] = pk(0.f, 0.f);
#pragma unroll
  for (int i = 0; i < BY + 2 * R; ++i) {
    const u64 v = pk1(col[i * ews]);
#pragma unroll
    for (int m = 0; m < BY / 2; ++m) {
      const int ti = i - 2 * m;
      if (ti >= 0 && ti < 2 * R + 2) acc[m] = fma2(v, tp[ti], acc[m]);
    }
  }
#pragma unroll
  for (int m = 0; m < BY / 2; ++m) upk(acc[m], res[2 * m], res[2 * m + 1]);
}

// Vertical pass in place (u > 1): a thread owns one column of one map and walks it top to bottom
// in chunks, so the rows it overwrites are never read again.
template <int R>
__device__ __forceinline__ void vpass_inplace(float* maps, int map_stride, int ews, int tw, int th,
                                              const u64 (&tp)[2 * R + 2], int tid, int nthreads) {
  constexpr int BY = kVBlock;
  for (int item = tid; item < 3 * tw; item += nthreads) {
    const int q = item >= 2 * tw ? 2 : (item >= tw ? 1 : 0), x = item - q * tw;
    float* col = maps + q * map_stride + x;
    for (int y0 = 0; y0 < th; y0 += BY) {
      float res[BY];
      vcolumn<R>(col + y0 * ews, ews, tp, res);
#pragma unroll
      for (int o = 0; o < BY; ++o)
        if (y0 + o < th) col[(y0 + o) * ews] = res[o];
    }
  }
}

// ---- the passes of the fast path (u == 1) ------------------------------------------------
// The vertical pass keeps two horizontally adjacent pixels in one 64-bit register pair and multiplies by a
// broadcast tap pair (t, t), so every FFMA2 does two useful FMAs on aligned pairs; symmetric taps: only
// R + 1 tap pairs live in registers.  The horizontal pass broadcasts the INPUT instead (hpass_b).
template <int R>
__device__ __forceinline__ void load_tap_bcast(const float* taps, u64 (&tb)[R + 1]) {
#pragma unroll
  for (int i = 0; i <= R; ++i) tb[i] = pk1(taps[i]);
}
template <int R>
__device__ __forceinline__ u64 tap_sym(const u64 (&tb)[R + 1], int j) {   // j in [0, 2R]
  return tb[j <= R ? j : 2 * R - j];
}

// Horizontal pass, in place, with BROADCAST inputs.  A row of one map is owned by a group of lanes of one warp
// (each lane 4 consecutive outputs), which loads everything it needs before it stores.  An output pair
// (x, x + 1) receives from input v[i] the tap pair (w[i], w[i - 1]) (w[-1] = w[2R + 1] = 0) -- 2R + 2 FFMA2 per
// pair instead of 2R + 1, but FFMA2 takes the scalar v[i] as it is, where multiplying aligned pixel pairs by a
// broadcast tap has to build every odd-offset input pair with two MOVs (the earlier form of this pass: 78 FFMA2
// + 56 MOV per 12 outputs).  The tap pairs are read from shared memory (`tp`, one 8-byte broadcast read each).
template <int R>
__device__ __forceinline__ void hpass_b(float* maps, int map_stride, int ews, int EH, int tw, const u64* tp,
                                        int tid, int nthreads) {
  constexpr int NV4 = (4 + 2 * R + 3) / 4;
  const int lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
  const int nx4 = (tw + 3) >> 2;
  int lpr_log = 0;
  while ((1 << lpr_log) < nx4 && lpr_log < 5) ++lpr_log;
  const int lpr = 1 << lpr_log;                 // lanes per row
  const int rpp = 32 >> lpr_log;                // rows per pass
  const int l = lane & (lpr - 1), rsub = lane >> lpr_log;
  const int nchunks = (nx4 + lpr - 1) >> lpr_log;
  const int npass = (EH + rpp - 1) / rpp;
  for (int job = warp; job < npass; job += nwarps) {
    const int row = job * rpp + rsub;
    for (int chunk = 0; chunk < nchunks; ++chunk) {
      const int x0 = ((chunk << lpr_log) + l) << 2;
      const bool active = row < EH && x0 < tw;
      float* rowp = maps + row * ews + x0;
      float4 res[3];
      if (active) {
#pragma unroll
        for (int q = 0; q < 3; ++q) {
          float v[NV4 * 4];
#pragma unroll
          for (int i = 0; i < NV4; ++i) {
            const float4 f = *reinterpret_cast<const float4*>(rowp + q * map_stride + 4 * i);
            v[4 * i] = f.x, v[4 * i + 1] = f.y, v[4 * i + 2] = f.z, v[4 * i + 3] = f.w;
          }
          u64 o0 = pk(0.f, 0.f), o1 = o0;
#pragma unroll
          for (int i = 0; i < 2 * R + 2; ++i) {
            const u64 t = tp[i];
            o0 = fma2(t, pk1(v[i]), o0);
            if (i + 2 < NV4 * 4) o1 = fma2(t, pk1(v[i + 2]), o1);
          }
          upk(o0, res[q].x, res[q].y);
          upk(o1, res[q].z, res[q].w);
        }
      }
      __syncwarp();
      if (active) {
#pragma unroll
        for (int q = 0; q < 3; ++q) *reinterpret_cast<float4*>(rowp + q * map_stride) = res[q];
      }
      __syncwarp();
    }
  }
}

// Vertical pass fused with moments and chi^2 (u == 1): a thread owns BY consecutive rows of a
// column PAIR; lanes run along x, so the 8-byte shared-memory reads are conflict-free and the
// global accesses coalesced.  Rows past the tile are read from the (allocated, never written)
// padding of the plane and only feed outputs that are discarded; likewise the second column of the
// last pair when the tile width is odd.
template <int R, int BY, bool OUT>
__device__ __forceinline__ float vpass_x_moments(const DevProblem& dp, const EvalArgs& a,
                                                 const RowConst& rc, long long k, const float* maps,
                                                 int map_stride, int ews, int tw, int th, int tx0,
                                                 int ty0, const u64 (&tb)[R + 1], int tid,
                                                 int nthreads) {
  const int nxp = (tw + 1) >> 1, nyb = (th + BY - 1) / BY;
  const unsigned magic = div_magic(nxp);
  float chi = 0.0f;
  for (int item = tid; item < nxp * nyb; item += nthreads) {
    const int yb = div_fast(item, magic), x = (item - yb * nxp) << 1, y0 = yb * BY;
    u64 res[3][BY];
#pragma unroll
    for (int q = 0; q < 3; ++q) {
      const float* col = maps + q * map_stride + y0 * ews + x;
#pragma unroll
      for (int m = 0; m < BY; ++m) res[q][m] = pk(0.f, 0.f);
#pragma unroll
      for (int i = 0; i < BY + 2 * R; ++i) {
        GBK_CHECK(col + 1 < maps + (q + 1) * map_stride && col >= maps + q * map_stride);
        const u64 v = *reinterpret_cast<const u64*>(col);
        col += ews;
#pragma unroll
        for (int m = 0; m < BY; ++m) {
          const int ti = i - m;
          if (ti >= 0 && ti <= 2 * R) res[q][m] = fma2(tap_sym<R>(tb, ti), v, res[q][m]);
        }
      }
    }
    const int pix0 = (ty0 + y0) * dp.nx + tx0 + x;
    const bool second = x + 1 < tw;
    float acc = 0.0f;     // per item, so the sum stays in a register (chi itself is long-lived and spills)
#pragma unroll
    for (int m = 0; m < BY; ++m)
      if (y0 + m < th) {
        const int pix = pix0 + m * dp.nx;
        float s0a, s0b, s1a, s1b, s2a, s2b;
        upk(res[0][m], s0a, s0b);
        upk(res[1][m], s1a, s1b);
        upk(res[2][m], s2a, s2b);
        acc += spaxel_finish<OUT>(dp, a, rc, k, pix, load_obs(dp, rc, pix), s0a, s1a, s2a);
        if (second)
          acc += spaxel_finish<OUT>(dp, a, rc, k, pix + 1, load_obs(dp, rc, pix + 1), s0b, s1b, s2b);
      }
    chi += acc;
  }
  return chi;
}

// a6 + a7/a8 for u > 1 after both in-place passes: block sums over u x u fine pixels.
template <bool OUT>
__device__ __forceinline__ float moments_blocks(const DevProblem& dp, const EvalArgs& a,
                                                const RowConst& rc, long long k, const float* p0,
                                                const float* p1, const float* p2, int ews, int tw,
                                                int th, int tx0, int ty0, int tid, int nthreads) {
  const int u = dp.u, sw = tw / u, sh = th / u;
  const unsigned magic = div_magic(sw);
  float chi = 0.0f;
  for (int item = tid; item < sw * sh; item += nthreads) {
    const int Y = div_fast(item, magic), X = item - Y * sw;
    const int pix = (ty0 / u + Y) * dp.nx + tx0 / u + X;
    const float4 ob = load_obs(dp, rc, pix);
    float s0 = 0.f, s1 = 0.f, s2 = 0.f;
    if (u == 1) {                                  // no down-sampling: one value per map
      const int o = Y * ews + X;
      s0 = p0[o], s1 = p1[o], s2 = p2[o];
    } else {
      for (int dy = 0; dy < u; ++dy)
        for (int dx = 0; dx < u; ++dx) {
          const int o = (Y * u + dy) * ews + X * u + dx;
          s0 += p0[o], s1 += p1[o], s2 += p2[o];
        }
    }
    chi += spaxel_finish<OUT>(dp, a, rc, k, pix, ob, s0, s1, s2);
  }
  return chi;
}

// General 2-D PSF image (any u): direct sum per spaxel from shared memory.  The image is stored
// flipped at create, so this correlation is the true convolution.
template <bool OUT>
__device__ __noinline__ float conv2d_moments(const DevProblem& dp, const EvalArgs& a,
                                             const RowConst& rc, long long k, const float* maps,
                                             int map_stride, int ews, int tw, int th, int tx0,
                                             int ty0, const float* taps, int tid, int nthreads) {
  const int u = dp.u, sw = tw / u, sh = th / u, n = 2 * rc.r_p + 1;
  float chi = 0.0f;
  for (int item = tid; item < sw * sh; item += nthreads) {
    const int Y = item / sw, X = item - Y * sw;
    const int pix = (ty0 / u + Y) * dp.nx + tx0 / u + X;
    const float4 ob = load_obs(dp, rc, pix);
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
    chi += spaxel_finish<OUT>(dp, a, rc, k, pix, ob, s0, s1, s2);
  }
  return chi;
}

// Register-tiled general 2-D PSF (image side N <= kMaxFastPsfN): out[y][x] = sum_ky sum_kx
// W[ky][kx] in[y + ky][x + kx] with W the flipped image (true convolution).  A thread produces an
// 8-pixel chunk of two rows (y and y + th/2): per kernel row it holds the N taps as (w, w) pairs
// (one 8-byte broadcast read each) and applies them to the two input rows (float4 reads; lanes run
// along y and the row stride is 4 mod 8 floats, so they are conflict-free), i.e. 8 N FFMA2 for
// N + 1 + 2 NV4 shared-memory reads.  `out` is a different plane than `in`.  (The two end terms of an
// output pair's N + 1 tap pairs carry half a pair each and share one FFMA2: 8 N - 8 + 8 per kernel row.)
// FIN (u == 1 only): the plane convolved is S2, the last of the three; its outputs stay in registers and each
// pixel is finished on the spot with its S0 and S1 read from `fin.s0`, `fin.s1` (the planes the first two
// passes wrote) -- no store of S2, no barrier and no separate pass over the spaxels.  Returns the thread's chi^2.
struct ConvFinish {
  const float *s0, *s1;     // convolved planes (same row stride)
  long long k;
  int tx0, ty0;
};
template <int N, bool FIN, bool OUT>
__device__ __forceinline__ float conv2d_plane(const DevProblem& dp, const EvalArgs& a, const RowConst& rc,
                                              const ConvFinish& fin, const float* in, float* out, int ews, int tw,
                                              int th, const u64* w64, int tid, int nthreads) {
  float chi = 0.0f;
  constexpr int NV4 = (8 + N - 1 + 3) / 4;
  const int nxc = (tw + 7) >> 3, half = (th + 1) >> 1;
  const unsigned magic = div_magic(half);
  for (int item = tid; item < nxc * half; item += nthreads) {
    const int xc = div_fast(item, magic), l = item - xc * half;
    const bool two = l + half < th;
    const int yy[2] = {l, two ? l + half : l};
    u64 acc[2][4];
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
      for (int p = 0; p < 4; ++p) acc[m][p] = pk(0.f, 0.f);
#pragma unroll 1
    for (int ky = 0; ky < N; ++ky) {
      // an output pair (x + 2p, x + 2p + 1) receives from input v[i] the tap pair (W[i - 2p], W[i - 2p - 1])
      // times the broadcast input: N + 1 FFMA2 per pair and kernel row, and no register shuffling
      u64 w[N + 1];
#pragma unroll
      for (int j = 0; j <= N; ++j) w[j] = w64[ky * (N + 1) + j];
      u64 wend;
      {
        float w0, wz, wl;
        upk(w[0], w0, wz), upk(w[N], wz, wl);
        wend = pk(w0, wl);
      }
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        const float* rowp = in + (yy[m] + ky) * ews + (xc << 3);
        float v[NV4 * 4];
#pragma unroll
        for (int i = 0; i < NV4; ++i) {
          const float4 f = *reinterpret_cast<const float4*>(rowp + 4 * i);
          v[4 * i] = f.x, v[4 * i + 1] = f.y, v[4 * i + 2] = f.z, v[4 * i + 3] = f.w;
        }
#pragma unroll
        for (int i = 0; i < 8 + N - 1; ++i)
#pragma unroll
          for (int p = 0; p < 4; ++p)
            if (i - 2 * p >= 1 && i - 2 * p <= N - 1) acc[m][p] = fma2(w[i - 2 * p], pk1(v[i]), acc[m][p]);
        // the two end terms have half a tap pair each, (W[0], 0) v[2p] and (0, W[N-1]) v[2p+N]: one FFMA2
#pragma unroll
        for (int p = 0; p < 4; ++p) acc[m][p] = fma2(wend, pk(v[2 * p], v[2 * p + N]), acc[m][p]);
      }
    }
#pragma unroll
    for (int m = 0; m < 2; ++m)
      if (m == 0 || two) {
        float4 f0, f1;
        upk(acc[m][0], f0.x, f0.y);
        upk(acc[m][1], f0.z, f0.w);
        upk(acc[m][2], f1.x, f1.y);
        upk(acc[m][3], f1.z, f1.w);
        const int o = yy[m] * ews + (xc << 3);
        if (FIN) {
          const float s2[8] = {f0.x, f0.y, f0.z, f0.w, f1.x, f1.y, f1.z, f1.w};
          const float4 a0 = *reinterpret_cast<const float4*>(fin.s0 + o), a1 = *reinterpret_cast<const float4*>(fin.s0 + o + 4);
          const float4 b0 = *reinterpret_cast<const float4*>(fin.s1 + o), b1 = *reinterpret_cast<const float4*>(fin.s1 + o + 4);
          const float s0[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
          const float s1[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
          const int pix0 = (fin.ty0 + yy[m]) * dp.nx + fin.tx0 + (xc << 3);
          float part = 0.0f;
#pragma unroll
          for (int e = 0; e < 8; ++e)
            if ((xc << 3) + e < tw)
              part += spaxel_finish<OUT>(dp, a, rc, fin.k, pix0 + e, load_obs(dp, rc, pix0 + e), s0[e], s1[e], s2[e]);
          chi += part;
        } else {
          *reinterpret_cast<float4*>(out + o) = f0;
          *reinterpret_cast<float4*>(out + o + 4) = f1;
        }
      }
  }
  return chi;
}

// a5..a9 for an image PSF on the fast path: the three maps are convolved plane by plane, each into
// a plane that is free by then (S0 -> spare, S1 -> plane 0, S2 -> plane 1), then block sums.
template <int N, bool OUT>
__device__ __forceinline__ float image_phase(const DevProblem& dp, const EvalArgs& a, const RowConst& rc,
                                          long long k, float* maps, float* spare, int map_stride, int tw,
                                          int th, int tx0, int ty0, const float* taps, int tid,
                                          int nthreads) {
  const u64* w64 = reinterpret_cast<const u64*>(taps);
  const ConvFinish fin{spare, maps, k, tx0, ty0};
  conv2d_plane<N, false, OUT>(dp, a, rc, fin, maps, spare, dp.ews, tw, th, w64, tid, nthreads);
  __syncthreads();
  conv2d_plane<N, false, OUT>(dp, a, rc, fin, maps + map_stride, maps, dp.ews, tw, th, w64, tid, nthreads);
  __syncthreads();
  if (dp.u == 1)   // no down-sampling: finish every pixel from the registers of the third pass
    return conv2d_plane<N, true, OUT>(dp, a, rc, fin, maps + 2 * map_stride, nullptr, dp.ews, tw, th, w64, tid,
                                      nthreads);
  conv2d_plane<N, false, OUT>(dp, a, rc, fin, maps + 2 * map_stride, maps + map_stride, dp.ews, tw, th, w64, tid,
                              nthreads);
  __syncthreads();
  return moments_blocks<OUT>(dp, a, rc, k, spare, maps, maps + map_stride, dp.ews, tw, th, tx0, ty0, tid,
                             nthreads);
}

template <int R, bool OUT, bool U1>   // U1: no down-sampling (u == 1); otherwise u > 1
__device__ __forceinline__ float separable_phase(const DevProblem& dp, const EvalArgs& a,
                                              const RowConst& rc, long long k, float* maps,
                                              int map_stride, int EH, int tw, int th, int tx0,
                                              int ty0, const float* taps, int tid, int nthreads) {
  if (U1) {
    u64 tb[R + 1];
    load_tap_bcast<R>(taps, tb);
    hpass_b<R>(maps, map_stride, dp.ews, EH, tw, reinterpret_cast<const u64*>(taps + round_up4(dp.psf_stride)), tid,
               nthreads);
    __syncthreads();
    return vpass_x_moments<R, kVBlockX, OUT>(dp, a, rc, k, maps, map_stride, dp.ews, tw, th, tx0, ty0,
                                             tb, tid, nthreads);
  }
  u64 tp[2 * R + 2];
  load_tap_pairs<R>(taps, tp);
  hpass<R>(maps, map_stride, dp.ews, EH, tw, tp, tid, nthreads);
  __syncthreads();
  vpass_inplace<R>(maps, map_stride, dp.ews, tw, th, tp, tid, nthreads);
  __syncthreads();
  return moments_blocks<OUT>(dp, a, rc, k, maps, maps + map_stride, maps + 2 * map_stride, dp.ews, tw, th,
                             tx0, ty0, tid, nthreads);
}

// ------------------------------------------------------------------------ a2, a3, a4 --------
// Geometry of one horizontally adjacent pixel pair (dx = x - x_o of both, dy = y - y_o shared):
// returns the line-centre offsets d0 (in units of 1/s, from extended channel 0) and writes the
// brightness I/I0 of both.
// Tabulated radial profile at table position t = (r / r0) / mesh: linear interpolation between the
// nodes, the last value beyond them.
__device__ __forceinline__ float table_profile(const float* tab, int n, float t) {
  const float tc = fminf(t, (float)(n - 1));
  const int j = min((int)tc, n - 2);
  const float lo = __ldg(tab + j), hi = __ldg(tab + j + 1);
  return fmaf(tc - (float)j, hi - lo, lo);
}

__device__ __forceinline__ u64 table_profile2(const float* tab, int n, u64 t) {
  float ta, tb;
  upk(t, ta, tb);
  return pk(table_profile(tab, n, ta), table_profile(tab, n, tb));
}
__device__ __forceinline__ u64 epinat_factor2(u64 q, float ea, float eg) {
  float qa, qb, na, nb, da, db;
  upk(q, qa, qb);
  const u64 lq = pk(lg2_approx(qa), lg2_approx(qb));                 // q = 0: -inf -> q^g = q^a = 0
  upk(mul2(lq, pk1(eg)), na, nb);
  upk(mul2(lq, pk1(ea)), da, db);
  return mul2(pk(ex2_approx(na), ex2_approx(nb)),
              pk(rcp_approx(1.0f + ex2_approx(da)), rcp_approx(1.0f + ex2_approx(db))));
}

template <bool GENERAL>
__device__ __forceinline__ u64 pair_geometry(const DevProblem& dp, const RowConst& rc, u64 dx,
                                             float dy, u64& brightness) {
  const u64 xe = fma2(pk1(rc.nsp), dx, pk1(dy * rc.cp));            // eq. 1
  const u64 yd = fma2(pk1(rc.ncp_ci), dx, pk1(dy * rc.nsp_ci));     // eq. 2 / cos i
  const u64 r2 = fma2(xe, xe, mul2(yd, yd));                         // eq. 3
  float r2a, r2b;
  upk(r2, r2a, r2b);
  // r = 0: cos(theta) := 0 and V_rot(0) = 0 (A8) -- x_e = r^2 = 0 there, so a finite 1/r gives exactly that
  // without a select
  const u64 rs = pk(rsqrt_approx(fmaxf(r2a, 1e-30f)), rsqrt_approx(fmaxf(r2b, 1e-30f)));
  const u64 r = mul2(r2, rs);
  const u64 cos_t = mul2(xe, rs);                                    // eq. 4
  if (GENERAL && dp.tab_n > 0) {                                     // tabulated T(r / r0)
    brightness = table_profile2(dp.tab, dp.tab_n, mul2(r, pk1(rc.tab_scale)));
  } else {
    float ea, eb;
    upk(mul2(r, pk1(rc.nl2e_inv_r0)), ea, eb);
    brightness = pk(ex2_approx(ea), ex2_approx(eb));                 // eq. 5 / I0
  }
  const u64 q = mul2(r, pk1(rc.inv_rt));
  u64 f;
  if (GENERAL && dp.rc_model == GBK_RC_EPINAT) {                     // eq. 7 without V_t: q^g / (1 + q^a)
    f = epinat_factor2(q, rc.ea, rc.eg);
  } else if (dp.rc_model == GBK_RC_ARCTAN) {                         // eq. 6 without (2/pi) V_t
    float qa, qb, ia, ib;
    upk(q, qa, qb);
    upk(mul2(rs, pk1(rc.rt)), ia, ib);                               // 1/q = r_t / r
    // atan(q) = pi/2 - atan(1/q) for q > 1: the polynomial argument is the smaller of q and 1/q (one min)
    float ata, atb;
    upk(atan01_2(pk(fminf(qa, ia), fminf(qb, ib))), ata, atb);
    f = pk(qa > 1.0f ? 1.5707963267948966f - ata : ata, qb > 1.0f ? 1.5707963267948966f - atb : atb);
  } else {                                                           // ramp: min(r/r_t, 1)
    float qa, qb;
    upk(q, qa, qb);
    f = pk(fminf(qa, 1.0f), fminf(qb, 1.0f));
  }
  return fma2(mul2(f, pk1(rc.k1)), cos_t, pk1(rc.k0));               // eq. 8 -> line centre
}

// The less common models (Epinat curve, tabulated profile) take ONE out-of-line call per pixel pair, so
// that they do not weigh on the register allocation of the headline path (arctan / ramp, exponential disc).
struct PairGeom {
  u64 d0, brightness;
};
__device__ __noinline__ PairGeom pair_geometry_general(const DevProblem& dp, const RowConst* rcp, u64 dx, float dy) {
  const RowConst rc = *rcp;
  PairGeom g;
  g.d0 = pair_geometry<true>(dp, rc, dx, dy, g.brightness);
  return g;
}

// Precise rows (RowConst::precise): eq. 1-4, 6 (or the ramp) and 8 of ONE fine sample in FP64.  Returns
// the line-centre offset d0 as a float pair hi + lo and the brightness I/I0 (FP32 is enough for that).
__device__ __noinline__ void sample_geometry_f64(const DevProblem& dp, const RowConstD* rdp, float nl2e_inv_r0,
                                                 double x, double y, float* hi, float* lo,
                                                 float* bright) {
  const int rc_model = dp.rc_model;
  const RowConstD rd = *rdp;
  const double dx = x - rd.xo, dy = y - rd.yo;
  const double xe = rd.nsp * dx + rd.cp * dy;                       // eq. 1
  const double yd = rd.ncp_ci * dx + rd.nsp_ci * dy;                // eq. 2 / cos i
  const double r2 = xe * xe + yd * yd;                              // eq. 3
  double r = 0.0, cos_t = 0.0;                                      // r = 0: cos(theta) := 0 (A8)
  if (r2 > 0.0) {
    r = sqrt(r2);
    cos_t = xe / r;                                                 // eq. 4
  }
  if (dp.tab_n > 0) {                                               // tabulated T(r / r0)
    const double tc = fmin(r * rd.tab_scale, (double)(dp.tab_n - 1));
    const int j = min((int)tc, dp.tab_n - 2);
    const double t0 = (double)__ldg(dp.tab + j), t1 = (double)__ldg(dp.tab + j + 1);
    *bright = (float)(t0 + (tc - (double)j) * (t1 - t0));
  } else {
    *bright = ex2_approx((float)r * nl2e_inv_r0);                   // eq. 5 / I0
  }
  const double q = r * rd.inv_rt;
  double f;
  if (rc_model == GBK_RC_ARCTAN) f = atan(q);                       // eq. 6 without (2/pi) V_t
  else if (rc_model == GBK_RC_RAMP) f = fmin(q, 1.0);               // ramp (A7)
  else f = q > 0.0 ? pow(q, rd.eg) / (1.0 + pow(q, rd.ea)) : 0.0;   // eq. 7 without V_t
  const double d0 = rd.k1 * f * cos_t + rd.k0;                      // eq. 8 -> line centre
  const float h = (float)d0;
  *hi = h;
  *lo = (float)(d0 - (double)h);
}

// ---- pieces of the voxel loop -------------------------------------------------------------
// With d_c = d0 + c step the line is g_c = 2^-(d_c^2), so g_{c+1} = g_c r_c with
// r_c = 2^-(2 d_c step + step^2) and r_{c+1} = r_c q, q = 2^-(2 step^2) a row constant.
// Block polynomial (exact in exact arithmetic): within a block of kChanBlock = 8 channels starting at
// cb, g_j = g_0 r_0^j q^(j(j-1)/2), so the block's contribution to S_m is
//   g_0 * sum_j C_m[cb + j] r_0^j,   C_m[c] = w_m[c] q^(j(j-1)/2)  (row table, see the prologue):
// two ex2 (anchor, ratio) and three degree-7 Horner chains per pixel and block -- 3.4 FP32 lane-ops
// per voxel instead of 5, and no ex2 per voxel.  The anchor must be the block's LARGEST voxel, or the
// sum of a block on the far wing of a line loses its relative accuracy (and a ratio > 1 to the 7th
// power overflows): blocks the lines of the whole warp item are leaving are anchored at their first
// channel (FWD, ratio r_0 <= 2^14.6), blocks they are approaching at their last one with the mirrored
// table (g_{7-i} = g_7 rho^i q^(i(i-1)/2), rho = 2^(2 d_7 step - step^2)), and the rare block where the
// item's lines do both is summed voxel by voxel.
template <int NP>
struct VoxelAcc {
  u64 d0[NP], d0lo[NP];              // line-centre offset at extended channel 0 (hi, lo)
  u64 s0[NP], s1[NP], s2[NP];    // the three weighted sums
  u64 refp[NP];                          // precise rows: the pixel's own reference velocity of s1, s2
};

// Precise rows: a block's sums P0, P1, P2 are about the block's centre velocity vb (build_row_tables); the
// pixel accumulates them about its own reference ref (its line centre clamped to the band), D = vb - ref:
//   s0 += g P0,   s1 += g (P1 + D P0),   s2 += g (P2 + 2 D P1 + D^2 P0).
// The blocks that matter for a pixel lie around ref, so D is small where g is not: no cancellation.
template <int NP>
__device__ __forceinline__ void accumulate_recentred(VoxelAcc<NP>& v, int j, u64 g, u64 P0, u64 P1, u64 P2, float vb) {
  const u64 D = add2(pk1(vb), mul2(v.refp[j], pk1(-1.0f)));
  v.s0[j] = fma2(g, P0, v.s0[j]);
  v.s1[j] = fma2(g, fma2(D, P0, P1), v.s1[j]);
  v.s2[j] = fma2(g, fma2(D, fma2(D, P0, add2(P1, P1)), P2), v.s2[j]);
}

template <bool PRECISE, bool FWD, int NP>
__device__ __forceinline__ bool poly_block(const DevProblem& dp, const RowConst& rc, const Smem& sm, int b,
                                           VoxelAcc<NP>& v) {
  const float nchan = (float)(b * kChanBlock + (FWD ? 0 : kChanBlock - 1));   // the anchor channel
  const float anchor_hi = nchan * rc.step;
  const u64 slope = pk1(FWD ? rc.m2step : -rc.m2step), ms2 = pk1(rc.mstep2);
  u64 g[NP], r[NP];
#pragma unroll
  for (int j = 0; j < NP; ++j) {
    u64 d;
    if (PRECISE) {   // n * step as a float pair (n * step_hi is not exact in FP32)
      const float anchor_lo = fmaf(nchan, rc.step, -anchor_hi) + nchan * rc.step_lo;
      d = add2(add2(pk1(anchor_hi), v.d0[j]), add2(pk1(anchor_lo), v.d0lo[j]));
    } else {
      d = add2(pk1(anchor_hi), v.d0[j]);
    }
    float ea, eb, ra, rb;
    upk(mul2(d, d), ea, eb);
    upk(fma2(d, slope, ms2), ra, rb);
    g[j] = pk(ex2_approx(-ea), ex2_approx(-eb));
    r[j] = pk(ex2_approx(fminf(ra, 15.0f)), ex2_approx(fminf(rb, 15.0f)));   // <= 2^14.6 unless garbage
  }
  // The anchor is the largest voxel of the block for every pixel here (up to the margin), so a block
  // whose anchors have all flushed to zero contributes exactly 0: skipping is bit-identical.
  u64 any_g = g[0];
#pragma unroll
  for (int j = 1; j < NP; ++j) any_g |= g[j];
  if (!__any_sync(0xffffffffu, any_g != 0ull)) return false;
  // scalar coefficients: FFMA2 takes a broadcast FP32 operand, so no (C, C) pairs are needed
  GBK_CHECK(b >= 0 && (const float*)((FWD ? sm.coef : sm.coefb) + (b + 1) * (3 * kChanBlock)) <=
                          (FWD ? (const float*)sm.coefb : (const float*)sm.rcd));
  const float4* C = reinterpret_cast<const float4*>((FWD ? sm.coef : sm.coefb) + b * (3 * kChanBlock));
  u64 P[3][NP];
#pragma unroll
  for (int m = 0; m < 3; ++m) {
    float c[kChanBlock];
#pragma unroll
    for (int i = 0; i < kChanBlock / 4; ++i) {
      const float4 t = C[m * (kChanBlock / 4) + i];
      c[4 * i] = t.x, c[4 * i + 1] = t.y, c[4 * i + 2] = t.z, c[4 * i + 3] = t.w;
    }
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      u64 Q = pk1(c[kChanBlock - 1]);
#pragma unroll
      for (int i = kChanBlock - 2; i >= 0; --i) Q = fma2(Q, r[j], pk1(c[i]));
      if (PRECISE) {
        P[m][j] = Q;
      } else {
        if (m == 0) v.s0[j] = fma2(g[j], Q, v.s0[j]);
        if (m == 1) v.s1[j] = fma2(g[j], Q, v.s1[j]);
        if (m == 2) v.s2[j] = fma2(g[j], Q, v.s2[j]);
      }
    }
  }
  if (PRECISE) {
    const float vb = block_centre_velocity(dp, b);
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      if ((rc.precise == kSqueezed)) {
        accumulate_recentred(v, j, g[j], P[0][j], P[1][j], P[2][j], vb);
      } else {
        v.s0[j] = fma2(g[j], P[0][j], v.s0[j]);
        v.s1[j] = fma2(g[j], P[1][j], v.s1[j]);
        v.s2[j] = fma2(g[j], P[2][j], v.s2[j]);
      }
    }
  }
  return true;
}

// One channel summed directly: the Gaussian line of PAPER.md:199 by one ex2 per voxel.
template <bool PRECISE, int NP>
__device__ __forceinline__ void direct_channel(const DevProblem& dp, const RowConst& rc, const float4 w, VoxelAcc<NP>& v) {
#pragma unroll
  for (int j = 0; j < NP; ++j) {
    u64 d = fma2(pk1(w.x), pk1(rc.step), v.d0[j]);
    if (PRECISE) d = add2(d, fma2(pk1(w.x), pk1(rc.step_lo), v.d0lo[j]));
    float ea, eb;
    upk(mul2(d, d), ea, eb);
    const u64 g = pk(ex2_approx(-ea), ex2_approx(-eb));
    if (PRECISE && (rc.precise == kSqueezed)) {   // the channel's weights are about the centre of its block
      accumulate_recentred(v, j, g, pk1(w.y), pk1(w.z), pk1(w.w), block_centre_velocity(dp, (int)w.x >> 3));
    } else {
      v.s0[j] = fma2(pk1(w.y), g, v.s0[j]);
      v.s1[j] = fma2(pk1(w.z), g, v.s1[j]);
      v.s2[j] = fma2(pk1(w.w), g, v.s2[j]);
    }
  }
}

// Pair index of a tile -> extended pixel: the pairs are walked strip by strip (kStripPairs pairs wide,
// row-major inside a strip), so that the 64 pairs of a warp item form a compact patch (16 x 8 pixels)
// instead of 1.7 rows of the tile: the line centres of a patch lie close together, so the window of
// channel blocks the item has to look at is hardly wider than that of a single line.
struct StripMap {
  int ppr, EH, full, nfull, wlast;
  unsigned magic_full, magic_last;
};
__device__ __forceinline__ StripMap strip_map(int EW, int EH) {
  StripMap m;
  m.ppr = (EW + 1) >> 1, m.EH = EH;
  m.full = kStripPairs * EH;
  m.nfull = m.ppr / kStripPairs;
  m.wlast = m.ppr - m.nfull * kStripPairs;      // pairs per row of the last, narrower strip (0: none)
  m.magic_full = div_magic(m.full);
  m.magic_last = div_magic(m.wlast > 0 ? m.wlast : 1);
  return m;
}
__device__ __forceinline__ void strip_pixel(const StripMap& m, int pi, int& ey, int& ex) {
  const int s = min(div_fast(pi, m.magic_full), m.nfull);
  const int rem = pi - s * m.full;
  const bool last = s == m.nfull;
  const int y = last ? div_fast(rem, m.magic_last) : rem / kStripPairs;
  const int w = last ? m.wlast : kStripPairs;
  ey = y;
  ex = (s * kStripPairs + rem - y * w) << 1;
}

// The voxel loop: a warp takes items of 32 lanes x kPairs pixel pairs, evaluates the Gaussian line
// of each pixel at every extended channel and accumulates the three LSF-folded weighted sums.
// PRECISE (rows whose lines may be centred outside the band, RowConst::precise): the geometry is
// evaluated in FP64 and the line offset is carried as hi + lo, with the channel offsets c * step
// compensated likewise, so that d at the voxels that matter (|d| < 12) is good to ~5e-7.
template <bool PRECISE, int NP>
__device__ __forceinline__ void voxel_phase(const DevProblem& dp, const RowConst& rc, const Smem& sm,
                                            int tx0, int ty0, int EW, int EH, int R, int tid,
                                            int nthreads, unsigned long long* counters) {
  const StripMap smap = strip_map(EW, EH);
  const bool general = dp.rc_model == GBK_RC_EPINAT || dp.tab_n > 0;
  int n_poly = 0, n_direct = 0, n_items = 0;     // work counters of this warp (gbk_eval_batch_counted)
  const int npairs = smap.ppr * EH;
  const int lane = tid & 31, warp = tid >> 5, nwarps = nthreads >> 5;
  constexpr int kPerItem = 32 * NP;
  const int nitems = (npairs + kPerItem - 1) / kPerItem;
  const int map_stride = dp.ehs * dp.ews;
  const float inv_u = dp.inv_u;
  for (int item = warp; item < nitems; item += nwarps) {
    VoxelAcc<NP> v;
    u64 In[NP];
    int sidx[NP];
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      const int pi = item * kPerItem + j * 32 + lane;
      int ey, ex;
      strip_pixel(smap, min(pi, npairs - 1), ey, ex);
      sidx[j] = pi < npairs ? ey * dp.ews + ex : -1;
      if (PRECISE) {
        const double inv_ud = 1.0 / (double)dp.u;
        const double xa = ((double)(tx0 + ex - R) + 0.5) * inv_ud - 0.5;
        const double y = ((double)(ty0 + ey - R) + 0.5) * inv_ud - 0.5;
        float ha, la, ba, hb, lb, bb;
        sample_geometry_f64(dp, sm.rcd, rc.nl2e_inv_r0, xa, y, &ha, &la, &ba);
        sample_geometry_f64(dp, sm.rcd, rc.nl2e_inv_r0, xa + inv_ud, y, &hb, &lb, &bb);
        v.d0[j] = pk(ha, hb), v.d0lo[j] = pk(la, lb), In[j] = pk(ba, bb);
        // the pixel's reference velocity: its line centre (offset -d0 from extended channel 0, in units of
        // dv / step), clamped to the in-band channels
        const float to_v = dp.dv / rc.step;
        v.refp[j] = pk(fminf(fmaxf(dp.vrel_first - ha * to_v, -dp.vhalf), dp.vhalf),
                       fminf(fmaxf(dp.vrel_first - hb * to_v, -dp.vhalf), dp.vhalf));
      } else {
        const float gx = (float)(tx0 + ex - R), gy = (float)(ty0 + ey - R);
        const float xa = (gx + 0.5f) * inv_u - 0.5f, xb = (gx + 1.5f) * inv_u - 0.5f;
        const float y = (gy + 0.5f) * inv_u - 0.5f;
        if (general) {
          const PairGeom pg = pair_geometry_general(dp, sm.rc, pk(xa - rc.xo, xb - rc.xo), y - rc.yo);
          v.d0[j] = pg.d0, In[j] = pg.brightness;
        } else {
          v.d0[j] = pair_geometry<false>(dp, rc, pk(xa - rc.xo, xb - rc.xo), y - rc.yo, In[j]);
        }
        v.d0lo[j] = 0ull;
      }
      v.s0[j] = v.s1[j] = v.s2[j] = pk(0.f, 0.f);
    }
    // range of the line-centre offsets of the item's 128 pixels (at extended channel 0)
    float dmin = 3.0e38f, dmax = -3.0e38f;
#pragma unroll
    for (int j = 0; j < NP; ++j) {
      float da, db;
      upk(v.d0[j], da, db);
      dmin = fminf(dmin, fminf(da, db));
      dmax = fmaxf(dmax, fmaxf(da, db));
    }
    dmin = ordered_float(__reduce_min_sync(0xffffffffu, ordered_key(dmin)));
    dmax = ordered_float(__reduce_max_sync(0xffffffffu, ordered_key(dmax)));
    // How far from its centre a line is summed.  A voxel with |d| >= 11.4 is flushed to zero by
    // ex2.approx.ftz (2^-(11.4^2) is far below 2^-126), so 11.4 loses nothing.  A line CENTRED IN THE
    // BAND (all 128 of the item) has a voxel of weight >= 1/2 within half a channel of its centre, so
    // what lies beyond |d| = kTruncD = 6.5 (7.7 sigma_0) is below 2^-42 = 2e-13 of its sum -- six
    // orders of magnitude under the FP32 rounding of the sums -- and is left out, like the PSF and LSF
    // taps beyond 4 sigma (A10), only a million times more conservatively.  Lines centred near or
    // beyond a band edge keep the full extent: there the far wing is all a spaxel sees.
    const bool centred = -dmax >= rc.cen_lo && -dmin <= rc.cen_hi;
    const float D = centred ? kTruncD : 11.4f;
    if (rc.use_poly) {
      const int nblk = dp.nvx_pad / kChanBlock;
      const float span = (float)(kChanBlock - 1) * rc.step;
      // blocks with a voxel |d| < D for some pixel of the item (infinite offsets give an empty range)
      const int b_lo = min(max(__float2int_rd((-D - span - dmax) * rc.inv_bstep), 0), nblk);
      const int b_hi = max(min(__float2int_ru((D - dmin) * rc.inv_bstep), nblk) - 1, -1);
      // how far past the anchor a line centre may lie: the anchor 2^-(A^2) must stay a normal number
      // (A <= 10.5) and (2^(2 A step))^7 times a coefficient <= 2^23 must not overflow (A step <= 7.3)
      const float A = rc.anchor_margin;
      // FWD is safe from block b_f on (every line centred at most A past the block's first channel),
      // the mirrored anchor up to block b_b (every line centred at most A before its last channel)
      const int b_f = min(max(__float2int_ru((-A - dmin) * rc.inv_bstep), b_lo), b_hi + 1);
      const int b_b = max(min(__float2int_rd((A - span - dmax) * rc.inv_bstep), b_f - 1), b_lo - 1);
      for (int b = b_lo; b <= b_b; ++b) n_poly += poly_block<PRECISE, false, NP>(dp, rc, sm, b, v) ? NP / 2 : 0;
      for (int b = b_b + 1; b < b_f; ++b) {      // lines of this item on both sides of the block
#pragma unroll
        for (int cc = 0; cc < kChanBlock; ++cc) {
          GBK_CHECK(b >= 0 && b * kChanBlock + cc < dp.nvx_pad);
          direct_channel<PRECISE, NP>(dp, rc, sm.chan[b * kChanBlock + cc], v);
        }
        n_direct += kChanBlock * (NP / 2);
      }
      for (int b = b_f; b <= b_hi; ++b) n_poly += poly_block<PRECISE, true, NP>(dp, rc, sm, b, v) ? NP / 2 : 0;
    } else {
      const float inv_step = rc.inv_bstep * (float)kChanBlock;
      const int c_lo = min(max(__float2int_rd((-D - dmax) * inv_step), 0), dp.nvx);
      const int c_hi = max(min(__float2int_ru((D - dmin) * inv_step), dp.nvx) - 1, -1);
#pragma unroll 4
      for (int c = c_lo; c <= c_hi; ++c) {
        GBK_CHECK(c >= 0 && c < dp.nvx);
        direct_channel<PRECISE, NP>(dp, rc, sm.chan[c], v);
      }
      n_direct += max(c_hi - c_lo + 1, 0) * (NP / 2);
    }
    n_items += NP / 2;     // the counters' unit is 128 samples (gbk.h)
#pragma unroll
    for (int j = 0; j < NP; ++j)
      if (sidx[j] >= 0) {
        float2 o;
        GBK_CHECK(sidx[j] + 1 < map_stride && (sidx[j] & 1) == 0);
        if (PRECISE && (rc.precise == kSqueezed)) {
          // these rows keep, per fine pixel, the flux S0 I, the mean velocity M1 (about the row's v_ref) and the
          // CENTRAL variance V of its line sums -- both formed about the pixel's own reference, where nothing
          // cancels; precise_finish mixes them through the PSF by the parallel-axis rule
          float s0a, s0b, s1a, s1b, s2a, s2b, ra, rb;
          upk(v.s0[j], s0a, s0b), upk(v.s1[j], s1a, s1b), upk(v.s2[j], s2a, s2b), upk(v.refp[j], ra, rb);
          // a line sum below 1e-36 (it would overflow the reciprocal) counts as no flux at all
          const bool ha = s0a > 1e-36f, hb = s0b > 1e-36f;
          const float ia = ha ? 1.0f / s0a : 0.0f, ib = hb ? 1.0f / s0b : 0.0f;
          const float ma = s1a * ia, mb = s1b * ib;
          upk(mul2(v.s0[j], In[j]), o.x, o.y);
          if (!ha) o.x = 0.0f;
          if (!hb) o.y = 0.0f;
          *reinterpret_cast<float2*>(sm.maps + sidx[j]) = o;
          o.x = ha ? (ra - rc.v_ref) + ma : 0.0f, o.y = hb ? (rb - rc.v_ref) + mb : 0.0f;
          *reinterpret_cast<float2*>(sm.maps + map_stride + sidx[j]) = o;
          o.x = fmaxf(fmaf(-ma, ma, s2a * ia), 0.0f), o.y = fmaxf(fmaf(-mb, mb, s2b * ib), 0.0f);
          *reinterpret_cast<float2*>(sm.maps + 2 * map_stride + sidx[j]) = o;
          continue;
        }
        upk(mul2(v.s0[j], In[j]), o.x, o.y);
        *reinterpret_cast<float2*>(sm.maps + sidx[j]) = o;
        upk(mul2(v.s1[j], In[j]), o.x, o.y);
        *reinterpret_cast<float2*>(sm.maps + map_stride + sidx[j]) = o;
        upk(mul2(v.s2[j], In[j]), o.x, o.y);
        *reinterpret_cast<float2*>(sm.maps + 2 * map_stride + sidx[j]) = o;
      }
  }
  if (counters && lane == 0) {
    atomicAdd(&counters[GBK_CNT_ITEMS], (unsigned long long)n_items);
    atomicAdd(&counters[GBK_CNT_POLY_BLOCKS], (unsigned long long)n_poly);
    atomicAdd(&counters[GBK_CNT_DIRECT_CHANNELS], (unsigned long long)n_direct);
    if (PRECISE) atomicAdd(&counters[GBK_CNT_PRECISE_ITEMS], (unsigned long long)n_items);
  }
}

// a5..a9 of a precise row.  The planes hold, per fine pixel i, the flux F_i = S0_i I_i, the mean velocity
// M_i (about the row's v_ref) and the central variance V_i of its line sums.  A spaxel is the PSF-weighted
// (and u x u block-summed) mixture of its pixels, so by the parallel-axis rule
//   S0 = sum_i w_i F_i,   m1 = sum_i w_i F_i M_i / S0,   var = sum_i w_i F_i (V_i + (M_i - m1)^2) / S0
// -- two passes over the footprint, the second about the spaxel's own mean: nothing cancels even when the
// spectrum is squeezed into the band's edge channel a hundred km/s from v_ref (m2 ~ 0.1 km/s), where
// S2/S0 - m1^2 in FP32 is off by more than the tolerance.  Direct 2-D sums, (2R+1)^2 taps per pass: about
// ten times the work of the separable passes, on rows that are rare.
template <bool OUT>
__device__ __noinline__ float precise_finish(const DevProblem& dp, const EvalArgs& a, const RowConst* rcp, long long k,
                                             const float* maps, int map_stride, int tw, int th, int tx0, int ty0,
                                             const float* taps, int tid, int nthreads) {
  const RowConst rc = *rcp;
  const int u = dp.u, sw = tw / u, sh = th / u, n = 2 * rc.r_p + 1, ews = dp.ews;
  const bool image = dp.psf_kind == GBK_PSF_IMAGE;
  float chi = 0.0f;
  for (int item = tid; item < sw * sh; item += nthreads) {
    const int Y = item / sw, X = item - Y * sw;
    const int pix = (ty0 / u + Y) * dp.nx + tx0 / u + X;
    const float4 ob = load_obs(dp, rc, pix);
    float A0 = 0.0f, A1 = 0.0f, A2 = 0.0f, m1 = 0.0f;
    for (int pass = 0; pass < 2; ++pass) {
      for (int dy = 0; dy < u; ++dy)
        for (int dx = 0; dx < u; ++dx) {
          const float* base = maps + (Y * u + dy) * ews + X * u + dx;
          for (int ky = 0; ky < n; ++ky)
            for (int kx = 0; kx < n; ++kx) {
              // Gaussian: outer product of the 1-D taps; image: the flipped image (pairs layout on the fast path)
              const float w = !image ? taps[ky] * taps[kx]
                                     : (dp.img_fast ? taps[2 * (ky * (n + 1) + kx)] : taps[ky * n + kx]);
              const float* q = base + ky * ews + kx;
              const float wf = w * q[0];
              if (pass == 0) {
                A0 += wf;
                A1 = fmaf(wf, q[map_stride], A1);
              } else {
                const float dm = q[map_stride] - m1;
                A2 = fmaf(wf, fmaf(dm, dm, q[2 * map_stride]), A2);
              }
            }
        }
      if (pass == 0) m1 = A1 / A0;
    }
    const bool dark = !(A0 >= rc.dark_s0);
    chi += spaxel_finish_moments<OUT>(dp, a, rc, k, pix, ob, A0, dark ? f_nan() : m1, A2 / A0, dark);
  }
  return chi;
}

// Out of line: precise rows are rare, and the FP64 path must not weigh on the register allocation of
// the common one.
__device__ __noinline__ void voxel_phase_precise(const DevProblem& dp, unsigned char* smem_raw, int tx0,
                                                 int ty0, int EW, int EH, int R, int tid, int nthreads,
                                                 unsigned long long* counters) {
  const Smem sm = carve(dp, smem_raw);
  const RowConst rc = *sm.rc;
  voxel_phase<true, kPairs>(dp, rc, sm, tx0, ty0, EW, EH, R, tid, nthreads, counters);
}

// Channel table, and the coefficients of the block polynomial of this row (voxel loop):
// C_m[c] = w_m[c] q^(j(j-1)/2), j = c mod 8, q = 2^(-2 step^2), stored as scalars (and the mirrored table).
// The row's moment weights are the problem's w_q about v_center shifted in FP64 to a reference velocity vr,
//   w1' = w1 - vr w0,   w2' = w2 - 2 vr w1 + vr^2 w0:
// the row's v_ref (RowConst::v_ref) for ordinary rows; for precise rows (per_block) the velocity of the
// centre of the channel's own block, so that the block sums of the voxel loop involve small velocities only
// and each pixel can re-reference them to a velocity of its own without cancellation (precise_finish).
__device__ __forceinline__ void build_row_tables(const DevProblem& dp, const EvalArgs& a, long long k, const Smem& sm,
                                                 bool per_block, int tid, int nthreads) {
  const float sigma0 = a.params[k * dp.row_stride + 7];
  const float s_ = 1.0f / (sigma0 * 1.1774100225154747f);
  const float step = s_ * dp.dv;
  const bool poly = step <= kPolyMaxStep;        // false for NaN: the row is out of domain anyway
  const double vrow = (double)fminf(fmaxf(a.params[k * dp.row_stride + 4] - dp.v_center, -dp.vhalf), dp.vhalf);
  for (int c = tid; c < dp.nvx_pad; c += nthreads) {
    const double vr = per_block ? (double)block_centre_velocity(dp, c >> 3) : vrow;
    const double w0 = dp.chan_w[3 * c], w1 = dp.chan_w[3 * c + 1], w2 = dp.chan_w[3 * c + 2];
    const float4 w = make_float4((float)c, (float)w0, (float)(w1 - vr * w0),
                                 (float)(w2 - vr * (2.0 * w1 - vr * w0)));
    sm.chan[c] = w;
    if (poly) {
      const int j = c & (kChanBlock - 1);
      const float f = exp2f(-step * step * (float)(j * (j - 1)));
      float* dst = sm.coef + (c >> 3) * (3 * kChanBlock) + j;
      dst[0] = w.y * f;
      dst[kChanBlock] = w.z * f;
      dst[2 * kChanBlock] = w.w * f;
      const int i = kChanBlock - 1 - j;            // the same channel counted from the block's end
      const float fb = exp2f(-step * step * (float)(i * (i - 1)));
      dst = sm.coefb + (c >> 3) * (3 * kChanBlock) + i;
      dst[0] = w.y * fb;
      dst[kChanBlock] = w.z * fb;
      dst[2 * kChanBlock] = w.w * fb;
    }
  }
}

__device__ __noinline__ void build_block_tables(const DevProblem& dp, const EvalArgs& a, long long k,
                                                unsigned char* smem_raw, int tid, int nthreads) {
  build_row_tables(dp, a, k, carve(dp, smem_raw), true, tid, nthreads);
}

// ------------------------------------------------------------------------------ the kernel ---
// PATH: which PSF passes the instantiation holds (path_of picks by problem) -- kPathSepU1 the separable Gaussian
// passes without down-sampling (configs 1, 3, 5), kPathSepUN the separable passes with down-sampling (config 2),
// kPathImage the register-tiled image pass (config 4; images up to kMaxFastPsfN a side, any u), kPathAny the
// general 2-D sum for larger images.  One function with every path inlined spilt ~1750 B inside 80 registers;
// separate instantiations also let each path have the launch bounds that fit it (fused_kernel below).
constexpr int kPathAny = 0, kPathSepU1 = 1, kPathImage = 2, kPathSepUN = 3;
template <bool OUT, bool COUNT, int PATH>
__global__ void __launch_bounds__(kMaxThreads, (PATH == kPathImage || PATH == kPathSepUN) ? 2 : kMinBlocks)
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

  if (tid == 0) row_constants(dp, a, k, sm.rc, sm.rcd);
  build_row_tables(dp, a, k, sm, false, tid, nthreads);
  __syncthreads();
  const RowConst rc = *sm.rc;   // by value: registers, no aliasing with the map stores
  if ((rc.precise == kSqueezed) && rc.valid) {  // moment weights about the centre of every channel block (build_row_tables)
    build_block_tables(dp, a, k, smem_raw, tid, nthreads);
    __syncthreads();
  }
  if (PATH == kPathImage) {   // rows of tap pairs (W[ky][i], W[ky][i-1]), i = 0..N, with W[ky][-1] = W[ky][N] = 0
    const int n = 2 * rc.r_p + 1;
    const float* W = dp.psf_taps + (size_t)rc.psf_set * dp.psf_stride;
    for (int j = tid; j < n * (n + 1); j += nthreads) {
      const int ky = j / (n + 1), i = j - ky * (n + 1);
      reinterpret_cast<u64*>(sm.taps)[j] = pk(i < n ? W[ky * n + i] : 0.0f, i >= 1 ? W[ky * n + i - 1] : 0.0f);
    }
  } else {
    for (int j = tid; j < dp.psf_stride; j += nthreads)
      sm.taps[j] = dp.psf_taps[(size_t)rc.psf_set * dp.psf_stride + j];
    if (PATH == kPathSepU1) {   // tap pairs (w[i], w[i - 1]) of the horizontal pass (hpass_b)
      const float* W = dp.psf_taps + (size_t)rc.psf_set * dp.psf_stride;
      const int n = 2 * rc.r_p + 1;
      u64* tp = reinterpret_cast<u64*>(sm.taps + round_up4(dp.psf_stride));
      for (int i = tid; i <= n; i += nthreads) tp[i] = pk(i < n ? W[i] : 0.0f, i >= 1 ? W[i - 1] : 0.0f);
    }
  }

  float chi = 0.0f;
  if (!rc.valid) {
    // out-of-domain row: chi^2 = +INF, NaN maps and residuals for this tile's spaxels
    if (OUT) {
      const int u = dp.u, sw = tw / u, sh = th / u, npix = dp.nx * dp.ny;
      for (int item = tid; item < sw * sh; item += nthreads) {
        const int Y = item / sw, X = item - Y * sw;
        const size_t pix = (size_t)(ty0 / u + Y) * dp.nx + tx0 / u + X;
        if (a.m0) a.m0[k * npix + pix] = f_nan();
        if (a.m1) a.m1[k * npix + pix] = f_nan();
        if (a.m2) a.m2[k * npix + pix] = f_nan();
        if (a.resid) a.resid[2 * k * npix + pix] = a.resid[(2 * k + 1) * npix + pix] = f_nan();
      }
    }
    chi = f_inf();
  } else {
    const int R = rc.r_p;
    const int EW = tw + 2 * R, EH = th + 2 * R;
    // The PSF passes read whole register blocks, i.e. up to 10 columns and 7 rows past the extended tile
    // inside the plane's allocation (ews x ehs, sized for that in gbk_api.cu).  Nobody writes that padding:
    // what is read there only feeds outputs that are discarded (columns >= tw, rows >= th), and zeroing it
    // would cost 5 % on config 5 and 10 % on config 1 for no change in any result.  -DGBK_DEBUG_BOUNDS
    // checks that every such access stays inside the allocation.
    if (rc.precise)
      voxel_phase_precise(dp, smem_raw, tx0, ty0, EW, EH, R, tid, nthreads, COUNT ? a.counters : nullptr);
    else
      voxel_phase<false, PATH == kPathImage ? 2 * kPairs : kPairs>(dp, rc, sm, tx0, ty0, EW, EH, R, tid, nthreads,
                                                                    COUNT ? a.counters : nullptr);
    __syncthreads();
    // ------------------------------------------------------------------ a5 .. a9 ---------
    if ((rc.precise == kSqueezed)) {
      chi = precise_finish<OUT>(dp, a, sm.rc, k, sm.maps, map_stride, tw, th, tx0, ty0, sm.taps, tid, nthreads);
    } else if (PATH == kPathImage) {
#define GBK_IMG_CASE(NN)                                                                          \
  case NN:                                                                                        \
    chi = image_phase<NN, OUT>(dp, a, rc, k, sm.maps, sm.spare, map_stride, tw, th, tx0, ty0,     \
                               sm.taps, tid, nthreads);                                           \
    break;
      switch (2 * R + 1) {
        GBK_IMG_CASE(1) GBK_IMG_CASE(3) GBK_IMG_CASE(5) GBK_IMG_CASE(7) GBK_IMG_CASE(9)
        GBK_IMG_CASE(11) GBK_IMG_CASE(13) GBK_IMG_CASE(15)
        default: break;
      }
#undef GBK_IMG_CASE
    } else if (PATH == kPathAny) {
      chi = conv2d_moments<OUT>(dp, a, rc, k, sm.maps, map_stride, dp.ews, tw, th, tx0, ty0, sm.taps,
                                tid, nthreads);
    } else if (PATH == kPathSepU1 || PATH == kPathSepUN) {
#define GBK_SEP_CASE(RR)                                                                          \
  case RR:                                                                                        \
    chi = separable_phase<RR, OUT, PATH == kPathSepU1>(dp, a, rc, k, sm.maps, map_stride, EH, tw, th, tx0, ty0, \
                                   sm.taps, tid, nthreads);                                       \
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
  if ((tid & 31) == 0) sm.red[tid >> 5] = chi;
  __syncthreads();
  if (tid == 0) {
    float tot = 0.0f;
    for (int w = 0; w < (nthreads >> 5); ++w) tot += sm.red[w];
    if (!(tot < f_inf())) tot = f_inf();
    if (dp.ntiles == 1) {
      a.chi2[k] = tot;
    } else {
      // the block that finishes a row's last tile adds the row's partials in tile order: one launch,
      // and still the same sum whichever block comes last
      a.partial[bid] = tot;
      __threadfence();
      if (atomicAdd(&a.tile_count[k], 1u) == (unsigned)dp.ntiles - 1u) {
        __threadfence();
        const volatile float* part = a.partial + k * dp.ntiles;
        float sum = 0.0f;
        for (int t = 0; t < dp.ntiles; ++t) sum += part[t];
        if (!(sum < f_inf())) sum = f_inf();
        a.chi2[k] = sum;
        a.tile_count[k] = 0u;     // ready for the next launch
      }
    }
  }
}

}  // namespace

size_t fused_smem_bytes(const DevProblem& dp) {
  return sizeof(float) * (3 * (size_t)dp.ehs * dp.ews + dp.spare_plane) + sizeof(float4) * dp.nvx_pad +
         sizeof(float) * 6 * dp.nvx_pad + sizeof(RowConstD) + sizeof(float) * taps_floats(dp) + sizeof(RowConst) +
         sizeof(float) * 32;
}

namespace {
// the instantiation a problem runs (see kPath* above)
int path_of(const DevProblem& dp) {
  if (dp.psf_kind == GBK_PSF_GAUSSIAN) return dp.u == 1 ? kPathSepU1 : kPathSepUN;
  if (dp.psf_kind == GBK_PSF_IMAGE && dp.img_fast) return kPathImage;
  return kPathAny;
}
typedef void (*FusedFn)(const DevProblem, const EvalArgs);
FusedFn fused_fn(int path, bool out, bool count) {
#define GBK_PATH_FN(PP)                                                  \
  case PP:                                                               \
    return out ? fused_kernel<true, false, PP> : (count ? fused_kernel<false, true, PP> : fused_kernel<false, false, PP>);
  switch (path) {
    GBK_PATH_FN(kPathSepU1) GBK_PATH_FN(kPathImage) GBK_PATH_FN(kPathSepUN)
    default: break;
  }
  return out ? fused_kernel<true, false, kPathAny> : (count ? fused_kernel<false, true, kPathAny> : fused_kernel<false, false, kPathAny>);
#undef GBK_PATH_FN
}
}  // namespace

cudaError_t fused_prepare(const FusedLaunch& fl) {
  for (int path = 0; path < 4; ++path)
    for (int v = 0; v < 3; ++v) {
      const cudaError_t e = cudaFuncSetAttribute(reinterpret_cast<const void*>(fused_fn(path, v == 1, v == 2)),
                                                 cudaFuncAttributeMaxDynamicSharedMemorySize, fl.smem_bytes);
      if (e != cudaSuccess) return e;
    }
  return cudaSuccess;
}

cudaError_t fused_occupancy(const DevProblem& dp, const FusedLaunch& fl, int* n) {
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(n, reinterpret_cast<const void*>(fused_fn(path_of(dp), false, false)),
                                                       fl.threads, fl.smem_bytes);
}

cudaError_t launch_fused(const DevProblem& dp, const EvalArgs& a, const FusedLaunch& fl,
                         cudaStream_t st) {
  const long long nblocks = a.K * dp.ntiles;
  const bool out = a.m0 || a.m1 || a.m2 || a.resid;
  fused_fn(path_of(dp), out, !out && a.counters)<<<(unsigned)nblocks, fl.threads, fl.smem_bytes, st>>>(dp, a);
  return cudaGetLastError();
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
