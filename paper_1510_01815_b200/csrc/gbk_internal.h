// Internal declarations shared by the translation units of libgbk (CUDA side only; the CPU
// oracle under oracle/ shares nothing with this tree).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/gbk.h"

namespace gbk {

constexpr int kMaxSepR = 16;    // largest separable (Gaussian) PSF tap radius, fine pixels
constexpr int kMaxPsfN = 33;    // largest PSF image side
constexpr int kMaxFastPsfN = 15; // largest PSF image side of the register-tiled 2-D pass
constexpr int kMaxLsfR = 64;    // largest LSF tap radius, channels
constexpr int kVBlock = 8;      // output rows per thread in the vertical pass
constexpr int kChanBlock = 8;   // channels summed by one block polynomial of the voxel loop (gbk_fused.cu)
constexpr float kPolyMaxStep = 0.8f;  // the block polynomial is used for step <= this (sigma0/dv >= 1.06)

// Everything the kernels need to know about a problem; passed by value (__grid_constant__).
struct DevProblem {
  int nx, ny, nv, u;        // spaxels, channels, up-sampling
  int n_gal;
  int row_stride;           // floats per parameter row (GBK_P, or GBK_P_EPINAT)
  int tab_n;                // > 0: tabulated radial profile I(r) = I0 T(r/r0) instead of eq. 5
  float tab_inv_dx;         // 1 / mesh of the table (in units of r/r0)
  const float* tab;         // [tab_n]
  int fw, fh;               // fine grid = u*nx, u*ny
  int r_v, nvx;             // LSF radius, nv + 2 r_v extended channels
  int nvx_pad;              // nvx rounded up to kChanBlock; the padding channels have zero weights
  int rc_model, psf_kind, has_disp, psf_per_gal;
  int tile_w, tile_h;       // tile, fine pixels (multiples of u)
  int tiles_x, tiles_y, ntiles;
  int r_p_max;              // largest PSF radius
  int ews, ehs;             // shared-memory row stride (floats) and rows of one moment map
  int psf_stride;           // floats per PSF set in psf_taps
  int img_fast;             // image PSF small enough for the register-tiled 2-D pass (gbk_fused.cu)
  int spare_plane;          // floats of the extra output plane of that pass (0 if unused)
  float dv, v_center;
  float vrel_first;         // velocity of extended channel 0 relative to v_center
  float inv_u, inv_u2;
  float vhalf;              // velocity of the last in-band channel relative to v_center, (nv-1)/2 dv
  const double* chan_w;     // [nvx_pad][3] LSF-folded moment weights w0, w1, w2 about v_center (FP64:
                            // every row shifts them to its own reference velocity, RowConst::v_ref)
  const float* psf_taps;    // [n_psf][psf_stride]: Gaussian 1-D taps, or flipped PSF image
  const int* psf_r;         // [n_psf] tap radius of each PSF set
  const float4* obs;        // [n_gal][ny][nx] {vobs - v_center, 1/E_v (0 = masked), sobs, 1/E_s}
};

struct EvalArgs {
  const float* params;      // [K][row_stride]
  const int32_t* gal_index; // [K] or null
  long long K;
  float* chi2;              // [K]
  float *m0, *m1, *m2;      // [K][ny][nx] or null
  float* resid;             // [K][2][ny][nx] or null
  float* partial;           // [K][ntiles] cross-tile scratch (ntiles > 1)
  unsigned* tile_count;     // [K] tiles of a row finished so far (self-resetting; ntiles > 1)
  unsigned long long* counters;  // [GBK_N_COUNTERS] work counters (gbk_eval_batch_counted) or null
};

// Per-row constants (a1 of SURVEY.md section 8(a)), computed once per block.
struct RowConst {
  float xo, yo, sp, cp;
  float nsp;          // -sin(PA):            x_e = nsp * dx + cp * dy             (eq. 1)
  float ncp_ci;       // -cos(PA) / cos(i):   y_e / cos i = ncp_ci * dx + nsp_ci * dy   (eq. 2-3)
  float nsp_ci;       // -sin(PA) / cos(i)
  float inv_rt, rt;
  float nl2e_inv_r0;  // -log2(e)/r0
  float tab_scale;    // 1 / (r0 * table mesh): position in the intensity table per pixel of radius
  float ea, eg;       // Epinat slopes a, g (eq. 7)
  float step;         // s * dv with s = 1/(sigma0 sqrt(2 ln 2)): exp(-dv^2/(2 sigma0^2)) = 2^-(s dv)^2
  float m2step;       // -2 step
  float mstep2;       // -step^2
  int use_poly;       // step <= kPolyMaxStep: the block polynomial is safe
  float inv_bstep;    // 1 / (kChanBlock * step): blocks per unit of the line-centre offset d
  float k1;           // -s * V_t sin i (* 2/pi for the arctan curve)
  float k0;           // s * (velocity of extended channel 0 - V_sys): the line-centre offset of a
                      // sample from extended channel 0 is  d0 = k1 * f(r/r_t) * cos(theta) + k0
  float v_ref;        // reference velocity of the row's moment sums S1, S2, relative to v_center: V_sys
                      // clamped to the band, so the FP32 cancellation in m2^2 = S2/S0 - m1^2 involves the
                      // distance of the line from V_sys (or from the band edge) and not from v_center
  float anchor_margin;   // how far past a block's anchor a line centre may lie (gbk_fused.cu, voxel loop)
  float cen_lo, cen_hi;  // offsets (from extended channel 0) of the first and last in-band channel
  float amp;          // I0 * dv / (sigma0 sqrt(2 pi) u^2): scales the S0 block sum to m0
  float dark_s0;      // S0 block sums below this are model-dark (m0 < 1e-30 I0)
  int valid;
  int r_p;            // PSF radius of this row's data set
  int psf_set, gal;
  int precise;        // some line of this row may be centred outside the extended band by more than
                      // kPreciseMargin: the voxel loop takes the FP64-geometry path
                      // = 2 (kSqueezed) when a line may be centred more than kSqueezedMargin outside: a spaxel
                      // can then see its line squeezed into the edge channel (m2 << dv), where S2/S0 - m1^2
                      // cancels in FP32 -- such rows keep per-pixel central moments (gbk_fused.cu, precise_finish)
  float step_lo;      // step = step + step_lo to FP64 accuracy (precise rows only)
};

// The row constants of the geometry in FP64, filled for precise rows only (see RowConst::precise):
// the far wing of a line, 2^-(d^2) at |d| ~ 9, turns an error of d into 2 d ln2 = 12 times that
// relative error of the voxel, so d must be known to ~1e-6 there while the line-centre offset itself
// reaches hundreds -- beyond FP32, which carries the product V_t sin i atan(r/r_t) cos(theta) / sigma_0
// to ~3e-7 relative at best.
struct RowConstD {
  double xo, yo;
  double nsp, cp, ncp_ci, nsp_ci;   // as in RowConst
  double inv_rt, rt;
  double k1, k0;                    // d0 = k1 * f(r/r_t) * cos(theta) + k0
  double ea, eg;                    // Epinat slopes
  double tab_scale;                 // 1 / (r0 * table mesh)
};

constexpr float kPreciseMargin = 2.5f;   // in units of the line offset d (1.18 sigma_0 each)

#ifdef __CUDACC__
// sup over the extended field of |f(r / r_t)|, the shape of the rotation curve (v_rot = V_t f, with the 2/pi
// of eq. 6 left out): bounds how far from V_sys a line of the row can be centred.  v = the parameter row.
__device__ inline float curve_sup(const DevProblem& dp, const float* v, float inv_ci) {
  float fsup = dp.rc_model == GBK_RC_ARCTAN ? 1.5707963267948966f : 1.0f;
  if (dp.rc_model == GBK_RC_EPINAT && v[11] > v[10]) {
    // q^g / (1 + q^a) <= max(1, q^(g - a)): bounded by the largest deprojected radius of the extended field
    const float R = (float)dp.r_p_max * dp.inv_u + 1.0f;
    const float ax = fmaxf(fabsf(v[0] + R), fabsf((float)dp.nx + R - v[0]));
    const float ay = fmaxf(fabsf(v[1] + R), fabsf((float)dp.ny + R - v[1]));
    const float qmax = sqrtf(ax * ax + ay * ay) * fabsf(inv_ci) / v[6];
    fsup = fmaxf(1.0f, powf(qmax, v[11] - v[10]));
  }
  return fsup;
}
// With d0 = k1 f cos(theta) + k0 the offset of a line from extended channel 0 in units of `step` per channel:
// can a line of the row be centred more than `margin` outside the extended band?
__device__ inline bool line_leaves_band(const DevProblem& dp, float k0, float k1, float fsup, float step,
                                        float margin) {
  const float tmax = fabsf(k1) * fsup * 1.0001f + 1e-3f;
  const float band = (float)(dp.nvx - 1) * step;
  return k0 + tmax > margin || k0 - tmax < -(band + margin);
}
#endif

struct FusedLaunch {
  int threads;
  int smem_bytes;
};

cudaError_t launch_fused(const DevProblem& dp, const EvalArgs& a, const FusedLaunch& fl,
                         cudaStream_t st);
cudaError_t fused_occupancy(const DevProblem& dp, const FusedLaunch& fl, int* blocks_per_sm);
cudaError_t fused_prepare(const FusedLaunch& fl);  // opt in to large dynamic shared memory
size_t fused_smem_bytes(const DevProblem& dp);

// unfused comparison path (gbk_unfused.cu)
size_t unfused_bytes_per_row(const DevProblem& dp);
double unfused_algorithmic_bytes_per_row(const DevProblem& dp);
cudaError_t launch_unfused(const DevProblem& dp, const EvalArgs& a, const float* lsf_taps, float* scratch,
                           long long chunk_rows, int sm_count, int extraction, cudaStream_t st);

// velocity-field strategy (gbk_vfield.cu): EvalArgs.m1 = velocity maps, EvalArgs.resid = [K][ny][nx]
cudaError_t launch_vfield(const DevProblem& dp, const EvalArgs& a, cudaStream_t st);

// Makes `device` current for the scope and restores the caller's device afterwards.
struct DeviceGuard {
  int prev = -1;
  cudaError_t status = cudaSuccess;
  explicit DeviceGuard(int device) {
    status = cudaGetDevice(&prev);
    if (status == cudaSuccess && prev != device) status = cudaSetDevice(device);
    else if (status == cudaSuccess) prev = -1;   // nothing to restore
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
  DeviceGuard(const DeviceGuard&) = delete;
  DeviceGuard& operator=(const DeviceGuard&) = delete;
};

// error reporting shared by the translation units (message read by gbk_last_error)
int fail(int code, const char* fmt, ...);
void clear_error();

cudaError_t launch_probe_umma(int iters, int blocks, float* out, cudaStream_t st);   // gbk_probe_umma.cu
cudaError_t launch_probe(int which, long long iters, int blocks, int threads, float* sink,
                         cudaStream_t st);

}  // namespace gbk
