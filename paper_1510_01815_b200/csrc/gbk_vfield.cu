// Velocity-field modelling strategy of libgbk (gbk_eval_vfield_batch of include/gbk.h).
//
// PAPER.md:189-195 (section 2.2.1): the radial-velocity model of eq. 8 is evaluated
// at every spaxel, steps 2.2.2-2.2.5 (cube, PSF/LSF, down-sampling, moments) are skipped
// (PAPER.md:195), and the iteration continues with the velocity residual and the
// first term of eq. 11.  The paper assigns one thread per pixel of ONE velocity
// field; here K fields are evaluated per launch: a block takes kRows parameter rows and walks over
// the spaxels once, so the packed observation {v_obs - v_center, 1/E_v, ., .} is read once per
// kRows rows when all rows share a data set.  Per spaxel and row: ~30 FP32 instructions, one
// MUFU.RSQ, no memory traffic besides that 16-byte read; chi^2 by warp shuffles and a fixed-order
// block sum (bit-reproducible).
#include <math.h>

#include "gbk_internal.h"

namespace gbk {

namespace {

constexpr int kRows = 4;        // parameter rows per block
constexpr int kThreads = 256;

struct VRow {
  float xo, yo, cp, nsp, ncp_ci, nsp_ci;   // eq. 1-3 as in RowConst
  float inv_rt, rt;
  float k1;                                 // V_t sin i (x 2/pi for the arctan curve)
  float v0;                                 // V_sys - v_center
  int valid, gal;
};

__device__ __forceinline__ float vf_rsqrt(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// atan(z), z in [0, 1]: z * P(z^2), 8 terms, max error 1.4e-7 rad (the polynomial of the fused
// kernel, scalar here).
__device__ __forceinline__ float vf_atan01(float z) {
  const float t = z * z;
  float p = -0.00405439967289567f;
  p = fmaf(p, t, 0.02186231128871441f);
  p = fmaf(p, t, -0.05591132491827011f);
  p = fmaf(p, t, 0.09642117470502853f);
  p = fmaf(p, t, -0.13908594846725464f);
  p = fmaf(p, t, 0.1994655877351761f);
  p = fmaf(p, t, -0.33329859375953674f);
  p = fmaf(p, t, 0.9999993443489075f);
  return p * z;
}

__device__ void vf_row(const DevProblem& dp, const EvalArgs& a, long long k, VRow* r) {
  const float* p = a.params + k * GBK_P;
  bool finite = true;
  float v[7];
#pragma unroll
  for (int j = 0; j < 7; ++j) {      // only the kinematic parameters enter eq. 8
    v[j] = p[j];
    finite = finite && isfinite(v[j]);
  }
  float sp, cp, si, ci;
  sincospif(v[2] * (1.0f / 180.0f), &sp, &cp);
  sincospif(v[3] * (1.0f / 180.0f), &si, &ci);
  int gal = a.gal_index ? a.gal_index[k] : 0;
  const bool gal_ok = gal >= 0 && gal < dp.n_gal;
  r->gal = gal_ok ? gal : 0;
  r->valid = (finite && gal_ok && v[6] > 0.f && !(fabsf(ci) < 1e-6f)) ? 1 : 0;
  const float inv_ci = 1.0f / ci;
  r->xo = v[0], r->yo = v[1];
  r->cp = cp, r->nsp = -sp, r->ncp_ci = -cp * inv_ci, r->nsp_ci = -sp * inv_ci;
  r->inv_rt = 1.0f / v[6], r->rt = v[6];
  r->k1 = (dp.rc_model == GBK_RC_ARCTAN ? 0.63661977236758134f : 1.0f) * v[5] * si;
  r->v0 = v[4] - dp.v_center;
}

// eq. 1-4, 6 (or the ramp), 8 at the spaxel (x, y): velocity relative to v_center.
__device__ __forceinline__ float vf_velocity(const DevProblem& dp, const VRow& r, float x, float y) {
  const float dx = x - r.xo, dy = y - r.yo;
  const float xe = fmaf(r.nsp, dx, dy * r.cp);              // eq. 1
  const float yd = fmaf(r.ncp_ci, dx, dy * r.nsp_ci);       // eq. 2 / cos i
  const float r2 = fmaf(xe, xe, yd * yd);                   // eq. 3
  const float rs = r2 > 1e-30f ? vf_rsqrt(r2) : 0.0f;       // r = 0: cos(theta) := 0 (A8)
  const float rad = r2 * rs, cos_t = xe * rs;               // eq. 4
  const float q = rad * r.inv_rt;
  float f;
  if (dp.rc_model == GBK_RC_ARCTAN) {                       // eq. 6 without (2/pi) V_t
    const bool big = q > 1.0f;
    const float at = vf_atan01(big ? rs * r.rt : q);
    f = big ? 1.5707963267948966f - at : at;
  } else {
    f = fminf(q, 1.0f);                                     // ramp (A7)
  }
  return fmaf(r.k1 * f, cos_t, r.v0);                       // eq. 8
}

template <bool OUT, bool SHARED_OBS>
__global__ void __launch_bounds__(kThreads) vfield_kernel(const __grid_constant__ DevProblem dp,
                                                          const __grid_constant__ EvalArgs a) {
  __shared__ VRow rows[kRows];
  __shared__ float red[kRows][kThreads / 32];
  const int tid = threadIdx.x;
  const long long k0 = (long long)blockIdx.x * kRows;
  const int nrows = (int)min((long long)kRows, a.K - k0);
  if (tid < nrows) vf_row(dp, a, k0 + tid, &rows[tid]);
  __syncthreads();
  const int npix = dp.nx * dp.ny;
  const float inf = __int_as_float(0x7f800000), nan = __int_as_float(0x7fc00000);
  float chi[kRows];
#pragma unroll
  for (int j = 0; j < kRows; ++j) chi[j] = 0.0f;
  for (int pix = tid; pix < npix; pix += kThreads) {
    const int iy = pix / dp.nx, ix = pix - iy * dp.nx;
    const float x = (float)ix, y = (float)iy;
    float4 ob;
    if (SHARED_OBS) ob = __ldg(&dp.obs[pix]);
#pragma unroll
    for (int j = 0; j < kRows; ++j) {
      if (j >= nrows) break;
      const VRow& r = rows[j];
      if (!SHARED_OBS) ob = __ldg(&dp.obs[(size_t)r.gal * npix + pix]);
      float v = r.valid ? vf_velocity(dp, r, x, y) : nan;
      float t = (v - ob.x) * ob.y;
      const bool unmasked = ob.y > 0.0f;
      float c = t * t;
      c = unmasked ? (c < inf ? c : inf) : 0.0f;
      chi[j] += c;
      if (OUT) {
        const size_t o = (size_t)(k0 + j) * npix + pix;
        if (a.m1) a.m1[o] = v + dp.v_center;
        if (a.resid) a.resid[o] = unmasked ? (c < inf ? t : nan) : 0.0f;
      }
    }
  }
#pragma unroll
  for (int j = 0; j < kRows; ++j) {
    float c = chi[j];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) c += __shfl_down_sync(0xffffffffu, c, off);
    if ((tid & 31) == 0) red[j][tid >> 5] = c;
  }
  __syncthreads();
  if (tid < nrows) {
    float tot = 0.0f;
    for (int w = 0; w < kThreads / 32; ++w) tot += red[tid][w];   // fixed order
    if (!(tot < inf) || !rows[tid].valid) tot = inf;
    a.chi2[k0 + tid] = tot;
  }
}

}  // namespace

// EvalArgs: m1 = velocity maps [K][ny][nx] or null, resid = velocity residuals [K][ny][nx] or null.
cudaError_t launch_vfield(const DevProblem& dp, const EvalArgs& a, cudaStream_t st) {
  const unsigned blocks = (unsigned)((a.K + kRows - 1) / kRows);
  const bool out = a.m1 || a.resid, shared = a.gal_index == nullptr;
  if (out && shared) vfield_kernel<true, true><<<blocks, kThreads, 0, st>>>(dp, a);
  else if (out) vfield_kernel<true, false><<<blocks, kThreads, 0, st>>>(dp, a);
  else if (shared) vfield_kernel<false, true><<<blocks, kThreads, 0, st>>>(dp, a);
  else vfield_kernel<false, false><<<blocks, kThreads, 0, st>>>(dp, a);
  return cudaGetLastError();
}

}  // namespace gbk
