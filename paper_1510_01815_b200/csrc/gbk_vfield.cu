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

#include "gbk_device.cuh"
#include "gbk_internal.h"

namespace gbk {

namespace {

constexpr int kRows = 4;        // parameter rows per block
constexpr int kThreads = 256;

struct VRow {
  u64 ea, eg;                               // Epinat slopes a, g (eq. 7), packed
  u64 nsp, ncp_ci, inv_rt, rt, k1, v0;     // packed (c, c): eq. 1-3 constants as in RowConst,
                                            // k1 = V_t sin i (x 2/pi for the arctan curve), v0 = V_sys - v_center
  float xo, yo, cp, nsp_ci;
  int valid, gal;
};

__device__ void vf_row(const DevProblem& dp, const EvalArgs& a, long long k, VRow* r) {
  const float* p = a.params + k * dp.row_stride;
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
  if (dp.rc_model == GBK_RC_EPINAT) {       // slopes a, g of eq. 7: slots 10, 11 of the 12-float row
    const float ea = p[10], eg = p[11];
    if (!(isfinite(ea) && isfinite(eg) && ea > 0.f && eg > 0.f)) r->valid = 0;
    r->ea = pk1(ea), r->eg = pk1(eg);
  }
  const float inv_ci = 1.0f / ci;
  r->xo = v[0], r->yo = v[1];
  r->cp = cp, r->nsp_ci = -sp * inv_ci;
  r->nsp = pk1(-sp), r->ncp_ci = pk1(-cp * inv_ci);
  r->inv_rt = pk1(1.0f / v[6]), r->rt = pk1(v[6]);
  r->k1 = pk1((dp.rc_model == GBK_RC_ARCTAN ? 0.63661977236758134f : 1.0f) * v[5] * si);
  r->v0 = pk1(v[4] - dp.v_center);
}

// eq. 1-4, 6 (or the ramp), 8 at the spaxel pair (x, y), (x + 1, y): velocities relative to
// v_center, in packed FP32.
__device__ __forceinline__ u64 vf_velocity2(const DevProblem& dp, const VRow& r, u64 dx, float dy) {
  const u64 xe = fma2(r.nsp, dx, pk1(dy * r.cp));               // eq. 1
  const u64 yd = fma2(r.ncp_ci, dx, pk1(dy * r.nsp_ci));        // eq. 2 / cos i
  const u64 r2 = fma2(xe, xe, mul2(yd, yd));                    // eq. 3
  float r2a, r2b;
  upk(r2, r2a, r2b);
  // r = 0: cos(theta) := 0 (A8) -- xe = 0 there, so a finite 1/r gives exactly that without a select
  const u64 rs = pk(rsqrt_approx(fmaxf(r2a, 1e-30f)), rsqrt_approx(fmaxf(r2b, 1e-30f)));
  const u64 rad = mul2(r2, rs), cos_t = mul2(xe, rs);           // eq. 4
  const u64 q = mul2(rad, r.inv_rt);
  float qa, qb;
  upk(q, qa, qb);
  u64 f;
  if (dp.rc_model == GBK_RC_ARCTAN) {                           // eq. 6 without (2/pi) V_t
    float ia, ib;
    upk(mul2(rs, r.rt), ia, ib);                                // 1/q = r_t / r
    // atan q = pi/2 - atan(1/q) for q > 1: the polynomial argument is the smaller of q and 1/q (one min)
    float ata, atb;
    upk(atan01_2(pk(fminf(qa, ia), fminf(qb, ib))), ata, atb);
    f = pk(qa > 1.0f ? 1.5707963267948966f - ata : ata, qb > 1.0f ? 1.5707963267948966f - atb : atb);
  } else if (dp.rc_model == GBK_RC_RAMP) {
    f = pk(fminf(qa, 1.0f), fminf(qb, 1.0f));                   // ramp (A7)
  } else {                                                      // eq. 7: q^g / (1 + q^a)
    const u64 lq = pk(lg2_approx(qa), lg2_approx(qb));          // q = 0: -inf -> q^g = q^a = 0
    float na, nb, da, db;
    upk(mul2(lq, r.eg), na, nb);
    upk(mul2(lq, r.ea), da, db);
    f = mul2(pk(ex2_approx(na), ex2_approx(nb)),
             pk(rcp_approx(1.0f + ex2_approx(da)), rcp_approx(1.0f + ex2_approx(db))));
  }
  return fma2(mul2(f, r.k1), cos_t, r.v0);                      // eq. 8
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
  const int ppr = (dp.nx + 1) >> 1;                 // spaxel pairs per map row
  const unsigned magic = div_magic(ppr);
  for (int item = tid; item < ppr * dp.ny; item += kThreads) {
    const int iy = div_fast(item, magic), ix = (item - iy * ppr) << 1;
    const int pix = iy * dp.nx + ix;
    const bool second = ix + 1 < dp.nx;
    const float x = (float)ix, y = (float)iy;
    float4 oa, ob = make_float4(0.f, 0.f, 0.f, 0.f);
    if (SHARED_OBS) {
      oa = __ldg(&dp.obs[pix]);
      if (second) ob = __ldg(&dp.obs[pix + 1]);
    }
#pragma unroll
    for (int j = 0; j < kRows; ++j) {
      if (j >= nrows) break;
      const VRow& r = rows[j];
      if (!SHARED_OBS) {
        const float4* o = dp.obs + (size_t)r.gal * npix + pix;
        oa = __ldg(o);
        if (second) ob = __ldg(o + 1);
      }
      float va, vb;
      upk(vf_velocity2(dp, r, pk(x - r.xo, x + 1.0f - r.xo), y - r.yo), va, vb);
      if (OUT && !r.valid) va = vb = nan;     // chi^2 of an out-of-domain row is set to +INF at the end whatever its sum
      const float ta = (va - oa.x) * oa.y, tb = (vb - ob.x) * ob.y;
      float ca = ta * ta, cb = tb * tb;
      // NaN or Inf -> +INF (fminf drops the NaN), masked -> 0: one min and one select each, no nested branch
      ca = oa.y > 0.0f ? fminf(ca, inf) : 0.0f;
      cb = ob.y > 0.0f ? fminf(cb, inf) : 0.0f;           // ob.y = 0 for the missing second spaxel
      chi[j] += ca + cb;
      if (OUT) {
        const size_t o = (size_t)(k0 + j) * npix + pix;
        if (a.m1) {
          a.m1[o] = va + dp.v_center;
          if (second) a.m1[o + 1] = vb + dp.v_center;
        }
        if (a.resid) {
          a.resid[o] = oa.y > 0.0f ? (ca < inf ? ta : nan) : 0.0f;
          if (second) a.resid[o + 1] = ob.y > 0.0f ? (cb < inf ? tb : nan) : 0.0f;
        }
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
