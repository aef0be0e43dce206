// Host side of libgbk: descriptor validation, table building, tiling, the C ABI of include/gbk.h.
// No CPU fallback: every compute call ends in a kernel launch or an error code.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <new>
#include <vector>

#include "gbk_internal.h"

using namespace gbk;

namespace {
thread_local char g_err[512] = "";
}

namespace gbk {
int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
void clear_error() { g_err[0] = 0; }
}  // namespace gbk

namespace {

#define GBK_CUDA(expr)                                                                  \
  do {                                                                                  \
    cudaError_t e_ = (expr);                                                            \
    if (e_ != cudaSuccess)                                                              \
      return fail(e_ == cudaErrorMemoryAllocation ? GBK_ERR_ALLOC : GBK_ERR_CUDA,       \
                  "%s: %s", #expr, cudaGetErrorString(e_));                             \
  } while (0)

int round_up4(int v) { return (v + 3) & ~3; }

// Gaussian taps exp(-j^2 / 2 sigma^2), j in [-R, R], R = ceil(4 sigma), normalised to sum 1
// (eq. 9 of the paper sampled on the grid).  sigma <= 0: delta.
std::vector<double> gaussian_taps(double sigma) {
  if (!(sigma > 0.0)) return {1.0};
  const int R = (int)ceil(4.0 * sigma);
  std::vector<double> t(2 * R + 1);
  double sum = 0.0;
  for (int j = -R; j <= R; ++j) sum += (t[j + R] = exp(-0.5 * (double)j * j / (sigma * sigma)));
  for (double& v : t) v /= sum;
  return t;
}

}  // namespace

struct gbk_problem {
  gbk_problem_desc d{};       // scalars only are meaningful after create
  DevProblem dp{};
  FusedLaunch fl{};
  // smaller tilings of the same problem for batches too small to fill the GPU (automatic tiling
  // only): level 0 is {dp, fl}; every further level halves the tile
  struct Level {
    DevProblem dp;
    FusedLaunch fl;
    int blocks_per_sm;   // resident blocks of this shape
    int rounds;          // passes of the voxel loop over the tile (4 pixels per thread and pass)
  };
  std::vector<Level> levels;
  int device = 0;
  int strategy = GBK_STRATEGY_CUBE;
  int extraction = GBK_EXTRACT_MOMENTS;
  int sm_count = 0, blocks_per_sm = 0;
  long long ext_voxels = 0;
  // device allocations owned by the problem
  double* chan_w = nullptr;
  float* tab = nullptr;         // tabulated intensity profile
  float* psf_taps = nullptr;
  int* psf_r = nullptr;
  float4* obs = nullptr;
  // Scratch of the eval calls, one set per CUDA stream the problem has been used on, so that
  // launches issued on different streams may overlap (they never share a buffer).
  struct StreamScratch {
    cudaStream_t stream = nullptr;
    float* partial = nullptr;         // [partial_cap] cross-tile chi^2 partials (tiled launches)
    unsigned* tile_count = nullptr;   // [count_cap] zeroed at allocation, self-resetting afterwards
    long long partial_cap = 0, count_cap = 0;
    float* st_params = nullptr;       // staging of gbk_eval_batch_host
    int32_t* st_gal = nullptr;
    float* st_chi2 = nullptr;
    long long st_cap = 0;
  };
  std::vector<StreamScratch*> scratch;
  std::mutex mu;                      // guards `scratch` (lookup and growth)
  // scratch of the unfused path
  float* uf_scratch = nullptr;
  long long uf_rows = 0;        // rows the scratch holds
  float* lsf_taps = nullptr;    // [2 r_v + 1], unfused path only
};

// ---- gbk_eval_batch_static: cross-tile scratch that nobody allocates ---------------------------
// [GBK_STATIC_MAX_PARTIALS] chi^2 partials (float) followed by [GBK_STATIC_MAX_ROWS] tile counters (unsigned,
// same size), in the device image of this translation unit: every device that loads the library holds it.
// The NAME below is a host-side stand-in in host code, not a device address: kernels get the address that
// cudaGetSymbolAddress returns for the current device (static_scratch_address).
static __device__ __align__(256) float g_static_scratch[GBK_STATIC_MAX_PARTIALS + GBK_STATIC_MAX_ROWS];

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mu;
float* g_static_addr[kMaxDevices] = {};        // device address of g_static_scratch on device i
cudaError_t g_static_err[kMaxDevices] = {};    // why it is missing

// Looks the address up once per device.  `device` must be current (cudaGetSymbolAddress answers for the
// current device; the first call also loads this unit's device image, which is why gbk_create_problem
// makes it at set-up and gbk_eval_batch_static only reads the table).
float* static_scratch_address(int device, bool lookup) {
  if (device < 0 || device >= kMaxDevices) return nullptr;
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (!g_static_addr[device] && lookup) {
    void* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);
    g_static_err[device] = e;
    if (e == cudaSuccess) g_static_addr[device] = static_cast<float*>(ptr);
    else (void)cudaGetLastError();             // not sticky for the caller's next CUDA call
  }
  return g_static_addr[device];
}
}  // namespace

extern "C" const char* gbk_last_error(void) { return g_err; }

extern "C" int gbk_destroy(gbk_problem* p) {
  if (!p) return GBK_OK;
  cudaFree(p->chan_w);
  cudaFree(p->tab);
  cudaFree(p->psf_taps);
  cudaFree(p->psf_r);
  cudaFree(p->obs);
  for (gbk_problem::StreamScratch* sc : p->scratch) {
    cudaFree(sc->partial), cudaFree(sc->tile_count);
    cudaFree(sc->st_params), cudaFree(sc->st_gal), cudaFree(sc->st_chi2);
    delete sc;
  }
  cudaFree(p->uf_scratch);
  cudaFree(p->lsf_taps);
  delete p;
  return GBK_OK;
}

extern "C" int gbk_create_problem(const gbk_problem_desc* d, gbk_problem** out) {
  g_err[0] = 0;
  if (!d || !out) return fail(GBK_ERR_ARG, "null descriptor or output pointer");
  *out = nullptr;
  if (d->nx < 1 || d->ny < 1 || d->nv < 1 || d->u < 1 || d->n_gal < 1)
    return fail(GBK_ERR_ARG, "nx, ny, nv, u and n_gal must be >= 1");
  if ((long long)d->nx * d->u > 16384 || (long long)d->ny * d->u > 16384 || d->nv > 16384)
    return fail(GBK_ERR_ARG, "grid too large");
  if (!(d->dv > 0.f) || !isfinite(d->dv) || !isfinite(d->v_center))
    return fail(GBK_ERR_ARG, "dv must be > 0 and finite, v_center finite");
  if (d->rc_model != GBK_RC_ARCTAN && d->rc_model != GBK_RC_RAMP && d->rc_model != GBK_RC_EPINAT)
    return fail(GBK_ERR_ARG, "unknown rc_model %d", d->rc_model);
  if (!d->vobs || !d->verr) return fail(GBK_ERR_ARG, "vobs and verr are required");
  if ((d->sobs == nullptr) != (d->serr == nullptr))
    return fail(GBK_ERR_ARG, "sobs and serr must both be given or both be NULL");
  if (d->psf_kind != GBK_PSF_GAUSSIAN && d->psf_kind != GBK_PSF_IMAGE)
    return fail(GBK_ERR_ARG, "unknown psf_kind %d", d->psf_kind);
  if (!isfinite(d->lsf_sigma)) return fail(GBK_ERR_ARG, "lsf_sigma must be finite");
  if (d->intensity_table) {
    if (d->intensity_n < 2 || d->intensity_n > (1 << 20) || !(d->intensity_dx > 0.f) || !isfinite(d->intensity_dx))
      return fail(GBK_ERR_ARG, "intensity_table needs 2 <= intensity_n <= 2^20 and intensity_dx > 0");
    for (int j = 0; j < d->intensity_n; ++j)
      if (!isfinite(d->intensity_table[j]) || d->intensity_table[j] < 0.f)
        return fail(GBK_ERR_ARG, "intensity_table[%d] must be finite and >= 0", j);
  }

  const int n_psf = d->psf_per_gal ? d->n_gal : 1;
  const size_t npix = (size_t)d->nx * d->ny;

  // ---- LSF taps and the LSF-folded channel weights (a4) ---------------------------------
  const std::vector<double> lsf = gaussian_taps(d->lsf_sigma > 0.f ? (double)d->lsf_sigma / d->dv : 0.0);
  const int r_v = (int)(lsf.size() / 2);
  if (r_v > kMaxLsfR) return fail(GBK_ERR_UNSUPPORTED, "LSF radius %d > %d channels", r_v, kMaxLsfR);
  const int nvx = d->nv + 2 * r_v;
  // w_q[c] = sum over in-band channels k of L[k - ch] * v'_k^q, ch = c - r_v,
  // v'_k = (k - (nv-1)/2) dv  (velocities relative to v_center).
  const int nvx_pad = (nvx + kChanBlock - 1) / kChanBlock * kChanBlock;
  std::vector<double> chan(3 * (size_t)nvx_pad, 0.0);   // weightless padding channels past nvx
  for (int c = 0; c < nvx; ++c) {
    const int ch = c - r_v;
    double w[3] = {0, 0, 0};
    for (int k = std::max(0, ch - r_v); k <= std::min(d->nv - 1, ch + r_v); ++k) {
      const double L = lsf[(k - ch) + r_v];
      const double v = ((double)k - 0.5 * (d->nv - 1)) * (double)d->dv;
      w[0] += L;
      w[1] += L * v;
      w[2] += L * v * v;
    }
    chan[3 * c] = w[0], chan[3 * c + 1] = w[1], chan[3 * c + 2] = w[2];
  }

  // ---- PSF sets ------------------------------------------------------------------------
  std::vector<int> psf_r(n_psf);
  std::vector<float> psf_taps;
  int psf_stride = 0, r_p_max = 0;
  if (d->psf_kind == GBK_PSF_GAUSSIAN) {
    if (!d->psf_fwhm) return fail(GBK_ERR_ARG, "psf_fwhm is required for a Gaussian PSF");
    std::vector<std::vector<double>> sets(n_psf);
    for (int g = 0; g < n_psf; ++g) {
      const double fwhm = d->psf_fwhm[g];
      if (!isfinite(fwhm)) return fail(GBK_ERR_ARG, "psf_fwhm[%d] is not finite", g);
      const double sigma_f = (double)d->u * fwhm / (2.0 * sqrt(2.0 * log(2.0)));
      sets[g] = gaussian_taps(sigma_f);
      psf_r[g] = (int)(sets[g].size() / 2);
      r_p_max = std::max(r_p_max, psf_r[g]);
    }
    if (r_p_max > kMaxSepR)
      return fail(GBK_ERR_UNSUPPORTED, "Gaussian PSF radius %d fine pixels > %d", r_p_max, kMaxSepR);
    psf_stride = 2 * r_p_max + 1;
    psf_taps.assign((size_t)n_psf * psf_stride, 0.f);
    for (int g = 0; g < n_psf; ++g)
      for (size_t j = 0; j < sets[g].size(); ++j) psf_taps[(size_t)g * psf_stride + j] = (float)sets[g][j];
  } else {
    if (!d->psf_image) return fail(GBK_ERR_ARG, "psf_image is required for an image PSF");
    if (d->psf_n < 1 || (d->psf_n & 1) == 0) return fail(GBK_ERR_ARG, "psf_n must be odd and >= 1");
    if (d->psf_n > kMaxPsfN) return fail(GBK_ERR_UNSUPPORTED, "psf_n %d > %d", d->psf_n, kMaxPsfN);
    const int n = d->psf_n;
    psf_stride = n * n;
    r_p_max = n / 2;
    psf_taps.resize((size_t)n_psf * psf_stride);
    for (int g = 0; g < n_psf; ++g) {
      const float* img = d->psf_image + (size_t)g * psf_stride;
      double sum = 0.0;
      for (int i = 0; i < psf_stride; ++i) {
        if (!isfinite(img[i])) return fail(GBK_ERR_ARG, "psf_image has a non-finite value");
        sum += img[i];
      }
      if (!(sum > 0.0)) return fail(GBK_ERR_ARG, "psf_image must have a positive sum");
      // stored flipped: the kernel correlates, which is then the true convolution
      for (int y = 0; y < n; ++y)
        for (int x = 0; x < n; ++x)
          psf_taps[(size_t)g * psf_stride + y * n + x] = (float)(img[(n - 1 - y) * n + (n - 1 - x)] / sum);
      psf_r[g] = n / 2;
    }
  }

  // ---- packed observation: {vobs - v_center, 1/E_v (0 = masked), sobs, 1/E_s} ------------
  std::vector<float4> obs((size_t)d->n_gal * npix);
  for (size_t i = 0; i < obs.size(); ++i) {
    const bool unmasked = !d->mask || d->mask[i] != 0;
    float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
    if (unmasked) {
      const float v = d->vobs[i], ev = d->verr[i];
      if (!isfinite(v) || !isfinite(ev) || !(ev > 0.f))
        return fail(GBK_ERR_ARG, "unmasked spaxel %zu: vobs/verr must be finite and verr > 0", i);
      o.x = (float)((double)v - (double)d->v_center);
      o.y = (float)(1.0 / (double)ev);
      if (d->sobs) {
        const float s = d->sobs[i], es = d->serr[i];
        if (!isfinite(s) || !isfinite(es) || !(es > 0.f))
          return fail(GBK_ERR_ARG, "unmasked spaxel %zu: sobs/serr must be finite and serr > 0", i);
        o.z = s;
        o.w = (float)(1.0 / (double)es);
      }
      if (!(o.y > 0.f)) return fail(GBK_ERR_ARG, "unmasked spaxel %zu: verr too large", i);
    }
    obs[i] = o;
  }

  // ---- device and tiling ---------------------------------------------------------------
  int dev = d->device;
  if (dev < 0) GBK_CUDA(cudaGetDevice(&dev));
  DeviceGuard guard(dev);
  GBK_CUDA(guard.status);
  cudaDeviceProp prop;
  GBK_CUDA(cudaGetDeviceProperties(&prop, dev));
  const size_t smem_cap = prop.sharedMemPerBlockOptin;

  gbk_problem* p = new (std::nothrow) gbk_problem;
  if (!p) return fail(GBK_ERR_ALLOC, "out of host memory");
  p->d = *d;
  p->device = dev;
  p->strategy = d->rc_model == GBK_RC_EPINAT ? GBK_STRATEGY_VFIELD : GBK_STRATEGY_CUBE;
  p->sm_count = prop.multiProcessorCount;
  DevProblem& dp = p->dp;
  dp.nx = d->nx, dp.ny = d->ny, dp.nv = d->nv, dp.u = d->u, dp.n_gal = d->n_gal;
  dp.fw = d->u * d->nx, dp.fh = d->u * d->ny;
  dp.r_v = r_v, dp.nvx = nvx, dp.nvx_pad = nvx_pad;
  dp.rc_model = d->rc_model, dp.psf_kind = d->psf_kind;
  dp.row_stride = d->rc_model == GBK_RC_EPINAT ? GBK_P_EPINAT : GBK_P;
  dp.tab_n = d->intensity_table ? d->intensity_n : 0;
  dp.tab_inv_dx = d->intensity_table ? 1.0f / d->intensity_dx : 0.0f;
  dp.has_disp = d->sobs ? 1 : 0, dp.psf_per_gal = d->psf_per_gal ? 1 : 0;
  dp.r_p_max = r_p_max, dp.psf_stride = psf_stride;
  dp.dv = d->dv, dp.v_center = d->v_center;
  dp.vrel_first = (float)((-(double)r_v - 0.5 * (d->nv - 1)) * (double)d->dv);
  dp.vhalf = (float)(0.5 * (d->nv - 1) * (double)d->dv);
  dp.inv_u = 1.0f / (float)d->u, dp.inv_u2 = 1.0f / ((float)d->u * (float)d->u);

  auto set_tile = [&](int tws, int ths) {   // in spaxels
    dp.tile_w = tws * d->u, dp.tile_h = ths * d->u;
    dp.tiles_x = (d->nx + tws - 1) / tws, dp.tiles_y = (d->ny + ths - 1) / ths;
    dp.ntiles = dp.tiles_x * dp.tiles_y;
    dp.ews = round_up4(dp.tile_w) + 4 * ((2 * r_p_max + 4 + 3) / 4) - 4;
    dp.ehs = (dp.tile_h + kVBlock - 1) / kVBlock * kVBlock + 2 * r_p_max;  // the vertical pass reads whole blocks
    dp.img_fast = d->psf_kind == GBK_PSF_IMAGE && d->psf_n <= kMaxFastPsfN ? 1 : 0;
    dp.spare_plane = 0;
    if (dp.img_fast) {
      // the 2-D pass reads 8-pixel chunks plus the kernel width as float4s, with lanes along y:
      // a row stride = 4 (mod 8) floats keeps those 16-byte reads free of bank conflicts
      const int nxc = (dp.tile_w + 7) / 8, nv4 = (8 + 2 * r_p_max + 3) / 4;
      dp.ews = std::max(dp.ews, 8 * nxc - 8 + 4 * nv4);
      while (dp.ews % 8 != 4) ++dp.ews;
      dp.spare_plane = dp.tile_h * dp.ews;
    }
    return fused_smem_bytes(dp);
  };
  int tws = d->tile_w > 0 ? std::min(d->tile_w, d->nx) : d->nx;
  int ths = d->tile_h > 0 ? std::min(d->tile_h, d->ny) : d->ny;
  size_t smem = set_tile(tws, ths);
  if (d->tile_w <= 0 || d->tile_h <= 0) {
    // automatic: halve the longer side until two blocks fit on an SM (or at least one does)
    const size_t want = (smem_cap - 2048) / 2;
    while (smem > want && (tws > 8 || ths > 8)) {
      if (d->tile_w <= 0 && (tws >= ths || d->tile_h > 0) && tws > 8) tws = (tws + 1) / 2;
      else if (d->tile_h <= 0 && ths > 8) ths = (ths + 1) / 2;
      else break;
      smem = set_tile(tws, ths);
    }
  }
  if (smem > smem_cap) {
    delete p;
    return fail(GBK_ERR_UNSUPPORTED, "tile %dx%d spaxels needs %zu B of shared memory (max %zu)", tws,
                ths, smem, smem_cap);
  }
  // launch shape: P pixels per thread in the voxel loop, threads per block
  const int n_ext = (dp.tile_w + 2 * r_p_max) * (dp.tile_h + 2 * r_p_max);
  p->fl.smem_bytes = (int)smem;
  // 256 threads: three blocks of a whole-field config-3 tile are resident per SM (70.7 KB and
  // <= 85 registers x 256 threads each), so their phases overlap (measured best of 128..384)
  auto threads_for = [&](const DevProblem& q) {
    const int ne = (q.tile_w + 2 * r_p_max) * (q.tile_h + 2 * r_p_max);
    return std::min(256, std::max(64, ((ne + 3) / 4 + 31) / 32 * 32));
  };
  p->fl.threads = threads_for(dp);
  (void)n_ext;
  long long ext = 0;
  for (int ty = 0; ty < dp.tiles_y; ++ty)
    for (int tx = 0; tx < dp.tiles_x; ++tx) {
      const int tw = std::min(dp.tile_w, dp.fw - tx * dp.tile_w), th = std::min(dp.tile_h, dp.fh - ty * dp.tile_h);
      ext += (long long)(tw + 2 * r_p_max) * (th + 2 * r_p_max) * nvx;
    }
  p->ext_voxels = ext;

  auto bail = [&](int code) {
    gbk_destroy(p);
    return code;
  };
#define GBK_CUDA_P(expr)                                                                       \
  do {                                                                                         \
    cudaError_t e_ = (expr);                                                                   \
    if (e_ != cudaSuccess)                                                                     \
      return bail(fail(e_ == cudaErrorMemoryAllocation ? GBK_ERR_ALLOC : GBK_ERR_CUDA, "%s: %s", \
                       #expr, cudaGetErrorString(e_)));                                        \
  } while (0)
  GBK_CUDA_P(cudaMalloc(&p->chan_w, sizeof(double) * chan.size()));
  GBK_CUDA_P(cudaMalloc(&p->psf_taps, sizeof(float) * psf_taps.size()));
  GBK_CUDA_P(cudaMalloc(&p->psf_r, sizeof(int) * n_psf));
  GBK_CUDA_P(cudaMalloc(&p->obs, sizeof(float4) * obs.size()));
  {
    std::vector<float> lsf_f(lsf.begin(), lsf.end());
    GBK_CUDA_P(cudaMalloc(&p->lsf_taps, sizeof(float) * lsf_f.size()));
    GBK_CUDA_P(cudaMemcpy(p->lsf_taps, lsf_f.data(), sizeof(float) * lsf_f.size(), cudaMemcpyHostToDevice));
  }
  GBK_CUDA_P(cudaMemcpy(p->chan_w, chan.data(), sizeof(double) * chan.size(), cudaMemcpyHostToDevice));
  if (d->intensity_table) {
    GBK_CUDA_P(cudaMalloc(&p->tab, sizeof(float) * (size_t)d->intensity_n));
    GBK_CUDA_P(cudaMemcpy(p->tab, d->intensity_table, sizeof(float) * (size_t)d->intensity_n, cudaMemcpyHostToDevice));
  }
  dp.tab = p->tab;
  GBK_CUDA_P(cudaMemcpy(p->psf_taps, psf_taps.data(), sizeof(float) * psf_taps.size(), cudaMemcpyHostToDevice));
  GBK_CUDA_P(cudaMemcpy(p->psf_r, psf_r.data(), sizeof(int) * n_psf, cudaMemcpyHostToDevice));
  GBK_CUDA_P(cudaMemcpy(p->obs, obs.data(), sizeof(float4) * obs.size(), cudaMemcpyHostToDevice));
  dp.chan_w = p->chan_w, dp.psf_taps = p->psf_taps, dp.psf_r = p->psf_r, dp.obs = p->obs;
  {
    // opt in to the device's largest dynamic shared memory once and for all: the attribute belongs
    // to the kernel, not to this problem, and a later problem with a smaller tile must not lower it
    FusedLaunch cap = p->fl;
    cap.smem_bytes = (int)smem_cap;
    GBK_CUDA_P(fused_prepare(cap));
  }
  GBK_CUDA_P(fused_occupancy(dp, p->fl, &p->blocks_per_sm));
  auto rounds_for = [&](const DevProblem& q, const FusedLaunch& f) {
    const int ne = (q.tile_w + 2 * r_p_max) * (q.tile_h + 2 * r_p_max);
    return (ne + 4 * f.threads - 1) / (4 * f.threads);
  };
  p->levels.push_back({dp, p->fl, std::max(1, p->blocks_per_sm), rounds_for(dp, p->fl)});
  if (d->tile_w <= 0 && d->tile_h <= 0) {
    const DevProblem dp0 = dp;
    int lw = tws, lh = ths;
    while (std::max(lw, lh) > 4) {
      lw = std::max(4, (lw + 1) / 2), lh = std::max(4, (lh + 1) / 2);
      FusedLaunch lf = p->fl;
      lf.smem_bytes = (int)set_tile(lw, lh);
      lf.threads = threads_for(dp);
      int bps = 1;
      GBK_CUDA_P(fused_occupancy(dp, lf, &bps));
      p->levels.push_back({dp, lf, std::max(1, bps), rounds_for(dp, lf)});
    }
    dp = dp0;
  }
#undef GBK_CUDA_P
  // set-up of gbk_eval_batch_static on this device (a failure is reported by that call, not here)
  (void)static_scratch_address(dev, true);
  // host pointers of the descriptor are not kept
  p->d.vobs = p->d.verr = p->d.sobs = p->d.serr = nullptr;
  p->d.mask = nullptr;
  p->d.psf_fwhm = p->d.psf_image = nullptr;
  p->d.intensity_table = nullptr;
  *out = p;
  return GBK_OK;
}

extern "C" int gbk_get_info(const gbk_problem* p, gbk_problem_info* info) {
  if (!p || !info) return fail(GBK_ERR_ARG, "null argument");
  const DevProblem& dp = p->dp;
  info->nx = dp.nx, info->ny = dp.ny, info->nv = dp.nv, info->u = dp.u, info->n_gal = dp.n_gal;
  info->r_v = dp.r_v, info->r_p_max = dp.r_p_max;
  info->tile_w = dp.tile_w / dp.u, info->tile_h = dp.tile_h / dp.u;
  info->tiles_x = dp.tiles_x, info->tiles_y = dp.tiles_y;
  info->block_threads = p->fl.threads, info->smem_bytes = p->fl.smem_bytes;
  info->blocks_per_sm = p->blocks_per_sm, info->sm_count = p->sm_count;
  info->ext_voxels_per_eval = p->ext_voxels;
  info->device = p->device;
  info->strategy = p->strategy;
  info->unfused_bytes_per_eval = (int64_t)unfused_algorithmic_bytes_per_row(p->dp);
  info->row_stride = dp.row_stride;
  info->extraction = p->extraction;
  return GBK_OK;
}

extern "C" int gbk_set_strategy(gbk_problem* p, int32_t strategy) {
  g_err[0] = 0;
  if (!p) return fail(GBK_ERR_ARG, "null problem");
  if (strategy != GBK_STRATEGY_CUBE && strategy != GBK_STRATEGY_VFIELD)
    return fail(GBK_ERR_ARG, "unknown strategy %d", strategy);
  p->strategy = strategy;
  return GBK_OK;
}

extern "C" int gbk_set_extraction(gbk_problem* p, int32_t extraction) {
  g_err[0] = 0;
  if (!p) return fail(GBK_ERR_ARG, "null problem");
  if (extraction != GBK_EXTRACT_MOMENTS && extraction != GBK_EXTRACT_GAUSSFIT)
    return fail(GBK_ERR_ARG, "unknown extraction %d", extraction);
  p->extraction = extraction;
  return GBK_OK;
}

static int check_eval_args(gbk_problem* p, const float* params, int64_t K, float* chi2) {
  if (!p) return fail(GBK_ERR_ARG, "null problem");
  if (K < 0) return fail(GBK_ERR_ARG, "K must be >= 0");
  if (K > 0 && (!params || !chi2)) return fail(GBK_ERR_ARG, "params and chi2 are required");
  return GBK_OK;
}

// The tiling level a batch of K rows runs on: the one with the fewest (waves of blocks) x
// (voxel-loop passes per block); ties go to the larger tile (less halo work).
static size_t pick_level(const gbk_problem* p, int64_t K) {
  size_t lv = 0;
  long long best_cost = 0;
  for (size_t i = 0; i < p->levels.size(); ++i) {
    const auto& L = p->levels[i];
    const long long slots = (long long)p->sm_count * L.blocks_per_sm;
    const long long cost = ((long long)K * L.dp.ntiles + slots - 1) / slots * L.rounds;
    if (i == 0 || cost < best_cost) best_cost = cost, lv = i;
  }
  return lv;
}

static gbk_problem::StreamScratch* scratch_of(gbk_problem* p, cudaStream_t st) {
  for (gbk_problem::StreamScratch* sc : p->scratch)
    if (sc->stream == st) return sc;
  gbk_problem::StreamScratch* sc = new (std::nothrow) gbk_problem::StreamScratch;
  if (!sc) return nullptr;
  sc->stream = st;
  p->scratch.push_back(sc);
  return sc;
}

// Grows the cross-tile scratch of a stream to `need` partials and `rows` counters.  Never during a
// stream capture: allocation is illegal there, so the caller has to gbk_reserve beforehand.
static int grow_tile_scratch(gbk_problem::StreamScratch* sc, long long need, long long rows, cudaStream_t st) {
  if (need <= sc->partial_cap && rows <= sc->count_cap) return GBK_OK;
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  GBK_CUDA(cudaStreamIsCapturing(st, &cap));
  if (cap != cudaStreamCaptureStatusNone)
    return fail(GBK_ERR_ARG, "the stream is being captured and the cross-tile scratch is too small: call "
                             "gbk_reserve(problem, K, stream) before the capture");
  if (need > sc->partial_cap) {
    if (sc->partial) GBK_CUDA(cudaFree(sc->partial));   // waits for launches that still use it
    sc->partial = nullptr, sc->partial_cap = 0;
    GBK_CUDA(cudaMalloc(&sc->partial, sizeof(float) * (size_t)need));
    sc->partial_cap = need;
  }
  if (rows > sc->count_cap) {
    if (sc->tile_count) GBK_CUDA(cudaFree(sc->tile_count));
    sc->tile_count = nullptr, sc->count_cap = 0;
    GBK_CUDA(cudaMalloc(&sc->tile_count, sizeof(unsigned) * (size_t)rows));
    GBK_CUDA(cudaMemsetAsync(sc->tile_count, 0, sizeof(unsigned) * (size_t)rows, st));
    sc->count_cap = rows;
  }
  return GBK_OK;
}

extern "C" int gbk_reserve(gbk_problem* p, int64_t K_max, void* cuda_stream) {
  g_err[0] = 0;
  if (!p) return fail(GBK_ERR_ARG, "null problem");
  if (K_max < 0) return fail(GBK_ERR_ARG, "K_max must be >= 0");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  GBK_CUDA(guard.status);
  // the largest K x tiles any batch of up to K_max rows asks for (the tiling depends on K)
  long long need = 0, rows = 0;
  for (int64_t K = 1; K <= K_max; ++K) {
    const int ntiles = p->levels[pick_level(p, K)].dp.ntiles;
    if (ntiles > 1) need = std::max(need, (long long)K * ntiles), rows = K;
  }
  std::lock_guard<std::mutex> lock(p->mu);
  gbk_problem::StreamScratch* sc = scratch_of(p, st);
  if (!sc) return fail(GBK_ERR_ALLOC, "out of host memory");
  if (int rc = grow_tile_scratch(sc, need, rows, st)) return rc;
  if (K_max > sc->st_cap) {
    cudaFree(sc->st_params), cudaFree(sc->st_gal), cudaFree(sc->st_chi2);
    sc->st_params = nullptr, sc->st_gal = nullptr, sc->st_chi2 = nullptr, sc->st_cap = 0;
    GBK_CUDA(cudaMalloc(&sc->st_params, sizeof(float) * GBK_P_MAX * (size_t)K_max));
    GBK_CUDA(cudaMalloc(&sc->st_gal, sizeof(int32_t) * (size_t)K_max));
    GBK_CUDA(cudaMalloc(&sc->st_chi2, sizeof(float) * (size_t)K_max));
    sc->st_cap = K_max;
  }
  return GBK_OK;
}

static int eval_batch_impl(gbk_problem* p, const float* params, const int32_t* gal_index, int64_t K,
                           float* chi2, float* m0, float* m1, float* m2, float* resid,
                           unsigned long long* counters, void* cuda_stream);

extern "C" int gbk_eval_batch(gbk_problem* p, const float* params, const int32_t* gal_index, int64_t K,
                              float* chi2, float* m0, float* m1, float* m2, float* resid,
                              void* cuda_stream) {
  return eval_batch_impl(p, params, gal_index, K, chi2, m0, m1, m2, resid, nullptr, cuda_stream);
}

extern "C" int gbk_eval_batch_counted(gbk_problem* p, const float* params, const int32_t* gal_index,
                                      int64_t K, float* chi2, uint64_t* counters, void* cuda_stream) {
  if (!counters) return fail(GBK_ERR_ARG, "counters is required");
  return eval_batch_impl(p, params, gal_index, K, chi2, nullptr, nullptr, nullptr, nullptr,
                         reinterpret_cast<unsigned long long*>(counters), cuda_stream);
}

static int eval_unfused_impl(gbk_problem* p, const float* params, const int32_t* gal_index, int64_t K,
                             float* chi2, float* m0, float* m1, float* m2, float* resid, void* cuda_stream);

static int eval_batch_impl(gbk_problem* p, const float* params, const int32_t* gal_index, int64_t K,
                           float* chi2, float* m0, float* m1, float* m2, float* resid,
                           unsigned long long* counters, void* cuda_stream) {
  g_err[0] = 0;
  if (int rc = check_eval_args(p, params, K, chi2)) return rc;
  if (K == 0) return GBK_OK;
  if (p->extraction == GBK_EXTRACT_GAUSSFIT) {   // needs whole spectra: the multi-kernel pipeline
    if (counters) return fail(GBK_ERR_UNSUPPORTED, "work counters belong to the fused kernel (moment extraction)");
    return eval_unfused_impl(p, params, gal_index, K, chi2, m0, m1, m2, resid, cuda_stream);
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  GBK_CUDA(guard.status);
  const size_t lv = pick_level(p, K);
  const DevProblem& dp = p->levels[lv].dp;
  if (K * (int64_t)dp.ntiles > 0x7fffffffLL) return fail(GBK_ERR_ARG, "K * tiles exceeds the grid limit");
  float* partial = nullptr;
  unsigned* tile_count = nullptr;
  if (dp.ntiles > 1) {
    std::lock_guard<std::mutex> lock(p->mu);
    gbk_problem::StreamScratch* sc = scratch_of(p, st);
    if (!sc) return fail(GBK_ERR_ALLOC, "out of host memory");
    if (int rc = grow_tile_scratch(sc, (long long)K * dp.ntiles, K, st)) return rc;
    partial = sc->partial, tile_count = sc->tile_count;
  }
  EvalArgs a{params, gal_index, (long long)K, chi2, m0, m1, m2, resid, partial, tile_count, counters};
  GBK_CUDA(launch_fused(dp, a, p->levels[lv].fl, st));
  return GBK_OK;
}

// gbk_eval_batch with the cross-tile scratch in g_static_scratch: no allocation of any kind (no scratch table,
// no cudaMalloc), one cudaMemsetAsync and one launch on the caller's stream.
extern "C" int gbk_eval_batch_static(gbk_problem* p, const float* params, const int32_t* gal_index, int64_t K,
                                     float* chi2, float* m0, float* m1, float* m2, float* resid,
                                     void* cuda_stream) {
  g_err[0] = 0;
  if (int rc = check_eval_args(p, params, K, chi2)) return rc;
  if (K == 0) return GBK_OK;
  if (p->extraction == GBK_EXTRACT_GAUSSFIT)
    return fail(GBK_ERR_UNSUPPORTED, "gbk_eval_batch_static: GBK_EXTRACT_GAUSSFIT runs the multi-kernel pipeline, "
                                     "which needs a model cube of scratch; use gbk_eval_batch");
  const DevProblem& dp = p->levels[pick_level(p, K)].dp;
  const FusedLaunch& fl = p->levels[pick_level(p, K)].fl;
  if (K > (int64_t)GBK_STATIC_MAX_ROWS)
    return fail(GBK_ERR_ARG, "gbk_eval_batch_static: K = %lld rows exceeds GBK_STATIC_MAX_ROWS = %d; split the batch "
                             "or use gbk_eval_batch", (long long)K, (int)GBK_STATIC_MAX_ROWS);
  if (K * (int64_t)dp.ntiles > (int64_t)GBK_STATIC_MAX_PARTIALS)
    return fail(GBK_ERR_ARG, "gbk_eval_batch_static: K x tiles = %lld x %d exceeds GBK_STATIC_MAX_PARTIALS = %d; "
                             "split the batch or use gbk_eval_batch", (long long)K, dp.ntiles,
                (int)GBK_STATIC_MAX_PARTIALS);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  GBK_CUDA(guard.status);
  float* scratch = static_scratch_address(p->device, false);
  if (!scratch)
    return fail(GBK_ERR_CUDA, "gbk_eval_batch_static: no device address of the static scratch on device %d "
                              "(cudaGetSymbolAddress at gbk_create_problem: %s)", p->device,
                p->device >= 0 && p->device < kMaxDevices ? cudaGetErrorString(g_static_err[p->device])
                                                          : "device ordinal beyond the table");
  float* partial = scratch;
  unsigned* tile_count = reinterpret_cast<unsigned*>(scratch + GBK_STATIC_MAX_PARTIALS);
  // the array keeps whatever the last call (of any problem) left: the counters must start at zero; the
  // partials are all written before they are read
  if (dp.ntiles > 1) GBK_CUDA(cudaMemsetAsync(tile_count, 0, sizeof(unsigned) * (size_t)K, st));
  EvalArgs a{params, gal_index, (long long)K, chi2, m0, m1, m2, resid, partial, tile_count, nullptr};
  GBK_CUDA(launch_fused(dp, a, fl, st));
  return GBK_OK;
}

extern "C" int gbk_eval_vfield_batch(gbk_problem* p, const float* params, const int32_t* gal_index,
                                     int64_t K, float* chi2, float* vmap, float* resid,
                                     void* cuda_stream) {
  g_err[0] = 0;
  if (int rc = check_eval_args(p, params, K, chi2)) return rc;
  if (K == 0) return GBK_OK;
  DeviceGuard guard(p->device);
  GBK_CUDA(guard.status);
  EvalArgs a{params, gal_index, (long long)K, chi2, nullptr, vmap, nullptr, resid, nullptr, nullptr, nullptr};
  GBK_CUDA(launch_vfield(p->dp, a, (cudaStream_t)cuda_stream));
  return GBK_OK;
}

extern "C" int gbk_eval_batch_host(gbk_problem* p, const float* params, const int32_t* gal_index,
                                   int64_t K, float* chi2, void* cuda_stream) {
  g_err[0] = 0;
  if (int rc = check_eval_args(p, params, K, chi2)) return rc;
  if (K == 0) return GBK_OK;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(p->device);
  GBK_CUDA(guard.status);
  gbk_problem::StreamScratch* sc;
  {
    std::lock_guard<std::mutex> lock(p->mu);
    sc = scratch_of(p, st);
  }
  if (!sc) return fail(GBK_ERR_ALLOC, "out of host memory");
  if (K > sc->st_cap)
    if (int rc = gbk_reserve(p, K, cuda_stream)) return rc;
  GBK_CUDA(cudaMemcpyAsync(sc->st_params, params, sizeof(float) * p->dp.row_stride * (size_t)K, cudaMemcpyHostToDevice, st));
  if (gal_index)
    GBK_CUDA(cudaMemcpyAsync(sc->st_gal, gal_index, sizeof(int32_t) * (size_t)K, cudaMemcpyHostToDevice, st));
  if (int rc = gbk_eval_batch(p, sc->st_params, gal_index ? sc->st_gal : nullptr, K, sc->st_chi2, nullptr,
                              nullptr, nullptr, nullptr, cuda_stream))
    return rc;
  GBK_CUDA(cudaMemcpyAsync(chi2, sc->st_chi2, sizeof(float) * (size_t)K, cudaMemcpyDeviceToHost, st));
  GBK_CUDA(cudaStreamSynchronize(st));
  return GBK_OK;
}

extern "C" int gbk_eval_batch_unfused(gbk_problem* p, const float* params, const int32_t* gal_index,
                                      int64_t K, float* chi2, float* m0, float* m1, float* m2,
                                      float* resid, void* cuda_stream) {
  g_err[0] = 0;
  if (int rc = check_eval_args(p, params, K, chi2)) return rc;
  if (K == 0) return GBK_OK;
  return eval_unfused_impl(p, params, gal_index, K, chi2, m0, m1, m2, resid, cuda_stream);
}

static int eval_unfused_impl(gbk_problem* p, const float* params, const int32_t* gal_index, int64_t K,
                             float* chi2, float* m0, float* m1, float* m2, float* resid, void* cuda_stream) {
  DeviceGuard guard(p->device);
  GBK_CUDA(guard.status);
  // scratch: two cubes + one contribution map per row, for a chunk of rows (<= 2 GiB, grown lazily)
  const size_t per_row = unfused_bytes_per_row(p->dp);
  const long long cap_rows = std::max<long long>(1, (long long)((size_t(2) << 30) / per_row));
  const long long want = std::min<long long>(K, cap_rows);
  if (want > p->uf_rows) {
    if (p->uf_scratch) GBK_CUDA(cudaFree(p->uf_scratch));
    p->uf_scratch = nullptr, p->uf_rows = 0;
    GBK_CUDA(cudaMalloc(&p->uf_scratch, per_row * (size_t)want));
    p->uf_rows = want;
  }
  EvalArgs a{params, gal_index, (long long)K, chi2, m0, m1, m2, resid, nullptr, nullptr, nullptr};
  GBK_CUDA(launch_unfused(p->dp, a, p->lsf_taps, p->uf_scratch, p->uf_rows, p->sm_count, p->extraction,
                          (cudaStream_t)cuda_stream));
  return GBK_OK;
}

extern "C" int gbk_probe_pipe(int which, int64_t iters, int blocks, int threads, float* sink,
                              double* ops_per_launch, void* cuda_stream) {
  g_err[0] = 0;
  if ((which != 0 && which != 1) || iters < 1 || blocks < 1 || threads < 32 || threads > 1024 || !sink)
    return fail(GBK_ERR_ARG, "bad probe arguments");
  if (ops_per_launch) *ops_per_launch = 16.0 * (double)iters * (double)blocks * (double)threads;
  GBK_CUDA(launch_probe(which, iters, blocks, threads, sink, (cudaStream_t)cuda_stream));
  return GBK_OK;
}

extern "C" int gbk_probe_umma(int iters, int blocks, float* check, double* flops_per_launch, void* cuda_stream) {
  g_err[0] = 0;
  if (iters < 1 || blocks < 1 || !check) return fail(GBK_ERR_ARG, "bad probe arguments");
  if (flops_per_launch)
    *flops_per_launch = (double)blocks * iters * (15.0 * 3.0 * 5.0) * ((128.0 + 64.0) * 64.0 * 16.0 * 2.0);
  GBK_CUDA(launch_probe_umma(iters, blocks, check, (cudaStream_t)cuda_stream));
  return GBK_OK;
}
