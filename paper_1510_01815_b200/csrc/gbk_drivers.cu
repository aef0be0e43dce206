// Host drivers of libgbk: nested grids, Levenberg-Marquardt and nested sampling
// written as callers of the batched hot path.  They use only the public calls of include/gbk.h
// (gbk_get_info, gbk_eval_batch) plus three small device reductions of their own (row building,
// argmin, J^T J), so an optimiser iteration moves a few hundred bytes across PCIe instead of the
// residual maps the paper copies back every iteration.
#include <math.h>
#include <stdint.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <mutex>
#include <new>
#include <vector>

#include "gbk_internal.h"

using namespace gbk;

namespace {

#define DRV_CUDA(expr)                                                                      \
  do {                                                                                      \
    cudaError_t e_ = (expr);                                                                \
    if (e_ != cudaSuccess)                                                                  \
      return fail(e_ == cudaErrorMemoryAllocation ? GBK_ERR_ALLOC : GBK_ERR_CUDA, "%s: %s", \
                  #expr, cudaGetErrorString(e_));                                           \
  } while (0)
#define DRV_TRY(expr)            \
  do {                           \
    if (int rc_ = (expr)) return rc_; \
  } while (0)

// Workspace of the drivers: ONE device block and ONE pinned host block per device, kept across calls
// (cudaMallocHost alone costs ~0.1 ms per buffer, more than a small fit) and carved into typed
// buffers by Buf::alloc.  The drivers block until their fit is done and hold the lock meanwhile.
struct Workspace {
  int device = -1;
  char* d = nullptr;
  char* h = nullptr;
  size_t d_cap = 0, h_cap = 0, d_used = 0, h_used = 0;
};
std::mutex g_ws_mu;
std::vector<Workspace*> g_ws;

Workspace* workspace_for(int device) {
  for (Workspace* w : g_ws)
    if (w->device == device) return w;
  Workspace* w = new (std::nothrow) Workspace;
  if (w) w->device = device, g_ws.push_back(w);
  return w;
}

// Sizes are requested first (plan = true: only adds up), then the blocks are grown if needed, then
// the same sequence of alloc calls hands out the pointers.
struct Arena {
  Workspace* ws;
  bool plan = true;
  size_t d_need = 0, h_need = 0;
  explicit Arena(Workspace* w) : ws(w) {}
  static size_t up(size_t n) { return (n + 255) & ~size_t(255); }
  cudaError_t commit() {
    cudaError_t e = cudaSuccess;
    if (d_need > ws->d_cap) {
      cudaFree(ws->d);
      ws->d = nullptr, ws->d_cap = 0;
      e = cudaMalloc(&ws->d, d_need);
      if (e != cudaSuccess) return e;
      ws->d_cap = d_need;
    }
    if (h_need > ws->h_cap) {
      cudaFreeHost(ws->h);
      ws->h = nullptr, ws->h_cap = 0;
      e = cudaMallocHost(&ws->h, h_need);
      if (e != cudaSuccess) return e;
      ws->h_cap = h_need;
    }
    ws->d_used = ws->h_used = 0;
    plan = false;
    return e;
  }
};

template <typename T>
struct Buf {
  T* d = nullptr;
  T* h = nullptr;
  size_t n = 0;
  void alloc(Arena& ar, size_t count, bool host = true, bool dev = true) {
    n = count;
    const size_t bytes = Arena::up(sizeof(T) * std::max<size_t>(count, 1));
    if (ar.plan) {
      if (dev) ar.d_need += bytes;
      if (host) ar.h_need += bytes;
      return;
    }
    if (dev) d = reinterpret_cast<T*>(ar.ws->d + ar.ws->d_used), ar.ws->d_used += bytes;
    if (host) h = reinterpret_cast<T*>(ar.ws->h + ar.ws->h_used), ar.ws->h_used += bytes;
  }
  cudaError_t to_device(size_t count, cudaStream_t st) {
    return cudaMemcpyAsync(d, h, sizeof(T) * count, cudaMemcpyHostToDevice, st);
  }
  cudaError_t to_host(size_t count, cudaStream_t st) {
    return cudaMemcpyAsync(h, d, sizeof(T) * count, cudaMemcpyDeviceToHost, st);
  }
};

struct Clock {
  std::chrono::steady_clock::time_point t0 = std::chrono::steady_clock::now();
  float ms() const {
    return std::chrono::duration<float, std::milli>(std::chrono::steady_clock::now() - t0).count();
  }
};

// One batch through the strategy the problem is set to (gbk_set_strategy).  `resid` is
// [K][2][ny][nx] for the cube strategy and [K][ny][nx] for the velocity-field strategy.
int eval_rows(gbk_problem* p, const gbk_problem_info& info, const float* rows, const int32_t* gal,
              int64_t K, float* chi2, float* resid, void* stream) {
  if (info.strategy == GBK_STRATEGY_VFIELD)
    return gbk_eval_vfield_batch(p, rows, gal, K, chi2, nullptr, resid, stream);
  return gbk_eval_batch(p, rows, gal, K, chi2, nullptr, nullptr, nullptr, resid, stream);
}

bool finite_row(const float* r, int S) {
  for (int j = 0; j < S; ++j)
    if (!isfinite(r[j])) return false;
  return true;
}

int check_box(int n, const int32_t* idx, const float* lo, const float* hi, int S) {
  if (n < 1 || n > S || !idx || !lo || !hi) return fail(GBK_ERR_ARG, "bad parameter box");
  for (int a = 0; a < n; ++a) {
    if (idx[a] < 0 || idx[a] >= S) return fail(GBK_ERR_ARG, "parameter index %d out of range", idx[a]);
    if (!isfinite(lo[a]) || !isfinite(hi[a]) || !(hi[a] > lo[a]))
      return fail(GBK_ERR_ARG, "box of parameter %d is empty or not finite", idx[a]);
    for (int b = 0; b < a; ++b)
      if (idx[b] == idx[a]) return fail(GBK_ERR_ARG, "parameter %d listed twice", idx[a]);
  }
  return GBK_OK;
}

// ------------------------------------------------------------------------- nested grids ----
constexpr int kNgMaxAxes = 6, kNgMaxNodes = 32;

struct NgAxes {
  int n_axes, S;              // S: floats per row
  int nodes[kNgMaxAxes];
  int param[kNgMaxAxes];
  float value[kNgMaxAxes][kNgMaxNodes];
  float base[GBK_P_MAX];
};

// Row r of the level: flat index with axis 0 slowest.
__global__ void ng_rows_kernel(const __grid_constant__ NgAxes ax, int n_rows, float* __restrict__ rows) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_rows) return;
  float row[GBK_P_MAX];
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j) row[j] = ax.base[j];
  int rem = r;
  for (int a = ax.n_axes - 1; a >= 0; --a) {
    const int j = rem % ax.nodes[a];
    rem /= ax.nodes[a];
    row[ax.param[a]] = ax.value[a][j];
  }
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j)
    if (j < ax.S) rows[(size_t)r * ax.S + j] = row[j];
}

// Smallest chi^2 and its lowest index (NaN never wins; +INF only if everything is +INF).
__global__ void argmin_kernel(const float* __restrict__ chi2, int n, int* __restrict__ out_idx,
                              float* __restrict__ out_val) {
  __shared__ float sv[1024];
  __shared__ int si[1024];
  float best = __int_as_float(0x7f800000);
  int bi = 0x7fffffff;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const float v = chi2[i];
    if (v < best || (v == best && i < bi)) best = v, bi = i;
  }
  sv[threadIdx.x] = best, si[threadIdx.x] = bi;
  __syncthreads();
  for (int s = blockDim.x >> 1; s > 0; s >>= 1) {
    if (threadIdx.x < s) {
      const float v = sv[threadIdx.x + s];
      const int i = si[threadIdx.x + s];
      if (v < sv[threadIdx.x] || (v == sv[threadIdx.x] && i < si[threadIdx.x]))
        sv[threadIdx.x] = v, si[threadIdx.x] = i;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) out_idx[0] = si[0] == 0x7fffffff ? 0 : si[0], out_val[0] = sv[0];
}

}  // namespace

extern "C" int gbk_fit_ng(gbk_problem* p, const float* base_row, int32_t gal, int32_t n_axes,
                          const int32_t* axis_param, const float* axis_lo, const float* axis_hi,
                          const int32_t* axis_nodes, const float* axis_accuracy, int32_t max_levels,
                          float* best_row, float* best_chi2, gbk_fit_stats* stats, void* cuda_stream) {
  clear_error();
  Clock clock;
  gbk_problem_info info;
  DRV_TRY(gbk_get_info(p, &info));
  if (!base_row || !best_row || !best_chi2 || !axis_nodes) return fail(GBK_ERR_ARG, "null argument");
  if (n_axes > kNgMaxAxes || max_levels < 1 || max_levels > 30)
    return fail(GBK_ERR_ARG, "need n_axes <= %d and 1 <= max_levels <= 30", kNgMaxAxes);
  DRV_TRY(check_box(n_axes, axis_param, axis_lo, axis_hi, info.row_stride));
  if (gal < 0 || gal >= info.n_gal) return fail(GBK_ERR_ARG, "gal out of range");
  double n_rows_d = 1.0;
  for (int a = 0; a < n_axes; ++a) {
    if (axis_nodes[a] < 2 || axis_nodes[a] > kNgMaxNodes)
      return fail(GBK_ERR_ARG, "need 2 <= axis_nodes <= %d", kNgMaxNodes);
    if (axis_accuracy && !(axis_accuracy[a] > 0.f)) return fail(GBK_ERR_ARG, "axis_accuracy must be > 0");
    n_rows_d *= axis_nodes[a];
  }
  if (n_rows_d > (double)(1 << 24)) return fail(GBK_ERR_ARG, "the grid exceeds 2^24 rows");
  const int n_rows = (int)n_rows_d;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(info.device);
  DRV_CUDA(guard.status);

  std::lock_guard<std::mutex> ws_lock(g_ws_mu);
  Workspace* ws = workspace_for(info.device);
  if (!ws) return fail(GBK_ERR_ALLOC, "out of host memory");
  Arena ar(ws);
  Buf<float> rows, chi2, best_v;
  Buf<int> best_i, gal_idx;
  for (int pass = 0; pass < 2; ++pass) {
    rows.alloc(ar, (size_t)n_rows * GBK_P_MAX, false);
    chi2.alloc(ar, n_rows, false);
    best_v.alloc(ar, 1);
    best_i.alloc(ar, 1);
    if (gal != 0) gal_idx.alloc(ar, n_rows);
    if (pass == 0) DRV_CUDA(ar.commit());
  }
  if (gal != 0) {
    std::fill(gal_idx.h, gal_idx.h + n_rows, gal);
    DRV_CUDA(gal_idx.to_device(n_rows, st));
  }
  DRV_TRY(gbk_reserve(p, n_rows, cuda_stream));

  NgAxes ax;
  memset(&ax, 0, sizeof(ax));
  const int S = info.row_stride;
  ax.n_axes = n_axes, ax.S = S;
  memcpy(ax.base, base_row, sizeof(float) * S);
  double centre[kNgMaxAxes];
  for (int a = 0; a < n_axes; ++a) {
    ax.param[a] = axis_param[a], ax.nodes[a] = axis_nodes[a];
    centre[a] = 0.5 * ((double)axis_lo[a] + (double)axis_hi[a]);
  }
  gbk_fit_stats fs{};
  bool reached = false;
  for (int level = 0; level < max_levels && !reached; ++level) {
    reached = axis_accuracy != nullptr;
    for (int a = 0; a < n_axes; ++a) {
      const int nodes = axis_nodes[a];
      const double lo = axis_lo[a], hi = axis_hi[a];
      const double h = (hi - lo) / ((double)nodes * (double)(1u << level));
      if (axis_accuracy && h > (double)axis_accuracy[a]) reached = false;   // this level is not the last
      const bool wraps = axis_param[a] == 2 && hi - lo >= 360.0;
      double first = centre[a] - 0.5 * (nodes - 1) * h;
      if (!wraps) {   // shift the whole axis back inside the box
        const double last = first + (nodes - 1) * h;
        first += std::max(0.0, lo - first) - std::max(0.0, last - hi);
      }
      for (int j = 0; j < nodes; ++j) {
        double v = first + j * h;
        if (wraps) v = lo + fmod(fmod(v - lo, 360.0) + 360.0, 360.0);
        ax.value[a][j] = (float)v;
      }
    }
    ng_rows_kernel<<<(n_rows + 255) / 256, 256, 0, st>>>(ax, n_rows, rows.d);
    DRV_CUDA(cudaGetLastError());
    DRV_TRY(eval_rows(p, info, rows.d, gal != 0 ? gal_idx.d : nullptr, n_rows, chi2.d, nullptr, cuda_stream));
    argmin_kernel<<<1, 1024, 0, st>>>(chi2.d, n_rows, best_i.d, best_v.d);
    DRV_CUDA(cudaGetLastError());
    DRV_CUDA(best_i.to_host(1, st));
    DRV_CUDA(best_v.to_host(1, st));
    DRV_CUDA(cudaStreamSynchronize(st));
    int rem = best_i.h[0];
    for (int a = n_axes - 1; a >= 0; --a) {
      centre[a] = ax.value[a][rem % axis_nodes[a]];
      rem /= axis_nodes[a];
    }
    fs.evals += n_rows, fs.launches += 1, fs.iterations += 1;
  }
  memcpy(best_row, base_row, sizeof(float) * S);
  for (int a = 0; a < n_axes; ++a) best_row[axis_param[a]] = (float)centre[a];
  *best_chi2 = best_v.h[0];
  // converged: the accuracy thresholds were reached (or none were asked for) with a finite chi^2
  fs.converged = (isfinite(best_v.h[0]) && (reached || !axis_accuracy)) ? 1 : 0;
  fs.ms_total = clock.ms();
  if (stats) *stats = fs;
  return GBK_OK;
}

// ------------------------------------------------------------------ Levenberg-Marquardt ----
// Device-resident (PAPER.md:758 names a GPU-only LM as future work):
// the state of every fit (row, chi^2, damping factor, status) lives in device memory, and one
// iteration is six launches on the caller's stream with no host round trip between them --
//   lm_jacobian_rows   base + n one-sided difference rows per listed fit
//   gbk_eval_batch     their chi^2 and weighted residuals
//   lm_normal_kernel   J^T J, J^T r in FP64
//   lm_trial_rows      the damped 7x7 Cholesky solves (four damping factors per fit), trial rows
//   gbk_eval_batch     chi^2 of the trial rows
//   lm_update          accept / reject, damping update, stopping rules, count of fits still active
// The host reads back ONE integer (fits still active) every kLmReadback iterations, and compacts the
// list of fits when it has shrunk; fits that stop in between cost an out-of-domain row per slot (a
// thread block that exits at once).
namespace {

enum { LM_ACTIVE = 0, LM_CONVERGED = 1, LM_STALLED = 2, LM_FAILED = 3, LM_MAXITER = 4, LM_BAD_START = 5 };
constexpr int kLmTrials = 4;
constexpr int kLmReadback = 4;
__constant__ double kLmFactor[kLmTrials] = {0.1, 1.0, 10.0, 100.0};

struct LmSetup {
  int n, M, n_terms, max_iter, S;   // S: floats per row
  int free_param[GBK_P_MAX];
  float lo[GBK_P_MAX], hi[GBK_P_MAX];
  float rel_step, ftol;
};

struct LmState {         // device arrays, one entry per fit
  float* row;            // [n_fits][S]
  double* chi2;          // chi^2 of `row` (+inf until evaluated)
  double* lambda;
  int* iters;
  int* status;
  int* gal;
  float* hstep;          // [n_fits][n] finite-difference steps actually taken (FP32)
  unsigned long long* evals;   // [1] rows evaluated for fits that were active
};

// One thread per (slot, r): row r of the slot's Jacobian batch.  r = 0 is the base row.
__global__ void lm_jacobian_rows(const __grid_constant__ LmSetup su, const LmState stt, const int* __restrict__ list,
                                 int n_list, float* __restrict__ rows, int* __restrict__ gidx) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int slot = t / (su.n + 1), r = t - slot * (su.n + 1);
  if (slot >= n_list) return;
  const int f = list[slot];
  float row[GBK_P_MAX];
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j) row[j] = j < su.S ? stt.row[(size_t)f * su.S + j] : 0.0f;
  gidx[t] = stt.gal[f];
  if (stt.status[f] != LM_ACTIVE) {
    row[0] = __int_as_float(0x7fc00000);          // finished: an out-of-domain row costs next to nothing
  } else if (r > 0) {
    const int a = r - 1, j = su.free_param[a];
    float h = su.rel_step * (su.hi[a] - su.lo[a]);
    float moved = row[j] + h;
    for (int k = 0; k < 30 && moved == row[j]; ++k) h *= 2.0f, moved = row[j] + h;   // a step below one ulp
    if (moved > su.hi[a]) h = -h, moved = row[j] + h;                                  // backward at the wall
    stt.hstep[(size_t)f * su.n + a] = moved - row[j];   // the step actually taken in FP32 (0: see lm_trial_rows)
    row[j] = moved;
  } else {
    atomicAdd(stt.evals, (unsigned long long)(su.n + 1));
  }
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j)
    if (j < su.S) rows[(size_t)t * su.S + j] = row[j];
}

// One block per (term, slot).  Terms: n(n+1)/2 entries of J^T J (upper triangle, row-major),
// n entries of J^T r, and r.r; J_a = (r_a - r_0) / h_a from the one-sided difference rows.
// resid: [n_list][n+1][M]; out: [n_list][n_terms] (double).
__global__ void lm_normal_kernel(const float* __restrict__ resid, const LmState stt, const int* __restrict__ list,
                                 int n, int M, double* __restrict__ out) {
  const int n_tri = n * (n + 1) / 2, n_terms = n_tri + n + 1;
  const int term = blockIdx.x, slot = blockIdx.y;
  const int f = list[slot];
  if (stt.status[f] != LM_ACTIVE) return;
  int a = -1, b = -1;   // a = b = -1: r.r;  b = -1: (J^T r)_a
  if (term < n_tri) {
    int t = term;
    a = 0;
    while (t >= n - a) t -= n - a, ++a;
    b = a + t;
  } else if (term < n_tri + n) {
    a = term - n_tri;
  }
  const float* r0 = resid + (size_t)slot * (n + 1) * M;
  const float* ra = a >= 0 ? r0 + (size_t)(a + 1) * M : r0;
  const float* rb = b >= 0 ? r0 + (size_t)(b + 1) * M : r0;
  double acc = 0.0;
  for (int i = threadIdx.x; i < M; i += blockDim.x) {
    const double z = r0[i];
    const double x = a >= 0 ? (double)ra[i] - z : z;
    const double y = b >= 0 ? (double)rb[i] - z : z;
    acc += x * y;
  }
  __shared__ double red[256];
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int s = blockDim.x >> 1; s > 0; s >>= 1) {
    if (threadIdx.x < s) red[threadIdx.x] += red[threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double v = red[0];
    if (a >= 0) v /= (double)stt.hstep[(size_t)f * n + a];
    if (b >= 0) v /= (double)stt.hstep[(size_t)f * n + b];
    out[(size_t)slot * n_terms + term] = v;
  }
}

// Solves (A + lambda diag(A)) x = -g by Cholesky (A symmetric, upper triangle packed row-major).
__device__ bool solve_damped(int n, const double* tri, const double* g, double lambda, double* x) {
  double L[GBK_P_MAX][GBK_P_MAX];
  int t = 0;
  for (int a = 0; a < n; ++a)
    for (int b = a; b < n; ++b, ++t) L[a][b] = L[b][a] = tri[t];
  for (int a = 0; a < n; ++a) {
    if (!(L[a][a] > 0.0) || !isfinite(L[a][a])) return false;
    L[a][a] *= 1.0 + lambda;
  }
  for (int j = 0; j < n; ++j) {
    double d = L[j][j];
    for (int k = 0; k < j; ++k) d -= L[j][k] * L[j][k];
    if (!(d > 0.0) || !isfinite(d)) return false;
    L[j][j] = sqrt(d);
    for (int i = j + 1; i < n; ++i) {
      double s = L[i][j];
      for (int k = 0; k < j; ++k) s -= L[i][k] * L[j][k];
      L[i][j] = s / L[j][j];
    }
  }
  double y[GBK_P_MAX];
  for (int i = 0; i < n; ++i) {
    double s = -g[i];
    for (int k = 0; k < i; ++k) s -= L[i][k] * y[k];
    y[i] = s / L[i][i];
  }
  for (int i = n - 1; i >= 0; --i) {
    double s = y[i];
    for (int k = i + 1; k < n; ++k) s -= L[k][i] * x[k];
    x[i] = s / L[i][i];
    if (!isfinite(x[i])) return false;
  }
  return true;
}

// One thread per (slot, trial): books the base chi^2 of the Jacobian batch, applies the stopping
// rules that need no trial (bad start, iteration limit, unusable Jacobian), and writes the trial row
// of damping factor lambda x kLmFactor[trial].  jac_chi2: [n_list][n+1]; normal: [n_list][n_terms].
__global__ void lm_trial_rows(const __grid_constant__ LmSetup su, const LmState stt, const int* __restrict__ list,
                              int n_list, const float* __restrict__ jac_chi2, const double* __restrict__ normal,
                              float* __restrict__ rows, int* __restrict__ gidx) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  const int slot = t / kLmTrials, trial = t - slot * kLmTrials;
  if (slot >= n_list) return;
  const int f = list[slot], n = su.n;
  float row[GBK_P_MAX];
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j) row[j] = j < su.S ? stt.row[(size_t)f * su.S + j] : 0.0f;
  gidx[t] = stt.gal[f];
  int status = stt.status[f];
  if (status == LM_ACTIVE) {
    const float* c = jac_chi2 + (size_t)slot * (n + 1);
    const double base = c[0];
    bool jac_ok = true;           // every difference row in domain and every step non-zero
    for (int a = 0; a < n; ++a) jac_ok = jac_ok && isfinite(c[a + 1]) && stt.hstep[(size_t)f * n + a] != 0.0f;
    if (!isfinite(base)) status = stt.iters[f] == 0 ? LM_BAD_START : LM_FAILED;
    else if (stt.iters[f] >= su.max_iter) status = LM_MAXITER;
    else if (!jac_ok) status = LM_FAILED;
    const double* nm = normal + (size_t)slot * su.n_terms;
    double dx[GBK_P_MAX];
    bool solved = false;
    if (status == LM_ACTIVE) {
      solved = solve_damped(n, nm, nm + n * (n + 1) / 2, stt.lambda[f] * kLmFactor[trial], dx);
      if (solved)
        for (int a = 0; a < n; ++a) {
          const int j = su.free_param[a];
          row[j] = (float)fmin((double)su.hi[a], fmax((double)su.lo[a], (double)row[j] + dx[a]));
        }
    }
    if (trial == 0) {             // one thread per slot writes the state
      if (isfinite(base) || stt.iters[f] == 0) stt.chi2[f] = base;
      if (status == LM_ACTIVE) atomicAdd(stt.evals, (unsigned long long)kLmTrials);
      else stt.status[f] = status;
    }
    if (status == LM_ACTIVE && !solved) row[0] = __int_as_float(0x7fc00000);   // this factor gives no step
  }
  if (status != LM_ACTIVE) row[0] = __int_as_float(0x7fc00000);
#pragma unroll
  for (int j = 0; j < GBK_P_MAX; ++j)
    if (j < su.S) rows[(size_t)t * su.S + j] = row[j];
}

// One thread per slot: best of the four trials, accept / reject, damping update, stopping rules.
__global__ void lm_update(const __grid_constant__ LmSetup su, const LmState stt, const int* __restrict__ list,
                          int n_list, const float* __restrict__ trial_rows, const float* __restrict__ trial_chi2,
                          int* __restrict__ n_active) {
  const int slot = blockIdx.x * blockDim.x + threadIdx.x;
  if (slot >= n_list) return;
  const int f = list[slot];
  if (stt.status[f] != LM_ACTIVE) return;
  int best = -1, n_finite = 0;
  double best_chi = stt.chi2[f];
  for (int t = 0; t < kLmTrials; ++t) {
    const double c = trial_chi2[(size_t)slot * kLmTrials + t];
    n_finite += isfinite(c) ? 1 : 0;
    if (c < best_chi) best_chi = c, best = t;
  }
  stt.iters[f] += 1;
  int status = LM_ACTIVE;
  if (best >= 0) {
    const double rel = (stt.chi2[f] - best_chi) / stt.chi2[f];
    for (int j = 0; j < su.S; ++j)
      stt.row[(size_t)f * su.S + j] = trial_rows[((size_t)slot * kLmTrials + best) * su.S + j];
    stt.lambda[f] = fmax(1e-9, stt.lambda[f] * kLmFactor[best] * 0.3);
    stt.chi2[f] = best_chi;
    if (rel < (double)su.ftol) status = LM_CONVERGED;
  } else {
    stt.lambda[f] *= 1e4;
    // no downhill step up to the largest damping: a stationary point of chi^2 as far as LM can tell --
    // unless no trial was ever evaluated (singular or non-finite normal equations): that is a failure
    if (stt.lambda[f] > 1e10) status = n_finite > 0 ? LM_STALLED : LM_FAILED;
  }
  if (status != LM_ACTIVE) stt.status[f] = status;
  else atomicAdd(n_active, 1);
}

// Stable compaction of the list of fits to those still active (one block; lists are short).
__global__ void lm_compact(const LmState stt, const int* __restrict__ list, int n_list, int* __restrict__ out) {
  __shared__ int base;
  __shared__ int warp_tot[32];
  if (threadIdx.x == 0) base = 0;
  __syncthreads();
  for (int i0 = 0; i0 < n_list; i0 += blockDim.x) {
    const int i = i0 + threadIdx.x;
    const int f = i < n_list ? list[i] : -1;
    const bool keep = f >= 0 && stt.status[f] == LM_ACTIVE;
    const unsigned m = __ballot_sync(0xffffffffu, keep);
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (lane == 0) warp_tot[w] = __popc(m);
    __syncthreads();
    int off = base;
    for (int k = 0; k < w; ++k) off += warp_tot[k];
    if (keep) out[off + __popc(m & ((1u << lane) - 1u))] = f;
    __syncthreads();
    if (threadIdx.x == 0) {
      int tot = 0;
      for (int k = 0; k < (int)(blockDim.x >> 5); ++k) tot += warp_tot[k];
      base += tot;
    }
    __syncthreads();
  }
}

}  // namespace

extern "C" int gbk_fit_lm(gbk_problem* p, int32_t n_fits, const float* start_rows, const int32_t* gal,
                          int32_t n_free, const int32_t* free_param, const float* lo, const float* hi,
                          float rel_step, int32_t max_iter, float ftol, float* fit_rows,
                          float* fit_chi2, int32_t* fit_iters, gbk_fit_stats* stats,
                          void* cuda_stream) {
  clear_error();
  Clock clock;
  gbk_problem_info info;
  DRV_TRY(gbk_get_info(p, &info));
  if (n_fits < 0 || (n_fits > 0 && (!start_rows || !fit_rows || !fit_chi2)))
    return fail(GBK_ERR_ARG, "null argument");
  if (!(rel_step > 0.f) || !isfinite(rel_step) || max_iter < 0 || !(ftol >= 0.f))
    return fail(GBK_ERR_ARG, "need rel_step > 0, max_iter >= 0, ftol >= 0");
  DRV_TRY(check_box(n_free, free_param, lo, hi, info.row_stride));
  for (int f = 0; f < n_fits; ++f)
    if (gal && (gal[f] < 0 || gal[f] >= info.n_gal)) return fail(GBK_ERR_ARG, "gal[%d] out of range", f);
  gbk_fit_stats fs{};
  if (n_fits == 0) {
    if (stats) *stats = fs;
    return GBK_OK;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(info.device);
  DRV_CUDA(guard.status);
  LmSetup su{};
  su.n = n_free, su.M = (info.strategy == GBK_STRATEGY_VFIELD ? 1 : 2) * info.nx * info.ny;
  su.n_terms = su.n * (su.n + 1) / 2 + su.n + 1, su.max_iter = max_iter;
  su.rel_step = rel_step, su.ftol = ftol, su.S = info.row_stride;
  const int S = su.S;
  for (int a = 0; a < su.n; ++a) su.free_param[a] = free_param[a], su.lo[a] = lo[a], su.hi[a] = hi[a];
  const int n = su.n;
  // fits per chunk: the residual buffer of a chunk stays below 1 GiB
  const size_t resid_per_fit = sizeof(float) * (size_t)(n + 1) * su.M;
  const int chunk = (int)std::max<size_t>(1, std::min<size_t>(n_fits, (size_t(1) << 30) / resid_per_fit));
  const int rows_per_fit = std::max(n + 1, kLmTrials);
  std::lock_guard<std::mutex> ws_lock(g_ws_mu);
  Workspace* ws = workspace_for(info.device);
  if (!ws) return fail(GBK_ERR_ALLOC, "out of host memory");
  Arena ar(ws);
  Buf<float> rows, chi2, resid, state_row, hstep;
  Buf<int> gidx, list_a, list_b, iters, status, galb, n_active;
  Buf<double> normal, state_chi2, lambda;
  Buf<unsigned long long> evals;
  for (int pass = 0; pass < 2; ++pass) {
    rows.alloc(ar, (size_t)chunk * rows_per_fit * S, false);
    chi2.alloc(ar, (size_t)chunk * rows_per_fit, false);
    gidx.alloc(ar, (size_t)chunk * rows_per_fit, false);
    resid.alloc(ar, (size_t)chunk * (n + 1) * su.M, false);
    normal.alloc(ar, (size_t)chunk * su.n_terms, false);
    hstep.alloc(ar, (size_t)n_fits * n, false);
    state_row.alloc(ar, (size_t)n_fits * S);
    state_chi2.alloc(ar, n_fits);
    lambda.alloc(ar, n_fits);
    iters.alloc(ar, n_fits);
    status.alloc(ar, n_fits);
    galb.alloc(ar, n_fits);
    list_a.alloc(ar, chunk);
    list_b.alloc(ar, chunk, false);
    n_active.alloc(ar, kLmReadback + 1);
    evals.alloc(ar, 1);
    if (pass == 0) DRV_CUDA(ar.commit());
  }
  for (int f = 0; f < n_fits; ++f) {
    float* row = state_row.h + (size_t)f * S;
    memcpy(row, start_rows + (size_t)f * S, sizeof(float) * S);
    for (int a = 0; a < n; ++a)   // start inside the box
      row[free_param[a]] = std::min(hi[a], std::max(lo[a], row[free_param[a]]));
    state_chi2.h[f] = INFINITY, lambda.h[f] = 1e-3, iters.h[f] = 0;
    status.h[f] = finite_row(row, S) ? LM_ACTIVE : LM_BAD_START;
    galb.h[f] = gal ? gal[f] : 0;
  }
  evals.h[0] = 0;
  DRV_CUDA(state_row.to_device((size_t)n_fits * S, st));
  DRV_CUDA(state_chi2.to_device(n_fits, st));
  DRV_CUDA(lambda.to_device(n_fits, st));
  DRV_CUDA(iters.to_device(n_fits, st));
  DRV_CUDA(status.to_device(n_fits, st));
  DRV_CUDA(galb.to_device(n_fits, st));
  DRV_CUDA(evals.to_device(1, st));
  DRV_TRY(gbk_reserve(p, (int64_t)chunk * rows_per_fit, cuda_stream));
  const LmState stt{state_row.d, state_chi2.d, lambda.d, iters.d, status.d, galb.d, hstep.d, evals.d};

  for (int c0 = 0; c0 < n_fits; c0 += chunk) {
    const int c1 = std::min(n_fits, c0 + chunk);
    int n_list = 0;
    for (int f = c0; f < c1; ++f)
      if (status.h[f] == LM_ACTIVE) list_a.h[n_list++] = f;
    if (n_list == 0) continue;
    DRV_CUDA(list_a.to_device(n_list, st));
    int* list = list_a.d;
    int* spare = list_b.d;
    // every fit stops after at most max_iter + 1 iterations (the last one only books chi^2)
    for (int it = 0; n_list > 0 && it <= max_iter + kLmReadback; it += kLmReadback) {
      DRV_CUDA(cudaMemsetAsync(n_active.d, 0, sizeof(int) * (kLmReadback + 1), st));
      for (int sub = 0; sub < kLmReadback; ++sub) {
        const int kj = n_list * (n + 1), kt = n_list * kLmTrials;
        lm_jacobian_rows<<<(kj + 127) / 128, 128, 0, st>>>(su, stt, list, n_list, rows.d, gidx.d);
        DRV_CUDA(cudaGetLastError());
        DRV_TRY(eval_rows(p, info, rows.d, gidx.d, kj, chi2.d, resid.d, cuda_stream));
        lm_normal_kernel<<<dim3(su.n_terms, n_list), 256, 0, st>>>(resid.d, stt, list, n, su.M, normal.d);
        DRV_CUDA(cudaGetLastError());
        lm_trial_rows<<<(kt + 127) / 128, 128, 0, st>>>(su, stt, list, n_list, chi2.d, normal.d, rows.d, gidx.d);
        DRV_CUDA(cudaGetLastError());
        // the Jacobian chi^2 are consumed by lm_trial_rows before this launch overwrites them (stream order)
        DRV_TRY(eval_rows(p, info, rows.d, gidx.d, kt, chi2.d, nullptr, cuda_stream));
        lm_update<<<(n_list + 127) / 128, 128, 0, st>>>(su, stt, list, n_list, rows.d, chi2.d, n_active.d + sub);
        DRV_CUDA(cudaGetLastError());
        fs.launches += 2;
      }
      DRV_CUDA(n_active.to_host(kLmReadback, st));
      DRV_CUDA(cudaStreamSynchronize(st));
      const int left = n_active.h[kLmReadback - 1];
      if (left == 0) break;
      if (left < n_list - n_list / 4 || left <= 64) {     // the list has shrunk: drop the finished fits
        lm_compact<<<1, 1024, 0, st>>>(stt, list, n_list, spare);
        DRV_CUDA(cudaGetLastError());
        std::swap(list, spare);
        n_list = left;
      }
    }
  }
  DRV_CUDA(state_row.to_host((size_t)n_fits * S, st));
  DRV_CUDA(state_chi2.to_host(n_fits, st));
  DRV_CUDA(iters.to_host(n_fits, st));
  DRV_CUDA(status.to_host(n_fits, st));
  DRV_CUDA(evals.to_host(1, st));
  DRV_CUDA(cudaStreamSynchronize(st));
  for (int f = 0; f < n_fits; ++f) {
    memcpy(fit_rows + (size_t)f * S, state_row.h + (size_t)f * S, sizeof(float) * S);
    fit_chi2[f] = (float)state_chi2.h[f];
    if (fit_iters) fit_iters[f] = iters.h[f];
    fs.iterations = std::max(fs.iterations, iters.h[f]);
    fs.converged += (status.h[f] == LM_CONVERGED || status.h[f] == LM_STALLED) ? 1 : 0;
    fs.failed += (status.h[f] == LM_FAILED || status.h[f] == LM_BAD_START) ? 1 : 0;
  }
  fs.evals = (int64_t)evals.h[0];
  fs.ms_total = clock.ms();
  if (stats) *stats = fs;
  return GBK_OK;
}

// --------------------------------------------------------------------- nested sampling ----
namespace {

struct Xoshiro {   // xoshiro256** seeded by splitmix64 (public-domain algorithm, re-stated)
  uint64_t s[4];
  explicit Xoshiro(uint64_t seed) {
    for (int i = 0; i < 4; ++i) {
      seed += 0x9E3779B97F4A7C15ull;
      uint64_t z = seed;
      z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
      z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
      s[i] = z ^ (z >> 31);
    }
  }
  static uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
  uint64_t next() {
    const uint64_t r = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
    s[2] ^= s[0], s[3] ^= s[1], s[1] ^= s[2], s[0] ^= s[3], s[2] ^= t, s[3] = rotl(s[3], 45);
    return r;
  }
  double uniform() { return (double)(next() >> 11) * (1.0 / 9007199254740992.0); }
};

double log_add(double a, double b) {
  if (a == -INFINITY) return b;
  if (b == -INFINITY) return a;
  const double m = std::max(a, b);
  return m + log(exp(a - m) + exp(b - m));
}

}  // namespace

extern "C" int gbk_fit_ns(gbk_problem* p, const float* base_row, int32_t gal, int32_t n_free,
                          const int32_t* free_param, const float* lo, const float* hi, int32_t n_live,
                          int32_t batch, int32_t max_batches, float enlarge, float tol, uint64_t seed,
                          float* best_row, float* best_chi2, float* mean_row, double* log_evidence,
                          gbk_fit_stats* stats, void* cuda_stream) {
  clear_error();
  Clock clock;
  gbk_problem_info info;
  DRV_TRY(gbk_get_info(p, &info));
  if (!base_row || !best_row || !best_chi2) return fail(GBK_ERR_ARG, "null argument");
  if (n_live < 2 || batch < 1 || max_batches < 0 || !(enlarge >= 0.f) || !(tol > 0.f))
    return fail(GBK_ERR_ARG, "need n_live >= 2, batch >= 1, max_batches >= 0, enlarge >= 0, tol > 0");
  DRV_TRY(check_box(n_free, free_param, lo, hi, info.row_stride));
  if (gal < 0 || gal >= info.n_gal) return fail(GBK_ERR_ARG, "gal out of range");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard guard(info.device);
  DRV_CUDA(guard.status);
  const int n = n_free, cap = std::max(n_live, batch), S = info.row_stride;
  std::lock_guard<std::mutex> ws_lock(g_ws_mu);
  Workspace* ws = workspace_for(info.device);
  if (!ws) return fail(GBK_ERR_ALLOC, "out of host memory");
  Arena ar(ws);
  Buf<float> rows, chi2;
  Buf<int> gidx;
  for (int pass = 0; pass < 2; ++pass) {
    rows.alloc(ar, (size_t)cap * S);
    chi2.alloc(ar, cap);
    gidx.alloc(ar, cap);
    if (pass == 0) DRV_CUDA(ar.commit());
  }
  std::fill(gidx.h, gidx.h + cap, gal);
  DRV_CUDA(gidx.to_device(cap, st));
  Xoshiro rng(seed);
  gbk_fit_stats fs{};

  auto evaluate = [&](int k) -> int {   // rows.h[0..k) -> chi2.h[0..k)
    DRV_CUDA(rows.to_device((size_t)k * S, st));
    DRV_TRY(eval_rows(p, info, rows.d, gidx.d, k, chi2.d, nullptr, cuda_stream));
    DRV_CUDA(chi2.to_host(k, st));
    DRV_CUDA(cudaStreamSynchronize(st));
    fs.evals += k, fs.launches += 1;
    return GBK_OK;
  };
  auto draw = [&](float* row, const double* blo, const double* bhi) {
    memcpy(row, base_row, sizeof(float) * S);
    for (int a = 0; a < n; ++a) row[free_param[a]] = (float)(blo[a] + (bhi[a] - blo[a]) * rng.uniform());
  };

  // live points from the whole prior box
  std::vector<double> plo(lo, lo + n), phi(hi, hi + n);
  std::vector<float> live((size_t)n_live * S);
  std::vector<double> live_lnl(n_live);
  for (int i = 0; i < n_live; ++i) draw(rows.h + (size_t)i * S, plo.data(), phi.data());
  DRV_TRY(evaluate(n_live));
  memcpy(live.data(), rows.h, sizeof(float) * live.size());
  for (int i = 0; i < n_live; ++i) live_lnl[i] = isfinite(chi2.h[i]) ? -0.5 * (double)chi2.h[i] : -INFINITY;

  // dead points: ln L, ln w and the free parameters, for the evidence and the posterior mean
  std::vector<double> dead_lnl, dead_lnw, dead_x;
  double lnz = -INFINITY;
  long long n_dead = 0;
  bool done = false;
  std::vector<double> blo(n), bhi(n);
  for (int b = 0; b < max_batches && !done; ++b) {
    // Sampling region: the ellipsoid of the live points (their mean and covariance, scaled to hold
    // every live point, then enlarged), intersected with the bounding box of the live points
    // (enlarged likewise) and the prior box -- single-ellipsoid nested sampling (the scheme
    // MultiNest generalises).  Falls back to the box alone while the covariance
    // is singular.  Parameters are scaled to the prior box so the covariance is well conditioned.
    for (int a = 0; a < n; ++a) {
      double mn = INFINITY, mx = -INFINITY;
      for (int i = 0; i < n_live; ++i) {
        const double v = live[(size_t)i * S + free_param[a]];
        mn = std::min(mn, v), mx = std::max(mx, v);
      }
      const double pad = 0.5 * enlarge * (mx - mn) + 1e-6 * (phi[a] - plo[a]);
      blo[a] = std::max(plo[a], mn - pad), bhi[a] = std::min(phi[a], mx + pad);
    }
    double mu[GBK_P_MAX], Lc[GBK_P_MAX][GBK_P_MAX], scale = 0.0;
    bool ellipsoid = n_live > 2 * n;
    if (ellipsoid) {
      double cov[GBK_P_MAX][GBK_P_MAX] = {};
      for (int a = 0; a < n; ++a) {
        mu[a] = 0.0;
        for (int i = 0; i < n_live; ++i)
          mu[a] += (live[(size_t)i * S + free_param[a]] - plo[a]) / (phi[a] - plo[a]);
        mu[a] /= n_live;
      }
      for (int i = 0; i < n_live; ++i) {
        double dlt[GBK_P_MAX];
        for (int a = 0; a < n; ++a)
          dlt[a] = (live[(size_t)i * S + free_param[a]] - plo[a]) / (phi[a] - plo[a]) - mu[a];
        for (int a = 0; a < n; ++a)
          for (int c = 0; c <= a; ++c) cov[a][c] += dlt[a] * dlt[c] / (n_live - 1);
      }
      for (int j = 0; j < n && ellipsoid; ++j) {            // Cholesky, lower triangle
        double d = cov[j][j];
        for (int q = 0; q < j; ++q) d -= Lc[j][q] * Lc[j][q];
        if (!(d > 1e-24)) {
          ellipsoid = false;
          break;
        }
        Lc[j][j] = sqrt(d);
        for (int i = j + 1; i < n; ++i) {
          double t = cov[i][j];
          for (int q = 0; q < j; ++q) t -= Lc[i][q] * Lc[j][q];
          Lc[i][j] = t / Lc[j][j];
        }
      }
      if (ellipsoid) {                                       // largest Mahalanobis distance of a live point
        for (int i = 0; i < n_live; ++i) {
          double y[GBK_P_MAX], d2 = 0.0;
          for (int a = 0; a < n; ++a) {
            double t = (live[(size_t)i * S + free_param[a]] - plo[a]) / (phi[a] - plo[a]) - mu[a];
            for (int q = 0; q < a; ++q) t -= Lc[a][q] * y[q];
            y[a] = t / Lc[a][a];
            d2 += y[a] * y[a];
          }
          scale = std::max(scale, d2);
        }
        scale = sqrt(scale) * (1.0 + enlarge);
      }
    }
    for (int i = 0; i < batch; ++i) {
      float* row = rows.h + (size_t)i * S;
      if (!ellipsoid) {
        draw(row, blo.data(), bhi.data());
        continue;
      }
      memcpy(row, base_row, sizeof(float) * S);
      for (int attempt = 0;; ++attempt) {
        // uniform in the unit n-ball: Gaussian direction, radius U^(1/n)
        double z[GBK_P_MAX], nrm = 0.0;
        for (int a = 0; a < n; a += 2) {
          const double u1 = std::max(rng.uniform(), 1e-300), u2 = rng.uniform();
          const double rr = sqrt(-2.0 * log(u1));
          z[a] = rr * cos(6.283185307179586 * u2);
          if (a + 1 < n) z[a + 1] = rr * sin(6.283185307179586 * u2);
        }
        for (int a = 0; a < n; ++a) nrm += z[a] * z[a];
        const double rad = scale * pow(rng.uniform(), 1.0 / n) / sqrt(nrm);
        bool inside = true;
        for (int a = 0; a < n; ++a) {
          double t = mu[a];
          for (int q = 0; q <= a; ++q) t += Lc[a][q] * z[q] * rad;
          const double v = plo[a] + t * (phi[a] - plo[a]);
          if (!(v >= blo[a] && v <= bhi[a])) inside = false;
          row[free_param[a]] = (float)v;
        }
        if (inside) break;
        if (attempt >= 1000) {                               // pathological: fall back to the box
          draw(row, blo.data(), bhi.data());
          break;
        }
      }
    }
    DRV_TRY(evaluate(batch));
    fs.iterations += 1;
    for (int i = 0; i < batch && !done; ++i) {
      const double lnl = isfinite(chi2.h[i]) ? -0.5 * (double)chi2.h[i] : -INFINITY;
      int worst = 0;
      for (int j = 1; j < n_live; ++j)
        if (live_lnl[j] < live_lnl[worst]) worst = j;
      if (!(lnl > live_lnl[worst])) continue;   // rejected: outside the current iso-likelihood contour
      // the worst live point dies: X_i = exp(-i / n_live), w_i = X_{i-1} - X_i
      const double x_prev = -(double)n_dead / n_live, x_now = -(double)(n_dead + 1) / n_live;
      const double lnw = x_prev + log1p(-exp(x_now - x_prev));
      dead_lnl.push_back(live_lnl[worst]), dead_lnw.push_back(lnw);
      for (int a = 0; a < n; ++a) dead_x.push_back(live[(size_t)worst * S + free_param[a]]);
      lnz = log_add(lnz, live_lnl[worst] + lnw);
      ++n_dead;
      memcpy(&live[(size_t)worst * S], rows.h + (size_t)i * S, sizeof(float) * S);
      live_lnl[worst] = lnl;
      const double lmax = *std::max_element(live_lnl.begin(), live_lnl.end());
      if (lmax + x_now < lnz + log((double)tol)) done = true;   // what is left cannot change Z by > tol
    }
  }
  // the live points share the remaining volume X = exp(-n_dead / n_live)
  const double ln_rest = -(double)n_dead / n_live - log((double)n_live);
  for (int i = 0; i < n_live; ++i) {
    dead_lnl.push_back(live_lnl[i]), dead_lnw.push_back(ln_rest);
    for (int a = 0; a < n; ++a) dead_x.push_back(live[(size_t)i * S + free_param[a]]);
    lnz = log_add(lnz, live_lnl[i] + ln_rest);
  }
  int best = 0;
  for (int j = 1; j < n_live; ++j)
    if (live_lnl[j] > live_lnl[best]) best = j;
  memcpy(best_row, &live[(size_t)best * S], sizeof(float) * S);
  *best_chi2 = live_lnl[best] == -INFINITY ? INFINITY : (float)(-2.0 * live_lnl[best]);
  if (mean_row) {
    memcpy(mean_row, base_row, sizeof(float) * S);
    std::vector<double> acc(n, 0.0);
    for (size_t i = 0; i < dead_lnl.size(); ++i) {
      const double w = exp(dead_lnl[i] + dead_lnw[i] - lnz);
      if (w > 0.0)
        for (int a = 0; a < n; ++a) acc[a] += w * dead_x[i * n + a];
    }
    for (int a = 0; a < n; ++a) mean_row[free_param[a]] = (float)acc[a];
  }
  if (log_evidence) *log_evidence = lnz;
  fs.converged = done ? 1 : 0;
  fs.ms_total = clock.ms();
  if (stats) *stats = fs;
  return GBK_OK;
}
