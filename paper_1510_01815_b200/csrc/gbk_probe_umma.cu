// A measured answer to "would tcgen05 help the 15 x 15 image-PSF pass?" (gbk_probe_umma of include/gbk.h).
//
// The pass of config 4 is a banded contraction: out[y][x] = sum_ky sum_kx W[ky][kx] in[y + ky][x + kx] on
// three maps.  As a tensor-core GEMM per kernel row ky:  D[(y, q)][x] += A_ky[(y, q)][x'] B_ky[x][x'],
// with A_ky the three maps (rows interleaved as 3 y + q, so that the shift by ky rows is a shift of the start
// address), K = x' over the 80 (78, padded) extended columns of a 64-wide tile, and B_ky[x][x'] = W[ky][x' - x]
// the Toeplitz band -- 15 of every 80 entries are non-zero.  FP32 accuracy (m0 1e-4, m2 a difference of sums)
// needs the maps as BF16 hi + lo and the taps as hi + lo: three products (hi hi, hi lo, lo hi).  Per 64 x 64
// tile that is 15 kernel rows x 3 products x 5 K-steps x (one M = 128 and one M = 64 MMA, N = 64, K = 16).
//
// This kernel issues exactly that sequence of tcgen05.mma instructions (single thread, operands in shared
// memory in the K-major no-swizzle canonical layout, accumulators in TMEM) `iters` times per CTA and is timed
// by the caller; before that it runs ONE MMA on known small integers and compares the accumulator, read back
// with tcgen05.ld, with the exact product, so that the descriptors are known to mean what they should.
// It is a probe, not a product path: the result is recorded in profiles/ and DESIGN.md.
#include <cuda_bf16.h>
#include <stdint.h>

#include "gbk_internal.h"

namespace gbk {
namespace {

constexpr int kRows = 240;        // 3 maps x 78 extended rows = 234, padded to a multiple of 8
constexpr int kPanels = 10;       // K = 80 columns = 10 panels of 8 BF16 (16 bytes)
constexpr int kSplits = 2;        // hi, lo
constexpr int kN = 64;            // output columns of the tile
constexpr uint32_t kABytes = kSplits * kPanels * kRows * 16;   // 76 800
constexpr uint32_t kBBytes = kSplits * kPanels * kN * 16;      // 20 480

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// K-major, no swizzle: element (r, k) of a K = 16 operand at  start + (k / 8) LBO + (r / 8) SBO + (r % 8) 16 + (k % 8) 2.
__device__ __forceinline__ uint64_t umma_desc(uint32_t addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((addr & 0x3FFFFu) >> 4);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
  d |= (uint64_t)1 << 46;          // descriptor version of sm_100
  return d;                        // base offset 0, layout type 0 = no swizzle
}

// kind::f16 instruction descriptor: D = F32, A = B = BF16, both K-major, N, M.
__device__ __forceinline__ uint32_t umma_idesc(int M, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

__device__ __forceinline__ void umma_bf16(uint32_t tmem_d, uint64_t a, uint64_t b, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t"
      "}\n" ::"r"(tmem_d), "l"(a), "l"(b), "r"(idesc), "r"(accumulate)
      : "memory");
}

__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}\n" ::"r"(bar), "r"(parity)
      : "memory");
}

__global__ void __launch_bounds__(128) probe_umma_band(int iters, float* __restrict__ out) {
  extern __shared__ __align__(128) unsigned char smem[];
  __nv_bfloat16* A = reinterpret_cast<__nv_bfloat16*>(smem);
  __nv_bfloat16* B = reinterpret_cast<__nv_bfloat16*>(smem + kABytes);
  uint64_t* bar = reinterpret_cast<uint64_t*>(smem + kABytes + kBBytes);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar + 1);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  // operands: small integers (exact in BF16) in the canonical layout.  a(r, k) = ((r + k) % 5) - 2,
  // b(n, k) = ((n + 2 k) % 7) - 3 for the first split; the other split gets the same values (timing only).
  for (int i = tid; i < kSplits * kPanels * kRows * 8; i += blockDim.x) {
    const int e = i & 7, r = (i >> 3) % kRows, p = ((i >> 3) / kRows) % kPanels;
    A[i] = __float2bfloat16((float)(((r + p * 8 + e) % 5) - 2));
  }
  for (int i = tid; i < kSplits * kPanels * kN * 8; i += blockDim.x) {
    const int e = i & 7, n = (i >> 3) % kN, p = ((i >> 3) / kN) % kPanels;
    B[i] = __float2bfloat16((float)(((n + 2 * (p * 8 + e)) % 7) - 3));
  }
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(bar)));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 0) {   // 128 TMEM columns: 64 for the M = 128 accumulator, 64 for the M = 64 one
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 128;" ::"r"(smem_u32(tmem_slot)) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic-proxy stores -> async-proxy reads
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_slot;
  const uint32_t a0 = smem_u32(A), b0 = smem_u32(B), barp = smem_u32(bar);
  const uint32_t lbo_a = kRows * 16, lbo_b = kN * 16, sbo = 128;
  uint32_t phase = 0;

  // ---- one MMA on known integers: D[m][n] = sum_k a(m, k) b(n, k), k < 16 -------------------------
  if (tid == 32) {
    umma_bf16(tmem, umma_desc(a0, lbo_a, sbo), umma_desc(b0, lbo_b, sbo), umma_idesc(128, kN), 0u);
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(barp) : "memory");
  }
  mbar_wait(barp, phase);
  phase ^= 1;
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  float max_err = 0.0f;
  {
    const int m = warp * 32 + lane;                                // TMEM lane = row of D
    for (int n0 = 0; n0 < kN; n0 += 8) {
      uint32_t v[8];
      const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)n0;
      asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                   : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                   : "r"(taddr));
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        float want = 0.0f;
        for (int k = 0; k < 16; ++k) want += (float)(((m + k) % 5) - 2) * (float)(((n0 + j + 2 * k) % 7) - 3);
        max_err = fmaxf(max_err, fabsf(__uint_as_float(v[j]) - want));
      }
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();

  // ---- the MMA sequence of one 64 x 64 tile of the 15 x 15 pass, `iters` times ----------------------
  if (tid == 32) {
    const uint32_t id128 = umma_idesc(128, kN), id64 = umma_idesc(64, kN);
    for (int it = 0; it < iters; ++it) {
      uint32_t acc = 0;
      for (int ky = 0; ky < 15; ++ky)
        for (int prod = 0; prod < 3; ++prod) {            // (A hi, B hi), (A hi, B lo), (A lo, B hi)
          const int sa = prod == 2 ? 1 : 0, sb = prod == 1 ? 1 : 0;
          for (int ks = 0; ks < kPanels / 2; ++ks) {
            const uint32_t a = a0 + ((uint32_t)((sa * kPanels + 2 * ks) * kRows + 3 * ky)) * 16;
            const uint32_t b = b0 + ((uint32_t)((sb * kPanels + 2 * ks) * kN)) * 16;
            umma_bf16(tmem, umma_desc(a, lbo_a, sbo), umma_desc(b, lbo_b, sbo), id128, acc);
            umma_bf16(tmem + 64, umma_desc(a + 128 * 16, lbo_a, sbo), umma_desc(b, lbo_b, sbo), id64, acc);
            acc = 1;
          }
        }
      asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(barp) : "memory");
      mbar_wait(barp, phase);
      phase ^= 1;
    }
  }
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 128;" ::"r"(tmem) : "memory");
  // the largest error of the check over the CTA (block 0 reports)
  for (int off = 16; off > 0; off >>= 1) max_err = fmaxf(max_err, __shfl_xor_sync(0xffffffffu, max_err, off));
  __shared__ float red[4];
  if (lane == 0) red[warp] = max_err;
  __syncthreads();
  if (blockIdx.x == 0 && tid == 0) out[0] = fmaxf(fmaxf(red[0], red[1]), fmaxf(red[2], red[3]));
}

}  // namespace

cudaError_t launch_probe_umma(int iters, int blocks, float* out, cudaStream_t st) {
  const int smem = (int)(kABytes + kBBytes + 64);
  cudaError_t e = cudaFuncSetAttribute(probe_umma_band, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e != cudaSuccess) return e;
  probe_umma_band<<<blocks, 128, smem, st>>>(iters, out);
  return cudaGetLastError();
}

}  // namespace gbk
