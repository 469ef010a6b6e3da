// peaks.cuh -- self-written peak microbenchmarks ("the builder measures them with tiny self-written
// microbenchmarks ... before quoting any fraction"): back-to-back tcgen05.mma.kind::tf32 (operands from shared memory,
// the a-operand from TMEM, or on a CTA pair), FFMA and DFMA loops, and an L2 -> shared-memory TMA stream.  bench.py --peaks
// prints them beside the nominal figures; they are the denominators DESIGN.md 7 argues with.  Not on the walker step's path.
#pragma once
#include "gemm_tf32.cuh"

namespace afq {
namespace pk {

using namespace tc;

// mode 0: SS (a, b from shared memory), one CTA;  1: TS (a from TMEM);  2: SS on a CTA pair (M = 256)
// Every CTA issues `iters` k-blocks of 4 MMAs (K = 8 each) into one accumulator; out[blockIdx] = clocks of the issue loop
// (first MMA issued -> last MMA completed).
template <int MODE>
__global__ void __launch_bounds__(320, 1) k_peak_mma(int N, int iters, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t done_bar_s[2];
  uint64_t& done_bar = done_bar_s[0];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float* a = reinterpret_cast<float*>(smem);                    // 128 rows x 32 columns, K-major (content irrelevant to timing;
  float* b = reinterpret_cast<float*>(smem + 16384);            // N rows x 32 columns     small finite numbers, no NaN patterns)
  for (int e = threadIdx.x; e < (128 + 256) * 32; e += blockDim.x) a[e] = (float)((e * 2654435761u) >> 20) * (1.0f / 4096.0f) - 0.5f;
  if (threadIdx.x == 0) { mbar_init(&done_bar, 1); mbar_init(&done_bar + 1, 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (warp == 0) {
    if (MODE == 2) {
      asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512u) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
    } else {
      asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512u) : "memory");
      asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  if (MODE == 2) cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  const uint32_t rank = MODE == 2 ? cluster_ctarank() : 0u;
  if (warp == 1 && lane == 0 && rank == 0) {
    const uint32_t idesc = make_idesc(MODE == 2 ? 256 : 128, N);
    const uint64_t ad = make_desc(smem_u32(a)), bd = make_desc(smem_u32(b));
    const uint32_t a_t = tmem + 256;      // TS: a-operand rows = lanes, K elements = columns 256.. (uninitialised TMEM: timing only)
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint64_t adv = (uint64_t)(k * 2);
        const uint32_t acc = (it | k) ? 1u : 0u;
        if (MODE == 0) umma_tf32(tmem, ad + adv, bd + adv, idesc, acc);
        if (MODE == 1) umma_tf32_ts(tmem, a_t + k * 8, bd + adv, idesc, acc);
        if (MODE == 2) umma_tf32_pair(tmem, ad + adv, bd + adv, idesc, acc);
        if (MODE >= 3) {   // the Taylor kernel's k-step: X_hi [T_hi | T_lo] (N = 128) then X_lo T_hi (N = 64), rotating stage slots
          const uint64_t as = make_desc(smem_u32(smem + 49152 + (it % 3) * 32768));
          umma_tf32(tmem, as + adv, bd + adv, make_idesc(128, 128), acc);
          umma_tf32(tmem + 64, as + 1024 + adv, bd + adv, make_idesc(128, 64), 1u);
        }
      }
      if (MODE >= 3 && (it & 1)) tc_commit(&done_bar + 1);
      if (MODE == 3 && N == 144) { tc_commit(&done_bar + 1); tc_commit(&done_bar + 1); }               // two commits per 8 MMAs
      if (MODE == 3 && N == 160) { tc_commit(&done_bar + 1); mbar_wait(&done_bar + 1, 0); }             // + an (already complete) wait
    }
    if (MODE == 2) tc_commit_pair(&done_bar); else tc_commit(&done_bar);
    mbar_wait(&done_bar, 0);
    out[blockIdx.x] = clock64() - t0;
  } else if (MODE == 2 && warp == 1 && lane == 0) {
    mbar_wait(&done_bar, 0);      // the peer's copy of the barrier receives the multicast commit
  } else if (MODE == 4 && warp >= 2) {
    // other warps keep the shared-memory ports busy the way the Taylor epilogue does (scalar stores + loads)
    volatile float* z = reinterpret_cast<volatile float*>(smem + 49152 + 3 * 32768);
    float acc2 = 0.f;
    for (int it = 0; it < iters * 6; ++it) {
#pragma unroll
      for (int u = 0; u < 8; ++u) { z[((threadIdx.x - 64) * 33 + u * 67 + it) & 4095] = acc2; acc2 += z[(threadIdx.x * 17 + u * 129 + it) & 4095]; }
    }
    if (acc2 == -1.f) out[1] = 0;
  }
  tc_fence_before();
  __syncthreads();
  if (MODE == 2) cluster_sync_all();
  if (warp == 0) {
    if (MODE == 2) asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
    else asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
  }
}

// The Taylor kernel's issue pattern, warp-uniform issue (elect_one): per iteration 4 k-steps of [N = 128 into d, N = 64 into
// d + 64] on rotating a-tiles, followed by NC tcgen05.commit (NC = 0: one commit at the very end only).
template <int NC, int POLL>
__global__ void __launch_bounds__(384, 1) k_peak_taylor(int iters, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[4];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float* a = reinterpret_cast<float*>(smem);
  for (int e = threadIdx.x; e < (16384 + 6 * 16384) / 4; e += blockDim.x) a[e] = (float)((e * 2654435761u) >> 20) * (1.0f / 4096.0f) - 0.5f;
  if (threadIdx.x == 0) { for (int i = 0; i < 4; ++i) mbar_init(&bars[i], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  if (warp == 1) {
    const uint32_t base = smem_u32(smem);
    const uint64_t bd = make_desc(base);                       // T planes stand-in: 128 rows
    int s = 0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
      const uint64_t xh = make_desc(base + 16384 + (uint32_t)s * 32768), xl = make_desc(base + 32768 + (uint32_t)s * 32768);
      const uint32_t d = tmem + (uint32_t)(it & 3) * 128;
      if (elect_one()) {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint64_t adv = (uint64_t)(k * 2);
          umma_tf32(d, xh + adv, bd + adv, make_idesc(128, 128), (it | k) ? 1u : 0u);
          umma_tf32(d + 64, xl + adv, bd + adv, make_idesc(128, 64), 1u);
        }
#pragma unroll
        for (int c = 0; c < NC; ++c) tc_commit(&bars[1 + c]);
      }
      __syncwarp();
      if (++s == 3) s = 0;
    }
    if (elect_one()) tc_commit(&bars[0]);
    __syncwarp();
    mbar_wait(&bars[0], 0);
    if (lane == 0) out[blockIdx.x] = clock64() - t0;
  } else if (POLL && warp >= 2) {
    mbar_wait(&bars[0], 0);      // the other warps poll a barrier that completes at the very end, as the epilogue warps do
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

// Table-driven MMA pattern: per iteration the warp issues tab.n MMAs {a offset, b offset (bytes from the 1024-aligned base),
// N, accumulator column}, uniform issue; used to compare operand orderings (which operand slices repeat back to back).
struct MmaTab { int n; int a[64]; int b[64]; int nn[64]; int d[64]; };
__global__ void __launch_bounds__(64, 1) k_peak_tab(const __grid_constant__ MmaTab tab, int iters, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[2];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float* a = reinterpret_cast<float*>(smem);
  for (int e = threadIdx.x; e < 220 * 1024 / 4; e += blockDim.x) a[e] = (float)((e * 2654435761u) >> 20) * (1.0f / 4096.0f) - 0.5f;
  if (threadIdx.x == 0) { mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  if (warp == 1) {
    const uint32_t base = smem_u32(smem);
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
      for (int m = 0; m < tab.n; ++m) {
        const uint64_t ad = make_desc(base + (uint32_t)tab.a[m]), bd = make_desc(base + (uint32_t)tab.b[m]);
        const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(tab.nn[m] >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
        if (elect_one()) umma_tf32(tmem + (uint32_t)tab.d[m], ad, bd, idesc, (it | m) ? 1u : 0u);
        __syncwarp();
      }
    }
    if (elect_one()) tc_commit(&bars[0]);
    __syncwarp();
    mbar_wait(&bars[0], 0);
    if (lane == 0) out[blockIdx.x] = clock64() - t0;
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

// Compile-time MMA orderings for the Taylor product, uniform issue, operands rotating through shared memory the
// way the real kernel's do: T k-blocks (NB of them, 16 KB apart from offset 0) and X tiles (from 112 KB on).
//   PAT 0  current:  per (k-block, plane): 4 x [X_hi (N=128, b = T slice) ; X_lo (N=64, same b)]
//   PAT 1  swapped:  T slice is the a-operand (128 rows), X tiles (208 rows) the b-operand: 4 x [X_hi ; X_lo], N = 208
//   PAT 2  grouped:  per k-block 4 x [X_r_hi, X_i_hi (N=128), X_r_lo, X_i_lo (N=64)] all on the same T slice
// out = clocks per k-block-plane equivalent (PAT 2 covers two planes per group: reported per plane).
template <int PAT, int NB, int EXTRA>
__global__ void __launch_bounds__(64, 1) k_peak_pat(int iters, long long* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bars[4];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  float* a = reinterpret_cast<float*>(smem);
  for (int e = threadIdx.x; e < 224 * 1024 / 4; e += blockDim.x) a[e] = (float)((e * 2654435761u) >> 20) * (1.0f / 4096.0f) - 0.5f;
  if (threadIdx.x == 0) { for (int i = 0; i < 4; ++i) mbar_init(&bars[i], 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  if (warp == 1) {
    const uint32_t base = smem_u32(smem), xb = base + 112 * 1024;
    int kb = 0, s = 0;
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
      const uint64_t t = make_desc(base + (uint32_t)kb * 16384);
      if (PAT == 0) {
        const uint64_t xh = make_desc(xb + (uint32_t)s * 16384), xl = make_desc(xb + (uint32_t)(s + 1) * 16384);
        const uint32_t d = tmem + (uint32_t)(it & 3) * 128;
        if (EXTRA & 2) mbar_wait(&bars[1], 1);      // a wait that is already satisfied: its latency only
        if (EXTRA & 4) tc_fence_after();
        if (elect_one()) {
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            umma_tf32(d, xh + 2 * k, t + 2 * k, make_idesc(128, 128), (it | k) ? 1u : 0u);
            umma_tf32(d + 64, xl + 2 * k, t + 2 * k, make_idesc(128, 64), 1u);
          }
          if (EXTRA & 1) { tc_commit(&bars[2]); tc_commit(&bars[3]); }
        }
        __syncwarp();
        s += 2; if (s >= 6) s = 0;
        if (it & 1) { if (++kb == NB) kb = 0; }        // two planes per k-block
      } else if (PAT == 1) {
        const uint64_t xh = make_desc(xb + (uint32_t)s * 53248), xl = make_desc(xb + (uint32_t)s * 53248 + 26624);
        const uint32_t d = tmem + (uint32_t)(it & 1) * 256;
        if (elect_one()) {
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            umma_tf32(d, t + 2 * k, xh + 2 * k, make_idesc(128, 208), (it | k) ? 1u : 0u);
            umma_tf32(d, t + 2 * k, xl + 2 * k, make_idesc(128, 208), 1u);
          }
        }
        __syncwarp();
        s ^= 1;
        if (it & 1) { if (++kb == NB) kb = 0; }
      } else {
        const uint64_t x0 = make_desc(xb + (uint32_t)s * 65536), x1 = make_desc(xb + (uint32_t)s * 65536 + 16384),
                       x2 = make_desc(xb + (uint32_t)s * 65536 + 32768), x3 = make_desc(xb + (uint32_t)s * 65536 + 49152);
        if (elect_one()) {
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            umma_tf32(tmem, x0 + 2 * k, t + 2 * k, make_idesc(128, 128), (it | k) ? 1u : 0u);
            umma_tf32(tmem + 128, x1 + 2 * k, t + 2 * k, make_idesc(128, 128), (it | k) ? 1u : 0u);
            umma_tf32(tmem + 64, x2 + 2 * k, t + 2 * k, make_idesc(128, 64), 1u);
            umma_tf32(tmem + 192, x3 + 2 * k, t + 2 * k, make_idesc(128, 64), 1u);
          }
        }
        __syncwarp();
        s = (s + 1) % 1;      // 4 x 16 KB tiles per group: only one group slot fits beside 112 KB of planes here
        if (++kb == NB) kb = 0;
      }
    }
    if (elect_one()) tc_commit(&bars[0]);
    __syncwarp();
    mbar_wait(&bars[0], 0);
    if (lane == 0) out[blockIdx.x] = (clock64() - t0) / (PAT == 2 ? 2 : 1);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

// Correctness probe for the TS-mode Taylor design: A (128 x 32 tf32) is written to TMEM by tcgen05.st (thread = row, 32 columns),
// B is N rows of a K-major SWIZZLE_128B tile starting r0 rows into the tile; D[128][N] is read back.  a[r][c] = ((r * 3 + c * 5) % 17) - 8,
// b[n][c] = ((n * 7 + c * 11) % 13) - 6 (small integers: exact in TF32), out[r * N + n] = sum_c a[r][c] b[r0 + n][c].
__global__ void __launch_bounds__(128, 1) k_probe_ts(int N, int r0, float* out) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t bar;
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  for (int e = threadIdx.x; e < 128 * 32; e += blockDim.x) {
    const int n = e >> 5, c = e & 31;
    const float v = (float)(((n * 7 + c * 11) % 13) - 6);
    *reinterpret_cast<float*>(smem + n * 128 + ((((c >> 2) ^ (n & 7)) << 4) | ((c & 3) << 2))) = v;
  }
  if (threadIdx.x == 0) { mbar_init(&bar, 1); asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(512u) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  {
    const int r = warp * 32 + lane;
    uint32_t a[32];
#pragma unroll
    for (int c = 0; c < 32; ++c) a[c] = __float_as_uint((float)(((r * 3 + c * 5) % 17) - 8));
    const uint32_t taddr = tmem + ((uint32_t)(warp * 32) << 16) + 256;
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};"
        ::"r"(taddr), "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(a[4]), "r"(a[5]), "r"(a[6]), "r"(a[7]), "r"(a[8]), "r"(a[9]),
          "r"(a[10]), "r"(a[11]), "r"(a[12]), "r"(a[13]), "r"(a[14]), "r"(a[15]), "r"(a[16]), "r"(a[17]), "r"(a[18]), "r"(a[19]),
          "r"(a[20]), "r"(a[21]), "r"(a[22]), "r"(a[23]), "r"(a[24]), "r"(a[25]), "r"(a[26]), "r"(a[27]), "r"(a[28]), "r"(a[29]),
          "r"(a[30]), "r"(a[31])
        : "memory");
    asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  if (warp == 1) {
    const uint64_t bd = make_desc(smem_u32(smem) + (uint32_t)r0 * 128);
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    if (elect_one()) {
#pragma unroll
      for (int k = 0; k < 4; ++k) umma_tf32_ts(tmem, tmem + 256 + k * 8, bd + 2 * k, idesc, k ? 1u : 0u);
      tc_commit(&bar);
    }
    __syncwarp();
  }
  mbar_wait(&bar, 0);
  tc_fence_after();
  for (int c0 = 0; c0 < N; c0 += 28) {        // 28-column steps on purpose: the design reads at offsets that are multiples of 28
    float v[32];
    tmem_ld32(tmem + ((uint32_t)(warp * 32) << 16) + c0, v);
    const int r = warp * 32 + lane;
    for (int j = 0; j < 28 && c0 + j < N; ++j) out[r * N + c0 + j] = v[j];
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(512u) : "memory");
}

// FFMA / DFMA: 8 independent chains per thread, 8 * 2 * iters flops per thread
template <typename T> __global__ void __launch_bounds__(512) k_peak_fma(int iters, T seed, T* out) {
  T v[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = seed + (T)(threadIdx.x + i);
  const T m = (T)0.999, c = (T)1e-3;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) v[i] = fma(v[i], m, c);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += v[i];
  if (s == (T)-12345) out[0] = s;     // never true: keeps the chains alive
}

// L2 -> shared memory: every CTA streams `iters` boxes of 128 rows x 32 floats (16 KB) by TMA through a 4-deep ring from a
// buffer of `rows` rows (small enough to stay L2 resident), starting at a CTA-dependent row.
__global__ void __launch_bounds__(64, 1) k_peak_tma(const __grid_constant__ CUtensorMap map, int rows, int iters) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full[4];
  if (threadIdx.x == 0) {
    for (int s = 0; s < 4; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    const int nbox = rows / 128;
    int box = (blockIdx.x * 37) % nbox;
    for (int it = 0; it < iters + 4; ++it) {
      const int s = it & 3;
      if (it >= 4) mbar_wait(&full[s], ((it - 4) >> 2) & 1);
      if (it < iters) {
        mbar_expect_tx(&full[s], 16384);
        tma_load_2d(smem + s * 16384, &map, &full[s], 0, box * 128);
        box = box + 1 == nbox ? 0 : box + 1;
      }
    }
  }
}

}  // namespace pk
}  // namespace afq
