// taylor_tc.cuh -- H7 on the tensor pipe: Phi' = E_h [sum_{k<=K} A^k/k!] E_h Phi  (R3, R9).
// Persistent CTAs, one walker at a time.  Every product X * T (X = E_h real or A_w complex symmetric, T complex
// M x N_t) is a set of real tcgen05.mma.kind::tf32 products with the 3xTF32 split:
//     D_re = X_r T_r - X_i T_i ,  D_im = X_r T_i + X_i T_r      (the minus sign via the descriptor's negate-B bit)
// a-operand: 128-row x 32-column tiles of X (hi / lo planes) streamed by TMA through a 3-stage ring;
// b-operand: T as four K-major planes (T_r, T_i) x (hi, lo), [32 rows (walker columns)][KP] in shared memory,
//            rewritten by the epilogue warps after every Taylor term (generic -> async proxy fence);
// accumulators: TMEM, 64 columns per 128-row tile (32 re | 32 im).  The running sum P lives in registers.
// Supported: M <= 256, N_t <= 32 (else the SIMT kernel of taylor.cuh runs).
#pragma once
#include "gemm_tf32.cuh"

namespace afq {
namespace tt {

using namespace tc;

enum { NST = 3, TILE_BYTES = 128 * 128, STG_BYTES = 2 * TILE_BYTES, PLANE_KB_BYTES = 32 * 128, EPW = 8, NTHREADS = (EPW + 2) * 32 };

struct TaylorMaps {
  CUtensorMap A[2][2];   // [hi/lo][0: 128-row box, 1: last-tile box]  over Abuf viewed as [N_w*M][2*MP]
  CUtensorMap E[2][2];   // same for E_h [M][MP]
};

struct TaylorTcArgs {
  int M, MP, nt, K, nw;
  int mtiles, rows_last, nkb;   // 128-row tiles, rows of the last one (multiple of 8), 32-column k-blocks
  cplx<float>* phi;             // [nw][M][nt] in/out
};

inline size_t smem_bytes(int nkb) { return (size_t)4 * nkb * PLANE_KB_BYTES + (size_t)NST * STG_BYTES + 1024; }

// byte offset of element (row b, column j) inside one K-major SWIZZLE_128B plane
__device__ __forceinline__ uint32_t plane_off(int b, int j) {
  const int kb = j >> 5, jj = j & 31;
  return (uint32_t)(kb * PLANE_KB_BYTES + b * 128 + ((((jj >> 2) ^ (b & 7)) << 4) | ((jj & 3) << 2)));
}

__global__ void __launch_bounds__(NTHREADS, 1) k_taylor_tc(const __grid_constant__ TaylorMaps maps, TaylorTcArgs g) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[NST];
  __shared__ __align__(8) uint64_t empty_bar[NST];
  __shared__ __align__(8) uint64_t tmem_full_bar;
  __shared__ __align__(8) uint64_t b_ready_bar;
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int M = g.M, nt = g.nt, nkb = g.nkb, mtiles = g.mtiles;
  const uint32_t plane_bytes = (uint32_t)nkb * PLANE_KB_BYTES;
  uint8_t* planes = smem;                                   // [Tr_hi | Tr_lo | Ti_hi | Ti_lo]
  uint8_t* stages = smem + 4 * (size_t)plane_bytes;
  const int nphase = g.K + 2;
  const uint32_t tmem_cols = mtiles > 1 ? 128u : 64u;

  // zero the planes once: rows >= nt and columns >= M must stay 0 for the whole kernel
  for (uint32_t o = threadIdx.x * 16; o < 4 * plane_bytes; o += NTHREADS * 16)
    *reinterpret_cast<uint4*>(planes + o) = make_uint4(0, 0, 0, 0);
  if (warp == EPW && lane == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    mbar_init(&tmem_full_bar, 1);
    mbar_init(&b_ready_bar, EPW);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == EPW + 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "r"(tmem_cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  if (warp == EPW) {
    if (lane == 0) {   // ===== TMA producer: streams X tiles for every (walker, phase, tile, k-block, plane) =====
      uint32_t it = 0;
      for (int w = blockIdx.x; w < g.nw; w += gridDim.x)
        for (int ph = 0; ph < nphase; ++ph) {
          const bool cx = ph >= 1 && ph <= g.K;           // complex A_w, else real E_h
          for (int mt = 0; mt < mtiles; ++mt) {
            const int last = mt == mtiles - 1;
            const uint32_t bytes = 2u * (uint32_t)(last ? g.rows_last : 128) * 128u;
            for (int kb = 0; kb < nkb; ++kb)
              for (int p = 0; p < (cx ? 2 : 1); ++p, ++it) {
                const int s = it % NST;
                mbar_wait(&empty_bar[s], ((it / NST) & 1) ^ 1);
                uint8_t* st = stages + (size_t)s * STG_BYTES;
                mbar_expect_tx(&full_bar[s], bytes);
                if (cx) {
                  tma_load_2d(st, &maps.A[0][last], &full_bar[s], p * g.MP + kb * 32, w * M + mt * 128);
                  tma_load_2d(st + TILE_BYTES, &maps.A[1][last], &full_bar[s], p * g.MP + kb * 32, w * M + mt * 128);
                } else {
                  tma_load_2d(st, &maps.E[0][last], &full_bar[s], kb * 32, mt * 128);
                  tma_load_2d(st + TILE_BYTES, &maps.E[1][last], &full_bar[s], kb * 32, mt * 128);
                }
              }
          }
        }
    }
  } else if (warp == EPW + 1) {
    if (lane == 0) {   // ===== MMA issuer =====
      constexpr uint32_t idesc = make_idesc(128, 32);
      constexpr uint32_t idesc_negb = idesc | (1u << 14);
      const uint32_t pl = smem_u32(planes);
      uint32_t it = 0, gph = 0;
      for (int w = blockIdx.x; w < g.nw; w += gridDim.x)
        for (int ph = 0; ph < nphase; ++ph, ++gph) {
          const bool cx = ph >= 1 && ph <= g.K;
          mbar_wait(&b_ready_bar, gph & 1);               // T planes of this phase are in shared memory
          tc_fence_after();
          for (int mt = 0; mt < mtiles; ++mt) {
            const uint32_t d_re = tmem + mt * 64, d_im = d_re + 32;
            for (int kb = 0; kb < nkb; ++kb)
              for (int p = 0; p < (cx ? 2 : 1); ++p, ++it) {
                const int s = it % NST;
                mbar_wait(&full_bar[s], (it / NST) & 1);
                tc_fence_after();
                const uint32_t sa = smem_u32(stages + (size_t)s * STG_BYTES);
                const uint64_t x_hi = make_desc(sa), x_lo = make_desc(sa + TILE_BYTES);
                const uint32_t kboff = (uint32_t)kb * PLANE_KB_BYTES;
                const uint64_t tr_hi = make_desc(pl + kboff), tr_lo = make_desc(pl + plane_bytes + kboff);
                const uint64_t ti_hi = make_desc(pl + 2 * plane_bytes + kboff), ti_lo = make_desc(pl + 3 * plane_bytes + kboff);
                // p == 0: D_re += X_r T_r, D_im += X_r T_i ;  p == 1: D_re -= X_i T_i, D_im += X_i T_r
                const uint64_t bre_hi = p ? ti_hi : tr_hi, bre_lo = p ? ti_lo : tr_lo;
                const uint64_t bim_hi = p ? tr_hi : ti_hi, bim_lo = p ? tr_lo : ti_lo;
                const uint32_t id_re = p ? idesc_negb : idesc;
                const bool first = kb == 0 && p == 0;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                  const uint64_t adv = (uint64_t)(k * 2);   // 8 tf32 = 32 bytes = 2 x 16 B
                  umma_tf32(d_re, x_lo + adv, bre_hi + adv, id_re, (first && k == 0) ? 0u : 1u);
                  umma_tf32(d_re, x_hi + adv, bre_lo + adv, id_re, 1u);
                  umma_tf32(d_re, x_hi + adv, bre_hi + adv, id_re, 1u);
                  umma_tf32(d_im, x_lo + adv, bim_hi + adv, idesc, (first && k == 0) ? 0u : 1u);
                  umma_tf32(d_im, x_hi + adv, bim_lo + adv, idesc, 1u);
                  umma_tf32(d_im, x_hi + adv, bim_hi + adv, idesc, 1u);
                }
                tc_commit(&empty_bar[s]);
              }
          }
          tc_commit(&tmem_full_bar);
        }
    }
  } else {   // ===== epilogue warps 0..7: TMEM lane quarter = warp & 3, half = warp >> 2 (0: real part, 1: imaginary) =====
    const int q = warp & 3, half = warp >> 2;
    uint8_t* pl_hi = planes + (size_t)(2 * half) * plane_bytes;       // T_r or T_i, hi
    uint8_t* pl_lo = pl_hi + plane_bytes;
    uint32_t gph = 0;
    float P[2][32];
    for (int w = blockIdx.x; w < g.nw; w += gridDim.x) {
      float* phi_w = reinterpret_cast<float*>(g.phi + (size_t)w * M * nt);
      // phase-0 operand: planes <- Phi_w  (row b = walker column, column j = basis index)
      for (int e = (warp & 3) * 32 + lane; e < M * nt; e += 128) {
        const int j = e / nt, b = e - j * nt;
        float hi, lo;
        tf32_split(phi_w[2 * e + half], hi, lo);
        const uint32_t o = plane_off(b, j);
        *reinterpret_cast<float*>(pl_hi + o) = hi;
        *reinterpret_cast<float*>(pl_lo + o) = lo;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&b_ready_bar)) : "memory");
      for (int ph = 0; ph < nphase; ++ph, ++gph) {
        mbar_wait(&tmem_full_bar, gph & 1);
        tc_fence_after();
        const bool last_phase = ph == nphase - 1;
        const float scale = (ph >= 1 && ph <= g.K) ? 1.0f / (float)ph : 1.0f;
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          if (mt < mtiles) {
            float v[32];
            tmem_ld32(tmem + ((uint32_t)(q * 32) << 16) + mt * 64 + half * 32, v);
            const int i = mt * 128 + q * 32 + lane;     // output row = basis index
#pragma unroll
            for (int b = 0; b < 32; ++b) {
              float t = v[b] * scale;
              if (ph == 0) P[mt][b] = t; else P[mt][b] += t;
              if (ph == g.K) t = P[mt][b];               // operand of the closing E_h product is the sum
              v[b] = t;
            }
            if (i < M) {
              if (last_phase) {
                for (int b = 0; b < nt; ++b) phi_w[2 * (i * nt + b) + half] = v[b];
              } else {
#pragma unroll
                for (int b = 0; b < 32; ++b) {
                  if (b < nt) {
                    float hi, lo;
                    tf32_split(v[b], hi, lo);
                    const uint32_t o = plane_off(b, i);
                    *reinterpret_cast<float*>(pl_hi + o) = hi;
                    *reinterpret_cast<float*>(pl_lo + o) = lo;
                  }
                }
              }
            }
          }
        }
        tc_fence_before();
        if (!last_phase) {
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          __syncwarp();
          if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&b_ready_bar)) : "memory");
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == EPW + 1) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(tmem_cols) : "memory");
  }
}

}  // namespace tt
}  // namespace afq
