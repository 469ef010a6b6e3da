// taylor_tc.cuh -- H7 on the tensor pipe: Phi' = E_h [sum_{k<=K} A^k/k!] E_h Phi  (R3, R9).
// Persistent CTAs, one walker at a time.  Every product X * T (X = E_h real or A_w complex symmetric, T complex
// M x N_t) is a set of real tcgen05.mma.kind::tf32 products with the 3xTF32 split:
//     D1 = X_r [T_r | T_i] ,  D2 = X_i [T_r | T_i];  D_re = D1[0:32] - D2[32:64],  D_im = D1[32:64] + D2[0:32]
//     are combined by the epilogue warps.  Measured: with N this small the kernel is bound by the tensor pipe's
//     shared-memory operand fetch (~64 B/clk/SM; every MMA re-reads its 4 KB a-operand slice), so the products are
//     packed into as few, as wide MMAs as possible: X_hi [T_hi | T_lo] is ONE N = 128 MMA (columns 0-63: hi*hi,
//     64-127: hi*lo) and X_lo T_hi one N = 64 MMA into columns 0-63; the epilogue adds the two column halves.
// a-operand: 128-row x 32-column tiles of X (hi / lo planes) streamed by TMA through a 3-stage ring;
// b-operand: T K-major in shared memory, per 32-column k-block 128 rows: [T_r, T_i (hi) | T_r, T_i (lo)],
//            rewritten by the epilogue warps after every Taylor term (generic -> async proxy fence);
// accumulators: TMEM, 128 columns per (128-row tile, plane).  The running sum P lives in registers.
// Supported: M <= 256, N_t <= 32 (else the SIMT kernel of taylor.cuh runs).
#pragma once
#include "gemm_tf32.cuh"

namespace afq {
namespace tt {

using namespace tc;

enum { NST = 3, TILE_BYTES = 128 * 128, STG_BYTES = 2 * TILE_BYTES, PLANE_KB_BYTES = 128 * 128, EPW = 8, NTHREADS = (EPW + 2) * 32 };

struct TaylorMaps {
  CUtensorMap A[2][2];   // [hi/lo][0: 128-row box, 1: last-tile box]  over Abuf viewed as [N_w*M][2*MP]
  CUtensorMap E[2][2];   // same for E_h [M][MP]
};

struct TaylorTcArgs {
  int M, MP, nt, K, nw;
  int mtiles, rows_last, nkb;   // 128-row tiles, rows of the last one (multiple of 8), 32-column k-blocks
  int nch, chunk_kb;            // accumulation chunks per tile (each its own 64 TMEM columns) and k-blocks per chunk:
                                // the tensor pipe truncates when it adds into its accumulator, so one long chain
                                // drifts; chunks are summed round-to-nearest in registers by the epilogue warps
  cplx<float>* phi;             // [nw][M][nt] in/out
};

inline size_t smem_bytes(int nkb) { return (size_t)nkb * PLANE_KB_BYTES + (size_t)NST * STG_BYTES + 1024; }

// byte offset of element (row b in 0..127, column j) inside the K-major SWIZZLE_128B T operand
__device__ __forceinline__ uint32_t plane_off(int b, int j) {
  const int kb = j >> 5, jj = j & 31;
  return (uint32_t)(kb * PLANE_KB_BYTES + b * 128 + ((((jj >> 2) ^ (b & 7)) << 4) | ((jj & 3) << 2)));
}

__global__ void __launch_bounds__(NTHREADS, 1) k_taylor_tc(const __grid_constant__ TaylorMaps maps, TaylorTcArgs g) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[NST];
  __shared__ __align__(8) uint64_t empty_bar[NST];
  __shared__ __align__(8) uint64_t tmem_full_bar[2];   // per 128-row tile: tile 0 is post-processed while tile 1 is issued
  __shared__ __align__(8) uint64_t b_ready_bar;
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int M = g.M, nt = g.nt, nkb = g.nkb, mtiles = g.mtiles;
  const uint32_t plane_bytes = (uint32_t)nkb * PLANE_KB_BYTES;
  uint8_t* planes = smem;                                   // rows 0-31 T_r hi, 32-63 T_i hi, 64-95 T_r lo, 96-127 T_i lo
  uint8_t* stages = smem + (size_t)plane_bytes;
  const int nphase = g.K + 2;
  const uint32_t tmem_cols = 512u;

  // zero the planes once: rows >= nt and columns >= M must stay 0 for the whole kernel
  for (uint32_t o = threadIdx.x * 16; o < plane_bytes; o += NTHREADS * 16)
    *reinterpret_cast<uint4*>(planes + o) = make_uint4(0, 0, 0, 0);
  if (warp == EPW && lane == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    mbar_init(&tmem_full_bar[0], 1); mbar_init(&tmem_full_bar[1], 1);
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
      constexpr uint32_t idesc128 = make_idesc(128, 128), idesc64 = make_idesc(128, 64);
      const uint32_t pl = smem_u32(planes);
      uint32_t it = 0, gph = 0;
      for (int w = blockIdx.x; w < g.nw; w += gridDim.x)
        for (int ph = 0; ph < nphase; ++ph, ++gph) {
          const bool cx = ph >= 1 && ph <= g.K;
          mbar_wait(&b_ready_bar, gph & 1);               // T planes of this phase are in shared memory
          tc_fence_after();
          for (int mt = 0; mt < mtiles; ++mt) {
            for (int kb = 0; kb < nkb; ++kb)
              for (int p = 0; p < (cx ? 2 : 1); ++p, ++it) {
                const uint32_t d = tmem + (mt * 2 + p) * 128;
                const int s = it % NST;
                mbar_wait(&full_bar[s], (it / NST) & 1);
                tc_fence_after();
                const uint32_t sa = smem_u32(stages + (size_t)s * STG_BYTES);
                const uint64_t x_hi = make_desc(sa), x_lo = make_desc(sa + TILE_BYTES);
                const uint32_t kboff = (uint32_t)kb * PLANE_KB_BYTES;
                const uint64_t t_all = make_desc(pl + kboff);   // 128 rows: hi then lo; its first 64 rows = T_hi
                const bool first = kb == 0;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                  const uint64_t adv = (uint64_t)(k * 2);   // 8 tf32 = 32 bytes = 2 x 16 B
                  umma_tf32(d, x_hi + adv, t_all + adv, idesc128, (first && k == 0) ? 0u : 1u);
                  umma_tf32(d, x_lo + adv, t_all + adv, idesc64, 1u);
                }
                tc_commit(&empty_bar[s]);
              }
            tc_commit(&tmem_full_bar[mt]);
          }
        }
    }
  } else {   // ===== epilogue warps 0..7: TMEM lane quarter = warp & 3, half = warp >> 2 (0: real part, 1: imaginary) =====
    const int q = warp & 3, half = warp >> 2;
    uint8_t* pl_hi = planes;
    uint8_t* pl_lo = planes + 64 * 128;       // lo rows start 64 rows further down inside every k-block
    const int rb = half * 32;                 // plane row base: T_r rows 0-31, T_i rows 32-63
    uint32_t gph = 0;
    float P[2][32];
    for (int w = blockIdx.x; w < g.nw; w += gridDim.x) {
      float* phi_w = reinterpret_cast<float*>(g.phi + (size_t)w * M * nt);
      // phase-0 operand: planes <- Phi_w  (row b = walker column, column j = basis index)
      for (int e = (warp & 3) * 32 + lane; e < M * nt; e += 128) {
        const int b = e / M, j = e - b * M;     // lanes along j: conflict-free plane writes
        float hi, lo;
        tf32_split(phi_w[2 * (j * nt + b) + half], hi, lo);
        const uint32_t o = plane_off(rb + b, j);
        *reinterpret_cast<float*>(pl_hi + o) = hi;
        *reinterpret_cast<float*>(pl_lo + o) = lo;
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&b_ready_bar)) : "memory");
      for (int ph = 0; ph < nphase; ++ph, ++gph) {
        const bool last_phase = ph == nphase - 1;
        const float scale = (ph >= 1 && ph <= g.K) ? 1.0f / (float)ph : 1.0f;
        const bool cxp = ph >= 1 && ph <= g.K;
        const uint32_t tl = tmem + ((uint32_t)(q * 32) << 16);
        float vv[2][32];
        // pass 1 (tile 0 overlaps the MMAs of tile 1): D_re = D1[0:32] - D2[32:64], D_im = D1[32:64] + D2[0:32],
        // summed over the accumulation chunks; scale, add into the running sum
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          if (mt < mtiles) {
            mbar_wait(&tmem_full_bar[mt], gph & 1);
            tc_fence_after();
#pragma unroll
            for (int b = 0; b < 32; ++b) vv[mt][b] = 0.f;
            {
              float u[32];
              tmem_ld32(tl + (mt * 2 + 0) * 128 + half * 32, u);              // X_r: hi*hi + lo*hi
#pragma unroll
              for (int b = 0; b < 32; ++b) vv[mt][b] += u[b];
              tmem_ld32(tl + (mt * 2 + 0) * 128 + 64 + half * 32, u);         // X_r: hi*lo
#pragma unroll
              for (int b = 0; b < 32; ++b) vv[mt][b] += u[b];
              if (cxp) {
                tmem_ld32(tl + (mt * 2 + 1) * 128 + (1 - half) * 32, u);
#pragma unroll
                for (int b = 0; b < 32; ++b) vv[mt][b] = half ? vv[mt][b] + u[b] : vv[mt][b] - u[b];
                tmem_ld32(tl + (mt * 2 + 1) * 128 + 64 + (1 - half) * 32, u);
#pragma unroll
                for (int b = 0; b < 32; ++b) vv[mt][b] = half ? vv[mt][b] + u[b] : vv[mt][b] - u[b];
              }
            }
#pragma unroll
            for (int b = 0; b < 32; ++b) {
              float t = vv[mt][b] * scale;
              if (ph == 0) P[mt][b] = t; else P[mt][b] += t;
              if (ph == g.K) t = P[mt][b];               // operand of the closing E_h product is the sum
              vv[mt][b] = t;
            }
          }
        }
        // pass 2: every MMA of this phase has completed, the T planes may be overwritten
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          if (mt < mtiles) {
            const int i = mt * 128 + q * 32 + lane;     // output row = basis index
            if (i < M) {
              if (last_phase) {
#pragma unroll
                for (int b = 0; b < 32; ++b)
                  if (b < nt) phi_w[2 * (i * nt + b) + half] = vv[mt][b];
              } else {
#pragma unroll
                for (int b = 0; b < 32; ++b) {
                  if (b < nt) {
                    float hi, lo;
                    tf32_split(vv[mt][b], hi, lo);
                    const uint32_t o = plane_off(rb + b, i);
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
