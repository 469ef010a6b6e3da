// taylor_tc.cuh -- H7 on the tensor pipe: Phi' = E_h [sum_{k<=K} A^k/k!] E_h Phi  (R3, R9).
// Persistent CTAs, one walker at a time.  Every product X * T (X = D_h = E_h - 1 real, or A_w complex symmetric; T complex
// M x N_t) is a set of real tcgen05.mma.kind::tf32 products with the 3xTF32 split:
//     D1 = X_r [T_r | T_i] ,  D2 = X_i [T_r | T_i];  D_re = D1[0:32] - D2[32:64],  D_im = D1[32:64] + D2[0:32]
//     are combined by the epilogue warps.  X_hi [T_hi | T_lo] is ONE N = 128 MMA (columns 0-63: hi*hi, 64-127: hi*lo) and
//     X_lo T_hi one N = 64 MMA into columns 64-127 (the cross terms share an accumulator; the epilogue adds the halves).
// a-operand: X is stored ONCE, in FP32 (A_w as the assembly GEMM wrote it).  128-row x 32-column tiles are streamed by TMA
//            through a ring of NF stages; the tensor pipe ignores the low 13 mantissa bits of a kind::tf32 operand (measured:
//            feeding raw FP32 as the hi operand is exact), so the raw tile IS X_hi = trunc(X), and two "splitter" warps
//            write X_lo = rn_tf32(X - trunc(X)) into one of NL lo buffers (same swizzled offsets, elementwise).  Against
//            storing hi / lo planes in HBM this halves the bytes A_w costs everywhere: the assembly epilogue's stores, the
//            Taylor kernel's HBM and L2 reads, and the set of live walkers (148 x 320 KB) now fits the L2, so passes 2-6
//            over A_w hit it (measured before: the TMA stream alone, MMAs off, took 1.0 ms of the kernel's 1.6).
// b-operand: T K-major in shared memory, per 32-column k-block 128 rows: [T_r, T_i (hi) | T_r, T_i (lo)],
//            rewritten by the epilogue warps after every Taylor term (generic -> async proxy fence);
// accumulators: TMEM, 128 columns per (128-row tile, plane).  The running sum P lives in registers.
// Supported: M <= 256, N_t <= 32 (else the SIMT kernel of taylor.cuh runs).
#pragma once
#include "gemm_tf32.cuh"

namespace afq {
namespace tt {

using namespace tc;

#ifndef TAYLOR_NL
#define TAYLOR_NL 3
#endif
#ifndef TAYLOR_NGROUP
#define TAYLOR_NGROUP 3
#endif
enum { NL = TAYLOR_NL, TILE_BYTES = 128 * 128, PLANE_KB_BYTES = 128 * 128, EPW = 8, NSPLIT = 6, NGROUP = TAYLOR_NGROUP, WPG = NSPLIT / NGROUP, NTHREADS = 16 * 32 };
// NSPLIT <= NL <= NF: a parity wait on an mbarrier is only unambiguous within one phase of it.  A splitter that has finished
// tile it - NSPLIT knows the MMAs of tile it - NSPLIT - NL are done; its wait for the lo buffer of tile `it` needs those of tile
// it - 2 NL done (a warp that runs two phases ahead sees the parity it waits for as already complete and reads a tile that has
// not landed -- seen as a hang: the producer's next expect_tx then over-arrives on the full barrier).
// 16 warps: the two epilogue warpgroups take 200 registers per thread, the producer / MMA / splitter warpgroups 56 (setmaxnreg)
enum { REGS_EPI = 200, REGS_AUX = 56 };
// warp roles: 0..EPW-1 epilogue, then the splitters, then the TMA producer, and the MMA issuer LAST: the warp scheduler favours the
// highest warp id of a sub-partition, and the MMA warp's few instructions between two tiles are the kernel's critical path
enum { W_SPLIT0 = EPW, W_PROD = EPW + NSPLIT, W_MMA = EPW + NSPLIT + 1 };
static_assert(W_MMA == 15, "16 warps");

struct TaylorMaps {
  CUtensorMap A[2];   // [0: 128-row box, 1: last-tile box] over Abuf viewed as [N_w*M][2*MP] FP32
  CUtensorMap E[2];   // same for D_h = E_h - 1 [M][MP] FP32
};

struct TaylorTcArgs {
  int M, MP, nt, K, nw;
  int mtiles, rows_last, nkb;   // 128-row tiles, rows of the last one (multiple of 8), 32-column k-blocks
  int nf;                       // FP32 tile stages in the TMA ring (what shared memory leaves: 5, or 4 at nkb = 8)
  cplx<float>* phi;             // [nw][M][nt] in/out
};

enum { NF_MAX = 6 };
static_assert(NGROUP <= NL && NSPLIT == WPG * NGROUP, "see above");
inline int pick_nf(int nkb) {   // >= NL (the splitters' wait order relies on it)
  const int left = 227 * 1024 - 1024 - 512 - nkb * PLANE_KB_BYTES - NL * TILE_BYTES;
  const int nf = left / TILE_BYTES;
  return nf > NF_MAX ? NF_MAX : nf;
}
inline size_t smem_bytes(int nkb) { return (size_t)nkb * PLANE_KB_BYTES + (size_t)(pick_nf(nkb) + NL) * TILE_BYTES + 1024; }

// byte offset of element (row b in 0..127, column j) inside the K-major SWIZZLE_128B T operand
__device__ __forceinline__ uint32_t plane_off(int b, int j) {
  const int kb = j >> 5, jj = j & 31;
  return (uint32_t)(kb * PLANE_KB_BYTES + b * 128 + ((((jj >> 2) ^ (b & 7)) << 4) | ((jj & 3) << 2)));
}

// Staged result [M][nt] complex inside the planes: only the non-padding rows of the first k-blocks are used (chunks of
// nt plane rows x 128 B = 16 result rows of nt complex, 4 chunks per k-block), so the zero padding the MMAs rely on is
// never touched.  Needs ceil(M / 16) <= 4 * floor(M / 32) (true for M >= 64).
__device__ __forceinline__ uint32_t stage_chunk(int c) { return (uint32_t)((c >> 2) * PLANE_KB_BYTES + (c & 3) * (32 * 128)); }
__device__ __forceinline__ uint32_t stage_row(int i, int nt) { return stage_chunk(i >> 4) + (uint32_t)((i & 15) * nt * 8); }
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void sts128(uint32_t a, uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void sts32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ float2 lds64(uint32_t a) {
  float2 v;
  asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(a) : "memory");
  return v;
}
// staged result -> global, 16-row chunks are contiguous on both sides
__device__ __forceinline__ void stage_flush(uint32_t pl, float2* dst, int M, int nt, int et) {
  const int per = 16 * nt;
  for (int c = 0; c * 16 < M; ++c) {
    const int n = min(16, M - c * 16) * nt;
    const uint32_t base = pl + stage_chunk(c);
    for (int idx = et; idx < n; idx += EPW * 32) dst[c * per + idx] = lds64(base + idx * 8);
  }
}
enum { MAXE = 32 };   // complex elements of Phi_w per epilogue thread: M * N_t <= 256 * 32 = MAXE * 256

__global__ void __launch_bounds__(NTHREADS, 1) k_taylor_tc(const __grid_constant__ TaylorMaps maps, TaylorTcArgs g) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[NF_MAX];   // TMA has landed an FP32 tile (= X_hi)
  __shared__ __align__(8) uint64_t empty_bar[NF_MAX];  // the MMAs of the tile in this stage have completed (waited for by the producer AND by the splitter that reuses the tile's lo buffer)
  __shared__ __align__(8) uint64_t lo_full_bar[NL];    // both warps of a splitter group have written their half of X_lo
  __shared__ __align__(8) uint64_t tmem_full_bar[2];   // per 128-row tile: tile 0 is post-processed while tile 1 is issued
  __shared__ __align__(8) uint64_t b_ready_bar[2];     // per tile of the PREVIOUS product = 4 k-blocks of the T operand (8 warps arrive)
  __shared__ __align__(8) uint64_t t_free_bar[4];      // last tile has consumed k-block kb < 4 of the current T
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int M = g.M, nt = g.nt, nkb = g.nkb, mtiles = g.mtiles, NF = g.nf;
  const uint32_t plane_bytes = (uint32_t)nkb * PLANE_KB_BYTES;
  uint8_t* planes = smem;                                   // rows 0-31 T_r hi, 32-63 T_i hi, 64-95 T_r lo, 96-127 T_i lo
  uint8_t* stages = smem + (size_t)plane_bytes;             // NF FP32 tiles, then NL lo tiles
  uint8_t* lobufs = stages + (size_t)NF * TILE_BYTES;
  const int nphase = g.K + 2;
  const uint32_t tmem_cols = 512u;

  // zero the planes once (rows >= nt and columns >= M must stay 0 for the whole kernel) and the tile buffers (rows past a
  // short last tile are never written by TMA and must not hold NaN patterns)
  for (uint32_t o = threadIdx.x * 16; o < plane_bytes + (uint32_t)(NF + NL) * TILE_BYTES; o += NTHREADS * 16)
    *reinterpret_cast<uint4*>(planes + o) = make_uint4(0, 0, 0, 0);
  if (warp == W_PROD && lane == 0) {
    for (int s = 0; s < NF_MAX; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
    for (int s = 0; s < NL; ++s) mbar_init(&lo_full_bar[s], WPG);   // the warps of a splitter group
    mbar_init(&tmem_full_bar[0], 1); mbar_init(&tmem_full_bar[1], 1);
    mbar_init(&b_ready_bar[0], EPW); mbar_init(&b_ready_bar[1], EPW);
    for (int x = 0; x < 4; ++x) mbar_init(&t_free_bar[x], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == W_MMA) {
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
  // tiles of this CTA: every (walker, phase, tile, k-block, plane), in this order in all three pipeline roles
  const int n_mine = blockIdx.x < g.nw ? (g.nw - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
  const uint32_t tiles_per_walker = (uint32_t)(mtiles * nkb) * (uint32_t)(2 * g.K + 2);

  if (warp == W_PROD) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"((int)REGS_AUX));
    if (lane == 0) {   // ===== TMA producer: streams FP32 X tiles =====
      int s = 0;
      uint32_t par = 1;
      for (int w = blockIdx.x; w < g.nw; w += gridDim.x)
        for (int ph = 0; ph < nphase; ++ph) {
          const bool cx = ph >= 1 && ph <= g.K;           // complex A_w, else real D_h
          for (int mt = 0; mt < mtiles; ++mt) {
            const int last = mt == mtiles - 1;
            const uint32_t bytes = (uint32_t)(last ? g.rows_last : 128) * 128u;
            for (int kb = 0; kb < nkb; ++kb)
              for (int p = 0; p < (cx ? 2 : 1); ++p) {
                mbar_wait(&empty_bar[s], par);
                uint8_t* st = stages + (size_t)s * TILE_BYTES;
                mbar_expect_tx(&full_bar[s], bytes);
                if (cx) tma_load_2d(st, &maps.A[last], &full_bar[s], p * g.MP + kb * 32, w * M + mt * 128);
                else tma_load_2d(st, &maps.E[last], &full_bar[s], kb * 32, mt * 128);
                if (++s == NF) { s = 0; par ^= 1; }
              }
          }
        }
    }
  } else if (warp >= W_SPLIT0 && warp < W_PROD) {
    // ===== splitter warps: X_lo = (X - trunc13 X)(1 + 2^-11), elementwise at the same (swizzled) offsets.  NGROUP groups of two
    // warps take the tiles round robin (group = tile mod NGROUP <= NL, see above), each warp one half of the tile: the chain
    // "MMAs of tile it - NL done -> split tile it -> MMAs of tile it" is what paces the kernel, and two warps halve its split part =====
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"((int)REGS_AUX));
    const int sw = warp - W_SPLIT0, grp = sw / WPG, half = sw % WPG;
    const uint32_t total = (uint32_t)n_mine * tiles_per_walker;
    // (phase, index inside the phase) of this group's current tile; a phase is [m-tile 0 | m-tile 1], each nkb x planes tiles
    // (mtiles == 1: half_len is unused)
    int ph = 0, half_len = nkb, rr = grp;
    const int slabs_last = (g.rows_last + 15) >> 4;
    if (mtiles == 2) while (rr >= 2 * half_len) { rr -= 2 * half_len; ++ph; half_len = nkb * ((ph >= 1 && ph <= g.K) ? 2 : 1); }
    for (uint32_t it = grp; it < total; it += NGROUP) {
      const int s = it % NF, sl = it % NL;
      // lo buffer sl was last read by the MMAs of tile it - NL, whose completion is the (only) tcgen05.commit of that tile, on the
      // empty barrier of ITS stage: no separate barrier (a commit costs ~50 clk of tensor-pipe time, the pipe has no queue).
      // Order matters: a parity wait is only unambiguous within one phase of the barrier.  Tile it - NL done means every tile
      // up to it - NL has been loaded, and NL <= NF: the previous user of stage s is among them, so full_bar[s] is exactly in
      // the phase this tile completes; and empty_bar[(it - NL) % NF] cannot be a phase further on, because tile it - NL + NF > it
      // is issued after tile `it`, which needs this group's lo buffer.
      if (it >= NL) mbar_wait(&empty_bar[(it - NL) % NF], ((it - NL) / NF) & 1);
      mbar_wait(&full_bar[s], (it / NF) & 1);
      // the two warps take alternate 16-row slabs (2 KB = 4 warp-wide 16-byte accesses); a short last tile (rows_last of 128 rows,
      // M = 200: 72) has only ceil(rows_last / 16) of them: TMA wrote nothing beyond and the MMAs' extra rows are never read back
      // explicit shared-space accesses (LDS.128 / STS.128): through generic pointers ptxas emitted LD.E.128 / ST.E.128
      const uint32_t src = smem_u32(stages + (size_t)s * TILE_BYTES) + lane * 16;
      const uint32_t dst = smem_u32(lobufs + (size_t)sl * TILE_BYTES) + lane * 16;
      const int slabs = (mtiles == 2 && rr >= half_len) ? slabs_last : 8;     // second m-tile of its phase?
#pragma unroll 1
      for (int sb = half; sb < slabs; sb += 2 * WPG) {       // two slabs (sb, sb + WPG) per iteration: 8 accesses in flight
        uint4 v[8];
        const bool two = sb + WPG < slabs;
#pragma unroll
        for (int x = 0; x < 4; ++x) v[x] = lds128(src + (sb * 4 + x) * 512);
        if (two) {
#pragma unroll
          for (int x = 0; x < 4; ++x) v[4 + x] = lds128(src + ((sb + WPG) * 4 + x) * 512);
        }
#pragma unroll
        for (int x = 0; x < 4; ++x) {
          uint4 q;
          q.x = tf32_lo_bits(v[x].x); q.y = tf32_lo_bits(v[x].y); q.z = tf32_lo_bits(v[x].z); q.w = tf32_lo_bits(v[x].w);
          sts128(dst + (sb * 4 + x) * 512, q);
        }
        if (two) {
#pragma unroll
          for (int x = 0; x < 4; ++x) {
            uint4 q;
            q.x = tf32_lo_bits(v[4 + x].x); q.y = tf32_lo_bits(v[4 + x].y); q.z = tf32_lo_bits(v[4 + x].z); q.w = tf32_lo_bits(v[4 + x].w);
            sts128(dst + ((sb + WPG) * 4 + x) * 512, q);
          }
        }
      }
      // advance (phase, index inside the phase) by NGROUP tiles without divisions
      rr += NGROUP;
      while (rr >= 2 * half_len) {
        rr -= 2 * half_len;
        if (++ph == nphase) ph = 0;
        half_len = nkb * ((ph >= 1 && ph <= g.K) ? 2 : 1);
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&lo_full_bar[sl])) : "memory");
    }
  } else if (warp == W_MMA) {
    // ===== MMA issuer warp.  The whole warp runs the loop (uniform control flow) and ONE elected lane issues: with the
    // descriptors computed under uniform control flow ptxas keeps them in uniform registers and the MMAs of a tile are
    // back-to-back UTCHMMA (inside an `if (lane == 0)` region it wraps every MMA in an ELECT / 5 x R2UR / branch-back sequence).
    // Measured (csrc/peaks.cuh k_peak_pat): a tile's 448 clk of pipe time, a tcgen05.commit (~50 clk) and a satisfied mbarrier
    // wait (~92 clk) add up -- the pipe does not run ahead of the issuing warp -- so there is one wait and one commit per tile.
    // Tried and dropped (B200, cfg 5): two issuer warps alternating tiles with a named-barrier hand-over (1.50 ms against 1.38);
    // two issuer warps each owning one plane's chain, no hand-over at all (1.43 ms against 1.38).  Trimming the last k-block to
    // the k-steps it really has (M = 200: 25 instead of 28 k-steps) removed 10 % of the MMAs and changed the time by 0.3 %:
    // the tensor pipe is not what paces this kernel -- the chain TMA -> splitter -> MMA over a 3-deep lo ring is. =====
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"((int)REGS_AUX));
    constexpr uint32_t idesc128 = make_idesc(128, 128), idesc64 = make_idesc(128, 64);
    const uint64_t xh0 = make_desc(smem_u32(stages)), xl0 = make_desc(smem_u32(lobufs)), t0 = make_desc(smem_u32(planes));
    constexpr uint64_t TSTEP = TILE_BYTES >> 4;     // descriptor address field counts 16-byte units
    const int klast = (M - 32 * (nkb - 1) + 7) >> 3;     // k-steps of 8 columns the last k-block really has (columns >= M are padding)
    uint64_t xh = xh0, xl = xl0;
    uint32_t gph = 0;
    int s = 0, sl = 0;
    uint32_t lpar = 0;
    for (int w = blockIdx.x; w < g.nw; w += gridDim.x)
      for (int ph = 0; ph < nphase; ++ph, ++gph) {
        const int np = (ph >= 1 && ph <= g.K) ? 2 : 1;
        for (int mt = 0; mt < mtiles; ++mt) {
          uint64_t t_all = t0;                       // k-block kb of T: 128 rows (hi then lo); its first 64 rows = T_hi
          for (int kb = 0; kb < nkb; ++kb, t_all += TSTEP) {
            // k-blocks 4 j .. 4 j + 3 of this phase's T are in shared memory, and (all 8 epilogue warps arrive after their
            // TMEM loads) the accumulators of tile j have been read
            if (mt == 0 && (kb & 3) == 0) mbar_wait(&b_ready_bar[kb >> 2], gph & 1);
            const int kn = kb == nkb - 1 ? klast : 4;
            for (int p = 0; p < np; ++p) {
              {
                const uint32_t d = tmem + (mt * 2 + p) * 128;
                mbar_wait(&lo_full_bar[sl], lpar);     // the splitter arrives after it has seen the TMA tile: X_hi is in place too
                tc_fence_after();
                if (elect_one()) {
#pragma unroll
                  for (int k = 0; k < 4; ++k) {
                    if (k < kn) {
                      const uint64_t adv = (uint64_t)(k * 2);   // 8 tf32 = 32 bytes = 2 x 16 B
                      umma_tf32(d, xh + adv, t_all + adv, idesc128, (kb == 0 && k == 0) ? 0u : 1u);
                      // X_lo T_hi joins the other cross term in columns 64-127: the large hi*hi accumulator of columns 0-63 then
                      // sees half as many (truncating) accumulations, the small cross-term accumulator's truncation is 2^-11 down
                      umma_tf32(d + 64, xl + adv, t_all + adv, idesc64, 1u);
                    }
                  }
                  tc_commit(&empty_bar[s]);
                }
                __syncwarp();
              }
              xh += TSTEP; xl += TSTEP;
              if (++s == NF) { s = 0; xh = xh0; }
              if (++sl == NL) { sl = 0; xl = xl0; lpar ^= 1; }
            }
            // this warp's chain (or, in a real phase, its empty share) has passed k-block kb of tile mt
            if ((mtiles == 2 && mt == 1 && kb < 4) || kb == nkb - 1) {
              if (elect_one()) {
                if (mtiles == 2 && mt == 1 && kb < 4) tc_commit(&t_free_bar[kb]);
                if (kb == nkb - 1) tc_commit(&tmem_full_bar[mt]);
              }
              __syncwarp();
            }
          }
        }
      }
  } else if (warp < EPW) {   // ===== epilogue warps 0..7: TMEM lane quarter = warp & 3, half = warp >> 2 (0: real part, 1: imaginary) =====
    // Rows i = mt*128 + q*32 + lane of the product are k-block mt*4+q of the next T operand.  Tile 0 is post-processed
    // and written back while tile 1 is being issued (each k-block as soon as tile 1 has consumed it), and the next
    // phase starts on k-blocks 0-3 while tile 1 is post-processed: the tensor pipe does not wait between phases.
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"((int)REGS_EPI));
    const int q = warp & 3, half = warp >> 2;
    const uint32_t plu = smem_u32(planes);
    const uint32_t pl_hi = plu, pl_lo = plu + 64 * 128;   // lo rows start 64 rows further down inside every k-block
    const int rb = half * 32;                 // plane row base: T_r rows 0-31, T_i rows 32-63
    uint32_t gph = 0;
    float P[2][32];
    const int et = (int)threadIdx.x;      // epilogue threads are 0..255
    int w_last = -1;
    for (int w = blockIdx.x; w < g.nw; w += gridDim.x) {
      float* phi_w = reinterpret_cast<float*>(g.phi + (size_t)w * M * nt);
      // phase-0 operand: planes <- Phi_w (row b = walker column, column i = basis index).  Phi_w is read as
      // consecutive complex numbers (coalesced, all loads in flight at once); every MMA of the previous walker has
      // completed (each warp has observed tmem_full of its last tile)
      {
        // The next walker of this CTA is pulled into L2 now, a whole walker ahead: its first touch would otherwise be a DRAM round trip on
        // the critical path (nothing else runs on this SM between two walkers).
        float2 f[MAXE / 2];
        const float2* src = reinterpret_cast<const float2*>(phi_w);
#pragma unroll
        for (int k = 0; k < MAXE / 2; ++k) {
          const int e = et + k * (EPW * 32);
          if (e < M * nt) f[k] = src[e];
        }
        if (w + (int)gridDim.x < g.nw) {
          const char* nxt = reinterpret_cast<const char*>(g.phi + (size_t)(w + gridDim.x) * M * nt);
          for (int o = et * 128; o < M * nt * 8; o += EPW * 32 * 128) asm volatile("prefetch.global.L2 [%0];" ::"l"(nxt + o));
        }
        if (w != (int)blockIdx.x) {
          // the previous walker's result is staged in the planes: write it out before they are overwritten
          asm volatile("bar.sync 1, 256;" ::: "memory");
          float2* dst = reinterpret_cast<float2*>(g.phi + (size_t)(w - gridDim.x) * M * nt);
          stage_flush(plu, dst, M, nt, et);
          asm volatile("bar.sync 1, 256;" ::: "memory");
        }
        int ci = et / nt, cbb = et - ci * nt;            // (row, column) of element e, stepped without divisions
        const int di = (EPW * 32) / nt, db = (EPW * 32) - di * nt;
#pragma unroll
        for (int hb = 0; hb < 2; ++hb) {
          if (hb == 1) {
#pragma unroll
            for (int k = 0; k < MAXE / 2; ++k) {
              const int e = et + (k + MAXE / 2) * (EPW * 32);
              if (e < M * nt) f[k] = src[e];
            }
          }
#pragma unroll
          for (int k = 0; k < MAXE / 2; ++k) {
            const int e = et + (k + hb * (MAXE / 2)) * (EPW * 32);
            if (e < M * nt) {
              const float2 fv = f[k];
              float h0, l0, h1, l1;
              tf32_split_raw(fv.x, h0, l0);     // hi = raw FP32 (the pipe truncates it), lo = centred low part
              tf32_split_raw(fv.y, h1, l1);
              const uint32_t o = plane_off(cbb, ci);
              sts32(pl_hi + o, h0);
              sts32(pl_lo + o, l0);
              sts32(pl_hi + o + 32 * 128, h1);    // T_i rows are 32 rows below the T_r rows
              sts32(pl_lo + o + 32 * 128, l1);
            }
            ci += di; cbb += db;
            if (cbb >= nt) { cbb -= nt; ++ci; }
          }
          // the first half holds the elements e < 4096, i.e. basis indices i < 4096 / N_t >= 128 (N_t <= 32): k-blocks 0-3 are
          // complete and the MMA warp can start on the first m-tile while the rest is being written
          asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
          tc_fence_before();
          asm volatile("bar.sync 1, 256;" ::: "memory");
          if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&b_ready_bar[hb])) : "memory");
        }
      }
      for (int ph = 0; ph < nphase; ++ph, ++gph) {
        const bool last_phase = ph == nphase - 1;
        const float scale = (ph >= 1 && ph <= g.K) ? 1.0f / (float)ph : 1.0f;
        const bool cxp = ph >= 1 && ph <= g.K;
        const uint32_t tl = tmem + ((uint32_t)(q * 32) << 16);
#pragma unroll
        for (int mt = 0; mt < 2; ++mt) {
          if (mt < mtiles) {
            // D_re = D1[0:32] - D2[32:64], D_im = D1[32:64] + D2[0:32]; columns 64.. hold the hi*lo products
            float v[32];
            mbar_wait(&tmem_full_bar[mt], gph & 1);
            tc_fence_after();
            {
              float u0[32], u1[32];
              tmem_ld32x2(tl + (mt * 2 + 0) * 128 + half * 32, tl + (mt * 2 + 0) * 128 + 64 + half * 32, u0, u1);
#pragma unroll
              for (int b = 0; b < 32; ++b) v[b] = u0[b] + u1[b];
              if (cxp) {
                // (single loads here: a second pair in flight would not fit the 168-register budget beside P)
                tmem_ld32(tl + (mt * 2 + 1) * 128 + (1 - half) * 32, u0);
#pragma unroll
                for (int b = 0; b < 32; ++b) v[b] = half ? v[b] + u0[b] : v[b] - u0[b];
                tmem_ld32(tl + (mt * 2 + 1) * 128 + 64 + (1 - half) * 32, u0);
#pragma unroll
                for (int b = 0; b < 32; ++b) v[b] = half ? v[b] + u0[b] : v[b] - u0[b];
              }
            }
            const int i = mt * 128 + q * 32 + lane;       // output row = basis index
            if (ph == 0) {
              // the streamed operand of the two one-body phases is D_h = E_h - 1 (|D_h| ~ dt |h'| / 2 << 1): E_h T = T + D_h T
              // with the addition in FP32 round-to-nearest here, so the tensor pipe's truncating accumulation acts on the
              // small correction only.  T (= Phi_w) is read back from the hi plane (raw FP32), before this thread overwrites it
              const int ic = i < M ? i : 0;
#pragma unroll
              for (int b = 0; b < 32; ++b)
                if (b < nt) {
                  const uint32_t o = plane_off(rb + b, ic);
                  float th;
                  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(th) : "r"(pl_hi + o) : "memory");
                  v[b] += th;                 // the hi plane holds the raw FP32 value (tf32_split_raw)
                }
            }
#pragma unroll
            for (int b = 0; b < 32; ++b) {
              float t = v[b] * scale;
              if (last_phase) t += P[mt][b];              // E_h P = P + D_h P
              else if (ph == 0) P[mt][b] = t;
              else P[mt][b] += t;
              if (ph == g.K) t = P[mt][b];               // operand of the closing E_h product is the sum
              v[b] = t;
            }
            if (last_phase) {
              // result rows stay in registers (P is dead) until every MMA has completed, then go to the staging
              // area inside the planes (the non-padding bytes, all rewritten by the next walker's operand)
#pragma unroll
              for (int b = 0; b < 32; ++b) P[mt][b] = v[b];
              if (mt == mtiles - 1) {
#pragma unroll
                for (int m2 = 0; m2 < 2; ++m2) {
                  const int i2 = m2 * 128 + q * 32 + lane;
                  if (m2 < mtiles && i2 < M) {
                    const uint32_t srow = plu + stage_row(i2, nt) + half * 4;
#pragma unroll
                    for (int b = 0; b < 32; ++b)
                      if (b < nt) sts32(srow + b * 8, P[m2][b]);
                  }
                }
              }
            } else {
              float hi[32], lo[32];
#pragma unroll
              for (int b = 0; b < 32; ++b) tf32_split_raw(v[b], hi[b], lo[b]);
              // k-block mt*4+q of T may be overwritten once every MMA that reads it has completed: for the last
              // tile that is tmem_full (above), for tile 0 of two the last tile's pass over that k-block
              if (mt == 0 && mtiles == 2) mbar_wait(&t_free_bar[q], gph & 1);
              if (i < M) {
#pragma unroll
                for (int b = 0; b < 32; ++b)
                  if (b < nt) {
                    const uint32_t o = plane_off(rb + b, i);
                    sts32(pl_hi + o, hi[b]);
                    sts32(pl_lo + o, lo[b]);
                  }
              }
              asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
              tc_fence_before();
              __syncwarp();
              if (lane == 0)
                asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&b_ready_bar[mt])) : "memory");
            }
          }
        }
      }
      w_last = w;
    }
    if (w_last >= 0) {   // the last walker's result is still staged
      asm volatile("bar.sync 1, 256;" ::: "memory");
      float2* dst = reinterpret_cast<float2*>(g.phi + (size_t)w_last * M * nt);
      stage_flush(plu, dst, M, nt, et);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == W_MMA) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(tmem_cols) : "memory");
  }
}

}  // namespace tt
}  // namespace afq
