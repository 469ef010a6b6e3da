// gemm_tf32.cuh -- tcgen05 / TMEM / TMA "NT" GEMM with the 3xTF32 operand split (sm_100a only).
//   C[m][n] = sum_k A[m][k] B[n][k],  A = A_hi + A_lo, B = B_hi + B_lo (each plane exactly TF32),
//   C ~= A_lo B_hi + A_hi B_lo + A_hi B_hi  accumulated in FP32 in TMEM (error ~ 2^-22, DESIGN.md
//   "Precision split").  Operands are K-major FP32 planes in HBM, moved by TMA (128B swizzle) into a
//   2-stage shared-memory ring; one elected thread issues tcgen05.mma.kind::tf32 (M=128, N=256, K=8);
//   four epilogue warps read the 128 x 256 accumulator with tcgen05.ld and apply the fused epilogue.
// Used for H4 (force bias), H6 (operator assembly), H9 (energy): PAPER.md:59, :80, :87.
// Three kernels: k_gemm_tf32 (one CTA per 128 x 256 tile, gemm_path 2), k_gemm_tf32_pair (one cta_group::2 pair per
// 256 x 256 tile pair: the multi-determinant TT GEMM and fallbacks) and k_gemm_tf32_pair_ps (persistent pairs, 16 warps:
// H6 with its tile handed to dedicated store warps; H4 and H9 with both spins in one launch over host-built tile lists).
#pragma once
#include <cuda.h>
#include "common.cuh"

namespace afq {
namespace tc {

enum { BM = 128, BN = 256, BK = 32, STAGES = 2, UMMA_K = 8, TMEM_COLS = 512, THREADS = 320 };
// The tensor pipe adds into its FP32 accumulator with truncation, so the error of one long accumulation grows
// linearly with K (measured 6.4e-9 per K element: 1.7e-5 at K = 2600).  The accumulation is therefore cut into
// chunks of CHUNK_KB k-blocks (128 K elements); each chunk lands in one of two TMEM buffers and is added to a
// running FP32 sum in registers (round-to-nearest) by the epilogue warps while the next chunk is being issued.
enum { CHUNK_KB = 4, EPI_WARPS = 8, COLS_PER_WARP = BN / 2 };
enum { A_BYTES = BM * BK * 4, B_BYTES = BN * BK * 4, STAGE_BYTES = 2 * A_BYTES + 2 * B_BYTES };
enum { SMEM_BYTES = STAGES * STAGE_BYTES + 1024 };
enum { B_BOX = 128 };   // rows per TMA box of the b-operand maps

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n.reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}
// one lane of a fully active warp (the same one every time)
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
               : "memory");
}
// D[tmem] (+)= A[smem] * B[smem], kind::tf32, one CTA
__device__ __forceinline__ void umma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
      : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem] (TS mode): A = 128 lanes (rows) x 8 consecutive 32-bit columns (the K elements)
__device__ __forceinline__ void umma_tf32_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n}"
      ::"r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(acc)
      : "memory");
}
// 32 registers of this thread -> its TMEM lane, 32 consecutive columns; waits for the store to complete
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&a)[32]) {
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
// ---- CTA pair (cta_group::2) forms.  Shared-window addresses of the two CTAs of a pair differ in bit 24; clearing
// it addresses the even (leader) CTA's copy of the same variable.
constexpr uint32_t PEER_MASK = 0xFEFFFFFFu;
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// TMA load into this CTA's shared memory, transaction bytes counted on the LEADER CTA's mbarrier
__device__ __forceinline__ void tma_load_2d_pair(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar) & PEER_MASK), "r"(c0), "r"(c1)
      : "memory");
}
// the same with an L2 eviction-priority hint (createpolicy encodings: whole-fraction evict_first / evict_last)
constexpr uint64_t L2_EVICT_FIRST = 0x12F0000000000000ull, L2_EVICT_LAST = 0x14F0000000000000ull;
__device__ __forceinline__ void tma_load_2d_pair_hint(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.tensor.2d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4}], [%2], %5;"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar) & PEER_MASK), "r"(c0), "r"(c1), "l"(pol)
      : "memory");
}
// arrive on the same barrier in both CTAs of the pair once all MMAs issued so far have completed
__device__ __forceinline__ void tc_commit_pair(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(smem_u32(bar)), "h"((uint16_t)3)
               : "memory");
}
// arrive on the leader CTA's copy of a barrier.  Default semantics (release at CTA scope): the arrive only hands a drained
// TMEM buffer back (ordered by tcgen05.fence::before_thread_sync), no generic-memory data travels with it; the
// .release.cluster form costs a MEMBAR.ALL.GPU + ERRBAR per arrive (measured: 1650 clk each, 18 % of the epilogue warps' time).
__device__ __forceinline__ void mbar_arrive_leader(uint64_t* bar) {
  asm volatile(
      "{\n.reg .b32 ra;\nmapa.shared::cluster.u32 ra, %0, 0;\nmbarrier.arrive.shared::cluster.b64 _, [ra];\n}"
      ::"r"(smem_u32(bar))
      : "memory");
}
// D[tmem of both CTAs] (+)= A * B with M = 256 (128 rows per CTA), the N rows of B split between the two CTAs
__device__ __forceinline__ void umma_tf32_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t acc) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::tf32 [%0], %1, %2, %3, p;\n}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(acc)
      : "memory");
}
// K-major, SWIZZLE_128B shared-memory matrix descriptor (rows 128 B apart, 8-row atoms 1024 B apart)
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3FFFF) >> 4);          // start address, bits [0,14)
  d |= (uint64_t)1 << 16;                           // leading byte offset (unused for swizzled K-major), bits [16,30)
  d |= (uint64_t)(1024 >> 4) << 32;                 // stride byte offset = 1024 B, bits [32,46)
  d |= (uint64_t)1 << 46;                           // descriptor version (sm_100)
  d |= (uint64_t)2 << 61;                           // layout type SWIZZLE_128B
  return d;
}
// instruction descriptor: FP32 accumulate, TF32 x TF32, both K-major, M x N
__host__ __device__ constexpr uint32_t make_idesc(int M, int N) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// 32 lanes x 32 columns of FP32 accumulators -> 32 registers per thread (thread = TMEM lane)
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}

// two 32-column loads in flight, one wait (the load latency is paid once)
__device__ __forceinline__ void tmem_ld32x2(uint32_t ta, uint32_t tb, float (&va)[32], float (&vb)[32]) {
  uint32_t ra[32], rb[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%64];\n"
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63}, [%65];\n"
      "tcgen05.wait::ld.sync.aligned;"
      : "=r"(ra[0]), "=r"(ra[1]), "=r"(ra[2]), "=r"(ra[3]), "=r"(ra[4]), "=r"(ra[5]), "=r"(ra[6]), "=r"(ra[7]), "=r"(ra[8]), "=r"(ra[9]), "=r"(ra[10]), "=r"(ra[11]), "=r"(ra[12]), "=r"(ra[13]), "=r"(ra[14]), "=r"(ra[15]), "=r"(ra[16]), "=r"(ra[17]), "=r"(ra[18]), "=r"(ra[19]), "=r"(ra[20]), "=r"(ra[21]), "=r"(ra[22]), "=r"(ra[23]), "=r"(ra[24]), "=r"(ra[25]), "=r"(ra[26]), "=r"(ra[27]), "=r"(ra[28]), "=r"(ra[29]), "=r"(ra[30]), "=r"(ra[31]),
        "=r"(rb[0]), "=r"(rb[1]), "=r"(rb[2]), "=r"(rb[3]), "=r"(rb[4]), "=r"(rb[5]), "=r"(rb[6]), "=r"(rb[7]), "=r"(rb[8]), "=r"(rb[9]), "=r"(rb[10]), "=r"(rb[11]), "=r"(rb[12]), "=r"(rb[13]), "=r"(rb[14]), "=r"(rb[15]), "=r"(rb[16]), "=r"(rb[17]), "=r"(rb[18]), "=r"(rb[19]), "=r"(rb[20]), "=r"(rb[21]), "=r"(rb[22]), "=r"(rb[23]), "=r"(rb[24]), "=r"(rb[25]), "=r"(rb[26]), "=r"(rb[27]), "=r"(rb[28]), "=r"(rb[29]), "=r"(rb[30]), "=r"(rb[31])
      : "r"(ta), "r"(tb)
      : "memory");
#pragma unroll
  for (int i = 0; i < 32; ++i) { va[i] = __uint_as_float(ra[i]); vb[i] = __uint_as_float(rb[i]); }
}

struct Maps {
  CUtensorMap a_hi, a_lo, b_hi, b_lo;   // 2-D {K, rows}, box {BK, BM} / {BK, BN}, SWIZZLE_128B
};


// ---- epilogues: called per epilogue thread with its accumulator row and 32 consecutive columns -------------
// explicit shared-space accesses for the staging area (generic LD / ST cost an address-space check and a uniform
// descriptor each)
__device__ __forceinline__ float4 ld_s128(uint32_t a) {
  float4 v;
  asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ float ld_s32(uint32_t a) {
  float v;
  asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a));
  return v;
}
// 16-byte global store that asks L2 to evict the line first (streamed output, not read again by this kernel)
__device__ __forceinline__ void st_g128_hint(void* p, float4 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w),
               "l"(pol)
               : "memory");
}
__device__ __forceinline__ void st_s32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }

struct EpiStoreT {      // H4: out[col][row]
  static constexpr bool kStaged = false;
  float* out; int ldo, m_real, n_real;
  __device__ __forceinline__ void operator()(int r, int c0, const float (&v)[32]) const {
    if (r >= m_real) return;
#pragma unroll
    for (int j = 0; j < 32; ++j)
      if (c0 + j < n_real) out[(size_t)(c0 + j) * ldo + r] = v[j];
  }
};
// H6: col = 2w + p -> A[w][i][p][MP] (+ j); out_lo != null: TF32 hi / lo planes.
// blk == null: row = i*M + j (all M^2 elements).  blk != null: A_w is symmetric, only the 8 x 16 element blocks that
// touch the upper triangle are computed: row = block*128 + (i % 8)*16 + (j % 16), blk[block] = (i / 8, j / 16); lanes
// run along j (64-byte segments).  The lower triangle is filled afterwards by k_symmetrize (misc.cuh).
struct EpiAssemble {
  static constexpr bool kStaged = false;
  float* out; float* out_lo; const int2* blk; int M, MP, m_real, n_real;
  __device__ __forceinline__ void put(size_t o, float v) const {
    if (out_lo) {
      float hi, lo;
      tf32_split(v, hi, lo);
      out[o] = hi; out_lo[o] = lo;
    } else {
      out[o] = v;
    }
  }
  __device__ __forceinline__ void operator()(int r, int c0, const float (&v)[32]) const {
    if (r >= m_real) return;
    int ii, jj;
    if (blk) {
      const int2 b = blk[r >> 7];
      ii = b.x * 8 + ((r >> 4) & 7); jj = b.y * 16 + (r & 15);
      if (ii >= M || jj >= M) return;
    } else {
      ii = r / M; jj = r - ii * M;
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      const int c = c0 + j;
      if (c < n_real) {
        const size_t base = (size_t)(c >> 1) * M * (2 * MP) + (c & 1) * MP;
        put(base + (size_t)ii * (2 * MP) + jj, v[j]);
      }
    }
  }
};
// H6, symmetric and staged (M % 4 == 0): the 128 x 256 tile (one 8 x 16 block of (i, j) for 128 walkers x 2 planes)
// goes through the now idle stage memory, S[col][i%8][j%16], and leaves as 16-byte vectors in BOTH orientations:
// A[w][i][p][j..j+3] (64-byte runs) and A[w][j][p][i..i+3] (32-byte runs), so no separate symmetrize pass is needed.
struct EpiAssembleSym {
  static constexpr bool kStaged = true;
  float* out; float* out_lo; const int2* blk; int M, MP, n_real;
  uint64_t st_pol = 0x1000000000000000ull;   // L2 eviction priority of the persistent kernel's stores
  __device__ __forceinline__ void operator()(int, int, const float (&)[32]) const {}
  __device__ __forceinline__ void put4(size_t o, float4 v) const {
    if (out_lo) {
      float4 h, l;
      tf32_split(v.x, h.x, l.x); tf32_split(v.y, h.y, l.y); tf32_split(v.z, h.z, l.z); tf32_split(v.w, h.w, l.w);
      *reinterpret_cast<float4*>(out + o) = h;
      *reinterpret_cast<float4*>(out_lo + o) = l;
    } else {
      *reinterpret_cast<float4*>(out + o) = v;
    }
  }
  // t = thread index among the 256 epilogue threads; S = staged tile, S[c * 128 + ii * 16 + jj]
  __device__ __forceinline__ void flush(const float* S, int m0, int n0, int t) const {
    const int2 b = blk[m0 >> 7];
    const int i0 = b.x * 8, j0 = b.y * 16;
    for (int u = t; u < 256 * 32; u += 256) {          // direct: (column c, row ii, vector v of 4 jj)
      const int c = u >> 5, ii = (u >> 2) & 7, v = u & 3;
      const int col = n0 + c, i = i0 + ii, j = j0 + 4 * v;
      if (col >= n_real || i >= M || j >= M) continue;
      const float4 x = *reinterpret_cast<const float4*>(S + c * 128 + ii * 16 + 4 * v);
      put4((size_t)(col >> 1) * M * (2 * MP) + (col & 1) * MP + (size_t)i * (2 * MP) + j, x);
    }
    for (int u = t; u < 256 * 32; u += 256) {          // mirrored: (column c, row jj, vector v of 4 ii)
      const int c = u >> 5, jj = (u >> 1) & 15, v = u & 1;
      const int col = n0 + c, j = j0 + jj, i = i0 + 4 * v;
      if (col >= n_real || i >= M || j >= M) continue;
      const float* p = S + c * 128 + (4 * v) * 16 + jj;
      const float4 x = make_float4(p[0], p[16], p[32], p[48]);
      put4((size_t)(col >> 1) * M * (2 * MP) + (col & 1) * MP + (size_t)j * (2 * MP) + i, x);
    }
  }
  // Persistent kernel, store warps.  One round = 16 columns of each half of the tile in a staging buffer,
  // S[sc][row], sc = half * 16 + j  <->  tile column half * 128 + r * 16 + j, row = ii * 16 + jj of the 8 x 16 block.
  // Thread t of 128 owns a fixed (row, vector) of the block in either orientation and the staged columns (t >> 5) + 4 k,
  // k = 0..7: plane p = (t >> 5) & 1 is fixed, the walkers of its eight stores are 2 apart (and 64 apart between halves).
  struct StoreCtx { char* pd; char* pm; uint32_t ad, am, mv, W2B; int limd, limm; };
  __device__ __forceinline__ StoreCtx store_ctx(int m0, int n0, int t) const {
    StoreCtx c;
    const int2 b = blk[m0 >> 7];
    const int ws = t >> 5, c0 = n0 + ws;
    const int lim = n_real - c0;                                 // a store at tile-column offset o is real iff o < lim
    c.W2B = (uint32_t)M * (uint32_t)(2 * MP) * 8u;               // bytes per two walkers
    char* wb = reinterpret_cast<char*>(out) + ((size_t)(c0 >> 1) * M * (2 * MP) + (size_t)(c0 & 1) * MP) * 4;
    {                                                            // direct: row ii, vector v of 4 jj
      const int ii = (t >> 2) & 7, v = t & 3, i = b.x * 8 + ii, j = b.y * 16 + 4 * v;
      c.ad = (uint32_t)(ws * 128 + (ii ^ (ii >> 2)) * 16 + 4 * v) * 4;   // staged row ii*16+jj has bit 4 flipped for ii >= 4
      c.limd = (i < M && j < M) ? lim : 0;
      c.pd = wb + ((size_t)i * (2 * MP) + j) * 4;
    }
    {                                                            // mirrored: row jj, vector v of 4 ii
      const int jj = (t >> 1) & 15, v = t & 1, j = b.y * 16 + jj, i = b.x * 8 + 4 * v;
      c.am = (uint32_t)(ws * 128 + (4 * v) * 16 + jj) * 4;
      c.mv = (uint32_t)v * 64;                                   // rows 4v+x sit at (x ^ v) * 16: both v hit different banks
      c.limm = (i < M && j < M) ? lim : 0;
      c.pm = wb + ((size_t)j * (2 * MP) + i) * 4;
    }
    return c;
  }
  __device__ __forceinline__ void flush_round(const StoreCtx& c, uint32_t sSb, int r) const {
    const size_t ro = (size_t)(4 * r) * c.W2B;
    const int lr = r * 16;
    float4 x[8], y[8];                      // all 40 shared-memory loads of the round are in flight before the first store
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = ld_s128(sSb + c.ad + k * 2048);
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const uint32_t ak = sSb + c.am + k * 2048;
      y[k] = make_float4(ld_s32(ak + c.mv), ld_s32(ak + (64 ^ c.mv)), ld_s32(ak + (128 + c.mv)), ld_s32(ak + (128 + (64 ^ c.mv))));
    }
    char* p = c.pd + ro;
#pragma unroll
    for (int k = 0; k < 8; ++k)
      if (lr + (k >> 2) * 128 + (k & 3) * 4 < c.limd)
        st_g128_hint(p + (size_t)((k >> 2) * 32 + (k & 3)) * c.W2B, x[k], st_pol);
    p = c.pm + ro;
#pragma unroll
    for (int k = 0; k < 8; ++k)
      if (lr + (k >> 2) * 128 + (k & 3) * 4 < c.limm)
        st_g128_hint(p + (size_t)((k >> 2) * 32 + (k & 3)) * c.W2B, y[k], st_pol);
  }
};

struct EpiTT {          // H10: row = g*nact + q, col = (w*nt + a)*2 + p -> TT[w][g][q][a] (interleaved complex)
  static constexpr bool kStaged = false;
  float* out; int ng1, nact, nt, m_real, n_real;
  __device__ __forceinline__ void operator()(int r, int c0, const float (&v)[32]) const {
    if (r >= m_real) return;
    const int g = r / nact, q = r - g * nact;
    float* orow = out + ((size_t)g * nact + q) * (2 * nt);
    const size_t wstride = (size_t)ng1 * nact * (2 * nt);
    if ((nt & 1) == 0) {     // 2nt % 4 == 0: float4 groups never straddle a walker and stay 16-byte aligned
#pragma unroll
      for (int j = 0; j < 32; j += 4) {
        const int c = c0 + j;
        if (c < n_real) {
          const int w = c / (2 * nt), rem = c - w * 2 * nt;
          *reinterpret_cast<float4*>(orow + w * wstride + rem) = make_float4(v[j], v[j + 1], v[j + 2], v[j + 3]);
        }
      }
    } else {
#pragma unroll
      for (int j = 0; j < 32; ++j) {
        const int c = c0 + j;
        if (c < n_real) {
          const int w = c / (2 * nt), rem = c - w * 2 * nt;
          orow[w * wstride + rem] = v[j];
        }
      }
    }
  }
};
struct EpiEnergy {      // H9: eloc[w] += sum_rows v[row] (0.5 C[row][w] + hrot[row]), v = Theta of the walker
  static constexpr bool kStaged = false;
  // v is read from the interleaved Theta [N_w][M][N_t] (one 8-byte load per element: Re and Im together) rather than
  // from the four planar hi/lo operands: the epilogue is bound by the latency of its loads (ncu / tri = 0 experiment:
  // ~40 us per tile with 64 loads per 32 x 32 block, profiles/r1b_ncu_full.md), and this needs a quarter of them
  const float2* theta; int M, nt, off, n;      // row r of the spin block = (orbital k = r / n, column off + r % n)
  const float* hrot; double* eloc; int m_real, n_real;
  __device__ __forceinline__ void operator()(int r, int c0, const float (&v)[32]) const {
    const bool rok = r < m_real;
    const float hr = rok ? hrot[r] : 0.f;
    const int lane = threadIdx.x & 31;
    const int k = r / n, a = r - k * n;
    const float2* tp = theta + (size_t)k * nt + off + a;
    const size_t wstride = (size_t)M * nt;
    float2 t[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const int c = c0 + 2 * j;
      t[j] = (rok && c < n_real) ? tp[(size_t)(c >> 1) * wstride] : make_float2(0.f, 0.f);
    }
    float x[32];             // x[2p] / x[2p+1] = this row's contribution to Re / Im of walker (c0/2 + p)
#pragma unroll
    for (int j = 0; j < 32; j += 2) {
      const float vr = t[j >> 1].x, vi = t[j >> 1].y;
      const float ur = v[j] + hr, ui = v[j + 1];   // v = Y' Theta with Y' = triu(Y), diag / 2: Theta^T Y' Theta = 1/2 Theta^T Y Theta
      x[j] = vr * ur - vi * ui;
      x[j + 1] = vr * ui + vi * ur;
    }
    // transpose-reduce over the 32 rows of this warp: 31 shuffles, lane l ends with the sum of x[l]
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
#pragma unroll
      for (int i = 0; i < s; ++i) {
        const float keep = (lane & s) ? x[i + s] : x[i];
        const float send = (lane & s) ? x[i] : x[i + s];
        x[i] = keep + __shfl_xor_sync(0xffffffffu, send, s);
      }
    }
    if (c0 + lane < n_real) atomicAdd(&eloc[c0 + lane], (double)x[0]);
  }
};

template <class Epi>
__global__ void __launch_bounds__(THREADS, 1) k_gemm_tf32(const __grid_constant__ Maps maps, int K, int tri, Epi epi) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[STAGES];
  __shared__ __align__(8) uint64_t empty_bar[STAGES];
  __shared__ __align__(8) uint64_t tmem_full_bar[2];
  __shared__ __align__(8) uint64_t tmem_empty_bar[2];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  // tri != 0: the a-operand is upper triangular in 128 x 128 blocks (H9: Y' = triu(Y) with half the diagonal), so
  // the k-blocks left of this row tile are all zero and are skipped
  const int kb0 = tri ? m0 / BK : 0;
  const int nkb = K / BK - kb0;
  const int nchunk = (nkb + CHUNK_KB - 1) / CHUNK_KB;

  if (warp == EPI_WARPS && lane == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
#pragma unroll
    for (int b = 0; b < 2; ++b) { mbar_init(&tmem_full_bar[b], 1); mbar_init(&tmem_empty_bar[b], EPI_WARPS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.a_hi) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.a_lo) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.b_hi) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.b_lo) : "memory");
  }
  if (warp == EPI_WARPS + 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "r"((uint32_t)TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  if (warp == EPI_WARPS) {
    if (lane == 0) {   // ===== TMA producer =====
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % STAGES;
        const uint32_t ph = (kb / STAGES) & 1;
        mbar_wait(&empty_bar[s], ph ^ 1);
        uint8_t* st = smem + (size_t)s * STAGE_BYTES;
        mbar_expect_tx(&full_bar[s], STAGE_BYTES);
        const int kc = (kb0 + kb) * BK;
        tma_load_2d(st, &maps.a_hi, &full_bar[s], kc, m0);
        tma_load_2d(st + A_BYTES, &maps.a_lo, &full_bar[s], kc, m0);
        // the b-operand maps have 128-row boxes (shared with the CTA-pair kernel): two loads per plane
        tma_load_2d(st + 2 * A_BYTES, &maps.b_hi, &full_bar[s], kc, n0);
        tma_load_2d(st + 2 * A_BYTES + B_BYTES / 2, &maps.b_hi, &full_bar[s], kc, n0 + B_BOX);
        tma_load_2d(st + 2 * A_BYTES + B_BYTES, &maps.b_lo, &full_bar[s], kc, n0);
        tma_load_2d(st + 2 * A_BYTES + B_BYTES + B_BYTES / 2, &maps.b_lo, &full_bar[s], kc, n0 + B_BOX);
      }
    }
  } else if (warp == EPI_WARPS + 1) {
    if (lane == 0) {   // ===== MMA issuer =====
      constexpr uint32_t idesc = make_idesc(BM, BN);
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % STAGES;
        const uint32_t ph = (kb / STAGES) & 1;
        const int ci = kb / CHUNK_KB, buf = ci & 1;
        const bool chunk_start = (kb % CHUNK_KB) == 0;
        if (chunk_start) {   // the epilogue must have drained this TMEM buffer
          mbar_wait(&tmem_empty_bar[buf], ((ci >> 1) & 1) ^ 1);
          tc_fence_after();
        }
        mbar_wait(&full_bar[s], ph);
        tc_fence_after();
        const uint32_t d = tmem + buf * BN;
        const uint32_t sa = smem_u32(smem + (size_t)s * STAGE_BYTES);
        const uint64_t a_hi = make_desc(sa), a_lo = make_desc(sa + A_BYTES);
        const uint64_t b_hi = make_desc(sa + 2 * A_BYTES), b_lo = make_desc(sa + 2 * A_BYTES + B_BYTES);
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k) {
          const uint64_t adv = (uint64_t)((k * UMMA_K * 4) >> 4);
          umma_tf32(d, a_lo + adv, b_hi + adv, idesc, (chunk_start && k == 0) ? 0u : 1u);
          umma_tf32(d, a_hi + adv, b_lo + adv, idesc, 1u);
          umma_tf32(d, a_hi + adv, b_hi + adv, idesc, 1u);
        }
        tc_commit(&empty_bar[s]);                    // frees the stage once these MMAs have read it
        if ((kb % CHUNK_KB) == CHUNK_KB - 1 || kb == nkb - 1) tc_commit(&tmem_full_bar[buf]);
      }
    }
  } else {             // ===== epilogue warps 0..7: TMEM lane quarter = warp % 4, column half = warp / 4 =====
    const int q = warp & 3, half = warp >> 2;
    const int row = m0 + q * 32 + lane;
    float acc[COLS_PER_WARP];
#pragma unroll
    for (int i = 0; i < COLS_PER_WARP; ++i) acc[i] = 0.f;
    for (int ci = 0; ci < nchunk; ++ci) {
      const int buf = ci & 1;
      mbar_wait(&tmem_full_bar[buf], (ci >> 1) & 1);
      tc_fence_after();
      const uint32_t t0 = tmem + ((uint32_t)(q * 32) << 16) + buf * BN + half * COLS_PER_WARP;
#pragma unroll
      for (int cb = 0; cb < COLS_PER_WARP / 32; ++cb) {
        float v[32];
        tmem_ld32(t0 + cb * 32, v);
#pragma unroll
        for (int j = 0; j < 32; ++j) acc[cb * 32 + j] += v[j];
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(&tmem_empty_bar[buf])) : "memory");
    }
    if constexpr (Epi::kStaged) {
      // all MMAs have completed (last tmem_full observed) and no TMA load is pending: the stage memory is free
      float* S = reinterpret_cast<float*>(smem);
#pragma unroll
      for (int j = 0; j < COLS_PER_WARP; ++j) S[(half * COLS_PER_WARP + j) * BM + q * 32 + lane] = acc[j];
      asm volatile("bar.sync 1, 256;" ::: "memory");
      epi.flush(S, m0, n0, (int)threadIdx.x);
    } else {
#pragma unroll
      for (int cb = 0; cb < COLS_PER_WARP / 32; ++cb) {
        float v[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = acc[cb * 32 + j];
        epi(row, n0 + half * COLS_PER_WARP + cb * 32, v);
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == EPI_WARPS + 1) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)TMEM_COLS) : "memory");
  }
}

// ---- CTA-pair version: two CTAs of one TPC (cluster of 2 along grid x: a cluster of (1, 2, 1) is rejected at launch for cta_group::2 code) run one 256 x 256 tile with
// tcgen05.mma.cta_group::2.  Each CTA holds its own 128 rows of A and HALF of the 256 b-operand rows, so every MMA
// fetches 4 KB + 4 KB per SM for 128 math cycles instead of 4 KB + 8 KB: the shared-memory operand fetch that caps
// the one-CTA kernel at 66 % of the pipe no longer binds.  The leader (even) CTA issues the MMAs; both CTAs run a
// TMA producer (transaction bytes of both land on the leader's full barrier) and 8 epilogue warps on their own
// 128 TMEM lanes.  Stage = 64 KB per CTA, three stages.
enum { STAGES2 = 3, HB_BYTES = B_BYTES / 2, STAGE2_BYTES = 2 * A_BYTES + 2 * HB_BYTES };
static_assert(STAGES2 * STAGE2_BYTES + 1024 <= SMEM_BYTES, "pair kernel uses the same dynamic smem size");
static_assert(STAGES2 * STAGE2_BYTES >= BM * BN * 4, "staged epilogue needs the tile in shared memory");

template <class Epi>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(THREADS, 1)
k_gemm_tf32_pair(const __grid_constant__ Maps maps, int K, int tri, int m_tiles, int n_tiles, Epi epi) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[STAGES2];     // used in the leader only
  __shared__ __align__(8) uint64_t empty_bar[STAGES2];    // one in each CTA (multicast commit)
  __shared__ __align__(8) uint64_t tmem_full_bar[2];      // one in each CTA (multicast commit)
  __shared__ __align__(8) uint64_t tmem_empty_bar[2];     // leader only: 2 x 8 epilogue warps arrive
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  // 1-D grid of pairs; the column tile varies fastest, so the CTAs running at one time share a few row tiles of A
  // (each fetched from HBM once) and all of B stays in L2
  const int pair = blockIdx.x >> 1, mt = (pair / n_tiles) * 2 + (int)rank;
  const int m0 = mt * BM, n0 = (pair % n_tiles) * BN;
  const int kb0 = tri ? ((mt & ~1) * BM) / BK : 0;   // the pair starts at the leader's diagonal block
  const int nkb = K / BK - kb0;
  const int nchunk = (nkb + CHUNK_KB - 1) / CHUNK_KB;

  if (warp == EPI_WARPS && lane == 0) {
#pragma unroll
    for (int s = 0; s < STAGES2; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
#pragma unroll
    for (int b = 0; b < 2; ++b) { mbar_init(&tmem_full_bar[b], 1); mbar_init(&tmem_empty_bar[b], 2 * EPI_WARPS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.a_hi) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.a_lo) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.b_hi) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps.b_lo) : "memory");
  }
  if (warp == EPI_WARPS + 1) {   // the same warp in both CTAs allocates the pair's TMEM columns
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "r"((uint32_t)TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();      // the peer's barriers are initialised before anything is signalled across the pair
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;

  if (warp == EPI_WARPS) {
    if (lane == 0) {   // ===== TMA producer (both CTAs): own A rows, own half of the B rows =====
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % STAGES2;
        const uint32_t ph = (kb / STAGES2) & 1;
        mbar_wait(&empty_bar[s], ph ^ 1);
        uint8_t* st = smem + (size_t)s * STAGE2_BYTES;
        if (rank == 0) mbar_expect_tx(&full_bar[s], 2 * STAGE2_BYTES);
        const int kc = (kb0 + kb) * BK, nb = n0 + (int)rank * B_BOX;
        tma_load_2d_pair(st, &maps.a_hi, &full_bar[s], kc, m0);
        tma_load_2d_pair(st + A_BYTES, &maps.a_lo, &full_bar[s], kc, m0);
        tma_load_2d_pair(st + 2 * A_BYTES, &maps.b_hi, &full_bar[s], kc, nb);
        tma_load_2d_pair(st + 2 * A_BYTES + HB_BYTES, &maps.b_lo, &full_bar[s], kc, nb);
      }
    }
  } else if (warp == EPI_WARPS + 1) {
    if (lane == 0 && rank == 0) {   // ===== MMA issuer (leader CTA) =====
      constexpr uint32_t idesc = make_idesc(2 * BM, BN);
      for (int kb = 0; kb < nkb; ++kb) {
        const int s = kb % STAGES2;
        const uint32_t ph = (kb / STAGES2) & 1;
        const int ci = kb / CHUNK_KB, buf = ci & 1;
        const bool chunk_start = (kb % CHUNK_KB) == 0;
        if (chunk_start) {   // the epilogue warps of both CTAs must have drained this TMEM buffer
          mbar_wait(&tmem_empty_bar[buf], ((ci >> 1) & 1) ^ 1);
          tc_fence_after();
        }
        mbar_wait(&full_bar[s], ph);
        tc_fence_after();
        const uint32_t d = tmem + buf * BN;
        const uint32_t sa = smem_u32(smem + (size_t)s * STAGE2_BYTES);
        const uint64_t a_hi = make_desc(sa), a_lo = make_desc(sa + A_BYTES);
        const uint64_t b_hi = make_desc(sa + 2 * A_BYTES), b_lo = make_desc(sa + 2 * A_BYTES + HB_BYTES);
#pragma unroll
        for (int k = 0; k < BK / UMMA_K; ++k) {
          const uint64_t adv = (uint64_t)((k * UMMA_K * 4) >> 4);
          umma_tf32_pair(d, a_lo + adv, b_hi + adv, idesc, (chunk_start && k == 0) ? 0u : 1u);
          umma_tf32_pair(d, a_hi + adv, b_lo + adv, idesc, 1u);
          umma_tf32_pair(d, a_hi + adv, b_hi + adv, idesc, 1u);
        }
        tc_commit_pair(&empty_bar[s]);
        if ((kb % CHUNK_KB) == CHUNK_KB - 1 || kb == nkb - 1) tc_commit_pair(&tmem_full_bar[buf]);
      }
    }
  } else {             // ===== epilogue warps 0..7 of each CTA: its own 128 accumulator rows =====
    const int q = warp & 3, half = warp >> 2;
    const int row = m0 + q * 32 + lane;
    float acc[COLS_PER_WARP];
#pragma unroll
    for (int i = 0; i < COLS_PER_WARP; ++i) acc[i] = 0.f;
    for (int ci = 0; ci < nchunk; ++ci) {
      const int buf = ci & 1;
      mbar_wait(&tmem_full_bar[buf], (ci >> 1) & 1);
      tc_fence_after();
      const uint32_t t0 = tmem + ((uint32_t)(q * 32) << 16) + buf * BN + half * COLS_PER_WARP;
#pragma unroll
      for (int cb = 0; cb < COLS_PER_WARP / 32; ++cb) {
        float v[32];
        tmem_ld32(t0 + cb * 32, v);
#pragma unroll
        for (int j = 0; j < 32; ++j) acc[cb * 32 + j] += v[j];
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive_leader(&tmem_empty_bar[buf]);
    }
    if (mt < m_tiles) {   // the grid is padded to an even number of row tiles
      if constexpr (Epi::kStaged) {
        // every MMA of the pair has completed (last tmem_full observed), no TMA load is pending: the stages are free
        float* S = reinterpret_cast<float*>(smem);
#pragma unroll
        for (int j = 0; j < COLS_PER_WARP; ++j) S[(half * COLS_PER_WARP + j) * BM + q * 32 + lane] = acc[j];
        asm volatile("bar.sync 1, 256;" ::: "memory");
        epi.flush(S, m0, n0, (int)threadIdx.x);
      } else {
#pragma unroll
        for (int cb = 0; cb < COLS_PER_WARP / 32; ++cb) {
          float v[32];
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] = acc[cb * 32 + j];
          epi(row, n0 + half * COLS_PER_WARP + cb * 32, v);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();      // neither CTA leaves while the other may still read its shared memory or signal its barriers
  if (warp == EPI_WARPS + 1) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)TMEM_COLS) : "memory");
  }
}

// ---- persistent CTA-pair version for staged epilogues (H6): one pair per TPC loops over the tile pairs.  The operand
// ring (3 x 64 KB) and the staging area (2 x 16 KB) are separate, and the tile leaves through a second set of warps:
//   warps 0-7   epilogue: add each accumulation chunk from TMEM into registers; after the last chunk, hand the tile to
//               the store warps 16 columns per half at a time (16 STS per thread and round, nothing else)
//   warp  8     TMA producer        warp 9   MMA issuer (leader CTA)        warps 10-11 idle
//   warps 12-15 store warps: staging area -> HBM in both orientations (LDS + STG), everything they need in registers
// so the epilogue warps are back at the next tile's first chunk after ~8 x (16 STS + a barrier), well inside the two
// chunks the MMA issuer may run ahead.  (One set of warps doing both took 21k clk per tile at two warps per scheduler
// -- spills and constant reloads beside 128 live accumulators -- against 12k clk of slack: 0.73 ms; profiles/r2_ncu_full.md.)
// Barrier phases run on across tiles (global k-block / chunk / round counters).
// Chunk length of the persistent kernel: the truncation bias of the tensor pipe's accumulation is linear in it (A_w is
// 8e-7 low at 4 k-blocks, 4e-7 at 2), and S = det(overlap) picks that bias up N_elec-fold.  With the store warps the hand-over
// takes ~9k clk per tile, so two chunks of 2 k-blocks (6.1k clk of MMA) almost cover it.  Measured, B200 cfg 5:
// 4 -> 0.648 ms, 3 -> 0.658 ms, 2 -> 0.677 ms; per-step error of S on cfg 5: 3.5e-5 / - / 2.6e-5 (profiles/parity_r2.md).
#ifndef AFQMC_PS_CHUNK_KB
#define AFQMC_PS_CHUNK_KB 2
#endif
enum { PS_CHUNK_KB = AFQMC_PS_CHUNK_KB };
enum { PS_THREADS = 512, PS_STORE_WARP0 = 12, STG_COLS = 32, STG_BYTES = BM * STG_COLS * 4, STG_ROUNDS = BN / STG_COLS,
       SMEM_PS_BYTES = STAGES2 * STAGE2_BYTES + 2 * STG_BYTES + 1024 };
// L2 eviction-priority hints (bit 0: L rows evict_first, bit 1: field rows evict_last, bit 2: output stores evict_first).
// Measured on B200, cfg 5, H6: none changes the time (0.653-0.664 ms against 0.655; bit 0 costs 0.03-0.05 ms), but the
// DRAM reads go from 836 MB (no hint) to 675 MB (bit 1: the 33 MB of field planes, re-read by every row pair, stay in L2
// under the 650 MB output stream) and 569 MB (bits 1 + 2).  Default: bit 1 here; the stores' hint is chosen at run time
// (EpiAssembleSym::st_pol: evict_first only when A_w is larger than the L2, so that a small A_w stays there for H7).
#ifndef AFQMC_PS_POL
#define AFQMC_PS_POL 2
#endif
constexpr uint64_t L2_EVICT_NORMAL = 0x1000000000000000ull;
constexpr uint64_t PS_POL_A = (AFQMC_PS_POL & 1) ? L2_EVICT_FIRST : L2_EVICT_NORMAL;
constexpr uint64_t PS_POL_B = (AFQMC_PS_POL & 2) ? L2_EVICT_LAST : L2_EVICT_NORMAL;
constexpr uint64_t PS_POL_ST = (AFQMC_PS_POL & 4) ? L2_EVICT_FIRST : L2_EVICT_NORMAL;
enum { PS_REGS_EPI = 168, PS_REGS_AUX = 64, PS_REGS_STORE = 96 };
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// Work description of the persistent kernel.  Up to two problems (same column count; H9: the two spins) share one launch;
// `sched` (device, may be null) holds for every CTA pair its tile list, `sched_stride` entries per pair, -1 terminated,
// entry = problem << 24 | tile pair index (row-pair major, column tile fastest); used by the LIST instantiation only.
// tri: the a-operand is upper triangular in 128 x 128 blocks, a row pair starts at its leader's diagonal k-block.
struct PsWork {
  int K[2], m_tiles[2], n_tiles, n_pairs, tri, sched_stride;
  const int* sched;
};
struct PsTile { int prob, mt, m0, n0, kb0, nkb; bool valid; };
// LIST = false: one problem, full K range, pairs dealt round-robin (everything about a tile but its origin is loop-invariant)
template <bool LIST>
__device__ __forceinline__ bool ps_tile(const PsWork& wk, int cid, int ncl, int rank, int k, PsTile& t) {
  int e;
  if (LIST) {
    if (k >= wk.sched_stride) return false;
    e = wk.sched[(size_t)cid * wk.sched_stride + k];
    if (e < 0) return false;
  } else {
    e = cid + k * ncl;
    if (e >= wk.n_pairs) return false;
  }
  t.prob = LIST ? e >> 24 : 0;
  const int tp = LIST ? (e & 0xFFFFFF) : e, mp = tp / wk.n_tiles;
  t.mt = mp * 2 + rank; t.m0 = t.mt * BM; t.n0 = (tp - mp * wk.n_tiles) * BN;
  t.kb0 = (LIST && wk.tri) ? (mp * 2 * BM) / BK : 0;
  t.nkb = wk.K[t.prob] / BK - t.kb0;
  t.valid = t.mt < wk.m_tiles[t.prob];
  return true;
}

template <class Epi, int CHUNK = PS_CHUNK_KB, bool LIST = false>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PS_THREADS, 1)
k_gemm_tf32_pair_ps(const __grid_constant__ Maps maps0, const __grid_constant__ Maps maps1, const __grid_constant__ PsWork wk,
                    const __grid_constant__ Epi epi0, const __grid_constant__ Epi epi1) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>(((uintptr_t)smem_raw + 1023) & ~(uintptr_t)1023);
  __shared__ __align__(8) uint64_t full_bar[STAGES2];     // used in the leader only
  __shared__ __align__(8) uint64_t empty_bar[STAGES2];
  __shared__ __align__(8) uint64_t tmem_full_bar[2];
  __shared__ __align__(8) uint64_t tmem_empty_bar[2];     // leader only: 2 x 8 epilogue warps arrive
  __shared__ __align__(8) uint64_t stg_full_bar[2];       // 8 epilogue warps arrive
  __shared__ __align__(8) uint64_t stg_free_bar[2];       // 4 store warps arrive
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;
  const uint32_t sS = smem_u32(smem + (size_t)STAGES2 * STAGE2_BYTES);

  if (warp == EPI_WARPS && lane == 0) {
#pragma unroll
    for (int s = 0; s < STAGES2; ++s) { mbar_init(&full_bar[s], 1); mbar_init(&empty_bar[s], 1); }
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      mbar_init(&tmem_full_bar[b], 1); mbar_init(&tmem_empty_bar[b], 2 * EPI_WARPS);
      mbar_init(&stg_full_bar[b], EPI_WARPS); mbar_init(&stg_free_bar[b], 4);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps0.a_hi) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps0.a_lo) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps0.b_hi) : "memory");
    asm volatile("prefetch.tensormap [%0];" ::"l"(&maps0.b_lo) : "memory");
  }
  if (warp == EPI_WARPS + 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)),
                 "r"((uint32_t)TMEM_COLS)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  PsTile tl;

  if (warp >= PS_STORE_WARP0) {          // ===== store warps (staged epilogues only) =====
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"((int)PS_REGS_STORE));
    if constexpr (Epi::kStaged) {
      const int t = (int)threadIdx.x - PS_STORE_WARP0 * 32;
      uint32_t sr = 0;
      for (int ti = 0; ps_tile<LIST>(wk, cid, ncl, (int)rank, ti, tl); ++ti) {
        const Epi* const epp = (LIST && tl.prob) ? &epi1 : &epi0;
        const Epi epi = *epp;
        typename Epi::StoreCtx sc = epi.store_ctx(tl.valid ? tl.m0 : 0, tl.n0, t);
#pragma unroll 1
        for (int r = 0; r < STG_ROUNDS; ++r, ++sr) {
          const int b = sr & 1;
          mbar_wait(&stg_full_bar[b], (sr >> 1) & 1);
          if (tl.valid) epi.flush_round(sc, sS + b * STG_BYTES, r);
          __syncwarp();
          if (lane == 0) mbar_arrive(&stg_free_bar[b]);   // release: the loads above have completed
        }
      }
    }
  } else if (warp >= EPI_WARPS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"((int)PS_REGS_AUX));
    if (warp == EPI_WARPS) {
      if (lane == 0) {   // ===== TMA producer (both CTAs) =====
        uint32_t it = 0;
        for (int ti = 0; ps_tile<LIST>(wk, cid, ncl, (int)rank, ti, tl); ++ti) {
          const Maps* mp = (LIST && tl.prob) ? &maps1 : &maps0;
          const int nb = tl.n0 + (int)rank * B_BOX;
          for (int kb = 0; kb < tl.nkb; ++kb, ++it) {
            const int s = it % STAGES2;
            mbar_wait(&empty_bar[s], ((it / STAGES2) & 1) ^ 1);
            uint8_t* st = smem + (size_t)s * STAGE2_BYTES;
            if (rank == 0) mbar_expect_tx(&full_bar[s], 2 * STAGE2_BYTES);
            const int kc = (tl.kb0 + kb) * BK;
            tma_load_2d_pair_hint(st, &mp->a_hi, &full_bar[s], kc, tl.m0, PS_POL_A);
            tma_load_2d_pair_hint(st + A_BYTES, &mp->a_lo, &full_bar[s], kc, tl.m0, PS_POL_A);
            // the b-operand hint is for H6's field planes only (33 MB, read by every row pair); H4 / H9 stream 165 MB of Theta planes
            constexpr uint64_t polb = LIST ? L2_EVICT_NORMAL : PS_POL_B;
            tma_load_2d_pair_hint(st + 2 * A_BYTES, &mp->b_hi, &full_bar[s], kc, nb, polb);
            tma_load_2d_pair_hint(st + 2 * A_BYTES + HB_BYTES, &mp->b_lo, &full_bar[s], kc, nb, polb);
          }
        }
      }
    } else if (warp == EPI_WARPS + 1) {
      if (rank == 0) {   // ===== MMA issuer (leader CTA).  The whole warp runs the loop and one elected lane issues: with
        // uniform control flow the descriptors live in uniform registers and a k-block's 12 MMAs are back-to-back UTCHMMA
        // (inside `if (lane == 0)` every MMA is wrapped in an ELECT / R2UR sequence; taylor_tc.cuh has the measurement) =====
        constexpr uint32_t idesc = make_idesc(2 * BM, BN);
        constexpr uint64_t SSTEP = STAGE2_BYTES >> 4;     // the descriptor's address field counts 16-byte units
        const uint64_t d0 = make_desc(smem_u32(smem));
        uint64_t ds = d0;
        int s = 0;
        uint32_t fpar = 0, cg = 0;
        for (int ti = 0; ps_tile<LIST>(wk, cid, ncl, 0, ti, tl); ++ti) {
          int kc = 0;                                      // k-block within the chunk
          for (int kb = 0; kb < tl.nkb; ++kb) {
            const int buf = cg & 1;
            if (kc == 0) {   // both CTAs' epilogue warps have drained this TMEM buffer (two chunks ago)
              mbar_wait(&tmem_empty_bar[buf], ((cg >> 1) & 1) ^ 1);
            }
            mbar_wait(&full_bar[s], fpar);
            tc_fence_after();
            const bool chunk_end = kc == CHUNK - 1 || kb == tl.nkb - 1;
            if (elect_one()) {
              const uint32_t d = tmem + buf * BN;
              const uint64_t a_hi = ds, a_lo = ds + (A_BYTES >> 4);
              const uint64_t b_hi = ds + ((2 * A_BYTES) >> 4), b_lo = ds + ((2 * A_BYTES + HB_BYTES) >> 4);
#pragma unroll
              for (int k = 0; k < BK / UMMA_K; ++k) {
                const uint64_t adv = (uint64_t)((k * UMMA_K * 4) >> 4);
                umma_tf32_pair(d, a_lo + adv, b_hi + adv, idesc, (kc == 0 && k == 0) ? 0u : 1u);
                umma_tf32_pair(d, a_hi + adv, b_lo + adv, idesc, 1u);
                umma_tf32_pair(d, a_hi + adv, b_hi + adv, idesc, 1u);
              }
              tc_commit_pair(&empty_bar[s]);
              if (chunk_end) tc_commit_pair(&tmem_full_bar[buf]);
            }
            __syncwarp();
            if (chunk_end) { ++cg; kc = 0; } else ++kc;
            ds += SSTEP;
            if (++s == STAGES2) { s = 0; ds = d0; fpar ^= 1; }
          }
        }
      }
    }
  } else {             // ===== epilogue warps 0..7 of each CTA =====
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"((int)PS_REGS_EPI));
    const int q = warp & 3, half = warp >> 2;
    // staged row = (q * 32 + lane) with bit 4 flipped in the upper half of the block (conflict-free mirrored reads, see StoreCtx)
    const uint32_t sW = sS + (uint32_t)((half * (STG_COLS / 2)) * BM + ((q * 32 + lane) ^ ((q >> 1) << 4))) * 4;
    uint32_t cg = 0, sr = 0;
    for (int ti = 0;; ++ti) {
      int nchunk;
      {   // only the chunk count stays live beside the 128 accumulators; the tile is looked up again after the loop
        PsTile t0;
        if (!ps_tile<LIST>(wk, cid, ncl, (int)rank, ti, t0)) break;
        nchunk = (t0.nkb + CHUNK - 1) / CHUNK;
      }
      float acc[COLS_PER_WARP];
#pragma unroll
      for (int i = 0; i < COLS_PER_WARP; ++i) acc[i] = 0.f;
      for (int ci = 0; ci < nchunk; ++ci, ++cg) {
        const int buf = cg & 1;
        mbar_wait(&tmem_full_bar[buf], (cg >> 1) & 1);
        tc_fence_after();
        const uint32_t t0 = tmem + ((uint32_t)(q * 32) << 16) + buf * BN + half * COLS_PER_WARP;
#pragma unroll
        for (int cb = 0; cb < COLS_PER_WARP / 32; ++cb) {
          float v[32];
          tmem_ld32(t0 + cb * 32, v);
#pragma unroll
          for (int j = 0; j < 32; ++j) acc[cb * 32 + j] += v[j];
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive_leader(&tmem_empty_bar[buf]);
      }
      // the tile sits in registers and both TMEM buffers are released: the next tile's MMAs run while it leaves
      if constexpr (Epi::kStaged) {
#pragma unroll
        for (int r = 0; r < STG_ROUNDS; ++r, ++sr) {
          const int b = sr & 1;
          mbar_wait(&stg_free_bar[b], ((sr >> 1) & 1) ^ 1);
#pragma unroll
          for (int j = 0; j < STG_COLS / 2; ++j) st_s32(sW + b * STG_BYTES + j * (BM * 4), acc[r * (STG_COLS / 2) + j]);
          __syncwarp();
          if (lane == 0) mbar_arrive(&stg_full_bar[b]);   // release: this warp's 16 x 32 values are in place
        }
      } else {
        ps_tile<LIST>(wk, cid, ncl, (int)rank, ti, tl);
        if (tl.valid) {
          // by address: `cond ? epi1 : epi0` on the two parameter structs picked epi0 for every tile of the EpiStoreT instantiation
          const Epi* const epp = (LIST && tl.prob) ? &epi1 : &epi0;
          const Epi epi = *epp;
#pragma unroll
          for (int cb = 0; cb < COLS_PER_WARP / 32; ++cb) {
            float v[32];
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] = acc[cb * 32 + j];
            epi(tl.m0 + q * 32 + lane, tl.n0 + half * COLS_PER_WARP + cb * 32, v);
          }
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == EPI_WARPS + 1) {
    __syncwarp();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"((uint32_t)TMEM_COLS) : "memory");
  }
}

// ---- host: tensor maps ------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// K-major FP32 plane [rows][ld], logical extent {K, rows}; box {BK, box_rows}; out-of-range rows read as 0
inline bool make_map(CUtensorMap* m, const void* base, uint64_t K, uint64_t rows, uint64_t ld, uint32_t box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[2] = {K, rows};
  cuuint64_t strides[1] = {ld * 4};
  cuuint32_t box[2] = {BK, box_rows};
  cuuint32_t estr[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tc
}  // namespace afq
