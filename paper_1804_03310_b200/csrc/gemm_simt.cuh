// gemm_simt.cuh -- register-tiled "NT" GEMM on the FP32 / FP64 SIMT pipes with fused epilogues.
//   C[m][n] = sum_k A[m][k] * B[n][k]      (both operands K-major, zero padded to a multiple of BK)
// Used for H4 (force bias), H6 (one-body operator assembly), H9 (energy) on the FP64 path (always) and
// on the FP32 path when the tcgen05 3xTF32 kernel is not selected.  PAPER.md:59, :80, :87.
#pragma once
#include "common.cuh"

namespace afq {

template <typename T> struct VecOf;
template <> struct VecOf<float> { typedef float4 type; enum { N = 4 }; };
template <> struct VecOf<double> { typedef double2 type; enum { N = 2 }; };

template <typename T> struct GemmCfg;
template <> struct GemmCfg<float> { enum { BM = 128, BN = 128, BK = 8, TM = 8, TN = 8 }; };
template <> struct GemmCfg<double> { enum { BM = 64, BN = 64, BK = 8, TM = 4, TN = 4 }; };

// ---- epilogues: called once per thread with its TM x TN accumulators.  Row index of acc[i][.]:
// i < TM/2 ? r0 + i : r1 + (i - TM/2); same for columns.  scratch = the CTA's (now free) tile memory.

// H4: f_s[col][row] = C[row][col]  (col = (walker, re/im plane), row = gamma)
template <typename T> struct EpiStoreT {
  T* out; int ldo; int m_real, n_real;
  template <int TM, int TN>
  __device__ void operator()(T (&acc)[TM][TN], int r0, int r1, int c0, int c1, void*) const {
#pragma unroll
    for (int j = 0; j < TN; ++j) {
      int c = j < TN / 2 ? c0 + j : c1 + j - TN / 2;
      if (c >= n_real) continue;
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        int r = i < TM / 2 ? r0 + i : r1 + i - TM / 2;
        if (r < m_real) out[(size_t)c * ldo + r] = acc[i][j];
      }
    }
  }
};

// H6: row = i*M + j (matrix element), col = 2*w + p.  A_w stored [w][j][p][MP] (symmetric, so the
// (i,j) element is written at row j, plane p, column i); "assembly of the one-body operator".
template <typename T> struct EpiAssemble {
  T* out; int M, MP; int m_real, n_real;
  template <int TM, int TN>
  __device__ void operator()(T (&acc)[TM][TN], int r0, int r1, int c0, int c1, void*) const {
#pragma unroll
    for (int i = 0; i < TM; ++i) {
      int r = i < TM / 2 ? r0 + i : r1 + i - TM / 2;
      if (r >= m_real) continue;
      int ii = r / M, jj = r - ii * M;
#pragma unroll
      for (int j = 0; j < TN; ++j) {
        int c = j < TN / 2 ? c0 + j : c1 + j - TN / 2;
        if (c >= n_real) continue;
        int w = c >> 1, p = c & 1;
        out[((size_t)w * M + ii) * (2 * MP) + p * MP + jj] = acc[i][j];
      }
    }
  }
};

// H9: per column pair (walker w): e += sum_rows v[row] * (C[row][w] + hrot[row]), C = Y' v, v = planar Theta
// block of this spin, complex bilinear (no conjugation).  Accumulated into eloc[w] (FP64 atomics).
template <typename T> struct EpiEnergy {
  const T* thp; const T* thp_lo; int KT; int soff;   // v_re = thp[(2w)*KT + soff + row] (+ lo plane if split)
  const T* hrot;                                     // [Ks] one-body row vector Psi^T h, same index as v
  double* eloc;                                      // [nw][2]
  int m_real, n_real;
  template <int TM, int TN>
  __device__ void operator()(T (&acc)[TM][TN], int r0, int r1, int c0, int c1, void* scratch) const {
    double* red = reinterpret_cast<double*>(scratch);   // [BN] doubles: (re, im) per walker of the tile
    const int BN = (int)GemmCfg<T>::BN;
    for (int e = threadIdx.x; e < BN; e += blockDim.x) red[e] = 0.0;
    __syncthreads();
    const int cbase = blockIdx.x * BN;
#pragma unroll
    for (int jp = 0; jp < TN / 2; ++jp) {
      int j = 2 * jp;
      int c = j < TN / 2 ? c0 + j : c1 + j - TN / 2;   // even column = real plane of walker c/2
      if (c >= n_real) continue;
      int w = c >> 1;
      double er = 0.0, ei = 0.0;
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        int r = i < TM / 2 ? r0 + i : r1 + i - TM / 2;
        if (r >= m_real) continue;
        size_t o = (size_t)(2 * w) * KT + soff + r;
        T vr = thp[o], vi = thp[o + KT];
        if (thp_lo) { vr += thp_lo[o]; vi += thp_lo[o + KT]; }
        T ur = acc[i][j] + hrot[r];          // acc = Y' v with Y' = triu(Y), diagonal halved: v^T Y' v = 1/2 v^T Y v
        T ui = acc[i][j + 1];
        er += (double)(vr * ur - vi * ui);
        ei += (double)(vr * ui + vi * ur);
      }
      atomicAdd(&red[c - cbase], er);
      atomicAdd(&red[c - cbase + 1], ei);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < BN; e += blockDim.x) {
      int c = cbase + e;
      if (c < n_real && red[e] != 0.0) atomicAdd(&eloc[c], red[e]);
    }
  }
};

// H10: row = g*nact + q, col = (w*nt + a)*2 + p  ->  TT[w][g][q][a] (interleaved complex; columns contiguous)
template <typename T> struct EpiTT {
  T* out; int ng1, nact, nt; int m_real, n_real;
  template <int TM, int TN>
  __device__ void operator()(T (&acc)[TM][TN], int r0, int r1, int c0, int c1, void*) const {
#pragma unroll
    for (int j = 0; j < TN; ++j) {
      int c = j < TN / 2 ? c0 + j : c1 + j - TN / 2;
      if (c >= n_real) continue;
      int w = c / (2 * nt), rem = c - w * 2 * nt;
#pragma unroll
      for (int i = 0; i < TM; ++i) {
        int r = i < TM / 2 ? r0 + i : r1 + i - TM / 2;
        if (r >= m_real) continue;
        int g = r / nact, q = r - g * nact;
        out[(((size_t)w * ng1 + g) * nact + q) * (2 * nt) + rem] = acc[i][j];
      }
    }
  }
};

// grid = (ceil(N/BN), ceil(M/BM)), 256 threads.
template <typename T, class Epi>
__global__ void __launch_bounds__(256) k_gemm_nt(const T* __restrict__ A, int lda, int m_rows,
                                                 const T* __restrict__ B, int ldb, int n_rows, int K, Epi epi) {
  typedef GemmCfg<T> C;
  typedef typename VecOf<T>::type V;
  enum { BM = C::BM, BN = C::BN, BK = C::BK, TM = C::TM, TN = C::TN, VN = VecOf<T>::N, PAD = 4 };
  static_assert(BM * BK / 256 == VN && BN * BK / 256 == VN, "one vector load per thread per operand");
  __shared__ __align__(16) T As[2][BK][BM + PAD];
  __shared__ __align__(16) T Bs[2][BK][BN + PAD];
  const int tid = threadIdx.x;
  const int m0 = blockIdx.y * BM, n0 = blockIdx.x * BN;
  const int lrow = tid / (BK / VN), lk = (tid % (BK / VN)) * VN;
  const bool a_ok = (m0 + lrow) < m_rows, b_ok = (n0 + lrow) < n_rows;
  const T* ap = A + (size_t)(m0 + lrow) * lda + lk;
  const T* bp = B + (size_t)(n0 + lrow) * ldb + lk;
  const int ty = tid / 16, tx = tid % 16;
  T acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = T(0);

  V va, vb;
  T zero[VN];
#pragma unroll
  for (int i = 0; i < VN; ++i) zero[i] = T(0);
  auto gload = [&](int k0) {
    va = a_ok ? *reinterpret_cast<const V*>(ap + k0) : *reinterpret_cast<const V*>(zero);
    vb = b_ok ? *reinterpret_cast<const V*>(bp + k0) : *reinterpret_cast<const V*>(zero);
  };
  auto sstore = [&](int st) {
    const T* pa = reinterpret_cast<const T*>(&va);
    const T* pb = reinterpret_cast<const T*>(&vb);
#pragma unroll
    for (int i = 0; i < VN; ++i) {
      As[st][lk + i][lrow] = pa[i];
      Bs[st][lk + i][lrow] = pb[i];
    }
  };
  const int nk = K / BK;
  gload(0);
  sstore(0);
  __syncthreads();
  for (int kb = 0; kb < nk; ++kb) {
    const int st = kb & 1;
    if (kb + 1 < nk) gload((kb + 1) * BK);
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      T a[TM], b[TN];
#pragma unroll
      for (int i = 0; i < TM / 2; ++i) {
        a[i] = As[st][k][ty * (TM / 2) + i];
        a[i + TM / 2] = As[st][k][BM / 2 + ty * (TM / 2) + i];
      }
#pragma unroll
      for (int j = 0; j < TN / 2; ++j) {
        b[j] = Bs[st][k][tx * (TN / 2) + j];
        b[j + TN / 2] = Bs[st][k][BN / 2 + tx * (TN / 2) + j];
      }
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    if (kb + 1 < nk) {
      sstore(st ^ 1);
      __syncthreads();
    }
  }
  __syncthreads();
  epi(acc, m0 + ty * (TM / 2), m0 + BM / 2 + ty * (TM / 2), n0 + tx * (TN / 2), n0 + BN / 2 + tx * (TN / 2),
      (void*)&As[0][0][0]);
}

}  // namespace afq
