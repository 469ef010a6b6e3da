// taylor.cuh -- H7: Phi' = E_h [sum_{k<=K} A^k / k!] E_h Phi, one CTA per walker (
// DESIGN.md R3, R9).  A_w = i sqrt(dt) sum_g xs_g L_g is complex symmetric, E_h real symmetric, so the
// row block j0..j0+JB of the matrix IS the column block the product needs: it is streamed with cp.async
// as one contiguous chunk and read conflict-free (lane <-> output row i).
//   thread (i, chunk) owns output row i, CW columns; T_k lives in shared memory, the running sum in registers.
#pragma once
#include "common.cuh"

namespace afq {

template <typename T> struct TaylorArgs {
  int M, MP, nt, K, nchunks;
  cplx<T>* phi;      // [nw][M][nt] in/out
  const T* A;        // [nw][M][2][MP]  (re plane, im plane per row)
  const T* Eh;       // [M][MP]
};

enum { TAYLOR_JB = 16 };

template <typename T, int CW> struct TaylorCfg {
  enum { CWP = (CW + 3) & ~3 };  // padded chunk width (vector loads)
};

template <typename T> inline size_t taylor_smem_bytes(int M, int MP, int nchunks, int CWP) {
  size_t v = (size_t)M * nchunks * 2 * CWP * sizeof(T);
  size_t a = (size_t)2 * TAYLOR_JB * 2 * MP * sizeof(T);
  return v + a;
}

// acc += X[:, j] * V[j, :] over all j, X streamed in row blocks of JB rows.
// CPLX: X rows are [re(MP) | im(MP)], else [re(MP)].
template <typename T, int CW, bool CPLX>
__device__ __forceinline__ void apply_sym(const T* __restrict__ X, int M, int MP, const T* Vs, int vstride, T* As,
                                          int i, int chunk, bool active, T (&ar)[CW], T (&ai)[CW]) {
  enum { JB = TAYLOR_JB, CWP = TaylorCfg<T, CW>::CWP, VPE = 16 / sizeof(T) };
  const int rowlen = CPLX ? 2 * MP : MP;       // elements per matrix row
  const int stage_elems = JB * 2 * MP;          // stage stride (sized for complex)
  const int nblk = (M + JB - 1) / JB;
  const int tid = threadIdx.x, nthr = blockDim.x;
#pragma unroll
  for (int c = 0; c < CW; ++c) { ar[c] = T(0); ai[c] = T(0); }
  auto prefetch = [&](int b) {
    int rows = min(JB, M - b * JB);
    int nvec = rows * rowlen / VPE;
    const T* src = X + (size_t)b * JB * rowlen;
    T* dst = As + (b & 1) * stage_elems;
    for (int v = tid; v < nvec; v += nthr) cp_async16(dst + v * VPE, src + v * VPE);
    cp_async_commit();
  };
  prefetch(0);
  for (int b = 0; b < nblk; ++b) {
    if (b + 1 < nblk) { prefetch(b + 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
    __syncthreads();
    if (active) {
      const T* Ab = As + (b & 1) * stage_elems;
      const int rows = min(JB, M - b * JB);
      for (int jj = 0; jj < rows; ++jj) {
        const T xr = Ab[jj * rowlen + i];
        const T xi = CPLX ? Ab[jj * rowlen + MP + i] : T(0);
        const T* vrow = Vs + (size_t)(b * JB + jj) * vstride + chunk * 2 * CWP;
        __align__(16) T vr[CWP];
        __align__(16) T vi[CWP];
#pragma unroll
        for (int c = 0; c < CWP; c += VPE) {
          if (sizeof(T) == 4) {
            *reinterpret_cast<float4*>(&vr[c]) = *reinterpret_cast<const float4*>(vrow + c);
            *reinterpret_cast<float4*>(&vi[c]) = *reinterpret_cast<const float4*>(vrow + CWP + c);
          } else {
            *reinterpret_cast<double2*>(&vr[c]) = *reinterpret_cast<const double2*>(vrow + c);
            *reinterpret_cast<double2*>(&vi[c]) = *reinterpret_cast<const double2*>(vrow + CWP + c);
          }
        }
#pragma unroll
        for (int c = 0; c < CW; ++c) {
          ar[c] = fma(xr, vr[c], ar[c]);
          ai[c] = fma(xr, vi[c], ai[c]);
          if (CPLX) {
            ar[c] = fma(-xi, vi[c], ar[c]);
            ai[c] = fma(xi, vr[c], ai[c]);
          }
        }
      }
    }
    __syncthreads();
  }
}

template <typename T, int CW, int MAXT>
__global__ void __launch_bounds__(MAXT) k_taylor(TaylorArgs<T> g) {
  enum { CWP = TaylorCfg<T, CW>::CWP };
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int M = g.M, MP = g.MP, nt = g.nt, nch = g.nchunks;
  const int vstride = nch * 2 * CWP;
  T* Vs = reinterpret_cast<T*>(smem_raw);
  T* As = Vs + (size_t)M * vstride;
  const int w = blockIdx.x, tid = threadIdx.x;
  const int chunk = tid / M, i = tid - chunk * M;
  const bool active = chunk < nch;
  cplx<T>* phi_w = g.phi + (size_t)w * M * nt;

  // V <- Phi (planar per chunk, zero padded)
  for (int e = tid; e < M * vstride; e += blockDim.x) Vs[e] = T(0);
  __syncthreads();
  for (int e = tid; e < M * nt; e += blockDim.x) {
    int k = e / nt, c = e - k * nt;
    int ch = c / CW, cc = c - ch * CW;
    cplx<T> v = phi_w[e];
    Vs[k * vstride + ch * 2 * CWP + cc] = v.x;
    Vs[k * vstride + ch * 2 * CWP + CWP + cc] = v.y;
  }
  __syncthreads();

  T ar[CW], ai[CW], pr[CW], pi[CW];
  auto storeV = [&](const T (&xr)[CW], const T (&xi)[CW]) {
    if (active) {
      T* vrow = Vs + (size_t)i * vstride + chunk * 2 * CWP;
#pragma unroll
      for (int c = 0; c < CW; ++c) { vrow[c] = xr[c]; vrow[CWP + c] = xi[c]; }
    }
    __syncthreads();
  };
  // T_0 = E_h Phi
  apply_sym<T, CW, false>(g.Eh, M, MP, Vs, vstride, As, i, chunk, active, ar, ai);
#pragma unroll
  for (int c = 0; c < CW; ++c) { pr[c] = ar[c]; pi[c] = ai[c]; }
  storeV(ar, ai);
  // T_k = A T_{k-1} / k ; P += T_k
  const T* Aw = g.A + (size_t)w * M * 2 * MP;
  for (int k = 1; k <= g.K; ++k) {
    apply_sym<T, CW, true>(Aw, M, MP, Vs, vstride, As, i, chunk, active, ar, ai);
    const T inv = T(1) / T(k);
#pragma unroll
    for (int c = 0; c < CW; ++c) { ar[c] *= inv; ai[c] *= inv; pr[c] += ar[c]; pi[c] += ai[c]; }
    storeV(ar, ai);
  }
  // Phi' = E_h P
  storeV(pr, pi);
  apply_sym<T, CW, false>(g.Eh, M, MP, Vs, vstride, As, i, chunk, active, ar, ai);
  storeV(ar, ai);
  for (int e = tid; e < M * nt; e += blockDim.x) {
    int k = e / nt, c = e - k * nt;
    int ch = c / CW, cc = c - ch * CW;
    phi_w[e] = mk<T>(Vs[k * vstride + ch * 2 * CWP + cc], Vs[k * vstride + ch * 2 * CWP + CWP + cc]);
  }
}

}  // namespace afq
