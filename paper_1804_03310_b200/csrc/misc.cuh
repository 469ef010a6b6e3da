// misc.cuh -- H5 field shift, force-bias finish, and the FP64 init-time precompute kernels (H11).
#pragma once
#include "common.cuh"

namespace afq {

// ---------------------------------------------------------------------------------------------
// H5 ("each auxiliary-field is shifted by a force-bias"; R1, R2):
//   xbar = -i sqrt(dt) f ; xs = x - xbar ; z = i sqrt(dt) xs  (coefficient of L_g in A) ;
//   c = sum_g x xbar - 1/2 sum_g xbar^2 (no conjugation).  One CTA per walker.
// Z planar [2*nw][NGP]: row 2w = Re z, row 2w+1 = Im z (K-major operand of the assembly GEMM).
// ---------------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128) k_shift(int n_chol, int NGP, double dt, const cplx<T>* fb, const T* x, T* Z,
                                               T* Z_lo, int split, zcplx* cshift) {
  const int w = blockIdx.x, tid = threadIdx.x;
  const double sdt = sqrt(dt);
  double cr = 0.0, ci = 0.0;
  for (int g = tid; g < n_chol; g += 128) {
    cplx<T> f = fb[(size_t)w * n_chol + g];
    double xg = (double)x[(size_t)w * n_chol + g];
    double xbr = sdt * (double)f.y, xbi = -sdt * (double)f.x;
    cr += xg * xbr - 0.5 * (xbr * xbr - xbi * xbi);
    ci += xg * xbi - xbr * xbi;
    double zr = sdt * xbi;             // Re(i sdt (xg - xbr - i xbi)) = sdt * xbi
    double zi = sdt * (xg - xbr);
    size_t o = (size_t)(2 * w) * NGP + g;
    if (split) {
      float h0, l0, h1, l1;
      tf32_split((float)zr, h0, l0);
      tf32_split((float)zi, h1, l1);
      Z[o] = (T)h0; Z[o + NGP] = (T)h1;
      Z_lo[o] = (T)l0; Z_lo[o + NGP] = (T)l1;
    } else {
      Z[o] = (T)zr; Z[o + NGP] = (T)zi;
    }
  }
  __shared__ double red[2][4];
  cr = warp_sum(cr); ci = warp_sum(ci);
  if ((tid & 31) == 0) { red[0][tid >> 5] = cr; red[1][tid >> 5] = ci; }
  __syncthreads();
  if (tid == 0) cshift[w] = mk<double>(red[0][0] + red[0][1] + red[0][2] + red[0][3],
                                       red[1][0] + red[1][1] + red[1][2] + red[1][3]);
}

// Per-spin planar traces fs[s][2w+p][NGP] -> fb[w][g] = f^a + f^b (interleaved complex), and
// eloc[w] := sum_g f^a_g f^b_g (cross-spin Coulomb term of E_L, R8) if eloc != null.
template <typename T>
__global__ void __launch_bounds__(128) k_fb_finish(int n_chol, int NGP, int nw, const T* fs, cplx<T>* fb, zcplx* eloc) {
  const int w = blockIdx.x, tid = threadIdx.x;
  const T* fa = fs + (size_t)(2 * w) * NGP;
  const T* fbt = fs + (size_t)2 * nw * NGP + (size_t)(2 * w) * NGP;
  double cr = 0.0, ci = 0.0;
  for (int g = tid; g < n_chol; g += 128) {
    T ar = fa[g], ai = fa[NGP + g], br = fbt[g], bi = fbt[NGP + g];
    if (fb) fb[(size_t)w * n_chol + g] = mk<T>(ar + br, ai + bi);
    cr += (double)ar * (double)br - (double)ai * (double)bi;
    ci += (double)ar * (double)bi + (double)ai * (double)br;
  }
  if (eloc) {
    __shared__ double red[2][4];
    cr = warp_sum(cr); ci = warp_sum(ci);
    if ((tid & 31) == 0) { red[0][tid >> 5] = cr; red[1][tid >> 5] = ci; }
    __syncthreads();
    if (tid == 0) eloc[w] = mk<double>(red[0][0] + red[0][1] + red[0][2] + red[0][3],
                                       red[1][0] + red[1][1] + red[1][2] + red[1][3]);
  }
}

// ---------------------------------------------------------------------------------------------
// Init-time FP64 precompute (H11; "need only be computed once at the start").
// Plain one-thread-per-output kernels: run once, not on the timed path.
// ---------------------------------------------------------------------------------------------

// h' = h - 1/2 sum_g L_g L_g   (H_2 = -1/2 sum v^2, v = i L)
__global__ void k_init_hprime(int M, int ng, const double* h, const double* L, double* hp) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= M * M) return;
  int i = e / M, j = e % M;
  double s = 0.0;
  for (int g = 0; g < ng; ++g) {
    const double* Lg = L + (size_t)g * M * M;
    double sg = 0.0;
    for (int k = 0; k < M; ++k) sg = fma(Lg[i * M + k], Lg[k * M + j], sg);
    s += sg;
  }
  hp[e] = h[e] - 0.5 * s;
}

// C = alpha * A B + beta * D   (all M x M, row-major, FP64)
__global__ void k_dgemm_small(int M, double alpha, const double* A, const double* B, double beta, const double* D,
                              double* C) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= M * M) return;
  int i = e / M, j = e % M;
  double s = 0.0;
  for (int k = 0; k < M; ++k) s = fma(A[i * M + k], B[k * M + j], s);
  C[e] = alpha * s + (D ? beta * D[e] : 0.0);
}
__global__ void k_dscale_eye(int M, double alpha, const double* A, double add_eye, double* C) {
  int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= M * M) return;
  C[e] = alpha * A[e] + ((e / M == e % M) ? add_eye : 0.0);
}

// Rd[g][soff + k*n + a] = sum_i C[i][a] X_g[i][k]   (X = L, ng matrices; or X = h with ng = 1)
__global__ void k_init_rot(int M, int n, int ldc, const double* C, int ng, const double* X, int soff, int KT, double* Rd) {
  size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  size_t tot = (size_t)ng * M * n;
  if (e >= tot) return;
  int g = (int)(e / ((size_t)M * n));
  int r = (int)(e - (size_t)g * M * n);
  int k = r / n, a = r % n;
  const double* Xg = X + (size_t)g * M * M;
  double s = 0.0;
  for (int i = 0; i < M; ++i) s = fma(C[i * ldc + a], Xg[i * M + k], s);
  Rd[(size_t)g * KT + soff + r] = s;
}

// Y^s[(k,a)][(l,b)] = sum_g R[g][(k,a)] R[g][(l,b)] - R[g][(l,a)] R[g][(k,b)]   (Eq.(5); R8).
// Y is symmetric and only enters through v^T Y v, so what is stored is Y' = upper triangle with the diagonal halved
// (v^T Y' v = 1/2 v^T Y v): the energy GEMM then skips the all-zero blocks below the diagonal.
template <typename T>
__global__ void k_init_Y(int M, int n, int ng, const double* Rd, int soff, int KT, T* Y, T* Y_lo, int ldy, int split) {
  int c = blockIdx.x * blockDim.x + threadIdx.x;
  int r = blockIdx.y;
  int Ks = M * n;
  if (c >= Ks) return;
  int k = r / n, a = r % n, l = c / n, b = c % n;
  const double* R = Rd + soff;
  double s = 0.0;
  for (int g = 0; g < (c >= r ? ng : 0); ++g) {
    const double* Rg = R + (size_t)g * KT;
    s = fma(Rg[r], Rg[c], s);
    s = fma(-Rg[l * n + a], Rg[k * n + b], s);
  }
  if (c == r) s *= 0.5;
  size_t o = (size_t)r * ldy + c;
  if (split) {
    float hi, lo;
    tf32_split((float)s, hi, lo);
    Y[o] = (T)hi; Y_lo[o] = (T)lo;
  } else {
    Y[o] = (T)s;
  }
}

// dst[r][c] (ld = ldd) = (T) src[c][r] (ld = lds), rows r < nr, cols c < nc ; optional tf32 split
template <typename T>
__global__ void k_transpose_cast(int nr, int nc, const double* src, size_t lds, T* dst, T* dst_lo, size_t ldd, int split) {
  __shared__ double tile[32][33];
  int c0 = blockIdx.x * 32, r0 = blockIdx.y * 32;
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int c = c0 + j, r = r0 + threadIdx.x;
    tile[j][threadIdx.x] = (c < nc && r < nr) ? src[(size_t)c * lds + r] : 0.0;
  }
  __syncthreads();
  for (int j = threadIdx.y; j < 32; j += blockDim.y) {
    int r = r0 + j, c = c0 + threadIdx.x;
    if (r < nr && c < nc) {
      double v = tile[threadIdx.x][j];
      size_t o = (size_t)r * ldd + c;
      if (split) {
        float hi, lo;
        tf32_split((float)v, hi, lo);
        dst[o] = (T)hi; dst_lo[o] = (T)lo;
      } else {
        dst[o] = (T)v;
      }
    }
  }
}

// dst[r][c] (ld = ldd) = (T) src[r][c] (ld = lds) ; optional split
template <typename T>
__global__ void k_cast2d(int nr, int nc, const double* src, size_t lds, T* dst, T* dst_lo, size_t ldd, int split) {
  size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (size_t)nr * nc) return;
  int r = (int)(e / nc), c = (int)(e % nc);
  double v = src[(size_t)r * lds + c];
  size_t o = (size_t)r * ldd + c;
  if (split) {
    float hi, lo;
    tf32_split((float)v, hi, lo);
    dst[o] = (T)hi; dst_lo[o] = (T)lo;
  } else {
    dst[o] = (T)v;
  }
}


// ---- multi-determinant energy: operands of the TT = C_act^T X Theta_0 GEMM (X = L_g for all g, then h) ----
// thT[((w*nt + a)*2 + p)*MPK + k] = Re/Im Theta_0[w][k][a]   (K-major rows (walker, column, plane), zero padded)
template <typename T>
__global__ void __launch_bounds__(128) k_thT(int M, int nt, int MPK, const cplx<T>* theta, T* thT, T* thT_lo) {
  const int w = blockIdx.x;
  for (int e = threadIdx.x; e < M * nt; e += blockDim.x) {
    int k = e / nt, a = e - k * nt;
    cplx<T> v = theta[(size_t)w * M * nt + e];
    const size_t o0 = (((size_t)w * nt + a) * 2 + 0) * MPK + k, o1 = o0 + MPK;
    if (thT_lo) {
      float h0, l0, h1, l1;
      tf32_split((float)v.x, h0, l0);
      tf32_split((float)v.y, h1, l1);
      thT[o0] = (T)h0; thT[o1] = (T)h1; thT_lo[o0] = (T)l0; thT_lo[o1] = (T)l1;
    } else {
      thT[o0] = v.x; thT[o1] = v.y;
    }
  }
}
// RactT[(g*nact + q)*MPK + k] = (C_act^T L_g)[q][k] for g < ng, (C_act^T h)[q][k] for g == ng
template <typename T>
__global__ void k_init_ractT(int ng, int nact, int M, int MPK, const double* Rd, int KT, const double* hrotd, T* out, T* out_lo) {
  size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  size_t tot = (size_t)(ng + 1) * nact * M;
  if (e >= tot) return;
  int k = (int)(e % M);
  int q = (int)((e / M) % nact);
  int g = (int)(e / ((size_t)M * nact));
  double v = g < ng ? Rd[(size_t)g * KT + k * nact + q] : hrotd[k * nact + q];
  const size_t o = ((size_t)g * nact + q) * MPK + k;
  if (out_lo) {
    float hi, lo;
    tf32_split((float)v, hi, lo);
    out[o] = (T)hi; out_lo[o] = (T)lo;
  } else {
    out[o] = (T)v;
  }
}


// Symmetric-packed K-major L for the tcgen05 assembly GEMM: row = block*128 + (i%8)*16 + (j%16) (see tc::EpiAssemble)
template <typename T>
__global__ void k_pack_Lt(int M, int ng, int NGP, int nblk, const int2* blk, const double* L, T* Lt, T* Lt_lo) {
  size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= (size_t)nblk * 128 * ng) return;
  int g = (int)(e % ng), r = (int)(e / ng);
  const int2 b = blk[r >> 7];
  int i = b.x * 8 + ((r >> 4) & 7), j = b.y * 16 + (r & 15);
  double v = (i < M && j < M) ? L[(size_t)g * M * M + (size_t)i * M + j] : 0.0;
  float hi, lo;
  tf32_split((float)v, hi, lo);
  Lt[(size_t)r * NGP + g] = (T)hi;
  Lt_lo[(size_t)r * NGP + g] = (T)lo;
}


// A[w][i][p][j] := A[w][j][p][i] for i > j (A_w is symmetric; the assembly GEMM wrote the upper blocks only).
// grid = (walkers, tile pairs TI >= TJ), block = 32 x 8; each CTA moves one 32 x 32 tile of both planes of both
// buffers (hi / lo) through shared memory: 16 independent loads per thread in flight.
template <typename T>
__global__ void __launch_bounds__(256) k_symmetrize(int M, int MP, T* A, T* A_lo) {
  __shared__ T tile[4][32][33];
  int t = blockIdx.y, TI = 0;
  while (t > TI) { t -= TI + 1; ++TI; }
  const int TJ = t;                        // TI >= TJ
  const int nbuf = A_lo ? 2 : 1;
  const size_t woff = ((size_t)blockIdx.x * M) * (2 * MP);
  const int tx = threadIdx.x, ty = threadIdx.y;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (q >= 2 * nbuf) break;
    const T* src = (q >> 1 ? A_lo : A) + woff + (q & 1) * MP;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
      int j = TJ * 32 + r, i = TI * 32 + tx;
      tile[q][r][tx] = (j < M && i < M) ? src[(size_t)j * (2 * MP) + i] : T(0);
    }
  }
  __syncthreads();
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    if (q >= 2 * nbuf) break;
    T* dst = (q >> 1 ? A_lo : A) + woff + (q & 1) * MP;
#pragma unroll
    for (int r = ty; r < 32; r += 8) {
      int i = TI * 32 + r, j = TJ * 32 + tx;
      if (i < M && j < M && i > j) dst[(size_t)i * (2 * MP) + j] = tile[q][tx][r];
    }
  }
}

}  // namespace afq
