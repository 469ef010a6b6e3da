// green.cuh -- H1-H3 + H8: overlap matrix, LU determinant / inverse, Theta, phaseless weight update.
// One CTA per walker; Phi is read from HBM once and Theta written once (HBM-bound stage).
// PAPER.md:51 (overlap, force bias, weights), :53 (phaseless rule), :61, :68 (A = psi_T^dagger phi).
#pragma once
#include "common.cuh"

namespace afq {

// Gauss-Jordan with partial pivoting on the augmented n x 2n matrix [A | I] held in shared memory,
// executed by ONE warp.  On exit the right block is A^-1; det = product of pivots (FP64, R17).
// sing bit 0: a pivot was exactly zero / NaN or below eps*max|A|.
template <typename T>
__device__ void warp_gauss_jordan(cplx<T>* aug, int n, int ld, cplx<T>* fac, int lane, zcplx& det, int& sing, T eps) {
  double dre = 1.0, dim = 0.0;
  sing = 0;
  T amax = T(0);
  for (int e = lane; e < n * n; e += 32) amax = fmax(amax, cabs2(aug[(e / n) * ld + (e % n)]));
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) amax = fmax(amax, __shfl_xor_sync(0xffffffffu, amax, o));
  const T thresh = amax * eps * eps;  // compare squared magnitudes
  for (int col = 0; col < n; ++col) {
    int r = col + lane;
    T mag = (r < n) ? cabs2(aug[r * ld + col]) : T(-1);
    int idx = r;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      T om = __shfl_xor_sync(0xffffffffu, mag, o);
      int oi = __shfl_xor_sync(0xffffffffu, idx, o);
      if (om > mag || (om == mag && oi < idx)) { mag = om; idx = oi; }
    }
    if (idx != col) {
      for (int c = lane; c < 2 * n; c += 32) {
        cplx<T> t = aug[col * ld + c];
        aug[col * ld + c] = aug[idx * ld + c];
        aug[idx * ld + c] = t;
      }
      dre = -dre; dim = -dim;
    }
    __syncwarp();
    cplx<T> p = aug[col * ld + col];
    if (!(mag > T(0))) { sing = 1; dre = 0.0; dim = 0.0; break; }
    if (mag < thresh) sing = 1;
    double nr = dre * (double)p.x - dim * (double)p.y;
    dim = dre * (double)p.y + dim * (double)p.x;
    dre = nr;
    cplx<T> ip = cinv(p);
    __syncwarp();
    for (int c = lane; c < 2 * n; c += 32) aug[col * ld + c] = cmul(aug[col * ld + c], ip);
    for (int rr = lane; rr < n; rr += 32) fac[rr] = aug[rr * ld + col];
    __syncwarp();
    for (int rr = 0; rr < n; ++rr) {
      if (rr == col) continue;
      cplx<T> f = fac[rr];
      for (int c = lane; c < 2 * n; c += 32) {
        cplx<T> v = aug[rr * ld + c];
        cplx<T> pr = aug[col * ld + c];
        v.x = fma(-f.x, pr.x, v.x); v.x = fma(f.y, pr.y, v.x);
        v.y = fma(-f.x, pr.y, v.y); v.y = fma(-f.y, pr.x, v.y);
        aug[rr * ld + c] = v;
      }
    }
    __syncwarp();
  }
  det = mk<double>(dre, dim);
}

template <typename T> struct GreenArgs {
  int M, na, nb, nw;
  const cplx<T>* phi;     // [nw][M][nt]
  const T* psi_a;         // [M][na]
  const T* psi_b;         // [M][nb]
  cplx<T>* theta;         // [nw][M][nt] or null
  T* thp;                 // planar [nw][2][KT]: spin-blocked index s_off + k*n_s + a ; may be null
  T* thp_lo;              // tf32 low plane (split != 0)
  int KA, KT, split;
  zcplx* ovlp;            // in: S (do_weight) ; out: S'
  int do_weight;
  const zcplx* cshift;    // c = x.xbar - xbar.xbar/2 per walker
  double* weight;
  const zcplx* eloc_pre;
  int weight_mode;
  double dt, E0;
  int* flags;
};

// shared-memory bytes needed by k_green
template <typename T> inline size_t green_smem_bytes(int M, int na, int nb) {
  int nt = na + nb, ns = na > nb ? na : nb;
  size_t b = ((size_t)M * nt * sizeof(cplx<T>) + 15) & ~size_t(15);   // phi_s
  b += (size_t)2 * ns * (2 * ns + 1) * sizeof(zcplx);   // aug per spin (FP64 on both precision paths)
  b += (size_t)2 * ns * sizeof(zcplx);                  // fac per spin
  b += 2 * sizeof(zcplx) + 4 * sizeof(int);
  return (b + 15) & ~size_t(15);
}

// Phaseless hybrid / local-energy weight update (R5, R6).  All FP64.
__device__ inline void weight_update(zcplx S_old, zcplx S_new, zcplx c, double w_old, double dt, double E0, int mode,
                                     double e_pre_re, double& w_new, int& flag) {
  zcplx rho = zdiv(S_new, S_old);
  double dtheta = atan2(rho.y, rho.x);
  double cosd = cos(dtheta);
  double fac;
  if (mode == 0) {
    double absI = exp(log(hypot(rho.x, rho.y)) + c.x);
    fac = exp(dt * E0) * absI;
  } else {
    fac = exp(-dt * (e_pre_re - E0));
  }
  bool killed = (cosd <= 0.0) || (w_old == 0.0);
  w_new = killed ? 0.0 : w_old * fac * cosd;
  if (cosd <= 0.0) flag |= FLAG_KILLED;
  if (!isfinite(w_new)) flag |= FLAG_NONFINITE;
}

template <typename T>
__global__ void __launch_bounds__(256) k_green(GreenArgs<T> g) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x;
  const int M = g.M, na = g.na, nb = g.nb, nt = na + nb, ns = na > nb ? na : nb;
  const int ld = 2 * ns + 1;
  cplx<T>* phi_s = reinterpret_cast<cplx<T>*>(smem_raw);
  // the small N x N work (overlap matrix, LU, inverse) is FP64 on both precision paths: it is
  // 0.3 % of the flops and keeps S, Theta accurate to cond(A) * eps of the FP32 walker itself
  zcplx* aug = reinterpret_cast<zcplx*>(smem_raw + (((size_t)M * nt * sizeof(cplx<T>) + 15) & ~size_t(15)));
  zcplx* fac = aug + 2 * ns * ld;
  zcplx* dets = fac + 2 * ns;
  int* sing = reinterpret_cast<int*>(dets + 2);

  const cplx<T>* phi_w = g.phi + (size_t)w * M * nt;
  for (int e = tid; e < M * nt; e += nthr) phi_s[e] = phi_w[e];
  __syncthreads();

  // A_s[a][b] = sum_k psi_s[k][a] phi[k][off+b]  (real x complex), augmented with the identity
  for (int e = tid; e < na * na + nb * nb; e += nthr) {
    int s = e >= na * na;
    int ee = s ? e - na * na : e;
    int n = s ? nb : na, off = s ? na : 0;
    const T* psi = s ? g.psi_b : g.psi_a;
    int a = ee / n, b = ee % n;
    double sr = 0.0, si = 0.0;
    for (int k = 0; k < M; ++k) {
      double p = (double)psi[k * n + a];
      cplx<T> v = phi_s[k * nt + off + b];
      sr = fma(p, (double)v.x, sr);
      si = fma(p, (double)v.y, si);
    }
    zcplx* A = aug + s * ns * ld;
    A[a * ld + b] = mk<double>(sr, si);
    A[a * ld + n + b] = mk<double>(a == b ? 1.0 : 0.0, 0.0);
  }
  __syncthreads();
  if (warp < 2) {
    int n = warp ? nb : na;
    zcplx det = mk<double>(1.0, 0.0);
    int sg = 0;
    if (n > 0) warp_gauss_jordan<double>(aug + warp * ns * ld, n, ld, fac + warp * ns, lane, det, sg, sizeof(T) == 4 ? 1e-6 : 1e-13);
    if (lane == 0) { dets[warp] = det; sing[warp] = sg; }
  }
  __syncthreads();

  // Theta_s = Phi_s A_s^-1
  for (int s = 0; s < 2; ++s) {
    int n = s ? nb : na, off = s ? na : 0, soff = s ? g.KA : 0;
    const zcplx* inv = aug + s * ns * ld + n;
    for (int e = tid; e < M * n; e += nthr) {
      int k = e / n, b = e % n;
      zcplx accd = mk<double>(0.0, 0.0);
      for (int a = 0; a < n; ++a) cfma(accd, to_z(phi_s[k * nt + off + a]), inv[a * ld + b]);
      cplx<T> acc = mk<T>((T)accd.x, (T)accd.y);
      if (g.theta) g.theta[(size_t)w * M * nt + k * nt + off + b] = acc;
      if (g.thp) {
        size_t o = (size_t)(2 * w) * g.KT + soff + e;
        if (g.split) {
          float h0, l0, h1, l1;
          tf32_split((float)acc.x, h0, l0);
          tf32_split((float)acc.y, h1, l1);
          g.thp[o] = (T)h0; g.thp[o + g.KT] = (T)h1;
          g.thp_lo[o] = (T)l0; g.thp_lo[o + g.KT] = (T)l1;
        } else {
          g.thp[o] = acc.x; g.thp[o + g.KT] = acc.y;
        }
      }
    }
  }

  if (tid == 0) {
    zcplx da = dets[0], db = dets[1];
    zcplx S_new = mk<double>(da.x * db.x - da.y * db.y, da.x * db.y + da.y * db.x);
    int flag = (sing[0] | sing[1]) ? FLAG_SINGULAR : 0;
    if (!isfinite(S_new.x) || !isfinite(S_new.y)) flag |= FLAG_NONFINITE;
    if (g.do_weight) {
      double w_new;
      double epre = g.eloc_pre ? g.eloc_pre[w].x : 0.0;
      weight_update(g.ovlp[w], S_new, g.cshift[w], g.weight[w], g.dt, g.E0, g.weight_mode, epre, w_new, flag);
      g.weight[w] = w_new;
    }
    g.ovlp[w] = S_new;
    if (g.flags && flag) atomicOr(&g.flags[w], flag);
  }
}

// Full Green's function on request: G_s[i][j] = sum_a Theta_s[j][a] psi_s[i][a]  (R15).
template <typename T>
__global__ void k_gfull(int M, int na, int nb, const cplx<T>* theta, const T* psi_a, const T* psi_b, cplx<T>* G) {
  const int w = blockIdx.y, s = blockIdx.z, nt = na + nb;
  const int n = s ? nb : na, off = s ? na : 0;
  const T* psi = s ? psi_b : psi_a;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < M * M; e += gridDim.x * blockDim.x) {
    int i = e / M, j = e % M;
    T sr = T(0), si = T(0);
    for (int a = 0; a < n; ++a) {
      cplx<T> t = theta[(size_t)w * M * nt + j * nt + off + a];
      T p = psi[i * n + a];
      sr = fma(p, t.x, sr);
      si = fma(p, t.y, si);
    }
    G[((size_t)(w * 2 + s) * M + i) * M + j] = mk<T>(sr, si);
  }
}

// interleaved Theta [nw][M][nt] -> planar spin-blocked [nw][2][KT] (hi/lo split on request)
template <typename T>
__global__ void k_planarize(int M, int na, int nb, int KA, int KT, int split, const cplx<T>* theta, T* thp, T* thp_lo) {
  const int w = blockIdx.x, nt = na + nb;
  for (int e = threadIdx.x; e < M * nt; e += blockDim.x) {
    int k = e / nt, c = e % nt;
    int s = c >= na;
    int n = s ? nb : na, b = s ? c - na : c;
    cplx<T> v = theta[(size_t)w * M * nt + e];
    size_t o = (size_t)(2 * w) * KT + (s ? KA : 0) + k * n + b;
    if (split) {
      float h0, l0, h1, l1;
      tf32_split((float)v.x, h0, l0);
      tf32_split((float)v.y, h1, l1);
      thp[o] = (T)h0; thp[o + KT] = (T)h1;
      thp_lo[o] = (T)l0; thp_lo[o + KT] = (T)l1;
    } else {
      thp[o] = v.x; thp[o + KT] = v.y;
    }
  }
}

}  // namespace afq
