// green.cuh -- H1-H3 + H8: overlap matrix, LU determinant / inverse, Theta, phaseless weight update.
// One CTA per walker; Phi is read from HBM once and Theta written once (HBM-bound stage).
// PAPER.md:51 (overlap, force bias, weights), :53 (phaseless rule), :61, :68 (A = psi_T^dagger phi).
#pragma once
#include "common.cuh"

namespace afq {

// In-place Gauss-Jordan inverse with partial (row) pivoting, executed by a GROUP of 128 threads (4 warps, named barrier
// `bar_id`).  The n x n matrix ping-pongs between two dense buffers (row stride n): every pivot step reads one and writes
// the other, so a step costs two group barriers (factors ready; update done).  No augmentation with the identity: the
// column of the pivot is overwritten with the column the identity would have produced (-f / p, and 1 / p in the pivot
// row), which halves the update work and the shared memory of the augmented form.  Row interchanges of A are column
// interchanges of the inverse, applied at the end in reverse order -- here composed into cperm[]: inverse[a][b] =
// result[a * n + cperm[b]].  The pivot search is done by every warp of the group redundantly (same shuffles, same
// result): no barrier between the search and the factor computation.  det / sing are identical in all threads.
// Returns the buffer that holds the result.
__device__ inline zcplx* group_gauss_jordan(zcplx* bufA, zcplx* bufB, int n, zcplx* fac, zcplx* prow, int* ipiv, int* cperm, int gtid,
                                            int bar_id, zcplx& det, int& sing, double eps) {
  const int lane = gtid & 31, gwarp = gtid >> 5;
  double dre = 1.0, dim = 0.0;
  sing = 0;
  double thresh = 0.0;
  {
    double amax = 0.0;
    for (int e = lane; e < n * n; e += 32) amax = fmax(amax, cabs2(bufA[e]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = fmax(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    thresh = amax * eps * eps;
  }
  zcplx* cur = bufA;
  zcplx* nxt = bufB;
  int done = 0;
  for (int col = 0; col < n; ++col) {
    int piv;
    zcplx ip = mk<double>(0.0, 0.0);
    {
      int r = col + lane;
      double mag = (r < n) ? cabs2(cur[r * n + col]) : -1.0;
      int idx = r;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        double om = __shfl_xor_sync(0xffffffffu, mag, o);
        int oi = __shfl_xor_sync(0xffffffffu, idx, o);
        if (om > mag || (om == mag && oi < idx)) { mag = om; idx = oi; }
      }
      const bool dead = !(mag > 0.0);
      if (dead) { sing = 1; dre = 0.0; dim = 0.0; piv = -1; }
      else {
        if (mag < thresh) sing = 1;
        if (idx != col) { dre = -dre; dim = -dim; }
        const zcplx p = cur[idx * n + col];
        double nr = dre * p.x - dim * p.y;
        dim = dre * p.y + dim * p.x;
        dre = nr;
        piv = idx;
        if (gtid < n) ip = cinv(p);     // only the threads that scale the pivot row need the FP64 reciprocal
      }
    }
    if (piv < 0) break;                                   // exactly singular: uniform exit (all warps agree)
    // scaled pivot row (its pivot-column entry is the reciprocal itself) and the factors (column col, rows permuted)
    if (gtid < n) prow[gtid] = gtid == col ? ip : cmul(cur[piv * n + gtid], ip);
    for (int r = gtid; r < n; r += 128) fac[r] = cur[(r == col ? piv : (r == piv ? col : r)) * n + col];
    if (gtid == 0) ipiv[col] = piv;
    asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
    // new row r <- (rows col, piv swapped) - fac[r] * prow, with 0 in place of the old pivot-column entry; new row col <- prow
    if (lane < n) {
      const int c = lane;
      const zcplx pr = prow[c];
      for (int r = gwarp; r < n; r += 4) {
        zcplx v;
        if (r == col) v = pr;
        else {
          const int src = (r == piv) ? col : r;            // the old row `col` moves to position piv
          v = c == col ? mk<double>(0.0, 0.0) : cur[src * n + c];
          const zcplx f = fac[r];
          v.x = fma(-f.x, pr.x, v.x); v.x = fma(f.y, pr.y, v.x);
          v.y = fma(-f.x, pr.y, v.y); v.y = fma(-f.y, pr.x, v.y);
        }
        nxt[r * n + c] = v;
      }
    }
    asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
    zcplx* t = cur; cur = nxt; nxt = t;
    ++done;
  }
  if (gtid == 0) {   // column order of the inverse: undo the row interchanges, last one first
    for (int c = 0; c < n; ++c) cperm[c] = c;
    for (int col = done - 1; col >= 0; --col) {
      const int q = ipiv[col];
      if (q != col) { const int t = cperm[col]; cperm[col] = cperm[q]; cperm[q] = t; }
    }
  }
  asm volatile("bar.sync %0, 128;" ::"r"(bar_id) : "memory");
  det = mk<double>(dre, dim);
  return cur;
}

template <typename T> struct GreenArgs {
  int M, na, nb, nw;
  const cplx<T>* phi;     // [nw][M][nt]
  const T* psi_a;         // [M][na]
  const T* psi_b;         // [M][nb]
  const double* psid_a;   // FP64 copies (no per-iteration conversion in the overlap loop)
  const double* psid_b;
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
  b += (size_t)4 * ns * ns * sizeof(zcplx);             // per spin: two ping-pong n x n buffers (FP64 on both precision paths)
  b += (size_t)4 * ns * sizeof(zcplx);                  // per spin: factors, scaled pivot row
  b += 2 * sizeof(zcplx) + (8 + 4 * ns) * sizeof(int);  // dets; sing, result buffer, ipiv, cperm
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
  // max{0, cos dtheta}: cos dtheta = Re(rho)/|rho|, so the decision is taken on Re(rho) itself (reading R6b): cos(atan2(y, x))
  // is 6e-17 > 0 at x = 0 and for tiny negative x
  const bool dead = rho.x <= 0.0;
  bool killed = dead || (w_old == 0.0);
  w_new = killed ? 0.0 : w_old * fac * cosd;
  if (dead) flag |= FLAG_KILLED;
  if (!isfinite(w_new)) flag |= FLAG_NONFINITE;
}

template <typename T>
__global__ void __launch_bounds__(256, 4) k_green(GreenArgs<T> g) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int w = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nthr = blockDim.x;
  const int M = g.M, na = g.na, nb = g.nb, nt = na + nb, ns = na > nb ? na : nb;
  cplx<T>* phi_s = reinterpret_cast<cplx<T>*>(smem_raw);
  // the small N x N work (overlap matrix, inverse) is FP64 on both precision paths: it is
  // 0.3 % of the flops and keeps S, Theta accurate to cond(A) * eps of the FP32 walker itself
  zcplx* mats = reinterpret_cast<zcplx*>(smem_raw + (((size_t)M * nt * sizeof(cplx<T>) + 15) & ~size_t(15)));   // [spin][2][ns*ns]
  zcplx* fac = mats + 4 * ns * ns;           // [spin][ns] factors, then [spin][ns] scaled pivot rows
  zcplx* dets = fac + 4 * ns;
  int* sing = reinterpret_cast<int*>(dets + 2);
  int* resb = sing + 2;                      // which ping-pong buffer holds the inverse of spin s
  int* ipiv = sing + 8;                      // [spin][ns]
  int* cperm = ipiv + 2 * ns;                // [spin][ns]

  const cplx<T>* phi_w = g.phi + (size_t)w * M * nt;
  for (int e = tid; e < M * nt; e += nthr) phi_s[e] = phi_w[e];
  __syncthreads();

  // A_s[a][b] = sum_k psi_s[k][a] phi[k][off+b]  (real x complex, FP64), dense n x n in the first ping-pong buffer of spin s.
  // FP64 issue slots are the scarce resource here (conversions included), so one work item = (spin, column b, group
  // of 4 rows a, half of the k range): phi[k][b] is converted once and reused for 4 rows; halves meet in shared atomics.
  for (int e = tid; e < 4 * ns * ns; e += nthr) mats[e] = mk<double>(0.0, 0.0);
  __syncthreads();
  {
    const int ga = (na + 3) >> 2, gb = (nb + 3) >> 2;
    const int items_a = na * ga * 2, items = items_a + nb * gb * 2;
    for (int e = tid; e < items; e += nthr) {
      const int s = e >= items_a;
      const int ee = s ? e - items_a : e;
      const int n = s ? nb : na, off = s ? na : 0, gn = s ? gb : ga;
      const double* psi = s ? g.psid_b : g.psid_a;
      const int kh = ee & 1, b = (ee >> 1) % n, a0 = ((ee >> 1) / n) * 4;
      (void)gn;
      const int k0 = kh ? (M >> 1) : 0, k1 = kh ? M : (M >> 1);
      double sr[4] = {0.0, 0.0, 0.0, 0.0}, si[4] = {0.0, 0.0, 0.0, 0.0};
      for (int k = k0; k < k1; ++k) {
        const cplx<T> v = phi_s[k * nt + off + b];
        const double vr = (double)v.x, vi = (double)v.y;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const double pu = (a0 + u < n) ? psi[k * n + a0 + u] : 0.0;
          sr[u] = fma(pu, vr, sr[u]);
          si[u] = fma(pu, vi, si[u]);
        }
      }
      zcplx* A = mats + s * 2 * ns * ns;     // dense n x n, row stride n
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (a0 + u < n) {
          double* dst = reinterpret_cast<double*>(&A[(a0 + u) * n + b]);
          atomicAdd(dst, sr[u]); atomicAdd(dst + 1, si[u]);
        }
    }
  }
  __syncthreads();
  {
    // warps 0-3 invert A_alpha, warps 4-7 A_beta (named barriers 1 / 2)
    const int grp = warp >> 2, n = grp ? nb : na;
    zcplx det = mk<double>(1.0, 0.0);
    int sg = 0;
    zcplx* res = mats + grp * 2 * ns * ns;
    if (n > 0)
      res = group_gauss_jordan(mats + grp * 2 * ns * ns, mats + grp * 2 * ns * ns + ns * ns, n, fac + grp * ns, fac + 2 * ns + grp * ns,
                               ipiv + grp * ns, cperm + grp * ns, tid & 127, 1 + grp, det, sg, sizeof(T) == 4 ? 1e-6 : 1e-13);
    if ((tid & 127) == 0) { dets[grp] = det; sing[grp] = sg; resb[grp] = res != mats + grp * 2 * ns * ns; }
  }
  __syncthreads();

  // Theta_s = Phi_s A_s^-1.  FP32 path: the FP64 inverse is split into FP32 hi + lo parts and the product runs on the
  // FP32 pipe (the walker itself is FP32, so FP64 products bought nothing but FP64 issue slots); FP64 path unchanged.
  // inverse of spin s: res_s[a * n + cperm_s[b]]; its FP32 hi / lo split goes into the OTHER ping-pong buffer of that spin
  // ([n*n][hi, lo] complex64 = the same bytes as n*n complex128)
  if constexpr (sizeof(T) == 4) {
    for (int e = tid; e < na * na + nb * nb; e += nthr) {
      const int s = e >= na * na, ee = s ? e - na * na : e, n = s ? nb : na;
      const zcplx* res = mats + (s * 2 + resb[s]) * ns * ns;
      cplx<float>* invf = reinterpret_cast<cplx<float>*>(mats + (s * 2 + (resb[s] ^ 1)) * ns * ns);
      const zcplx v = res[(ee / n) * n + cperm[s * ns + (ee % n)]];
      const float hr = (float)v.x, hi = (float)v.y;
      invf[ee * 2 + 0] = mk<float>(hr, hi);
      invf[ee * 2 + 1] = mk<float>((float)(v.x - (double)hr), (float)(v.y - (double)hi));
    }
    __syncthreads();
  }
  if constexpr (sizeof(T) == 4) {
    // register tile: one thread = column b of four rows k, k + Mq, k + 2 Mq, k + 3 Mq (Mq = ceil(M/4)); the hi/lo pair of
    // inv[a][b] is one 16-byte shared load reused by the four rows, and for a fixed row slot consecutive threads
    // write consecutive elements of Theta and of the planar operand
    const int Mq = (M + 3) >> 2;
    for (int s = 0; s < 2; ++s) {
      const int n = s ? nb : na, off = s ? na : 0, soff = s ? g.KA : 0;
      const float4* iv = reinterpret_cast<const float4*>(mats + (s * 2 + (resb[s] ^ 1)) * ns * ns);
      for (int e = tid; e < Mq * n; e += nthr) {
        const int kg = e / n, b = e - kg * n;
        cplx<float> ah[4], al[4];
        int kk[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          ah[u] = mk<float>(0.f, 0.f); al[u] = mk<float>(0.f, 0.f);
          const int k = kg + u * Mq;
          kk[u] = k < M ? k : M - 1;
        }
        for (int a = 0; a < n; ++a) {
          const float4 v = iv[a * n + b];
          const cplx<float> vh = mk<float>(v.x, v.y), vl = mk<float>(v.z, v.w);
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const cplx<T> p = phi_s[kk[u] * nt + off + a];
            const cplx<float> ph = mk<float>((float)p.x, (float)p.y);
            cfma(ah[u], ph, vh);
            cfma(al[u], ph, vl);
          }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int k = kg + u * Mq;
          if (k >= M) continue;
          const cplx<T> acc = mk<T>((T)(ah[u].x + al[u].x), (T)(ah[u].y + al[u].y));
          if (g.theta) g.theta[(size_t)w * M * nt + k * nt + off + b] = acc;
          if (g.thp) {
            const size_t o = (size_t)(2 * w) * g.KT + soff + k * n + b;
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
    }
  } else {
    for (int s = 0; s < 2; ++s) {
      int n = s ? nb : na, off = s ? na : 0, soff = s ? g.KA : 0;
      const zcplx* inv = mats + (s * 2 + resb[s]) * ns * ns;
      const int* cp = cperm + s * ns;
      for (int e = tid; e < M * n; e += nthr) {
        int k = e / n, b = e % n;
        zcplx accd = mk<double>(0.0, 0.0);
        for (int a = 0; a < n; ++a) cfma(accd, to_z(phi_s[k * nt + off + a]), inv[a * n + cp[b]]);
        cplx<T> acc = mk<T>((T)accd.x, (T)accd.y);
        if (g.theta) g.theta[(size_t)w * M * nt + k * nt + off + b] = acc;
        if (g.thp) {
          size_t o = (size_t)(2 * w) * g.KT + soff + e;
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
  const int w = blockIdx.x, s = blockIdx.z, nt = na + nb;
  const int n = s ? nb : na, off = s ? na : 0;
  const T* psi = s ? psi_b : psi_a;
  for (int e = blockIdx.y * blockDim.x + threadIdx.x; e < M * M; e += gridDim.y * blockDim.x) {
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
