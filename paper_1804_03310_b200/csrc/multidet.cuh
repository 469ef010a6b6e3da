// multidet.cuh -- H10: multi-determinant trial |Psi_T> = sum_i c_i |psi_i> (Eq.(4)).
// Every determinant is the reference with <= 2 columns per spin replaced by active-space orbitals, so
// all overlaps / Green's functions follow from the reference by Sherman-Morrison-Woodbury rank-E updates:
//   Q = C_act^T Theta_0,  Q_i = Q[P_i,H_i] (E x E),  det A_i / det A_0 = det Q_i,  Z_i = Q_i^-1,
//   Theta_i psi_i^T = Theta_0 psi_0^T + Theta_0[:,H_i] Z_i R[P_i,:],  R = C_virt^T - Q_virt psi_0^T.
// One CTA per walker; determinant-level scalars are FP64 on both precision paths (H10).
#pragma once
#include "common.cuh"
#include "green.cuh"

namespace afq {

__device__ __forceinline__ zcplx zmul(zcplx a, zcplx b) { return mk<double>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ zcplx zadd(zcplx a, zcplx b) { return mk<double>(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ zcplx zsub(zcplx a, zcplx b) { return mk<double>(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ zcplx zscale(zcplx a, double s) { return mk<double>(a.x * s, a.y * s); }

struct MdConst {
  int M, na, nb, nact, ndet;
  int emax;                // slots per spin in exc: 2 (excitation rank <= 2, closed forms) or 4 (rank <= 4, general small elimination)
  const void* C;           // [M][nact]  (T)
  const double* coeff;     // [ndet]
  const int32_t* exc;      // [ndet][2][emax][2] (hole, particle) or -1
};

// Shared-memory view used by both multi-det kernels.
struct MdSmem {
  zcplx* Qv[2];    // [nvirt_s][n_s]     Q_virt = C_virt^T Theta_0
  zcplx* Z;        // [ndet][2][emax^2]  Z_i^s[f][e] (row = hole slot f, col = particle slot e), index md_zidx(rank, f, e)
  zcplx* omega;    // [ndet]             c_i S_i / S
  int8_t* rank;    // [ndet][2]          excitation rank per spin
  zcplx* red;      // [64] reduction scratch
  int* flag;       // bit 0: a determinant has exactly zero overlap with the walker (its Z is undefined)
};

inline size_t md_smem_bytes(int na, int nb, int nact, int ndet, int emax = 2) {
  size_t b = (size_t)((nact - na) * na + (nact - nb) * nb) * sizeof(zcplx);
  b += (size_t)ndet * 2 * emax * emax * sizeof(zcplx) + (size_t)ndet * sizeof(zcplx) + 64 * sizeof(zcplx);
  b += ((size_t)ndet * 2 + 15) & ~size_t(15);
  b += 16;
  return b;
}

__device__ inline unsigned char* md_carve(unsigned char* p, const MdConst& m, MdSmem& s) {
  s.Qv[0] = reinterpret_cast<zcplx*>(p); p += (size_t)(m.nact - m.na) * m.na * sizeof(zcplx);
  s.Qv[1] = reinterpret_cast<zcplx*>(p); p += (size_t)(m.nact - m.nb) * m.nb * sizeof(zcplx);
  s.Z = reinterpret_cast<zcplx*>(p); p += (size_t)m.ndet * 2 * m.emax * m.emax * sizeof(zcplx);
  s.omega = reinterpret_cast<zcplx*>(p); p += (size_t)m.ndet * sizeof(zcplx);
  s.red = reinterpret_cast<zcplx*>(p); p += 64 * sizeof(zcplx);
  s.rank = reinterpret_cast<int8_t*>(p); p += ((size_t)m.ndet * 2 + 15) & ~size_t(15);
  s.flag = reinterpret_cast<int*>(p); p += 16;
  return p;
}

// block-wide complex sum (all threads call); result broadcast
__device__ inline zcplx block_sum(zcplx v, zcplx* red) {
  v.x = warp_sum(v.x); v.y = warp_sum(v.y);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nwarp = (blockDim.x + 31) >> 5;
  __syncthreads();
  if (lane == 0) red[wid] = v;
  __syncthreads();
  zcplx t = mk<double>(0.0, 0.0);
  for (int i = 0; i < nwarp; ++i) t = zadd(t, red[i]);
  __syncthreads();
  return t;
}

// canonical (hole, particle) slots of determinant i, spin sp (valid pairs first, in list order); returns the rank
__device__ __forceinline__ int md_exc(const MdConst& m, int i, int sp, int (&h)[4], int (&p)[4]) {
  const int32_t* ex = m.exc + ((size_t)i * 2 + sp) * 2 * m.emax;
  int rk = 0;
#pragma unroll
  for (int e = 0; e < 4; ++e) { h[e] = -1; p[e] = -1; }
  for (int e = 0; e < m.emax; ++e)
    if (ex[2 * e] >= 0) { h[rk] = ex[2 * e]; p[rk] = ex[2 * e + 1]; ++rk; }
  return rk;
}

// index of Z[f][e] inside a determinant's block: rank 1 and 2 keep the layout of the closed forms, rank 3 and 4 use rows of 4
__device__ __forceinline__ int md_zidx(int rk, int f, int e) { return rk == 1 ? 0 : (rk == 2 ? f * 2 + e : f * 4 + e); }

// determinant and inverse of the rk x rk matrix A (rk <= 4, row-major, stride 4) by Gauss-Jordan with partial pivoting; inv row-major
// stride 4.  An exactly singular matrix returns det = 0 and leaves inv zero (the caller flags the walker).  FP64.
__device__ inline zcplx md_small_inverse(int rk, zcplx (&A)[16], zcplx (&inv)[16]) {
  for (int e = 0; e < 16; ++e) inv[e] = mk<double>(((e >> 2) == (e & 3)) ? 1.0 : 0.0, 0.0);
  zcplx det = mk<double>(1.0, 0.0);
  for (int c = 0; c < rk; ++c) {
    int piv = c; double best = cabs2(A[c * 4 + c]);
    for (int r = c + 1; r < rk; ++r) { const double m2 = cabs2(A[r * 4 + c]); if (m2 > best) { best = m2; piv = r; } }
    if (!(best > 0.0)) {
      for (int e = 0; e < 16; ++e) inv[e] = mk<double>(0.0, 0.0);
      return mk<double>(0.0, 0.0);
    }
    if (piv != c) {
      for (int k = 0; k < rk; ++k) {
        zcplx t = A[c * 4 + k]; A[c * 4 + k] = A[piv * 4 + k]; A[piv * 4 + k] = t;
        t = inv[c * 4 + k]; inv[c * 4 + k] = inv[piv * 4 + k]; inv[piv * 4 + k] = t;
      }
      det = mk<double>(-det.x, -det.y);
    }
    const zcplx pv = A[c * 4 + c];
    det = zmul(det, pv);
    const zcplx ip = zdiv(mk<double>(1.0, 0.0), pv);
    for (int k = 0; k < rk; ++k) { A[c * 4 + k] = zmul(A[c * 4 + k], ip); inv[c * 4 + k] = zmul(inv[c * 4 + k], ip); }
    for (int r = 0; r < rk; ++r) {
      if (r == c) continue;
      const zcplx f = A[r * 4 + c];
      for (int k = 0; k < rk; ++k) {
        A[r * 4 + k] = zsub(A[r * 4 + k], zmul(f, A[c * 4 + k]));
        inv[r * 4 + k] = zsub(inv[r * 4 + k], zmul(f, inv[c * 4 + k]));
      }
    }
  }
  return det;
}

// From Theta_0 (shared, [M][nt] complex T): Q_virt, per-determinant ratios r_i, Z_i, mixing weights
// omega_i = c_i r_i^a r_i^b / sum_j c_j r_j^a r_j^b.  Returns the sum (S / S_0).  All threads call.
template <typename T>
__device__ zcplx md_prepare(const MdConst& m, const cplx<T>* th0, MdSmem& s) {
  const int nt = m.na + m.nb, tid = threadIdx.x, nthr = blockDim.x;
  const T* C = reinterpret_cast<const T*>(m.C);
  if (tid == 0) *s.flag = 0;
  for (int sp = 0; sp < 2; ++sp) {
    const int n = sp ? m.nb : m.na, off = sp ? m.na : 0, nv = m.nact - n;
    for (int e = tid; e < nv * n; e += nthr) {
      int p = e / n, h = e - p * n;
      double sr = 0.0, si = 0.0;
      for (int k = 0; k < m.M; ++k) {
        double c = (double)C[k * m.nact + n + p];
        cplx<T> v = th0[k * nt + off + h];
        sr = fma(c, (double)v.x, sr);
        si = fma(c, (double)v.y, si);
      }
      s.Qv[sp][e] = mk<double>(sr, si);
    }
  }
  __syncthreads();
  zcplx part = mk<double>(0.0, 0.0);
  for (int i = tid; i < m.ndet; i += nthr) {
    zcplx ratio = mk<double>(1.0, 0.0);
    for (int sp = 0; sp < 2; ++sp) {
      const int n = sp ? m.nb : m.na;
      int hs[4], ps[4];
      const int rk = md_exc(m, i, sp, hs, ps);
      const int h0 = hs[0], p0 = ps[0], h1 = hs[1], p1 = ps[1];
      s.rank[i * 2 + sp] = (int8_t)rk;
      zcplx* Zi = s.Z + ((size_t)i * 2 + sp) * m.emax * m.emax;
      const zcplx* Q = s.Qv[sp];
      if (rk == 1) {
        zcplx q = Q[(p0 - n) * n + h0];
        ratio = zmul(ratio, q);
        if (q.x == 0.0 && q.y == 0.0) { Zi[0] = q; atomicOr(s.flag, 1); }   // zero overlap: dropped, flagged
        else Zi[0] = zdiv(mk<double>(1.0, 0.0), q);
      } else if (rk == 2) {
        zcplx a = Q[(p0 - n) * n + h0], b = Q[(p0 - n) * n + h1];
        zcplx c = Q[(p1 - n) * n + h0], d = Q[(p1 - n) * n + h1];
        zcplx det = zsub(zmul(a, d), zmul(b, c));
        const bool zero = det.x == 0.0 && det.y == 0.0;
        zcplx id = zero ? det : zdiv(mk<double>(1.0, 0.0), det);
        if (zero) atomicOr(s.flag, 1);
        ratio = zmul(ratio, det);
        // inverse of [[a,b],[c,d]] (rows = particle slot, cols = hole slot): Z[f][e]
        Zi[0] = zmul(d, id);
        Zi[1] = zmul(mk<double>(-b.x, -b.y), id);
        Zi[2] = zmul(mk<double>(-c.x, -c.y), id);
        Zi[3] = zmul(a, id);
      } else if (rk >= 3) {
        // Q_i[e][f] = Q[p_e][h_f] (rows = particle slot, columns = hole slot); Z = Q_i^-1, Z[f][e]
        zcplx A[16], inv[16];
        for (int e = 0; e < rk; ++e)
          for (int f = 0; f < rk; ++f) A[e * 4 + f] = Q[(ps[e] - n) * n + hs[f]];
        const zcplx det = md_small_inverse(rk, A, inv);
        if (det.x == 0.0 && det.y == 0.0) atomicOr(s.flag, 1);
        ratio = zmul(ratio, det);
        for (int f = 0; f < rk; ++f)
          for (int e = 0; e < rk; ++e) Zi[f * 4 + e] = inv[f * 4 + e];
      }
    }
    zcplx cr = zscale(ratio, m.coeff[i]);
    s.omega[i] = cr;
    part = zadd(part, cr);
  }
  zcplx tot = block_sum(part, s.red);
  for (int i = tid; i < m.ndet; i += nthr) s.omega[i] = zdiv(s.omega[i], tot);
  __syncthreads();
  return tot;
}


template <typename T> struct MdOverlapArgs {
  MdConst m;
  const cplx<T>* theta0;   // [nw][M][nt]   reference Theta_0 (from k_green)
  const zcplx* ovlp0;      // [nw]          reference overlap det A_0^a det A_0^b
  cplx<T>* thtil;          // [nw][M][2*nact]  generalised half-rotated mixed Green's function:
                           //   mixed G_s^T = Thtil_s C_act^T,  Thtil_s = [Theta_0 - Theta_0 B Q_virt | Theta_0 B]
  zcplx* ovlp;             // in: S (do_weight) ; out: S' = S_0 sum_i c_i r_i
  int do_weight;
  const zcplx* cshift; double* weight; const zcplx* eloc_pre; int weight_mode; double dt, E0;
  int* flags;
};

inline size_t md_overlap_smem(int M, int na, int nb, int nact, int ndet, int ts, int emax = 2) {
  size_t b = md_smem_bytes(na, nb, nact, ndet, emax);
  b += ((size_t)M * (na + nb) * 2 * ts + 15) & ~size_t(15);
  b += (size_t)(na * (nact - na) + nb * (nact - nb)) * sizeof(zcplx);   // Btil
  b += (size_t)(na * na + nb * nb) * sizeof(zcplx);                     // Btil Q_virt
  return b;
}

template <typename T>
__global__ void __launch_bounds__(256) k_md_overlap(MdOverlapArgs<T> g) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const MdConst& m = g.m;
  const int w = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x, nt = m.na + m.nb, M = m.M;
  MdSmem s;
  unsigned char* p = md_carve(smem_raw, m, s);
  cplx<T>* th0 = reinterpret_cast<cplx<T>*>(p);
  p += ((size_t)M * nt * sizeof(cplx<T>) + 15) & ~size_t(15);
  zcplx* Bt[2]; zcplx* BQ[2];
  Bt[0] = reinterpret_cast<zcplx*>(p); Bt[1] = Bt[0] + m.na * (m.nact - m.na);
  BQ[0] = Bt[1] + m.nb * (m.nact - m.nb); BQ[1] = BQ[0] + m.na * m.na;
  for (int e = tid; e < M * nt; e += nthr) th0[e] = g.theta0[(size_t)w * M * nt + e];
  const int nbt = m.na * (m.nact - m.na) + m.nb * (m.nact - m.nb);
  for (int e = tid; e < nbt; e += nthr) Bt[0][e] = mk<double>(0.0, 0.0);
  __syncthreads();
  zcplx tot = md_prepare<T>(m, th0, s);
  // Btil_s[h][p] = sum_i omega_i Z_i^s[f][e] at (h_f, p_e)
  for (int i = tid; i < m.ndet; i += nthr) {
    zcplx om = s.omega[i];
    for (int sp = 0; sp < 2; ++sp) {
      int h[4], pp[4];
      int rk = md_exc(m, i, sp, h, pp);
      const int n = sp ? m.nb : m.na, nv = m.nact - n;
      const zcplx* Zi = s.Z + ((size_t)i * 2 + sp) * m.emax * m.emax;
      for (int f = 0; f < rk; ++f)
        for (int e = 0; e < rk; ++e) {
          zcplx v = zmul(om, Zi[md_zidx(rk, f, e)]);
          double* dst = reinterpret_cast<double*>(&Bt[sp][h[f] * nv + (pp[e] - n)]);
          atomicAdd(dst, v.x); atomicAdd(dst + 1, v.y);
        }
    }
  }
  __syncthreads();
  for (int sp = 0; sp < 2; ++sp) {
    const int n = sp ? m.nb : m.na, nv = m.nact - n;
    for (int e = tid; e < n * n; e += nthr) {
      int h1 = e / n, h2 = e - h1 * n;
      zcplx a = mk<double>(0.0, 0.0);
      for (int q = 0; q < nv; ++q) a = zadd(a, zmul(Bt[sp][h1 * nv + q], s.Qv[sp][q * n + h2]));
      BQ[sp][e] = a;
    }
  }
  __syncthreads();
  for (int sp = 0; sp < 2; ++sp) {
    const int n = sp ? m.nb : m.na, nv = m.nact - n, off = sp ? m.na : 0;
    for (int e = tid; e < M * m.nact; e += nthr) {
      int k = e / m.nact, q = e - k * m.nact;
      zcplx a;
      if (q < n) {
        a = to_z(th0[k * nt + off + q]);
        for (int h = 0; h < n; ++h) a = zsub(a, zmul(to_z(th0[k * nt + off + h]), BQ[sp][h * n + q]));
      } else {
        a = mk<double>(0.0, 0.0);
        for (int h = 0; h < n; ++h) a = zadd(a, zmul(to_z(th0[k * nt + off + h]), Bt[sp][h * nv + (q - n)]));
      }
      g.thtil[((size_t)w * M + k) * (2 * m.nact) + sp * m.nact + q] = mk<T>((T)a.x, (T)a.y);
    }
  }
  if (tid == 0) {
    zcplx S_new = zmul(g.ovlp0[w], tot);
    int flag = (*s.flag & 1) ? FLAG_SINGULAR : 0;
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


// ---------------------------------------------------------------------------------------------
// Mixed local energy E_L = sum_i omega_i E_L^(i) with rank-E closed forms (H10):
// per operator X in {L_g, h}:  TT = C_act^T X Theta_0 (nact x N),  T0 = its top N rows,
//   W = TT_virt - Q_virt T0,  WT = W T0,  f0 = Tr T0,  X0 = Tr(T0 T0);  per determinant and spin
//   t = f0 + Tr(Z W[P,H]),  xch = X0 + 2 Tr(Z WT[P,H]) + Tr((Z W[P,H])^2);
//   E^(i) = sum_s t^s(h) + 1/2 sum_g [(t^a + t^b)^2 - xch^a - xch^b].
// ---------------------------------------------------------------------------------------------
template <typename T> struct MdEnergyArgs {
  MdConst m;
  int ng, ldr;
  const cplx<T>* theta0;   // [nw][M][nt]
  const cplx<T>* TTg;      // [nw][ng+1][nact][nt] : TT = C_act^T X Theta_0 for X = L_0..L_{ng-1}, h  (batched GEMM,
                           //                        run before this kernel; H10)
  zcplx* eloc;             // [nw]
};

inline size_t md_energy_smem(int M, int na, int nb, int nact, int ndet, int ts, int emax = 2) {
  size_t b = md_smem_bytes(na, nb, nact, ndet, emax);
  b += ((size_t)M * (na + nb) * 2 * ts + 15) & ~size_t(15);
  const size_t nw_ = (size_t)(nact - na) * na + (size_t)(nact - nb) * nb;
  // TT, W, WT, Q_virt copy, Z copy, 4 scalars: complex T (the bulk arithmetic follows the walker precision;
  // per-determinant energies and the final mixture are accumulated in FP64)
  b += ((size_t)2 * nact * (na + nb) + 3 * nw_ + 4) * 2 * ts + 16;   // TT is double buffered; Z is read from md_prepare's FP64 copy
  return b;
}

enum { MD_THREADS = 128 };  // determinants per thread DPT in {1, 2, 4, 8} (ndet <= 8 * 128)

template <typename T, int MD_DPT>
__global__ void __launch_bounds__(MD_THREADS) k_md_energy(MdEnergyArgs<T> g) {
  typedef cplx<T> C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const MdConst& m = g.m;
  const int w = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x, nt = m.na + m.nb, M = m.M, nact = m.nact;
  const int lane = tid & 31, wid = tid >> 5;
  MdSmem s;
  unsigned char* p = md_carve(smem_raw, m, s);
  C* th0 = reinterpret_cast<C*>(p);
  p += ((size_t)M * nt * sizeof(C) + 15) & ~size_t(15);
  const int nwa = (nact - m.na) * m.na, nwb = (nact - m.nb) * m.nb;
  C* TT0 = reinterpret_cast<C*>(p);
  C* Wm[2]; C* WTm[2]; C* Qc[2];
  Wm[0] = TT0 + 2 * nact * nt; Wm[1] = Wm[0] + nwa;
  WTm[0] = Wm[1] + nwb; WTm[1] = WTm[0] + nwa;
  Qc[0] = WTm[1] + nwb; Qc[1] = Qc[0] + nwa;
  C* scal = Qc[1] + nwb;               // f0[2], X0[2]   (Z_i is read from s.Z, FP64: a second copy in T would not fit 1000 determinants)
  for (int e = tid; e < M * nt; e += nthr) th0[e] = g.theta0[(size_t)w * M * nt + e];
  __syncthreads();
  md_prepare<T>(m, th0, s);
  for (int e = tid; e < nwa + nwb; e += nthr) Qc[0][e] = mk<T>((T)s.Qv[0][e].x, (T)s.Qv[0][e].y);

  zcplx Eacc[MD_DPT];
#pragma unroll
  for (int j = 0; j < MD_DPT; ++j) Eacc[j] = mk<double>(0.0, 0.0);
  // excitation pattern of this thread's determinants (constant over the gamma loop): packed 4 x 8 bits per spin
  uint32_t pat[MD_DPT][2]; int rks[MD_DPT];
#pragma unroll
  for (int j = 0; j < MD_DPT; ++j) {
    const int i = tid + j * MD_THREADS;
    rks[j] = 0; pat[j][0] = pat[j][1] = 0;
    if (i < m.ndet)
      for (int sp = 0; sp < 2; ++sp) {
        int h[4], pp[4];
        const int rk = md_exc(m, i, sp, h, pp);
        const int n = sp ? m.nb : m.na;
        rks[j] |= rk << (4 * sp);
        pat[j][sp] = (uint32_t)(h[0] & 255) | ((uint32_t)((pp[0] - n) & 255) << 8) | ((uint32_t)(h[1] & 255) << 16) |
                     ((uint32_t)((pp[1] - n) & 255) << 24);
      }
  }
  __syncthreads();

  // 1. TT[q][a] = (C_act^T X Theta_0)[q][a], precomputed for all X by one GEMM over all walkers; the tile of the
  //    next X is fetched into registers while this one is processed (double buffer in shared memory)
  enum { TTPF = 8 };   // nact * nt <= TTPF * MD_THREADS (checked on the host)
  const C* srcw = g.TTg + (size_t)w * (g.ng + 1) * nact * nt;
  for (int e = tid; e < nact * nt; e += nthr) TT0[e] = srcw[e];
  __syncthreads();
  for (int gi = 0; gi <= g.ng; ++gi) {
    const bool is_h = gi == g.ng;
    C* TT = TT0 + (gi & 1) * nact * nt;
    C pre[TTPF];
    if (gi < g.ng) {
      const C* src = srcw + (size_t)(gi + 1) * nact * nt;
#pragma unroll
      for (int u = 0; u < TTPF; ++u) {
        const int e = tid + u * MD_THREADS;
        if (e < nact * nt) pre[u] = src[e];
      }
    }
    // 2. W = TT_virt - Q_virt T0 ; f0, X0 by warps 0 / 1
    for (int sp = 0; sp < 2; ++sp) {
      const int n = sp ? m.nb : m.na, nv = nact - n, off = sp ? m.na : 0;
      for (int e = tid; e < nv * n; e += nthr) {
        int pv = e / n, a = e - pv * n;
        C acc = TT[(n + pv) * nt + off + a];
        for (int h = 0; h < n; ++h) acc = csub(acc, cmul(Qc[sp][pv * n + h], TT[h * nt + off + a]));
        Wm[sp][e] = acc;
      }
    }
    if (wid < 2) {
      const int sp = wid, n = sp ? m.nb : m.na, off = sp ? m.na : 0;
      C f0 = mk<T>(T(0), T(0)), x0 = mk<T>(T(0), T(0));
      for (int e = lane; e < n * n; e += 32) {
        int a = e / n, b = e - a * n;
        if (a == b) f0 = cadd(f0, TT[a * nt + off + a]);
        x0 = cadd(x0, cmul(TT[a * nt + off + b], TT[b * nt + off + a]));
      }
      f0.x = warp_sum(f0.x); f0.y = warp_sum(f0.y); x0.x = warp_sum(x0.x); x0.y = warp_sum(x0.y);
      if (lane == 0) { scal[sp] = f0; scal[2 + sp] = x0; }
    }
    __syncthreads();
    // 3. WT = W T0
    if (!is_h) {
      for (int sp = 0; sp < 2; ++sp) {
        const int n = sp ? m.nb : m.na, nv = nact - n, off = sp ? m.na : 0;
        for (int e = tid; e < nv * n; e += nthr) {
          int pv = e / n, a = e - pv * n;
          C acc = mk<T>(T(0), T(0));
          for (int b = 0; b < n; ++b) cfma(acc, Wm[sp][pv * n + b], TT[b * nt + off + a]);
          WTm[sp][e] = acc;
        }
      }
      __syncthreads();
    }
    // 4. per determinant: E x E work only
#pragma unroll
    for (int j = 0; j < MD_DPT; ++j) {
      const int i = tid + j * MD_THREADS;
      if (i >= m.ndet) continue;
      C tsum = mk<T>(T(0), T(0)), xsum = mk<T>(T(0), T(0));
#pragma unroll
      for (int sp = 0; sp < 2; ++sp) {
        const int n = sp ? m.nb : m.na;
        const int rk = (rks[j] >> (4 * sp)) & 15;
        const uint32_t pt = pat[j][sp];
        const int h0 = pt & 255, p0 = (pt >> 8) & 255, h1 = (pt >> 16) & 255, p1 = (pt >> 24) & 255;
        const zcplx* Zd = s.Z + ((size_t)i * 2 + sp) * m.emax * m.emax;
        C Zi[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) Zi[u] = mk<T>((T)Zd[u].x, (T)Zd[u].y);
        C t = scal[sp], xch = scal[2 + sp];
        if (rk >= 3) {
          // general rank (3, 4): A = Z W[P,H] (rk x rk), t += Tr A, xch += 2 Tr(Z WT[P,H]) + Tr(A A)
          int hh[4], pq[4];
          md_exc(m, i, sp, hh, pq);
          C A[16];
          for (int f = 0; f < rk; ++f)
            for (int f2 = 0; f2 < rk; ++f2) {
              C acc = mk<T>(T(0), T(0));
              for (int e = 0; e < rk; ++e) {
                const zcplx zd = Zd[f * 4 + e];
                cfma(acc, mk<T>((T)zd.x, (T)zd.y), Wm[sp][(pq[e] - n) * n + hh[f2]]);
              }
              A[f * 4 + f2] = acc;
            }
          for (int f = 0; f < rk; ++f) t = cadd(t, A[f * 4 + f]);
          if (!is_h) {
            C tr2 = mk<T>(T(0), T(0));
            for (int f = 0; f < rk; ++f)
              for (int e = 0; e < rk; ++e) {
                const zcplx zd = Zd[f * 4 + e];
                cfma(tr2, mk<T>((T)zd.x, (T)zd.y), WTm[sp][(pq[e] - n) * n + hh[f]]);
              }
            xch = cadd(xch, mk<T>(2 * tr2.x, 2 * tr2.y));
            for (int f = 0; f < rk; ++f)
              for (int f2 = 0; f2 < rk; ++f2) cfma(xch, A[f * 4 + f2], A[f2 * 4 + f]);
          }
        } else if (rk == 1) {
          C zw = cmul(Zi[0], Wm[sp][p0 * n + h0]);
          t = cadd(t, zw);
          if (!is_h) {
            C zt = cmul(Zi[0], WTm[sp][p0 * n + h0]);
            xch = cadd(xch, mk<T>(2 * zt.x, 2 * zt.y));
            cfma(xch, zw, zw);
          }
        } else if (rk == 2) {
          // (Z W)[f][f'] = sum_e Z[f][e] W[p_e][h_f']
          const C w00 = Wm[sp][p0 * n + h0], w01 = Wm[sp][p0 * n + h1], w10 = Wm[sp][p1 * n + h0], w11 = Wm[sp][p1 * n + h1];
          const C z00 = Zi[0], z01 = Zi[1], z10 = Zi[2], z11 = Zi[3];
          C a00 = cmul(z00, w00); cfma(a00, z01, w10);
          C a01 = cmul(z00, w01); cfma(a01, z01, w11);
          C a10 = cmul(z10, w00); cfma(a10, z11, w10);
          C a11 = cmul(z10, w01); cfma(a11, z11, w11);
          t = cadd(t, cadd(a00, a11));
          if (!is_h) {
            const C v00 = WTm[sp][p0 * n + h0], v10 = WTm[sp][p1 * n + h0], v01 = WTm[sp][p0 * n + h1], v11 = WTm[sp][p1 * n + h1];
            C b00 = cmul(z00, v00); cfma(b00, z01, v10);
            C b11 = cmul(z10, v01); cfma(b11, z11, v11);
            xch = cadd(xch, mk<T>(2 * (b00.x + b11.x), 2 * (b00.y + b11.y)));
            cfma(xch, a00, a00); cfma(xch, a11, a11);
            C cr = cmul(a01, a10);
            xch = cadd(xch, mk<T>(2 * cr.x, 2 * cr.y));
          }
        }
        tsum = cadd(tsum, t);
        xsum = cadd(xsum, xch);
      }
      if (is_h) {
        Eacc[j].x += (double)tsum.x; Eacc[j].y += (double)tsum.y;
      } else {
        C e2 = csub(cmul(tsum, tsum), xsum);
        Eacc[j].x += 0.5 * (double)e2.x; Eacc[j].y += 0.5 * (double)e2.y;
      }
    }
    if (gi < g.ng) {
      C* TTn = TT0 + ((gi + 1) & 1) * nact * nt;
#pragma unroll
      for (int u = 0; u < TTPF; ++u) {
        const int e = tid + u * MD_THREADS;
        if (e < nact * nt) TTn[e] = pre[u];
      }
    }
    __syncthreads();
  }
  zcplx part = mk<double>(0.0, 0.0);
#pragma unroll
  for (int j = 0; j < MD_DPT; ++j) {
    const int i = tid + j * MD_THREADS;
    if (i < m.ndet) part = zadd(part, zmul(s.omega[i], Eacc[j]));
  }
  zcplx tot = block_sum(part, s.red);
  if (tid == 0) g.eloc[w] = tot;
}


// ---------------------------------------------------------------------------------------------
// Batched-gamma version of k_md_energy (same arithmetic).  The kernel above walks the operators one at a time with three
// CTA barriers each and a fraction of its threads busy; here MDB_G operators are processed per pass:
//   A. one thread per (operator, spin, virtual row pv): the W row (n x n complex MACs against Q_virt), then the WT row
//      (n x n more), rows in registers, T0 read from the TT tiles that cp.async double-buffers in shared memory;
//   A2. f0 = Tr T0 and X0 = Tr(T0 T0) reduced from per-row partials;
//   B. one thread per determinant, looping over the operators of the batch with its Z and excitation pattern in registers.
// Three barriers per MDB_G operators.  Needs n_sigma <= NMAX and 16-byte multiples for the tiles (host checks).
// ---------------------------------------------------------------------------------------------
enum { MDB_G = 6, MDB_PAD = 2 };   // tiles MDB_PAD complex apart in shared memory: operators of a batch hit different banks

inline size_t md_energy_b_smem(int M, int na, int nb, int nact, int ndet, int ts) {
  size_t b = md_smem_bytes(na, nb, nact, ndet);
  b += ((size_t)M * (na + nb) * 2 * ts + 15) & ~size_t(15);
  const size_t nva = nact - na, nvb = nact - nb, nw_ = nva * na + nvb * nb, nvm = nva > nvb ? nva : nvb;
  const size_t celems = (size_t)2 * MDB_G * (nact * (na + nb) + MDB_PAD) + (size_t)2 * MDB_G * nw_ + nw_ + (size_t)ndet * 8 +
                        (size_t)MDB_G * 4 + (size_t)MDB_G * 2 * (nvm ? nvm : 1) * 2;
  return b + celems * 2 * ts + 32;
}

template <typename T, int NMAX, int MD_DPT>
__global__ void __launch_bounds__(MD_THREADS) k_md_energy_b(MdEnergyArgs<T> g) {
  typedef cplx<T> C;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const MdConst& m = g.m;
  const int w = blockIdx.x, tid = threadIdx.x, nthr = blockDim.x, nt = m.na + m.nb, M = m.M, nact = m.nact;
  MdSmem s;
  unsigned char* p = md_carve(smem_raw, m, s);
  C* th0 = reinterpret_cast<C*>(p);
  p += ((size_t)M * nt * sizeof(C) + 15) & ~size_t(15);
  const int nva = nact - m.na, nvb = nact - m.nb, nvt = nva + nvb, nvm = nva > nvb ? nva : nvb;
  const int nwa = nva * m.na, nwb = nvb * m.nb, nwt = nwa + nwb, tile = nact * nt;
  const int tstr = tile + MDB_PAD;             // padded tile stride
  C* TTb = reinterpret_cast<C*>(p);            // [2][MDB_G][tstr]   (16-byte aligned: cp.async destination)
  C* Wb = TTb + 2 * MDB_G * tstr;              // [MDB_G][nwa + nwb]
  C* WTb = Wb + MDB_G * nwt;
  C* Qc[2]; Qc[0] = WTb + MDB_G * nwt; Qc[1] = Qc[0] + nwa;
  C* Zc = Qc[1] + nwb;                         // [ndet][2][4]
  C* scal = Zc + (size_t)m.ndet * 8;           // [MDB_G][f0 a, f0 b, X0 a, X0 b]
  C* part = scal + MDB_G * 4;                  // [MDB_G][2][nvm][f0, X0]
  const int nop = g.ng + 1, nbatch = (nop + MDB_G - 1) / MDB_G;
  const C* srcw = g.TTg + (size_t)w * nop * tile;
  auto fetch = [&](int bi) {
    const int g0 = bi * MDB_G, gc = min(MDB_G, nop - g0);
    const int t16 = (int)((size_t)tile * sizeof(C) / 16);
    const unsigned char* src = reinterpret_cast<const unsigned char*>(srcw + (size_t)g0 * tile);
    unsigned char* dst = reinterpret_cast<unsigned char*>(TTb + (size_t)(bi & 1) * MDB_G * tstr);
    for (int e = tid; e < gc * t16; e += nthr) {
      const int gl = e / t16, r = e - gl * t16;
      cp_async16(dst + ((size_t)gl * tstr * sizeof(C) + (size_t)r * 16), src + (size_t)e * 16);
    }
    cp_async_commit();
  };
  fetch(0);

  for (int e = tid; e < M * nt; e += nthr) th0[e] = g.theta0[(size_t)w * M * nt + e];
  __syncthreads();
  md_prepare<T>(m, th0, s);
  for (int e = tid; e < nwt; e += nthr) Qc[0][e] = mk<T>((T)s.Qv[0][e].x, (T)s.Qv[0][e].y);
  for (int e = tid; e < m.ndet * 8; e += nthr) Zc[e] = mk<T>((T)s.Z[e].x, (T)s.Z[e].y);

  zcplx Eacc[MD_DPT];
  uint32_t pat[MD_DPT][2]; int rks[MD_DPT];
#pragma unroll
  for (int j = 0; j < MD_DPT; ++j) {
    Eacc[j] = mk<double>(0.0, 0.0);
    const int i = tid + j * MD_THREADS;
    rks[j] = 0; pat[j][0] = pat[j][1] = 0;
    if (i < m.ndet)
      for (int sp = 0; sp < 2; ++sp) {
        int h[4], pp[4];
        const int rk = md_exc(m, i, sp, h, pp);
        const int n = sp ? m.nb : m.na;
        rks[j] |= rk << (2 * sp);
        pat[j][sp] = (uint32_t)(h[0] & 255) | ((uint32_t)((pp[0] - n) & 255) << 8) | ((uint32_t)(h[1] & 255) << 16) |
                     ((uint32_t)((pp[1] - n) & 255) << 24);
      }
  }

  for (int bi = 0; bi < nbatch; ++bi) {
    const int g0 = bi * MDB_G, gc = min(MDB_G, nop - g0);
    if (bi + 1 < nbatch) { fetch(bi + 1); cp_async_wait<1>(); } else { cp_async_wait<0>(); }
    __syncthreads();   // this batch's tiles have landed; the previous pass no longer reads W / WT / scal
    const C* TT = TTb + (size_t)(bi & 1) * MDB_G * tstr;
    // ---- A: W = TT_virt - Q_virt T0 and WT = W T0, one row per thread
    for (int it = tid; it < gc * nvt; it += nthr) {
      const int gl = it / nvt, r = it - gl * nvt, sp = r >= nva, pv = sp ? r - nva : r;
      const int n = sp ? m.nb : m.na, nv = sp ? nvb : nva, off = sp ? m.na : 0;
      const C* T0 = TT + (size_t)gl * tstr + off;          // T0[h * nt + a]
      const int wo = gl * nwt + (sp ? nwa : 0) + pv * n;
      C wr[NMAX];
#pragma unroll
      for (int a = 0; a < NMAX; ++a) wr[a] = a < n ? T0[(n + pv) * nt + a] : mk<T>(T(0), T(0));
      for (int h = 0; h < n; ++h) {
        const C q = Qc[sp][pv * n + h];
#pragma unroll
        for (int a = 0; a < NMAX; ++a)
          if (a < n) wr[a] = csub(wr[a], cmul(q, T0[h * nt + a]));
      }
#pragma unroll
      for (int a = 0; a < NMAX; ++a)
        if (a < n) Wb[wo + a] = wr[a];
      C wt[NMAX];
#pragma unroll
      for (int a = 0; a < NMAX; ++a) wt[a] = mk<T>(T(0), T(0));
      for (int b = 0; b < n; ++b) {
        const C wb = Wb[wo + b];
#pragma unroll
        for (int a = 0; a < NMAX; ++a)
          if (a < n) cfma(wt[a], wb, T0[b * nt + a]);
      }
#pragma unroll
      for (int a = 0; a < NMAX; ++a)
        if (a < n) WTb[wo + a] = wt[a];
      C f0 = mk<T>(T(0), T(0)), x0 = mk<T>(T(0), T(0));
      for (int a = pv; a < n; a += nv) {
        f0 = cadd(f0, T0[a * nt + a]);
        for (int b = 0; b < n; ++b) cfma(x0, T0[a * nt + b], T0[b * nt + a]);
      }
      part[((gl * 2 + sp) * nvm + pv) * 2 + 0] = f0;
      part[((gl * 2 + sp) * nvm + pv) * 2 + 1] = x0;
    }
    __syncthreads();
    // ---- A2: f0, X0 per (operator, spin)
    for (int it = tid; it < gc * 2; it += nthr) {
      const int gl = it >> 1, sp = it & 1, n = sp ? m.nb : m.na, nv = sp ? nvb : nva, off = sp ? m.na : 0;
      C f0 = mk<T>(T(0), T(0)), x0 = mk<T>(T(0), T(0));
      if (nv > 0) {
        for (int pv = 0; pv < nv; ++pv) {
          f0 = cadd(f0, part[((gl * 2 + sp) * nvm + pv) * 2 + 0]);
          x0 = cadd(x0, part[((gl * 2 + sp) * nvm + pv) * 2 + 1]);
        }
      } else {   // no virtual orbital for this spin: nobody computed the partials
        const C* T0 = TT + (size_t)gl * tstr + off;
        for (int a = 0; a < n; ++a) {
          f0 = cadd(f0, T0[a * nt + a]);
          for (int b = 0; b < n; ++b) cfma(x0, T0[a * nt + b], T0[b * nt + a]);
        }
      }
      scal[gl * 4 + sp] = f0; scal[gl * 4 + 2 + sp] = x0;
    }
    __syncthreads();
    // ---- B: per determinant, E x E work per operator
#pragma unroll
    for (int j = 0; j < MD_DPT; ++j) {
      const int i = tid + j * MD_THREADS;
      if (i >= m.ndet) continue;
      C zz[2][4];
#pragma unroll
      for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int u = 0; u < 4; ++u) zz[sp][u] = Zc[((size_t)i * 2 + sp) * 4 + u];
      for (int gl = 0; gl < gc; ++gl) {
        const bool is_h = g0 + gl == g.ng;
        C tsum = mk<T>(T(0), T(0)), xsum = mk<T>(T(0), T(0));
#pragma unroll
        for (int sp = 0; sp < 2; ++sp) {
          const int n = sp ? m.nb : m.na;
          const int rk = (rks[j] >> (2 * sp)) & 3;
          const uint32_t pt = pat[j][sp];
          const int h0 = pt & 255, p0 = (pt >> 8) & 255, h1 = (pt >> 16) & 255, p1 = (pt >> 24) & 255;
          const C* Wm = Wb + gl * nwt + (sp ? nwa : 0);
          const C* WTm = WTb + gl * nwt + (sp ? nwa : 0);
          C t = scal[gl * 4 + sp], xch = scal[gl * 4 + 2 + sp];
          if (rk == 1) {
            C zw = cmul(zz[sp][0], Wm[p0 * n + h0]);
            t = cadd(t, zw);
            if (!is_h) {
              C zt = cmul(zz[sp][0], WTm[p0 * n + h0]);
              xch = cadd(xch, mk<T>(2 * zt.x, 2 * zt.y));
              cfma(xch, zw, zw);
            }
          } else if (rk == 2) {
            const C w00 = Wm[p0 * n + h0], w01 = Wm[p0 * n + h1], w10 = Wm[p1 * n + h0], w11 = Wm[p1 * n + h1];
            const C z00 = zz[sp][0], z01 = zz[sp][1], z10 = zz[sp][2], z11 = zz[sp][3];
            C a00 = cmul(z00, w00); cfma(a00, z01, w10);
            C a01 = cmul(z00, w01); cfma(a01, z01, w11);
            C a10 = cmul(z10, w00); cfma(a10, z11, w10);
            C a11 = cmul(z10, w01); cfma(a11, z11, w11);
            t = cadd(t, cadd(a00, a11));
            if (!is_h) {
              const C v00 = WTm[p0 * n + h0], v10 = WTm[p1 * n + h0], v01 = WTm[p0 * n + h1], v11 = WTm[p1 * n + h1];
              C b00 = cmul(z00, v00); cfma(b00, z01, v10);
              C b11 = cmul(z10, v01); cfma(b11, z11, v11);
              xch = cadd(xch, mk<T>(2 * (b00.x + b11.x), 2 * (b00.y + b11.y)));
              cfma(xch, a00, a00); cfma(xch, a11, a11);
              C cr = cmul(a01, a10);
              xch = cadd(xch, mk<T>(2 * cr.x, 2 * cr.y));
            }
          }
          tsum = cadd(tsum, t);
          xsum = cadd(xsum, xch);
        }
        if (is_h) {
          Eacc[j].x += (double)tsum.x; Eacc[j].y += (double)tsum.y;
        } else {
          C e2 = csub(cmul(tsum, tsum), xsum);
          Eacc[j].x += 0.5 * (double)e2.x; Eacc[j].y += 0.5 * (double)e2.y;
        }
      }
    }
  }
  zcplx partE = mk<double>(0.0, 0.0);
#pragma unroll
  for (int j = 0; j < MD_DPT; ++j) {
    const int i = tid + j * MD_THREADS;
    if (i < m.ndet) partE = zadd(partE, zmul(s.omega[i], Eacc[j]));
  }
  zcplx tot = block_sum(partE, s.red);
  if (tid == 0) g.eloc[w] = tot;
}

}  // namespace afq
