// popctl.cuh -- the two steps either side of the walker step:
//   k_ortho        walker orthonormalisation, PAPER.md:97 ("orthonormalized after every two propagation steps")
//   k_comb_parents / k_comb_pack / k_comb_unpack   "simple combing" population control
// Both are HBM-bound by design (read + write the walker once); the arithmetic is FP64 on both precision paths.
#pragma once
#include "common.cuh"

namespace afq {

// ------------------------------------------------------------------------------------------------
// Thin QR of each spin block by modified Gram-Schmidt, R with a real positive diagonal (reading R21):
// Phi_s = Q_s R_s, walker <- Q, S <- S / (det R_a det R_b) because |Phi> = det R_a det R_b |Q>.
// One CTA per walker, one warp per trailing column (ortho_threads).  The walker is held in shared memory in FP64, one column after the
// other with an odd leading dimension (conflict-free both for the transposing load/store and for the column
// sweeps).  Right-looking elimination without an intermediate scaling: at step j every warp that owns a
// trailing column k computes d = <v_j, v_k> in one sweep and applies v_k -= (d/|v_j|^2) v_j in a second one; v_j itself is only read, so one CTA barrier per step is enough.  Columns are scaled by 1/|v_j|
// when the walker is written back.  Theta = Phi A^-1 is invariant, so nothing else of the state changes.
// ------------------------------------------------------------------------------------------------
__host__ __device__ inline int ortho_ld(int M) { return M | 1; }
inline int ortho_threads(int na, int nb) {
  int w = na + nb - 2;   // trailing columns of both spins at the first elimination step
  w = w < 8 ? 8 : (w > 16 ? 16 : w);     // <= 512 threads: two CTAs per SM by registers and (cfg 5) shared memory
  return 32 * w;
}
inline size_t ortho_smem_bytes(int M, int nt) { return (size_t)nt * ortho_ld(M) * sizeof(zcplx) + 136 * sizeof(double); }

template <typename T>
__global__ void __launch_bounds__(512, 2) k_ortho(int M, int na, int nb, cplx<T>* __restrict__ phi, zcplx* __restrict__ ovlp,
                                               int32_t* __restrict__ flags) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  zcplx* V = (zcplx*)smem_raw;
  const int nt = na + nb, ld = ortho_ld(M);
  double* nrm = (double*)(V + (size_t)nt * ld);   // [nt] squared norms of the orthogonalised columns
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nth = blockDim.x, nwp = nth >> 5;
  cplx<T>* g = phi + (size_t)blockIdx.x * M * nt;
  for (int e = tid; e < M * nt; e += nth) {
    const int i = e / nt, k = e - i * nt;
    V[k * ld + i] = to_z(g[e]);
  }
  __syncthreads();
  // nrm[k] = |v_k|^2 of the fully orthogonalised column k.  Column 0 of each spin is final from the start; column
  // j + 1 becomes final in elimination step j, and the warp that updates it accumulates its norm in the same sweep.
  if (warp < 2) {
    const int n = warp ? nb : na, c0 = warp ? na : 0;
    if (n > 0) {
      const zcplx* v0 = V + (size_t)c0 * ld;
      double nn = 0.0;
      for (int i = lane; i < M; i += 32) { const zcplx a = v0[i]; nn = fma(a.x, a.x, nn); nn = fma(a.y, a.y, nn); }
      nn = warp_sum(nn);
      if (lane == 0) nrm[c0] = nn;
    }
  }
  __syncthreads();
  const int nmax = na > nb ? na : nb;
  for (int j = 0; j + 1 < nmax; ++j) {
    // trailing columns of both spins at this step, dealt round-robin to the warps (up to 16 per CTA)
    const int ta = na - 1 - j > 0 ? na - 1 - j : 0, tb = nb - 1 - j > 0 ? nb - 1 - j : 0;
    for (int t = warp; t < ta + tb; t += nwp) {
      const int s_off = t < ta ? 0 : na;
      const int k = t < ta ? j + 1 + t : j + 1 + (t - ta);
      const zcplx* vj = V + (size_t)(s_off + j) * ld;
      zcplx* vk = V + (size_t)(s_off + k) * ld;
      const double nn = nrm[s_off + j];
      // two rows per iteration on separate accumulators: the sweep is a chain of dependent DFMAs otherwise
      double dr = 0.0, di = 0.0, dr2 = 0.0, di2 = 0.0;
      int i = lane;
      for (; i + 32 < M; i += 64) {
        const zcplx a = vj[i], b = vk[i], a2 = vj[i + 32], b2 = vk[i + 32];
        dr = fma(a.x, b.x, dr); dr = fma(a.y, b.y, dr);      // conj(a) * b
        di = fma(a.x, b.y, di); di = fma(-a.y, b.x, di);
        dr2 = fma(a2.x, b2.x, dr2); dr2 = fma(a2.y, b2.y, dr2);
        di2 = fma(a2.x, b2.y, di2); di2 = fma(-a2.y, b2.x, di2);
      }
      if (i < M) {
        const zcplx a = vj[i], b = vk[i];
        dr = fma(a.x, b.x, dr); dr = fma(a.y, b.y, dr);
        di = fma(a.x, b.y, di); di = fma(-a.y, b.x, di);
      }
      dr = warp_sum(dr + dr2); di = warp_sum(di + di2);
      double nk = 0.0;
      if (nn > 0.0) {
        const double inv = 1.0 / nn, cr = dr * inv, ci = di * inv;
        for (int r = lane; r < M; r += 32) {
          const zcplx a = vj[r];
          zcplx b = vk[r];
          b.x = fma(-cr, a.x, b.x); b.x = fma(ci, a.y, b.x);
          b.y = fma(-cr, a.y, b.y); b.y = fma(-ci, a.x, b.y);
          vk[r] = b;
          if (k == j + 1) { nk = fma(b.x, b.x, nk); nk = fma(b.y, b.y, nk); }
        }
      } else if (k == j + 1) {
        for (int r = lane; r < M; r += 32) { const zcplx b = vk[r]; nk = fma(b.x, b.x, nk); nk = fma(b.y, b.y, nk); }
      }
      if (k == j + 1) {
        nk = warp_sum(nk);
        if (lane == 0) nrm[s_off + k] = nk;
      }
    }
    __syncthreads();
  }
  if (tid < nt) nrm[72 + tid] = 1.0 / sqrt(nrm[tid]);
  __syncthreads();
  if (tid < 32) {
    // det R_a det R_b = prod |v_k| (real, positive); a vanishing or non-finite column flags the walker
    double r = (tid < nt) ? sqrt(nrm[tid]) : 1.0;
    int bad = (tid < nt) && !(r > 0.0 && isfinite(r));
    bad = __any_sync(0xffffffffu, bad);
    double prod = r;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) prod *= __shfl_xor_sync(0xffffffffu, prod, o);
    if (nt > 32) {   // n_alpha, n_beta <= 32 each: a second round covers columns 32..63
      double r2 = (tid + 32 < nt) ? sqrt(nrm[tid + 32]) : 1.0;
      int bad2 = (tid + 32 < nt) && !(r2 > 0.0 && isfinite(r2));
      bad |= __any_sync(0xffffffffu, bad2);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) r2 *= __shfl_xor_sync(0xffffffffu, r2, o);
      prod *= r2;
    }
    if (tid == 0) {
      if (!bad) {
        zcplx s = ovlp[blockIdx.x];
        ovlp[blockIdx.x] = mk<double>(s.x / prod, s.y / prod);
      } else if (flags) {
        flags[blockIdx.x] |= isfinite(prod) ? FLAG_SINGULAR : FLAG_NONFINITE;
      }
      nrm[64] = bad ? 1.0 : 0.0;
    }
  }
  __syncthreads();
  if (nrm[64] != 0.0) return;   // degenerate walker: left as it was (flagged)
  for (int e = tid; e < M * nt; e += nth) {
    const int i = e / nt, k = e - i * nt;
    const double inv = nrm[72 + k];
    const zcplx v = V[k * ld + i];
    g[e] = mk<T>((T)(v.x * inv), (T)(v.y * inv));
  }
}

// ------------------------------------------------------------------------------------------------
// Comb (reading R22): teeth t_i = (i + u) W / N_w; parent(i) = first p with c_p > t_i, c = running sum of w in
// index order.  The running sum decides integers, so it is accumulated SEQUENTIALLY in FP64 in the same order as
// the definition (one thread, chunks staged through shared memory by the whole CTA): bit-identical parents.
// One CTA.  cum [N_w] scratch; wnew[0] = W / N_w, wnew[1] = W.  W == 0 or non-finite: identity map, wnew[0] = -1
// (the unpack kernel then keeps the weights).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_comb_parents(int nw, const double* __restrict__ w, double u, double* __restrict__ cum,
                                                        int32_t* __restrict__ parent, double* __restrict__ wnew) {
  __shared__ double buf[1024];
  __shared__ double carry;
  const int tid = threadIdx.x;
  if (tid == 0) carry = 0.0;
  for (int base = 0; base < nw; base += 1024) {
    const int n = min(1024, nw - base);
    if (tid < n) buf[tid] = w[base + tid];
    __syncthreads();
    if (tid == 0) {
      double c = carry;
      for (int i = 0; i < n; ++i) { c = __dadd_rn(c, buf[i]); buf[i] = c; }
      carry = c;
    }
    __syncthreads();
    if (tid < n) cum[base + tid] = buf[tid];
    __syncthreads();
  }
  const double W = carry;
  const bool ok = W > 0.0 && isfinite(W);
  if (tid == 0) { wnew[0] = ok ? __ddiv_rn(W, (double)nw) : -1.0; wnew[1] = W; }
  const double step = __ddiv_rn(W, (double)nw);
  for (int i = tid; i < nw; i += 1024) {
    int p = i;
    if (ok) {
      const double t = __dmul_rn(__dadd_rn((double)i, u), step);
      int lo = 0, hi = nw;                 // first index with cum > t
      while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if (cum[mid] > t) hi = mid; else lo = mid + 1;
      }
      p = lo < nw - 1 ? lo : nw - 1;
    }
    parent[i] = p;
  }
}

// Walkers whose parent is another slot are first copied (phi, theta, fb, S of the PARENT) into a scratch slot of
// their own, then (second kernel) from there into place: out of place, so any map is allowed; slots that keep their
// walker move no bytes.  Sizes in 8-byte words (a complex64 or one double).
struct CombMove {
  uint2 *phi, *theta, *fb, *s_phi, *s_theta, *s_fb;
  zcplx *ovlp, *s_ovlp;
  int words_phi, words_fb;   // per walker
};

__global__ void __launch_bounds__(256) k_comb_pack(CombMove m, const int32_t* __restrict__ parent) {
  const int i = blockIdx.x, p = parent[i];
  if (p == i) return;
  const size_t op = (size_t)p * m.words_phi, oi = (size_t)i * m.words_phi;
  for (int e = threadIdx.x; e < m.words_phi; e += 256) {
    m.s_phi[oi + e] = m.phi[op + e];
    m.s_theta[oi + e] = m.theta[op + e];
  }
  const size_t fp = (size_t)p * m.words_fb, fi = (size_t)i * m.words_fb;
  for (int e = threadIdx.x; e < m.words_fb; e += 256) m.s_fb[fi + e] = m.fb[fp + e];
  if (threadIdx.x == 0) m.s_ovlp[i] = m.ovlp[p];
}

__global__ void __launch_bounds__(256) k_comb_unpack(CombMove m, const int32_t* __restrict__ parent, double* __restrict__ weight,
                                                      const double* __restrict__ wnew) {
  const int i = blockIdx.x;
  if (threadIdx.x == 0 && wnew[0] >= 0.0) weight[i] = wnew[0];
  if (parent[i] == i) return;
  const size_t oi = (size_t)i * m.words_phi;
  for (int e = threadIdx.x; e < m.words_phi; e += 256) {
    m.phi[oi + e] = m.s_phi[oi + e];
    m.theta[oi + e] = m.s_theta[oi + e];
  }
  const size_t fi = (size_t)i * m.words_fb;
  for (int e = threadIdx.x; e < m.words_fb; e += 256) m.fb[fi + e] = m.s_fb[fi + e];
  if (threadIdx.x == 0) m.ovlp[i] = m.s_ovlp[i];
}

// ------------------------------------------------------------------------------------------------
// Comb over a population sharded across ranks: every rank runs
// k_comb_parents on the all-gathered weights (same bits everywhere), packs the records of ITS walkers that the map
// hands out (to itself or to peers) in global-slot order -- the map is monotone, so these slots are one contiguous
// range and the all-to-all's receive buffer arrives in slot order -- and unpacks the received records in place.
// Record = [phi | theta | fb | S] in 8-byte words.
// ------------------------------------------------------------------------------------------------
struct CombRecord {
  uint2 *phi, *theta, *fb;
  zcplx* ovlp;
  int words_phi, words_fb, words_rec;   // words_rec = 2 words_phi + words_fb + 2
};

__global__ void __launch_bounds__(256) k_comb_pack_send(CombRecord m, const int32_t* __restrict__ parent_all, long long slot_lo,
                                                         long long first_local, uint2* __restrict__ sendbuf) {
  const long long j = blockIdx.x;
  const long long p = (long long)parent_all[slot_lo + j] - first_local;   // local index of the parent
  uint2* dst = sendbuf + j * m.words_rec;
  const uint2* sp = m.phi + p * m.words_phi;
  const uint2* st = m.theta + p * m.words_phi;
  for (int e = threadIdx.x; e < m.words_phi; e += 256) { dst[e] = sp[e]; dst[m.words_phi + e] = st[e]; }
  const uint2* sf = m.fb + p * m.words_fb;
  for (int e = threadIdx.x; e < m.words_fb; e += 256) dst[2 * m.words_phi + e] = sf[e];
  if (threadIdx.x == 0) {   // 8-byte stores: a record is only 8-byte aligned
    const zcplx sv = m.ovlp[p];
    double* d = reinterpret_cast<double*>(dst + 2 * m.words_phi + m.words_fb);
    d[0] = sv.x; d[1] = sv.y;
  }
}

__global__ void __launch_bounds__(256) k_comb_unpack_recv(CombRecord m, const uint2* __restrict__ recvbuf, double* __restrict__ weight,
                                                           const double* __restrict__ wnew) {
  const long long i = blockIdx.x;
  const uint2* src = recvbuf + i * m.words_rec;
  uint2* dp = m.phi + i * m.words_phi;
  uint2* dt = m.theta + i * m.words_phi;
  for (int e = threadIdx.x; e < m.words_phi; e += 256) { dp[e] = src[e]; dt[e] = src[m.words_phi + e]; }
  uint2* df = m.fb + i * m.words_fb;
  for (int e = threadIdx.x; e < m.words_fb; e += 256) df[e] = src[2 * m.words_phi + e];
  if (threadIdx.x == 0) {
    const double* d = reinterpret_cast<const double*>(src + 2 * m.words_phi + m.words_fb);
    m.ovlp[i] = mk<double>(d[0], d[1]);
    if (wnew[0] >= 0.0) weight[i] = wnew[0];
  }
}

// ------------------------------------------------------------------------------------------------
// Mixed-estimator sums of one measurement ("weighted sum"; the (sum w, sum w E_L) pair that
// is all-reduced across ranks): out = { sum_w w, Re sum_w w E_L, Im sum_w w E_L }, FP64.  One CTA, fixed-shape tree
// (thread t sums walkers t, t + 1024, ... in order; then a shared-memory tree): the result does not depend on timing.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_mixed_sums(int nw, const double* __restrict__ w, const zcplx* __restrict__ eloc,
                                                      double* __restrict__ out) {
  __shared__ double sh[3][1024];
  const int tid = threadIdx.x;
  double a = 0.0, b = 0.0, c = 0.0;
  for (int i = tid; i < nw; i += 1024) {
    const double wi = w[i];
    const zcplx e = eloc[i];
    a += wi;
    if (wi != 0.0) { b = fma(wi, e.x, b); c = fma(wi, e.y, c); }   // a dead walker's E_L may be Inf/NaN: weight 0 drops it
  }
  sh[0][tid] = a; sh[1][tid] = b; sh[2][tid] = c;
  __syncthreads();
  for (int o = 512; o > 0; o >>= 1) {
    if (tid < o) { sh[0][tid] += sh[0][tid + o]; sh[1][tid] += sh[1][tid + o]; sh[2][tid] += sh[2][tid + o]; }
    __syncthreads();
  }
  if (tid < 3) out[tid] = sh[tid][0];
}

// E_mix[m] = (sums[m][1] + i sums[m][2]) / sums[m][0] for n measurements (the sums are afqmc_mixed_sums' output, possibly
// all-reduced across ranks in between); a dead population (sum of weights 0) gives NaN.
__global__ void k_mixed_ratio(int n, const double* __restrict__ sums, zcplx* __restrict__ out) {
  const int m = blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= n) return;
  const double w = sums[3 * m];
  out[m] = w != 0.0 ? mk<double>(sums[3 * m + 1] / w, sums[3 * m + 2] / w) : mk<double>(nan(""), nan(""));
}

}  // namespace afq
