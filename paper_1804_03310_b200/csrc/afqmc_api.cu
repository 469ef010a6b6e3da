// afqmc_api.cu -- C-ABI entry points (include/afqmc.h) of the B200-native ph-AFQMC walker step.
// Host-side orchestration only: every arithmetic step of the path runs in the kernels of this directory.
#include "../../include/afqmc.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <new>
#include <algorithm>
#include <vector>

#include "common.cuh"
#include "gemm_simt.cuh"
#include "gemm_tf32.cuh"
#include "green.cuh"
#include "misc.cuh"
#include "multidet.cuh"
#include "taylor.cuh"
#include "taylor_tc.cuh"
#include "popctl.cuh"
#include "peaks.cuh"

using namespace afq;

namespace {

inline size_t rup(size_t v, size_t a) { return (v + a - 1) / a * a; }

#ifndef AFQMC_EN_CHUNK
#define AFQMC_EN_CHUNK 4
#endif
enum { EN_SCHED_INTS = 16384, EN_CHUNK = AFQMC_EN_CHUNK };   // room for the persistent energy GEMM's tile lists

struct Carver {
  size_t off = 0;
  char* base = nullptr;
  void* take(size_t bytes) {
    void* p = base ? base + off : nullptr;
    off += rup(bytes, 256);
    return p;
  }
};

thread_local char g_init_err[256] = "";

}  // namespace

struct afqmc_ctx {
  afqmc_params p;
  cudaStream_t stream;
  int M, MP, na, nb, nt, ng, NGP, nw, KA, KB, KT, ts;  // ts = sizeof(T)
  int split, path;
  // multi-determinant trial (md != 0): ca/cb = columns per spin of the generalised Theta (n_act), else n_alpha/n_beta
  int md, nact, ndet, ca, cb, emax;   // emax: slots per spin of the normalised excitation list (2, or 4 when max_exc > 2)
  void* Cact; double* coeff; int32_t* exc;
  double *psid_ac, *psid_bc;   // FP64 trial orbitals (constants)
  void *thtil, *th_scr; zcplx *ovlp0, *ovlp_scr;
  void *RactT, *RactT_lo, *thT, *thT_lo, *TTg; int MPK; tc::Maps map_tt;
  size_t mdo_smem, mde_smem; int mde_attr_done;
  int tay_cw, tay_nch, tay_threads;
  size_t tay_smem, green_smem;
  // constants
  void *psi_a, *psi_b, *Eh, *Lt, *Lt_lo, *Rall, *Rall_lo, *Y[2], *Y_lo[2], *hrot;
  // per-step work
  void *Z, *Z_lo, *Abuf, *thp, *thp_lo, *fs;
  zcplx *cshift, *eloc_scratch;
  // device staging for afqmc_step_host
  void *h_phi, *h_theta, *h_fb, *h_x;
  zcplx *h_ovlp, *h_eloc;
  double* h_weight;
  int32_t* h_flags;
  void* h_x2; zcplx* h_eloc2;            // second field / energy staging buffers: copies overlap the previous step
  cudaStream_t copy_stream; cudaEvent_t ev_x[2], ev_done[2], ev_e[2]; int copy_ready;
  cudaEvent_t ev_phi; int ev_phi_armed;   // afqmc_step_host: recorded once the walker of the call's last step is final (after H7)
  // orthonormalisation / comb population control (popctl.cuh)
  size_t ortho_smem;
  void *pc_phi, *pc_theta, *pc_fb; zcplx* pc_ovlp; double *pc_cum, *pc_wnew; int32_t* pc_parent;
  // init staging (FP64)
  double *Ld, *hd, *hpd, *Rd, *hrotd, *ex[4], *psid;
  tc::Maps map_asm, map_fb[2], map_en[2];
  int nblk; int2* blk;   // symmetric block list of the tcgen05 assembly GEMM
  int cta2;   // tcgen05 GEMMs run on CTA pairs (cta_group::2), gemm_path 3
  int ps_ok;  // the persistent pair kernel's shared-memory request was accepted
  int* fb_sched; int fb_stride, fb_ok;   // H4: the same for the force-bias GEMM (both spins, one launch)
  int* en_sched; int en_stride, en_ok;   // H9: tile lists of the persistent energy GEMM (both spins in one launch), [n_sm/2][en_stride]
  int tay_tc; tt::TaylorMaps map_tay; tt::TaylorTcArgs tay_args; size_t tay_tc_smem; int n_sm;   // TMA descriptors of the tcgen05 path (path == 2)
  char err[256];
  int64_t launches;
  // optional per-stage timing (afqmc_profile_enable)
  int prof;
  cudaEvent_t pev[AFQMC_N_STAGES][64][2];
  int pcount[AFQMC_N_STAGES];
};

namespace {

afqmc_status fail(afqmc_ctx* c, afqmc_status s, const char* fmt, const char* a = "") {
  char* dst = c ? c->err : g_init_err;
  snprintf(dst, 256, fmt, a);
  return s;
}

#define CUDA_OK(c, call)                                                              \
  do {                                                                                \
    cudaError_t e_ = (call);                                                          \
    if (e_ != cudaSuccess) return fail((c), AFQMC_ECUDA, "CUDA: %s", cudaGetErrorString(e_)); \
  } while (0)

#define LAUNCH(c, kern, grid, block, smem, ...)                                       \
  do {                                                                                \
    kern<<<(grid), (block), (smem), (c)->stream>>>(__VA_ARGS__);                      \
    (c)->launches++;                                                                  \
    cudaError_t e_ = cudaGetLastError();                                              \
    if (e_ != cudaSuccess) return fail((c), AFQMC_ECUDA, #kern ": %s", cudaGetErrorString(e_)); \
  } while (0)

struct StageScope {
  afqmc_ctx* c; int stage; int slot;
  StageScope(afqmc_ctx* c_, int stage_) : c(c_), stage(stage_), slot(-1) {
    if (c->prof && c->pcount[stage] < 64) {
      slot = c->pcount[stage]++;
      cudaEventRecord(c->pev[stage][slot][0], c->stream);
    }
  }
  ~StageScope() {
    if (slot >= 0) cudaEventRecord(c->pev[stage][slot][1], c->stream);
  }
};

// Taylor kernel configuration: chunk width CW (compile-time), chunks, threads.
template <typename T> int taylor_maxt(int cw) {
  int cwp = (cw + 3) & ~3;
  if (sizeof(T) == 4) return cwp >= 16 ? 448 : cwp >= 12 ? 576 : cwp >= 8 ? 768 : 1024;
  return cwp >= 8 ? 448 : 768;
}
template <typename T> bool taylor_pick(int M, int nt, int& cw, int& nch) {
  const int cwmax = sizeof(T) == 4 ? 16 : 8;
  for (nch = 1; nch <= nt; ++nch) {
    cw = (nt + nch - 1) / nch;
    if (cw <= cwmax && M * nch <= taylor_maxt<T>(cw)) return true;
  }
  return false;
}

struct Layout {
  int M, MP, na, nb, nt, ng, NGP, nw, KA, KB, KT, ts;
  size_t const_bytes, work_bytes;
};

// gemm_path 0 (auto): tcgen05 3xTF32 wherever it exists (complex64 walkers), else SIMT
int resolve_path(const afqmc_params* p) {
  if (p->gemm_path) return p->gemm_path >= 2 ? 2 : 1;
  return p->precision == 0 ? 2 : 1;
}
// the tcgen05 GEMMs run on CTA pairs unless gemm_path 2 asks for the one-CTA kernels
int resolve_cta2(const afqmc_params* p) { return resolve_path(p) == 2 && p->gemm_path != 2; }
// tensor-pipe Taylor kernel (taylor_tc.cuh): complex64 walkers on the tcgen05 path, 96 <= M <= 256, N_t <= 32.  Below
// M = 96 a 128-row tile is mostly padding and the FP32 SIMT kernel is competitive and free of the tensor pipe's
// truncation bias
bool will_tay_tc(const afqmc_params* p) {
  return resolve_path(p) == 2 && p->M >= 96 && p->M <= 256 && p->n_alpha + p->n_beta <= 32;
}

afqmc_status check_params(const afqmc_params* p, char* err) {
  if (!p) { snprintf(err, 256, "params is NULL"); return AFQMC_EINVAL; }
  if (p->M < 1 || p->n_alpha < 1 || p->n_beta < 0 || p->n_chol < 1 || p->n_walkers < 0 ||
      p->n_alpha > p->M || p->n_beta > p->M) {
    snprintf(err, 256, "bad sizes: need M>=1, 1<=n_alpha<=M, 0<=n_beta<=M, n_chol>=1, n_walkers>=0");
    return AFQMC_EINVAL;
  }
  if (p->precision != 0 && p->precision != 1) { snprintf(err, 256, "precision must be 0 or 1"); return AFQMC_EINVAL; }
  if (p->taylor_order < 1 || p->taylor_order > 20) { snprintf(err, 256, "taylor_order must be in 1..20"); return AFQMC_EINVAL; }
  if (p->weight_mode != 0 && p->weight_mode != 1) { snprintf(err, 256, "weight_mode must be 0 or 1"); return AFQMC_EINVAL; }
  if (!(p->dt > 0.0) || !isfinite(p->dt) || !isfinite(p->E0)) { snprintf(err, 256, "dt must be > 0 and finite"); return AFQMC_EINVAL; }
  if (p->gemm_path < 0 || p->gemm_path > 3) { snprintf(err, 256, "gemm_path must be 0, 1, 2 or 3"); return AFQMC_EINVAL; }
  if (p->n_alpha > 32 || p->n_beta > 32) { snprintf(err, 256, "n_alpha, n_beta <= 32 supported"); return AFQMC_EUNSUPPORTED; }
  if (p->n_det < 1) { snprintf(err, 256, "n_det must be >= 1"); return AFQMC_EINVAL; }
  if (p->n_det > 1) {
    if (p->n_act < p->n_alpha || p->n_act < p->n_beta || p->n_act > p->M || p->n_beta < 1) {
      snprintf(err, 256, "multi-det: need max(n_alpha, n_beta) <= n_act <= M and n_beta >= 1"); return AFQMC_EINVAL;
    }
    if (p->max_exc < 1 || p->max_exc > 4) { snprintf(err, 256, "max_exc (excitation rank per spin) must be 1..4"); return AFQMC_EUNSUPPORTED; }
    if (p->n_det > 1024) { snprintf(err, 256, "n_det <= 1024 supported"); return AFQMC_EUNSUPPORTED; }
    if (p->n_act * (p->n_alpha + p->n_beta) > 1024) { snprintf(err, 256, "n_act * N_t <= 1024 supported"); return AFQMC_EUNSUPPORTED; }
    const int ts_ = p->precision ? 8 : 4, emax_ = p->max_exc > 2 ? 4 : 2;
    if (md_energy_smem(p->M, p->n_alpha, p->n_beta, p->n_act, p->n_det, ts_, emax_) > 200 * 1024 ||
        md_overlap_smem(p->M, p->n_alpha, p->n_beta, p->n_act, p->n_det, ts_, emax_) > 200 * 1024) {
      snprintf(err, 256, "multi-det working set exceeds one CTA's shared memory"); return AFQMC_EUNSUPPORTED;
    }
  }
  if (p->gemm_path >= 2 && p->precision != 0) {
    snprintf(err, 256, "gemm_path 2/3 (tcgen05 3xTF32) needs precision 0 (complex64 walkers)");
    return AFQMC_EUNSUPPORTED;
  }
  if (!will_tay_tc(p)) {   // the one-CTA SIMT Taylor kernel's size limit applies only where the tensor-pipe kernel does not run
    int cw, nch;
    bool ok = p->precision ? taylor_pick<double>(p->M, p->n_alpha + p->n_beta, cw, nch)
                           : taylor_pick<float>(p->M, p->n_alpha + p->n_beta, cw, nch);
    if (!ok) { snprintf(err, 256, "M * ceil(N_t / chunk) exceeds one CTA (M too large for the SIMT Taylor kernel; the tensor-pipe kernel needs complex64, 96 <= M <= 256, N_t <= 32)"); return AFQMC_EUNSUPPORTED; }
  }
  size_t gs = p->precision ? green_smem_bytes<double>(p->M, p->n_alpha, p->n_beta)
                           : green_smem_bytes<float>(p->M, p->n_alpha, p->n_beta);
  if (gs > 200 * 1024) { snprintf(err, 256, "walker does not fit one CTA's shared memory"); return AFQMC_EUNSUPPORTED; }
  return AFQMC_OK;
}

// Carve (or just size, when base pointers are null) every buffer.
void carve(const afqmc_params* p, afqmc_ctx* c, char* cbase, char* wbase, size_t* cb, size_t* wb) {
  const int M = p->M, na = p->n_alpha, nb = p->n_beta, nt = na + nb, ng = p->n_chol, nw = p->n_walkers;
  const int ts = p->precision ? 8 : 4;
  const int MP = (M + 3) & ~3, NGP = (int)rup(ng, 32);
  const int md = p->n_det > 1;
  const int ca = md ? p->n_act : na, cb_ = md ? p->n_act : nb;
  const int KA = (int)rup((size_t)M * ca, 32), KB = (int)rup((size_t)M * cb_, 32), KT = KA + KB;
  c->md = md; c->nact = md ? p->n_act : 0; c->ndet = p->n_det; c->ca = ca; c->cb = cb_;
  c->M = M; c->MP = MP; c->na = na; c->nb = nb; c->nt = nt; c->ng = ng; c->NGP = NGP; c->nw = nw;
  c->KA = KA; c->KB = KB; c->KT = KT; c->ts = ts;
  const int split = c->split;
  Carver cc; cc.base = cbase;
  c->psi_a = cc.take((size_t)M * na * ts);
  c->psi_b = cc.take((size_t)M * (nb ? nb : 1) * ts);
  c->psid_ac = (double*)cc.take((size_t)M * na * 8);
  c->psid_bc = (double*)cc.take((size_t)M * (nb ? nb : 1) * 8);
  c->Eh = cc.take((size_t)M * MP * ts);
  // tcgen05 path: only the 8 x 16 blocks (i-block, j-block) that touch the upper triangle of the symmetric A_w
  c->nblk = 0;
  for (int ib = 0; ib * 8 < M; ++ib)
    for (int jb = 0; jb * 16 < M; ++jb)
      if (ib * 8 <= jb * 16 + 15) ++c->nblk;
  const size_t lt_rows = split ? (size_t)c->nblk * 128 : (size_t)M * M;
  c->Lt = cc.take(lt_rows * NGP * ts);
  c->Lt_lo = split ? cc.take(lt_rows * NGP * ts) : nullptr;
  c->blk = (int2*)cc.take((size_t)(c->nblk ? c->nblk : 1) * sizeof(int2));
  c->en_sched = (int*)cc.take(EN_SCHED_INTS * sizeof(int));
  c->fb_sched = (int*)cc.take(EN_SCHED_INTS * sizeof(int));
  c->Rall = cc.take((size_t)rup(ng, 128) * KT * ts);
  c->Rall_lo = split ? cc.take((size_t)rup(ng, 128) * KT * ts) : nullptr;
  const size_t ya = md ? 32 : KA, yb = (md || !KB) ? 32 : KB;   // Y is not used by the multi-det energy
  c->Y[0] = cc.take(ya * ya * ts);
  c->Y[1] = cc.take(yb * yb * ts);
  c->Y_lo[0] = split ? cc.take(ya * ya * ts) : nullptr;
  c->Y_lo[1] = split ? cc.take(yb * yb * ts) : nullptr;
  c->hrot = cc.take((size_t)KT * ts);
  c->Cact = cc.take((size_t)M * (md ? p->n_act : 1) * ts);
  c->coeff = (double*)cc.take((size_t)p->n_det * 8);
  c->exc = (int32_t*)cc.take((size_t)p->n_det * 16 * 4);      // [n_det][2][emax <= 4][2]
  c->MPK = (int)rup(M, 32);   // K of the TT GEMM, padded to the tcgen05 k-block
  c->RactT = cc.take(md ? (size_t)(ng + 1) * p->n_act * c->MPK * ts : 256);
  c->RactT_lo = (md && split) ? cc.take((size_t)(ng + 1) * p->n_act * c->MPK * ts) : nullptr;
  *cb = cc.off;

  Carver w; w.base = wbase;
  const size_t nw1 = nw ? nw : 1;
  c->Z = w.take(2 * nw1 * NGP * ts);
  c->Z_lo = split ? w.take(2 * nw1 * NGP * ts) : nullptr;
  c->Abuf = w.take(nw1 * M * 2 * MP * ts);
  c->thp = w.take(2 * nw1 * KT * ts);
  c->thp_lo = split ? w.take(2 * nw1 * KT * ts) : nullptr;
  c->fs = w.take(2 * 2 * nw1 * NGP * ts);
  c->thtil = w.take(md ? nw1 * M * 2 * p->n_act * 2 * ts : 256);
  c->th_scr = w.take(md ? nw1 * M * nt * 2 * ts : 256);
  c->thT = w.take(md ? nw1 * 2 * nt * c->MPK * ts : 256);
  c->thT_lo = (md && split) ? w.take(nw1 * 2 * nt * c->MPK * ts) : nullptr;
  c->TTg = w.take(md ? nw1 * (ng + 1) * p->n_act * nt * 2 * ts : 256);
  c->ovlp0 = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->ovlp_scr = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->cshift = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->eloc_scratch = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->h_phi = w.take(nw1 * M * nt * 2 * ts);
  c->h_theta = w.take(nw1 * M * nt * 2 * ts);
  c->h_fb = w.take(nw1 * ng * 2 * ts);
  c->h_x = w.take(nw1 * ng * ts);
  c->h_ovlp = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->h_eloc = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->h_weight = (double*)w.take(nw1 * sizeof(double));
  c->h_flags = (int32_t*)w.take(nw1 * sizeof(int32_t));
  c->h_x2 = w.take(nw1 * ng * ts);
  c->h_eloc2 = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->pc_phi = w.take(nw1 * M * nt * 2 * ts);
  c->pc_theta = w.take(nw1 * M * nt * 2 * ts);
  c->pc_fb = w.take(nw1 * ng * 2 * ts);
  c->pc_ovlp = (zcplx*)w.take(nw1 * sizeof(zcplx));
  c->pc_cum = (double*)w.take(nw1 * sizeof(double));
  c->pc_wnew = (double*)w.take(256);
  c->pc_parent = (int32_t*)w.take(nw1 * sizeof(int32_t));
  // FP64 init staging
  c->Ld = (double*)w.take((size_t)ng * M * M * 8);
  c->hd = (double*)w.take((size_t)M * M * 8);
  c->hpd = (double*)w.take((size_t)M * M * 8);
  c->Rd = (double*)w.take((size_t)ng * KT * 8);
  c->hrotd = (double*)w.take((size_t)KT * 8);
  for (int i = 0; i < 4; ++i) c->ex[i] = (double*)w.take((size_t)M * M * 8);
  c->psid = (double*)w.take((size_t)M * (nt + (md ? p->n_act : 0)) * 8);
  *wb = w.off;
}

template <typename T> afqmc_status init_device(afqmc_ctx* c, const double* h1, const double* L, const double* pa, const double* pb,
                                              const double* Cact_h, const double* coeff_h, const int32_t* exc_h) {
  const int M = c->M, MP = c->MP, na = c->na, nb = c->nb, ng = c->ng, NGP = c->NGP, KA = c->KA, KB = c->KB, KT = c->KT;
  cudaStream_t st = c->stream;
  size_t cb, wb;
  {
    afqmc_ctx tmp = *c;
    carve(&c->p, &tmp, nullptr, nullptr, &cb, &wb);
  }
  CUDA_OK(c, cudaMemsetAsync(c->psi_a, 0, cb, st));           // const_mem starts at psi_a
  CUDA_OK(c, cudaMemsetAsync(c->Z, 0, wb, st));               // work_mem starts at Z
  CUDA_OK(c, cudaMemcpyAsync(c->hd, h1, (size_t)M * M * 8, cudaMemcpyHostToDevice, st));
  CUDA_OK(c, cudaMemcpyAsync(c->Ld, L, (size_t)ng * M * M * 8, cudaMemcpyHostToDevice, st));
  double* psid_a = c->psid;
  double* psid_b = c->psid + (size_t)M * na;
  CUDA_OK(c, cudaMemcpyAsync(psid_a, pa, (size_t)M * na * 8, cudaMemcpyHostToDevice, st));
  if (nb) CUDA_OK(c, cudaMemcpyAsync(psid_b, pb, (size_t)M * nb * 8, cudaMemcpyHostToDevice, st));

  const int mm = M * M;
  LAUNCH(c, k_init_hprime, (mm + 127) / 128, 128, 0, M, ng, c->hd, c->Ld, c->hpd);
  // E_h = expm(-(dt/2) h') by scaling and squaring of an order-18 Taylor (Horner) series, FP64
  std::vector<double> hp((size_t)mm);
  CUDA_OK(c, cudaMemcpyAsync(hp.data(), c->hpd, (size_t)mm * 8, cudaMemcpyDeviceToHost, st));
  CUDA_OK(c, cudaStreamSynchronize(st));
  double n1 = 0.0;
  for (int j = 0; j < M; ++j) {
    double s = 0.0;
    for (int i = 0; i < M; ++i) s += fabs(hp[(size_t)i * M + j]);
    n1 = fmax(n1, s);
  }
  if (!isfinite(n1)) return fail(c, AFQMC_EINVAL, "h1 / L_chol contain non-finite values");
  n1 *= 0.5 * c->p.dt;
  int sq = 0;
  while (n1 > 0.5 && sq < 60) { n1 *= 0.5; ++sq; }
  double* X = c->ex[0];
  double* E = c->ex[1];
  double* Tm = c->ex[2];
  LAUNCH(c, k_dscale_eye, (mm + 127) / 128, 128, 0, M, -0.5 * c->p.dt / ldexp(1.0, sq), c->hpd, 0.0, X);
  LAUNCH(c, k_dscale_eye, (mm + 127) / 128, 128, 0, M, 0.0, c->hpd, 1.0, E);
  for (int k = 18; k >= 1; --k) {
    LAUNCH(c, k_dgemm_small, (mm + 127) / 128, 128, 0, M, 1.0 / k, X, E, 0.0, (const double*)nullptr, Tm);
    LAUNCH(c, k_dscale_eye, (mm + 127) / 128, 128, 0, M, 1.0, Tm, 1.0, E);
  }
  for (int s = 0; s < sq; ++s) {
    LAUNCH(c, k_dgemm_small, (mm + 127) / 128, 128, 0, M, 1.0, E, E, 0.0, (const double*)nullptr, Tm);
    double* t = E; E = Tm; Tm = t;
  }
  LAUNCH(c, k_cast2d<T>, (mm + 127) / 128, 128, 0, M, M, E, (size_t)M, (T*)c->Eh, (T*)nullptr, (size_t)MP, 0);
  if (c->tay_tc) {   // D_h = E_h - 1 in FP32 for the tensor-pipe Taylor kernel, which splits it on the fly (the SIMT kernel never runs then)
    LAUNCH(c, k_dscale_eye, (mm + 127) / 128, 128, 0, M, 1.0, E, -1.0, Tm);
    LAUNCH(c, k_cast2d<T>, (mm + 127) / 128, 128, 0, M, M, Tm, (size_t)M, (T*)c->Eh, (T*)nullptr, (size_t)MP, 0);
  }
  CUDA_OK(c, cudaMemcpyAsync(c->psid_ac, psid_a, (size_t)M * na * 8, cudaMemcpyDeviceToDevice, st));
  if (nb) CUDA_OK(c, cudaMemcpyAsync(c->psid_bc, psid_b, (size_t)M * nb * 8, cudaMemcpyDeviceToDevice, st));
  // trial orbitals in T
  LAUNCH(c, k_cast2d<T>, (M * na + 127) / 128, 128, 0, M, na, psid_a, (size_t)na, (T*)c->psi_a, (T*)nullptr, (size_t)na, 0);
  if (nb) LAUNCH(c, k_cast2d<T>, (M * nb + 127) / 128, 128, 0, M, nb, psid_b, (size_t)nb, (T*)c->psi_b, (T*)nullptr, (size_t)nb, 0);
  double* Cact_d = c->psid + (size_t)M * (na + nb);
  if (c->md) {
    const int nact = c->nact;
    CUDA_OK(c, cudaMemcpyAsync(Cact_d, Cact_h, (size_t)M * nact * 8, cudaMemcpyHostToDevice, st));
    CUDA_OK(c, cudaMemcpyAsync(c->coeff, coeff_h, (size_t)c->ndet * 8, cudaMemcpyHostToDevice, st));
    CUDA_OK(c, cudaMemcpyAsync(c->exc, exc_h, (size_t)c->ndet * 4 * c->emax * 4, cudaMemcpyHostToDevice, st));
    LAUNCH(c, k_cast2d<T>, (M * nact + 127) / 128, 128, 0, M, nact, Cact_d, (size_t)nact, (T*)c->Cact, (T*)nullptr,
           (size_t)nact, 0);
  }
  // R^s_g = Psi_s^T L_g and Psi_s^T h, spin-blocked index (s_off + k*n_s + a); multi-det: C_act^T L_g for both spins
  for (int s = 0; s < 2; ++s) {
    int n = s ? c->cb : c->ca, soff = s ? KA : 0;
    if (!n) continue;
    const double* C = c->md ? Cact_d : (s ? psid_b : psid_a);
    size_t tot = (size_t)ng * M * n;
    LAUNCH(c, k_init_rot, (unsigned)((tot + 127) / 128), 128, 0, M, n, n, C, ng, c->Ld, soff, KT, c->Rd);
    LAUNCH(c, k_init_rot, (M * n + 127) / 128, 128, 0, M, n, n, C, 1, c->hd, soff, KT, c->hrotd);
    int Ks = s ? KB : KA;
    if (!c->md)
    LAUNCH(c, k_init_Y<T>, dim3((M * n + 127) / 128, M * n), 128, 0, M, n, ng, c->Rd, soff, KT, (T*)c->Y[s],
           (T*)c->Y_lo[s], Ks, c->split);
  }
  if (c->md) {
    size_t tot = (size_t)(ng + 1) * c->nact * M;
    LAUNCH(c, k_init_ractT<T>, (unsigned)((tot + 127) / 128), 128, 0, ng, c->nact, M, c->MPK, c->Rd, KT, c->hrotd, (T*)c->RactT, (T*)c->RactT_lo);
  }
  {
    size_t tot = (size_t)ng * KT;
    LAUNCH(c, k_cast2d<T>, (unsigned)((tot + 127) / 128), 128, 0, ng, KT, c->Rd, (size_t)KT, (T*)c->Rall, (T*)c->Rall_lo,
           (size_t)KT, c->split);
    LAUNCH(c, k_cast2d<T>, (KT + 127) / 128, 128, 0, 1, KT, c->hrotd, (size_t)KT, (T*)c->hrot, (T*)nullptr, (size_t)KT, 0);
  }
  // Lt[ij][g] = L[g][ij]  (K-major operand of the assembly GEMM); tcgen05 path: symmetric block packing
  if (c->split) {
    std::vector<int2> tab;
    for (int ib = 0; ib * 8 < M; ++ib)
      for (int jb = 0; jb * 16 < M; ++jb)
        if (ib * 8 <= jb * 16 + 15) tab.push_back(make_int2(ib, jb));
    // order: 32 x 32 super-blocks (4 ib x 2 jb), blocks row-major inside.  Tiles that run at the same time then write
    // whole 128-byte lines of A_w in both orientations (a block alone writes 64-byte runs (i, j..j+15) and 32-byte
    // runs (j, i..i+7)), which L2 merges before they reach HBM
    std::stable_sort(tab.begin(), tab.end(), [](const int2& a, const int2& b) {
      const int ka[4] = {a.x >> 2, a.y >> 1, a.x, a.y}, kb[4] = {b.x >> 2, b.y >> 1, b.x, b.y};
      for (int t = 0; t < 4; ++t) if (ka[t] != kb[t]) return ka[t] < kb[t];
      return false;
    });
    CUDA_OK(c, cudaMemcpyAsync(c->blk, tab.data(), tab.size() * sizeof(int2), cudaMemcpyHostToDevice, st));
    CUDA_OK(c, cudaStreamSynchronize(st));
    size_t tot = (size_t)c->nblk * 128 * ng;
    LAUNCH(c, k_pack_Lt<T>, (unsigned)((tot + 255) / 256), 256, 0, M, ng, NGP, c->nblk, c->blk, c->Ld, (T*)c->Lt, (T*)c->Lt_lo);
  } else
  LAUNCH(c, k_transpose_cast<T>, dim3((ng + 31) / 32, (mm + 31) / 32), dim3(32, 8), 0, mm, ng, c->Ld, (size_t)mm,
         (T*)c->Lt, (T*)c->Lt_lo, (size_t)NGP, c->split);
  CUDA_OK(c, cudaStreamSynchronize(st));
  return AFQMC_OK;
}

// ---- stage launchers -------------------------------------------------------------------------

template <typename T>
afqmc_status run_green(afqmc_ctx* c, const void* phi, void* ovlp, void* theta, int do_weight, double* weight,
                       const void* eloc_pre, int32_t* flags) {
  GreenArgs<T> g;
  g.M = c->M; g.na = c->na; g.nb = c->nb; g.nw = c->nw;
  g.phi = (const cplx<T>*)phi; g.psi_a = (const T*)c->psi_a; g.psi_b = (const T*)c->psi_b;
  g.psid_a = c->psid_ac; g.psid_b = c->psid_bc;
  g.theta = (cplx<T>*)theta; g.thp = (T*)c->thp; g.thp_lo = (T*)c->thp_lo;
  g.KA = c->KA; g.KT = c->KT; g.split = c->split;
  g.ovlp = (zcplx*)ovlp; g.do_weight = do_weight; g.cshift = c->cshift; g.weight = weight;
  g.eloc_pre = (const zcplx*)eloc_pre; g.weight_mode = c->p.weight_mode; g.dt = c->p.dt; g.E0 = c->p.E0;
  g.flags = flags;
  StageScope sc(c, AFQMC_STAGE_GREEN);
  if (c->md) {
    // reference determinant first (S_0 to scratch, no weights), then SMW over all determinants
    g.thp = nullptr; g.thp_lo = nullptr; g.ovlp = c->ovlp0; g.do_weight = 0;
    LAUNCH(c, k_green<T>, c->nw, 256, c->green_smem, g);
    MdOverlapArgs<T> a;
    a.m.M = c->M; a.m.na = c->na; a.m.nb = c->nb; a.m.nact = c->nact; a.m.ndet = c->ndet;
    a.m.C = c->Cact; a.m.coeff = c->coeff; a.m.exc = c->exc; a.m.emax = c->emax;
    a.theta0 = (const cplx<T>*)theta; a.ovlp0 = c->ovlp0; a.thtil = (cplx<T>*)c->thtil; a.ovlp = (zcplx*)ovlp;
    a.do_weight = do_weight; a.cshift = c->cshift; a.weight = weight; a.eloc_pre = (const zcplx*)eloc_pre;
    a.weight_mode = c->p.weight_mode; a.dt = c->p.dt; a.E0 = c->p.E0; a.flags = flags;
    LAUNCH(c, k_md_overlap<T>, c->nw, 256, c->mdo_smem, a);
    LAUNCH(c, k_planarize<T>, c->nw, 128, 0, c->M, c->nact, c->nact, c->KA, c->KT, c->split, (const cplx<T>*)c->thtil,
           (T*)c->thp, (T*)c->thp_lo);
    return AFQMC_OK;
  }
  LAUNCH(c, k_green<T>, c->nw, 256, c->green_smem, g);
  return AFQMC_OK;
}

template <typename T, class Epi>
afqmc_status run_gemm(afqmc_ctx* c, const T* A, int lda, int m, const T* B, int ldb, int n, int K, Epi epi) {
  typedef GemmCfg<T> G;
  dim3 grid((n + G::BN - 1) / G::BN, (m + G::BM - 1) / G::BM);
  auto kern = k_gemm_nt<T, Epi>;
  LAUNCH(c, kern, grid, 256, 0, A, lda, m, B, ldb, n, K, epi);
  return AFQMC_OK;
}

template <class Epi>
afqmc_status run_gemm_tc(afqmc_ctx* c, const tc::Maps& maps, int m, int n, int K, Epi epi, int tri = 0, bool pair_ok = true) {
  dim3 grid((n + tc::BN - 1) / tc::BN, (m + tc::BM - 1) / tc::BM);
  if (c->cta2 && pair_ok) {
    const int m_tiles = (int)grid.y;
    const int n_tiles = (int)grid.x;
    if constexpr (Epi::kStaged) {
      // persistent pairs: the staged epilogue of one tile overlaps the main loop of the next
      const int n_pairs = (m_tiles + 1) / 2 * n_tiles, slots = c->n_sm / 2;
      if (!tri && slots > 0 && c->ps_ok) {
        dim3 gridp(2 * (n_pairs < slots ? n_pairs : slots));
        tc::PsWork wk{};
        wk.K[0] = K; wk.m_tiles[0] = m_tiles; wk.n_tiles = n_tiles; wk.n_pairs = n_pairs;
        auto kernp = tc::k_gemm_tf32_pair_ps<Epi>;
        LAUNCH(c, kernp, gridp, tc::PS_THREADS, tc::SMEM_PS_BYTES, maps, maps, wk, epi, epi);
        return AFQMC_OK;
      }
    }
    dim3 grid2(((grid.y + 1) & ~1u) * grid.x);   // CTA pairs = clusters of two adjacent row tiles, 1-D grid
    auto kern2 = tc::k_gemm_tf32_pair<Epi>;
    LAUNCH(c, kern2, grid2, tc::THREADS, tc::SMEM_BYTES, maps, K, tri, m_tiles, n_tiles, epi);
    return AFQMC_OK;
  }
  auto kern = tc::k_gemm_tf32<Epi>;
  LAUNCH(c, kern, grid, tc::THREADS, tc::SMEM_BYTES, maps, K, tri, epi);
  return AFQMC_OK;
}

// per-spin traces f^s_g = sum R^s_g[a][k] Theta_s[k][a] from the planar Theta in ctx->thp
template <typename T> afqmc_status run_fb_gemm(afqmc_ctx* c) {
  StageScope sc(c, AFQMC_STAGE_FORCE_BIAS);
  if constexpr (sizeof(T) == 4) {
    if (c->path == 2 && c->cta2 && c->fb_ok) {   // both spins, one persistent launch; stores overlap the next tile's main loop
      tc::EpiStoreT e[2];
      tc::PsWork wk{};
      for (int s = 0; s < 2; ++s) {
        e[s].out = (float*)c->fs + (size_t)s * 2 * c->nw * c->NGP; e[s].ldo = c->NGP; e[s].m_real = c->ng; e[s].n_real = 2 * c->nw;
        wk.K[s] = s ? c->KB : c->KA; wk.m_tiles[s] = (c->ng + tc::BM - 1) / tc::BM;
      }
      wk.n_tiles = (2 * c->nw + tc::BN - 1) / tc::BN; wk.sched = c->fb_sched; wk.sched_stride = c->fb_stride;
      auto kernp = tc::k_gemm_tf32_pair_ps<tc::EpiStoreT, EN_CHUNK, true>;
      LAUNCH(c, kernp, dim3(2 * (c->n_sm / 2)), tc::PS_THREADS, tc::SMEM_PS_BYTES, c->map_fb[0], c->map_fb[c->cb ? 1 : 0], wk, e[0], e[1]);
      return AFQMC_OK;
    }
  }
  for (int s = 0; s < 2; ++s) {
    int n = s ? c->cb : c->ca, soff = s ? c->KA : 0, Ks = s ? c->KB : c->KA;
    if (!n) continue;
    if constexpr (sizeof(T) == 4) {
      if (c->path == 2) {
        tc::EpiStoreT e2;
        e2.out = (float*)c->fs + (size_t)s * 2 * c->nw * c->NGP; e2.ldo = c->NGP; e2.m_real = c->ng; e2.n_real = 2 * c->nw;
        afqmc_status st2 = run_gemm_tc(c, c->map_fb[s], c->ng, 2 * c->nw, Ks, e2);
        if (st2) return st2;
        continue;
      }
    }
    EpiStoreT<T> epi;
    epi.out = (T*)c->fs + (size_t)s * 2 * c->nw * c->NGP; epi.ldo = c->NGP; epi.m_real = c->ng; epi.n_real = 2 * c->nw;
    afqmc_status st = run_gemm<T>(c, (const T*)c->Rall + soff, c->KT, c->ng, (const T*)c->thp + soff, c->KT, 2 * c->nw, Ks, epi);
    if (st) return st;
  }
  return AFQMC_OK;
}

template <typename T> afqmc_status run_md_energy(afqmc_ctx* c, const void* theta, zcplx* eloc) {
  StageScope sc(c, AFQMC_STAGE_ENERGY);
  MdEnergyArgs<T> a;
  a.m.M = c->M; a.m.na = c->na; a.m.nb = c->nb; a.m.nact = c->nact; a.m.ndet = c->ndet;
  a.m.C = c->Cact; a.m.coeff = c->coeff; a.m.exc = c->exc; a.m.emax = c->emax;
  a.ng = c->ng; a.ldr = c->KT; a.theta0 = (const cplx<T>*)theta; a.TTg = (const cplx<T>*)c->TTg;
  a.eloc = eloc;
  // TT[w][g][q][a] = sum_k (C_act^T X_g)[q][k] Theta_0[w][k][a] for every g (and h) in one GEMM over all walkers
  LAUNCH(c, k_thT<T>, c->nw, 128, 0, c->M, c->nt, c->MPK, (const cplx<T>*)theta, (T*)c->thT, (T*)c->thT_lo);
  bool tt_done = false;
  if constexpr (sizeof(T) == 4) {
    if (c->path == 2) {
      tc::EpiTT e2;
      e2.out = (float*)c->TTg; e2.ng1 = c->ng + 1; e2.nact = c->nact; e2.nt = c->nt;
      e2.m_real = (c->ng + 1) * c->nact; e2.n_real = c->nw * 2 * c->nt;
      // K is one or two k-blocks here: the epilogue is the whole kernel and the pair's cluster barriers only cost
      afqmc_status st = run_gemm_tc(c, c->map_tt, e2.m_real, e2.n_real, c->MPK, e2, 0, false);
      if (st) return st;
      tt_done = true;
    }
  }
  if (!tt_done) {
    EpiTT<T> epi;
    epi.out = (T*)c->TTg; epi.ng1 = c->ng + 1; epi.nact = c->nact; epi.nt = c->nt;
    epi.m_real = (c->ng + 1) * c->nact; epi.n_real = c->nw * 2 * c->nt;
    afqmc_status st = run_gemm<T>(c, (const T*)c->RactT, c->MPK, epi.m_real, (const T*)c->thT, c->MPK, epi.n_real, c->MPK, epi);
    if (st) return st;
  }
  const int dpt = (c->ndet + MD_THREADS - 1) / MD_THREADS;
  if constexpr (sizeof(T) == 4) {
    // batched-gamma kernel (gemm_path 1 keeps the one-operator-at-a-time kernel): n_sigma <= 16, <= 2 determinants per thread (more would spill its per-determinant
    // registers), tiles that are 16-byte multiples, shared memory that fits
    const int nmax = c->na > c->nb ? c->na : c->nb;
    const size_t smb = md_energy_b_smem(c->M, c->na, c->nb, c->nact, c->ndet, c->ts);
    if (c->path == 2 && c->emax == 2 && nmax <= 16 && dpt <= 2 && ((size_t)c->nact * c->nt * 2 * c->ts) % 16 == 0 && smb <= 200 * 1024) {
#define MDB_LAUNCH(N, D)                                                                                           \
  {                                                                                                                \
    auto kern = k_md_energy_b<T, N, D>;                                                                            \
    if (smb > 48 * 1024 && !c->mde_attr_done)   /* once per context: the first energy call */                      \
      CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smb));               \
    c->mde_attr_done = 1;                                                                                          \
    LAUNCH(c, kern, c->nw, MD_THREADS, smb, a);                                                                    \
  }
#define MDB_PICK(N)                                                                                                \
  { if (dpt <= 1) MDB_LAUNCH(N, 1) else MDB_LAUNCH(N, 2) }
      if (nmax <= 8) MDB_PICK(8) else if (nmax <= 12) MDB_PICK(12) else MDB_PICK(16)
#undef MDB_PICK
#undef MDB_LAUNCH
      return AFQMC_OK;
    }
  }
#define MDE_LAUNCH(D)                                                                                              \
  {                                                                                                                \
    auto kern = k_md_energy<T, D>;                                                                                 \
    if (c->mde_smem > 48 * 1024 && !c->mde_attr_done)                                                              \
      CUDA_OK(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->mde_smem));       \
    c->mde_attr_done = 1;                                                                                          \
    LAUNCH(c, kern, c->nw, MD_THREADS, c->mde_smem, a);                                                            \
  }
  if (dpt <= 1) MDE_LAUNCH(1) else if (dpt <= 2) MDE_LAUNCH(2) else if (dpt <= 4) MDE_LAUNCH(4) else MDE_LAUNCH(8)
#undef MDE_LAUNCH
  return AFQMC_OK;
}

// Tile lists of the persistent pair kernel's LIST instantiation (H9, H4): every (problem, row pair, column tile) with its
// cost (k-blocks -- from the pair's diagonal block on when `tri` -- plus `epi_cost` for the epilogue), longest first onto the
// least loaded CTA pair (LPT).  Tiles of one row pair cost the same, sit next to each other in the order and so start
// at about the same time on different pairs: they share their rows of the a-operand in L2.
static bool build_pair_schedule(const afqmc_ctx* c, int tri, const int m_rows[2], const int K[2], int epi_cost,
                                std::vector<int>& out, int& stride) {
  const int slots = c->n_sm / 2, n_tiles = (2 * c->nw + tc::BN - 1) / tc::BN;
  if (slots <= 0) return false;
  struct Item { int cost, entry; };
  std::vector<Item> items;
  for (int sp = 0; sp < 2; ++sp) {
    if (!m_rows[sp] || !K[sp]) continue;
    const int m_tiles = (m_rows[sp] + tc::BM - 1) / tc::BM;
    for (int mp = 0; mp < (m_tiles + 1) / 2; ++mp) {
      const int nkb = K[sp] / tc::BK - (tri ? (mp * 2 * tc::BM) / tc::BK : 0);
      if (nkb <= 0) return false;
      for (int nt = 0; nt < n_tiles; ++nt) items.push_back({nkb + epi_cost, (sp << 24) | (mp * n_tiles + nt)});
    }
  }
  if (items.empty()) return false;
  std::stable_sort(items.begin(), items.end(), [](const Item& a, const Item& b) { return a.cost > b.cost; });
  std::vector<std::vector<int>> lists(slots);
  std::vector<long> load(slots, 0);
  for (const Item& it : items) {
    int best = 0;
    for (int k = 1; k < slots; ++k) if (load[k] < load[best]) best = k;
    lists[best].push_back(it.entry); load[best] += it.cost;
  }
  size_t longest = 0;
  for (auto& l : lists) longest = l.size() > longest ? l.size() : longest;
  stride = (int)longest + 1;
  if ((size_t)stride * slots > EN_SCHED_INTS) return false;
  out.assign((size_t)stride * slots, -1);
  for (int k = 0; k < slots; ++k) for (size_t j = 0; j < lists[k].size(); ++j) out[(size_t)k * stride + j] = lists[k][j];
  return true;
}

template <typename T> afqmc_status run_energy_gemm(afqmc_ctx* c, const void* theta, zcplx* eloc) {
  StageScope sc(c, AFQMC_STAGE_ENERGY);
  if constexpr (sizeof(T) == 4) {
    if (c->path == 2 && c->cta2 && c->en_ok) {   // both spins, one persistent launch
      tc::EpiEnergy e[2];
      tc::PsWork wk{};
      for (int s = 0; s < 2; ++s) {
        const int n = s ? c->nb : c->na, soff = s ? c->KA : 0;
        e[s].theta = (const float2*)theta; e[s].M = c->M; e[s].nt = c->nt; e[s].off = s ? c->na : 0; e[s].n = n ? n : 1;
        e[s].hrot = (const float*)c->hrot + soff; e[s].eloc = (double*)eloc; e[s].m_real = c->M * n; e[s].n_real = 2 * c->nw;
        wk.K[s] = s ? c->KB : c->KA; wk.m_tiles[s] = (c->M * n + tc::BM - 1) / tc::BM;
      }
      wk.n_tiles = (2 * c->nw + tc::BN - 1) / tc::BN; wk.tri = 1; wk.sched = c->en_sched; wk.sched_stride = c->en_stride;
      auto kernp = tc::k_gemm_tf32_pair_ps<tc::EpiEnergy, EN_CHUNK, true>;
      LAUNCH(c, kernp, dim3(2 * (c->n_sm / 2)), tc::PS_THREADS, tc::SMEM_PS_BYTES, c->map_en[0], c->map_en[c->nb ? 1 : 0], wk, e[0], e[1]);
      return AFQMC_OK;
    }
  }
  for (int s = 0; s < 2; ++s) {
    int n = s ? c->nb : c->na, soff = s ? c->KA : 0, Ks = s ? c->KB : c->KA;
    if (!n) continue;
    if constexpr (sizeof(T) == 4) {
      if (c->path == 2) {
        tc::EpiEnergy e2;
        e2.theta = (const float2*)theta; e2.M = c->M; e2.nt = c->nt; e2.off = s ? c->na : 0; e2.n = n;
        e2.hrot = (const float*)c->hrot + soff; e2.eloc = (double*)eloc; e2.m_real = c->M * n; e2.n_real = 2 * c->nw;
        afqmc_status st2 = run_gemm_tc(c, c->map_en[s], c->M * n, 2 * c->nw, Ks, e2, 1);
        if (st2) return st2;
        continue;
      }
    }
    EpiEnergy<T> epi;
    epi.thp = (const T*)c->thp; epi.thp_lo = (const T*)c->thp_lo; epi.KT = c->KT; epi.soff = soff;
    epi.hrot = (const T*)c->hrot + soff; epi.eloc = (double*)eloc; epi.m_real = c->M * n; epi.n_real = 2 * c->nw;
    afqmc_status st = run_gemm<T>(c, (const T*)c->Y[s], Ks, c->M * n, (const T*)c->thp + soff, c->KT, 2 * c->nw, Ks, epi);
    if (st) return st;
  }
  return AFQMC_OK;
}

template <typename T> afqmc_status run_taylor(afqmc_ctx* c, void* phi) {
  TaylorArgs<T> g;
  g.M = c->M; g.MP = c->MP; g.nt = c->nt; g.K = c->p.taylor_order; g.nchunks = c->tay_nch;
  g.phi = (cplx<T>*)phi; g.A = (const T*)c->Abuf; g.Eh = (const T*)c->Eh;
  StageScope sc(c, AFQMC_STAGE_TAYLOR);
  if constexpr (sizeof(T) == 4) {
    if (c->tay_tc) {
      tt::TaylorTcArgs a = c->tay_args;
      a.phi = (cplx<float>*)phi;
      const int grid = c->nw < c->n_sm ? c->nw : c->n_sm;
      LAUNCH(c, tt::k_taylor_tc, grid, tt::NTHREADS, c->tay_tc_smem, c->map_tay, a);
      return AFQMC_OK;
    }
  }
#define TAY_CASE(CW)                                                                                        \
  case CW: {                                                                                                \
    constexpr int MT = sizeof(T) == 4 ? (((CW + 3) & ~3) >= 16 ? 448 : ((CW + 3) & ~3) >= 12 ? 576 : ((CW + 3) & ~3) >= 8 ? 768 : 1024) \
                                      : (((CW + 3) & ~3) >= 8 ? 448 : 768);                                 \
    auto kern = k_taylor<T, CW, MT>;                                                                        \
    LAUNCH(c, kern, c->nw, c->tay_threads, c->tay_smem, g);                                                 \
  } break;
  switch (c->tay_cw) {
    TAY_CASE(1) TAY_CASE(2) TAY_CASE(3) TAY_CASE(4) TAY_CASE(5) TAY_CASE(6) TAY_CASE(7) TAY_CASE(8)
    default:
      if constexpr (sizeof(T) == 4) {
        switch (c->tay_cw) {
          TAY_CASE(9) TAY_CASE(10) TAY_CASE(11) TAY_CASE(12) TAY_CASE(13) TAY_CASE(14) TAY_CASE(15) TAY_CASE(16)
          default: return fail(c, AFQMC_EUNSUPPORTED, "taylor chunk width");
        }
      } else {
        return fail(c, AFQMC_EUNSUPPORTED, "taylor chunk width");
      }
  }
#undef TAY_CASE
  return AFQMC_OK;
}

// dynamic shared-memory opt-in of the SIMT Taylor instantiation that run_taylor will launch (called once, from afqmc_init)
template <typename T> cudaError_t set_taylor_smem(int cw, size_t smem) {
#define TAY_SET(CW)                                                                                          \
  case CW: {                                                                                                \
    constexpr int MT = sizeof(T) == 4 ? (((CW + 3) & ~3) >= 16 ? 448 : ((CW + 3) & ~3) >= 12 ? 576 : ((CW + 3) & ~3) >= 8 ? 768 : 1024) \
                                      : (((CW + 3) & ~3) >= 8 ? 448 : 768);                                 \
    return cudaFuncSetAttribute(k_taylor<T, CW, MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
  }
  switch (cw) {
    TAY_SET(1) TAY_SET(2) TAY_SET(3) TAY_SET(4) TAY_SET(5) TAY_SET(6) TAY_SET(7) TAY_SET(8)
    default:
      if constexpr (sizeof(T) == 4) {
        switch (cw) {
          TAY_SET(9) TAY_SET(10) TAY_SET(11) TAY_SET(12) TAY_SET(13) TAY_SET(14) TAY_SET(15) TAY_SET(16)
          default: break;
        }
      }
  }
#undef TAY_SET
  return cudaErrorInvalidValue;
}

template <typename T>
afqmc_status do_propagate(afqmc_ctx* c, void* phi, const void* x, const void* fb, void* ovlp, double* weight, void* theta,
                          const void* eloc_pre, int32_t* flags) {
  {
    StageScope sc(c, AFQMC_STAGE_SHIFT);
    LAUNCH(c, k_shift<T>, c->nw, 128, 0, c->ng, c->NGP, c->p.dt, (const cplx<T>*)fb, (const T*)x, (T*)c->Z, (T*)c->Z_lo,
           c->split, c->cshift);
  }
  afqmc_status st;
  {
    StageScope sc(c, AFQMC_STAGE_ASSEMBLE);
    bool done = false;
    if constexpr (sizeof(T) == 4) {
      if (c->path == 2) {
        if (c->M % 4 == 0) {   // staged epilogue writes both triangles: no symmetrize pass
          tc::EpiAssembleSym e3;
          e3.out = (float*)c->Abuf; e3.out_lo = nullptr;   // A_w is stored once, in FP32: the Taylor kernel splits it on the fly
          e3.blk = c->blk; e3.M = c->M;
          e3.MP = c->MP; e3.n_real = 2 * c->nw;
          // A_w beyond the L2 (126 MB) is streamed: its lines are asked to leave first, the field planes stay (gemm_tf32.cuh)
          e3.st_pol = ((size_t)c->nw * c->M * 2 * c->MP * 4 > ((size_t)96 << 20) || (AFQMC_PS_POL & 4)) ? tc::L2_EVICT_FIRST : tc::L2_EVICT_NORMAL;
          st = run_gemm_tc(c, c->map_asm, c->nblk * 128, 2 * c->nw, c->NGP, e3);
          done = true;
        }
        tc::EpiAssemble e2;
        e2.out = (float*)c->Abuf; e2.out_lo = nullptr; e2.blk = c->blk; e2.M = c->M; e2.MP = c->MP; e2.m_real = c->nblk * 128; e2.n_real = 2 * c->nw;
        if (!done) st = run_gemm_tc(c, c->map_asm, c->nblk * 128, 2 * c->nw, c->NGP, e2);
        done = true;
      }
    }
    if (!done) {
    EpiAssemble<T> epi;
    epi.out = (T*)c->Abuf; epi.M = c->M; epi.MP = c->MP; epi.m_real = c->M * c->M; epi.n_real = 2 * c->nw;
    st = run_gemm<T>(c, (const T*)c->Lt, c->NGP, c->M * c->M, (const T*)c->Z, c->NGP, 2 * c->nw, c->NGP, epi);
    }
  }
  if constexpr (sizeof(T) == 4) {
    if (!st && c->path == 2 && c->M % 4 != 0) {
      StageScope sc(c, AFQMC_STAGE_SYMMETRIZE);
      const int nt32 = (c->M + 31) / 32;
      dim3 sg(c->nw, nt32 * (nt32 + 1) / 2);   // walkers on grid x (no 65535 cap)
      LAUNCH(c, k_symmetrize<float>, sg, dim3(32, 8), 0, c->M, c->MP, (float*)c->Abuf, (float*)nullptr);
    }
  }
  if (st) return st;
  st = run_taylor<T>(c, phi);
  if (st) return st;
  if (c->ev_phi_armed) {   // the walker is final: afqmc_step_host starts its download under the rest of the step
    c->ev_phi_armed = 0;
    CUDA_OK(c, cudaEventRecord(c->ev_phi, c->stream));
  }
  return run_green<T>(c, phi, ovlp, theta, 1, weight, eloc_pre, flags);
}

template <typename T> afqmc_status do_force_bias(afqmc_ctx* c, const void* phi, const void* theta, void* fb) {
  if (c->md) {
    // the mixed Green's function needs the determinant ratios: rebuild them from the walker itself
    afqmc_status st0 = run_green<T>(c, phi, c->ovlp_scr, c->th_scr, 0, nullptr, nullptr, nullptr);
    if (st0) return st0;
    st0 = run_fb_gemm<T>(c);
    if (st0) return st0;
    LAUNCH(c, k_fb_finish<T>, c->nw, 128, 0, c->ng, c->NGP, c->nw, (const T*)c->fs, (cplx<T>*)fb, (zcplx*)nullptr);
    return AFQMC_OK;
  }
  LAUNCH(c, k_planarize<T>, c->nw, 128, 0, c->M, c->na, c->nb, c->KA, c->KT, c->split, (const cplx<T>*)theta, (T*)c->thp,
         (T*)c->thp_lo);
  afqmc_status st = run_fb_gemm<T>(c);
  if (st) return st;
  LAUNCH(c, k_fb_finish<T>, c->nw, 128, 0, c->ng, c->NGP, c->nw, (const T*)c->fs, (cplx<T>*)fb, (zcplx*)nullptr);
  return AFQMC_OK;
}

// energy of the walkers whose planar Theta is in ctx->thp; runs the force-bias GEMM too (fb may be null)
template <typename T> afqmc_status do_fb_energy_planar(afqmc_ctx* c, const void* theta, void* fb, zcplx* eloc) {
  afqmc_status st = run_fb_gemm<T>(c);
  if (st) return st;
  if (c->md) {
    if (fb) LAUNCH(c, k_fb_finish<T>, c->nw, 128, 0, c->ng, c->NGP, c->nw, (const T*)c->fs, (cplx<T>*)fb, (zcplx*)nullptr);
    return run_md_energy<T>(c, theta, eloc);
  }
  LAUNCH(c, k_fb_finish<T>, c->nw, 128, 0, c->ng, c->NGP, c->nw, (const T*)c->fs, (cplx<T>*)fb, eloc);
  return run_energy_gemm<T>(c, theta, eloc);
}

// E_L from an interleaved Theta handed in by the caller
template <typename T> afqmc_status do_energy_from_theta(afqmc_ctx* c, const void* theta, zcplx* eloc) {
  if (c->md) return run_md_energy<T>(c, theta, eloc);
  LAUNCH(c, k_planarize<T>, c->nw, 128, 0, c->M, c->na, c->nb, c->KA, c->KT, c->split, (const cplx<T>*)theta, (T*)c->thp,
         (T*)c->thp_lo);
  return do_fb_energy_planar<T>(c, theta, nullptr, eloc);
}

template <typename T>
afqmc_status do_step(afqmc_ctx* c, void* phi, double* weight, void* ovlp, void* theta, void* fb, const void* x, int n_steps,
                     void* eloc, int32_t* flags) {
  zcplx* el = (zcplx*)eloc;
  const zcplx* epre = nullptr;
  if (c->p.weight_mode == 1) {
    // E_L of the walkers on entry
    afqmc_status st = do_energy_from_theta<T>(c, theta, c->eloc_scratch);
    if (st) return st;
    epre = c->eloc_scratch;
  }
  for (int s = 0; s < n_steps; ++s) {
    const T* xs = (const T*)x + (size_t)s * c->nw * c->ng;
    afqmc_status st = do_propagate<T>(c, phi, xs, fb, ovlp, weight, theta, epre, flags);
    if (st) return st;
    st = do_fb_energy_planar<T>(c, theta, fb, el + (size_t)s * c->nw);
    if (st) return st;
    epre = el + (size_t)s * c->nw;
  }
  return AFQMC_OK;
}

template <typename T> afqmc_status do_ortho(afqmc_ctx* c, void* phi, void* ovlp, int32_t* flags) {
  if (c->ortho_smem > 227 * 1024) return fail(c, AFQMC_EUNSUPPORTED, "%s", "afqmc_orthonormalize: walker exceeds one CTA's shared memory in FP64");
  StageScope sc(c, AFQMC_STAGE_ORTHO);
  LAUNCH(c, k_ortho<T>, c->nw, ortho_threads(c->na, c->nb), c->ortho_smem, c->M, c->na, c->nb, (cplx<T>*)phi, (zcplx*)ovlp, flags);
  return AFQMC_OK;
}

template <typename T>
afqmc_status do_popctl(afqmc_ctx* c, void* phi, double* weight, void* ovlp, void* theta, void* fb, double u, int32_t* parent) {
  StageScope sc(c, AFQMC_STAGE_POPCTL);
  LAUNCH(c, k_comb_parents, 1, 1024, 0, c->nw, (const double*)weight, u, c->pc_cum, c->pc_parent, c->pc_wnew);
  CombMove m;
  m.phi = (uint2*)phi; m.theta = (uint2*)theta; m.fb = (uint2*)fb; m.ovlp = (zcplx*)ovlp;
  m.s_phi = (uint2*)c->pc_phi; m.s_theta = (uint2*)c->pc_theta; m.s_fb = (uint2*)c->pc_fb; m.s_ovlp = c->pc_ovlp;
  m.words_phi = c->M * c->nt * 2 * c->ts / 8; m.words_fb = c->ng * 2 * c->ts / 8;
  LAUNCH(c, k_comb_pack, c->nw, 256, 0, m, (const int32_t*)c->pc_parent);
  LAUNCH(c, k_comb_unpack, c->nw, 256, 0, m, (const int32_t*)c->pc_parent, weight, (const double*)c->pc_wnew);
  if (parent) CUDA_OK(c, cudaMemcpyAsync(parent, c->pc_parent, (size_t)c->nw * 4, cudaMemcpyDeviceToDevice, c->stream));
  return AFQMC_OK;
}

// The paper's schedule around the walker step; hybrid weights only.
template <typename T>
afqmc_status do_run(afqmc_ctx* c, void* phi, double* weight, void* ovlp, void* theta, void* fb, const void* x, int n_steps,
                    int energy_every, int ortho_every, int pc_every, const double* u, void* eloc, double* w_meas,
                    int32_t* parents, int32_t* flags) {
  zcplx* el = (zcplx*)eloc;
  int n_meas = 0, n_pc = 0;
  for (int s = 1; s <= n_steps; ++s) {
    const T* xs = (const T*)x + (size_t)(s - 1) * c->nw * c->ng;
    afqmc_status st = do_propagate<T>(c, phi, xs, fb, ovlp, weight, theta, nullptr, flags);
    if (st) return st;
    if (energy_every && s % energy_every == 0) {
      st = do_fb_energy_planar<T>(c, theta, fb, el + (size_t)n_meas * c->nw);
      if (st) return st;
      if (w_meas) CUDA_OK(c, cudaMemcpyAsync(w_meas + (size_t)n_meas * c->nw, weight, (size_t)c->nw * 8, cudaMemcpyDeviceToDevice, c->stream));
      ++n_meas;
    } else {   // propagate-only step: the force bias of the new walker, no energy contraction
      st = run_fb_gemm<T>(c);
      if (st) return st;
      LAUNCH(c, k_fb_finish<T>, c->nw, 128, 0, c->ng, c->NGP, c->nw, (const T*)c->fs, (cplx<T>*)fb, (zcplx*)nullptr);
    }
    if (ortho_every && s % ortho_every == 0) {
      st = do_ortho<T>(c, phi, ovlp, flags);
      if (st) return st;
    }
    if (pc_every && s % pc_every == 0) {
      st = do_popctl<T>(c, phi, weight, ovlp, theta, fb, u[n_pc], parents ? parents + (size_t)n_pc * c->nw : nullptr);
      if (st) return st;
      ++n_pc;
    }
  }
  return AFQMC_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

afqmc_status afqmc_query_bytes(const afqmc_params* p, size_t* const_bytes, size_t* work_bytes) {
  afqmc_status s = check_params(p, g_init_err);
  if (s) return s;
  if (!const_bytes || !work_bytes) { snprintf(g_init_err, 256, "null output pointer"); return AFQMC_EINVAL; }
  afqmc_ctx tmp;
  memset(&tmp, 0, sizeof(tmp));
  tmp.p = *p;
  tmp.split = resolve_path(p) == 2;
  carve(p, &tmp, nullptr, nullptr, const_bytes, work_bytes);
  return AFQMC_OK;
}

afqmc_status afqmc_init(afqmc_ctx** out, const afqmc_params* p, const double* h1, const double* L_chol,
                        const double* psiT_a, const double* psiT_b, const double* C_act, const double* det_coeff,
                        const int32_t* det_exc, void* const_mem, void* work_mem, void* stream) {
  if (!out) { snprintf(g_init_err, 256, "out is NULL"); return AFQMC_EINVAL; }
  *out = nullptr;
  afqmc_status s = check_params(p, g_init_err);
  if (s) return s;
  const bool md = p->n_det > 1;
  if (!h1 || !L_chol || !const_mem || !work_mem || (!md && (!psiT_a || (p->n_beta && !psiT_b))) ||
      (md && (!C_act || !det_coeff || !det_exc))) {
    snprintf(g_init_err, 256, "null input pointer");
    return AFQMC_EINVAL;
  }
  // multi-det: reference orbitals = first n_sigma columns of C_act; excitation list normalised to 2 slots
  std::vector<double> pa_md, pb_md;
  const int emax = p->max_exc > 2 ? 4 : 2;
  std::vector<int32_t> exc2((size_t)p->n_det * 4 * emax, -1);
  if (md) {
    const int nact = p->n_act;
    pa_md.resize((size_t)p->M * p->n_alpha); pb_md.resize((size_t)p->M * p->n_beta);
    for (int k = 0; k < p->M; ++k) {
      for (int a = 0; a < p->n_alpha; ++a) pa_md[(size_t)k * p->n_alpha + a] = C_act[(size_t)k * nact + a];
      for (int a = 0; a < p->n_beta; ++a) pb_md[(size_t)k * p->n_beta + a] = C_act[(size_t)k * nact + a];
    }
    psiT_a = pa_md.data(); psiT_b = pb_md.data();
    for (int i = 0; i < p->n_det; ++i)
      for (int sp = 0; sp < 2; ++sp) {
        const int n = sp ? p->n_beta : p->n_alpha;
        int cnt = 0, hs[4] = {-1, -1, -1, -1}, ps[4] = {-1, -1, -1, -1};
        for (int e = 0; e < p->max_exc; ++e) {
          const int32_t* ex = det_exc + (((size_t)i * 2 + sp) * p->max_exc + e) * 2;
          if (ex[0] < 0) continue;
          bool dup = false;
          for (int q = 0; q < cnt; ++q) dup |= ex[0] == hs[q] || ex[1] == ps[q];
          if (ex[0] >= n || ex[1] < n || ex[1] >= nact || dup) {
            snprintf(g_init_err, 256, "det_exc: need hole < n_sigma <= particle < n_act, distinct within a determinant");
            return AFQMC_EINVAL;
          }
          hs[cnt] = ex[0]; ps[cnt] = ex[1]; ++cnt;
        }
        for (int e = 0; e < cnt; ++e) {
          exc2[((size_t)i * 2 + sp) * 2 * emax + 2 * e] = hs[e];
          exc2[((size_t)i * 2 + sp) * 2 * emax + 2 * e + 1] = ps[e];
        }
      }
  }
  if (((uintptr_t)const_mem & 255) || ((uintptr_t)work_mem & 255)) {
    snprintf(g_init_err, 256, "const_mem / work_mem must be 256-byte aligned");
    return AFQMC_EINVAL;
  }
  // h and every L_g must be symmetric: the kernels rely on it
  const int M = p->M;
  double amax = 0.0;
  for (size_t e = 0; e < (size_t)M * M; ++e) amax = fmax(amax, fabs(h1[e]));
  for (int i = 0; i < M; ++i)
    for (int j = 0; j < i; ++j)
      if (fabs(h1[(size_t)i * M + j] - h1[(size_t)j * M + i]) > 1e-10 * (amax + 1e-300)) {
        snprintf(g_init_err, 256, "h1 is not symmetric");
        return AFQMC_EINVAL;
      }
  for (int g = 0; g < p->n_chol; ++g) {
    const double* Lg = L_chol + (size_t)g * M * M;
    double lm = 0.0;
    for (size_t e = 0; e < (size_t)M * M; ++e) lm = fmax(lm, fabs(Lg[e]));
    if (!isfinite(lm)) { snprintf(g_init_err, 256, "L_chol contains non-finite values"); return AFQMC_EINVAL; }
    for (int i = 0; i < M; ++i)
      for (int j = 0; j < i; ++j)
        if (fabs(Lg[(size_t)i * M + j] - Lg[(size_t)j * M + i]) > 1e-10 * (lm + 1e-300)) {
          snprintf(g_init_err, 256, "L_chol[g] is not symmetric");
          return AFQMC_EINVAL;
        }
  }
  afqmc_ctx* c = new (std::nothrow) afqmc_ctx;
  if (!c) { snprintf(g_init_err, 256, "host allocation failed"); return AFQMC_ENOMEM; }
  memset(c, 0, sizeof(*c));
  c->p = *p;
  c->stream = (cudaStream_t)stream;
  c->path = resolve_path(p);
  c->split = c->path == 2;
  c->cta2 = resolve_cta2(p);
  c->emax = emax;
  {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
  }
  size_t cb, wb;
  carve(p, c, (char*)const_mem, (char*)work_mem, &cb, &wb);
  c->tay_tc = will_tay_tc(p) && c->nw > 0;
  c->green_smem = p->precision ? green_smem_bytes<double>(c->M, c->na, c->nb) : green_smem_bytes<float>(c->M, c->na, c->nb);
  if (!will_tay_tc(p)) {
    if (p->precision) {
      taylor_pick<double>(c->M, c->nt, c->tay_cw, c->tay_nch);
      c->tay_smem = taylor_smem_bytes<double>(c->M, c->MP, c->tay_nch, (c->tay_cw + 3) & ~3);
    } else {
      taylor_pick<float>(c->M, c->nt, c->tay_cw, c->tay_nch);
      c->tay_smem = taylor_smem_bytes<float>(c->M, c->MP, c->tay_nch, (c->tay_cw + 3) & ~3);
    }
    c->tay_threads = (int)rup((size_t)c->M * c->tay_nch, 32);
    if (c->tay_smem > 227 * 1024) {
      s = fail(nullptr, AFQMC_EUNSUPPORTED, "Taylor kernel tile exceeds shared memory");
      delete c;
      return s;
    }
    if (c->tay_smem > 48 * 1024) {
      cudaError_t e = p->precision ? set_taylor_smem<double>(c->tay_cw, c->tay_smem) : set_taylor_smem<float>(c->tay_cw, c->tay_smem);
      if (e != cudaSuccess) { snprintf(g_init_err, 256, "CUDA: %s", cudaGetErrorString(e)); delete c; return AFQMC_ECUDA; }
    }
  }
  if (c->md) {
    c->mdo_smem = md_overlap_smem(c->M, c->na, c->nb, c->nact, c->ndet, c->ts, c->emax);
    c->mde_smem = md_energy_smem(c->M, c->na, c->nb, c->nact, c->ndet, c->ts, c->emax);
    cudaError_t e1, e2;
    if (p->precision) {
      e1 = cudaFuncSetAttribute(k_md_overlap<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->mdo_smem);
      e2 = cudaSuccess;
    } else {
      e1 = cudaFuncSetAttribute(k_md_overlap<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->mdo_smem);
      e2 = cudaSuccess;
    }
    if (e1 != cudaSuccess || e2 != cudaSuccess) { snprintf(g_init_err, 256, "CUDA: cannot size multi-det shared memory"); delete c; return AFQMC_ECUDA; }
  }
  if (c->green_smem > 48 * 1024) {
    cudaError_t e = p->precision ? cudaFuncSetAttribute(k_green<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->green_smem)
                                 : cudaFuncSetAttribute(k_green<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->green_smem);
    if (e != cudaSuccess) { snprintf(g_init_err, 256, "CUDA: %s", cudaGetErrorString(e)); delete c; return AFQMC_ECUDA; }
  }
  c->ortho_smem = ortho_smem_bytes(c->M, c->nt);
  if (c->ortho_smem > 48 * 1024 && c->ortho_smem <= 227 * 1024) {
    cudaError_t e = p->precision ? cudaFuncSetAttribute(k_ortho<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ortho_smem)
                                 : cudaFuncSetAttribute(k_ortho<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->ortho_smem);
    // ask for the full shared-memory carve-out: with the default split only one 80 KB CTA fits an SM (ncu, round 1)
    if (e == cudaSuccess)
      e = p->precision ? cudaFuncSetAttribute(k_ortho<double>, cudaFuncAttributePreferredSharedMemoryCarveout, 100)
                       : cudaFuncSetAttribute(k_ortho<float>, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
    if (e != cudaSuccess) { snprintf(g_init_err, 256, "CUDA: %s", cudaGetErrorString(e)); delete c; return AFQMC_ECUDA; }
  }
  // tensor-pipe Taylor kernel for 96 <= M <= 256: below that a 128-row tile is mostly padding and the FP32 SIMT
  // kernel is both competitive and free of the tensor pipe's truncation bias
  if (c->tay_tc) {
    tt::TaylorTcArgs& a = c->tay_args;
    a.M = c->M; a.MP = c->MP; a.nt = c->nt; a.K = p->taylor_order; a.nw = c->nw;
    a.mtiles = (c->M + 127) / 128;
    a.rows_last = (int)rup((size_t)(c->M - 128 * (a.mtiles - 1)), 8);
    a.nkb = (c->M + 31) / 32;
    a.phi = nullptr;
    c->tay_tc_smem = tt::smem_bytes(a.nkb);
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
    bool ok = true;
    a.nf = tt::pick_nf(a.nkb);
    ok &= a.nf >= 3;
    for (int v = 0; v < 2; ++v) {
      const uint32_t rows = v ? (uint32_t)a.rows_last : 128u;
      ok &= tc::make_map(&c->map_tay.A[v], c->Abuf, 2 * (uint64_t)c->MP, (uint64_t)c->nw * c->M, 2 * (uint64_t)c->MP, rows);
      ok &= tc::make_map(&c->map_tay.E[v], c->Eh, (uint64_t)c->MP, (uint64_t)c->M, (uint64_t)c->MP, rows);
    }

    cudaError_t e0 = cudaFuncSetAttribute(tt::k_taylor_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->tay_tc_smem);
    if (!ok || e0 != cudaSuccess || c->n_sm <= 0) {
      snprintf(g_init_err, 256, "tensor-pipe Taylor kernel: tensor-map / shared-memory set-up failed");
      delete c;
      return AFQMC_ECUDA;
    }
  }
  if (c->path == 2 && c->nw > 0) {
    using namespace tc;
    bool ok = true;
    const uint64_t nrow = 2 * (uint64_t)c->nw;
    ok &= make_map(&c->map_asm.a_hi, c->Lt, c->NGP, (uint64_t)c->nblk * 128, c->NGP, BM);
    ok &= make_map(&c->map_asm.a_lo, c->Lt_lo, c->NGP, (uint64_t)c->nblk * 128, c->NGP, BM);
    ok &= make_map(&c->map_asm.b_hi, c->Z, c->NGP, nrow, c->NGP, B_BOX);
    ok &= make_map(&c->map_asm.b_lo, c->Z_lo, c->NGP, nrow, c->NGP, B_BOX);
    for (int sp = 0; sp < 2; ++sp) {
      const int n = sp ? c->cb : c->ca, soff = sp ? c->KA : 0, Ks = sp ? c->KB : c->KA;
      if (!n) continue;
      const float* R = (const float*)c->Rall + soff; const float* Rl = (const float*)c->Rall_lo + soff;
      const float* th = (const float*)c->thp + soff; const float* thl = (const float*)c->thp_lo + soff;
      ok &= make_map(&c->map_fb[sp].a_hi, R, Ks, c->ng, c->KT, BM);
      ok &= make_map(&c->map_fb[sp].a_lo, Rl, Ks, c->ng, c->KT, BM);
      ok &= make_map(&c->map_fb[sp].b_hi, th, Ks, nrow, c->KT, B_BOX);
      ok &= make_map(&c->map_fb[sp].b_lo, thl, Ks, nrow, c->KT, B_BOX);
      if (c->md) {           // the multi-determinant energy does not use Y; its TT GEMM has its own operands
        if (sp == 0) {
          const uint64_t r1 = (uint64_t)(c->ng + 1) * c->nact, r2 = (uint64_t)c->nw * 2 * c->nt;
          ok &= make_map(&c->map_tt.a_hi, c->RactT, c->MPK, r1, c->MPK, BM);
          ok &= make_map(&c->map_tt.a_lo, c->RactT_lo, c->MPK, r1, c->MPK, BM);
          ok &= make_map(&c->map_tt.b_hi, c->thT, c->MPK, r2, c->MPK, B_BOX);
          ok &= make_map(&c->map_tt.b_lo, c->thT_lo, c->MPK, r2, c->MPK, B_BOX);
        }
        continue;
      }
      ok &= make_map(&c->map_en[sp].a_hi, c->Y[sp], Ks, (uint64_t)c->M * n, Ks, BM);
      ok &= make_map(&c->map_en[sp].a_lo, c->Y_lo[sp], Ks, (uint64_t)c->M * n, Ks, BM);
      c->map_en[sp].b_hi = c->map_fb[sp].b_hi;
      c->map_en[sp].b_lo = c->map_fb[sp].b_lo;
    }
    cudaError_t e1 = cudaFuncSetAttribute(k_gemm_tf32<tc::EpiStoreT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    cudaError_t e2 = cudaFuncSetAttribute(k_gemm_tf32<tc::EpiAssemble>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    cudaError_t e3 = cudaFuncSetAttribute(k_gemm_tf32<tc::EpiEnergy>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32<tc::EpiTT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32<tc::EpiAssembleSym>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32_pair<tc::EpiStoreT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32_pair<tc::EpiAssemble>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32_pair<tc::EpiEnergy>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32_pair<tc::EpiTT>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (e3 == cudaSuccess) e3 = cudaFuncSetAttribute(k_gemm_tf32_pair<tc::EpiAssembleSym>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    c->ps_ok = cudaFuncSetAttribute(k_gemm_tf32_pair_ps<tc::EpiAssembleSym>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_PS_BYTES) == cudaSuccess;
    c->en_ok = c->cta2 && !c->md &&
               cudaFuncSetAttribute(k_gemm_tf32_pair_ps<tc::EpiEnergy, EN_CHUNK, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_PS_BYTES) == cudaSuccess;
    c->fb_ok = c->cta2 &&
               cudaFuncSetAttribute(k_gemm_tf32_pair_ps<tc::EpiStoreT, EN_CHUNK, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_PS_BYTES) == cudaSuccess;
    (void)cudaGetLastError();
    if (!ok || e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) {
      snprintf(g_init_err, 256, "tcgen05 path: tensor-map / shared-memory set-up failed");
      delete c;
      return AFQMC_ECUDA;
    }
  }
  s = p->precision ? init_device<double>(c, h1, L_chol, psiT_a, psiT_b, C_act, det_coeff, exc2.data())
                   : init_device<float>(c, h1, L_chol, psiT_a, psiT_b, C_act, det_coeff, exc2.data());
  if (s) {
    memcpy(g_init_err, c->err, 256);
    delete c;
    return s;
  }
  // after init_device: it clears the constant region the lists live in
  auto upload_sched = [&](int* dst, const std::vector<int>& v) {
    return cudaMemcpyAsync(dst, v.data(), v.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream) == cudaSuccess &&
           cudaStreamSynchronize(c->stream) == cudaSuccess;
  };
  if (c->en_ok) {
    std::vector<int> sched;
    const int rows[2] = {c->M * c->na, c->M * c->nb}, Ks[2] = {c->KA, c->nb ? c->KB : 0};
    c->en_ok = build_pair_schedule(c, 1, rows, Ks, 6, sched, c->en_stride) && upload_sched(c->en_sched, sched);
  }
  if (c->fb_ok) {
    std::vector<int> sched;
    const int rows[2] = {c->ca ? c->ng : 0, c->cb ? c->ng : 0}, Ks[2] = {c->KA, c->cb ? c->KB : 0};
    c->fb_ok = build_pair_schedule(c, 0, rows, Ks, 3, sched, c->fb_stride) && upload_sched(c->fb_sched, sched);
  }
  c->launches = 0;
  *out = c;
  return AFQMC_OK;
}

void afqmc_destroy(afqmc_ctx* ctx) {
  if (!ctx) return;
  afqmc_profile_enable(ctx, 0);
  if (ctx->copy_ready) {
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(ctx->ev_x[i]); cudaEventDestroy(ctx->ev_done[i]); cudaEventDestroy(ctx->ev_e[i]); }
    cudaEventDestroy(ctx->ev_phi);
    cudaStreamDestroy(ctx->copy_stream);
  }
  delete ctx;
}

afqmc_status afqmc_profile_enable(afqmc_ctx* c, int32_t enable) {
  if (!c) return AFQMC_EINVAL;
  if (c->prof) {
    for (int s = 0; s < AFQMC_N_STAGES; ++s)
      for (int i = 0; i < 64; ++i) { cudaEventDestroy(c->pev[s][i][0]); cudaEventDestroy(c->pev[s][i][1]); }
    c->prof = 0;
  }
  memset(c->pcount, 0, sizeof(c->pcount));
  if (enable) {
    for (int s = 0; s < AFQMC_N_STAGES; ++s)
      for (int i = 0; i < 64; ++i) {
        CUDA_OK(c, cudaEventCreate(&c->pev[s][i][0]));
        CUDA_OK(c, cudaEventCreate(&c->pev[s][i][1]));
      }
    c->prof = 1;
  }
  return AFQMC_OK;
}

afqmc_status afqmc_profile_read(afqmc_ctx* c, int32_t stage, double* total_ms, int32_t* launches) {
  if (!c || stage < 0 || stage >= AFQMC_N_STAGES || !total_ms || !launches) return AFQMC_EINVAL;
  double tot = 0.0;
  int n = c->prof ? c->pcount[stage] : 0;
  for (int i = 0; i < n; ++i) {
    float ms = 0.f;
    CUDA_OK(c, cudaEventElapsedTime(&ms, c->pev[stage][i][0], c->pev[stage][i][1]));
    tot += ms;
  }
  *total_ms = tot;
  *launches = n;
  return AFQMC_OK;
}

const char* afqmc_last_error(const afqmc_ctx* ctx) { return ctx ? ctx->err : g_init_err; }

afqmc_status afqmc_set_stream(afqmc_ctx* c, void* stream) {
  if (!c) return AFQMC_EINVAL;
  c->stream = (cudaStream_t)stream;
  return AFQMC_OK;
}

int64_t afqmc_launch_count(const afqmc_ctx* ctx) { return ctx ? ctx->launches : 0; }
int32_t afqmc_gemm_path(const afqmc_ctx* ctx) { return ctx ? (ctx->cta2 ? 3 : ctx->path) : 0; }

#define NEED(c, cond, msg) \
  do { if (!(cond)) return fail((c), AFQMC_EINVAL, "%s", msg); } while (0)
#define DISPATCH(c, fn, ...) ((c)->p.precision ? fn<double>(__VA_ARGS__) : fn<float>(__VA_ARGS__))

afqmc_status afqmc_overlap_green(afqmc_ctx* c, const void* phi, void* ovlp, void* theta, void* G_or_null, int32_t* flags) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, phi && ovlp && theta, "afqmc_overlap_green: null pointer");
  if (c->nw == 0) return AFQMC_OK;
  afqmc_status s = DISPATCH(c, run_green, c, phi, ovlp, theta, 0, nullptr, nullptr, flags);
  if (s) return s;
  if (G_or_null) {
    dim3 grid(c->nw, (c->M * c->M + 255) / 256 < 65535 ? (c->M * c->M + 255) / 256 : 65535, 2);   // walkers on grid x (no 65535 cap)
    if (c->md) {   // mixed G_s^T = Thtil_s C_act^T
      if (c->p.precision)
        LAUNCH(c, k_gfull<double>, grid, 256, 0, c->M, c->nact, c->nact, (const cplx<double>*)c->thtil,
               (const double*)c->Cact, (const double*)c->Cact, (cplx<double>*)G_or_null);
      else
        LAUNCH(c, k_gfull<float>, grid, 256, 0, c->M, c->nact, c->nact, (const cplx<float>*)c->thtil,
               (const float*)c->Cact, (const float*)c->Cact, (cplx<float>*)G_or_null);
    } else if (c->p.precision)
      LAUNCH(c, k_gfull<double>, grid, 256, 0, c->M, c->na, c->nb, (const cplx<double>*)theta, (const double*)c->psi_a,
             (const double*)c->psi_b, (cplx<double>*)G_or_null);
    else
      LAUNCH(c, k_gfull<float>, grid, 256, 0, c->M, c->na, c->nb, (const cplx<float>*)theta, (const float*)c->psi_a,
             (const float*)c->psi_b, (cplx<float>*)G_or_null);
  }
  return AFQMC_OK;
}

afqmc_status afqmc_force_bias(afqmc_ctx* c, const void* phi, const void* theta, void* fb) {
  (void)phi;
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, theta && fb, "afqmc_force_bias: null pointer");
  if (c->nw == 0) return AFQMC_OK;
  NEED(c, !c->md || phi, "afqmc_force_bias: multi-determinant trial needs phi");
  return DISPATCH(c, do_force_bias, c, phi, theta, fb);
}

afqmc_status afqmc_propagate(afqmc_ctx* c, void* phi, const void* x, const void* fb, void* ovlp, double* weight, void* theta,
                             const void* eloc_pre, int32_t* flags) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, phi && x && fb && ovlp && weight && theta, "afqmc_propagate: null pointer");
  NEED(c, c->p.weight_mode == 0 || eloc_pre, "afqmc_propagate: weight_mode 1 needs eloc_pre");
  if (c->nw == 0) return AFQMC_OK;
  return DISPATCH(c, do_propagate, c, phi, x, fb, ovlp, weight, theta, eloc_pre, flags);
}

afqmc_status afqmc_local_energy(afqmc_ctx* c, const void* phi, const void* theta, void* eloc) {
  (void)phi;
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, theta && eloc, "afqmc_local_energy: null pointer");
  if (c->nw == 0) return AFQMC_OK;
  return DISPATCH(c, do_energy_from_theta, c, theta, (zcplx*)eloc);
}

afqmc_status afqmc_step(afqmc_ctx* c, void* phi, double* weight, void* ovlp, void* theta, void* fb, const void* x,
                        int32_t n_steps, void* eloc, int32_t* flags) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, n_steps >= 0, "afqmc_step: n_steps < 0");
  if (c->nw == 0 || n_steps == 0) return AFQMC_OK;
  NEED(c, phi && weight && ovlp && theta && fb && x && eloc, "afqmc_step: null pointer");
  return DISPATCH(c, do_step, c, phi, weight, ovlp, theta, fb, x, n_steps, eloc, flags);
}

afqmc_status afqmc_orthonormalize(afqmc_ctx* c, void* phi, void* ovlp, int32_t* flags) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  if (c->nw == 0) return AFQMC_OK;
  NEED(c, phi && ovlp, "afqmc_orthonormalize: null pointer");
  return DISPATCH(c, do_ortho, c, phi, ovlp, flags);
}

afqmc_status afqmc_population_control(afqmc_ctx* c, void* phi, double* weight, void* ovlp, void* theta, void* fb, double u,
                                      int32_t* parent) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, u >= 0.0 && u < 1.0, "afqmc_population_control: u must be in [0, 1)");
  if (c->nw == 0) return AFQMC_OK;
  NEED(c, phi && weight && ovlp && theta && fb, "afqmc_population_control: null pointer");
  return DISPATCH(c, do_popctl, c, phi, weight, ovlp, theta, fb, u, parent);
}

size_t afqmc_comb_record_bytes(const afqmc_ctx* c) {
  if (!c) return 0;
  return (size_t)(2 * (c->M * c->nt * 2 * c->ts / 8) + c->ng * 2 * c->ts / 8 + 2) * 8;
}

static CombRecord comb_record(const afqmc_ctx* c, void* phi, void* ovlp, void* theta, void* fb) {
  CombRecord m;
  m.phi = (uint2*)phi; m.theta = (uint2*)theta; m.fb = (uint2*)fb; m.ovlp = (zcplx*)ovlp;
  m.words_phi = c->M * c->nt * 2 * c->ts / 8; m.words_fb = c->ng * 2 * c->ts / 8;
  m.words_rec = 2 * m.words_phi + m.words_fb + 2;
  return m;
}

afqmc_status afqmc_comb_map(afqmc_ctx* c, const double* weight_all, int64_t n_total, double u, double* cum_scratch,
                            int32_t* parent_all, double* w_new) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, n_total >= 0 && n_total < (int64_t)1 << 31, "afqmc_comb_map: n_total out of range");
  NEED(c, u >= 0.0 && u < 1.0, "afqmc_comb_map: u must be in [0, 1)");
  if (n_total == 0) return AFQMC_OK;
  NEED(c, weight_all && cum_scratch && parent_all && w_new, "afqmc_comb_map: null pointer");
  StageScope sc(c, AFQMC_STAGE_POPCTL);
  LAUNCH(c, k_comb_parents, 1, 1024, 0, (int)n_total, weight_all, u, cum_scratch, parent_all, w_new);
  return AFQMC_OK;
}

// ---- allocation-free variant of afqmc_comb_map: the running-sum scratch lives in a file-scope device array ----------------
// Every GPU that loads the library holds AFQMC_NOALLOC_MAX_WALKERS doubles (512 KiB) until exit.  In host code the array's name is
// a host-side stand-in, not a device address: the address is taken once per device with cudaGetSymbolAddress (that device
// current) and that pointer is what the kernel receives.
static __device__ __align__(256) double g_noalloc_cum[AFQMC_NOALLOC_MAX_WALKERS];
static double* g_noalloc_cum_ptr[64];    // per device ordinal; null until the first call on that device

afqmc_status afqmc_comb_map_noalloc(afqmc_ctx* c, const double* weight_all, int64_t n_total, double u, int32_t* parent_all,
                                    double* w_new) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, n_total >= 0, "afqmc_comb_map_noalloc: n_total < 0");
  if (n_total > (int64_t)AFQMC_NOALLOC_MAX_WALKERS)
    return fail(c, AFQMC_EUNSUPPORTED, "%s", "afqmc_comb_map_noalloc: n_total exceeds AFQMC_NOALLOC_MAX_WALKERS (65536), the size of the "
                                             "library's static scratch; use afqmc_comb_map with caller-provided scratch");
  NEED(c, u >= 0.0 && u < 1.0, "afqmc_comb_map_noalloc: u must be in [0, 1)");
  if (n_total == 0) return AFQMC_OK;
  NEED(c, weight_all && parent_all && w_new, "afqmc_comb_map_noalloc: null pointer");
  int dev = -1;
  CUDA_OK(c, cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(c, AFQMC_EUNSUPPORTED, "%s", "afqmc_comb_map_noalloc: device ordinal >= 64");
  if (!g_noalloc_cum_ptr[dev]) {           // set-up, once per device, with that device current
    double* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_cum);
    if (e != cudaSuccess || !ptr) return fail(c, AFQMC_ECUDA, "cudaGetSymbolAddress(g_noalloc_cum): %s", cudaGetErrorString(e));
    g_noalloc_cum_ptr[dev] = ptr;
  }
  // k_comb_parents writes cum[0 .. n_total) before it reads any of it: nothing of the previous call's contents is used
  StageScope sc(c, AFQMC_STAGE_POPCTL);
  LAUNCH(c, k_comb_parents, 1, 1024, 0, (int)n_total, weight_all, u, g_noalloc_cum_ptr[dev], parent_all, w_new);
  return AFQMC_OK;
}

afqmc_status afqmc_comb_pack(afqmc_ctx* c, const void* phi, const void* ovlp, const void* theta, const void* fb,
                             const int32_t* parent_all, int64_t slot_lo, int64_t count, int64_t first_local, void* sendbuf) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, count >= 0 && slot_lo >= 0 && first_local >= 0, "afqmc_comb_pack: negative index");
  if (count == 0 || c->nw == 0) return AFQMC_OK;
  NEED(c, phi && ovlp && theta && fb && parent_all && sendbuf, "afqmc_comb_pack: null pointer");
  StageScope sc(c, AFQMC_STAGE_POPCTL);
  CombRecord m = comb_record(c, (void*)phi, (void*)ovlp, (void*)theta, (void*)fb);
  LAUNCH(c, k_comb_pack_send, (unsigned)count, 256, 0, m, parent_all, (long long)slot_lo, (long long)first_local, (uint2*)sendbuf);
  return AFQMC_OK;
}

afqmc_status afqmc_comb_unpack(afqmc_ctx* c, const void* recvbuf, void* phi, double* weight, void* ovlp, void* theta, void* fb,
                               const double* w_new) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  if (c->nw == 0) return AFQMC_OK;
  NEED(c, recvbuf && phi && weight && ovlp && theta && fb && w_new, "afqmc_comb_unpack: null pointer");
  StageScope sc(c, AFQMC_STAGE_POPCTL);
  CombRecord m = comb_record(c, phi, ovlp, theta, fb);
  LAUNCH(c, k_comb_unpack_recv, c->nw, 256, 0, m, (const uint2*)recvbuf, weight, w_new);
  return AFQMC_OK;
}

afqmc_status afqmc_mixed_sums(afqmc_ctx* c, const double* weight, const void* eloc, double* out3) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, out3 && (c->nw == 0 || (weight && eloc)), "afqmc_mixed_sums: null pointer");
  LAUNCH(c, k_mixed_sums, 1, 1024, 0, c->nw, weight, (const zcplx*)eloc, out3);
  return AFQMC_OK;
}

afqmc_status afqmc_mixed_energy(afqmc_ctx* c, const double* sums, int32_t n, void* e_mix) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, n >= 0, "afqmc_mixed_energy: n < 0");
  if (n == 0) return AFQMC_OK;
  NEED(c, sums && e_mix, "afqmc_mixed_energy: null pointer");
  LAUNCH(c, k_mixed_ratio, (n + 127) / 128, 128, 0, n, sums, (zcplx*)e_mix);
  return AFQMC_OK;
}

// table-driven MMA ordering experiment (peaks.cuh): tab = {n, a[64], b[64], nn[64], d[64]} int32 HOST; clk = clocks per MMA
afqmc_status afqmc_peak_mma_table(const int32_t* tab, int32_t iters, void* scratch, void* stream, double* clk) {
  if (!tab || !scratch || !clk || tab[0] < 1 || tab[0] > 64) return AFQMC_EINVAL;
  pk::MmaTab t;
  memcpy(&t, tab, sizeof(t));
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, n_sm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  const int smem = 221 * 1024;
  cudaFuncSetAttribute(pk::k_peak_tab, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  pk::k_peak_tab<<<n_sm, 64, smem, st>>>(t, iters, (long long*)scratch);
  if (cudaStreamSynchronize(st) != cudaSuccess || cudaGetLastError() != cudaSuccess) return AFQMC_ECUDA;
  long long c0 = 0;
  cudaMemcpy(&c0, scratch, 8, cudaMemcpyDeviceToHost);
  *clk = (double)c0 / ((double)iters * t.n);
  return AFQMC_OK;
}

// ---- peak microbenchmarks (bench.py --peaks; not on the walker step's path) ----
afqmc_status afqmc_peak_probe(int32_t kind, int32_t n, int32_t iters, void* scratch, size_t scratch_bytes, void* stream,
                              double* ms, double* units, double* clk) {
  if (!ms || !units || !clk || iters < 1 || !scratch || scratch_bytes < (size_t)1 << 20) return AFQMC_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, n_sm = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return AFQMC_ECUDA;
  long long* out = (long long*)scratch;
  *clk = 0.0;
  cudaError_t err = cudaSuccess;
  auto finish = [&](double u) -> afqmc_status {
    cudaEventRecord(e1, st);
    err = cudaStreamSynchronize(st);
    float t = 0.f;
    cudaEventElapsedTime(&t, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (err == cudaSuccess) err = cudaGetLastError();
    *ms = t; *units = u;
    return err == cudaSuccess ? AFQMC_OK : AFQMC_ECUDA;
  };
  if (kind >= 0 && kind <= 2) {          // tcgen05.mma.kind::tf32: SS / TS / SS on CTA pairs; units = flops
    if (n < 16 || n > 256 || n % 16) return AFQMC_EINVAL;
    const int grid = kind == 2 ? (n_sm & ~1) : n_sm;
    const int smem = 16384 + 32768 + 1024;
    cudaFuncSetAttribute(pk::k_peak_mma<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaFuncSetAttribute(pk::k_peak_mma<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaFuncSetAttribute(pk::k_peak_mma<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaMemsetAsync(out, 0, 4096, st);
    cudaEventRecord(e0, st);
    if (kind == 0) pk::k_peak_mma<0><<<grid, 128, smem, st>>>(n, iters, out);
    if (kind == 1) pk::k_peak_mma<1><<<grid, 128, smem, st>>>(n, iters, out);
    if (kind == 2) {
      cudaLaunchConfig_t cfg = {};
      cfg.gridDim = dim3(grid); cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = smem; cfg.stream = st;
      cudaLaunchAttribute at[1];
      at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = 2; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
      cfg.attrs = at; cfg.numAttrs = 1;
      err = cudaLaunchKernelEx(&cfg, pk::k_peak_mma<2>, (int)n, (int)iters, out);
    }
    const double mrows = kind == 2 ? 256.0 : 128.0, ctas = kind == 2 ? grid / 2 : grid;
    afqmc_status s = finish(ctas * (double)iters * 4.0 * 2.0 * mrows * n * 8.0);
    if (s == AFQMC_OK) {
      long long c0 = 0;
      cudaMemcpy(&c0, out, 8, cudaMemcpyDeviceToHost);
      *clk = (double)c0 / ((double)iters * 4.0);      // clocks per MMA in CTA 0
    }
    return s;
  }
  if (kind == 6 || kind == 7) {          // the Taylor kernel's MMA pattern alone (6) and with the other warps loading the smem ports (7)
    const int smem = 49152 + 3 * 32768 + 16384 + 1024;
    cudaFuncSetAttribute(pk::k_peak_mma<3>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaFuncSetAttribute(pk::k_peak_mma<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    cudaMemsetAsync(out, 0, 4096, st);
    cudaEventRecord(e0, st);
    if (kind == 6) pk::k_peak_mma<3><<<n_sm, 128, smem, st>>>(n, iters, out);
    else pk::k_peak_mma<4><<<n_sm, 320, smem, st>>>(128, iters, out);
    afqmc_status s = finish((double)n_sm * iters * 4.0 * 2.0 * 128.0 * 192.0 * 8.0);
    if (s == AFQMC_OK) {
      long long c0 = 0;
      cudaMemcpy(&c0, out, 8, cudaMemcpyDeviceToHost);
      *clk = (double)c0 / ((double)iters * 4.0);      // clocks per (N = 128, N = 64) MMA pair
    }
    return s;
  }
  if (kind == 8) {                       // the Taylor kernel's MMA pattern, uniform issue; n = commits per 8 MMAs (0..2), + 10: 10 more warps poll an mbarrier
    const int smem = 16384 + 6 * 16384 + 1024;
    const int nc = n % 10, poll = n >= 10;
#define PT_LAUNCH(NC, PL)                                                                                         \
    {                                                                                                              \
      cudaFuncSetAttribute(pk::k_peak_taylor<NC, PL>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);          \
      cudaMemsetAsync(out, 0, 4096, st);                                                                           \
      cudaEventRecord(e0, st);                                                                                     \
      pk::k_peak_taylor<NC, PL><<<n_sm, PL ? 384 : 64, smem, st>>>(iters, out);                                    \
    }
    if (nc == 0 && !poll) PT_LAUNCH(0, 0) else if (nc == 1 && !poll) PT_LAUNCH(1, 0) else if (nc == 2 && !poll) PT_LAUNCH(2, 0)
    else if (nc == 0) PT_LAUNCH(0, 1) else if (nc == 1) PT_LAUNCH(1, 1) else PT_LAUNCH(2, 1)
#undef PT_LAUNCH
    afqmc_status s = finish((double)n_sm * iters * 4.0 * 2.0 * 128.0 * 192.0 * 8.0);
    if (s == AFQMC_OK) {
      long long c0 = 0;
      cudaMemcpy(&c0, out, 8, cudaMemcpyDeviceToHost);
      *clk = (double)c0 / ((double)iters * 4.0);      // clocks per (N = 128, N = 64) MMA pair
    }
    return s;
  }
  if (kind == 9) {                       // MMA orderings for the Taylor product: n = 10 * pattern + (1: seven T k-blocks cycle, 0: one)
    const int smem = 225 * 1024;
#define PP_LAUNCH(PAT, NB, EX)                                                                                    \
    {                                                                                                              \
      cudaFuncSetAttribute(pk::k_peak_pat<PAT, NB, EX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);        \
      cudaMemsetAsync(out, 0, 4096, st);                                                                           \
      cudaEventRecord(e0, st);                                                                                     \
      pk::k_peak_pat<PAT, NB, EX><<<n_sm, 64, smem, st>>>(iters, out);                                             \
    }
    switch (n) {
      case 0: PP_LAUNCH(0, 1, 0) break; case 1: PP_LAUNCH(0, 7, 0) break;
      case 10: PP_LAUNCH(1, 1, 0) break; case 11: PP_LAUNCH(1, 7, 0) break;
      case 20: PP_LAUNCH(2, 1, 0) break; case 21: PP_LAUNCH(2, 7, 0) break;
      case 101: PP_LAUNCH(0, 7, 1) break; case 102: PP_LAUNCH(0, 7, 2) break; case 103: PP_LAUNCH(0, 7, 3) break;
      case 104: PP_LAUNCH(0, 7, 4) break; case 107: PP_LAUNCH(0, 7, 7) break;
      default: cudaEventDestroy(e0); cudaEventDestroy(e1); return AFQMC_EINVAL;
    }
#undef PP_LAUNCH
    afqmc_status s = finish(0.0);
    if (s == AFQMC_OK) {
      long long c0 = 0;
      cudaMemcpy(&c0, out, 8, cudaMemcpyDeviceToHost);
      *clk = (double)c0 / (double)iters;      // clocks per (k-block, plane)
    }
    return s;
  }
  if (kind == 10) {                      // TS-mode correctness probe: n = N + 1000 * r0; scratch receives D[128][N] floats
    const int N = n % 1000, r0 = n / 1000;
    if (N < 16 || N > 128 || N % 16 || r0 + N > 128) { cudaEventDestroy(e0); cudaEventDestroy(e1); return AFQMC_EINVAL; }
    cudaFuncSetAttribute(pk::k_probe_ts, cudaFuncAttributeMaxDynamicSharedMemorySize, 32768);
    cudaEventRecord(e0, st);
    pk::k_probe_ts<<<1, 128, 32768, st>>>(N, r0, (float*)scratch);
    return finish(0.0);
  }
  if (kind == 3 || kind == 4) {          // FFMA / DFMA; units = flops
    const int grid = n_sm * 4, thr = 512;
    cudaEventRecord(e0, st);
    if (kind == 3) pk::k_peak_fma<float><<<grid, thr, 0, st>>>(iters, 1.0f, (float*)scratch);
    else pk::k_peak_fma<double><<<grid, thr, 0, st>>>(iters, 1.0, (double*)scratch);
    return finish((double)grid * thr * 8.0 * 2.0 * iters);
  }
  if (kind == 5) {                       // L2 -> smem TMA stream; units = bytes; n = MiB of the streamed buffer
    size_t bytes = (size_t)n << 20;
    if (bytes > scratch_bytes) bytes = scratch_bytes;
    const int rows = (int)(bytes / 128) / 128 * 128;
    CUtensorMap map;
    if (rows < 128 || !tc::make_map(&map, scratch, 32, (uint64_t)rows, 32, 128)) return AFQMC_EINVAL;
    const int smem = 4 * 16384 + 1024;
    cudaFuncSetAttribute(pk::k_peak_tma, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    pk::k_peak_tma<<<n_sm, 64, smem, st>>>(map, rows, 64);      // warm the L2
    cudaEventRecord(e0, st);
    pk::k_peak_tma<<<n_sm, 64, smem, st>>>(map, rows, iters);
    return finish((double)n_sm * iters * 16384.0);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  return AFQMC_EINVAL;
}

afqmc_status afqmc_run(afqmc_ctx* c, void* phi, double* weight, void* ovlp, void* theta, void* fb, const void* x,
                       int32_t n_steps, int32_t energy_every, int32_t ortho_every, int32_t pc_every, const double* u,
                       void* eloc, double* w_meas, int32_t* parents, int32_t* flags) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, n_steps >= 0 && energy_every >= 0 && ortho_every >= 0 && pc_every >= 0, "afqmc_run: negative count");
  NEED(c, c->p.weight_mode == 0, "afqmc_run: the schedule needs hybrid weights (weight_mode 0, PAPER.md:97)");
  if (c->nw == 0 || n_steps == 0) return AFQMC_OK;
  NEED(c, phi && weight && ovlp && theta && fb && x, "afqmc_run: null pointer");
  NEED(c, eloc || !energy_every || n_steps < energy_every, "afqmc_run: eloc is NULL");
  if (pc_every && n_steps >= pc_every) {
    NEED(c, u, "afqmc_run: u is NULL");
    for (int i = 0; i < n_steps / pc_every; ++i) NEED(c, u[i] >= 0.0 && u[i] < 1.0, "afqmc_run: u must be in [0, 1)");
  }
  return DISPATCH(c, do_run, c, phi, weight, ovlp, theta, fb, x, n_steps, energy_every, ortho_every, pc_every, u, eloc,
                  w_meas, parents, flags);
}

afqmc_status afqmc_step_host(afqmc_ctx* c, void* phi_h, double* weight_h, void* ovlp_h, const void* x_h, int32_t n_steps,
                             void* eloc_h, int32_t* flags_h, size_t* h2d_bytes, size_t* d2h_bytes) {
  if (!c) return AFQMC_EINVAL;
  c->err[0] = 0;
  NEED(c, n_steps >= 0, "afqmc_step_host: n_steps < 0");
  if (h2d_bytes) *h2d_bytes = 0;
  if (d2h_bytes) *d2h_bytes = 0;
  if (c->nw == 0) return AFQMC_OK;
  NEED(c, phi_h && weight_h && ovlp_h && (x_h || n_steps == 0) && (eloc_h || n_steps == 0), "afqmc_step_host: null pointer");
  const size_t nw = c->nw, ts = c->ts;
  const size_t phi_b = nw * c->M * c->nt * 2 * ts, x_b = nw * c->ng * ts;
  size_t up = 0, down = 0;
  cudaStream_t st = c->stream;
  CUDA_OK(c, cudaMemcpyAsync(c->h_phi, phi_h, phi_b, cudaMemcpyHostToDevice, st));
  CUDA_OK(c, cudaMemcpyAsync(c->h_weight, weight_h, nw * 8, cudaMemcpyHostToDevice, st));
  CUDA_OK(c, cudaMemsetAsync(c->h_flags, 0, nw * 4, st));
  up += phi_b + nw * 8;
  afqmc_status s = afqmc_overlap_green(c, c->h_phi, c->h_ovlp, c->h_theta, nullptr, c->h_flags);
  if (s) return s;
  s = afqmc_force_bias(c, c->h_phi, c->h_theta, c->h_fb);
  if (s) return s;
  // Fields go up and energies come down on a second (non-blocking) stream, double-buffered: the upload of step i+1 and
  // the download of step i-1 run under the kernels of step i (pinned host buffers; pageable ones serialise).
  if (!c->copy_ready && n_steps > 0) {
    CUDA_OK(c, cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_x[i], cudaEventDisableTiming));
      CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming));
      CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_e[i], cudaEventDisableTiming));
    }
    CUDA_OK(c, cudaEventCreateWithFlags(&c->ev_phi, cudaEventDisableTiming));
    c->copy_ready = 1;
  }
  cudaStream_t cs = c->copy_stream;
  void* xb[2] = {c->h_x, c->h_x2};
  zcplx* eb[2] = {c->h_eloc, c->h_eloc2};
  if (n_steps > 0) {   // the copy stream starts after everything already queued on the context's stream
    CUDA_OK(c, cudaEventRecord(c->ev_done[0], st));
    CUDA_OK(c, cudaStreamWaitEvent(cs, c->ev_done[0], 0));
  }
  auto upload = [&](int i) -> cudaError_t {   // fields of step i into buffer i & 1 (free once step i-2 is done)
    const int b = i & 1;
    cudaError_t e = cudaSuccess;
    if (i >= 2) e = cudaStreamWaitEvent(cs, c->ev_done[b], 0);
    if (e == cudaSuccess) e = cudaMemcpyAsync(xb[b], (const char*)x_h + (size_t)i * x_b, x_b, cudaMemcpyHostToDevice, cs);
    if (e == cudaSuccess) e = cudaEventRecord(c->ev_x[b], cs);
    up += x_b;
    return e;
  };
  if (n_steps > 0) CUDA_OK(c, upload(0));
  for (int i = 0; i < n_steps; ++i) {
    const int b = i & 1;
    if (i + 1 < n_steps) CUDA_OK(c, upload(i + 1));                      // queued ahead of step i's download
    CUDA_OK(c, cudaStreamWaitEvent(st, c->ev_x[b], 0));
    if (i >= 2) CUDA_OK(c, cudaStreamWaitEvent(st, c->ev_e[b], 0));      // energies of step i-2 have left buffer b
    const bool last = i == n_steps - 1;
    c->ev_phi_armed = last;
    s = afqmc_step(c, c->h_phi, c->h_weight, c->h_ovlp, c->h_theta, c->h_fb, xb[b], 1, eb[b], c->h_flags);
    c->ev_phi_armed = 0;
    if (s) return s;
    if (last) {   // the walker is final after H7: it goes down while overlap / force bias / energy of this step still run
      CUDA_OK(c, cudaStreamWaitEvent(cs, c->ev_phi, 0));
      CUDA_OK(c, cudaMemcpyAsync(phi_h, c->h_phi, phi_b, cudaMemcpyDeviceToHost, cs));
    }
    CUDA_OK(c, cudaEventRecord(c->ev_done[b], st));
    CUDA_OK(c, cudaStreamWaitEvent(cs, c->ev_done[b], 0));
    CUDA_OK(c, cudaMemcpyAsync((char*)eloc_h + (size_t)i * nw * 16, eb[b], nw * 16, cudaMemcpyDeviceToHost, cs));
    CUDA_OK(c, cudaEventRecord(c->ev_e[b], cs));
    down += nw * 16;
  }
  if (n_steps > 0) {   // the context's stream ends after the last download
    CUDA_OK(c, cudaEventRecord(c->ev_e[0], cs));
    CUDA_OK(c, cudaStreamWaitEvent(st, c->ev_e[0], 0));
  }
  if (n_steps == 0) CUDA_OK(c, cudaMemcpyAsync(phi_h, c->h_phi, phi_b, cudaMemcpyDeviceToHost, st));
  CUDA_OK(c, cudaMemcpyAsync(weight_h, c->h_weight, nw * 8, cudaMemcpyDeviceToHost, st));
  CUDA_OK(c, cudaMemcpyAsync(ovlp_h, c->h_ovlp, nw * 16, cudaMemcpyDeviceToHost, st));
  down += phi_b + nw * 8 + nw * 16;
  if (flags_h) {
    CUDA_OK(c, cudaMemcpyAsync(flags_h, c->h_flags, nw * 4, cudaMemcpyDeviceToHost, st));
    down += nw * 4;
  }
  CUDA_OK(c, cudaStreamSynchronize(st));
  if (h2d_bytes) *h2d_bytes = up;
  if (d2h_bytes) *d2h_bytes = down;
  return AFQMC_OK;
}

}  // extern "C"
