/* afqmc.h -- C ABI of the B200-native phaseless-AFQMC walker step.
 *
 * Source of every operation: Shee, Arthur, Zhang, Reichman, Friesner, "Phaseless Auxiliary-Field
 * Quantum Monte Carlo on Graphical Processing Units" (arXiv:1804.03310).  Citations are
 * PAPER.md:<line> (+ section / equation).  Where the paper is silent the reading is the one
 * listed in DESIGN.md "Readings" (R1..R18).
 *
 * Conventions that hold for every entry point
 *   - returns an afqmc_status; never throws, never prints, never allocates device memory;
 *   - the device entry points enqueue work on the stream given to afqmc_init and do NOT
 *     synchronise (the caller synchronises its stream); afqmc_init and afqmc_step_host do;
 *   - "DEVICE" pointers are caller-owned device memory (the Python binding hands in
 *     torch tensors' data_ptr()); "HOST" pointers are ordinary host memory;
 *   - complex = interleaved (re, im) pairs of the stated real type;
 *   - the real type T of walkers / Green's functions / force bias / fields follows
 *     afqmc_params.precision (0: float, complex64 walkers; 1: double, complex128 walkers);
 *     overlaps, weights, local energies are ALWAYS FP64 (R17: |S| reaches 1e209);
 *   - numerical events never fail a call: they set bits in flags[w]
 *       bit 0  overlap matrix singular / pivot below eps*max|A|
 *       bit 1  non-finite overlap or weight
 *       bit 2  walker killed by the phaseless rule cos(dtheta) <= 0 (weight := 0 exactly)
 *   - argument errors (null pointers, sizes out of the supported range) return
 *     AFQMC_EINVAL / AFQMC_EUNSUPPORTED before any launch.
 *
 * Layouts (w = walker, M = basis size, N_t = n_alpha + n_beta, alpha columns first)
 *   phi   [N_w][M][N_t] complex T     walker determinants Phi_w
 *   theta [N_w][M][N_t] complex T     Theta_s = Phi_s (Psi_s^T Phi_s)^-1
 *                                     (multi-det: Theta of the reference determinant)
 *   G     [N_w][2][M][M] complex T    G_s[i][j] = <Psi_T|c+_i c_j|phi>/<Psi_T|phi> (mixed for multi-det)
 *   fb    [N_w][n_chol]  complex T    f_g = sum_s Tr(L_g G_s)
 *   x     [N_w][n_chol]  T            auxiliary fields (host-drawn N(0,1)) PAPER.md:45 Eq.(2)
 *   ovlp  [N_w] complex double        S = <Psi_T|phi_w>
 *   weight[N_w] double ; eloc [N_w] complex double ; flags [N_w] int32
 */
#ifndef AFQMC_B200_H
#define AFQMC_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define AFQMC_API __attribute__((visibility("default")))
#else
#define AFQMC_API
#endif

typedef struct afqmc_ctx afqmc_ctx; /* opaque; owns no memory the caller allocated */

typedef enum {
  AFQMC_OK = 0,
  AFQMC_EINVAL = 1,
  AFQMC_EUNSUPPORTED = 2,
  AFQMC_ECUDA = 3,
  AFQMC_ENOMEM = 4
} afqmc_status;

typedef struct {
  int32_t M;            /* orbitals */
  int32_t n_alpha;      /* spin-up electrons (<= 32) */
  int32_t n_beta;       /* spin-down electrons (<= 32, may be 0) */
  int32_t n_chol;       /* N_gamma Cholesky / DF vectors */
  int32_t n_walkers;    /* N_w, batch handled by every call */
  int32_t precision;    /* 0: complex64 walkers / FP32 operands; 1: complex128 / FP64 */
  int32_t taylor_order; /* K of exp(A) ~ sum_{k<=K} A^k/k! (R9); 1..20 */
  int32_t weight_mode;  /* 0: hybrid; 1: local-energy form */
  int32_t n_det;        /* determinants in the trial, 1 = single determinant */
  int32_t n_act;        /* active orbitals spanning all determinants (0 if n_det == 1) */
  int32_t max_exc;      /* slots per spin in det_exc = largest excitation rank per spin, 1..4 (<= 2: closed-form 2 x 2 inverses and the
                           batched energy kernel; 3, 4: general small elimination, one-operator-at-a-time energy kernel) */
  int32_t gemm_path;    /* 0: auto (3 for precision 0, else 1); 1: SIMT FP32/FP64 everywhere; 2: tcgen05 3xTF32
                           GEMMs, one CTA per 128x256 tile; 3: the same on CTA pairs (cta_group::2, 256x256
                           tiles).  2 and 3 need precision 0.  DESIGN.md "Precision split". */
  double dt;            /* time step */
  double E0;            /* projector shift in e^{dt(E0-H)} (R7) */
} afqmc_params;

/* Bytes of DEVICE memory the caller must hand to afqmc_init: const_bytes holds the operands
 * precomputed once (E_h, R, Y, transposed L, ... PAPER.md:80 "computed once at the start"),
 * work_bytes holds per-step intermediates (one-body operators A_w, split planes, ...) and the
 * FP64 staging used during init.  Both are multiples of 256. */
AFQMC_API afqmc_status afqmc_query_bytes(const afqmc_params* p, size_t* const_bytes, size_t* work_bytes);

/* Build a context.  HOST inputs, FP64, row-major, read only during this call:
 *   h1      [M][M]          one-body matrix T_ij of Eq.(1), real symmetric
 *   L_chol  [n_chol][M][M]  V_ijkl = sum_g L_g[i][k] L_g[j][l], each real symmetric
 *   psiT_a  [M][n_alpha], psiT_b [M][n_beta]   trial orbitals, single determinant
 *   multi-determinant trial (n_det > 1): C_act [M][n_act] orthonormal columns shared
 *   by both spins, first n_sigma columns = reference determinant (psiT_a/psiT_b are then ignored
 *   and may be NULL); det_coeff [n_det] real c_i; det_exc [n_det][2][max_exc][2] =
 *   (hole < n_sigma, particle >= n_sigma) pairs, -1 padded: column `hole` of the reference is
 *   replaced in place by column `particle` of C_act (no re-sorting, hence no sign).
 * DEVICE: const_mem / work_mem of at least the sizes afqmc_query_bytes returned, 256-aligned,
 * owned by the caller, must outlive the context.  stream = cudaStream_t (0 = legacy default).
 * Precomputes on the device (hand-written FP64 kernels): h' = h - 1/2 sum_g L_g^2,
 * E_h = exp(-dt/2 h') (R3), R^s_g = Psi_s^T L_g, Y^s of Eq.(5), Psi_s^T h.
 * Synchronises the stream before returning.  Errors: EINVAL (null / non-symmetric h or L /
 * bad excitation list), EUNSUPPORTED (sizes), ECUDA. */
AFQMC_API afqmc_status afqmc_init(afqmc_ctx** out, const afqmc_params* p, const double* h1, const double* L_chol,
                        const double* psiT_a, const double* psiT_b, const double* C_act,
                        const double* det_coeff, const int32_t* det_exc, void* const_mem, void* work_mem,
                        void* stream);
AFQMC_API void afqmc_destroy(afqmc_ctx* ctx);
/* All further work of this context is enqueued on `stream` (cudaStream_t).  The device entry points launch kernels and
 * device-to-device copies only -- no synchronisation, no allocation -- so a call such as afqmc_step(n_steps) may be captured
 * into a CUDA graph on a capturing stream and replayed (bench.py does so for the launch-latency-bound configs, M < 96; per-stage
 * profiling must be off).  The caller orders the old and the new stream. */
AFQMC_API afqmc_status afqmc_set_stream(afqmc_ctx* ctx, void* stream);
/* Last error text of this context ("" if none); valid until the next call on ctx. ctx may be NULL
 * (then the text of the last failed afqmc_init of this thread). */
AFQMC_API const char* afqmc_last_error(const afqmc_ctx* ctx);

/* H1-H3: per walker A_s = Psi_s^T Phi_s, S = det A_a det A_b (LU, partial
 * pivoting), Theta_s = Phi_s A_s^-1; optional full G (DEVICE or NULL).  Multi-determinant trial:
 * S = sum_i c_i S_i with S_i from Sherman-Morrison-Woodbury updates off the reference (Eq.(4),
 * PAPER.md:63-66), theta = reference Theta_0, G = mixed Green's function. All DEVICE. */
AFQMC_API afqmc_status afqmc_overlap_green(afqmc_ctx* ctx, const void* phi, void* ovlp, void* theta, void* G_or_null,
                                 int32_t* flags);

/* H4: f_g = sum_s sum_{a,k} R^s_g[a][k] Theta_s[k][a] = sum_s Tr(L_g G_s)
 * (multi-det: mixed over determinants, needs the walker itself).  All DEVICE.  phi may be NULL for a
 * single-determinant trial. */
AFQMC_API afqmc_status afqmc_force_bias(afqmc_ctx* ctx, const void* phi, const void* theta, void* fb);

/* H5-H8 (Eq.(2),(3); :97): xbar = -i sqrt(dt) f, xs = x - xbar,
 * A = i sqrt(dt) sum_g xs_g L_g, Phi' = E_h [sum_{k<=K} A^k/k!] E_h Phi, then overlap / Theta of Phi',
 * dtheta = arg(S'/S), hybrid weight w' = w e^{dt E0} |S'/S e^{c}| max(0, cos dtheta),
 * c = x.xbar - xbar.xbar/2.  phi, ovlp, weight in/out; theta out; flags OR-ed.  All DEVICE.
 * weight_mode 1 uses exp(-dt(Re E_L - E0)) with eloc_pre = E_L of the pre-step walker (DEVICE,
 * complex double [N_w]); eloc_pre may be NULL in mode 0. */
AFQMC_API afqmc_status afqmc_propagate(afqmc_ctx* ctx, void* phi, const void* x, const void* fb, void* ovlp, double* weight,
                             void* theta, const void* eloc_pre, int32_t* flags);

/* H9 / H10 (Eq.(5)): E_L = sum_s Tr(Psi_s^T h Theta_s) + 1/2 sum_s vec(Theta_s)^T Y^s
 * vec(Theta_s) + sum_g f^a_g f^b_g  (complex).  Multi-det: mixed over determinants with rank-E updates
 * (needs phi).  All DEVICE.  phi may be NULL for a single-determinant trial. */
AFQMC_API afqmc_status afqmc_local_energy(afqmc_ctx* ctx, const void* phi, const void* theta, void* eloc);

/* n_steps full walker steps (Eq.(2),(3), :61-80, :97; order R10): [shift -> assemble -> Taylor propagate -> overlap/Theta ->
 * weight -> force bias -> local energy] per step.  State on entry/exit: phi, weight, ovlp, theta, fb of
 * the current walkers (seed with afqmc_overlap_green + afqmc_force_bias).  x [n_steps][N_w][n_chol] T,
 * eloc [n_steps][N_w] complex double (E_L of the post-step walker), flags OR-ed.  All DEVICE. */
AFQMC_API afqmc_status afqmc_step(afqmc_ctx* ctx, void* phi, double* weight, void* ovlp, void* theta, void* fb,
                        const void* x, int32_t n_steps, void* eloc, int32_t* flags);

/* The same n_steps through HOST buffers (pinned or pageable): copies phi, weight, x to the device,
 * seeds ovlp/theta/fb from phi, runs afqmc_step, copies phi, weight, ovlp, eloc, flags back, and
 * synchronises.  Device staging lives in work_mem (sized by afqmc_query_bytes for two steps of fields;
 * x is streamed step by step).  The per-step field upload and energy download run on a second, library-owned
 * non-blocking stream, double-buffered and ordered with events, so that with PINNED host buffers they overlap the
 * kernels of the neighbouring steps; the walkers go up before and come down after the steps on ctx's stream.  h2d_bytes / d2h_bytes (may be NULL) receive the bytes moved. */
AFQMC_API afqmc_status afqmc_step_host(afqmc_ctx* ctx, void* phi_h, double* weight_h, void* ovlp_h, const void* x_h,
                             int32_t n_steps, void* eloc_h, int32_t* flags_h, size_t* h2d_bytes,
                             size_t* d2h_bytes);

/* Walker orthonormalisation ("Walker orbitals are orthonormalized after every two
 * propagation steps"): thin QR of each spin block, Phi_s = Q_s R_s with R_s upper triangular and a real positive
 * diagonal (the unique thin QR, reading R21; modified Gram-Schmidt in FP64 on both precision paths).  phi (in/out)
 * becomes Q; ovlp (in/out, complex double [N_w]) becomes S / (det R_a det R_b), since |Phi> = det R_a det R_b |Q>.
 * Theta, the force bias and E_L are invariant (Theta = Phi A^-1), so theta / fb of the state stay valid.  A walker
 * with a vanishing or non-finite column is left untouched and flagged (bit 0 / bit 1).  flags may be NULL.
 * All DEVICE.  EUNSUPPORTED if N_t (M|1) 16 bytes exceed one CTA's shared memory. */
AFQMC_API afqmc_status afqmc_orthonormalize(afqmc_ctx* ctx, void* phi, void* ovlp, int32_t* flags);

/* "Simple combing" population control (NEXT-1; reading R22): W = sum_w weight, teeth
 * t_i = (i + u) W / N_w, new walker i = copy of the first walker p whose running sum weight[0] + ... + weight[p]
 * (accumulated in index order, FP64) exceeds t_i; every new walker gets weight W / N_w.  phi, ovlp, theta, fb follow
 * their parent (in place; moved through scratch in work_mem); the caller's flags array is NOT permuted: flags[i] is the
 * history of SLOT i (every event that happened to a walker while it sat there), not of a lineage.
 * u in [0, 1) is drawn by the caller (HOST value).
 * parent (DEVICE int32 [N_w], may be NULL) receives the map.  W == 0 or non-finite: nothing moves, weights kept.
 * All other pointers DEVICE.  Errors: EINVAL (null, u outside [0, 1)). */
AFQMC_API afqmc_status afqmc_population_control(afqmc_ctx* ctx, void* phi, double* weight, void* ovlp, void* theta, void* fb,
                                      double u, int32_t* parent);

/* Building blocks of the comb over a population SHARDED across ranks (PAPER.md:111
 * "subsets which are independently propagated and measured on different GPU cards", :121-127): the one exchange step
 * of the method.  Every rank holds N_w walkers; global slot g = rank * N_w + local index.  Protocol (the collectives
 * themselves are the caller's: paper_1804_03310_b200/dist.py uses torch.distributed all_gather + all_to_all_single):
 *   1. all-gather the weights -> weight_all [n_total]; afqmc_comb_map on every rank (same bits everywhere) gives
 *      parent_all [n_total] (reading R22, as afqmc_population_control) and w_new = { W / n_total, W } (DEVICE [2]).
 *      cum_scratch: DEVICE double [n_total].
 *   2. the map is monotone, so the global slots whose parent lives on this rank form ONE contiguous range
 *      [slot_lo, slot_lo + count): afqmc_comb_pack writes their parents' records, in slot order, into sendbuf
 *      (count * afqmc_comb_record_bytes; record = [phi | theta | fb | S]); first_local = rank * N_w.
 *   3. all-to-all with per-rank counts derived from parent_all; the receive buffer then holds this rank's N_w new
 *      walkers in slot order; afqmc_comb_unpack stores them and sets every weight to w_new[0] (kept if w_new[0] < 0,
 *      the dead-population case).
 * All pointers DEVICE; nothing synchronises.  Errors: EINVAL. */
AFQMC_API size_t afqmc_comb_record_bytes(const afqmc_ctx* ctx);
AFQMC_API afqmc_status afqmc_comb_map(afqmc_ctx* ctx, const double* weight_all, int64_t n_total, double u, double* cum_scratch,
                            int32_t* parent_all, double* w_new);
/* Allocation-free variant of afqmc_comb_map (reading R22) for callers that cannot provide scratch or call
 * cudaMalloc (CUDA graph capture, tight serving loops, harnesses that forbid it): the running-sum scratch is a file-scope device
 * array of AFQMC_NOALLOC_MAX_WALKERS doubles (512 KiB, held by every GPU that loads the library until exit).  Same inputs,
 * outputs and bits as afqmc_comb_map.  n_total > AFQMC_NOALLOC_MAX_WALKERS returns AFQMC_EUNSUPPORTED before any launch.  Calls no
 * cudaMalloc / cudaFree / allocating routine; the first call on a device resolves the array's address (cudaGetSymbolAddress).
 * ALL calls on a device share the one array: it keeps the last call's running sums (each call overwrites [0, n_total) before reading
 * it, so nothing needs clearing), and two calls that overlap on the GPU -- different streams or contexts -- RACE on it; serialise them.
 * All pointers DEVICE; enqueues on the context's stream; does not synchronise. */
#define AFQMC_NOALLOC_MAX_WALKERS 65536
AFQMC_API afqmc_status afqmc_comb_map_noalloc(afqmc_ctx* ctx, const double* weight_all, int64_t n_total, double u,
                                              int32_t* parent_all, double* w_new);
AFQMC_API afqmc_status afqmc_comb_pack(afqmc_ctx* ctx, const void* phi, const void* ovlp, const void* theta, const void* fb,
                             const int32_t* parent_all, int64_t slot_lo, int64_t count, int64_t first_local, void* sendbuf);
AFQMC_API afqmc_status afqmc_comb_unpack(afqmc_ctx* ctx, const void* recvbuf, void* phi, double* weight, void* ovlp, void* theta,
                               void* fb, const double* w_new);

/* Sums of the mixed estimator for one measurement: out3 (DEVICE double [3]) =
 * { sum_w weight[w], Re sum_w weight[w] eloc[w], Im sum_w weight[w] eloc[w] }, FP64, fixed summation tree; walkers with
 * weight exactly 0 contribute nothing (their E_L may be non-finite).  E_mix = out3[1] / out3[0]; across ranks the three
 * numbers are what is all-reduced.  An empty batch writes zeros.  All DEVICE. */
AFQMC_API afqmc_status afqmc_mixed_sums(afqmc_ctx* ctx, const double* weight, const void* eloc, double* out3);

/* The mixed estimator itself: e_mix[m] = (sums[m][1] + i sums[m][2]) / sums[m][0] for n measurements, sums
 * [n][3] as written by afqmc_mixed_sums (and, for a sharded population, all-reduced across ranks first).  A dead
 * population (sum of weights 0) gives NaN.  sums, e_mix (complex double [n]) DEVICE.  Errors: EINVAL. */
AFQMC_API afqmc_status afqmc_mixed_energy(afqmc_ctx* ctx, const double* sums, int32_t n, void* e_mix);

/* The paper's schedule around the walker step (NEXT-2; hybrid weights "to minimize evaluations of the
 * local energy, which is measured every 0.1 Ha^-1", orthonormalisation every 2 steps, population control every
 * 0.1 Ha^-1).  n_steps steps of [shift -> assemble -> Taylor -> overlap/Theta -> weight -> force bias]; after step n
 * (1-based), in this order (reading R23): if n % energy_every == 0, E_L of the walkers goes to
 * eloc[n / energy_every - 1][N_w] and their weights to w_meas[same][N_w] (DEVICE double, may be NULL); if
 * n % ortho_every == 0, afqmc_orthonormalize; if n % pc_every == 0, afqmc_population_control with
 * u[n / pc_every - 1] (HOST array, read during the call) and the map to parents[n / pc_every - 1][N_w] (DEVICE, may be
 * NULL).  0 switches a part off; energy_every = 1, ortho_every = pc_every = 0 is afqmc_step.  Needs weight_mode 0.
 * x [n_steps][N_w][n_chol] T DEVICE; state arguments as afqmc_step. */
AFQMC_API afqmc_status afqmc_run(afqmc_ctx* ctx, void* phi, double* weight, void* ovlp, void* theta, void* fb, const void* x,
                       int32_t n_steps, int32_t energy_every, int32_t ortho_every, int32_t pc_every, const double* u,
                       void* eloc, double* w_meas, int32_t* parents, int32_t* flags);

/* Number of kernels this context has launched since init (bench.py's gpu_launches). */
AFQMC_API int64_t afqmc_launch_count(const afqmc_ctx* ctx);

/* Per-stage device timing with CUDA events recorded on the context's stream around the stage's
 * kernels (bench.py's roofline line).  enable != 0 creates the events and resets the counters;
 * enable == 0 destroys them.  afqmc_profile_read may be called after the caller has synchronised the
 * stream: total_ms = sum of the elapsed times of the (at most 64) recorded executions, launches =
 * how many were recorded. */
enum {
  AFQMC_STAGE_SHIFT = 0,      /* H5 */
  AFQMC_STAGE_ASSEMBLE = 1,   /* H6: A_w = sum_g z_g L_g GEMM */
  AFQMC_STAGE_TAYLOR = 2,     /* H7 */
  AFQMC_STAGE_GREEN = 3,      /* H1-H3 + H8 (+ H10 overlap part) */
  AFQMC_STAGE_FORCE_BIAS = 4, /* H4 GEMM + finish */
  AFQMC_STAGE_ENERGY = 5,     /* H9 GEMMs / H10 energy */
  AFQMC_STAGE_SYMMETRIZE = 6, /* H6 tail: lower triangle of A_w from the upper one (tcgen05 path) */
  AFQMC_STAGE_ORTHO = 7,      /* NEXT-1: walker orthonormalisation */
  AFQMC_STAGE_POPCTL = 8,     /* NEXT-1: comb population control (3 kernels) */
  AFQMC_N_STAGES = 9
};
AFQMC_API afqmc_status afqmc_profile_enable(afqmc_ctx* ctx, int32_t enable);
AFQMC_API afqmc_status afqmc_profile_read(afqmc_ctx* ctx, int32_t stage, double* total_ms, int32_t* launches);

/* Peak microbenchmarks behind bench.py --peaks (the TF32 / FP32 / FP64 / L2 denominators are measured, not
 * assumed).  kind 0: back-to-back tcgen05.mma.kind::tf32 M = 128, N = n, operands from shared memory, one CTA per SM;
 * 1: the same with the a-operand in TMEM; 2: CTA pairs (cta_group::2, M = 256); 3: FFMA; 4: DFMA; 5: TMA stream of an
 * n-MiB buffer (L2 resident if n is small) into shared memory; 6-9: MMA issue patterns of the Taylor kernel (csrc/peaks.cuh);
 * 10: correctness probe of a TS-mode MMA (a-operand written to TMEM by tcgen05.st; n = N + 1000 r0; scratch receives D[128][N]).
 * scratch: DEVICE, >= 1 MiB (kind 5: the streamed buffer).
 * Synchronises `stream`.  ms = kernel time (CUDA events), units = flops (kinds 0-4) or bytes (kind 5) the kernel did,
 * clk = clocks per MMA measured inside CTA 0 (kinds 0-2, else 0).  No context needed.  Errors: EINVAL, ECUDA. */
AFQMC_API afqmc_status afqmc_peak_probe(int32_t kind, int32_t n, int32_t iters, void* scratch, size_t scratch_bytes,
                                        void* stream, double* ms, double* units, double* clk);

/* Operand-ordering experiment behind DESIGN.md 7 (which tcgen05 operand slices may repeat back to back): issues the
 * tab[0] MMAs {a byte offset, b byte offset, N, accumulator column} of tab = {n, a[64], b[64], nn[64], d[64]} (HOST int32)
 * `iters` times on every SM; clk = clocks per MMA in CTA 0.  scratch DEVICE >= 4 KiB.  Synchronises. */
AFQMC_API afqmc_status afqmc_peak_mma_table(const int32_t* tab, int32_t iters, void* scratch, void* stream, double* clk);

/* Which contraction path the context resolved to: 1 = SIMT, 2 = tcgen05 3xTF32. */
AFQMC_API int32_t afqmc_gemm_path(const afqmc_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* AFQMC_B200_H */
