/*
 * phi4smc.h -- C ABI of libphi4smc.so: the batched tempered-particle update of
 * "Particle Monte Carlo methods for Lattice Field Theory" (arxiv 2511.15196; PAPER.md) for
 * 2D phi^4 theory, as hand-written CUDA for sm_100a (NVIDIA B200).
 *
 * Model (PAPER.md:27-29 Eq. 1, :43): periodic L x L lattice, V = L*L sites, x = r*L + c,
 *   S_E(phi) = sum_x [ 1/2 (phi_{x+1hat}-phi_x)^2 + 1/2 (phi_{x+2hat}-phi_x)^2
 *                      + 1/2 m0sq phi_x^2 + lambda phi_x^4 ],
 *   U0(phi) = 1/2 sum_x phi_x^2,   p_beta(phi) ~ exp(-[U0 + beta S_E]),  beta in [0,1].
 * log Z means log int N(phi;0,I) exp(-S_E(phi)) dphi (reading A1).
 *
 * Conventions
 *  - Every function returns PHI4_OK (0) or a negative PHI4_E* code; nothing throws, aborts or
 *    prints.  phi4_strerror(code) names a code.  There is NO CPU fallback: without a CUDA device
 *    every compute entry point returns PHI4_ECUDA.
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers; everything else is by value.
 *  - The caller owns the device workspace (one allocation of *_workspace_bytes, 256-byte aligned)
 *    and the CUDA stream (a cudaStream_t passed as void*; NULL = the legacy default stream).  The
 *    library owns the opaque handle, keeps all state inside the workspace and never allocates
 *    device memory after *_init.  The workspace must outlive the handle.
 *  - The handle also owns one internal side stream (a host resource): independent branches of a
 *    step run there, forked from and joined back into the caller's stream by events inside the
 *    same call, so the caller's stream order is all a caller ever needs to reason about.
 *  - Work is enqueued on the handle's stream.  A function synchronises the stream only when it
 *    returns host values (an info struct, a host array, a double); this is stated per function.
 *  - Host-visible particle arrays are fp32, site-major and dense: h_phi[x*N + i], x = site,
 *    i = particle.  (Inside the workspace the particle stride is padded; not visible here.)
 *  - Random numbers: Philox4x32-10, key = (seed lo32, seed hi32), counter = (site quad or 0,
 *    slot, step counter, stream tag); readings R1/R2 fix the streams so that a CPU
 *    oracle can reproduce every draw.
 */
#ifndef PHI4SMC_H
#define PHI4SMC_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PHI4_OK 0
#define PHI4_EINVAL (-1)  /* bad argument, NULL handle, wrong sampler kind, workspace too small   */
#define PHI4_ENOMEM (-2)  /* host allocation failed                                               */
#define PHI4_ENOTPD (-3)  /* particle covariance not positive definite even after the jitter retry */
#define PHI4_ENAN (-4)    /* a non-finite action or weight was produced                           */
#define PHI4_ECUDA (-5)   /* a CUDA call failed or no device; see phi4_last_cuda_error()          */
#define PHI4_ETRUNC (-6)  /* ns_step / ns_run: the dead-point log (max_iters) filled up before the
                             stop rule fired.  Everything computed so far is valid, but log_Z()
                             is the dead-point evidence only (no live-point term was added).     */

#define PHI4_ETOOBIG (-7) /* a no-allocation entry point was given a size beyond its fixed capacity
                             (phi4_resample_noalloc: N > PHI4_NOALLOC_MAX_N)                     */

#define PHI4_HIST_BINS 80 /* B = 80 bins; fixed range [-1.6, 1.6] (reading A13)     */
#define PHI4_MAX_HOOK_STEPS 64 /* largest k accepted by smc_mutate when flags/margins are wanted  */
#define PHI4_NS_MAX_LIVE (1 << 20) /* nested sampling: largest n_live (k_delete: any value < n_live) */
#define PHI4_MAX_L 255    /* largest lattice side: several launches index sites by a grid
                             dimension limited to 65535 (V = 65025); *_workspace_bytes returns 0
                             and *_init PHI4_EINVAL beyond it                                    */

typedef struct phi4smc phi4smc; /* opaque sampler handle (SMC or NS) */

/* Free parameters of the outer kernel. */
typedef struct {
  int k_steps;      /* MCMC steps per tempering transition, n_MCMC >= 1           */
  float ess_target; /* target ESS fraction in (0,1) for adaptive tempering        */
  float step_scale; /* s in phi' = phi + s*Lc*z; 0 selects 2.38/sqrt(V) (A3)       */
  int mutation_path; /* 0 = automatic, 1 = generic (any V), 2 = fused tcgen05 (if it supports V),
                      * 3 = automatic with the large-V products (proposal L*z and covariance,
                      * L*L > 112) in 3xTF32 instead of the scaled 3xFP16 split of the same
                      * accuracy (reading A20, 5.2, 5.4); PHI4_EINVAL for L*L <= 112     */
  /* Rejuvenation kernel: 0 = RW-Metropolis (i), 1 = HMC (iii, :172; reading A14),
   * 2 = independent MH from the fitted Gaussian N(mu, Sigma) (ii, :200; reading A15; L*L <= 800).
   * HMC: mass matrix diag(1/var_x) from the particle covariance, hmc_leapfrog >= 1 leapfrog steps
   * of size hmc_eps > 0 per transition, k_steps transitions per temperature.  L <= 22 runs in one
   * register/shared-memory resident kernel per temperature; larger lattices keep position and
   * momentum in HBM scratch with one launch per leapfrog step (kick + drift in one pass).          */
  int kernel;
  float hmc_eps;
  int hmc_leapfrog;
  /* 1: global Z2 flips phi -> -phi (reading A17): after every resampling each
   * particle is flipped with probability 1/2 (always accepted: S_E and U0 are even).  0: off.   */
  int z2_flip;
} smc_params;

/* Inner kernel of nested sampling (PAPER.md:53(iv), :174).  inner = 0: constrained random walk of
 * n_walk steps (reading A5, the BASELINE.json configuration).  inner = 1: slice sampling along
 * covariance-drawn directions (reading A16): bracket of slice_width > 0 placed at random, at most
 * max_expand - 1 stepping-out moves (1..64), at most max_shrink shrinkages (1..256) per step;
 * n_walk is then the number of slice steps and accept_rate the fraction of steps that moved.   */
typedef struct {
  int inner;
  float slice_width;
  int max_expand;
  int max_shrink;
} ns_params;

/* One tempering transition, filled when smc_step is given a non-NULL pointer. */
typedef struct {
  double beta;        /* inverse temperature after the step                                      */
  double delta;       /* increment chosen by the ESS bisection (P1)                              */
  double ess_frac;    /* ESS/N of the incremental weights at delta                               */
  double dlogZ;       /* logsumexp(-delta S_E) - log N (P2)                                      */
  double logZ;        /* running sum of dlogZ                                                    */
  double accept_rate; /* mean Metropolis acceptance over the k_steps mutations    */
  int n_unique;       /* distinct ancestors chosen by the resampler                              */
  int chol_status;    /* 0 plain, 1 jitter retry used, -1 failed                                 */
  int temp_index;     /* 0-based index of this temperature                                       */
  int done;           /* 1 when beta == 1                                                        */
} smc_step_info;

typedef struct {
  double logX;           /* log prior volume after this iteration (reading A6)                   */
  double logZ;           /* log evidence accumulated from dead points (live term added when done) */
  double S_star;         /* likelihood threshold of this iteration: constraint S_E < S_star      */
  double accept_rate;    /* acceptance of the constrained walk                                   */
  double remaining_frac; /* X mean_live(e^-S) / (Z + X mean_live(e^-S))                          */
  int chol_status;
  int iter_index;
  int done; /* 0 running; 1 remaining_frac < stop_frac: the live term has been added to logZ;
             * 2 truncated: max_iters iterations were logged before the stop rule fired, logZ is
             * the dead-point evidence only (ns_step / ns_run then return PHI4_ETRUNC)            */
} ns_step_info;

typedef struct {
  double absM;         /* <|M|>, M = (1/V) sum_x phi_x                             */
  double M2;           /* <M^2>                                                                  */
  double chi;          /* V (<M^2> - <|M|>^2)                                                    */
  double mean_SE;      /* <S_E>                                                                  */
  double mode_balance; /* #(M>0) / #(M<0), zeros ignored, +inf if no negatives, 0 if no positives
                        * (PAPER.md:293); NS: weight mass on each side (reading A19)             */
  double hist[PHI4_HIST_BINS]; /* normalised (weighted) histogram of M on [-1.6, 1.6]            */
} phi4_observables;

const char* phi4_strerror(int code);
/* Text of the last CUDA error seen by this handle ("" if none); valid until the next call.
 * h == NULL: the message of the last smc_init / ns_init that failed in this process.        */
const char* phi4_last_cuda_error(const phi4smc* h);
/* Diagnostic: number of CUDA kernels this library has launched in this process so far. */
uint64_t phi4_kernel_launches(void);

/* Measurement aid: the roofline denominators that MEASURED_PEAKS.json does not hold,
 * measured on the current device with kernels that do nothing else: dense tcgen05 kind::tf32 and kind::f16
 * throughput (burst: best short launch; sustained: back-to-back launches for `seconds`, 0 < seconds
 * <= 30), FP32 FMA and 32x32->64 integer multiply rates in 1e12 lane-operations per second.
 * d_scratch: >= 4096 bytes of device memory (contents destroyed).  Synchronises.               */
typedef struct {
  double tf32_tflops_burst;
  double tf32_tflops_sustained;
  double ffma_tlaneops;       /* 1e12 FMA lane-operations / s (x2 for flop)                        */
  double imad_wide_tlaneops;  /* 1e12 IMAD.WIDE + LOP3 pairs / s: the unit of a Philox round       */
  int32_t sms;
  int32_t reserved;
  double dfma_tlaneops;       /* 1e12 FP64 FMA lane-operations / s (8 chains per thread): half the FP32 rate on a B200 */
  double f16_tflops_burst;    /* dense tcgen05.mma kind::f16 (FP16 operands, FP32 accumulator)     */
  double f16_tflops_sustained;
} phi4_peaks;
int phi4_measure_peaks(double seconds, phi4_peaks* out, void* d_scratch, size_t scratch_bytes,
                       void* cuda_stream);

/* ---------------------------------------------------------------- SMC-RW (PAPER.md:53(i)) ----
 * smc_workspace_bytes: bytes of device memory smc_init needs for an L x L lattice and N particles
 * (0 if L < 1, L > PHI4_MAX_L or N < 2).  Sized for 180 GB parts: C4 (L=64, N=131072) needs
 * about 15 GB.  m0sq, lambda (and kappa) must be finite, else *_init returns PHI4_EINVAL.        */
size_t smc_workspace_bytes(int L, int N);

/* Creates an SMC sampler: particles phi_i ~ N(0,I) from Philox stream INIT, S_E and U0 evaluated,
 * beta = 0, logZ = 0, Lc = I, defaults k_steps = 10, ess_target = 0.5, step_scale = 0 (2.38/sqrt V).
 * d_workspace: device memory of >= smc_workspace_bytes(L,N).  Enqueues on cuda_stream, no sync.  */
int smc_init(phi4smc** out, int L, float m0sq, float lambda, int N, uint64_t seed,
             void* d_workspace, size_t workspace_bytes, void* cuda_stream);
/* The kappa-lambda parameterisation (Appendix G; reading A18):
 *   Eq. 2: S_E(phi; kappa, lambda) = kappa/2 sum_{x,mu} (phi_{x+mu}-phi_x)^2
 *                                    + sum_x [ phi_x^2 + lambda (phi_x^2 - 1)^2 ],
 * kappa >= 0 the physical nearest-neighbour coupling that "scales only the kinetic term".  By
 * Eq. 4 this is Eq. 1's stencil with the kinetic term multiplied by kappa, m0sq = 2 (1 - 2 lambda)
 * and the same quartic coefficient; the additive constant V*lambda is dropped as in Eq. 5, so
 * every S_E and log_Z of such a handle refers to Eq. 5 (subtract V*lambda from log_Z for Eq. 2).
 * U0, the tempering path and everything else are as for smc_init; the same kernels run (the
 * kinetic coefficient is a model parameter of every stencil).  PHI4_EINVAL if kappa or lambda is
 * negative or not finite.                                                                       */
int smc_init_kl(phi4smc** out, int L, float kappa, float lambda, int N, uint64_t seed,
                void* d_workspace, size_t workspace_bytes, void* cuda_stream);
/* Re-initialises an existing handle (SMC or NS) with a new seed exactly as *_init would: fresh
 * particles from stream INIT, beta = 0, logZ = 0 (NS: -inf, logX = 0), Lc = I, history cleared.
 * Device work only (no host allocation); enqueue only.                                          */
int smc_reset(phi4smc* h, uint64_t seed);
int smc_destroy(phi4smc* h); /* synchronises the stream, frees host resources; NULL is a no-op    */
int smc_set_params(phi4smc* h, const smc_params* p);

/* One temperature (SURVEY 8(a) P1,P2,P3,P4,C1,C2,(M1-M4) x k_steps):
 * bisection for delta at the target ESS, incremental weights and log Z, systematic resampling,
 * gather, covariance + Cholesky of the resampled particles (A4), k_steps fused RW-Metropolis
 * mutations at the new beta.  info == NULL: enqueue only.  info != NULL: synchronises and fills
 * it.  Calling it when beta == 1 is a no-op that reports done = 1.                               */
int smc_step(phi4smc* h, smc_step_info* info);

/* Runs smc_step until beta == 1 or max_temps transitions were made; termination is decided on
 * the device, the host only polls a flag.  Synchronises.  *n_temps (may be NULL) = transitions
 * made by this call.  Returns PHI4_ENOTPD / PHI4_ENAN if a step failed, PHI4_ECUDA if the
 * stream reports an error or no step finishes for 120 s (the same holds for ns_run).            */
int smc_run(phi4smc* h, int max_temps, int* n_temps);

/* Per-temperature records of all transitions made so far (at most cap entries are copied;
 * returns the number available through *n).  Synchronises.                                       */
int smc_get_history(phi4smc* h, smc_step_info* h_info, int cap, int* n);

/* C1 + C2 from the current, equally weighted particles: mean, centred covariance with 1/(N-1),
 * lower Cholesky factor (readings A4, R6).  Enqueue only.                                        */
int estimate_cov_chol(phi4smc* h);

/* Magnetisation observables of the current particles (SMC: equal weights; NS: dead points and
 * live points with their nested-sampling weights).  Synchronises.                                */
int observables(phi4smc* h, phi4_observables* out);

/* Synchronises; SMC: sum of dlogZ so far; NS: log evidence (with the live term once done).
 * NaN if h is NULL.                                                                              */
double log_Z(const phi4smc* h);

/* ------------------------------------------------ nested sampling (PAPER.md:53(iv), :170) ---- */
size_t ns_workspace_bytes(int L, int n_live, int k_delete, int max_iters);

/* n_live points ~ N(0,I), likelihood exp(-S_E); per iteration the k_delete lowest-likelihood
 * points are deleted and each replaced by an n_walk-step covariance-preconditioned constrained
 * walk (accept iff S_E' < S_star and log u < -dU0, reading A5).  stop_frac: remaining-evidence
 * fraction at which the run ends (BASELINE configs: 1e-3).  max_iters bounds the dead-point log.
 * Requires 2 <= n_live <= PHI4_NS_MAX_LIVE and 1 <= k_delete < n_live (the paper's own setting,
 * N = 5000 with delete fraction 0.5, is ns_init(.., 5000, 2500, ..)); up to
 * 16384 live points are ordered by one CTA in shared memory, more by a multi-block network.      */
int ns_init(phi4smc** out, int L, float m0sq, float lambda, int n_live, int k_delete, int n_walk,
            uint64_t seed, double stop_frac, int max_iters, void* d_workspace,
            size_t workspace_bytes, void* cuda_stream);
/* ns_init for Eq. 2's (kappa, lambda); see smc_init_kl.                                         */
int ns_init_kl(phi4smc** out, int L, float kappa, float lambda, int n_live, int k_delete,
               int n_walk, uint64_t seed, double stop_frac, int max_iters, void* d_workspace,
               size_t workspace_bytes, void* cuda_stream);
/* One iteration N1-N4.  info != NULL synchronises.  No-op once done.              */
int ns_set_params(phi4smc* h, const ns_params* p); /* defaults: inner 0, width 1, 8, 32          */
int ns_step(phi4smc* h, ns_step_info* info);
/* Until done or max_iters more iterations; synchronises.  PHI4_ETRUNC if the handle's dead-point
 * log filled up first (see ns_step_info.done).                                                  */
int ns_run(phi4smc* h, int max_iters, int* n_iters);

/* ------------------------------------------------- test / checkpoint hooks (all synchronise) --
 * Needed for lockstep parity with the oracle.  Checkpoint / resume: the RNG is counter-based, so
 * the whole sampler state is the particles with their cached S_E, U0 (smc_get_state) plus the
 * scalars of phi4_run_state (smc_get_run_state); smc_restore puts both back and the run then
 * continues bit for bit as the uninterrupted one would (NS: add ns_get_dead / ns_set_dead).
 * Any output pointer may be NULL.  N below is the particle count (n_live for NS).               */
typedef struct {
  double beta;           /* SMC: current inverse temperature                                     */
  double delta;          /* SMC: last increment (the starting point of the next ESS root solve)  */
  double logZ;           /* SMC: running sum; NS: evidence of the dead points so far             */
  double logX;           /* NS: log prior volume                                                 */
  double S_star;         /* NS: last threshold                                                   */
  double remaining_frac; /* NS                                                                   */
  int32_t index;         /* transitions / iterations completed: keys the RESAMPLE, Z2 and NS
                            start-point streams                                                  */
  int32_t done;
  uint64_t step_counter; /* mutation steps made: keys the PROP / ACC streams                     */
} phi4_run_state;
int smc_get_run_state(phi4smc* h, phi4_run_state* out);
/* Replaces particles, cached actions and control scalars.  h_SE and h_U0 are either both given
 * (taken as they are: a bit-exact resume) or both NULL (recomputed from h_phi).                 */
int smc_restore(phi4smc* h, const float* h_phi, const float* h_SE, const float* h_U0,
                const phi4_run_state* rs);
int smc_get_state(phi4smc* h, float* h_phi, float* h_SE, float* h_U0, double* beta,
                  uint64_t* step_counter);
/* Replaces the particles (S_E, U0 are recomputed on the device), beta and the step counter.      */
int smc_set_state(phi4smc* h, const float* h_phi, double beta, uint64_t step_counter);
int smc_get_chol(phi4smc* h, float* h_Lc /* V*V row-major, strict upper = 0 */);
int smc_set_chol(phi4smc* h, const float* h_Lc);
int smc_get_cov(phi4smc* h, float* h_Sigma /* V*V row-major */);
int smc_get_mean(phi4smc* h, float* h_mu /* V: particle mean of the last covariance estimate */);
/* M1-M4 only: k mutation steps at the current beta and Lc; step counters continue from the
 * handle's counter.  h_accept[j*N+i] in {0,1}, h_margin[j*N+i] = g of reading R4 as the kernel
 * computed it (fp32).  k <= PHI4_MAX_HOOK_STEPS when either array is wanted.                     */
int smc_mutate(phi4smc* h, int k, uint8_t* h_accept, float* h_margin);
/* P1+P2 at the current beta: delta < 0 selects the bisection, otherwise the given delta is used.
 * Advances beta and logZ; h_w receives the max-shifted fp32 weights (max = 1).                   */
/* Measurement hook: enqueues `reps` back-to-back mutations of k steps each (as smc_mutate without
 * flags, no host synchronisation in between) bracketed by CUDA events on the handle's stream and
 * returns the average device time of one k-step mutation in milliseconds.                        */
int smc_time_mutation(phi4smc* h, int k, int reps, float* h_ms_per_call);
/* Measurement hook: one phase of the step, `reps` times back to back between two CUDA events on
 * the handle's stream; returns the average device time of one call in milliseconds.  Phases 1-3
 * exist only where a mutation step is three kernels (L*L > 112, mutation_path != 1).  The state
 * afterwards is valid but meaningless (e.g. a resampling without its reweighting): smc_reset or
 * smc_restore before using the handle for anything else.  PHASE_REWEIGHT advances beta.       */
#define PHI4_PHASE_MUTATION 0 /* k_steps x (M1-M4), as smc_step enqueues them                  */
#define PHI4_PHASE_PROPOSAL 1 /* M2: the tcgen05 proposal GEMM of one step, operands in place  */
#define PHI4_PHASE_NORMALS 2  /* M1: the normals of one step                                   */
#define PHI4_PHASE_ACCEPT 3   /* M3 + M4: action differences, decision, commit of one step     */
#define PHI4_PHASE_RESAMPLE 4 /* P3 + P4: integer scan, ancestors, gather                      */
#define PHI4_PHASE_GATHER 5   /* P4 alone (with the ancestors of the last resampling)          */
#define PHI4_PHASE_COVCHOL 6  /* C1 + C2                                                       */
#define PHI4_PHASE_REWEIGHT 7 /* P1 + P2                                                       */
int smc_time_phase(phi4smc* h, int phase, int reps, float* h_ms_per_call);
int smc_reweight(phi4smc* h, double delta, float* h_w, smc_step_info* info);
/* P3+P4: systematic resampling of the device weights (or of h_w if non-NULL) with the Philox
 * offset of the current temperature index, then the gather.  h_ancestors receives a_j.           */
int smc_resample(phi4smc* h, const float* h_w, int32_t* h_ancestors);
/* NS hooks: the last iteration's dead indices (k_delete, by decreasing S_E) and the dead-point
 * log so far (S_E, M, log w per dead point; n_dead = iterations * k_delete).                     */
int ns_get_dead(phi4smc* h, int32_t* h_last_dead_idx, float* h_dead_S, float* h_dead_M,
                double* h_dead_logw, int cap, int* n_dead);
/* Restores the first n_dead entries of the dead-point log (checkpoint / resume of observables). */
int ns_set_dead(phi4smc* h, const float* h_dead_S, const float* h_dead_M,
                const double* h_dead_logw, int n_dead);

/* ------------------------------------------------------------- no-allocation entry point ------
 * For callers that cannot allocate device memory (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): exact systematic resampling (P3; reading
 * R5) without a handle or a workspace.  The scratch of the kernels (64-bit integer CDF, block sums,
 * control block) is a file-scope __device__ array of PHI4_NOALLOC_SCRATCH_BYTES inside the library:
 * every GPU that loads libphi4smc.so holds that much until the process exits.  The call performs no
 * cudaMalloc / cudaFree and calls no allocating library routine; it only enqueues kernels.
 *   d_w          DEVICE, N fp32 weights in [0, 1] (the resampler's contract: max-shifted, max = 1)
 *   N            1 <= N <= PHI4_NOALLOC_MAX_N, else PHI4_ETOOBIG (nothing is enqueued)
 *   seed, t      the offset U is word 0 of the Philox draw (tag RESAMPLE, step t, slot 0): the same
 *                ancestors as smc_resample on a handle with this seed at temperature index t
 *   d_ancestors  DEVICE, receives N int32 ancestor indices (identity map if every weight is 0)
 * Enqueues on cuda_stream and returns without synchronising.  All calls share the one array, which
 * keeps the last call's contents (each call re-initialises what it reads): calls that overlap on
 * the GPU -- different streams or host threads -- race; serialise them.
 * phi4_noalloc_setup() looks up the array's device address for the CURRENT device (done lazily by
 * the first call otherwise; call it once per device before graph capture begins).              */
#define PHI4_NOALLOC_MAX_N 131072
#define PHI4_NOALLOC_SCRATCH_BYTES 1181952
int phi4_noalloc_setup(void);
int phi4_resample_noalloc(const float* d_w, int N, uint64_t seed, uint32_t t, int32_t* d_ancestors,
                          void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PHI4SMC_H */
