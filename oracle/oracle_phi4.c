/*
 * oracle_phi4.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, FP64 CPU restatement of the batched tempered-particle update
 * of "Particle Monte Carlo methods for Lattice Field Theory" for
 * 2D phi^4 theory.  It is the parity oracle for the CUDA library in
 * paper_2511_15196_b200/csrc and shares no code with it.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load it.
 *
 * Layout everywhere: particles are site-major, phi[x*N + i], x = r*L + c
 * (lattice site, row r, column c), i = particle index.  All arithmetic is
 * double; the only float is the weight vector handed to the resampler
 * (reading R5 fixes the resampler's input as fp32).
 *
 * Paper passages followed (line numbers of /root/reference/PAPER.md):
 *   Eq. 1  (:27-29)  S_E = sum_x [ 1/2 sum_mu (phi_{x+mu}-phi_x)^2
 *                                  + 1/2 m0^2 phi_x^2 + lambda phi_x^4 ],
 *                    periodic lattice {0..L-1}^2
 *   :37              magnetisation M = (1/V) sum_x phi_x
 *   :43              U0 = 1/2 sum_x phi_x^2, p_beta ~ exp(-[U0 + beta S_E])
 *   :53(i), :172     SMC-RW: Gaussian random-walk proposal scaled by the
 *                    particle covariance, scale 2.38^2/V on the covariance
 *   :161, :169, :244 adaptive tempering by target ESS
 *   :53(iv), :161, :170, :174  nested sampling with a delete fraction and a
 *                    hard likelihood constraint
 *   :293-295         mode balance; 80-bin histogram
 * Where the paper is silent the readings R1-R6 / A1-A13 of DESIGN.md apply;
 * each function names the one it follows.
 *
 * Pins (tests/test_oracle_*.py): Philox known-answer vectors; Gaussian
 * closed-form log Z, <M^2>, E[S_E]; 1-D and 4-D quadrature at L=1, L=2;
 * Z2 / translation invariance; plane-wave eigenvalues; finite differences;
 * exact-rational brute force of systematic resampling; numpy cov/cholesky.
 * Parity unpinned: the phi^4 (lambda>0) end-to-end runs at L>=4 have no
 * closed form; they are pinned only through the pieces.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_TAG_INIT 0u
#define ORC_TAG_PROP 1u
#define ORC_TAG_ACC 2u
#define ORC_TAG_RESAMPLE 3u
#define ORC_TAG_NS_START 4u
#define ORC_TAG_NS_PROP 5u
#define ORC_TAG_NS_ACC 6u

#define ORC_MODE_SMC 0
#define ORC_MODE_NS 1

static const double ORC_TWO_PI = 6.283185307179586476925286766559;

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------
 * R1: Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  Ten rounds; the
 * key is bumped by the Weyl constants between rounds.
 * ---------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2],
                       uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0;
    uint32_t n1 = lo1;
    uint32_t n2 = hi0 ^ c3 ^ k1;
    uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R1 counter layout: (c0, c1, c2, c3) = (site-quad q or 0, slot i, step t,
 * stream tag); key = (seed lo32, seed hi32). */
static void orc_draw(uint64_t seed, uint32_t tag, uint32_t t, uint32_t i,
                     uint32_t q, uint32_t out[4]) {
  uint32_t ctr[4] = {q, i, t, tag};
  uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
  orc_philox4x32_10(ctr, key, out);
}

/* R2: two 32-bit words -> two standard normals by Box-Muller.
 * radius uniform u_r = (k+1) 2^-24 in (0,1], angle theta = 2 pi k' 2^-24. */
static void orc_box_muller(uint32_t xa, uint32_t xb, double* za, double* zb) {
  double ur = ((double)(xa >> 8) + 1.0) * (1.0 / 16777216.0);
  double th = ORC_TWO_PI * ((double)(xb >> 8) * (1.0 / 16777216.0));
  double r = sqrt(-2.0 * log(ur));
  *za = r * cos(th);
  *zb = r * sin(th);
}

/* z[0..V-1] for (seed, tag, t, slot i): quad q gives sites 4q..4q+3, a
 * ragged last quad is truncated. */
void orc_normals(uint64_t seed, uint32_t tag, uint32_t t, uint32_t i, int V,
                 double* z) {
  int nq = (V + 3) / 4;
  for (int q = 0; q < nq; ++q) {
    uint32_t w[4];
    double zz[4];
    orc_draw(seed, tag, t, i, (uint32_t)q, w);
    orc_box_muller(w[0], w[1], &zz[0], &zz[1]);
    orc_box_muller(w[2], w[3], &zz[2], &zz[3]);
    for (int j = 0; j < 4; ++j)
      if (4 * q + j < V) z[4 * q + j] = zz[j];
  }
}

/* R2: accept uniform u = (k+1) 2^-24 from word 0 of the (c0 = 0) draw. */
double orc_uniform(uint64_t seed, uint32_t tag, uint32_t t, uint32_t i) {
  uint32_t w[4];
  orc_draw(seed, tag, t, i, 0u, w);
  return ((double)(w[0] >> 8) + 1.0) * (1.0 / 16777216.0);
}

/* raw 32-bit word 0 of the (c0 = 0) draw: resampling offset U (R5) and the
 * nested-sampling start-point choice (R1 tag 4). */
uint32_t orc_word0(uint64_t seed, uint32_t tag, uint32_t t, uint32_t i) {
  uint32_t w[4];
  orc_draw(seed, tag, t, i, 0u, w);
  return w[0];
}

/* ------------------------------------------------------------------------
 * O-1: the model.  One field f[0..V-1], x = r*L + c.  Eq. 1 verbatim with
 * periodic forward neighbours (reading A2: (c+1)%L and (r+1)%L also for
 * L = 1, 2).  If absum != NULL it receives sum_x(|kin_x|+|mass_x|+|quart_x|)
 * (the scale of reading A12's tolerance).
 * ---------------------------------------------------------------------- */
/* Appendix G ("Alternative parameterizations"): a physical
 * nearest-neighbour coupling kappa "that scales only the kinetic term",
 *   Eq. 2: S_E(phi; kappa, lambda) = kappa/2 sum_{x,mu} (phi_{x+mu}-phi_x)^2
 *                                    + sum_x [ phi_x^2 + lambda (phi_x^2-1)^2 ].
 * By Eq. 4, phi^2 + lambda (phi^2-1)^2 = lambda phi^4 + (1-2 lambda) phi^2 + lambda, so
 * Eq. 2 is Eq. 1 with the kinetic term multiplied by kappa, m0^2 = 2 (1 - 2 lambda), the
 * same quartic coefficient, plus the constant V lambda (Eq. 5 drops it: it "only shifts
 * log Z").  The oracle keeps one kinetic coefficient for the whole process (1 = Eq. 1);
 * every action, gradient, mutation and run below reads it.  orc_action_eq2_field is
 * Eq. 2 written out verbatim, constant included (reading A18). */
static double orc_kappa = 1.0;
void orc_set_kinetic(double kappa) { orc_kappa = kappa; }
double orc_get_kinetic(void) { return orc_kappa; }

double orc_action_eq2_field(const double* f, int L, double kappa, double lam) {
  double S = 0.0;
  for (int r = 0; r < L; ++r)
    for (int c = 0; c < L; ++c) {
      double p = f[r * L + c];
      double pr = f[r * L + (c + 1) % L], pd = f[((r + 1) % L) * L + c];
      S += 0.5 * kappa * ((pr - p) * (pr - p) + (pd - p) * (pd - p));
      S += p * p + lam * (p * p - 1.0) * (p * p - 1.0);
    }
  return S;
}

double orc_action_field(const double* f, int L, double m0sq, double lam,
                        double* absum) {
  double S = 0.0, A = 0.0;
  for (int r = 0; r < L; ++r) {
    for (int c = 0; c < L; ++c) {
      double p = f[r * L + c];
      double pr = f[r * L + (c + 1) % L];       /* x + 1-hat (next column) */
      double pd = f[((r + 1) % L) * L + c];     /* x + 2-hat (next row)    */
      double kin = 0.5 * orc_kappa * ((pr - p) * (pr - p) + (pd - p) * (pd - p));
      double mass = 0.5 * m0sq * p * p;
      double quart = lam * p * p * p * p;
      S += kin + mass + quart;
      A += fabs(kin) + fabs(mass) + fabs(quart);
    }
  }
  if (absum) *absum = A;
  return S;
}

/* PAPER.md:43  U0 = 1/2 sum_x phi_x^2 */
double orc_u0_field(const double* f, int V) {
  double u = 0.0;
  for (int x = 0; x < V; ++x) u += f[x] * f[x];
  return 0.5 * u;
}

/* Gradient dS_E/dphi_x of Eq. 1 (finite-difference pin, HMC force):
 * kappa sum_mu (2 phi_x - phi_{x+mu} - phi_{x-mu}) + m0^2 phi_x + 4 lambda phi_x^3 */
void orc_action_grad_field(const double* f, int L, double m0sq, double lam,
                           double* g) {
  for (int r = 0; r < L; ++r)
    for (int c = 0; c < L; ++c) {
      double p = f[r * L + c];
      double e = f[r * L + (c + 1) % L], w = f[r * L + (c + L - 1) % L];
      double s = f[((r + 1) % L) * L + c], n = f[((r + L - 1) % L) * L + c];
      g[r * L + c] = orc_kappa * (4.0 * p - e - w - s - n) + m0sq * p + 4.0 * lam * p * p * p;
    }
}

static void orc_get_field(const double* phi, int N, int V, int i, double* f) {
  for (int x = 0; x < V; ++x) f[x] = phi[(size_t)x * N + i];
}
static void orc_put_field(double* phi, int N, int V, int i, const double* f) {
  for (int x = 0; x < V; ++x) phi[(size_t)x * N + i] = f[x];
}

/* S_E, U0 (and optionally the A12 scale) of every particle. */
void orc_action_batch(const double* phi, int N, int L, double m0sq, double lam,
                      double* S, double* U0, double* absum) {
  int V = L * L;
#pragma omp parallel
  {
    double* f = (double*)malloc(sizeof(double) * V);
#pragma omp for
    for (int i = 0; i < N; ++i) {
      double a;
      orc_get_field(phi, N, V, i, f);
      S[i] = orc_action_field(f, L, m0sq, lam, &a);
      U0[i] = orc_u0_field(f, V);
      if (absum) absum[i] = a;
    }
    free(f);
  }
}

/* O-2 step 1: phi_i ~ N(0, I) from stream INIT (tag 0, t = 0). */
void orc_init_particles(uint64_t seed, int N, int V, double* phi) {
#pragma omp parallel
  {
    double* z = (double*)malloc(sizeof(double) * V);
#pragma omp for
    for (int i = 0; i < N; ++i) {
      orc_normals(seed, ORC_TAG_INIT, 0u, (uint32_t)i, V, z);
      orc_put_field(phi, N, V, i, z);
    }
    free(z);
  }
}

/* ------------------------------------------------------------------------
 * M1-M4, O-2 step 2(e): k covariance-preconditioned random-walk Metropolis
 * steps on every particle (PAPER.md:53(i), :172; reading A3: s multiplies
 * L_c z).  For step j = 0..k-1 the step counter is t0 + j.
 *   z        = normals(seed, tag_prop, t, i)
 *   phi'     = phi + s * Lc z                (Lc lower-triangular, row-major)
 *   SMC mode: g = -((U0'-U0) + beta (S'-S)) - ln u        (R4)
 *   NS  mode: g = -(U0'-U0) - ln u, and additionally S' < S_star (A5)
 *   accept iff g > 0 (and the constraint in NS mode); u from tag_acc.
 * accept_out[j*N+i] (0/1) and margin_out[j*N+i] (= g; in NS mode also
 * cmargin_out = S_star - S') may be NULL.  phi, S, U0 are updated in place.
 * slots (may be NULL = identity) gives the Philox slot of column i (R1:
 * streams are keyed by slot), so that a sub-sample of a large population
 * can be replayed with its own streams.
 * ---------------------------------------------------------------------- */
void orc_mutate(double* phi, double* S, double* U0, int N, int L, double m0sq,
                double lam, const double* Lc, double s, double beta, int mode,
                double S_star, uint64_t seed, uint32_t tag_prop,
                uint32_t tag_acc, uint32_t t0, int k, uint8_t* accept_out,
                double* margin_out, double* cmargin_out, const int32_t* slots) {
  int V = L * L;
#pragma omp parallel
  {
    double* f = (double*)malloc(sizeof(double) * V);
    double* fp = (double*)malloc(sizeof(double) * V);
    double* z = (double*)malloc(sizeof(double) * V);
#pragma omp for
    for (int i = 0; i < N; ++i) {
      orc_get_field(phi, N, V, i, f);
      double Si = S[i], Ui = U0[i];
      const uint32_t slot = slots ? (uint32_t)slots[i] : (uint32_t)i;
      for (int j = 0; j < k; ++j) {
        uint32_t t = t0 + (uint32_t)j;
        orc_normals(seed, tag_prop, t, slot, V, z);
        for (int x = 0; x < V; ++x) {
          double d = 0.0;
          for (int y = 0; y <= x; ++y) d += Lc[(size_t)x * V + y] * z[y];
          fp[x] = f[x] + s * d;
        }
        double Sp = orc_action_field(fp, L, m0sq, lam, NULL);
        double Up = orc_u0_field(fp, V);
        double u = orc_uniform(seed, tag_acc, t, slot);
        double g;
        int acc;
        if (mode == ORC_MODE_SMC) {
          g = -((Up - Ui) + beta * (Sp - Si)) - log(u);
          acc = g > 0.0;
        } else {
          g = -(Up - Ui) - log(u);
          acc = (g > 0.0) && (Sp < S_star);
          if (cmargin_out) cmargin_out[(size_t)j * N + i] = S_star - Sp;
        }
        if (margin_out) margin_out[(size_t)j * N + i] = g;
        if (accept_out) accept_out[(size_t)j * N + i] = (uint8_t)acc;
        if (acc) {
          memcpy(f, fp, sizeof(double) * V);
          Si = Sp;
          Ui = Up;
        }
      }
      orc_put_field(phi, N, V, i, f);
      S[i] = Si;
      U0[i] = Ui;
    }
    free(f); free(fp); free(z);
  }
}

/* ------------------------------------------------------------------------
 * P1/P2 (reading R3).
 * ---------------------------------------------------------------------- */
/* log sum_i exp(-c S_i), max-shifted. */
double orc_lse_neg(const double* S, int N, double c) {
  double m = -INFINITY;
  for (int i = 0; i < N; ++i) { double v = -c * S[i]; if (v > m) m = v; }
  double acc = 0.0;
  for (int i = 0; i < N; ++i) acc += exp(-c * S[i] - m);
  return m + log(acc);
}

/* ESS(delta)/N with ESS = (sum e^{-delta S})^2 / sum e^{-2 delta S}. */
double orc_ess_frac(const double* S, int N, double delta) {
  return exp(2.0 * orc_lse_neg(S, N, delta) - orc_lse_neg(S, N, 2.0 * delta)) /
         (double)N;
}

/* R3: delta in (0, 1-beta].  If ESS(1-beta)/N >= target: delta = 1-beta and
 * *final = 1.  Else 48 halvings of [0, 1-beta], mid kept in lo if
 * f(mid) > 0, result (lo+hi)/2. */
double orc_next_delta(const double* S, int N, double beta, double target,
                      int* final) {
  double hi = 1.0 - beta;
  if (orc_ess_frac(S, N, hi) - target >= 0.0) { *final = 1; return hi; }
  *final = 0;
  double lo = 0.0;
  for (int it = 0; it < 48; ++it) {
    double mid = 0.5 * (lo + hi);
    if (orc_ess_frac(S, N, mid) - target > 0.0) lo = mid; else hi = mid;
  }
  return 0.5 * (lo + hi);
}

/* P2: logw_i = -delta S_i (U0 cancels between p_beta and p_{beta+delta},
 * PAPER.md:43); returns dlogZ = lse(logw) - log N; w_i = exp(logw_i - max)
 * rounded to fp32 (the resampler's input type, R5), max w = 1.0f. */
double orc_reweight(const double* S, int N, double delta, float* w) {
  double m = -INFINITY;
  for (int i = 0; i < N; ++i) { double v = -delta * S[i]; if (v > m) m = v; }
  double acc = 0.0;
  for (int i = 0; i < N; ++i) {
    double e = exp(-delta * S[i] - m);
    acc += e;
    if (w) w[i] = (float)e;
  }
  return m + log(acc) - log((double)N);
}

/* ------------------------------------------------------------------------
 * P3 (reading R5): exact systematic resampling on integers.
 *   q_i = floor(w_i 2^40), C_i = sum_{m<=i} q_m, T = C_{N-1}
 *   t_j = floor(((j 2^32 + U) T) / (N 2^32)),  a_j = #{i : C_i <= t_j},
 *   clamped to N-1.  Returns 0, or -1 if T == 0.
 * ---------------------------------------------------------------------- */
int orc_resample_systematic(const float* w, int N, uint32_t U, int32_t* anc) {
  uint64_t* C = (uint64_t*)malloc(sizeof(uint64_t) * N);
  uint64_t run = 0;
  for (int i = 0; i < N; ++i) {
    run += (uint64_t)floor((double)w[i] * 1099511627776.0);
    C[i] = run;
  }
  uint64_t T = run;
  if (T == 0) { free(C); return -1; }
  int i = 0;
  for (int j = 0; j < N; ++j) {
    unsigned __int128 num =
        ((unsigned __int128)(((uint64_t)j << 32) + U)) * (unsigned __int128)T;
    unsigned __int128 den = (unsigned __int128)((uint64_t)N << 32);
    uint64_t tj = (uint64_t)(num / den);
    while (i < N - 1 && C[i] <= tj) ++i;   /* t_j is non-decreasing in j */
    anc[j] = i;
  }
  free(C);
  return 0;
}

/* P4: out[x][j] = in[x][anc_j]. */
void orc_gather(const double* in, int N, int V, const int32_t* anc,
                double* out) {
  for (int x = 0; x < V; ++x)
    for (int j = 0; j < N; ++j)
      out[(size_t)x * N + j] = in[(size_t)x * N + anc[j]];
}

/* ------------------------------------------------------------------------
 * C1/C2 (readings A4, R6): unweighted sample covariance with
 * the 1/(N-1) normalisation from centred sums, then lower Cholesky.  If a
 * pivot is <= 0, eps = 1e-6 tr(Sigma)/V is added to the diagonal once and
 * the factorisation restarted; a second failure returns -1.
 * Sigma and Lc are V x V row-major; Lc's strict upper triangle is zero.
 * Returns 0 (no jitter), 1 (jitter used) or -1.
 * ---------------------------------------------------------------------- */
void orc_covariance(const double* phi, int N, int V, double* mu,
                    double* Sigma) {
  for (int x = 0; x < V; ++x) {
    double m = 0.0;
    for (int i = 0; i < N; ++i) m += phi[(size_t)x * N + i];
    mu[x] = m / (double)N;
  }
#pragma omp parallel for schedule(dynamic, 4)
  for (int x = 0; x < V; ++x)
    for (int y = 0; y <= x; ++y) {
      double acc = 0.0;
      for (int i = 0; i < N; ++i)
        acc += (phi[(size_t)x * N + i] - mu[x]) * (phi[(size_t)y * N + i] - mu[y]);
      acc /= (double)(N - 1);
      Sigma[(size_t)x * V + y] = acc;
      Sigma[(size_t)y * V + x] = acc;
    }
}

static int orc_chol_once(const double* A, int V, double add, double* Lc) {
  memset(Lc, 0, sizeof(double) * (size_t)V * V);
  for (int j = 0; j < V; ++j) {
    double d = A[(size_t)j * V + j] + add;
    for (int m = 0; m < j; ++m) d -= Lc[(size_t)j * V + m] * Lc[(size_t)j * V + m];
    if (!(d > 0.0)) return -1;
    double ljj = sqrt(d);
    Lc[(size_t)j * V + j] = ljj;
    for (int r = j + 1; r < V; ++r) {
      double v = A[(size_t)r * V + j];
      for (int m = 0; m < j; ++m) v -= Lc[(size_t)r * V + m] * Lc[(size_t)j * V + m];
      Lc[(size_t)r * V + j] = v / ljj;
    }
  }
  return 0;
}

int orc_cholesky(const double* Sigma, int V, double* Lc) {
  if (orc_chol_once(Sigma, V, 0.0, Lc) == 0) return 0;
  double tr = 0.0;
  for (int x = 0; x < V; ++x) tr += Sigma[(size_t)x * V + x];
  if (orc_chol_once(Sigma, V, 1e-6 * tr / (double)V, Lc) == 0) return 1;
  return -1;
}

int orc_cov_chol(const double* phi, int N, int V, double* Sigma, double* Lc) {
  double* mu = (double*)malloc(sizeof(double) * V);
  orc_covariance(phi, N, V, mu, Sigma);
  free(mu);
  return orc_cholesky(Sigma, V, Lc);
}

/* ------------------------------------------------------------------------
 * O (reading A13): magnetisation observables with
 * optional log-weights logw (NULL = equal weights).
 * out[0]=<|M|>, out[1]=<M^2>, out[2]=chi=V(<M^2>-<|M|>^2), out[3]=<S_E>,
 * out[4]=mode balance (positive over negative samples, zeros
 *   ignored; +inf if no negatives, 0 if no positives).  With log-weights the
 *   "number of samples" on a side is its weight mass (reading A19): an
 *   unweighted count of nested-sampling dead points would describe the prior,
 *   not the weighted sample the other outputs describe.
 * out[5..84] = 80-bin normalised weighted histogram of M on [-1.6, 1.6],
 * out-of-range values clamped into the end bins.
 * ---------------------------------------------------------------------- */
void orc_magnetisation(const double* phi, int N, int V, double* M) {
  for (int i = 0; i < N; ++i) {
    double m = 0.0;
    for (int x = 0; x < V; ++x) m += phi[(size_t)x * N + i];
    M[i] = m / (double)V;
  }
}

void orc_observables_from_M(const double* M, const double* S,
                            const double* logw, int N, int V, double* out) {
  double mx = -INFINITY;
  if (logw) for (int i = 0; i < N; ++i) if (logw[i] > mx) mx = logw[i];
  double W = 0.0, a = 0.0, m2 = 0.0, se = 0.0;
  double wpos = 0.0, wneg = 0.0;
  for (int b = 0; b < 85; ++b) out[b] = 0.0;
  for (int i = 0; i < N; ++i) {
    double wi = logw ? exp(logw[i] - mx) : 1.0;
    W += wi;
    a += wi * fabs(M[i]);
    m2 += wi * M[i] * M[i];
    if (S) se += wi * S[i];
    if (M[i] > 0.0) wpos += wi; else if (M[i] < 0.0) wneg += wi;
    int b = (int)floor((M[i] + 1.6) / (3.2 / 80.0));
    if (b < 0) b = 0;
    if (b > 79) b = 79;
    out[5 + b] += wi;
  }
  out[0] = a / W;
  out[1] = m2 / W;
  out[2] = (double)V * (out[1] - out[0] * out[0]);
  out[3] = se / W;
  out[4] = wneg > 0.0 ? wpos / wneg : INFINITY;
  for (int b = 0; b < 80; ++b) out[5 + b] /= W;
}

void orc_observables(const double* phi, const double* S, int N, int V,
                     double* out) {
  double* M = (double*)malloc(sizeof(double) * N);
  orc_magnetisation(phi, N, V, M);
  orc_observables_from_M(M, S, NULL, N, V, out);
  free(M);
}

/* ------------------------------------------------------------------------
 * O-2: the SMC-RW run.  phi (V*N doubles) receives the final particles.
 * Per temperature m (m = 0..T-1) info[8*m + ...] = {beta', delta, ESS/N at
 * delta, dlogZ, accept rate, #unique ancestors, chol status, 0}.
 * Returns the number of temperatures T (<= max_temps), or -1 on a
 * Cholesky failure; *logZ_out = sum of dlogZ.
 * ---------------------------------------------------------------------- */
int orc_smc_run(int L, double m0sq, double lam, int N, uint64_t seed, int k,
                double ess_target, double step_scale, int max_temps,
                double* phi, double* S, double* U0, double* logZ_out,
                double* info) {
  int V = L * L;
  double s = step_scale > 0.0 ? step_scale : 2.38 / sqrt((double)V);
  double* tmp = (double*)malloc(sizeof(double) * (size_t)V * N);
  double* Sigma = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* Lc = (double*)malloc(sizeof(double) * (size_t)V * V);
  float* w = (float*)malloc(sizeof(float) * N);
  int32_t* anc = (int32_t*)malloc(sizeof(int32_t) * N);
  uint8_t* acc = (uint8_t*)malloc((size_t)k * N);
  orc_init_particles(seed, N, V, phi);
  orc_action_batch(phi, N, L, m0sq, lam, S, U0, NULL);
  double beta = 0.0, logZ = 0.0;
  uint32_t t = 0;
  int T = 0, rc = 0;
  while (beta < 1.0 && T < max_temps) {
    int final;
    double delta = orc_next_delta(S, N, beta, ess_target, &final);
    double beta_new = final ? 1.0 : beta + delta;
    double ess = orc_ess_frac(S, N, delta);
    double dlz = orc_reweight(S, N, delta, w);
    logZ += dlz;
    uint32_t U = orc_word0(seed, ORC_TAG_RESAMPLE, (uint32_t)T, 0u);
    orc_resample_systematic(w, N, U, anc);
    orc_gather(phi, N, V, anc, tmp);
    memcpy(phi, tmp, sizeof(double) * (size_t)V * N);
    orc_gather(S, N, 1, anc, tmp);  memcpy(S, tmp, sizeof(double) * N);
    orc_gather(U0, N, 1, anc, tmp); memcpy(U0, tmp, sizeof(double) * N);
    int uniq = 1;
    for (int j = 1; j < N; ++j) uniq += anc[j] != anc[j - 1];
    int st = orc_cov_chol(phi, N, V, Sigma, Lc);
    if (st < 0) { rc = -1; break; }
    orc_mutate(phi, S, U0, N, L, m0sq, lam, Lc, s, beta_new, ORC_MODE_SMC, 0.0,
               seed, ORC_TAG_PROP, ORC_TAG_ACC, t + 1, k, acc, NULL, NULL, NULL);
    t += (uint32_t)k;
    double nacc = 0.0;
    for (size_t m = 0; m < (size_t)k * N; ++m) nacc += acc[m];
    if (info) {
      double* o = info + 8 * T;
      o[0] = beta_new; o[1] = delta; o[2] = ess; o[3] = dlz;
      o[4] = nacc / ((double)k * N); o[5] = uniq; o[6] = st; o[7] = 0.0;
    }
    beta = beta_new;
    ++T;
  }
  *logZ_out = logZ;
  free(tmp); free(Sigma); free(Lc); free(w); free(anc); free(acc);
  return rc < 0 ? rc : T;
}

/* ------------------------------------------------------------------------
 * N1 (readings A6): indices of the k_del live points with the largest S_E,
 * ordered by S descending, ties by index ascending.
 * ---------------------------------------------------------------------- */
typedef struct { double s; int32_t i; } orc_si;
static int orc_cmp_desc(const void* a, const void* b) {
  const orc_si* p = (const orc_si*)a; const orc_si* q = (const orc_si*)b;
  if (p->s > q->s) return -1;
  if (p->s < q->s) return 1;
  return (p->i > q->i) - (p->i < q->i);
}
void orc_ns_select(const double* S, int n, int k_del, int32_t* dead) {
  orc_si* v = (orc_si*)malloc(sizeof(orc_si) * n);
  for (int i = 0; i < n; ++i) { v[i].s = S[i]; v[i].i = i; }
  qsort(v, n, sizeof(orc_si), orc_cmp_desc);
  for (int j = 0; j < k_del; ++j) dead[j] = v[j].i;
  free(v);
}

static double orc_logaddexp(double a, double b) {
  if (a == -INFINITY) return b;
  if (b == -INFINITY) return a;
  double m = a > b ? a : b;
  return m + log(exp(a - m) + exp(b - m));
}

/* log mean_i exp(-S_i) */
static double orc_log_mean_like(const double* S, int n) {
  return orc_lse_neg(S, n, 1.0) - log((double)n);
}

/* ------------------------------------------------------------------------
 * O-3: the nested-sampling run (PAPER.md:53(iv),161,170,174; readings A5,
 * A6; Skilling 2006 for the volume bookkeeping, PAPER.md:141 ref [37]).
 * Live points ~ N(0,I) (tag 0), likelihood exp(-S_E).  Per iteration it:
 *   Lc from all n live points (A5); N1 select; N2 for the j-th dead point
 *   (j = 1..k_del, lowest likelihood first) logX_j = logX_{j-1} - 1/(n-j+1),
 *   w_j = X_{j-1} - X_j, Z += w_j exp(-S_j); N3 walker j starts from survivor
 *   number (word0 mod (n-k_del)) in index order (tag 4, c1 = j-1, c2 = it),
 *   walks n_walk steps at step counters it*n_walk + 1 .. (tags 5/6, slot
 *   j-1) under S' < S_star = min dead S, and replaces dead slot dead[j-1];
 *   N4 stop when X mean_live(e^-S) / (Z + X mean_live(e^-S)) < stop_frac,
 *   then Z += X mean_live(e^-S).
 * dead_S / dead_M / dead_logw (capacity max_iter*k_del) record the deleted
 * points (logw = log w_j, without the likelihood).  info[6*it + ...] =
 * {logX, logZ so far, S_star, accept rate, remaining fraction, chol status}.
 * Returns the number of iterations done, or -1.
 * ---------------------------------------------------------------------- */
void orc_slice_walk(double* phi, double* S, double* U0, int N, int L,
                    double m0sq, double lam, const double* Lc, double width,
                    int m_expand, int max_shrink, double S_star, uint64_t seed,
                    uint32_t t0, int k, double* t_out, int32_t* nexp_out,
                    int32_t* nshr_out, double* amb_out, const int32_t* slots);

/* inner = 0: the constrained random walk of reading A5 (orc_mutate, MODE_NS);
 * inner = 1: the slice-sampling kernel of reading A16 (orc_slice_walk) with
 * bracket width slice_w, m_expand stepping-out moves, max_shrink shrinkages;
 * info[3] is then the fraction of steps that moved. */
int orc_ns_run_inner(int L, double m0sq, double lam, int n, int k_del, int n_walk,
                     uint64_t seed, double step_scale, double stop_frac,
                     int max_iter, int inner, double slice_w, int m_expand,
                     int max_shrink, double* phi, double* S, double* U0,
                     double* logZ_out, double* logX_out, double* dead_S,
                     double* dead_M, double* dead_logw, double* info) {
  int V = L * L;
  double s = step_scale > 0.0 ? step_scale : 2.38 / sqrt((double)V);
  double* Sigma = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* Lc = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* wphi = (double*)malloc(sizeof(double) * (size_t)V * k_del);
  double* wS = (double*)malloc(sizeof(double) * k_del);
  double* wU = (double*)malloc(sizeof(double) * k_del);
  int32_t* dead = (int32_t*)malloc(sizeof(int32_t) * k_del);
  int32_t* surv = (int32_t*)malloc(sizeof(int32_t) * n);
  uint8_t* isdead = (uint8_t*)malloc(n);
  uint8_t* acc = (uint8_t*)malloc((size_t)n_walk * k_del);
  orc_init_particles(seed, n, V, phi);
  orc_action_batch(phi, n, L, m0sq, lam, S, U0, NULL);
  double logX = 0.0, logZ = -INFINITY;
  int it = 0, rc = 0;
  for (; it < max_iter; ++it) {
    int st = orc_cov_chol(phi, n, V, Sigma, Lc);
    if (st < 0) { rc = -1; break; }
    orc_ns_select(S, n, k_del, dead);
    double S_star = S[dead[k_del - 1]];
    for (int j = 1; j <= k_del; ++j) {
      int d = dead[j - 1];
      double logX_new = logX - 1.0 / (double)(n - j + 1);
      /* log(X_{j-1} - X_j) = logX_{j-1} + log(1 - exp(logX_j - logX_{j-1})) */
      double logw = logX + log1p(-exp(logX_new - logX));
      logZ = orc_logaddexp(logZ, logw - S[d]);
      double m = 0.0;
      for (int x = 0; x < V; ++x) m += phi[(size_t)x * n + d];
      size_t slot = (size_t)it * k_del + (size_t)(j - 1);
      if (dead_S) dead_S[slot] = S[d];
      if (dead_M) dead_M[slot] = m / (double)V;
      if (dead_logw) dead_logw[slot] = logw;
      logX = logX_new;
    }
    memset(isdead, 0, n);
    for (int j = 0; j < k_del; ++j) isdead[dead[j]] = 1;
    int ns = 0;
    for (int i = 0; i < n; ++i) if (!isdead[i]) surv[ns++] = i;
    for (int j = 0; j < k_del; ++j) {
      uint32_t r = orc_word0(seed, ORC_TAG_NS_START, (uint32_t)it, (uint32_t)j);
      int src = surv[r % (uint32_t)ns];
      for (int x = 0; x < V; ++x)
        wphi[(size_t)x * k_del + j] = phi[(size_t)x * n + src];
      wS[j] = S[src];
      wU[j] = U0[src];
    }
    if (inner == 0) {
      orc_mutate(wphi, wS, wU, k_del, L, m0sq, lam, Lc, s, 0.0, ORC_MODE_NS,
                 S_star, seed, ORC_TAG_NS_PROP, ORC_TAG_NS_ACC,
                 (uint32_t)it * (uint32_t)n_walk + 1u, n_walk, acc, NULL, NULL,
                 NULL);
    } else {
      double* tt = (double*)malloc(sizeof(double) * (size_t)n_walk * k_del);
      orc_slice_walk(wphi, wS, wU, k_del, L, m0sq, lam, Lc, slice_w, m_expand,
                     max_shrink, S_star, seed,
                     (uint32_t)it * (uint32_t)n_walk + 1u, n_walk, tt, NULL,
                     NULL, NULL, NULL);
      for (size_t m = 0; m < (size_t)n_walk * k_del; ++m) acc[m] = tt[m] != 0.0;
      free(tt);
    }
    for (int j = 0; j < k_del; ++j) {
      int d = dead[j];
      for (int x = 0; x < V; ++x)
        phi[(size_t)x * n + d] = wphi[(size_t)x * k_del + j];
      S[d] = wS[j];
      U0[d] = wU[j];
    }
    double nacc = 0.0;
    for (size_t m = 0; m < (size_t)n_walk * k_del; ++m) nacc += acc[m];
    double log_live = logX + orc_log_mean_like(S, n);
    double rem = exp(log_live - orc_logaddexp(logZ, log_live));
    if (info) {
      double* o = info + 6 * it;
      o[0] = logX; o[1] = logZ; o[2] = S_star;
      o[3] = nacc / ((double)n_walk * k_del); o[4] = rem; o[5] = st;
    }
    if (rem < stop_frac) {
      logZ = orc_logaddexp(logZ, log_live);
      ++it;
      break;
    }
  }
  *logZ_out = logZ;
  *logX_out = logX;
  free(Sigma); free(Lc); free(wphi); free(wS); free(wU); free(dead);
  free(surv); free(isdead); free(acc);
  return rc < 0 ? rc : it;
}

int orc_ns_run(int L, double m0sq, double lam, int n, int k_del, int n_walk,
               uint64_t seed, double step_scale, double stop_frac,
               int max_iter, double* phi, double* S, double* U0,
               double* logZ_out, double* logX_out, double* dead_S,
               double* dead_M, double* dead_logw, double* info) {
  return orc_ns_run_inner(L, m0sq, lam, n, k_del, n_walk, seed, step_scale,
                          stop_frac, max_iter, 0, 0.0, 0, 0, phi, S, U0, logZ_out,
                          logX_out, dead_S, dead_M, dead_logw, info);
}

/* ------------------------------------------------------------------------
 * NEXT row f1 -- SMC-HMC rejuvenation (PAPER.md:53(iii), :172): "short HMC
 * trajectories", "diagonal mass matrix", "fixed trajectory of 20 leapfrog
 * steps".  Reading A14: target U(phi) = U0 + beta S_E; mass matrix
 * M = diag(1/var_x) with var_x the particle variance of site x (the diagonal
 * of the covariance of reading A4); momentum p = z / sqrt(var) with z the
 * PROP-stream normals; nfrog leapfrog steps of size eps:
 *     p <- p - eps/2 grad U;  nfrog x { phi <- phi + eps var p;
 *     p <- p - eps grad U (eps/2 after the last position update) };
 * H = U + 1/2 sum var_x p_x^2; margin g = (H_old - H_new) - ln u (ACC stream),
 * accept iff g > 0.  grad U = phi + beta grad S_E (orc_action_grad_field).
 * Same outputs / slot keying as orc_mutate.
 * ---------------------------------------------------------------------- */
static void orc_grad_u(const double* f, int L, double m0sq, double lam,
                       double beta, double* g) {
  orc_action_grad_field(f, L, m0sq, lam, g);
  for (int x = 0; x < L * L; ++x) g[x] = f[x] + beta * g[x];
}

void orc_hmc_mutate(double* phi, double* S, double* U0, int N, int L,
                    double m0sq, double lam, const double* var, double eps,
                    int nfrog, double beta, uint64_t seed, uint32_t t0, int k,
                    uint8_t* accept_out, double* margin_out,
                    const int32_t* slots) {
  int V = L * L;
#pragma omp parallel
  {
    double* f = (double*)malloc(sizeof(double) * V);
    double* q = (double*)malloc(sizeof(double) * V);
    double* p = (double*)malloc(sizeof(double) * V);
    double* g = (double*)malloc(sizeof(double) * V);
    double* z = (double*)malloc(sizeof(double) * V);
#pragma omp for
    for (int i = 0; i < N; ++i) {
      orc_get_field(phi, N, V, i, f);
      double Si = S[i], Ui = U0[i];
      const uint32_t slot = slots ? (uint32_t)slots[i] : (uint32_t)i;
      for (int j = 0; j < k; ++j) {
        uint32_t t = t0 + (uint32_t)j;
        orc_normals(seed, ORC_TAG_PROP, t, slot, V, z);
        double K0 = 0.0;
        for (int x = 0; x < V; ++x) {
          p[x] = z[x] / sqrt(var[x]);
          K0 += 0.5 * var[x] * p[x] * p[x];
          q[x] = f[x];
        }
        orc_grad_u(q, L, m0sq, lam, beta, g);
        for (int x = 0; x < V; ++x) p[x] -= 0.5 * eps * g[x];
        for (int s = 0; s < nfrog; ++s) {
          for (int x = 0; x < V; ++x) q[x] += eps * var[x] * p[x];
          orc_grad_u(q, L, m0sq, lam, beta, g);
          double h = (s + 1 == nfrog) ? 0.5 * eps : eps;
          for (int x = 0; x < V; ++x) p[x] -= h * g[x];
        }
        double K1 = 0.0;
        for (int x = 0; x < V; ++x) K1 += 0.5 * var[x] * p[x] * p[x];
        double Sp = orc_action_field(q, L, m0sq, lam, NULL);
        double Up = orc_u0_field(q, V);
        double u = orc_uniform(seed, ORC_TAG_ACC, t, slot);
        double gm = ((Ui + beta * Si + K0) - (Up + beta * Sp + K1)) - log(u);
        int acc = gm > 0.0;
        if (margin_out) margin_out[(size_t)j * N + i] = gm;
        if (accept_out) accept_out[(size_t)j * N + i] = (uint8_t)acc;
        if (acc) {
          memcpy(f, q, sizeof(double) * V);
          Si = Sp;
          Ui = Up;
        }
      }
      orc_put_field(phi, N, V, i, f);
      S[i] = Si;
      U0[i] = Ui;
    }
    free(f); free(q); free(p); free(g); free(z);
  }
}

/* One leapfrog trajectory of a single field with given momentum (pin helper:
 * reversibility and energy-error scaling).  q, p are updated in place;
 * returns H_new - H_old. */
double orc_leapfrog(double* q, double* p, int L, double m0sq, double lam,
                    const double* var, double eps, int nfrog, double beta) {
  int V = L * L;
  double* g = (double*)malloc(sizeof(double) * V);
  double H0 = orc_u0_field(q, V) + beta * orc_action_field(q, L, m0sq, lam, NULL);
  for (int x = 0; x < V; ++x) H0 += 0.5 * var[x] * p[x] * p[x];
  orc_grad_u(q, L, m0sq, lam, beta, g);
  for (int x = 0; x < V; ++x) p[x] -= 0.5 * eps * g[x];
  for (int s = 0; s < nfrog; ++s) {
    for (int x = 0; x < V; ++x) q[x] += eps * var[x] * p[x];
    orc_grad_u(q, L, m0sq, lam, beta, g);
    double h = (s + 1 == nfrog) ? 0.5 * eps : eps;
    for (int x = 0; x < V; ++x) p[x] -= h * g[x];
  }
  double H1 = orc_u0_field(q, V) + beta * orc_action_field(q, L, m0sq, lam, NULL);
  for (int x = 0; x < V; ++x) H1 += 0.5 * var[x] * p[x] * p[x];
  free(g);
  return H1 - H0;
}

/* SMC with HMC rejuvenation: orc_smc_run with step 2(e) replaced by k HMC
 * transitions; var = diag of the covariance of the resampled particles. */
int orc_smc_hmc_run(int L, double m0sq, double lam, int N, uint64_t seed, int k,
                    double ess_target, double eps, int nfrog, int max_temps,
                    double* phi, double* S, double* U0, double* logZ_out,
                    double* info) {
  int V = L * L;
  double* tmp = (double*)malloc(sizeof(double) * (size_t)V * N);
  double* Sigma = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* mu = (double*)malloc(sizeof(double) * V);
  double* var = (double*)malloc(sizeof(double) * V);
  float* w = (float*)malloc(sizeof(float) * N);
  int32_t* anc = (int32_t*)malloc(sizeof(int32_t) * N);
  uint8_t* acc = (uint8_t*)malloc((size_t)k * N);
  orc_init_particles(seed, N, V, phi);
  orc_action_batch(phi, N, L, m0sq, lam, S, U0, NULL);
  double beta = 0.0, logZ = 0.0;
  uint32_t t = 0;
  int T = 0;
  while (beta < 1.0 && T < max_temps) {
    int final;
    double delta = orc_next_delta(S, N, beta, ess_target, &final);
    double beta_new = final ? 1.0 : beta + delta;
    double ess = orc_ess_frac(S, N, delta);
    double dlz = orc_reweight(S, N, delta, w);
    logZ += dlz;
    uint32_t U = orc_word0(seed, ORC_TAG_RESAMPLE, (uint32_t)T, 0u);
    orc_resample_systematic(w, N, U, anc);
    orc_gather(phi, N, V, anc, tmp);
    memcpy(phi, tmp, sizeof(double) * (size_t)V * N);
    orc_gather(S, N, 1, anc, tmp);  memcpy(S, tmp, sizeof(double) * N);
    orc_gather(U0, N, 1, anc, tmp); memcpy(U0, tmp, sizeof(double) * N);
    orc_covariance(phi, N, V, mu, Sigma);
    for (int x = 0; x < V; ++x) var[x] = Sigma[(size_t)x * V + x];
    orc_hmc_mutate(phi, S, U0, N, L, m0sq, lam, var, eps, nfrog, beta_new, seed,
                   t + 1, k, acc, NULL, NULL);
    t += (uint32_t)k;
    double nacc = 0.0;
    for (size_t m = 0; m < (size_t)k * N; ++m) nacc += acc[m];
    if (info) {
      double* o = info + 8 * T;
      o[0] = beta_new; o[1] = delta; o[2] = ess; o[3] = dlz;
      o[4] = nacc / ((double)k * N); o[5] = 0; o[6] = 0; o[7] = 0.0;
    }
    beta = beta_new;
    ++T;
  }
  *logZ_out = logZ;
  free(tmp); free(Sigma); free(mu); free(var); free(w); free(anc); free(acc);
  return T;
}

/* ------------------------------------------------------------------------
 * NEXT row f2 -- SMC-IRMH rejuvenation (PAPER.md:53(ii): "independent
 * Metropolis-Hastings, with a Gaussian proposal fitted to the particles";
 * :200).  Reading A15: proposal q = N(mu, Sigma) with mu, Sigma
 * the particle mean and covariance of reading A4, Sigma = Lc Lc^T;
 *     phi' = mu + Lc z,  z = PROP-stream normals (same keying as orc_mutate);
 *     log q(phi) = -1/2 |Lc^-1 (phi - mu)|^2 + const,  log q(phi') = -1/2 |z|^2 + const;
 *     g = -[(U0' - U0) + beta (S' - S)] + 1/2 |z|^2 - 1/2 |w|^2 - ln u,
 *     w = Lc^-1 (phi - mu) of the CURRENT state (forward substitution; after an
 *     accepted move w = z), u from the ACC stream; accept iff g > 0.
 * Same outputs / slot keying as orc_mutate.
 * ---------------------------------------------------------------------- */
void orc_irmh_mutate(double* phi, double* S, double* U0, int N, int L,
                     double m0sq, double lam, const double* mu,
                     const double* Lc, double beta, uint64_t seed, uint32_t t0,
                     int k, uint8_t* accept_out, double* margin_out,
                     const int32_t* slots) {
  int V = L * L;
#pragma omp parallel
  {
    double* f = (double*)malloc(sizeof(double) * V);
    double* fp = (double*)malloc(sizeof(double) * V);
    double* z = (double*)malloc(sizeof(double) * V);
    double* w = (double*)malloc(sizeof(double) * V);
#pragma omp for
    for (int i = 0; i < N; ++i) {
      orc_get_field(phi, N, V, i, f);
      double Si = S[i], Ui = U0[i];
      const uint32_t slot = slots ? (uint32_t)slots[i] : (uint32_t)i;
      /* w = Lc^-1 (f - mu) */
      double W2 = 0.0;
      for (int x = 0; x < V; ++x) {
        double a = f[x] - mu[x];
        for (int y = 0; y < x; ++y) a -= Lc[(size_t)x * V + y] * w[y];
        w[x] = a / Lc[(size_t)x * V + x];
        W2 += w[x] * w[x];
      }
      for (int j = 0; j < k; ++j) {
        uint32_t t = t0 + (uint32_t)j;
        orc_normals(seed, ORC_TAG_PROP, t, slot, V, z);
        double Z2 = 0.0;
        for (int x = 0; x < V; ++x) {
          double a = mu[x];
          for (int y = 0; y <= x; ++y) a += Lc[(size_t)x * V + y] * z[y];
          fp[x] = a;
          Z2 += z[x] * z[x];
        }
        double Sp = orc_action_field(fp, L, m0sq, lam, NULL);
        double Up = orc_u0_field(fp, V);
        double u = orc_uniform(seed, ORC_TAG_ACC, t, slot);
        double gm = -((Up - Ui) + beta * (Sp - Si)) + 0.5 * Z2 - 0.5 * W2 - log(u);
        int acc = gm > 0.0;
        if (margin_out) margin_out[(size_t)j * N + i] = gm;
        if (accept_out) accept_out[(size_t)j * N + i] = (uint8_t)acc;
        if (acc) {
          memcpy(f, fp, sizeof(double) * V);
          Si = Sp; Ui = Up; W2 = Z2;
        }
      }
      orc_put_field(phi, N, V, i, f);
      S[i] = Si;
      U0[i] = Ui;
    }
    free(f); free(fp); free(z); free(w);
  }
}

/* SMC with IRMH rejuvenation: orc_smc_run with step 2(e) replaced by k IRMH
 * steps from N(mu, Sigma) of the resampled particles (A4 jitter rule). */
int orc_smc_irmh_run(int L, double m0sq, double lam, int N, uint64_t seed, int k,
                     double ess_target, int max_temps, double* phi, double* S,
                     double* U0, double* logZ_out, double* info) {
  int V = L * L;
  double* tmp = (double*)malloc(sizeof(double) * (size_t)V * N);
  double* Sigma = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* Lc = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* mu = (double*)malloc(sizeof(double) * V);
  float* w = (float*)malloc(sizeof(float) * N);
  int32_t* anc = (int32_t*)malloc(sizeof(int32_t) * N);
  uint8_t* acc = (uint8_t*)malloc((size_t)k * N);
  orc_init_particles(seed, N, V, phi);
  orc_action_batch(phi, N, L, m0sq, lam, S, U0, NULL);
  double beta = 0.0, logZ = 0.0;
  uint32_t t = 0;
  int T = 0, rc = 0;
  while (beta < 1.0 && T < max_temps) {
    int final;
    double delta = orc_next_delta(S, N, beta, ess_target, &final);
    double beta_new = final ? 1.0 : beta + delta;
    double ess = orc_ess_frac(S, N, delta);
    double dlz = orc_reweight(S, N, delta, w);
    logZ += dlz;
    uint32_t U = orc_word0(seed, ORC_TAG_RESAMPLE, (uint32_t)T, 0u);
    orc_resample_systematic(w, N, U, anc);
    orc_gather(phi, N, V, anc, tmp);
    memcpy(phi, tmp, sizeof(double) * (size_t)V * N);
    orc_gather(S, N, 1, anc, tmp);  memcpy(S, tmp, sizeof(double) * N);
    orc_gather(U0, N, 1, anc, tmp); memcpy(U0, tmp, sizeof(double) * N);
    orc_covariance(phi, N, V, mu, Sigma);
    int st = orc_cov_chol(phi, N, V, Sigma, Lc);
    if (st < 0) { rc = -1; break; }
    orc_irmh_mutate(phi, S, U0, N, L, m0sq, lam, mu, Lc, beta_new, seed, t + 1, k,
                    acc, NULL, NULL);
    t += (uint32_t)k;
    double nacc = 0.0;
    for (size_t m = 0; m < (size_t)k * N; ++m) nacc += acc[m];
    if (info) {
      double* o = info + 8 * T;
      o[0] = beta_new; o[1] = delta; o[2] = ess; o[3] = dlz;
      o[4] = nacc / ((double)k * N); o[5] = 0; o[6] = st; o[7] = 0.0;
    }
    beta = beta_new;
    ++T;
  }
  *logZ_out = logZ;
  free(tmp); free(Sigma); free(Lc); free(mu); free(w); free(anc); free(acc);
  return rc < 0 ? rc : T;
}

/* ------------------------------------------------------------------------
 * NEXT row f3 -- the slice-sampling inner kernel of nested sampling
 * (PAPER.md:53(iv), :174: "slice-sampling kernel (also tuned using the
 * particle covariance)", "bracketing and shrinkage"; ref [47]).  Reading A16
 * (DESIGN.md), one step of a walker at phi with S_E(phi) < S_star:
 *   1. direction d = Lc z, z = NS_PROP-stream normals (tag 5, same keying as
 *      orc_mutate); the particle covariance sets the scale of d.
 *   2. one draw of the NS_SLICE stream (tag 7, c0 = 0): height
 *      u_h = (w0>>8 + 1) 2^-24, bracket offset u_b = (w1>>8) 2^-24, stepping-out
 *      split u_j = (w2>>8) 2^-24.  log y = -U0(phi) + ln u_h.
 *      Inside(t) <=> S_E(phi + t d) < S_star and -U0(phi + t d) > log y
 *      (slice of the reference density N(0,I) under the hard constraint).
 *   3. bracket l = -width u_b, r = l + width; stepping out (Neal 2003, Fig. 3):
 *      J = floor(m_expand u_j), K = m_expand - 1 - J; while J > 0 and Inside(l):
 *      l -= width, --J; while K > 0 and Inside(r): r += width, --K.
 *   4. shrinkage: for i = 0 .. max_shrink-1: u_i = ((w>>8) + 0.5) 2^-24 from
 *      word i%4 of draw c0 = 1 + i/4; t = l + u_i (r - l); if Inside(t): move,
 *      phi <- phi + t d, stop; else l = t if t < 0 else r = t.  No move after
 *      max_shrink failures (t = 0).
 * Outputs per (step, walker): t (0 = no move), expansions, shrinkages used and
 * amb = the smallest |S_star - S_E| or |-U0 - log y| met in any Inside test
 * (how close the nearest decision was to flipping).
 * ---------------------------------------------------------------------- */
#define ORC_TAG_NS_SLICE 7u

typedef struct {
  const double* f; const double* d; double* tmp;
  int L; double m0sq, lam, S_star, logy, amb, S_last, U_last;
} orc_slice_ctx;

static int orc_slice_inside(orc_slice_ctx* c, double t) {
  int V = c->L * c->L;
  for (int x = 0; x < V; ++x) c->tmp[x] = c->f[x] + t * c->d[x];
  double Sx = orc_action_field(c->tmp, c->L, c->m0sq, c->lam, NULL);
  double Ux = orc_u0_field(c->tmp, V);
  double a1 = fabs(c->S_star - Sx), a2 = fabs(-Ux - c->logy);
  if (a1 < c->amb) c->amb = a1;
  if (a2 < c->amb) c->amb = a2;
  c->S_last = Sx; c->U_last = Ux;
  return Sx < c->S_star && -Ux > c->logy;
}

void orc_slice_walk(double* phi, double* S, double* U0, int N, int L,
                    double m0sq, double lam, const double* Lc, double width,
                    int m_expand, int max_shrink, double S_star, uint64_t seed,
                    uint32_t t0, int k, double* t_out, int32_t* nexp_out,
                    int32_t* nshr_out, double* amb_out, const int32_t* slots) {
  int V = L * L;
#pragma omp parallel
  {
    double* f = (double*)malloc(sizeof(double) * V);
    double* d = (double*)malloc(sizeof(double) * V);
    double* z = (double*)malloc(sizeof(double) * V);
    double* tmp = (double*)malloc(sizeof(double) * V);
#pragma omp for
    for (int i = 0; i < N; ++i) {
      orc_get_field(phi, N, V, i, f);
      double Si = S[i], Ui = U0[i];
      const uint32_t slot = slots ? (uint32_t)slots[i] : (uint32_t)i;
      for (int j = 0; j < k; ++j) {
        uint32_t t = t0 + (uint32_t)j;
        orc_normals(seed, ORC_TAG_NS_PROP, t, slot, V, z);
        for (int x = 0; x < V; ++x) {
          double a = 0.0;
          for (int y = 0; y <= x; ++y) a += Lc[(size_t)x * V + y] * z[y];
          d[x] = a;
        }
        uint32_t w[4];
        orc_draw(seed, ORC_TAG_NS_SLICE, t, slot, 0u, w);
        double u_h = ((double)(w[0] >> 8) + 1.0) * (1.0 / 16777216.0);
        double u_b = (double)(w[1] >> 8) * (1.0 / 16777216.0);
        double u_j = (double)(w[2] >> 8) * (1.0 / 16777216.0);
        orc_slice_ctx c = {f, d, tmp, L, m0sq, lam, S_star, -Ui + log(u_h), INFINITY, Si, Ui};
        double l = -width * u_b, r = l + width;
        int J = (int)floor((double)m_expand * u_j), K = m_expand - 1 - J, nexp = 0;
        while (J > 0 && orc_slice_inside(&c, l)) { l -= width; --J; ++nexp; }
        while (K > 0 && orc_slice_inside(&c, r)) { r += width; --K; ++nexp; }
        double tacc = 0.0;
        int nshr = 0;
        for (int m = 0; m < max_shrink; ++m) {
          if ((m & 3) == 0) orc_draw(seed, ORC_TAG_NS_SLICE, t, slot, 1u + (uint32_t)(m >> 2), w);
          double u = ((double)(w[m & 3] >> 8) + 0.5) * (1.0 / 16777216.0);
          double tt = l + u * (r - l);
          if (orc_slice_inside(&c, tt)) {
            tacc = tt;
            for (int x = 0; x < V; ++x) f[x] += tt * d[x];
            Si = c.S_last; Ui = c.U_last;
            break;
          }
          ++nshr;
          if (tt < 0.0) l = tt; else r = tt;
        }
        size_t o = (size_t)j * N + i;
        if (t_out) t_out[o] = tacc;
        if (nexp_out) nexp_out[o] = nexp;
        if (nshr_out) nshr_out[o] = nshr;
        if (amb_out) amb_out[o] = c.amb;
      }
      orc_put_field(phi, N, V, i, f);
      S[i] = Si;
      U0[i] = Ui;
    }
    free(f); free(d); free(z); free(tmp);
  }
}

/* ------------------------------------------------------------------------
 * NEXT row f4 -- global Z2 flips inside the particle method (PAPER.md:55,
 * :85: "It is also possible to simply encode the Z2 symmetry into particle
 * methods"; :176 describes the move for the AHMC control).  Reading A17
 * (DESIGN.md): S_E and U0 are even in phi, so phi -> -phi is a symmetry of every
 * p_beta and the flip is always accepted.  After the resampling of temperature
 * T, the particle in slot j is flipped iff the top bit of word 0 of the draw
 * (tag 8, t = T, slot j) is set.  S_E and U0 are unchanged.
 * ---------------------------------------------------------------------- */
#define ORC_TAG_Z2 8u
void orc_z2_flip(double* phi, int N, int V, uint64_t seed, uint32_t T,
                 uint8_t* flipped) {
  for (int j = 0; j < N; ++j) {
    uint32_t w = orc_word0(seed, ORC_TAG_Z2, T, (uint32_t)j);
    int f = (int)(w >> 31);
    if (flipped) flipped[j] = (uint8_t)f;
    if (f)
      for (int x = 0; x < V; ++x) phi[(size_t)x * N + j] = -phi[(size_t)x * N + j];
  }
}

/* orc_smc_run with the Z2 flip of reading A17 after every resampling. */
int orc_smc_run_z2(int L, double m0sq, double lam, int N, uint64_t seed, int k,
                   double ess_target, double step_scale, int max_temps,
                   double* phi, double* S, double* U0, double* logZ_out,
                   double* info) {
  int V = L * L;
  double s = step_scale > 0.0 ? step_scale : 2.38 / sqrt((double)V);
  double* tmp = (double*)malloc(sizeof(double) * (size_t)V * N);
  double* Sigma = (double*)malloc(sizeof(double) * (size_t)V * V);
  double* Lc = (double*)malloc(sizeof(double) * (size_t)V * V);
  float* w = (float*)malloc(sizeof(float) * N);
  int32_t* anc = (int32_t*)malloc(sizeof(int32_t) * N);
  uint8_t* acc = (uint8_t*)malloc((size_t)k * N);
  orc_init_particles(seed, N, V, phi);
  orc_action_batch(phi, N, L, m0sq, lam, S, U0, NULL);
  double beta = 0.0, logZ = 0.0;
  uint32_t t = 0;
  int T = 0, rc = 0;
  while (beta < 1.0 && T < max_temps) {
    int final;
    double delta = orc_next_delta(S, N, beta, ess_target, &final);
    double beta_new = final ? 1.0 : beta + delta;
    double ess = orc_ess_frac(S, N, delta);
    double dlz = orc_reweight(S, N, delta, w);
    logZ += dlz;
    uint32_t U = orc_word0(seed, ORC_TAG_RESAMPLE, (uint32_t)T, 0u);
    orc_resample_systematic(w, N, U, anc);
    orc_gather(phi, N, V, anc, tmp);
    memcpy(phi, tmp, sizeof(double) * (size_t)V * N);
    orc_gather(S, N, 1, anc, tmp);  memcpy(S, tmp, sizeof(double) * N);
    orc_gather(U0, N, 1, anc, tmp); memcpy(U0, tmp, sizeof(double) * N);
    orc_z2_flip(phi, N, V, seed, (uint32_t)T, NULL);
    int st = orc_cov_chol(phi, N, V, Sigma, Lc);
    if (st < 0) { rc = -1; break; }
    orc_mutate(phi, S, U0, N, L, m0sq, lam, Lc, s, beta_new, ORC_MODE_SMC, 0.0,
               seed, ORC_TAG_PROP, ORC_TAG_ACC, t + 1, k, acc, NULL, NULL, NULL);
    t += (uint32_t)k;
    double nacc = 0.0;
    for (size_t m = 0; m < (size_t)k * N; ++m) nacc += acc[m];
    if (info) {
      double* o = info + 8 * T;
      o[0] = beta_new; o[1] = delta; o[2] = ess; o[3] = dlz;
      o[4] = nacc / ((double)k * N); o[5] = 0; o[6] = st; o[7] = 0.0;
    }
    beta = beta_new;
    ++T;
  }
  *logZ_out = logZ;
  free(tmp); free(Sigma); free(Lc); free(w); free(anc); free(acc);
  return rc < 0 ? rc : T;
}
