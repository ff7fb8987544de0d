/*
 * sail_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, serial-per-walker CPU implementation (fp64, compile with -ffp-contract=off) of
 * the hot path of SAIL (arXiv 1609.07936): kernel table, forward transform, residue, the
 * sum-rule-preserving local move with Metropolis acceptance, the sweep with the update-amplitude
 * heuristic, the full-residual resync and imprinted branching.  Every function cites the passage
 * of /root/reference/PAPER.md it follows (PAPER.md:<line>, equation) and, where the paper is
 * silent or garbled, the reading taken in DESIGN.md §2 (G* / B* numbers as in SURVEY.md §8c).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  It shares no code with paper_1609_07936_b200/csrc (the CUDA
 * path): no common header, table generator or helper.  The two sides implement the same
 * counter-based generator (Philox4x32-10) independently.
 *
 * Pins (tests/test_oracle_*.py, run with -m "not gpu"):
 *   orc_philox4x32_10   published known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   orc_kernel_table    adaptive quadrature of the rectangle; flat-spectrum closed form
 *   orc_forward         Simpson F of the double Lorentzian, O(domega^2) convergence; M(0)=c_0 A
 *   orc_chi2            brute force on tiny grids
 *   orc_move            sum-rule invariance 1e-13, dM_0 = 0, homothety identity, incremental
 *                       vs from-scratch chi^2, Metropolis frequency exp(-D/T), T->0 / T->inf
 *   orc_amp_factor      Eq. 30 special values (y = a^2 for p=1, m=2)
 *   orc_branch          sum m = W, E[m] = w, t=1 copy / t=0 no-op, A,B preserved
 *   orc_branch_fraction_T  zeros(T) = 0 as T -> inf and grows as T falls; the T found brackets the target count
 *                       (zeros(T) >= n0 > zeros(T (1 + 1e-9))); the bracketing path itself (B6) is unpinned
 *   orc_stencil         cosine (DCT-II) modes are eigenvectors with eigenvalue 1 - 2s(1 - cos(pi n/N));
 *                       sum a kept, sum a w^m shifted by s domega (a_0 - a_{N-1}); s = 0 identity
 *   orc_smooth          A, B restored to 1e-13, positivity; the clamp branch: no negative coefficient, factor 0 at the
 *                       clamped end bin, sum a kept, B moved towards its target; the choice of renormalisation (S2)
 *                       itself is unpinned
 * Parity unpinned (paper silent; inputs identical on both sides): the width/shape of the
 * random move rho (eta, uniform), y_min, the acceptance window of Eq. 30, the comb choice of xi.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_TWO_PI 6.283185307179586476925286766559

/* ---------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon et al., SC'11).  The paper never mentions its RNG (reading G14):
 * key = (seed_lo, seed_hi), counter = (walker slot, absolute sweep, move, stream id).
 * ------------------------------------------------------------------------------------- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* uniform on (0,1) from 32 bits: (x + 0.5) * 2^-32, never 0 or 1 (reading G14) */
static double orc_u01(uint32_t x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

/* ---------------------------------------------------------------------------------------
 * O1  kernel table, Eq. 5-8:
 *   K[k][j] = (1/2pi) int_{omega_k}^{omega_k+domega} exp(-w tau_j) dw = c_j exp(-omega_k tau_j),
 *   c_j = domega/2pi (tau_j = 0),  (1 - exp(-domega tau_j)) / (2pi tau_j) otherwise (Eq. 8),
 * with expm1 for 1-exp(-x) (reading G2).  omega[] = bin LEFT edges, uniform.
 * ------------------------------------------------------------------------------------- */
double orc_domega(int n_omega, const double *omega)
{
    return (omega[n_omega - 1] - omega[0]) / (double)(n_omega - 1);
}

void orc_cvec(int n_omega, const double *omega, int n_tau, const double *tau, double *c)
{
    double dw = orc_domega(n_omega, omega);
    for (int j = 0; j < n_tau; ++j)
        c[j] = (tau[j] == 0.0) ? dw / ORC_TWO_PI : -expm1(-dw * tau[j]) / (ORC_TWO_PI * tau[j]);
}

void orc_kernel_table(int n_omega, const double *omega, int n_tau, const double *tau, double *K)
{
    double *c = (double *)malloc(sizeof(double) * (size_t)n_tau);
    orc_cvec(n_omega, omega, n_tau, tau, c);
    for (int k = 0; k < n_omega; ++k)
        for (int j = 0; j < n_tau; ++j)
            K[(size_t)k * n_tau + j] = c[j] * exp(-omega[k] * tau[j]);
    free(c);
}

/* ---------------------------------------------------------------------------------------
 * O2  forward transform, Eq. 7: M_j = sum_k a_k K[k][j], Neumaier-compensated.
 * ------------------------------------------------------------------------------------- */
void orc_forward(int n_omega, int n_tau, const double *K, const double *a, double *M)
{
    for (int j = 0; j < n_tau; ++j) {
        double sum = 0.0, comp = 0.0;
        for (int k = 0; k < n_omega; ++k) {
            double term = a[k] * K[(size_t)k * n_tau + j];
            double t = sum + term;
            if (fabs(sum) >= fabs(term)) comp += (sum - t) + term;
            else                         comp += (term - t) + sum;
            sum = t;
        }
        M[j] = sum + comp;
    }
}

/* ---------------------------------------------------------------------------------------
 * O3  residue, Eq. 9 with error bars (reading G3):
 *   chi^2 = sum_j ((M_j - F_j)/sigma_j)^2.   sigma == NULL means sigma_j = 1 (the paper's form).
 * ------------------------------------------------------------------------------------- */
double orc_chi2(int n_tau, const double *M, const double *F, const double *sigma)
{
    double s = 0.0;
    for (int j = 0; j < n_tau; ++j) {
        double D = (M[j] - F[j]) / (sigma ? sigma[j] : 1.0);
        s += D * D;
    }
    return s;
}

/* ---------------------------------------------------------------------------------------
 * O4  start spectrum (reading G4; the paper does not say how walkers start):
 *   a_k = alpha exp(-lambda (wm_k - wm_0)), wm_k = omega_k + domega/2, lambda by bisection so
 *   that sum a_k wm_k / sum a_k = B/A (Eq. 12-15), alpha from sum a_k = A.
 * Fixed 200 bisection steps on [-lam_max, lam_max], lam_max = 700/(wm_last - wm_0).
 * Returns 0, or -1 if B/A is outside (wm_0, wm_last).
 * ------------------------------------------------------------------------------------- */
int orc_init_tilt(int n_omega, const double *omega, double A, double B, double *a)
{
    double dw = orc_domega(n_omega, omega);
    double w0 = omega[0] + 0.5 * dw, wl = omega[n_omega - 1] + 0.5 * dw;
    double target = B / A;
    if (!(target > w0 && target < wl)) return -1;
    double lam_max = 700.0 / (wl - w0), lo = -lam_max, hi = lam_max, lam = 0.0;
    for (int it = 0; it < 200; ++it) {
        lam = 0.5 * (lo + hi);
        double s0 = 0.0, s1 = 0.0;
        for (int k = 0; k < n_omega; ++k) {
            double wm = omega[k] + 0.5 * dw;
            double e = exp(-lam * (wm - w0));
            s0 += e; s1 += e * wm;
        }
        if (s1 / s0 > target) lo = lam; else hi = lam;   /* mean too high -> tilt harder */
    }
    double s0 = 0.0;
    for (int k = 0; k < n_omega; ++k) {
        a[k] = exp(-lam * ((omega[k] + 0.5 * dw) - w0));
        s0 += a[k];
    }
    for (int k = 0; k < n_omega; ++k) a[k] *= A / s0;
    return 0;
}

/* ---------------------------------------------------------------------------------------
 * Problem description handed to the move / sweep / branch routines.
 * ------------------------------------------------------------------------------------- */
typedef struct {
    int32_t n_omega, n_tau;
    const double *omega;   /* [n_omega] bin left edges                        */
    const double *K;       /* [n_omega][n_tau] from orc_kernel_table           */
    const double *F;       /* [n_tau] data                                     */
    const double *sigma;   /* [n_tau] error bars (never NULL here; pass ones)  */
    double A, B;           /* sum constants, Eq. 12-15                         */
    double eta;            /* base move amplitude (reading G6)                 */
    int32_t amp_mode;      /* 0: y = 1 always; 1: Eq. 30                        */
    double amp_p, amp_m;   /* Eq. 30 parameters (paper: p = 1, m = 2)          */
    double y_min;          /* floor of y (reading G7)                          */
    uint32_t seed_lo, seed_hi;
    int32_t walk_len;      /* length L of the index-selection walk (section 2.3); 0 = uniform p, s (reading G11) */
    double walk_uniform;   /* fraction of moves that keep the uniform choice although L > 0 (:158 "a small fraction of
                            * the uniform distribution can be mixed in")                                            */
} orc_problem;

/* One traced move (what the parity tests compare). */
typedef struct {
    int32_t p, s;
    int32_t flags;          /* bit0 feasible (positivity passed), bit1 accepted          */
    int32_t move;
    double rho, delta_p, delta_s;
    double dchi2;           /* incremental Delta chi^2 (evaluated even if infeasible)     */
    double ln_u;            /* ln(u_acc)                                                  */
    double ap_new, as_new;  /* rho a_p + delta_p, rho a_s + delta_s                       */
    double l1;              /* tolerance scale: cancellation-aware L1 mass */
} orc_trace;

/* ---------------------------------------------------------------------------------------
 * O5  one attempted move of one walker, Eq. 17-22 + Eq. 10.
 *   1. (x0..x3) = Philox(key = seed, ctr = (walker, sweep, move, 0))
 *   2. p = (x0 N_w)>>32 ; s' = (x1 (N_w-1))>>32 ; s = s' + (s' >= p)   (uniform p, s != p; G11)
 *   3. u_rho, u_acc ; rho = 1 - y eta (2 u_rho - 1)                       (G6)
 *   4. delta_p = (1-rho)(B - A wm_s)/((p-s) domega), delta_s likewise    (Eq. 20-21)
 *   5. positivity: rho > 0, rho a_p + delta_p >= 0, rho a_s + delta_s >= 0
 *   6. d_j = ((rho-1) M_j + delta_p K_pj + delta_s K_sj)/sigma_j  (Eq. 22 with c_j, G1),
 *      D_j = (M_j - F_j)/sigma_j,  dchi2 = sum_j d_j (d_j + 2 D_j)
 *   7. accept iff feasible and dchi2/T + ln u_acc < 0                    (Eq. 10, Metropolis)
 *   8. on accept: a_k <- rho a_k (all k), a_p, a_s <- step-5 values, M_j <- rho M_j + ..., chi2 += dchi2
 * Returns flags.  tr may be NULL.
 * ------------------------------------------------------------------------------------- */
int orc_move(const orc_problem *P, int64_t walker, int64_t sweep, int32_t move, double T, double y,
             double *a, double *M, double *chi2, orc_trace *tr)
{
    const int n_omega = P->n_omega, n_tau = P->n_tau;
    const double dw = orc_domega(n_omega, P->omega);
    uint32_t ctr[4] = { (uint32_t)walker, (uint32_t)sweep, (uint32_t)move, 0u };
    uint32_t key[2] = { P->seed_lo, P->seed_hi };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);

    int32_t p = (int32_t)(((uint64_t)x[0] * (uint64_t)n_omega) >> 32);
    int32_t s = (int32_t)(((uint64_t)x[1] * (uint64_t)(n_omega - 1)) >> 32);
    /* Section 2.3 (reading F4): "a truncated Markov walk in the space of the
     * spectral coefficients" selects p and s; zero length = uniform, infinite length = P(j) = a_j / A.  The walk is
     * Metropolis on the bin index with uniform candidates: j <- c if u a_j < a_c.  Step l = 0 .. L-1 draws
     * Philox(ctr = (walker, sweep, move, 2 + l)) = (candidate for p, u for p, candidate for s, u for s); the whole
     * p-walk runs first, then s starts from its uniform draw on the bins other than the final p and walks on those. */
    /* the admixture: one more uniform, word 0 of Philox(ctr = (walker, sweep, move, 2 + L)); below walk_uniform the
     * move keeps its uniform indices */
    int walk_len = P->walk_len;
    if (walk_len > 0 && P->walk_uniform > 0.0) {
        uint32_t cm[4] = { (uint32_t)walker, (uint32_t)sweep, (uint32_t)move, (uint32_t)(2 + P->walk_len) }, xm[4];
        orc_philox4x32_10(cm, key, xm);
        if (orc_u01(xm[0]) < P->walk_uniform) walk_len = 0;
    }
    for (int l = 0; l < walk_len; ++l) {
        uint32_t cw[4] = { (uint32_t)walker, (uint32_t)sweep, (uint32_t)move, (uint32_t)(2 + l) }, xw[4];
        orc_philox4x32_10(cw, key, xw);
        int32_t c = (int32_t)(((uint64_t)xw[0] * (uint64_t)n_omega) >> 32);
        if (orc_u01(xw[1]) * a[p] < a[c]) p = c;
    }
    if (s >= p) s += 1;
    for (int l = 0; l < walk_len; ++l) {
        uint32_t cw[4] = { (uint32_t)walker, (uint32_t)sweep, (uint32_t)move, (uint32_t)(2 + l) }, xw[4];
        orc_philox4x32_10(cw, key, xw);
        int32_t c = (int32_t)(((uint64_t)xw[2] * (uint64_t)(n_omega - 1)) >> 32);
        if (c >= p) c += 1;
        if (orc_u01(xw[3]) * a[s] < a[c]) s = c;
    }
    double u_rho = orc_u01(x[2]), u_acc = orc_u01(x[3]);
    double rho = 1.0 - y * P->eta * (2.0 * u_rho - 1.0);

    double wm_p = P->omega[p] + 0.5 * dw, wm_s = P->omega[s] + 0.5 * dw;
    double delta_p = (1.0 - rho) * (P->B - P->A * wm_s) / ((double)(p - s) * dw);
    double delta_s = (1.0 - rho) * (P->B - P->A * wm_p) / ((double)(s - p) * dw);

    double ap_new = rho * a[p] + delta_p;
    double as_new = rho * a[s] + delta_s;
    int feasible = (rho > 0.0) && (ap_new >= 0.0) && (as_new >= 0.0);

    const double *Kp = P->K + (size_t)p * n_tau, *Ks = P->K + (size_t)s * n_tau;
    double dchi2 = 0.0, l1 = 0.0;
    for (int j = 0; j < n_tau; ++j) {
        double t1 = (rho - 1.0) * M[j], t2 = delta_p * Kp[j], t3 = delta_s * Ks[j];
        double d = (t1 + t2 + t3) / P->sigma[j];
        double D = (M[j] - P->F[j]) / P->sigma[j];
        dchi2 += d * (d + 2.0 * D);
        /* tolerance scale: rounding of the three cancelling terms of d_j and of M_j - F_j */
        double mass_d = (fabs(t1) + fabs(t2) + fabs(t3)) / P->sigma[j];
        double mass_D = (fabs(M[j]) + fabs(P->F[j])) / P->sigma[j];
        l1 += mass_d * (fabs(d) + 2.0 * fabs(D)) + mass_d * mass_d + 2.0 * fabs(d) * mass_D;
    }
    double ln_u = log(u_acc);
    int accepted = feasible && (dchi2 / T + ln_u < 0.0);

    if (tr) {
        tr->p = p; tr->s = s; tr->flags = (feasible ? 1 : 0) | (accepted ? 2 : 0); tr->move = move;
        tr->rho = rho; tr->delta_p = delta_p; tr->delta_s = delta_s; tr->dchi2 = dchi2;
        tr->ln_u = ln_u; tr->ap_new = ap_new; tr->as_new = as_new; tr->l1 = l1;
    }
    if (accepted) {
        for (int k = 0; k < n_omega; ++k) a[k] = rho * a[k];          /* Eq. 19 */
        a[p] = ap_new;                                                /* Eq. 17 */
        a[s] = as_new;                                                /* Eq. 18 */
        for (int j = 0; j < n_tau; ++j)                               /* Eq. 22 */
            M[j] = rho * M[j] + delta_p * Kp[j] + delta_s * Ks[j];
        *chi2 += dchi2;
    }
    return (feasible ? 1 : 0) | (accepted ? 2 : 0);
}

/* ---------------------------------------------------------------------------------------
 * Eq. 30: y = 1 if a >= p else (a/p)^m, floored at y_min (reading G7).
 * ------------------------------------------------------------------------------------- */
double orc_amp_factor(double acc_rate, double amp_p, double amp_m, double y_min)
{
    if (acc_rate >= amp_p) return 1.0;
    double y = pow(acc_rate / amp_p, amp_m);
    return y < y_min ? y_min : y;
}

/* ---------------------------------------------------------------------------------------
 * O6  one sweep ("macroupdate"): N_omega attempted moves at temperature T,
 * then y from this sweep's acceptance (per walker; reading G7).  Returns #accepted.
 * trace (may be NULL) receives n_omega records; flags8 (may be NULL) n_omega bytes.
 * ------------------------------------------------------------------------------------- */
int orc_sweep(const orc_problem *P, int64_t walker, int64_t sweep, double T,
              double *a, double *M, double *chi2, double *y, int64_t *n_feasible,
              orc_trace *trace, uint8_t *flags8)
{
    int acc = 0;
    for (int32_t m = 0; m < P->n_omega; ++m) {
        int fl = orc_move(P, walker, sweep, m, T, *y, a, M, chi2, trace ? trace + m : NULL);
        if (flags8) flags8[m] = (uint8_t)fl;
        if (fl & 2) acc++;
        if ((fl & 1) && n_feasible) (*n_feasible)++;
    }
    if (P->amp_mode == 1)
        *y = orc_amp_factor((double)acc / (double)P->n_omega, P->amp_p, P->amp_m, P->y_min);
    return acc;
}

/* ---------------------------------------------------------------------------------------
 * O7  full-residual resync (north_star item 3; not in the paper): M <- forward(a), chi2 <- O3.
 * ------------------------------------------------------------------------------------- */
void orc_resync(const orc_problem *P, int64_t W, const double *a, double *M, double *chi2)
{
    #pragma omp parallel for schedule(static)
    for (int64_t w = 0; w < W; ++w) {
        orc_forward(P->n_omega, P->n_tau, P->K, a + (size_t)w * P->n_omega, M + (size_t)w * P->n_tau);
        chi2[w] = orc_chi2(P->n_tau, M + (size_t)w * P->n_tau, P->F, P->sigma);
    }
}

/* ---------------------------------------------------------------------------------------
 * Anneal driver: sweeps sweep0 .. sweep0+n-1 for all walkers (independent chains between
 * branchings, PAPER.md:166 -> OpenMP over walkers), resync after every resync_every-th
 * absolute sweep.  Temperature T_sched[i] for sweep sweep0+i.
 *   trace_lo/hi: walkers whose per-move records are written to trace
 *                ([(w-lo)][i][n_omega] records);  flags8: [W][n][n_omega] bytes or NULL.
 *   acc_total / feas_total: per-walker running counters (may be NULL).
 * ------------------------------------------------------------------------------------- */
void orc_anneal(const orc_problem *P, int64_t W, double *a, double *M, double *chi2, double *y,
                const double *T_sched, int64_t sweep0, int64_t n, int64_t resync_every,
                int64_t *acc_total, int64_t *feas_total,
                int64_t trace_lo, int64_t trace_hi, orc_trace *trace, uint8_t *flags8)
{
    const int n_omega = P->n_omega, n_tau = P->n_tau;
    int64_t done = 0;
    while (done < n) {
        /* run up to the next resync boundary */
        int64_t chunk = n - done;
        if (resync_every > 0) {
            int64_t to_boundary = resync_every - ((sweep0 + done) % resync_every);
            if (to_boundary < chunk) chunk = to_boundary;
        }
        #pragma omp parallel for schedule(dynamic, 1)
        for (int64_t w = 0; w < W; ++w) {
            for (int64_t i = done; i < done + chunk; ++i) {
                orc_trace *tr = NULL;
                if (trace && w >= trace_lo && w < trace_hi)
                    tr = trace + ((size_t)(w - trace_lo) * n + i) * n_omega;
                uint8_t *f8 = flags8 ? flags8 + ((size_t)w * n + i) * n_omega : NULL;
                int64_t feas = 0;
                int acc = orc_sweep(P, w, sweep0 + i, T_sched[i], a + (size_t)w * n_omega,
                                    M + (size_t)w * n_tau, chi2 + w, y + w, &feas, tr, f8);
                if (acc_total) acc_total[w] += acc;
                if (feas_total) feas_total[w] += feas;
            }
        }
        done += chunk;
        if (resync_every > 0 && ((sweep0 + done) % resync_every) == 0)
            orc_resync(P, W, a, M, chi2);
    }
}

/* ---------------------------------------------------------------------------------------
 * O8  imprinted branching, Eq. 24-26 with readings B1-B5:
 *   B1  e_i = exp(-(chi2_i - chi2_min)/T), w_i = W e_i / sum e          (Delta = 1/T)
 *   B3  fixed point: E_i = floor(e_i 2^40); C = inclusive integer scan; S = C_{W-1}
 *   B2  comb: Xi = (x0 S)>>32 with x0 from Philox(ctr = (0, sweep, 0, 1));
 *       m_i = floor((C_i W + Xi)/S) - floor((C_{i-1} W + Xi)/S)         (Eq. 25 with a comb xi set,
 *       sum m = W by construction)
 *   B4  recipients {m_i = 0} in ascending index, rank r; donor extras x_i = max(m_i - 1, 0),
 *       exclusive scan X; recipient r takes the donor with X_i <= r < X_i + x_i
 *   Eq. 26  a(l1) <- t a(l2) + (1-t) a(l1); donor unchanged
 *   B5  M of the recipient recomputed by O2, chi2 by O3; y stays the recipient's.
 * Outputs: mult[W] multipliers, donor_of[W] (donor index for recipients, -1 otherwise).
 * Returns the number of recipients.
 * ------------------------------------------------------------------------------------- */
int64_t orc_branch(const orc_problem *P, int64_t W, double *a, double *M, double *chi2,
                   double T, double t_imprint, int64_t sweep, int32_t *mult, int64_t *donor_of)
{
    const int n_omega = P->n_omega, n_tau = P->n_tau;
    double cmin = chi2[0];
    for (int64_t i = 1; i < W; ++i) if (chi2[i] < cmin) cmin = chi2[i];

    uint64_t *C = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)W);
    uint64_t run = 0;
    for (int64_t i = 0; i < W; ++i) {
        double e = exp(-(chi2[i] - cmin) / T);
        run += (uint64_t)floor(e * 1099511627776.0);   /* 2^40 */
        C[i] = run;
    }
    const uint64_t S = run;

    uint32_t ctr[4] = { 0u, (uint32_t)sweep, 0u, 1u };
    uint32_t key[2] = { P->seed_lo, P->seed_hi };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    const unsigned __int128 Xi = ((unsigned __int128)x[0] * S) >> 32;

    uint64_t prev = (uint64_t)(Xi / S);                 /* = 0 */
    for (int64_t i = 0; i < W; ++i) {
        uint64_t cur = (uint64_t)(((unsigned __int128)C[i] * (uint64_t)W + Xi) / S);
        mult[i] = (int32_t)(cur - prev);
        prev = cur;
    }
    free(C);

    /* donor map (B4) */
    int64_t n_rec = 0;
    {
        int64_t donor = 0, left = 0;      /* walk donors in ascending index */
        for (int64_t i = 0; i < W; ++i) donor_of[i] = -1;
        for (int64_t i = 0; i < W; ++i) {
            if (mult[i] != 0) continue;
            while (left == 0) {           /* advance to the next donor with extras */
                while (mult[donor] < 2) donor++;
                left = mult[donor] - 1;
                if (left == 0) donor++;
            }
            donor_of[i] = donor;
            if (--left == 0) donor++;
            n_rec++;
        }
    }

    /* imprint (Eq. 26) — donors (m >= 2) and recipients (m = 0) are disjoint */
    for (int64_t i = 0; i < W; ++i) {
        if (donor_of[i] < 0) continue;
        double *ar = a + (size_t)i * n_omega;
        const double *ad = a + (size_t)donor_of[i] * n_omega;
        for (int k = 0; k < n_omega; ++k) ar[k] = t_imprint * ad[k] + (1.0 - t_imprint) * ar[k];
        orc_forward(n_omega, n_tau, P->K, ar, M + (size_t)i * n_tau);
        chi2[i] = orc_chi2(n_tau, M + (size_t)i * n_tau, P->F, P->sigma);
    }
    return n_rec;
}

/* ---------------------------------------------------------------------------------------
 * O8b  branching with a prescribed branching fraction:
 *   "Parameter Delta is found numerically such that a given fraction of walkers is assigned a zero
 *    multiplier."  Reading B6: Delta = 1/T is the smallest value on a doubling-then-bisection path for
 *   which the comb multipliers of O8 (same Philox offset for every trial value) give at least
 *   n0 = floor(fraction W + 1/2) zeros:
 *     beta_0 = 1/(chi2_max - chi2_min); bracket by doubling / halving from beta_0 (at most 200 steps)
 *     until Z(lo) < n0 <= Z(hi); 40 bisection steps on beta; T = 1/hi.
 *   orc_branch_zeros counts the zero multipliers for a given T without touching the state.
 *   Returns 0 and leaves *T_out = 0 when the population is degenerate (all chi2 equal) or n0 = 0.
 * ------------------------------------------------------------------------------------- */
int64_t orc_branch_zeros(const orc_problem *P, int64_t W, const double *chi2, double T, int64_t sweep)
{
    double cmin = chi2[0];
    for (int64_t i = 1; i < W; ++i) if (chi2[i] < cmin) cmin = chi2[i];
    uint64_t *C = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)W);
    uint64_t run = 0;
    for (int64_t i = 0; i < W; ++i) {
        run += (uint64_t)floor(exp(-(chi2[i] - cmin) / T) * 1099511627776.0);
        C[i] = run;
    }
    const uint64_t S = run;
    uint32_t ctr[4] = { 0u, (uint32_t)sweep, 0u, 1u };
    uint32_t key[2] = { P->seed_lo, P->seed_hi };
    uint32_t x[4];
    orc_philox4x32_10(ctr, key, x);
    const unsigned __int128 Xi = ((unsigned __int128)x[0] * S) >> 32;
    uint64_t prev = 0;
    int64_t zeros = 0;
    for (int64_t i = 0; i < W; ++i) {
        uint64_t cur = (uint64_t)(((unsigned __int128)C[i] * (uint64_t)W + Xi) / S);
        if (cur == prev) zeros++;
        prev = cur;
    }
    free(C);
    return zeros;
}

int orc_branch_fraction_T(const orc_problem *P, int64_t W, const double *chi2, double fraction, int64_t sweep,
                          double *T_out)
{
    *T_out = 0.0;
    const int64_t n0 = (int64_t)floor(fraction * (double)W + 0.5);
    double cmin = chi2[0], cmax = chi2[0];
    for (int64_t i = 1; i < W; ++i) { if (chi2[i] < cmin) cmin = chi2[i]; if (chi2[i] > cmax) cmax = chi2[i]; }
    if (n0 <= 0 || !(cmax > cmin)) return 0;
    double lo, hi = 1.0 / (cmax - cmin);
    if (orc_branch_zeros(P, W, chi2, 1.0 / hi, sweep) >= n0) {
        lo = 0.5 * hi;
        for (int it = 0; it < 200 && orc_branch_zeros(P, W, chi2, 1.0 / lo, sweep) >= n0; ++it) { hi = lo; lo = 0.5 * lo; }
    } else {
        lo = hi; hi = 2.0 * hi;
        int it = 0;
        for (; it < 200 && orc_branch_zeros(P, W, chi2, 1.0 / hi, sweep) < n0; ++it) { lo = hi; hi = 2.0 * hi; }
        if (it == 200) return 0;               /* the fraction cannot be reached (e.g. n0 >= W) */
    }
    for (int it = 0; it < 40; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (orc_branch_zeros(P, W, chi2, 1.0 / mid, sweep) >= n0) hi = mid; else lo = mid;
    }
    *T_out = 1.0 / hi;
    return 1;
}

/* ---------------------------------------------------------------------------------------
 * O9  smoothing, Eq. 27-29, SURVEY 8(f) row f3.
 *   Eq. 27: a_j <- s a_{j-1} + (1 - 2s) a_j + s a_{j+1},  0 < j < N-1
 *   Eq. 28: a_0 <- (1 - s) a_0 + s a_1          Eq. 29: a_{N-1} <- (1 - s) a_{N-1} + s a_{N-2}
 * Reading S1: the stencil is applied to all bins simultaneously (every right-hand side is the OLD
 * spectrum), terms added in the order written.  orc_stencil is exactly this and nothing else.
 * The stencil keeps sum a (Eq. 12) and shifts sum a w^m (Eq. 14) by s domega (a_0 - a_{N-1}); the
 * paper asks for "an additional renormalization" (:197) without saying which.  Reading S2:
 * multiply by a linear tilt about the new mean frequency,
 *      a_k <- a_k (1 + kappa (w^m_k - wbar)),  wbar = B'/A',  kappa = (B - B') / sum_k a_k (w^m_k - wbar)^2,
 * which leaves A' untouched, restores B and, kappa being O(s / N), keeps every coefficient positive.
 * (B is the problem's second sum, P->B.)  Afterwards the model and residue are recomputed (O7).
 * ------------------------------------------------------------------------------------- */
void orc_stencil(int n, double s, const double *a, double *out)
{
    const double c = 1.0 - 2.0 * s, e = 1.0 - s;
    if (n == 1) { out[0] = a[0]; return; }
    out[0] = e * a[0] + s * a[1];
    for (int j = 1; j < n - 1; ++j) out[j] = (s * a[j - 1] + c * a[j]) + s * a[j + 1];
    out[n - 1] = e * a[n - 1] + s * a[n - 2];
}

void orc_smooth(const orc_problem *P, int64_t W, double s, double *a, double *M, double *chi2)
{
    const int n = P->n_omega;
    const double half = 0.5 * orc_domega(n, P->omega);
    #pragma omp parallel for schedule(static)
    for (int64_t w = 0; w < W; ++w) {
        double *row = a + (size_t)w * n;
        double *tmp = (double *)malloc((size_t)n * sizeof(double));
        orc_stencil(n, s, row, tmp);
        double A1 = 0.0, B1 = 0.0, V = 0.0;
        for (int k = 0; k < n; ++k) { A1 += tmp[k]; B1 += tmp[k] * (P->omega[k] + half); }
        const double wbar = B1 / A1;
        for (int k = 0; k < n; ++k) { const double dw = (P->omega[k] + half) - wbar; V += tmp[k] * dw * dw; }
        double kappa = (V > 0.0) ? (P->B - B1) / V : 0.0;
        /* reading S2, positivity (Eq. 10 needs a_k >= 0): the tilt factor 1 + kappa (w^m_k - wbar) is linear in k, so it
         * is smallest at one of the two end bins; kappa is clamped so that it stays >= 0 there (the second sum rule is
         * then restored only in part; s of a few percent never gets near the clamp) */
        {
            const double d_lo = (P->omega[0] + half) - wbar, d_hi = (P->omega[n - 1] + half) - wbar;
            if (1.0 + kappa * d_lo < 0.0) kappa = -1.0 / d_lo;
            if (1.0 + kappa * d_hi < 0.0) kappa = -1.0 / d_hi;
        }
        for (int k = 0; k < n; ++k) row[k] = tmp[k] * (1.0 + kappa * ((P->omega[k] + half) - wbar));
        free(tmp);
        orc_forward(n, P->n_tau, P->K, row, M + (size_t)w * P->n_tau);
        chi2[w] = orc_chi2(P->n_tau, M + (size_t)w * P->n_tau, P->F, P->sigma);
    }
}

/* number of OpenMP threads the driver will use (reported as cpu_baseline.cores) */
#ifdef _OPENMP
#include <omp.h>
int orc_num_threads(void) { return omp_get_max_threads(); }
#else
int orc_num_threads(void) { return 1; }
#endif
