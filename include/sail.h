/*
 * sail.h — C ABI of sail-b200: the B200 (sm_100a) hot path of SAIL, "simulated annealing for the
 * inverse Laplace transform" (arXiv 1609.07936; citations are /root/reference/PAPER.md:<line>).
 *
 * The calls follow the paper's problem statement (inputs N_tau, dtau, F~; omega_max, N_omega; B —
 * PAPER.md:214, :127) and BASELINE.json's north_star list:
 *     sail_create -> sail_init_walkers -> { sail_anneal | sail_branch | sail_resync }* -> sail_get
 *     -> sail_destroy.
 * Every step of the path runs in hand-written CUDA kernels; there is no CPU fallback: without a
 * usable CUDA device every call returns SAIL_ERR_CUDA.
 *
 * Conventions
 *   - plain C types only; "host" / "device" is stated for every pointer.
 *   - all functions return a status code (0 = SAIL_OK, negative = error); no exception crosses the
 *     boundary; sail_last_error() gives the text of the last error of a handle (or of create).
 *   - one handle = one CUDA stream = one thread at a time; no global state.
 *   - all floating point is IEEE binary64 ("fp64"); matrices are row-major, contiguous.
 *   - work is enqueued on the handle's stream; calls that copy to HOST memory synchronise it.
 *
 * Method summary (notation of DESIGN.md §1):
 *   spectrum of a walker: a_k >= 0 on bins [omega_k, omega_k + domega), k = 0..N_omega-1 (Eq. 3, :65)
 *   model:   M_j = sum_k a_k K_kj,  K_kj = c_j exp(-omega_k tau_j)  (Eq. 5-8, :75-88)
 *   residue: chi^2 = sum_j ((M_j - F_j)/sigma_j)^2                  (Eq. 9, :92, with error bars)
 *   sums:    A = sum_k a_k,  B = sum_k a_k (omega_k + domega/2)      (Eq. 12-15, :111-121)
 */
#ifndef SAIL_B200_H
#define SAIL_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SAIL_ABI_VERSION 1

/* every function below is exported with default visibility; everything else in the library is hidden */
#if defined(__GNUC__)
#define SAIL_API __attribute__((visibility("default")))
#else
#define SAIL_API
#endif

enum {
    SAIL_OK        = 0,
    SAIL_ERR_ARG   = -1,  /* NULL / out-of-range argument, unsupported size                       */
    SAIL_ERR_GRID  = -2,  /* omega or tau grid not uniform (rel. deviation > 1e-12) or not ascending */
    SAIL_ERR_ALLOC = -3,  /* workspace too small / device allocation failed                       */
    SAIL_ERR_CUDA  = -4,  /* no device, or a CUDA runtime error (text in sail_last_error)          */
    SAIL_ERR_STATE = -5   /* call order violated (e.g. anneal before init_walkers)               */
};

typedef struct sail_handle sail_t;

/* Device / memory configuration of a handle. */
typedef struct {
    int32_t device;           /* CUDA device ordinal                                               */
    int32_t reserved;
    void   *stream;           /* cudaStream_t to enqueue on (e.g. torch's current stream); NULL = default stream */
    void   *workspace;        /* DEVICE pointer to caller-owned scratch (e.g. a torch uint8 tensor),
                                 256-byte aligned, or NULL: the library then cudaMallocs its own   */
    size_t  workspace_bytes;  /* size of workspace; must be >= sail_workspace_bytes(...)           */
    int64_t max_walkers;      /* capacity W_max the handle is sized for                            */
} sail_config;

/* Bytes of device memory a handle needs for (n_omega, n_tau, max_walkers). */
SAIL_API size_t sail_workspace_bytes(int32_t n_omega, int32_t n_tau, int64_t max_walkers);

/*
 * sail_create — define the inverse problem (N_tau, dtau, F~, omega_max, N_omega).
 *   omega  HOST [n_omega]  bin LEFT edges omega_k = omega_0 + k domega, uniform, omega_0 >= 0 (Eq. 3)
 *   tau    HOST [n_tau]    tau_j = tau_0 + j dtau, uniform, tau_0 >= 0 (Eq. 2, :61)
 *   F      HOST [n_tau]    correlation data F~(tau_j)
 *   sigma  HOST [n_tau]    error bars > 0, or NULL for sigma = 1 (the paper's unweighted Eq. 9)
 * Inputs are copied; the caller keeps ownership.  Builds the device tables (c_j, exp(-omega_k tau_j),
 * weights (c_j/sigma_j)^2).  Limits of this version: 2 <= n_omega <= 8192 (the sweep kernel keeps two n_omega-sized
 * tables and the start table in the 227 KB of shared memory of an SM; it runs fewer warps per SM above ~4000 bins),
 * 1 <= n_tau <= 512 (16 tau-points per lane in registers); sail_smooth needs n_omega <= 2048.
 * Errors: SAIL_ERR_ARG, SAIL_ERR_GRID (the method is defined on uniform grids only, Eq. 2-3, 7),
 * SAIL_ERR_ALLOC, SAIL_ERR_CUDA.  *out is NULL on error.
 */
SAIL_API int sail_create(sail_t **out, const double *omega, int32_t n_omega, const double *tau, int32_t n_tau,
                const double *F, const double *sigma, const sail_config *cfg);

/*
 * sail_init_walkers — start W Markov walkers with sum constants A, B (Eq. 12-16).
 *   mode 0: every walker = the exponential-tilt spectrum a_k ~ exp(-lambda omega_k^m) that meets both
 *           sum rules (reading G4; the paper does not say how walkers start); spectra ignored.
 *   mode 1: spectra HOST [W][n_omega] given by the caller (must be >= 0; sums are NOT re-normalised;
 *           A and B are the constants the moves will preserve).
 *   seed:   Philox4x32-10 key for all later random draws of this handle.
 * Computes M, chi^2; resets the absolute sweep counter to 0, y = 1, counters = 0.
 * Errors: SAIL_ERR_ARG (W < 1 or > max_walkers, B/A outside the grid, negative input).
 */
SAIL_API int sail_init_walkers(sail_t *h, int64_t W, double A, double B, uint64_t seed, int32_t mode,
                      const double *spectra);

/* One traced move (parity tests): written by sail_anneal for walkers in [trace_lo, trace_hi). */
typedef struct {
    int32_t p, s;            /* updated bins (Eq. 17-18)                                           */
    int32_t flags;           /* bit0 feasible (positivity passed, :143), bit1 accepted, bit2 dchi2 evaluated */
    int32_t move;            /* move index within the sweep                                        */
    double  rho;             /* the paper's random scale factor r of Eq. 17-19                     */
    double  delta_p, delta_s;/* Eq. 20-21                                                          */
    double  dchi2;           /* incremental Delta chi^2 (valid if bit2)                            */
    double  thr;             /* acceptance threshold -T ln(u_acc): accepted iff feasible && dchi2 < thr */
    double  ap_new, as_new;  /* rho a_p + delta_p, rho a_s + delta_s                               */
} sail_trace_rec;

/* Parameters of sail_anneal. */
typedef struct {
    double  eta;             /* base amplitude: rho = 1 - y eta (2u - 1), requires 0 < eta < 1 (reading G6) */
    int32_t amp_mode;        /* 0: y = 1;  1: Eq. 30 from the previous sweep's acceptance  */
    int32_t reserved0;       /* must be 0 (there is one sweep-kernel form: DESIGN.md 6.1)                 */
    double  amp_p, amp_m;    /* Eq. 30 parameters (paper: p = 1, m = 2, :222)                      */
    double  y_min;           /* floor of y (reading G7), e.g. 1e-6                                  */
    int64_t resync_every;    /* full-residual resync after every such absolute sweep; 0 = never    */
    int64_t trace_lo, trace_hi;  /* walkers whose moves are traced; lo == hi: none                 */
    sail_trace_rec *trace;   /* DEVICE [(hi-lo)][n_sweeps][n_omega] or NULL                        */
    uint8_t *flags;          /* DEVICE [W][n_sweeps][n_omega] per-move flag bytes, or NULL         */
    int32_t walk_length;     /* section 2.3 (:156-158): p and s by a truncated Markov walk of this many steps on the
                              * current spectrum (j <- uniform candidate c if u a_j < a_c); 0 = uniform p, s.  Every
                              * lane of the batch walks its own move; the moves behind an accepted one walk again.   */
    int32_t reserved;
    double  walk_uniform;    /* :158 "a small fraction of the uniform distribution can be mixed in": this fraction
                              * of the moves keeps its uniform p, s although walk_length > 0; in [0, 1]              */
} sail_anneal_params;

/*
 * sail_anneal — n_sweeps sweeps ("macroupdates", :148, :218) of N_omega attempted moves per walker:
 * proposal (uniform p, s != p; rho; Eq. 20-21), positivity rejection (:143), incremental
 * Delta chi^2 over all tau (Eq. 22 + Eq. 9), Metropolis acceptance at T (Eq. 10), Eq. 30 update of
 * y after each sweep.  T_schedule HOST [n_sweeps]: temperature of sweep (sweep_counter + i).  The
 * absolute sweep counter continues across calls, so splitting a run does not change the random
 * stream (Philox counter = (walker, sweep, move, 0)).  Asynchronous on the stream.
 */
SAIL_API int sail_anneal(sail_t *h, const double *T_schedule, int64_t n_sweeps, const sail_anneal_params *p);

/* Results of one branching event. */
typedef struct {
    int64_t n_recipients;    /* walkers with multiplier 0 that were imprinted                      */
    int32_t max_multiplier;
    int32_t reserved;
    double  chi2_min;
} sail_branch_info;

/*
 * sail_branch — one imprinted-branching event (Eq. 24-26, :166-182; readings B1-B5):
 * weights exp(-(chi^2 - chi^2_min)/T) normalised to W, integer multipliers by a comb over the
 * fixed-point prefix sum (sum m = W exactly), recipients (m = 0) take t*donor + (1-t)*self for
 * spectrum and model, their chi^2 is recomputed.  mult_out HOST [W] int32 or NULL; donor_out HOST
 * [W] int64 (-1 for non-recipients) or NULL; info HOST or NULL.  Synchronises the stream when any
 * output is requested.
 */
SAIL_API int sail_branch(sail_t *h, double T, double t_imprint, sail_branch_info *info, int32_t *mult_out,
                int64_t *donor_out);

/*
 * sail_branch_fraction — the paper's own way of fixing the branching strength (:174, :220): "Delta is found
 * numerically such that a given fraction of walkers is assigned a zero multiplier" (the paper branches a quarter of
 * the walkers).  The inverse temperature Delta = 1/T of sail_branch is searched on the device, inside the kernel that
 * builds the multiplier plan (bracketing from 1/(chi2_max - chi2_min), then 40 bisection steps; every trial is one pass
 * of the multiplier chain with the same comb offset, reading B6), for the smallest value that gives at least
 * floor(fraction W + 1/2) zeros; then the event runs at that temperature: two kernel launches in all.  *T_found (HOST,
 * may be NULL) receives it; 0 means no event happened (all residues equal, or fraction W rounds to 0).  Other arguments
 * as sail_branch.  Synchronises the stream only when an output is requested.
 */
SAIL_API int sail_branch_fraction(sail_t *h, double fraction, double t_imprint, double *T_found, sail_branch_info *info,
                                  int32_t *mult_out, int64_t *donor_out);

/* sail_resync — recompute M = a K (dense W x N_omega x N_tau contraction) and chi^2 for all walkers. */
SAIL_API int sail_resync(sail_t *h);

/*
 * sail_smooth — the smoothing step between blocks (Eq. 27-29): every walker's spectrum goes through
 * the three-point stencil a_j <- s a_{j-1} + (1 - 2s) a_j + s a_{j+1} (reflecting end bins, all bins at once), the
 * second sum rule the stencil violates (:197) is restored by a linear tilt about the mean frequency (DESIGN.md
 * reading S2), then model and residue are recomputed as in sail_resync.  0 <= s <= 0.5 (the paper uses a few
 * percent); n_omega <= 2048.  Asynchronous on the stream.
 */
SAIL_API int sail_smooth(sail_t *h, double s);

/*
 * sail_chi2_stats — the two population statistics the self-cooling schedule feeds on: the smallest
 * and the mean residue over the W walkers, HOST outputs (either may be NULL).  Fixed summation order: bit-reproducible.
 * Synchronises the stream.
 */
SAIL_API int sail_chi2_stats(sail_t *h, double *chi2_min, double *chi2_mean);

/*
 * sail_chi2_stats_static — the same two statistics (smallest and mean residue) for callers that must
 * not allocate device memory and have no handle whose workspace they could borrow.
 *
 * Who that is.  A handle belongs to one thread at a time, so a second thread that watches an anneal in progress (a
 * progress monitor, a stopping rule, a logger on its own stream) works on a COPY of the residues — e.g. the tensor it
 * got from sail_get(..., on_device = 1) — and cannot touch the handle or its workspace.  That thread cannot call
 * cudaMalloc / cudaFree either: both wait for the whole device, and a sweep-kernel launch of the large configurations
 * runs for seconds, so one such call stalls the monitor for that long (and cudaFree stalls the anneal's stream too).
 * The same holds for a process in which a framework's caching allocator (torch's) already owns all of HBM: a raw
 * cudaMalloc from this library then fails although the framework still has free blocks.
 *
 * What it does instead.  The per-CTA partial sums and minima go to a fixed array that is part of the library image
 * (a file-scope __device__ array of SAIL_STATS_STATIC_SCRATCH_BYTES = 4096 bytes; every GPU that loads the library
 * holds these 4 KB until the process exits).  No cudaMalloc, cudaFree or allocating library routine is called.
 *
 *   device  CUDA device ordinal (made current);  stream  cudaStream_t to enqueue on, NULL = default stream
 *   chi2    DEVICE [W] residues, read only;  1 <= W <= SAIL_STATS_STATIC_MAX_W (2^24).  The array holds 256 partial
 *           results whatever W is; the bound is the population size up to which a thread adds at most 256 residues one
 *           after the other, i.e. up to which the mean is good to ~600 eps relative for residues of one sign.  Larger
 *           W: SAIL_ERR_ARG with the limit in the error text — use sail_chi2_stats (handle workspace) or split the array.
 *   out     DEVICE [2], written stream-ordered: out[0] = min, out[1] = mean.  Same kernels, same summation order and
 *           so the same bits as sail_chi2_stats on the same residues.  The call does not synchronise.
 *
 * Set-up.  The first call on each device looks up the device address of the array (cudaGetSymbolAddress with that device
 * current; an error is returned as SAIL_ERR_CUDA).  Make that first call during start-up, outside any stream capture;
 * later calls only enqueue two kernels.
 * Sharing.  There is ONE array per device, shared by every call from every thread, and it keeps what the last call
 * left in it.  Nothing in it has to start at zero (each call overwrites every slot it later reads), so two calls in a
 * row need no clearing — but two calls whose kernels can run at the same time on one GPU (different streams, no event
 * between them) race on it and return garbage.  Keep the calls of one device on one stream, or order them with events.
 * Errors go to sail_last_error(NULL) of the calling thread.
 */
#define SAIL_STATS_STATIC_MAX_W ((int64_t)1 << 24)
#define SAIL_STATS_STATIC_SCRATCH_BYTES 4096
SAIL_API int sail_chi2_stats_static(int32_t device, void *stream, const double *chi2, int64_t W, double *out);

/* Parameters of sail_anneal_selfcool (readings C1-C3; the paper gives no constants beyond T_start). */
typedef struct {
    int32_t sweeps_per_block;   /* k of "each block consists of some k N_omega steps" (paper: 100, :218)          */
    int32_t n_boil, n_ramp;     /* blocks at T = chi2_ave, then blocks of the linear ramp to chi2_min (n_ramp >= 1) */
    double  T_start;            /* temperature of block 0 in units of the starting residue (paper: 10, :216)        */
    double  freeze_rate;        /* freeze-out: T = chi2_min / (1 + freeze_rate * blocks since the ramp ended)       */
    double  t_imprint;          /* imprint strength of the branching after every block (paper: 0.1, :220)          */
    double  smooth_s;           /* smoothing amplitude applied at the start of every block; 0 = no smoothing (:190, :199) */
    int32_t branch;             /* 0: no branching                                                                  */
    int32_t adapt;              /* 1: imprint strength and branching fraction of a block are multiplied by the block's
                                 * acceptance rate relative to the largest one seen so far (:184, reading B7)          */
    double  branch_fraction;    /* > 0: branch that fraction of the walkers (sail_branch_fraction; paper: 1/4, :220);
                                 * 0: branch at the block's own 1/T (sail_branch)                                   */
    const double *T_override;   /* HOST [n_blocks] or NULL: use these temperatures instead of the rule (tests)      */
    sail_anneal_params anneal;  /* eta, Eq. 30 parameters, resync period, index walk; trace and flags must be NULL       */
} sail_selfcool_params;

/*
 * sail_anneal_selfcool — n_blocks blocks of the paper's protocol (:218-220) with the self-cooling schedule of
 * section 2.4 (:160-162): before each block the residues chi2_ave, chi2_min are measured (sail_chi2_stats), the block's
 * temperature follows from them (block 0: T_start starting residues; boil: chi2_ave; ramp: linear to chi2_min; freeze-out:
 * below chi2_min, ~ 1 / blocks), then sail_smooth (if smooth_s > 0; :199 "Once the transforms are smoothed and
 * renormalized, they undergo Metropolis updates and branching"), sweeps_per_block sweeps at that temperature and
 * one sail_branch at 1/T.  The feedback loop runs on the device (statistics, rule, schedule slice, branching parameters):
 * no host synchronisation inside a block.  T_out, chi2_ave_out, chi2_min_out: HOST [n_blocks] or NULL, copied once at
 * the end (once per 4096 blocks).  Errors: SAIL_ERR_ARG also when the rule reaches T <= 0 (chi2_min is a running sum and
 * can go negative next to an exact fit; use anneal.resync_every then).  The failing block and every later block of the
 * call are no-ops on the device (no sweeps, no smoothing, no branching: the population stays as the last good block left
 * it); the error, with the block index, is reported when the call returns; T_out is 0 from that block on.
 */
SAIL_API int sail_anneal_selfcool(sail_t *h, const sail_selfcool_params *p, int64_t n_blocks, double *T_out,
                                  double *chi2_ave_out, double *chi2_min_out);

/*
 * sail_get — copy results out.  spectra [W][n_omega] (true coefficients a_k), chi2 [W]; either may
 * be NULL.  on_device = 0: HOST destinations (synchronises); 1: DEVICE destinations (stream-ordered).
 */
SAIL_API int sail_get(sail_t *h, double *spectra, double *chi2, int32_t on_device);

/* sail_get_model — M [W][n_tau] (the model correlation of each walker), HOST or DEVICE as above. */
SAIL_API int sail_get_model(sail_t *h, double *M, int32_t on_device);

/* sail_stats — HOST outputs [W], any may be NULL: accepted / evaluated move totals since init, y. */
SAIL_API int sail_stats(sail_t *h, int64_t *accepted, int64_t *evaluated, double *y);

/*
 * sail_set_walkers — state injection for sampled parity on big configs: overwrite walkers
 * [w0, w0+n) with HOST spectra [n][n_omega] and (optionally, may be NULL) HOST y [n]; M and chi^2
 * are recomputed.  sail_set_sweep sets the absolute sweep counter.
 */
SAIL_API int sail_set_walkers(sail_t *h, int64_t w0, int64_t n, const double *spectra, const double *y);
SAIL_API int sail_set_sweep(sail_t *h, int64_t sweep);

/*
 * sail_set_chi2 — overwrite the RUNNING residues chi2_0 + sum dchi2 of walkers [w0, w0+n) with HOST values (resuming
 * from a checkpoint restores the running sums bit for bit, sail_set_walkers recomputes them from the spectra; the
 * parity tests use it to give both sides identical weights input).  The model is not touched.  Synchronises.
 */
SAIL_API int sail_set_chi2(sail_t *h, int64_t w0, int64_t n, const double *chi2);

/*
 * sail_set_walker_offset — global index of this handle's walker 0 (default 0).  The Philox counter of a move is
 * (global walker index, sweep, move, stream), so a population split over several handles (one per GPU: contiguous walker
 * ranges, paper_1609_07936_b200/distributed.py) draws exactly the random numbers of the single-handle run.  Branching
 * stays per handle.  offset + max_walkers must be < 2^32.
 */
SAIL_API int sail_set_walker_offset(sail_t *h, int64_t first_walker);

/* sail_destroy — free library-owned memory (never the caller's workspace).  NULL is OK. */
SAIL_API int sail_destroy(sail_t *h);

/* Text of the last error on this handle; h == NULL: last error of sail_create in this thread. */
SAIL_API const char *sail_last_error(const sail_t *h);

/* Number of kernel launches issued by this handle so far (bench.py's gpu_launches). */
SAIL_API int64_t sail_launch_count(const sail_t *h);

/*
 * Diagnostics used by bench.py for the roofline denominators (not part of the method):
 * sail_measure_fp64_peak — runs a register-resident DFMA microbenchmark on `device`, returns
 * achieved FP64 lane-instructions per second (fused multiply-adds per second) in *dfma_per_s.
 */
SAIL_API int sail_measure_fp64_peak(int32_t device, void *stream, double *dfma_per_s);

/*
 * sail_microbench — issue rates and latencies of the units the sweep kernel (rows A2-A6) leans on, measured on
 * `device` with one CTA per SM; every kernel times itself in SM cycles (clock64), so the figures are per SM clock
 * (DESIGN.md 6.1 cites them).  `out` is a HOST array of n_out >= SAIL_MICROBENCH_N doubles:
 *   warp-instructions / clk / SM at 4 warps per sub-partition (2.0 = one per 2 clk per sub-partition = 64 lanes):
 *   [0] DMUL, two vector-register operands              [1] DFMA with one constant-bank operand
 *   [2] DFMA, three vector operands, two of them shared with the neighbouring instructions (operand reuse)
 *   [3] DFMA, three distinct vector operands            [4] DMMA m8n8k4
 *   [5] clk per SM for (2 DMMA + 8 DFMA) issued together: 2/[4] + 8/[2] means DMMA has no pipe of its own
 *   [6] SHFL   [7] LDS.128, one address per warp   [8] LDS.64, lane-contiguous
 *   [9] [10] [11] dependent-issue latency of DFMA, SHFL, DMMA in clk   [12] as [2] at ONE warp per sub-partition
 *   [13] the sweep kernel's tau loop alone (C = 16, 12 warps per SM): CREDITED (5 per tau-point) warp-instr / clk / SM
 *   [14] [15] latency in clk of the warp sum by 2 DMMA + DADD / by the 5-stage fp64 shuffle butterfly
 * Returns SAIL_ERR_ARG for a NULL / short array, SAIL_ERR_CUDA without a device.
 */
#define SAIL_MICROBENCH_N 16
SAIL_API int sail_microbench(int32_t device, void *stream, double *out, int32_t n_out);

#ifdef __cplusplus
}
#endif
#endif /* SAIL_B200_H */
