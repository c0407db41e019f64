/*
 * chem.h -- C ABI of the B200-native batched stiff-kinetics integrator
 * (hot path of arXiv 1607.03884, Curtis/Niemeyer/Sung: "An investigation of
 * GPU-based stiff chemical kinetics integration methods").
 *
 * PAPER.md = /root/reference/PAPER.md (text of the paper).  The operations:
 *   - the problem: many independent constant-pressure reactor IVPs, one per
 *     thermochemical state (T, Y_1..Y_{N-1}), advanced over ONE global time
 *     step; PAPER.md L47-L49 (Sec. 1), L134 (Sec. 3).
 *   - source term and analytical constant-pressure mass-fraction Jacobian
 *     (pyJac): PAPER.md L82 (Sec. 2.1), footnote L186.
 *   - 3-stage / 5th-order implicit Radau IIA with built-in adaptive stepping,
 *     Jacobian reuse "according to the built-in rules", rtol = 1e-6,
 *     atol = 1e-10: PAPER.md L86 (Sec. 2.1).
 *   - LU factorisation of the Jacobian-based matrices on the device:
 *     PAPER.md L86.
 *   - per-IVP internal step counts d_i (divergence measure, Eq. 3): L190.
 * DESIGN.md lists every reading (R1..R13) where the paper is silent.
 *
 * Conventions
 *   - units: cm, mol, s, K, g/mol, dyn/cm^2 (1 atm = 1.01325e6), Ea in cal/mol.
 *   - all functions return 0 on success or a negative CHEM_E_* code;
 *     chem_last_error() gives a thread-local message for the last failure.
 *   - "device" pointers are CUDA global-memory pointers on the current device;
 *     "host" pointers are ordinary host memory.  Nothing is retained after a
 *     call returns except inside the opaque chem_mech.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).
 *     Calls taking a stream are asynchronous with respect to the host.  Every launch takes its work-queue head and
 *     scratch from the stream-ordered allocator (cudaMallocFromPoolAsync on `stream`), so calls on different streams may
 *     run concurrently with the same chem_mech.  The memory comes from a pool the library creates for itself on each
 *     device it is used on; the device's default pool (the application's) is not touched.  The pool keeps its blocks (a
 *     few bytes; 277 MB for a full launch of the thread-per-state kernel) from call to call; chem_scratch_trim() or
 *     chem_mech_free() returns the unused ones to the driver.  chem_integrate_noalloc uses no allocator at all.
 *   - there is NO CPU fallback: without a CUDA device every compute call fails
 *     with CHEM_E_CUDA.
 */
#ifndef CHEM_H_
#define CHEM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define CHEM_OK 0
#define CHEM_E_ARG (-1)         /* invalid argument / inconsistent description      */
#define CHEM_E_UNSUPPORTED (-2) /* description outside the compiled limits           */
#define CHEM_E_CUDA (-3)        /* CUDA runtime error (see chem_last_error)          */
#define CHEM_E_NOMEM (-4)

/* reaction types */
#define CHEM_RXN_ELEMENTARY 0
#define CHEM_RXN_THREE_BODY 1        /* q = [M] (kf prod C - kr prod C)                */
#define CHEM_RXN_FALLOFF_LINDEMANN 2 /* k = k_inf Pr/(1+Pr), Pr = k_0 [M] / k_inf      */
#define CHEM_RXN_FALLOFF_TROE 3      /* ... times the Troe broadening factor F         */

/* Mechanism description: plain host arrays, borrowed for the duration of chem_mech_load.
 * All reactions are reversible; reverse rate constants follow from the equilibrium
 * constants of the NASA-7 thermo data.  The LAST species is the bath species removed
 * from the state vector (Y_N = 1 - sum Y_k). */
typedef struct chem_mech_desc {
    int32_t n_species;        /* N_sp >= 2; the state vector has N = N_sp entries (T, Y_1..Y_{N_sp-1}) */
    int32_t n_reactions;      /* >= 1                                                                 */
    const double *mol_weight; /* [n_species] g/mol                                                    */
    const double *nasa_lo;    /* [n_species][7] a0..a6 for T <= nasa_tmid                             */
    const double *nasa_hi;    /* [n_species][7] a0..a6 for T >  nasa_tmid                             */
    const double *nasa_tmid;  /* [n_species] K                                                        */
    const int32_t *rxn_type;  /* [n_reactions] CHEM_RXN_*                                             */
    const int32_t *reac_ptr;  /* [n_reactions+1] CSR offsets into reac_sp / reac_nu                    */
    const int32_t *reac_sp;   /* reactant species indices (0-based)                                   */
    const int32_t *reac_nu;   /* reactant stoichiometric coefficients, integers 1..3                  */
    const int32_t *prod_ptr;  /* same for products                                                    */
    const int32_t *prod_sp;
    const int32_t *prod_nu;
    const double *arr_A;      /* [n_reactions] k = A T^b exp(-Ea/(R T)); the high-pressure limit for falloff */
    const double *arr_b;
    const double *arr_Ea;     /* cal/mol */
    const double *low_A;      /* [n_reactions] low-pressure limit k_0 (read for falloff types only)   */
    const double *low_b;
    const double *low_Ea;
    const double *troe;       /* [n_reactions][4] alpha, T***, T*, T** (read for CHEM_RXN_FALLOFF_TROE) */
    const int32_t *eff_ptr;   /* [n_reactions+1] CSR of third-body efficiencies that differ from 1    */
    const int32_t *eff_sp;
    const double *eff_val;
} chem_mech_desc;

typedef struct chem_mech chem_mech; /* opaque: packed device tables + launch configuration */

/* Options of chem_integrate_ex.  Zero-initialise for the defaults. */
typedef struct chem_opts {
    double h0;           /* first internal step size; 0 -> t_end (R9)                      */
    int32_t max_steps;   /* limit on internal step attempts per state; 0 -> 100000                    */
    int32_t newton_max;  /* max simplified-Newton iterations per step; 0 -> 7                         */
    int32_t kernel;      /* 0 auto; 1 shared-memory group kernel (warp or CTA per state); 2 warp-per-state kernel and
                            3 thread-per-state kernel (both: small mechanisms only, N_sp <= 16, N_rx <= 32).
                            Results are bit-reproducible PER KERNEL ID.  Auto chooses by mechanism AND batch size (n_states),
                            so with kernel = 0 the bits of one state may differ between a small and a large batch (always
                            within the tolerance); chem_last_kernel tells which ran.  Fix the id where bits must not move. */
    int32_t reorder;     /* order in which the work queue starts the states ("reordering IVPs to increase similarity
                            of stiffness"; L184).  Results never depend on it, bit for bit.  1: by decreasing cost_hint (caller's
                            prediction); 2: by the library's own stiffness estimate, t_end ||f(y0) / (atol + rtol |y0|)||_rms, from
                            one extra source term per state (small mechanisms only, else CHEM_E_UNSUPPORTED); 0: auto = the
                            estimate where it is measured to pay (small mechanisms: the thread-per-state kernel from ~150,000
                            states on, the warp-per-state kernel from ~12,000), otherwise none; -1: off */
    const double *P_per_state;  /* device [n_states] or NULL: per-state pressure overriding P        */
    const int32_t *cost_hint;   /* device [n_states] or NULL: predicted cost per state, e.g. chem_stats.nstep of the
                                   previous global step; read only when reorder = 1.  Results do not depend on it. */
    int32_t fd_jacobian; /* 1: first-order finite-difference Jacobian "based on that of CVODE" (Sec. 3.4;
                            DESIGN.md R13) instead of the analytical one; costs N extra source terms per Jacobian */
    int32_t fixed_steps; /* > 0: take exactly this many equal internal steps without error control (the solver-verification
                            experiment of PAPER.md L106-L128, Fig. 2); a step that cannot be taken ends the state with
                            status -5 (R14); 0: adaptive (default) */
} chem_opts;

/* Per-state result record written by chem_integrate_ex (device array of n_states). */
typedef struct chem_stats {
    int32_t status;     /* 0 ok; -1 max_steps exceeded; -2 step size too small; -3 singular matrix 5x; -4 non-finite input;
                           -5 fixed_steps mode: a step could not be taken (singular matrix or non-finite iterate) */
    int32_t nstep;      /* internal step attempts that reached the Newton loop (d_i of PAPER.md Eq. 3) */
    int32_t naccpt;     /* accepted steps                                                              */
    int32_t nrejct;     /* error-test rejections (after the first accepted step)                       */
    int32_t nfcn;       /* source-term evaluations                                                     */
    int32_t njac;       /* Jacobian evaluations                                                        */
    int32_t ndec;       /* LU factorisations (each = one real + one complex N x N)                     */
    int32_t nsol;       /* Newton iterations (each = one real + one complex solve)                     */
    int32_t nnewt_fail; /* step attempts abandoned by the Newton convergence control                   */
    int32_t reserved;
    double h_last;      /* size of the last accepted internal step                                     */
} chem_stats;

/* Mechanism compiler: validates `desc` (host), packs it into device tables.
 * On success *out owns device memory; release with chem_mech_free. */
int chem_mech_load(const chem_mech_desc *desc, chem_mech **out);
void chem_mech_free(chem_mech *mech);
int chem_mech_info(const chem_mech *mech, int32_t *n_species, int32_t *n_reactions);

/* Source term f(T, Y; P) for a batch (test hook and building block).
 * y: device [n_states][N] row-major; f: device [n_states][N]. */
int chem_rhs(const chem_mech *mech, int32_t n_states, double P, const double *y, double *f, void *stream);

/* Analytical Jacobian J[s][i][j] = d f_i / d y_j, device [n_states][N][N] row-major. */
int chem_jacobian(const chem_mech *mech, int32_t n_states, double P, const double *y, double *J, void *stream);

/* Batched dense solve hook (the device routines the integrator uses: for n <= 16 those of the warp-per-state kernel,
 * a pivoted Gauss-Jordan inverse applied as a matrix-vector product; above that the LU + triangular solves of the
 * group kernels):
 * solves A_s x_s = b_s for s < batch.  A: device [batch][n][n] row-major (complex: interleaved re,im),
 * b: device [batch][n] (complex: interleaved), x: same shape as b.  info: device [batch], 0 or k+1 of a zero pivot. */
int chem_lu_solve(int32_t n, int32_t batch, int32_t is_complex, const double *A, const double *b, double *x,
                  int32_t *info, void *stream);

/* Test hook for the thread-per-state kernel's linear algebra (left-looking LU with partial pivoting +
 * triangular solves, one system per lane), on the two matrices of one Radau step built from a real n x n matrix J
 * (1 <= n <= 16):   (fac1 I - J) x1 = b1   and   ((alphn + i betan) I - J)(x2 + i x3) = b2 + i b3.
 * J: device [batch][n][n] row-major; b, x: device [batch][3][n] (b1, b2, b3 / x1, x2, x3); info: device [batch] or NULL,
 * 0 or j + 1 if a matrix has no usable pivot in column j (x is then not written). */
int chem_tps_radau_solve(int32_t n, int32_t batch, const double *J, double fac1, double alphn, double betan,
                         const double *b, double *x, int32_t *info, void *stream);

/* The hot path: integrate every state from t = 0 to t_end at constant pressure P.
 * y_in, y_out: device [n_states][N] row-major (may alias).  n_states == 0 is a no-op. */
int chem_integrate(const chem_mech *mech, int32_t n_states, double P, double t_end, double rtol, double atol,
                   const double *y_in, double *y_out, void *stream);

/* Same with options and per-state statistics (stats: device [n_states] or NULL). */
int chem_integrate_ex(const chem_mech *mech, int32_t n_states, double P, double t_end, double rtol, double atol,
                      const double *y_in, double *y_out, const chem_opts *opts, chem_stats *stats, void *stream);

/* End-to-end form with HOST buffers (the paper's timings include the transfers): integrates the states
 * of y_in_host into y_out_host (and stats_host if not NULL) and synchronises.  Page-locked (pinned) buffers are read and
 * written by the kernel itself through their device mapping, state by state, so the transfers overlap the integration;
 * pageable buffers are staged through device memory in two chunks on two internal streams.  The buffers may alias.
 * `reorder` = 1 / 2 are treated as 0 (auto) here; -1 switches the ordering pass off.  The kernel is chosen once from n_states, as chem_integrate_ex would, whether or not the
 * buffers are pinned (the chunks of the pageable path all run that kernel).  The internal streams belong to the mechanism
 * object: one chem_integrate_host call per mechanism at a time. */
int chem_integrate_host(const chem_mech *mech, int32_t n_states, double P, double t_end, double rtol, double atol,
                        const double *y_in_host, double *y_out_host, const chem_opts *opts, chem_stats *stats_host);

/* The hot path for callers that must not allocate device memory at call time.
 *
 * Every other compute call of this library takes a little device memory per launch from CUDA's stream-ordered allocator
 * (the work-queue head, the start order, the thread-per-state workspace).  Some hosts cannot afford that: an application
 * that claimed the whole card for its own memory arena at start-up (a flow solver, a training framework with a caching
 * allocator), so that a driver allocation fails or forces the arena to shrink; a process held to a fixed memory budget
 * on a shared or partitioned GPU; a time-critical loop in which a call that may take a driver lock or synchronise the
 * device is not acceptable.  chem_integrate_noalloc is chem_integrate_ex for them.  It runs the same shared-memory
 * kernels (chem_opts.kernel 0, 1 or 2; 0 picks the warp-per-state kernel where the mechanism allows it, else the group
 * kernel) and gives bit-identical y_out and stats for the same kernel id, but keeps its scratch in a fixed array that is
 * part of the library image.  It calls no cudaMalloc / cudaMallocAsync / cudaFree and no library routine that does.
 * The caller owns every buffer it passes (y_in, y_out, stats, opts->P_per_state, opts->cost_hint: device memory);
 * chem_mech_load DOES allocate, so load the mechanism at set-up time, before the no-allocation phase begins.
 *
 * Limits and rules:
 *   - at most CHEM_NOALLOC_MAX_STATES states per call (the array has one start-order slot per state); a larger n_states
 *     returns CHEM_E_UNSUPPORTED with a message and launches nothing.  Split a larger batch into several calls on one
 *     stream: the states are independent.
 *   - chem_opts.kernel = 3 (thread-per-state) returns CHEM_E_UNSUPPORTED: its workspace is 7 KB per resident state.
 *   - the array costs 4 MiB + 4352 B of device memory on EVERY GPU that loads libchem.so, from load until the process
 *     exits, whether or not this function is ever called.
 *   - the first call on each device looks up the array's device address (with that device current) and sets kernel
 *     attributes; CUDA may also load the kernels' code on a first launch.  Make one call per device during set-up
 *     (n_states = 1 is enough), before any stream capture and before the phase in which allocation is off limits.
 *   - all calls on a device share the one array, and it keeps the previous call's contents; each call clears, on its own
 *     stream, the part it starts from.  Calls that can overlap on the GPU (different streams, several host threads)
 *     race on the work queue and return wrong results or skip states: issue them on one stream or order them with events.
 *     This applies across mechanisms too.  chem_integrate / chem_integrate_ex do not use the array and may overlap freely.
 *   - opts->reorder = 0, 2 and -1 all mean "no ordering" here (the library's own estimate is not offered).
 *   - opts->reorder = 1 with opts->cost_hint orders the start of the states by decreasing cost with a counting sort over
 *     1024 cost classes (no sort library); as with chem_integrate_ex the results do not depend on it.
 * Otherwise as chem_integrate_ex: asynchronous on `stream`, y_in / y_out may alias, stats may be NULL, n_states == 0 is a
 * no-op.  PAPER.md L47-L49, L86, L134 (the operation), L194 (reordering). */
#define CHEM_NOALLOC_MAX_STATES 1048576
int chem_integrate_noalloc(const chem_mech *mech, int32_t n_states, double P, double t_end, double rtol, double atol,
                           const double *y_in, double *y_out, const chem_opts *opts, chem_stats *stats, void *stream);

/* Returns the launch scratch that the library's memory pool caches for the CURRENT device to the driver (blocks still in
 * use by queued work stay).  chem_mech_free does the same.  The next launch simply allocates again. */
int chem_scratch_trim(void);

/* Number of kernel launches issued by this library since load (for bench.py's gpu_launches). */
int64_t chem_launch_count(void);

/* Kernel id (1, 2 or 3 as in chem_opts.kernel) of the last chem_integrate / chem_integrate_ex / chem_integrate_host
 * launch issued with this mechanism; 0 before the first.  Not synchronised with concurrent callers. */
int chem_last_kernel(const chem_mech *mech);

/* Algorithmic floating-point operation counts of the compiled mechanism:
 * out[0] = one source-term evaluation, out[1] = one Jacobian evaluation, out[2] = one LU pair (real + complex),
 * out[3] = one Newton iteration's solves and vector work (excluding its 3 source terms), out[4] = error estimate. */
int chem_flop_model(const chem_mech *mech, double out[5]);
/* The same counts with every exp / log / pow / sqrt counted as 1 flop instead of the 20 of chem_flop_model's convention
 * (bench.py reports the roofline fraction both ways). */
int chem_flop_model_t1(const chem_mech *mech, double out[5]);

/* Diagnostic, not on the hot path: the fp64 FMA rate of the device measured with dependent-free DFMA streams
 * (`iters` fused multiply-adds x 8 accumulators per thread, 8 CTAs of 256 threads per SM, best of `reps` launches, in
 * TFLOP/s); bench.py reports it beside the derived peak of the "alu" roofline. */
int chem_fp64_probe(int32_t iters, int32_t reps, double *tflops_best);

const char *chem_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CHEM_H_ */
