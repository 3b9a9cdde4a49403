/*
 * landau.h -- C ABI of liblandau.so: the B200 (sm_100a) hot path of the multispecies
 * structure-preserving particle discretisation of the Landau collision operator
 * (Zonta, Pusztay, Hirvijoki, arXiv:2212.00663; citations are PAPER.md:<line>).
 *
 * What the library computes (3-V restatement, DESIGN.md "Readings" D1, D2, S1-S10, U1-U3):
 *
 *   pass 1  G_p = (1/w_p) dS_eps/dv_p, the gradient of the Gaussian-regularised entropy by tensor
 *           Gauss-Hermite quadrature                       Eq. (22); Eqs. 19-21
 *   pass 2  V_p = (1/m_s) sum_s' nu_ss' sum_{p' in s'} w_p' Q(v_p - v_p') (G_p/m_s - G_p'/m_s'),
 *           Q(z) = (|z|^2 I - z z^T)/|z|^3                 Eq. (23); Eqs. 4, 16, 17
 *   step    v^{n+1} = v^n + dt V[(v^n + v^{n+1})/2 ; G^n]  by Jacobi fixed-point iteration
 *                                                          Eqs. (24)-(25); Alg. 1
 *   moments n_s, P_s, K_s, S_eps,s                         Eqs. 26, 28, 33, 20
 *
 * Conventions
 *   - Every marker array argument is a DEVICE pointer (cudaMalloc'ed / torch CUDA tensor
 *     data_ptr) unless the function name ends in _host, in which case it is a HOST pointer and the
 *     library does the host<->device copies itself (on the context's stream, then synchronises).
 *   - v is [N x 3] row-major FP64, w is [N] FP64 (> 0), species_id is [N] int32 in 0..S-1 in any
 *     order.  Outputs are [N x 3] in the CALLER's marker order whatever the internal bucketing.
 *   - Small per-species outputs (moments) and landau_step_info are HOST memory.
 *   - Ownership: the caller owns every array it passes and may free or reuse it once the call
 *     returns (device arrays: once the context's stream has passed the call).  The library copies
 *     what it needs into its own SoA scratch and keeps no caller pointer.  The context owns its
 *     scratch (grown lazily, released by landau_destroy).
 *   - Streams: one context = one CUDA stream (opts->stream, NULL = the legacy default stream).
 *     Device-pointer calls are asynchronous on that stream except for the final status read-back;
 *     landau_step synchronises once at its end to fill landau_step_info.
 *   - Errors: every call returns an int.  0 = LANDAU_OK; 1 = LANDAU_NOT_CONVERGED (the step is
 *     still committed, as in the paper); negative = hard error, outputs are
 *     unspecified: -1 invalid argument (NULL, N < 1, species_id out of range, w <= 0, m <= 0,
 *     eps <= 0, non-symmetric nu, n_q out of range), -2 out of memory, -3 CUDA error,
 *     -4 non-finite input or result, -5 marker cloud too wide for the factorised entropy kernel
 *     AND the literal fallback disabled (never returned with default options).
 *     No exception or abort crosses this boundary; landau_last_error() returns a message.
 *   - There is NO CPU fallback: without a CUDA device landau_create fails with -3.
 */
#ifndef LANDAU_H
#define LANDAU_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LANDAU_OK 0
#define LANDAU_NOT_CONVERGED 1
#define LANDAU_EINVAL (-1)
#define LANDAU_ENOMEM (-2)
#define LANDAU_ECUDA (-3)
#define LANDAU_ENONFINITE (-4)
#define LANDAU_ERANGE (-5)

#define LANDAU_MAX_SPECIES 16
#define LANDAU_MAX_NQ 8

typedef struct landau_ctx landau_ctx; /* opaque, library-owned */

typedef struct {
    int n_q;          /* Gauss-Hermite knots per axis (reading S3); 0 -> 4; 2..8 */
    double nu0;       /* nu_ss' = nu0 q_s^2 q_s'^2 (reading U1); 0 -> 1.0            */
    const double* nu; /* optional HOST S x S override of nu_ss', must be symmetric; may be NULL   */
    int precision;    /* 0 = FP64 everywhere; 1 = FP32 arithmetic inside the pairwise sum of
                         landau_pair_field / landau_eval_field only (BASELINE config 4 variant)   */
    void* stream;     /* cudaStream_t; NULL = default stream                                      */
    int pair_kernel;  /* 0 = automatic; 1 = one-sided tiled kernel; 2 = symmetric (action-reaction)
                         kernel.  For tests and per-kernel timing.                                */
    int entropy_kernel; /* 0 = automatic (3 when the cloud is narrow enough, else 1); 1 = literal
                         separable form (3 n_q exponentials per pair); 2 = factorised form (1
                         exponential per pair) on the FP64 vector pipe; 3 = factorised form as an
                         FP64 tensor contraction (DMMA).  2 and 3 return LANDAU_ERANGE when the
                         cloud is too wide for the factorised form.  Form 3 streams a per-pass
                         product table of 544 B (n_q = 4) to 4352 B (n_q = 8) per marker; when
                         that exceeds a quarter of the device memory (or the environment variable
                         LANDAU_PRODTAB_BUDGET_MB, read by landau_create) 0 takes form 2 instead
                         and 3 returns LANDAU_ENOMEM.                                             */
    int device;       /* CUDA device ordinal; -1 = current device                                 */
} landau_opts;

typedef struct {
    int iterations;   /* fixed-point iterations done (k+1 of DESIGN.md O4) */
    double residual;  /* r_k of the last iteration                          */
    int converged;    /* 1 if r_k <= tol                                    */
} landau_step_info;

/* Fills *opts with the defaults (n_q 4, nu0 1, FP64, default stream, automatic kernels). */
void landau_default_opts(landau_opts* opts);

/* Species table: masses m_s > 0, charges q_s, mollifier covariances eps_s > 0 (Eq. 19,
 * PAPER.md:112-116; units velocity^2), all HOST arrays of n_species <= LANDAU_MAX_SPECIES
 * entries.  opts may be NULL (defaults). */
int landau_create(landau_ctx** out, int n_species, const double* mass, const double* charge,
                  const double* eps, const landau_opts* opts);
void landau_destroy(landau_ctx* ctx);

/* V_p of Eq. (23) with G from Eq. (22): pass 1 then pass 2.  Stateless with respect to the
 * markers held by landau_set_markers. */
int landau_eval_field(landau_ctx* ctx, int64_t N, const double* v, const double* w,
                      const int32_t* species_id, double* out);
int landau_eval_field_host(landau_ctx* ctx, int64_t N, const double* v, const double* w,
                           const int32_t* species_id, double* out);

/* Pass 1 alone: G_out[N x 3] = (1/w_p) dS_eps/dv_p (Eq. 22; Eq. 14).
 * S_eps_out: optional HOST array of S entries receiving S_eps,s (Eq. 20); may be NULL. */
int landau_entropy_grad(landau_ctx* ctx, int64_t N, const double* v, const double* w,
                        const int32_t* species_id, double* G_out, double* S_eps_out);

/* Pass 2 alone with the entropy gradient supplied: out[N x 3] = V_p of Eq. (23) for G_in. */
int landau_pair_field(landau_ctx* ctx, int64_t N, const double* v, const double* w,
                      const int32_t* species_id, const double* G_in, double* out);

/* Time stepping works on markers held by the context. */
int landau_set_markers(landau_ctx* ctx, int64_t N, const double* v, const double* w,
                       const int32_t* species_id);
int landau_set_markers_host(landau_ctx* ctx, int64_t N, const double* v, const double* w,
                            const int32_t* species_id);
int landau_get_markers(landau_ctx* ctx, double* v_out /* device, N x 3, caller order */);
int landau_get_markers_host(landau_ctx* ctx, double* v_out /* host */);

/* One step of Eq. (24): pass 1 once at v^n, then Jacobi fixed-point iterations, each one pass 2 at
 * the midpoint (Eq. 25) with G^n frozen, until r_k <= tol or max_iter iterations, where
 *   r_k = sqrt( sum_p w_p m_s |v^(k+1)_p - v^(k)_p|^2 / sum_p w_p m_s |v^(k+1)_p|^2 )  (reading S7).
 * The loop runs on the device (no host synchronisation per iteration).  info may be NULL.
 * Returns 0, or 1 if not converged (state still advanced; reading S8). */
int landau_step(landau_ctx* ctx, double dt, double tol, int max_iter, landau_step_info* info);

/* velocity-space dimension.  3 (default), or 2 = the paper's own 2-V setting (PAPER.md:110,
 * 180): markers must be given with v_z = 0 (v_z is ignored by the passes and left untouched by the steps).  The
 * passes then run native 2-V kernels: pass 1 sums the n_q^2 planar nodes (k_i, k_j, 0) -- the z-quadrature of
 * Eq. (22) is done in closed form, G_z is an exact zero -- and pass 2 does the two-component arithmetic of Eq. (23)
 * (22 instead of 30 FP64 instructions per unordered pair).  x/y results are the paper's 2-V Eqs. (22)-(24) and equal
 * what the 3-V kernels give on v_z = 0 data (reading D1; pass 2 bit for bit, pass 1 to round-off), and S_eps is the
 * 3-V value of that data, so 2-V and 3-V runs report comparable entropies.  (Clouds too wide for the factorised pass 1
 * and landau_cells_run use the 3-V arithmetic with G_z stored as zero.) */
int landau_set_dimension(landau_ctx* ctx, int dim);

/* SURVEY.md NEXT-4 (second half): Gaussian cutoff of pass 1.  on = 1 (default): a tile of 64 source markers is not
 * visited when the distance D (in units of sqrt(2 eps_s)) between its bounding box and the box of a block of 128
 * targets satisfies  D^2 - 2 D |k|_max >= 60 ln 2 + ln(w_max/w_min) + ln N_s  (|k|_max = sqrt(3) times the largest
 * Gauss-Hermite knot): everything skipped changes no node sum of Eq. (22) by more than 2^-60 relative (derivation in
 * csrc/entropy.cuh), so results agree with the all-pairs evaluation to round-off.  It pays when eps_s is small against
 * the extent of the cloud -- the paper's own rule eps_s = 1.2 (L_s/N)^1.98 -- and costs one
 * box test per tile pair otherwise.  on = 0: all pairs.  morton = 1 (default): clouds of 4096 .. 2^21 markers are
 * bucketed, inside every species, along a Morton curve through the cells of a mesh over the species' bounding box
 * (stable inside a cell), so that tiles are compact boxes whatever the caller's marker order; morton = 0 keeps the
 * caller's order inside a species (takes effect at the next landau_set_markers / field evaluation).  Outputs are
 * in caller order either way.  landau_cutoff_stats returns the number of (target block, source tile) pairs
 * considered / skipped by the LAST pass 1 (HOST outputs; synchronises). */
int landau_set_cutoff(landau_ctx* ctx, int on, int morton);
int landau_cutoff_stats(landau_ctx* ctx, int64_t* tiles_considered, int64_t* tiles_skipped);

/* How landau_step / landau_run issue a step whose cost is launch latency (small clouds).  mode 1 (default,
 * automatic): clouds of <= 32768 padded slots on the one-sided pair kernel with the paper's Jacobi iteration (no stiff-
 * pair treatment) run ALL iterations of a step inside one persistent kernel with grid-wide barriers (cooperative
 * launch; step_small.cuh); other clouds of <= 65536 padded slots replay the whole step as ONE CUDA graph whose fixed-
 * point body is a conditional WHILE node kept alive from the device (cudaGraphSetConditional in the update kernel) --
 * no launch per iteration, no pre-enqueued iterations that exit at once.  mode 0: always the plain launch sequence
 * (max_iter iterations enqueued up front, early exit on the device flag).  mode 2: the graph at any size (never the
 * persistent kernel).  The same kernel bodies in the same summation orders and bit-identical results in every mode
 * (for every solver of landau_set_solver); the graph is captured after the first ordinary step, is reused while shapes
 * and parameters stay the same, and neither graph nor persistent kernel is used while landau_profile_enable is on. */
int landau_set_step_graph(landau_ctx* ctx, int mode);

/* SURVEY.md NEXT-4 (robustness): what landau_step / landau_run do with a step whose fixed point does not converge
 * within max_iter.  max_halvings = 0 (default) is the paper's behaviour: the last iterate is committed and status 1
 * returned, at the price of an energy jump (reading S8).  max_halvings = k > 0: such a step
 * is NOT committed but redone as two steps of dt/2, recursively up to k levels (only the deepest level commits an
 * unconverged iterate).  Every sub-step is a step of Eq. (24), so the conservation laws hold for each of them.
 * info then reports the summed iterations, the largest residual and converged = all sub-steps converged.  The loop
 * is driven from the host (one synchronisation per sub-step). */
int landau_set_substep(landau_ctx* ctx, int max_halvings);

/* how landau_step / landau_run solve Eq. (24).  solver 0 (default) = the paper's plain
 * Jacobi fixed-point iteration (`depth` ignored); solver 1 = the same fixed point with Anderson acceleration of the
 * given depth (1..10, 3 to 5 is a good default); solver 2 = Jacobian-free Newton-Krylov: Newton's method on
 * F(x) = x - v^n - dt V[(x + v^n)/2 ; G^n] with GMRES(depth) (restart length 1..30, 20 is a good default) in the
 * energy inner product and Jacobian-vector products by one extra pass 2 each -- for the steps the fixed-point
 * iteration cannot converge.  The equation, the residual (evaluated at a true evaluation of
 * g(x) = v^n + dt V), the stopping rule, status codes and conservation properties are unchanged; only the iterates
 * between v^n and the converged v^{n+1} differ.  `iterations` counts pass-2 evaluations for every solver.  All
 * three are device driven (no host synchronisation inside a step). */
int landau_set_solver(landau_ctx* ctx, int solver, int depth);

/* SURVEY.md NEXT-4 (robustness): exact local treatment of stiff two-marker interactions inside landau_step /
 * landau_run (Jacobi and Anderson solvers).  The pair term of Eq. (23) is not Lipschitz at z = 0; two markers that have
 * drifted to within ~dt nu w |Gamma| / m of each other make the fixed-point map of Eq. (24) expand in their relative
 * coordinate, and the iteration ends at max_iter with a residual ~1e-8 -- the paper's "unable to fully converge on
 * occasion", reproduced step for step by the oracle.  theta > 0: pairs whose stiffness
 *   L_pq = (dt/2) nu_ss' (w_q/m_s + w_p/m_s') |g_p - g_q| / |v_p - v_q|^2   (at v^n)
 * exceeds theta are found by the first pass-2 evaluation of every step, and in every iteration their mutual term is
 * taken out of the explicit update and solved implicitly and exactly (a two-marker midpoint equation that reduces to
 * one scalar root; csrc/stiff_pairs.cuh).  SAME equation, residual, stopping rule and status codes: at convergence
 * every marker satisfies Eq. (24); only the path of the iteration changes, so steps that the plain iteration can
 * converge give the same v^{n+1} to ~tol.  0.2 is a good value.  theta = 0 (default): off, the paper's plain
 * iteration.  landau_stiff_pairs_last returns how many stiff pairs the last step found and how many of them its last
 * iteration had to leave to the plain update (HOST outputs; synchronises). */
int landau_set_stiff_pairs(landau_ctx* ctx, double theta);
int landau_stiff_pairs_last(landau_ctx* ctx, int* n_pairs, int* n_skipped);

/* Mixed-precision implicit step ("try FP32 pass-2 evaluations for the early iterations").  f32_until > 0:
 * while the Jacobi iterates of Eq. (24) still move by more than f32_until (the residual r_k of the last iteration),
 * pass 2 is evaluated by the FP32 flavour of the symmetric kernel (the BASELINE config-4 field variant: ~3e-6 relative
 * error in V, i.e. ~dt * 3e-6 in the iterate); below it, and always for the iteration that ends the step, by the FP64
 * kernel.  The fixed point, the stopping rule (r_k <= tol on an FP64 evaluation) and therefore the converged state and
 * its conservation properties are those of the FP64 step; only the early iterates differ.  A sensible value is 1e-7
 * (FP32 noise in the iterate is ~3e-9 at dt = 1e-3).  The decision is taken on the device, per iteration.  The last
 * iteration max_iter allows is an FP64 evaluation too, so a step that stops unconverged at max_iter also commits an
 * FP64 iterate (with max_iter = 1 the step is plain FP64).  A threshold the FP32 iterates can never reach would keep
 * every step in FP32 until that last iteration, so values in (0, 1e-10) are rejected with LANDAU_EINVAL.  Applies
 * to the Jacobi solver on clouds of >= 16384 markers in 3-V; ignored otherwise.  0 (default) = off. */
int landau_set_mixed_precision(landau_ctx* ctx, double f32_until);

/* n_steps consecutive steps with one host synchronisation at the end; info (optional, HOST,
 * n_steps entries) receives each step's record.  Returns 1 if any step did not converge. */
int landau_run(landau_ctx* ctx, int n_steps, double dt, double tol, int max_iter,
               landau_step_info* info);

/* one step of the discrete-gradient scheme, Eqs. (46)-(49), which adds
 * guaranteed entropy monotonicity (Eq. 49) to the conservation laws of Eq. (24).  Q is taken at the
 * midpoint (the discrete gradient of the quadratic K); the entropy gradient is Gonzalez' midpoint discrete
 * gradient  dbar S/dv_p = w_p G_p(u) + lambda (v_p^{n+1} - v_p^n)  (reading DG1).  Same Jacobi fixed
 * point, residual, status and info conventions as landau_step; every iteration costs two pass-1 and one
 * pass-2 evaluations.  Device driven: the entropies, lambda's sums and the residual are reduced on the device and
 * every kernel of an iteration exits at once when the step is done; the host enqueues iterations in chunks of 8 and
 * reads the done flag once per chunk (no read-back inside an iteration). */
int landau_step_dg(landau_ctx* ctx, double dt, double tol, int max_iter, landau_step_info* info);

/* many spatial collision cells in one call.  The bracket couples only markers of the same
 * cell; a PIC code has thousands of small cells.  Markers of cell k are rows
 * cell_offset[k] .. cell_offset[k+1]-1 of v / w / species_id (DEVICE arrays, any species order inside a cell;
 * cell_offset is a HOST array of n_cells + 1 entries).  Every cell is advanced by n_steps steps of Eq. (24)
 * (same Jacobi fixed point, residual, tolerance and readings as landau_step) by ONE kernel launch: one
 * persistent thread block per cell with the cell's state in shared memory.  v_out (DEVICE, same layout, may
 * alias v) receives the new velocities in caller order.  Limit: markers per cell <= 1024 (n_q <= 5), 970 / 878 /
 * 802 at n_q = 6 / 7 / 8 (the cell's state lives in the 227 KB of shared memory of one thread block);
 * landau_cells_max_markers(n_q) returns the limit the library enforces (host only, no GPU needed; 0 for an n_q
 * outside 2..8); a larger cell makes the call return LANDAU_EINVAL.  A cell too
 * wide for the factorised pass 1 takes the literal form, as the single-cell path does.
 * info (HOST, n_cells entries, may be NULL): per-cell status (0 ok, 1 = some step hit max_iter, < 0 = the
 * cell was rejected and copied through unchanged: -1 invalid markers, -4 non-finite), iterations summed over the
 * steps, the largest per-step count, and the last residual.
 * Returns 0, 1 (some cell did not converge) or the most negative cell status. */
typedef struct {
    int status;
    int iterations;
    int max_iterations;
    int steps_not_converged;
    double residual;
} landau_cell_info;
int landau_cells_max_markers(int n_q);
int landau_cells_run(landau_ctx* ctx, int n_cells, const int64_t* cell_offset, const double* v, const double* w,
                     const int32_t* species_id, double* v_out, int n_steps, double dt, double tol, int max_iter,
                     landau_cell_info* info);

/* Moments of the held markers, HOST outputs, any may be NULL:
 * n[S] = sum w (Eq. 33), P[S x 3] = m_s sum w v (Eq. 26), K[S] = (m_s/2) sum w |v|^2 (Eq. 28),
 * S_eps[S] = regularised entropy (Eq. 20; costs one pass 1). */
int landau_moments(landau_ctx* ctx, double* n, double* P, double* K, double* S_eps);
/* stress[S x 6] = m_s sum w v_i v_j (xx,yy,zz,xy,xz,yz); m4[S x 3] = sum w (v_i - u_i)^4
 * (per-axis temperatures Eqs. 30-31 and kurtosis are derived from these by the caller). */
int landau_moments_ext(landau_ctx* ctx, double* stress, double* m4);

/* The same n_s, P_s, K_s (Eqs. 33, 26, 28) WITHOUT a context and without
 * any device allocation, for callers that cannot call cudaMalloc: a host code whose own arrays (or
 * whose framework's fixed pool) already own all of HBM, or a diagnostics hook inside an asynchronous
 * time loop where cudaMalloc / cudaFree would synchronise the whole device under somebody else's
 * streams.  (landau_create and every context call allocate; this call never does.)
 *   v [N x 3], w [N], species_id [N] int32 in 0..n_species-1, any order: DEVICE, read only.
 *   mass [n_species] > 0: HOST (passed to the kernel by value).
 *   out [n_species x 5] = n_s, P_s,x, P_s,y, P_s,z, K_s per species: DEVICE, written on `stream`
 *       (cudaStream_t, NULL = default stream).  The call does not synchronise: read `out` after the
 *       stream has passed it.  A species_id outside the range turns every entry of `out` into NaN.
 *   Scratch is a 655 616-byte (640.25 KiB) __device__ array built into liblandau.so: every GPU that
 *       loads the library holds it until the process exits.  It bounds the problem:
 *       N <= LANDAU_MOMENTS_NOALLOC_MAX_N, n_species <= LANDAU_MAX_SPECIES; anything larger returns
 *       LANDAU_EINVAL (nothing is launched; landau_moments handles those sizes, and allocates).
 *   The array is shared by ALL calls on a device and keeps the last call's contents; the call clears
 *       the one word that has to start at zero.  Calls that can overlap on the GPU (two streams, two
 *       threads) race on it and return garbage: serialise them.
 *   The first call on each device looks up the array's device address (cudaGetSymbolAddress) with
 *       that device current, which can make the runtime load the library's device code: make that
 *       call once at start-up, before any stream capture.  The devices are told apart by
 *       cudaGetDevice at call time; `stream` and all pointers must belong to the current device.
 *   Returns 0, LANDAU_EINVAL (NULL, N < 1, sizes beyond the limits, mass <= 0) or LANDAU_ECUDA;
 *       landau_moments_noalloc_last_error() gives the calling thread's last message ("" if none).
 *   Sums are taken in a fixed order (deterministic), but not landau_moments' order: the two agree to
 *       rounding (tests: rtol 1e-12), not bit for bit. */
#define LANDAU_MOMENTS_NOALLOC_MAX_N 2097152 /* 2^21 markers */
int landau_moments_noalloc(int64_t N, const double* v, const double* w, const int32_t* species_id,
                           int n_species, const double* mass, double* out, void* stream);
const char* landau_moments_noalloc_last_error(void);

/* Gauss-Hermite rule the context uses (HOST outputs, n_q entries each). */
int landau_get_quadrature(const landau_ctx* ctx, double* knots, double* weights);

/* Names of the kernels the last field evaluation / step used, e.g. "pair=sym entropy=fact". */
const char* landau_last_kernels(const landau_ctx* ctx);
/* Number of kernel launches issued by this context so far. */
int64_t landau_launch_count(const landau_ctx* ctx);

/* Per-kernel timing for bench.py's roofline: when enabled, CUDA events are recorded on the
 * context's stream around every launch of the two all-pairs kernels (pass 2 "pair", pass 1
 * "entropy"); launches of fixed-point iterations that exited at once because the step had already
 * converged are not counted.  landau_profile_enable(ctx, on) also clears the sums.  Times are
 * accumulated when a call synchronises; read them after the call returns (HOST outputs). */
int landau_profile_enable(landau_ctx* ctx, int on);
int landau_profile_read(landau_ctx* ctx, double* pair_ms, int64_t* pair_launches, double* entropy_ms,
                        int64_t* entropy_launches);

/* FP64 ALU peak microbenchmark (dependent-free DFMA streams on every SM): runs `reps` launches and
 * returns the best rate in FLOP/s (2 per DFMA) through *flops_out (HOST). Used by bench.py for the
 * roofline denominator. */
int landau_fp64_peak(landau_ctx* ctx, int reps, double* flops_out);
/* Same for the FP64 tensor instructions (DMMA.8x8x4) that pass 1's contraction issues. */
int landau_fp64_peak_dmma(landau_ctx* ctx, int reps, double* flops_out);

const char* landau_last_error(const landau_ctx* ctx);
const char* landau_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LANDAU_H */
