/*
 * top.h -- C ABI of the B200-native Consensus-ADMM (CADMM) segment sweep of TOP
 * (arXiv 2507.10290).  Citations are PAPER.md:L<line> (+ equation) of the paper text.
 *
 * What the library computes: Algorithm 1 of the paper, closed-form
 * branch -- per sweep and per polynomial segment i of a piecewise polynomial trajectory
 * (Eq. 18; order 2s-1, s=3 jerk / s=4 snap):
 *     x-update  (Eq. 20a)      c_i  <- closed-form QP solve
 *     phi, w    (Eq. 14/20f/20g, L186-191, L250-252)  ball projections + their scaled duals
 *     z-update  (Eq. 6b/20b, L136, L235)      average of adjacent boundary derivatives
 *     residuals (Eq. 21-22)         r_p, r_d (two global sums per trajectory)
 *     s-update  (Eq. 10/20d, L166, L244)      slack projection of the box corridor
 *     u, v      (Eq. 6c/20c/20e, L139, L239-247)  scaled dual updates
 * Every step runs in CUDA kernels for sm_100a.  There is NO CPU fallback: without a CUDA
 * device every compute entry point returns TOP_E_CUDA.  The readings of the paper taken
 * where it is silent or garbled are listed in DESIGN.md ("Readings", A1-A19).
 *
 * Conventions
 *  - All INPUT pointers are HOST pointers to fp64 data and are copied inside top_create
 *    (the caller may free them as soon as top_create returns).
 *  - Output buffers are caller-owned.  Where an argument says "host or device" a flag tells
 *    which; device pointers must belong to the solver's device.
 *  - The handle owns all other host and device memory; top_destroy frees it.  The device memory of a
 *    solver is ONE allocation taken from a library-private stream-ordered memory pool of its device
 *    (cudaMallocFromPoolAsync); top_destroy returns it to that pool, which keeps up to 1 GiB for the
 *    next top_create (re-planning loops) and hands everything back to the driver at process exit.
 *  - Every call returns a top_status; nothing throws or aborts across the ABI.  A negative
 *    status leaves a message in top_last_error().  A handle is not thread-safe.
 *  - Kernels are enqueued on top_options.cuda_stream (a cudaStream_t passed as void*;
 *    NULL = the legacy default stream).  top_iterate is asynchronous with respect to the
 *    host; every call that returns data to the host synchronises that stream first.
 *    The stream must outlive the handle: top_destroy synchronises it and returns the arena to the pool in
 *    stream order (if the stream is gone or is being captured it falls back to a synchronising cudaFree).
 *
 * Environment variables (read by the library; none changes a result):
 *  - TOP_TRACE_CREATE=1     top_create / top_reset print their phase times (ms) to stderr.
 *  - TOP_SPLIT_TAIL=0|1     A/B switch of the tensor-core kernel's "split octets" launch shape: 0 = never
 *                           split, 1 = only the last octet of CTAs holding 4k+1 octets, unset = the planner's choice.
 *                           Read once per process.  Bit-identical results in every setting.
 *  - TOP_TEST_SEQ_START=n   test hook: the 64-bit counter whose low 32 bits number the inter-CTA mailbox messages starts at n
 *                           instead of 0 in solvers created afterwards (tests/test_gpu_cluster.py runs across the 2^32 wrap).
 */
#ifndef TOP_H
#define TOP_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define TOP_API __attribute__((visibility("default")))
#else
#define TOP_API
#endif

typedef struct top_solver top_solver;

typedef enum {
    TOP_OK = 0,
    TOP_NOT_CONVERGED = 1,   /* top_solve hit max_iter; the state is valid */
    TOP_E_INVALID = -1,      /* bad argument (see top_create)                      */
    TOP_E_NOMEM = -2,        /* host or device allocation failed                   */
    TOP_E_CUDA = -3,         /* CUDA runtime error, no device, or barrier time-out */
    TOP_E_UNSUPPORTED = -4,  /* valid request this build cannot run (size limits)  */
    TOP_E_NONFINITE = -5     /* a residual became NaN/Inf                          */
} top_status;

typedef enum { TOP_F64 = 0, TOP_F32 = 1 } top_dtype;
/* TOP_F64: state, evaluation, projections and the x-update all in fp64.
 * TOP_F32: state, evaluation and projections in fp32; the 2s x 2s x-update operator is kept
 *          and applied in fp64 (an all-fp32 operator loses Q against rho*G; R5). */

/* Waypoint handling (reading A2 of DESIGN.md; the paper's Alg. 1 leaves waypoints free). */
#define TOP_WAYPOINT_HARD     0u  /* sigma_i(0)=p_{i-1}, sigma_i(T_i)=p_i as equalities inside each segment QP (default) */
#define TOP_WAYPOINT_PINNED_Z 1u  /* Eq. 20a verbatim; the position row of every z_j is held at p_j */
#define TOP_WAYPOINT_FREE     2u  /* Alg. 1 verbatim: position rows are averaged as well */
#define TOP_WAYPOINT_MASK     3u
/* Which dual residual top_solve compares with eps (reading A8). */
#define TOP_RD_PAPER          0u  /* Eq. 22 in monomial physical-time coefficient space (default) */
#define TOP_RD_NORMALISED     4u  /* component k divided by T_i^k */
/* Tolerance scaling (reading A13). */
#define TOP_EPS_ABSOLUTE      0u  /* ||r|| < eps (default) */
#define TOP_EPS_N_SCALED      8u  /* ||r|| < N*eps, the paper's rule */
/* Inter-CTA synchronisation of the persistent kernel (a performance knob; results are identical). */
#define TOP_SYNC_AUTO         0u
#define TOP_SYNC_GRID         16u /* one grid-wide barrier per sweep */
#define TOP_SYNC_NEIGHBOUR    32u /* mailbox exchange with the two neighbouring CTAs only; one CTA barrier per sweep */
#define TOP_SYNC_PAIRWISE     48u /* the same, with warp-pair named barriers instead of the CTA barrier (what AUTO picks) */
#define TOP_SYNC_MASK         48u
/* Adaptive penalty (Eq. 24; Alg. 1 line 14): at every residual check of top_solve (every
 * check_every sweeps; the paper: every sweep) rho <- tau_incr*rho if r_p > mu*r_d, rho <- rho/tau_decr if
 * r_d > mu*r_p.  The change goes through top_set_rho. */
#define TOP_RHO_ADAPTIVE      64u
/* Kernel selection.  With 4 lanes per segment the sweep runs its two constant-matrix contractions (Eq. 20a second
 * bracket; evaluation of Eq. 20b, 20d-g) on the tensor cores (mma.sync m8n8k4 f64); with 8 lanes per segment
 * (lanes_per_segment = 8) it uses warp shuffles and synthetic division, no tensor cores.  The shuffle form of the 4-lane
 * kernel that this flag used to select was removed: together with 4 lanes it now returns TOP_E_UNSUPPORTED. */
#define TOP_KERNEL_NO_MMA     128u
/* Consensus width (reading A1 of DESIGN.md).  Default: every junction carries the derivative orders 0..s-1 (M is 2s x 2s).
 * TOP_CONSENSUS_WIDE: the paper's literal choice (M(t) stacks beta^0..beta^(d-1) with d = 2p-1; L257: each
 * x-update is over-determined; L259-264): orders 0..2s-2, i.e. n_c = 2s-1 rows per boundary; z_0 and z_N carry the given
 * end state (orders 0..s-1, Eq. 2c), so the orders s..2s-2 do not exist at the two trajectory ends.
 * top_get_state "z" is then [batch][N+1][2s-1][dims] and "u" [batch][N][2(2s-1)][dims] (rows that do not exist read 0).
 * TOP_F64 on the tensor-core kernel only; the trajectory must fit on chip (N <= 148 x 56; together with a polytope corridor
 * N <= 148 x 32); else TOP_E_UNSUPPORTED. */
#define TOP_CONSENSUS_WIDE    256u
/* x-update branch of Alg. 1 (PAPER.md:L266-270 lines 4-8).  Default: ClosedFormSolve (Eq. 20a, 20f, 20g).
 * TOP_XUPDATE_NUMERIC: NumericSolve (Eq. 15-17; L303) -- the ball sets ||sigma'|| <= vmax, ||sigma''|| <= amax
 * are treated as general convex inequality constraints g0_j(c) <= 0, replaced by g_j(c) = max{0, g0_j(c)}^2 = 0 (Eq. 15) with
 * one scaled multiplier per sample and ball, w_j <- w_j + g_j(c^{k+1}); the x-update minimises the augmented Lagrangian
 * (Eq. 17 added to Eq. 5 and to the slack penalty of the box, which keeps its slack form) with L-BFGS: memory 6, initial
 * inverse Hessian = the closed-form operator of the quadratic part, Armijo backtracking, stop when the step (proposed or taken) is below 1e-10
 * of the coefficients or after 50 iterations (the paper gives no parameters; reading A20 of DESIGN.md).
 * top_get_state "y_v" / "y_a" [batch][N][8] are the multipliers; "phi_*" / "w_*" read 0.  top_set_rho and TOP_RHO_ADAPTIVE
 * work as in the closed-form branch (the multipliers are scaled duals: times rho_old / rho_new).  TOP_F64 only; no polytope
 * corridor, TOP_CONSENSUS_WIDE or snapshots (TOP_E_UNSUPPORTED / TOP_E_INVALID). */
#define TOP_XUPDATE_NUMERIC   512u

/* The paper's convex sets, specialised as BASELINE.json's configs use them:
 * an axis-aligned box corridor per segment (K=6 half-spaces, linear set, Eq. 7-10) and Euclidean balls on
 * velocity and acceleration (quadratic sets, Eq. 11-14), all enforced at `samples` interior sample times
 * t_ij = T_i*j/(samples+1), j=1..samples (reading A10). */
typedef struct {
    int32_t samples;        /* Ms: 0 => no inequality constraints; otherwise 8 in this build (else TOP_E_UNSUPPORTED) */
    const double* box_lo;   /* host [batch][N][dims] or NULL => no box */
    const double* box_hi;   /* host [batch][N][dims]; lo < hi elementwise */
    double vmax;            /* > 0: ||sigma'(t_ij)||_2  <= vmax ; <= 0: off */
    double amax;            /* > 0: ||sigma''(t_ij)||_2 <= amax ; <= 0: off */
    /* General convex-polytope corridor (Eq. 7-10 "FIRI ... multiple linear inequality
     * constraints", L231 A_i^o in R^{MK x m(d+1)}): num_planes = K half-spaces a_k'p <= b_k per segment, enforced on the
     * position at the `samples` sample times, one slack and one scaled dual per (sample, plane) (Eq. 20d, 20e).
     * planes: host [batch][N][K][dims+1] = (a_k (dims), b_k); normals need not be unit but must be non-zero.
     * Replaces the box (box_lo/box_hi must be NULL).  1 <= K <= 16; TOP_F64 with the tensor-core kernel only
     * (lanes_per_segment 0 or 4, no TOP_KERNEL_NO_MMA), N up to 40 segments per SM (5 920 on a B200); else TOP_E_UNSUPPORTED.
     * num_planes == 0: no polytope. */
    int32_t num_planes;
    const double* planes;
} top_constraints;

typedef struct {
    uint32_t struct_size;   /* = sizeof(top_options); lets the struct grow */
    uint32_t flags;         /* OR of TOP_WAYPOINT_*, TOP_RD_*, TOP_EPS_*, TOP_SYNC_* */
    int32_t check_every;    /* top_solve evaluates the residuals every this many sweeps (default 32) */
    int32_t device;         /* CUDA device ordinal; -1 = current device */
    int64_t max_iter;       /* top_solve gives up after this many sweeps (default 1000000) */
    void* cuda_stream;      /* cudaStream_t; NULL = default stream */
    int32_t segs_per_cta;   /* segments per thread block, 0 = choose (a tuning knob; multiple of 4) */
    int32_t lanes_per_segment; /* threads per segment of the sweep kernel: 0 = choose, 4 or 8 (a tuning knob) */
    double adapt_mu;        /* Eq. 24: mu (> 1),       0 = the paper's 10 */
    double adapt_tau_incr;  /*         tau_incr (> 1), 0 = the paper's 1.1 */
    double adapt_tau_decr;  /*         tau_decr (> 1), 0 = the paper's 1.1 */
} top_options;

/*
 * top_create -- Init of Alg. 1 (PAPER.md:L270 line 1, L301): validates, uploads the caller's arrays as they are (one
 * device allocation, one host-to-device copy), precomputes per segment the x-update operator of Eq. 20a from T_i, rho and the
 * enabled constraint sets in a kernel (double-double arithmetic; with a polytope corridor: on the host in extended precision,
 * three operators per segment), and an init kernel derives every per-lane constant and iterate 0 (reading A9: chord at
 * constant speed, z0 from the chord, duals 0, slacks/phi = projections of the chord samples).  The device work is
 * asynchronous; an operator that is not positive definite (extreme durations / rho) is reported as TOP_E_INVALID by the next
 * call that synchronises.
 *   batch        number of independent trajectories (>= 1), each with N segments
 *   N            segments per trajectory (>= 1);  s in {3,4};  dims in {1,2,3}
 *   waypoints    host [batch][N+1][dims] metres       (the path P of Alg. 1)
 *   durations    host [batch][N] seconds, > 0
 *   start_derivs host [batch][s-1][dims], derivative orders 1..s-1 at t_0, or NULL = rest (Eq. 2c)
 *   end_derivs   same at t_N
 *   cons         NULL = unconstrained
 *   rho          > 0, penalty of Eq. 5; one rho for every penalty (A18)
 *   opt          NULL = defaults
 * Errors: TOP_E_INVALID (sizes, non-finite input, T<=0, lo>=hi, rho<=0, samples < 0), TOP_E_UNSUPPORTED (samples other
 * than 0 or 8: the paper's M is a parameter; this build evaluates at 8; more than 2^28 segments),
 * TOP_E_NOMEM, TOP_E_CUDA.  A trajectory longer than the on-chip capacity of the persistent
 * kernel (top_capacity) is streamed in pieces with halo segments (temporal blocking: same results, state
 * round-trips through device memory every 64 sweeps).  On error *out is NULL; top_last_error(NULL) has the message.
 */
TOP_API top_status top_create(top_solver** out, int32_t batch, int32_t N, int32_t s, int32_t dims, top_dtype dtype,
                      const double* waypoints, const double* durations,
                      const double* start_derivs, const double* end_derivs,
                      const top_constraints* cons, double rho, const top_options* opt);

/*
 * top_reset -- a NEW PROBLEM OF THE SAME SHAPE on an existing handle: Init of Alg. 1 again (PAPER.md:L270 line 1), as a
 * re-planning loop calls it.  batch, N, s, dims, dtype, options and the constraint
 * SELECTION (box present or not, vmax > 0 or not, amax > 0 or not) are those of top_create; waypoints, durations, end
 * states, box bounds, vmax, amax and rho are new (same layouts as top_create; host pointers, copied).  Nothing is
 * allocated: one host-to-device copy of the caller's arrays, the per-segment operator recomputed by the device kernel
 * that top_create uses (polytope corridors: on the host, as in top_create), one init kernel; the iterate is iterate 0
 * again and top_iteration() restarts at 0.  Asynchronous with respect to the host.
 * Errors: TOP_E_INVALID (as top_create, or a different constraint selection), TOP_E_CUDA, TOP_E_NOMEM.
 */
TOP_API top_status top_reset(top_solver* h, const double* waypoints, const double* durations,
                     const double* start_derivs, const double* end_derivs, const top_constraints* cons, double rho);

/* top_iterate -- exactly k sweeps of Alg. 1 lines 3-13 (k >= 0; k == 0 is a no-op), enqueued on the
 * stream, no host synchronisation.  Afterwards the observable state is iterate (previous + k) and the
 * residuals are those of the last sweep. */
TOP_API top_status top_iterate(top_solver* h, int64_t k);

/* top_solve -- sweep until, for every trajectory, r_p < eps and r_d < eps (Eq. 23, PAPER.md:L283-288;
 * readings A6, A7, A8, A13), testing every check_every sweeps, or until max_iter sweeps (of this call).
 *   iters  host [batch] or NULL: sweeps done (in this call) when that trajectory first passed the test,
 *          or the total if it never did.
 * One resident trajectory: a single launch, the test (and Eq. 24 with TOP_RHO_ADAPTIVE) runs inside the kernel.
 * Batches and streamed chains: launches of check_every sweeps with the test on the host (32 bytes D2H per test); the
 * call ends when every trajectory is below eps at the same test.
 * Returns TOP_OK, TOP_NOT_CONVERGED, TOP_E_NONFINITE, TOP_E_CUDA.  Synchronises the stream. */
TOP_API top_status top_solve(top_solver* h, double eps, int64_t* iters);

/* top_set_rho -- change the penalty parameter between sweeps (the primitive under Eq. 24).  The x-update operator
 * of every segment is re-evaluated on the device for the new rho (from the rho-independent spectral form that
 * top_create precomputes in extended precision), and the SCALED duals u, v, w are multiplied by rho_old/rho_new
 * so that the multipliers y = rho*u are unchanged (reading A16; the paper is silent; Boyd et al. 3.4.1).
 * Two small kernels on the stream.  The FIRST change of rho on a handle (or TOP_RHO_ADAPTIVE at top_create) builds the
 * spectral form on the host (per-segment eigen-solves in extended precision; synchronises once).
 * TOP_E_INVALID if rho <= 0 or not finite. */
TOP_API top_status top_set_rho(top_solver* h, double rho);

/* Current penalty parameter (NaN if h is NULL). */
TOP_API double top_get_rho(const top_solver* h);

/* top_get_residuals -- residuals of the last sweep, host [batch] each, any pointer may be NULL:
 *   r_primal       || stack_i (M c_i - z~_i) ||_2  over all consensus rows (reading A7)
 *   r_dual         rho || stack_i M(T_i)'(z~_i^{k+1} - z~_i^k) ||_2   (Eq. 22, reading A8)
 *   r_dual_norm    the same with component k divided by T_i^k
 *   r_primal_gap   Eq. 21 verbatim: junction gaps only
 * NaN before the first sweep.  Synchronises the stream. */
TOP_API top_status top_get_residuals(top_solver* h, double* r_primal, double* r_dual, double* r_dual_norm,
                             double* r_primal_gap);

/* top_get_coeffs -- the trajectory C of the current iterate in the paper's basis (Eq. 18, PAPER.md:L220:
 * ascending powers of (t - t_{i-1}), seconds, global frame), layout [batch][N][dims][2s] (dim-major per
 * segment, the "squeezed" c_i of PAPER.md:L231), element type = the solver's dtype.
 * out_is_device != 0: `out` is a device pointer, written on the stream without host synchronisation. */
TOP_API top_status top_get_coeffs(top_solver* h, void* out, int32_t out_is_device);

/* top_get_state -- one field of the current iterate as host fp64 (parity tests, warm-start snapshots).
 * field / layout:  "z" [batch][N+1][n_c][dims]   "u" [batch][N][2 n_c][dims]      (n_c = s, or 2s-1 with TOP_CONSENSUS_WIDE)
 *                  "s_pos","s_neg","v_pos","v_neg","phi_v","w_v","phi_a","w_a" [batch][N][Ms][dims]
 *                  "s_poly","v_poly" [batch][N][Ms][K]   (polytope corridor: slack / scaled dual per (sample, plane))
 *                  "y_v","y_a" [batch][N][Ms]            (TOP_XUPDATE_NUMERIC: scaled multipliers of Eq. 17)
 * count = number of doubles `out` holds; TOP_E_INVALID if it does not match or the field is unknown. */
TOP_API top_status top_get_state(top_solver* h, const char* field, double* out, size_t count);

/* Checkpoint / resume (warm start).  top_snapshot_save copies the complete iterate (z~, u, slack / ball variables and
 * their duals, coefficients, residuals, sweep count, rho) into a caller-owned HOST buffer of top_snapshot_bytes(h)
 * bytes; top_snapshot_restore puts it back into a solver that was created with the same sizes, dtype and constraint
 * selection, waypoint mode and N (checked: TOP_E_INVALID otherwise).  A restore also clears the barrier time-out flag
 * of the handle.  Sweeping on from a restored snapshot reproduces the uninterrupted
 * run bit for bit.  Both synchronise the stream.  The buffer layout is private to this library version. */
TOP_API size_t top_snapshot_bytes(const top_solver* h);
TOP_API top_status top_snapshot_save(top_solver* h, void* host_buf, size_t bytes);
TOP_API top_status top_snapshot_restore(top_solver* h, const void* host_buf, size_t bytes);

/* Sweeps done since top_create. */
TOP_API int64_t top_iteration(const top_solver* h);

/* top_numeric_info -- TOP_XUPDATE_NUMERIC solvers: the number of L-BFGS iterations spent so far, summed over segments and
 * sweeps (out may be NULL).  Synchronises the stream.  TOP_E_INVALID for a closed-form solver. */
TOP_API top_status top_numeric_info(top_solver* h, int64_t* inner_iterations);

/* Launch facts of this solver (for the bench's roofline arithmetic); any pointer may be NULL:
 * CTAs per launch, threads per CTA, segments per CTA, dynamic shared memory bytes per CTA,
 * waves (launches per top_iterate call) and kernels launched so far. */
TOP_API top_status top_launch_info(const top_solver* h, int32_t* ctas, int32_t* threads, int32_t* segs_per_cta,
                           int32_t* smem_bytes, int32_t* waves, int64_t* launches);

/* Memory facts of this solver; any pointer may be NULL: bytes of its (single) device allocation, and the bytes that
 * top_create / top_reset copy host-to-device per problem (the caller's arrays and 14 KB of Gram tables; with a polytope
 * corridor also the operator rows, which are then computed on the host). */
TOP_API top_status top_memory_info(const top_solver* h, int64_t* device_bytes, int64_t* h2d_bytes_per_problem);

/* Largest N (segments of ONE trajectory) the persistent kernel can hold ON CHIP on the given device (longer
 * trajectories are streamed)
 * (-1 = current) for this s / dtype / constraint selection -- computed by the rule top_create applies to a long chain
 * (4 lanes per segment, same shared-memory reserve); < 0 on error. */
TOP_API int64_t top_capacity(int32_t device, int32_t s, top_dtype dtype, int32_t constrained);

/* top_fma_peak -- measured plain-ALU FMA throughput of the device in FLOP/s (2 per FMA) for the given
 * dtype, from a dependent-chain-free FMA loop on all SMs (the denominator of the ALU roofline).
 * Runs `reps` launches on `stream` and returns the best.  < 0 on error. */
TOP_API double top_fma_peak(int32_t device, top_dtype dtype, int32_t reps, void* cuda_stream);

/* top_precompute_operator -- the host twin (extended precision) of the per-segment operator precompute that top_create
 * runs in a kernel (and on the host for polytope corridors and for the spectral form behind top_set_rho), exposed so that
 * it can be checked without a device (it launches nothing): the x-update operator of Eq. 20a in the
 * library's internal normalised-time basis c^_a = c_a T^a, for one segment of duration T between waypoints
 * p0, p1 (host [3]):  c^ = Pm_hat (rho R^) + c0_hat.   Pm_hat host [8][8] row-major (zero padded beyond 2s),
 * c0_hat host [8][3].  flags: TOP_WAYPOINT_*.  box/vel/acc != 0 enable the constraint blocks (8 samples). */
TOP_API top_status top_precompute_operator(int32_t s, double T, double rho, int32_t box, int32_t vel, int32_t acc,
                                           uint32_t flags, const double* p0, const double* p1,
                                           double* Pm_hat, double* c0_hat);

/* top_operator_rows_static -- the x-update operator of Eq. 20a (first bracket) for up to
 * TOP_STATIC_MAX_SEGMENTS segments, computed on the GPU by the same double-double kernel that top_create runs, WITHOUT
 * ANY ALLOCATION: no cudaMalloc / cudaFree / memory-pool call, no solver handle.  It is for callers that own their device
 * buffers but may not take new ones -- a plug-in inside a host application that reserved the whole device heap at start-up,
 * a fixed-rate re-planning loop that cannot afford the device-wide synchronisation and the unbounded latency of the
 * allocator, a thread that works while another thread of the process records a CUDA graph (an allocation call would break
 * that recording), a process with a fixed memory budget.  Everything else in this header needs a solver, and top_create
 * allocates one arena per solver.
 *   device      CUDA device ordinal, -1 = the current device
 *   nseg        number of segments, 1 <= nseg <= TOP_STATIC_MAX_SEGMENTS (more: TOP_E_UNSUPPORTED; split the call)
 *   s           3 (jerk) or 4 (snap)
 *   durations   HOST [nseg] seconds, finite and > 0 (copied inside the call)
 *   rho         > 0, penalty of Eq. 5
 *   box/vel/acc != 0: the penalty blocks of the box corridor / velocity ball / acceleration ball at the 8 sample times
 *               are part of the operator (readings A10, A11)
 *   flags       one TOP_WAYPOINT_* mode
 *   rows_out    DEVICE buffer of the selected device, 64 * nseg doubles, caller-owned and caller-allocated:
 *               rows_out[(b * nseg + g) * 8 + a] = rho * Pm_hat_g[a][b] (Pm_hat is symmetric), the operator of segment g in the
 *               normalised-time basis c^_a = c_a T^a -- rho times the Pm_hat that top_precompute_operator returns on the host
 *               for T = durations[g] -- zero for a >= 2s or b >= 2s
 *   cuda_stream the work is enqueued on this stream (NULL = legacy default stream) and the call waits for it: on return
 *               rows_out is complete and `durations` may be freed.
 * Where the working memory is.  The kernel's scratch (28 KB of Gram tables, the device copy of the durations, a status word;
 * 156.25 KB in all) is a static array inside libtop.so's device image: every GPU on which the process uses this library
 * holds it from module load to process exit, whether or not this function is ever called.  TOP_STATIC_MAX_SEGMENTS is what
 * that array was sized for.
 * First call.  The first call on each device looks up the array's device address and fills the Gram tables with one
 * synchronous copy (and, as for any kernel, the driver loads the code on first launch).  Make that first call during
 * start-up, before any stream capture begins; later calls enqueue two small copies, a memset and two kernels.
 * Sharing.  Every call on a device uses the same array, and the array keeps what the last call left in it (the call itself
 * re-zeroes the status word).  Two calls that ran on the GPU at the same time would overwrite each other's durations and
 * status: the library therefore holds a per-device lock for the whole (synchronous) call, so calls on one device are
 * serialised, from whatever threads and streams they come.  Different processes have separate copies of the array.
 * Errors: TOP_E_INVALID (arguments; rows_out is not device memory of that device; an operator that is not positive
 * definite -- rows_out is then unspecified), TOP_E_UNSUPPORTED (nseg beyond the maximum), TOP_E_CUDA.  The message is in
 * top_last_error(NULL). */
#define TOP_STATIC_MAX_SEGMENTS 16384
TOP_API top_status top_operator_rows_static(int32_t device, int32_t nseg, int32_t s, const double* durations, double rho,
                                            int32_t box, int32_t vel, int32_t acc, uint32_t flags, double* rows_out,
                                            void* cuda_stream);

TOP_API top_status top_destroy(top_solver* h);

/* Message of the last failing call on this handle (h == NULL: of the last failing top_create on this
 * thread).  Never NULL. */
TOP_API const char* top_last_error(const top_solver* h);

#ifdef __cplusplus
}
#endif
#endif /* TOP_H */
