// top_internal.h -- structures shared by the host side (top_api.cpp) and the kernels (top_kernels.cu).
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace top {

constexpr int LANES = 8;        // threads per segment: lane j <-> sample j, lane a <-> coefficient / consensus row a
constexpr int MS = 8;           // samples per segment (Ms)
constexpr int MAXN = 8;         // n = 2s <= 8
constexpr int DIMS = 3;         // flat dimensions are padded to 3 (unused ones carry zeros)
constexpr int KMAX = 16;        // general polytope corridor: at most this many half-spaces per segment

// segment flags
constexpr uint8_t SEG_FIRST = 1;  // first segment of its trajectory: left junction (z_0) is fixed
constexpr uint8_t SEG_LAST = 2;   // last segment: right junction (z_N) is fixed

// kernel flags
constexpr uint32_t KF_BOX = 1, KF_VEL = 2, KF_ACC = 4, KF_PIN_POS = 8 /* PINNED_Z: position row of z held */,
                   KF_NEIGHBOUR_SYNC = 16, KF_PAIRWISE = 32 /* warp-pair named barriers instead of the CTA barrier */,
                   KF_OPEN_LEFT = 64, KF_OPEN_RIGHT = 128 /* streaming: the launch range starts / ends inside a chain (halo) */,
                   KF_POLY = 256 /* general polytope corridor (K planes per segment, rotated per-segment frame) */,
                   KF_WIDE = 512 /* paper-literal consensus n_c = 2s-1: a second block of consensus rows (orders s..2s-2) */,
                   KF_CLUSTER = 1024 /* the launch is ONE thread-block cluster: boundary rows go through distributed shared memory */;

// Per-lane field arrays: element [f * stride + gseg * LANES + lane]; stride = padded lane count.
// "Real" is double (TOP_F64) or float (TOP_F32); the x-update operator is always double.
struct KParams {
    // ---- constants (read only)
    const double* Pm;       // [MAXN][stride]  row `lane` of rho * Pm_hat (normalised-time basis), zero padded
    const double* c0;       // [DIMS][stride]  row `lane` of c0_hat
    const void* invTk;      // Real [stride]   1 / T^k, k = derivative order of consensus row `lane`
    const void* Tpow;       // Real [stride]   T^lane (physical-time scaling of the dual residual, Eq. 22)
    const void* invT;       // Real [2][nseg_pad]  1/T, 1/T^2 per segment
    const void* lohi;       // Real [6][nseg_pad]  lo[3], hi[3] per segment
    const uint8_t* segflags;// [nseg_pad]
    const void* zoff;       // Real [DIMS][stride]  frame shift added to the neighbour's row (position rows only)
    // ---- state of iterate k (read at launch start, written at launch end)
    void* zt;               // Real [DIMS][stride]  consensus row `lane` of z~_i = (z_{i-1}; z_i)
    void* u;                // Real [DIMS][stride]  scaled dual of that row (Eq. 20c)
    void* qp;               // Real [DIMS][stride]  box + side: S+ = max(0,q), V+ = max(0,-q)  (Moreau pair)
    void* qn;               // Real [DIMS][stride]  box - side
    void* phv;              // Real [DIMS][stride]  phi of the velocity ball (Eq. 20f)
    void* wv;               // Real [DIMS][stride]  its scaled dual (Eq. 20g)
    void* pha;              // Real [DIMS][stride]
    void* wa;               // Real [DIMS][stride]
    void* chat;             // Real [DIMS][stride]  coefficient row `lane` in normalised time (c^_a = c_a T^a)
    // where the iterate is written at launch end (= the input arrays except in streaming mode: ping-pong buffers)
    void *zt_out, *u_out, *qp_out, *qn_out, *phv_out, *wv_out, *pha_out, *wa_out;
    // ---- exchange / reduction
    void* Bedge;            // mailbox [2 parity][max_ctas][2 sides][4][DIMS] x 16-byte LL slots: boundary rows at CTA edges
    double* part;           // [nseg_pad][4]  per-segment residual partial sums (rp2, rd2, rdn2, gap2)
    unsigned long long* bar;// [0] grid barrier counter (reset before each launch)
    int* abort_flag;        // set when a barrier wait times out
    // ---- sizes
    long long stride;       // lanes per field (>= nseg_pad * LANES)
    long long nseg_pad;
    long long seg_begin, seg_end;   // global segment range of this launch (a wave of whole trajectories)
    long long own_begin, own_end;   // segments whose results are written back (streaming: range minus its halos)
    int segs_per_cta;
    int k_sweeps;
    int split_octets;       // tensor-core kernel, SPLIT instantiation: the last this-many octets of a CTA run on three warps each
    uint32_t flags;
    int max_ctas;
    unsigned int seq_base;  // sweeps launched before this launch (mod 2^32): mailbox sequence numbers never repeat
    double rho, vmax, amax;
    // ---- in-kernel solve (cadmm_sweeps_kernel only; check_every == 0: plain k sweeps)
    int check_every;        // test the stop rule (Eq. 23) inside the kernel every this many sweeps
    int rd_sel;             // which dual residual is tested: 1 = Eq. 22, 2 = normalised
    int adaptive;           // apply Eq. 24 after every test
    int q;                  // spectral components (operator refresh)
    double tol, mu, tau_incr, tau_decr;
    void* resbox;           // [2][max_ctas][4] LL slots: per-CTA residual partial sums, all-gathered by every CTA
    double* solve_out;      // [8]: sweeps done, stopped (0/1), rho, r_p, r_d, r_d_norm, r_p_gap, unused
    const double *W, *lam, *g0, *dp;   // spectral operator data (RefreshParams)
    // ---- general polytope corridor (KF_POLY; fp64 tensor-core kernel only).  Every segment works in its own rotated frame
    // y = V'(p - o_i), V = eigenvectors of sum_k a_k a_k': there the dims decouple again (one operator per dim, Pm is
    // [DIMS][MAXN][stride]); consensus rows are rotated in and out, the planes are stored rotated.
    const double* rot;      // [9][nseg_pad]          V row-major: V[d][e] = component d (global) of axis e (rotated)
    const double* planes;   // [K][4][nseg_pad]       a'_k = V'a_k (3), b'_k = b_k - a_k'o_i
    void* qpl;              // double [K][stride]     Moreau value of (sample `lane`, plane k): s = max(0,q), v = max(0,-q)
    void* qpl_out;
    int K;
    // ---- paper-literal consensus n_c = 2s-1 (KF_WIDE; fp64 tensor-core kernel only): the second block of consensus rows.
    // Slot t < 4 of a segment = start-boundary row of derivative order s + t, slot 4 + t = end-boundary row of that order
    // (t <= s-2); invTk2 = 1/T^(s+t), and 0 for slots / rows that do not exist (reading A1).  Read and written in place.
    const void* invTk2;     // Real [stride]
    void* zt2;              // Real [DIMS][stride]
    void* u2;               // Real [DIMS][stride]
};

struct ConvParams {       // coefficient conversion to the paper's basis (Eq. 18)
    const double* rot;    // [9][nseg_pad] or null: rotate the dims back to the global frame first (polytope corridor)
    const void* chat;     // Real [DIMS][stride]
    const void* invT;     // Real [2][nseg_pad]
    const double* origin; // [3][nseg_pad]  origin of each segment's local frame (added to c_0)
    long long nseg_pad;
    void* out;            // Real [nseg][dims][2s]
    long long stride, nseg;
    int s, dims;
};

// launchers (top_kernels.cu).  dtype: 0 = f64, 1 = f32.  Return cudaError_t.
// 8 lanes per segment (cadmm_sweeps_kernel); the 4-lane kernel is cadmm_sweeps_mma_kernel below
cudaError_t launch_sweeps(const KParams& p, int dtype, int s, bool constrained, int lanes, int ctas, int threads,
                          size_t smem, cudaStream_t st);
size_t sweep_smem_bytes(int dtype, int s, bool constrained, int lanes, int segs_per_cta);
int max_threads_for(int dtype, int lanes);
cudaError_t sweep_kernel_limits(int dtype, int s, bool constrained, int lanes, int threads, size_t smem, int* max_ctas_per_sm);
// fp64 tensor-core variant of the 4-lane kernel (top_kernels_mma.cu: cadmm_sweeps_mma_kernel)
cudaError_t launch_sweeps_mma(const KParams& p, int dtype, int s, int ctas, int threads, size_t smem, cudaStream_t st);
// how many trailing octets of a CTA does a launch with these flags run on three warps each (top_kernels_mma.cu, "split
// octets")?  0 = none; the launch then has threads + 64 * that many threads per CTA
int split_octets_for(uint32_t kparam_flags, int check_every, int dtype, int ctas, int threads);
// can this problem use the SPLIT instantiation at all (fp64, box + velocity [+ acceleration], no polytope / wide consensus)?
bool split_supported(uint32_t kflags, int dtype);
size_t sweep_smem_bytes_mma(int dtype, bool constrained, bool poly, bool wide = false);
int max_threads_mma(int dtype, bool poly, bool wide = false);
cudaError_t sweep_kernel_limits_mma(int dtype, int s, uint32_t kflags, int threads, size_t smem, int* max_ctas_per_sm);
cudaError_t sweep_cluster_limits_mma(int dtype, int s, uint32_t kflags, int ctas, int threads, size_t smem, int* nclusters);
cudaError_t launch_convert(const ConvParams& p, int dtype, cudaStream_t st);
// rho Pm^ = W diag(rho/(lambda_i+rho)) W',  c0^ = c_chord - (rho Pm^) g0   (spectral form; top_api.cpp build_spectral)
struct RefreshParams {
    const double* W;      // [MAXN i][stride]  W[lane][i]
    const double* lam;    // [MAXN i][nseg_pad]
    const double* g0;     // [DIMS][stride]    (G c_chord)[lane][d]
    const double* dp;     // [DIMS][nseg_pad]  p_i - p_{i-1} (c_chord row 1; HARD mode), else zeros
    double* Pm;           // out [MAXN b][stride]
    double* c0;           // out [DIMS][stride]
    long long stride, nseg_pad, nseg;
    int q;                // number of spectral components (n-2 in HARD mode, else n)
    double rho;
};
cudaError_t launch_refresh_operator(const RefreshParams& p, cudaStream_t st);
// The x-update operator of Eq. 20a (first bracket) on the device, one thread per segment, in double-double
// arithmetic (106-bit significand: the host path uses the 64-bit significand of long double): H^ from the Gram tables
// of the constant normalised-time rows weighted by powers of 1/T_i, the waypoint equalities eliminated with the null-space
// basis (HARD), symmetric scaling by powers of two, Gauss-Jordan, rho * Pm^ rounded to fp64 into the per-lane layout.
constexpr int GRAM_TABLES = 14;      // Q1 | Gc[0..3] | Ge[0..2] | Gw[start][0..2] | Gw[end][0..2]
struct GramDD { double hi[GRAM_TABLES][MAXN * MAXN], lo[GRAM_TABLES][MAXN * MAXN]; };
struct PrecompParams {
    const GramDD* gram;           // device
    const double* durations;      // [nseg] (device copy of the caller's array)
    double* Pm;                   // out [MAXN b][stride]: element b of row `lane` of rho * Pm^
    long long stride, nseg;
    int N, s, hard, box, vel, acc, wide;
    double rho;
    int* bad;                     // set to 1 when a segment's operator is not positive definite
};
cudaError_t launch_precompute_operator(const PrecompParams& p, cudaStream_t st);
// host helpers of top_api.cpp for the entry point that lives outside it (top_static_scratch.cu): the Gram tables of
// order s in {3, 4} split into double-double, and the message behind top_last_error(NULL) (returns `status`)
void gram_tables_dd(int s, GramDD* out);
int report_error(int status, const char* msg);
// NumericSolve branch (top_kernels_numeric.cu): one sweep = x-update kernel + consensus kernel.  fp64 only.
struct NumParams {
    const double* Pm;         // [MAXN][stride] rho * Pm^ rows of the QUADRATIC part (no ball terms)
    const double* invT;       // [2][nseg_pad]
    const double* lohi;       // [6][nseg_pad]
    const double* origin;     // [3][nseg_pad]
    const uint8_t* segflags;
    const double* zoff;       // [3][stride]
    const double* Tpow;       // [stride]
    double *zt, *u, *qp, *qn, *chat;   // [3][stride] each (qp, qn: box only)
    double *yv, *ya;          // [stride] scaled multipliers of Eq. 17 (lane j = sample j)
    double* bnd;              // [3][stride] boundary rows B = M c of the newest coefficients
    double* part;             // [nseg_pad][4]
    unsigned long long* inner_iters;   // L-BFGS iterations, summed over segments and sweeps
    unsigned int* work_counter;        // work queue of the x-update kernel (next segment to fetch; reset by the consensus kernel)
    int max_blocks;                    // persistent grid of the x-update kernel: CTAs that are co-resident (3 per SM)
    long long stride, nseg_pad, nseg;
    int s, hard;
    uint32_t flags;           // KF_BOX | KF_VEL | KF_ACC | KF_PIN_POS
    double rho, vmax, amax;
};
cudaError_t launch_numeric_sweep(const NumParams& p, cudaStream_t st);
// Init of Alg. 1 (PAPER.md:L270 line 1, L301; reading A9) on the device: from the caller's arrays (uploaded as they are)
// and the per-segment operator rows, every per-lane constant and iterate 0.
struct InitParams {
    // the caller's arrays (device copies)
    const double* waypoints;      // [batch][N+1][dims]
    const double* durations;      // [batch][N]
    const double* box_lo;         // [batch][N][dims] or null
    const double* box_hi;
    const double* start_derivs;   // [batch][s-1][dims] or null = rest
    const double* end_derivs;
    // column 1 of the Gram matrix G of the penalty rows (G e_1 = sum_k T^-2k gc1[k] + 2 ge1[0] + T^-2 ge1[1] + T^-4 ge1[2],
    // the enabled blocks only): constants per s, the T weights are applied per segment
    double gc1[4][MAXN], ge1[3][MAXN];
    const double* Pm;             // [MAXN][stride] rho Pm^ rows (host precompute)
    // outputs
    double *c0, *g0, *dp, *origin;
    void *invTk, *Tpow, *invT, *lohi, *zoff, *zt, *chat, *qp, *qn, *phv;
    void* invTk2;                 // wide consensus (n_c = 2s-1): 1/T^(s+t) per slot of the second row block, 0 where no row exists; or null
    // polytope corridor: rotation and rotated planes (host precompute), per-dim box weight lambda_d (eigenvalues of sum a a'),
    // and the Moreau values of the chord samples (output)
    const double *rot, *planes, *lam3;   // [9][nseg_pad], [K][4][nseg_pad], [3][nseg_pad]
    double* qpl;                          // [K][stride]
    int K, has_poly, c0_only;
    uint8_t* segflags;
    long long stride, nseg_pad, nseg;
    int N, batch, s, dims, hard, has_box, has_vel, has_acc;
    double vmax;
};
cudaError_t launch_init(const InitParams& p, int dtype, cudaStream_t st);
// duals *= ratio after a change of rho: u, w (both balls), and the negative part of the Moreau values q (= -v)
struct RescaleParams { void *u, *qp, *qn, *wv, *wa; long long count; double ratio; void* qpl; long long qpl_count; void* u2;
                       double *yv, *ya; long long y_count; /* NumericSolve: multipliers of Eq. 17, [stride] each */ };
cudaError_t launch_rescale_duals(const RescaleParams& p, int dtype, cudaStream_t st);
cudaError_t launch_residual_reduce(const double* part, double* res, long long N, int batch, cudaStream_t st);
cudaError_t launch_fma_peak(int dtype, int blocks, int threads, long long iters, float* sink, cudaStream_t st);

}  // namespace top
