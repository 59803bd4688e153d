// top_kernels_mma.cu -- the fp64 CADMM sweep with its constant-matrix contractions on the tensor cores.
//
// Same sweep, same global-memory layout, same exchange protocol as cadmm_sweeps_kernel (top_kernels.cu), but FOUR lanes
// per segment, lane t owns inequality samples {t, t+4} and coefficient / consensus rows {t, t+4}; 8 segments per
// warp.  What differs is how the two contractions with CONSTANT matrices are done.  In the normalised-time basis
// (c^_a = c_a T^a) the evaluation matrices of Eq. 19 are the same for every segment:
//     a1  R^ = [M^' E0' E1' E2'] G        (Eq. 20a second bracket)   8 x 32 constant, G 32 x 3 per segment
//     a3  [B; P; V; A] = [M^; E0; E1; E2] c^   (Eq. 20b, 20d-g)   32 x 8 constant, c^ 8 x 3 per segment
// Both are issued as mma.sync.aligned.m8n8k4.f64 (DMMA) with the (segment, dim) pairs of the warp as the M dimension
// (8 segments x 3 dims = three m-tiles) and the constant matrix as the B operand, held in registers for the whole
// launch.  The fragment layout of m8n8k4 puts row g of the A operand in lanes 4g..4g+3 and column k in lane 4g + (k%4):
// exactly "lane t of segment g supplies its own items t, t+4", so operands are taken from the lane's own registers and
// results land in the lane that owns them: no shuffle reduce-scatter, no select instructions, no second all-gather.
// The only intra-segment exchange left is the all-gather of R^ (8 rows x 3 dims through shared memory) in front of the
// per-segment 8 x 8 operator apply a2 (Eq. 20a first bracket), which stays on DFMA: its matrix differs per segment.
// Measured on B200: DMMA m8n8k4 runs at the DFMA FLOP rate on the SAME pipe (16 cycles per instruction
// and scheduler, 26-cycle dependent latency, the issuing warp waits ~17 cycles after each), so the gain is not FLOPs
// but everything around them: the shuffle / select / synthetic-division form was bound by instruction issue and
// dependent-chain latency.
//
// Data flow of one lane (registers are short at 9 warps per SM: 168):
//   registers   the a1 OPERANDS gM, A0, gv, ga (the A fragments of the first contraction), each produced where its
//               inputs are updated (phase B, projections) so that a1 is 24 back-to-back MMAs with nothing in front
//   shared      the variables behind them, as pairs read and written once per sweep where they are updated:
//               (z~, u), the Moreau pair values (q+, q-), the ball variables (phi_v, phi_a) and (w_v, w_a);
//               the per-segment operator rows; the all-gather buffer; the boundary-row exchange buffer
// The constraint selection is a template parameter (the three combinations BASELINE.json's configs use, plus a
// run-time-flag variant for the others): no branch inside the sweep body except the exchange.
#include <stdlib.h>
#include <string.h>

#include "top_device.cuh"

namespace top {

namespace {

// D (8x8, lane (g,t): row g, cols 2t, 2t+1) += A (8x4, lane (g,t): row g, col t) * B (4x8, lane (g,t): row t, col g)
__device__ __forceinline__ void dmma884(double& d0, double& d1, double a, double b) {
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(d0), "+d"(d1) : "d"(a), "d"(b));
}

// A operand of one k-block of a contraction (the lane's two items x three dims), B operand (the two k-steps of the constant
// matrix that go with them), and the accumulator tiles of one contraction output: value (dim d, column 2t + j).
// TOP_F32 feeds fp32-rounded operands to the same fp64 tensor instructions (fp64 accumulation).  [Tried and dropped for
// TOP_F32: mma.sync m16n8k8 tf32 with the 3-term split a_hi b_hi + a_lo b_hi + a_hi b_lo on the regular tensor pipe -- 8 cycles
// per instruction and scheduler against 16 for DMMA, measured, and it frees the fp64 pipe; parity green, but config 5 ran at
// 5.9e9 instead of 6.5e9 segment-iterations/s: that kernel is bound by shared-memory wavefronts (73 % of peak, ncu) and
// issue slots, not by the fp64 pipe, and the split adds ~90 instructions per lane and sweep.]
struct AOp { double v[2][3]; };
struct BOp { double b0, b1; };
template <typename Real>
__device__ __forceinline__ AOp make_aop(const Real (&op)[2][3]) {
    AOp a;
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int d = 0; d < 3; ++d) a.v[h][d] = (double)op[h][d];
    return a;
}
struct Acc {
    double v[3][2] = {{0, 0}, {0, 0}, {0, 0}};
    __device__ __forceinline__ void blk(const AOp& a, const BOp& b) {
#pragma unroll
        for (int d = 0; d < 3; ++d) dmma884(v[d][0], v[d][1], a.v[0][d], b.b0);
#pragma unroll
        for (int d = 0; d < 3; ++d) dmma884(v[d][0], v[d][1], a.v[1][d], b.b1);
    }
    __device__ __forceinline__ double get(int d, int j) const { return v[d][j]; }
};

// 1/sqrt(x) for x > 0, normal: the hardware seed (MUFU.RSQ64H, ~2^-22 relative) and ONE cubically convergent step
// y (1 + e/2 + 3e^2/8), e = 1 - x y^2  =>  error ~ e^3: full double precision (a few ulp), 5 fp64 operations and no
// branch.  The library rsqrt() adds special-case branches that keep ptxas from interleaving independent projections.
__device__ __forceinline__ double rsqrt_pos(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-x * y, y, 1.0);
    return fma(y * e, fma(0.375, e, 0.5), y);
}

// max(-q, 0) on the integer pipe (the fp64 pipe is the bound of this kernel): -q where the sign bit of q is set, else +0
__device__ __forceinline__ double neg_part(double q) {
    const int hi = __double2hiint(q), lo = __double2loint(q);
    const int m = hi >> 31;
    return __hiloint2double((hi ^ 0x80000000) & m, lo & m);
}

__device__ __forceinline__ float rsqrt_pos(float x) { return rsqrtf(x); }
__device__ __forceinline__ float neg_part(float q) {
    const int b = __float_as_int(q);
    return __int_as_float((b ^ 0x80000000) & (b >> 31));
}

// Eq. 20f without a branch: the factor min(1, bound/||y||) of the projection of y onto ||.|| <= bound (reading A15)
template <typename Real>
__device__ __forceinline__ Real ball_scale(const Real (&y)[3], Real bound) {
    const Real n2 = fma(y[2], y[2], fma(y[1], y[1], y[0] * y[0]));      // (spelled out: the split-tail warps must round the same way)
    const Real sc = bound * rsqrt_pos(n2);                 // garbage (inf/NaN) when n2 == 0: not selected then
    return n2 > bound * bound ? sc : (Real)1;
}

// residual partial sums of one (row, dim) / one dim, spelled out with fma so that every path adds them in the same order
__device__ __forceinline__ void rp_accum(double& rp2, double& gap2, double res, bool gaprow, double own, double nb) {
    rp2 = fma(res, res, rp2);
    if (gaprow) { const double gp = own - nb; gap2 = fma(gp, gp, gap2); }      // Eq. 21
}
__device__ __forceinline__ void rd_accum(double& rd2, double& rdn2, double xr0, double xr1, double Tp0, double Tp1) {
    rdn2 = rdn2 + fma(xr1, xr1, xr0 * xr0);
    const double a = xr0 * Tp0, b = xr1 * Tp1;
    rd2 = rd2 + fma(b, b, a * a);
}

// the state of a lane lives in shared memory as pairs
template <typename Real> struct Pair;
template <> struct Pair<double> { typedef double2 type; };
template <> struct Pair<float> { typedef float2 type; };
__device__ __forceinline__ double2 make2(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ float2 make2(float a, float b) { return make_float2(a, b); }

// y = V'x (global -> rotated frame of the segment) and x = V y (back); V row-major 3x3 in shared memory
__device__ __forceinline__ void rot_in(const double* V, double (&x)[3]) {
    const double a = x[0], b = x[1], c = x[2];
#pragma unroll
    for (int e = 0; e < 3; ++e) x[e] = V[0 * 3 + e] * a + V[1 * 3 + e] * b + V[2 * 3 + e] * c;
}
__device__ __forceinline__ void rot_out(const double* V, double (&y)[3]) {
    const double a = y[0], b = y[1], c = y[2];
#pragma unroll
    for (int d = 0; d < 3; ++d) y[d] = V[d * 3 + 0] * a + V[d * 3 + 1] * b + V[d * 3 + 2] * c;
}

// one instantiation: <= 288 threads (9 warps of 8 segments; 3 warps on one scheduler: 168 registers per thread)
constexpr int MAXT_MMA = 288;
constexpr int MAXT_MMA_F32 = 384;
// constraint mask of an instantiation: KF_BOX | KF_VEL | KF_ACC, or CM_RUNTIME = read the flags at run time
constexpr int CM_RUNTIME = 8;

// polytope corridor instantiations: <= 160 threads (5 warps: 40 segments; the per-plane state needs the shared memory)
constexpr int MAXT_MMA_POLY = 160;
// paper-literal consensus n_c = 2s-1 (reading A1): a second block of consensus rows per segment (orders s..2s-2 at both
// boundaries: (z~, u) pairs, boundary-row buffer, mailbox slots); <= 224 threads (7 warps: 56 segments)
constexpr int MAXT_MMA_WIDE = 224;
// both at once (the paper's literal configuration: FIRI polytope corridor + 2s-1 consensus orders): <= 128 threads (32 segments)
constexpr int MAXT_MMA_POLY_WIDE = 128;
constexpr int PSTR = KMAX * 4 + 2;      // doubles per segment of the plane table (padded: the 8 segments of a warp hit distinct banks)
constexpr int VSTR = 10;                // doubles per segment of the rotation table

struct SmemLayoutMma {
    size_t pm, c0, zu, qs, ws, ph, ctab, lohi, xs, bs, zoff, qpl, pls, vs, zu2, bs2, total;
};
__host__ __device__ inline SmemLayoutMma smem_layout_mma(bool cons, int segs_alloc, bool poly = false, int rb = 8, bool wide = false) {
    SmemLayoutMma L;
    const int T = segs_alloc * 4;
    size_t off = 0;
    L.pm = off;   off = align16(off + (size_t)(poly ? 3 : 1) * 2 * 4 * T * sizeof(double2));   // rho*Pm^ rows, [d (poly)][h][b/2][thread] pairs
    L.c0 = off;   off = align16(off + (size_t)6 * T * sizeof(double));                 // c0^ rows, [h][d][thread]
    L.zu = off;   off = align16(off + (size_t)6 * T * 2 * rb);                // (z~, u) of the lane's two consensus rows, [h][d][thread]
    L.qs = off;   off = align16(off + (size_t)(cons && !poly ? 6 : 0) * T * 2 * rb);   // Moreau pair values (q+, q-) of the lane's two samples (box)
    L.ws = off;   off = align16(off + (size_t)(cons ? 6 : 0) * T * 2 * rb);   // ball duals (w_v, w_a) of the lane's two samples
    L.ph = off;   off = align16(off + (size_t)(cons ? 6 : 0) * T * 2 * rb);   // ball variables (phi_v, phi_a)
    L.ctab = off; off = align16(off + (size_t)20 * 32 * sizeof(double));               // constant MMA operands, [16 (+4: wide consensus)][lane of warp]
    L.lohi = off; off = align16(off + (size_t)(cons && !poly ? 6 : 0) * segs_alloc * rb);
    L.xs = off;   off = align16(off + (size_t)segs_alloc * XSTRIDE * sizeof(double));  // rhs rows, all-gather
    L.bs = off;   off = align16(off + (size_t)2 * (segs_alloc + 2) * 24 * rb);   // boundary rows, double buffered
    L.zoff = off; off = align16(off + (size_t)6 * segs_alloc * rb);        // frame shift of the neighbours' position rows
    L.qpl = off;  off = align16(off + (size_t)(poly ? KMAX * 2 : 0) * T * sizeof(double));          // Moreau values per (plane, sample of the lane)
    L.pls = off;  off = align16(off + (size_t)(poly ? segs_alloc : 0) * PSTR * sizeof(double));     // rotated planes (a'_k, b'_k) per segment
    L.vs = off;   off = align16(off + (size_t)(poly ? segs_alloc : 0) * VSTR * sizeof(double));     // rotation V per segment
    L.zu2 = off;  off = align16(off + (size_t)(wide ? 6 : 0) * T * 2 * rb);                         // (z~, u) of the lane's two rows of the second consensus block
    L.bs2 = off;  off = align16(off + (size_t)(wide ? 2 : 0) * (segs_alloc + 2) * 24 * rb);         // boundary rows of the second block, double buffered
    L.total = off;
    return L;
}

// Operator refresh of one coefficient row inside the solve kernel (Eq. 24 changed rho): row `row` of rho Pm^ and of c0^ from
// the rho-independent spectral data, as refresh_operator_kernel does for the arrays.  Rare path: kept out of line so
// that its registers do not count against the sweep loop.
template <int N2, int TS>
__device__ __noinline__ void refresh_operator_rows(const KParams& p, long long gseg, long long gt, int row, double rho_new,
                                                   double2* pm_row /* [4 pairs] stride TS */, double* c0_row /* [3] stride TS */) {
    double wd[MAXN];
    for (int i = 0; i < MAXN; ++i) {
        const double lam = i < p.q ? p.lam[i * p.nseg_pad + gseg] : 0.0;
        wd[i] = i < p.q ? p.W[i * p.stride + gt] * (rho_new / (lam + rho_new)) : 0.0;
    }
    double c0n[3];
    for (int d = 0; d < 3; ++d) c0n[d] = row == 1 ? p.dp[d * p.nseg_pad + gseg] : 0.0;
    for (int b = 0; b < 8; b += 2) {
        double v2[2];
        for (int e = 0; e < 2; ++e) {
            double v = 0.0;
            if (b + e < N2) for (int i = 0; i < p.q; ++i) v += wd[i] * p.W[i * p.stride + gseg * LANES + b + e];
            v2[e] = v;
            for (int d = 0; d < 3; ++d) c0n[d] -= v * p.g0[d * p.stride + gseg * LANES + b + e];
        }
        pm_row[(b >> 1) * TS] = make_double2(v2[0], v2[1]);
    }
    for (int d = 0; d < 3; ++d) c0_row[d * TS] = c0n[d];
}

// In-kernel stop rule, the CTA-wide part (every thread of the CTA calls it on a test sweep, after the per-octet partial sums are in
// wsum_sh): CTA partial in a fixed order, all-gather of the per-CTA partials through LL slots (every CTA reads all of them and
// adds them in the same order, so all CTAs take the same decision from the same numbers), Eq. 23, Eq. 24.
// Returns true when the launch ends here (converged: stopped = 1; or a failed gather / non-finite residual); otherwise rho_new is
// the penalty of the next sweep (== rho_cur unless Eq. 24 moved it).
// KF_CLUSTER: the all-gather goes through distributed shared memory -- every CTA stores its four sums straight into the result
// box of EVERY CTA of the cluster (cresbox: [2 parity][16 CTAs][4] LL slots in each CTA's shared memory) and polls its own copy:
// one one-way DSMEM store instead of an L2 round trip with polling (a test sweep of config 2: 3.6 -> 2.x us).
constexpr int CRES_BYTES = 2 * 16 * 4 * 16;
__device__ __forceinline__ bool solve_decide(const KParams& p, unsigned seq, int noct, double (*wsum_sh)[4], double (*allp_sh)[4], double* tot_sh,
                                             unsigned char* cresbox, int& ncheck, double rho_cur, double& rho_new, int& stopped) {
    const int tid = threadIdx.x, T = blockDim.x, cta = blockIdx.x, nctas = gridDim.x;
    const bool clus = (p.flags & KF_CLUSTER) != 0;
    __syncthreads();
    unsigned char* const rb = static_cast<unsigned char*>(p.resbox) + (size_t)(ncheck & 1) * p.max_ctas * 4 * 16;
    const unsigned cres_local = smem_u32(cresbox), cpar = (unsigned)((ncheck & 1) * 16 * 4 * 16);
    if (clus) {
        // lanes 0..3 of every warp add the octets' sums of quantity k = lane in the same fixed order; thread t delivers quantity
        // t & 3 to CTA t >> 2
        double acc = 0.0;
        if ((tid & 31) < 4) for (int w = 0; w < noct; ++w) acc += wsum_sh[w][tid & 3];
        acc = __shfl_sync(0xffffffffu, acc, tid & 3);
        for (int t = tid; t < nctas * 4; t += T)
            ll_store_cluster(cluster_map(cres_local, (unsigned)(t >> 2)) + cpar + (unsigned)((cta * 4 + (t & 3)) * 16), acc, seq);
    } else if (tid == 0) {
        for (int k = 0; k < 4; ++k) {
            double acc = 0.0;
            for (int w = 0; w < noct; ++w) acc += wsum_sh[w][k];
            ll_store(rb + ((size_t)cta * 4 + k) * 16, acc, seq);
        }
    }
    int gather_failed = 0;
    for (int tt = tid; tt < nctas; tt += T) {
        const long long t0 = global_ns();
        unsigned spins = 0;
        for (int k = 0; k < 4; ++k) {
            LLRaw r;
            const unsigned cslot = cres_local + cpar + (unsigned)((tt * 4 + k) * 16);
            if (clus) ll_issue_smem(cslot, r); else ll_issue(rb + ((size_t)tt * 4 + k) * 16, r);
            while (!ll_ok(r, seq)) {
                if ((++spins & 255u) == 0 && (*(volatile int*)p.abort_flag || global_ns() - t0 > WAIT_TIMEOUT_NS)) {
                    atomicExch(p.abort_flag, 1); gather_failed = 1; break;
                }
                if (clus) ll_issue_smem(cslot, r); else ll_issue(rb + ((size_t)tt * 4 + k) * 16, r);
            }
            allp_sh[tt][k] = ll_value(r);
        }
    }
    gather_failed = __syncthreads_or(gather_failed);
    if (tid < 4) {
        double acc = 0.0;
        for (int tt = 0; tt < nctas; ++tt) acc += allp_sh[tt][tid];
        tot_sh[tid] = acc;
    }
    __syncthreads();
    ++ncheck;
    const double rp = sqrt(tot_sh[0]), rd = sqrt(tot_sh[p.rd_sel]);
    const bool conv = rp < p.tol && rd < p.tol;
    if (conv || gather_failed || !(rp == rp) || !(rd == rd)) { stopped = conv ? 1 : 0; return true; }
    rho_new = rho_cur;
    if (p.adaptive) {      // Eq. 24
        if (rp > p.mu * rd) rho_new = rho_cur * p.tau_incr;
        else if (rd > p.mu * rp) rho_new = rho_cur / p.tau_decr;
    }
    return false;
}

// Constant operands of the two contractions, written once per launch by the first warp of the CTA (ctab = table base + lane of warp).
template <int S, bool WIDE>
__device__ __forceinline__ void fill_ctab(double* ctab, int lane32) {
    constexpr int N2 = 2 * S;
    const int lane = lane32 & 3, grp = lane32 >> 2;
    // ---- constant operands of the two contractions (B fragments: row k = 4*kstep + lane, column n = grp)
    // a1: k runs over the 32 items [consensus rows | E0 samples | E1 samples | E2 samples], n = coefficient row
    // a3: k = coefficient row, n runs over the items of one block, permuted so that the accumulator columns
    //     2*lane, 2*lane+1 are the lane's own items lane, lane+4
    {
        const int a = grp;
#pragma unroll
        for (int kk = 0; kk < 8; ++kk) {
            const int b = kk >> 1, item = lane + 4 * (kk & 1);
            const double tau = (double)(item + 1) / (double)(MS + 1);       // sample time (reading A10)
            double v = 0.0;
            if (a < N2) {
                if (b == 0) { if (item < N2) v = beta_entry(item % S, a, item < S ? 0.0 : 1.0); }
                else v = beta_entry(b - 1, a, tau);
            }
            ctab[kk * 32] = v;
        }
        const int item = (grp >> 1) + 4 * (grp & 1);
        const double tau = (double)(item + 1) / (double)(MS + 1);
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) {
            const int ar = 4 * kk + lane;
#pragma unroll
            for (int nt = 0; nt < 4; ++nt) {
                double v = 0.0;
                if (ar < N2) {
                    if (nt == 0) { if (item < N2) v = beta_entry(item % S, ar, item < S ? 0.0 : 1.0); }
                    else v = beta_entry(nt - 1, ar, tau);
                }
                ctab[(8 + kk * 4 + nt) * 32] = v;
            }
        }
        if (WIDE) {
            // second consensus block.  a1 operand of k-step h (h = 0 start, 1 end boundary): row k = lane <-> order S + lane,
            // column n = grp = coefficient row.  a3 operand of k-step kk: row k = coefficient row 4 kk + lane, column n = grp
            // <-> item (grp >> 1, side grp & 1), so that accumulator columns 2t, 2t+1 are the lane's own two rows.
#pragma unroll
            for (int h = 0; h < 2; ++h)
                ctab[(16 + h) * 32] = (a < N2 && lane <= S - 2) ? beta_entry(S + lane, a, h ? 1.0 : 0.0) : 0.0;
            const int t2 = grp >> 1, h2 = grp & 1;
#pragma unroll
            for (int kk = 0; kk < 2; ++kk) {
                const int ar = 4 * kk + lane;
                ctab[(18 + kk) * 32] = (ar < N2 && t2 <= S - 2) ? beta_entry(S + t2, ar, h2 ? 1.0 : 0.0) : 0.0;
            }
        }
    }
}

// ================================================================================================ split tail
// Load balance of the fp64 kernel when a CTA holds 4k+1 octets (config 4: 68 segments = 8 octets + 4 segments): as 4k+1 warps
// one scheduler carries k+1 warps, and all the others wait for it at the pair barriers.  In the SPLIT instantiation the LAST
// octet is run by THREE warps, one flat dimension each (4k+3 warps: the extra work is spread over three schedulers).  Everything
// in the sweep is independent per dimension -- both contractions (one accumulator tile instead of three), the operator apply,
// the box, the consensus, the duals -- except the ball projections, which need ||y||^2 over the three dims: the three warps
// exchange their y_d through shared memory around one named barrier.  The arithmetic of a (row, dim) is the one of the unsplit
// lane, operation for operation: results are bit-identical.  Towards the octet in front the three warps join that warp's pair
// barrier (128 threads); towards the next CTA each publishes and fetches its own dim's mailbox slots.
// (A kernel made of such warps ONLY was tried: 864 threads leave 72 registers and every operator row is read three times --
// shared-memory bound, slower.  Here only one octet pays that.)
// The same split applied to EVERY octet of a small CTA (<= 4 octets, 12 warps) shortens the dependent chain of a sweep and puts
// three light warps on every scheduler instead of one heavy one: the latency-bound short and mid-size chains gain most
// (p.split_octets = how many trailing octets are split; 1 for the tail case above).
constexpr int SPLIT_BALL_BAR = 15;      // named barrier of split octet j: 15 - j (the pair barriers use ids 0..8)
constexpr int SPLIT_MAX_ALL = 3;        // cluster CTAs of at most this many octets are split entirely

// octets [0, W) run on one warp each, octets [W, noct) on three: threads of the pair barrier that joins octets b and b + 1
__device__ __forceinline__ int pair_threads(int b, int W) { return (b >= W ? 96 : 32) + (b + 1 >= W ? 96 : 32); }

// SOLVE (in-kernel stop rule and Eq. 24, as in cadmm_sweeps_mma_kernel): only for CTAs that are split entirely; one CTA barrier
// per sweep instead of the pair barriers.
struct SolveShared { int* abort_sh; double (*wsum)[4]; double (*allp)[4]; double* tot; unsigned char* cres; };

template <int S, int CM, int MAXT, bool SOLVE>
__device__ __forceinline__ void split_tail_sweeps(const KParams& p, unsigned char* smem_raw, volatile int* abort_any, unsigned char* cmbox, const SolveShared sv) {
    constexpr int N2 = 2 * S;
    constexpr int TS = MAXT, SA = MAXT / 4, BPAR = (SA + 2) * 24, MBS = 24;
    const int nsplit = p.split_octets, tmain = (int)blockDim.x - 96 * nsplit;      // threads of the unsplit warps in front
    const int W = tmain >> 5, noct = W + nsplit, rel = (int)threadIdx.x - tmain, jsp = rel / 96;
    const int oct = W + jsp, d = (rel - 96 * jsp) >> 5, lane32 = threadIdx.x & 31;
    const int lane = lane32 & 3, grp = lane32 >> 2, sl = oct * 8 + grp, vt = sl * 4 + lane;      // vt: the thread an unsplit warp would be
    const int SEGS = p.segs_per_cta, cta = blockIdx.x, nctas = gridDim.x;
    const uint32_t flags = p.flags;
    constexpr bool has_box = (CM & (int)KF_BOX) != 0, has_vel = (CM & (int)KF_VEL) != 0, has_acc = (CM & (int)KF_ACC) != 0;
    static_assert(CM != CM_RUNTIME && CM != 0, "split tail: compile-time constraint sets only");
    const bool pin_pos = flags & KF_PIN_POS;

    const SmemLayoutMma L = smem_layout_mma(true, SA);
    double2* Pms = reinterpret_cast<double2*>(smem_raw + L.pm) + vt;                          // [(h*4 + b/2) * TS]  (shared by the three dims)
    double* c0s = reinterpret_cast<double*>(smem_raw + L.c0) + vt + (size_t)d * TS;           // [h*3 * TS]
    double2* zus = reinterpret_cast<double2*>(smem_raw + L.zu) + vt + (size_t)d * TS;         // [h*3 * TS]: (z~, u)
    double2* qs = reinterpret_cast<double2*>(smem_raw + L.qs) + vt + (size_t)d * TS;          // (q+, q-)
    double2* ws = reinterpret_cast<double2*>(smem_raw + L.ws) + vt + (size_t)d * TS;          // (w_v, w_a)
    double* ctab = reinterpret_cast<double*>(smem_raw + L.ctab) + lane32;                     // (filled by warp 0)
    double* lohi = reinterpret_cast<double*>(smem_raw + L.lohi) + sl;                         // [6 * SA]
    double* Xs = reinterpret_cast<double*>(smem_raw + L.xs) + (size_t)sl * XSTRIDE + d * 8;
    double* Bs = reinterpret_cast<double*>(smem_raw + L.bs);                                  // [2 parity][SA+2][8 rows][3]
    double* zoffs = reinterpret_cast<double*>(smem_raw + L.zoff) + sl;                        // [(side*3 + dim) * SA]
    // ball exchange buffer of this octet, [parity][item h][dim][lane of warp] (y_v, y_a): in the slot of the (phi_v, phi_a)
    // pairs, which the SPLIT instantiation does not keep in shared memory
    double2* nbuf = reinterpret_cast<double2*>(smem_raw + L.ph) + (size_t)jsp * (2 * 2 * 3 * 32) + lane32;
    const int ball_bar = SPLIT_BALL_BAR - jsp;

    const long long cta_first = p.seg_begin + (long long)cta * SEGS;
    const long long remaining = p.seg_end - cta_first;
    const int nact = remaining < SEGS ? (int)remaining : SEGS;
    const bool active = sl < nact;
    const long long gseg = active ? cta_first + sl : cta_first;
    const bool owned = active && gseg >= p.own_begin && gseg < p.own_end;
    const long long stride = p.stride;

    int jj[2]; long long gt[2]; bool isrow[2], right[2]; int korder[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        jj[h] = lane + 4 * h;
        gt[h] = gseg * LANES + jj[h];
        isrow[h] = S == 4 ? true : jj[h] < N2;
        right[h] = S == 4 ? h == 1 : jj[h] >= S;
        korder[h] = right[h] ? jj[h] - S : jj[h];
    }
    double invTk[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        if (d == 0) {
#pragma unroll
            for (int b = 0; b < 8; b += 2)
                Pms[(h * 4 + (b >> 1)) * TS] = make_double2(b < N2 ? p.Pm[(long long)b * stride + gt[h]] : 0.0,
                                                            b + 1 < N2 ? p.Pm[(long long)(b + 1) * stride + gt[h]] : 0.0);
        }
        c0s[h * 3 * TS] = p.c0[d * stride + gt[h]];
        invTk[h] = static_cast<const double*>(p.invTk)[gt[h]];
    }
    const double invT = static_cast<const double*>(p.invT)[gseg], invT2 = static_cast<const double*>(p.invT)[p.nseg_pad + gseg];
    if (d == 0) {
        lohi[lane * SA] = static_cast<const double*>(p.lohi)[lane * p.nseg_pad + gseg];
        if (lane < 2) lohi[(lane + 4) * SA] = static_cast<const double*>(p.lohi)[(lane + 4) * p.nseg_pad + gseg];
    }
    if (lane == 0) {      // frame shifts of the neighbours' position rows of this dim: left junction (row 0), right junction (row S)
        zoffs[d * SA] = static_cast<const double*>(p.zoff)[d * stride + gseg * LANES + 0];
        zoffs[(3 + d) * SA] = static_cast<const double*>(p.zoff)[d * stride + gseg * LANES + S];
    }
    const uint8_t sf = p.segflags[gseg];
    const bool open_l = (flags & KF_OPEN_LEFT) && gseg == p.seg_begin, open_r = (flags & KF_OPEN_RIGHT) && gseg == p.seg_end - 1;

    // ---- per-lane facts of the exchange (one dim per lane: one value per row)
    int own_off[2], nb_off[2], pub_off[2];
    bool fixed[2], zshift[2], gaprow[2], pub[2];
    bool need = false;
    int need_h = 0, need_off = 0;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        own_off[h] = (sl + 1) * 24 + jj[h] * 3 + d;
        nb_off[h] = (right[h] ? (sl + 2) * 24 + korder[h] * 3 : sl * 24 + (korder[h] + S) * 3) + d;
        fixed[h] = (right[h] ? (sf & SEG_LAST) : (sf & SEG_FIRST)) || (pin_pos && korder[h] == 0) || (right[h] ? open_r : open_l);
        zshift[h] = isrow[h] && korder[h] == 0;
        gaprow[h] = isrow[h] && right[h] && !(sf & SEG_LAST);
        const bool edge_l = active && isrow[h] && sl == 0 && !right[h] && cta > 0;
        const bool edge_r = active && isrow[h] && sl == nact - 1 && right[h] && cta + 1 < nctas;
        pub[h] = nctas > 1 && (edge_l || edge_r);
        pub_off[h] = (cta * 24 + (edge_r ? 12 : 0) + korder[h] * 3 + d) * 16;
        if (edge_l || edge_r) {
            need = true; need_h = h;
            need_off = (edge_l ? ((cta - 1) * 24 + 12 + korder[h] * 3) : ((cta + 1) * 24 + korder[h] * 3)) * 16 + d * 16;
        }
    }

    // ---- state of iterate k: the a1 operands in registers, the variables behind them in shared memory
    double gM[2], A0[2], gv[2], ga[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        const long long i = d * stride + gt[h];
        const double z0 = static_cast<const double*>(p.zt)[i], u0 = static_cast<const double*>(p.u)[i];
        zus[h * 3 * TS] = make_double2(z0, u0);
        gM[h] = (z0 - u0) * invTk[h];
        A0[h] = gv[h] = ga[h] = 0.0;
        double w_v = 0, w_a = 0;
        if (has_box) {
            const double lo = static_cast<const double*>(p.lohi)[d * p.nseg_pad + gseg], hi = static_cast<const double*>(p.lohi)[(3 + d) * p.nseg_pad + gseg];
            const double a = static_cast<const double*>(p.qp)[i], b = static_cast<const double*>(p.qn)[i];
            qs[h * 3 * TS] = make_double2(a, b);
            A0[h] = (hi - fabs(a)) + (lo + fabs(b));
        }
        if (has_vel) { w_v = static_cast<const double*>(p.wv)[i]; gv[h] = (static_cast<const double*>(p.phv)[i] - w_v) * invT; }
        if (has_acc) { w_a = static_cast<const double*>(p.wa)[i]; ga[h] = (static_cast<const double*>(p.pha)[i] - w_a) * invT2; }
        ws[h * 3 * TS] = make_double2(w_v, w_a);
    }
    // (phi of iterate k is not kept: it only enters through gv, ga; phi of the final iterate is written on the last sweep -- a
    // launch of zero sweeps writes nothing back at all)
    const double vmax = p.vmax, amax = p.amax;
    unsigned char* const mbox = static_cast<unsigned char*>(p.Bedge);
    // cluster exchange (KF_CLUSTER; see cadmm_sweeps_mma_kernel): the mailbox is the CTA's own shared memory
    const bool clus = (flags & KF_CLUSTER) != 0;
    const unsigned cm_local = smem_u32(cmbox);
    unsigned cm_remote[2] = {0, 0};
    if (clus) {
        cm_remote[0] = cta > 0 ? cluster_map(cm_local, (unsigned)(cta - 1)) : 0u;
        cm_remote[1] = cta + 1 < nctas ? cluster_map(cm_local, (unsigned)(cta + 1)) : 0u;
        cluster_barrier();
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const bool er = right[h];
            pub_off[h] = ((er ? 0 : 1) * (MBS / 2) + korder[h] * 3 + d) * 16;
            if (need && need_h == h) need_off = ((er ? 1 : 0) * (MBS / 2) + korder[h] * 3 + d) * 16;
        }
    }
    const size_t par_stride = clus ? (size_t)MBS * 16 : (size_t)p.max_ctas * MBS * 16;
    const int bfirst = (oct & 1) ? oct - 1 : oct, bsecond = (oct & 1) ? oct : oct - 1;      // pair barriers: the even id first, as every octet does
    const bool use_first = bfirst >= 0 && bfirst + 1 < noct, use_second = bsecond >= 0 && bsecond + 1 < noct;
    const int n_first = use_first ? pair_threads(bfirst, W) : 0, n_second = use_second ? pair_threads(bsecond, W) : 0;
    const int ce = SOLVE ? p.check_every : 0;
    double rho_cur = p.rho;
    int ncheck = 0, sweeps_done = p.k_sweeps, stopped = 0, since_test = 0;
    double phv_[2] = {0, 0}, pha_[2] = {0, 0};      // SOLVE: phi of the newest iterate (Eq. 24 rebuilds the operands gv, ga from it)
    __syncthreads();      // (the one CTA barrier of the launch: the unsplit warps arrive from cadmm_sweeps_mma_kernel)

    for (int it = 0; it < p.k_sweeps; ++it) {
        const unsigned seq = p.seq_base + (unsigned)it + 1u;
        const int par = (int)(seq & 1u);
        // sweeps on which residuals (and the coefficients) are materialised: the last one, and every test sweep
        bool test_sweep = false;      // (a counter, not (it + 1) % ce: the integer division showed up in the profile of short chains)
        if (SOLVE && ce > 0 && ++since_test == ce) { since_test = 0; test_sweep = true; }
        const bool last_sweep = (it == p.k_sweeps - 1) || test_sweep;
        double* const Bcur = Bs + par * BPAR;
        unsigned char* const mpar = mbox + par * par_stride;      // (cluster exchange: only the offset part is used)
        const unsigned cpar = (unsigned)(par * MBS * 16);
        double2* const nb = nbuf + par * (2 * 3 * 32);

        // ================= phase A: segment local, this dim =================
        double2 pm[2][4];
        double cacc[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
#pragma unroll
            for (int b = 0; b < 4; ++b) pm[h][b] = Pms[(h * 4 + b) * TS];
            cacc[h] = c0s[h * 3 * TS];
        }
        // a1 (Eq. 20a second bracket): one accumulator tile; lane t ends with rows 2t, 2t+1 of R^ of its segment and dim
        {
            double a0 = 0.0, a1 = 0.0;
            dmma884(a0, a1, gM[0], ctab[0 * 32]); dmma884(a0, a1, gM[1], ctab[1 * 32]);
            if (has_box) { dmma884(a0, a1, A0[0], ctab[2 * 32]); dmma884(a0, a1, A0[1], ctab[3 * 32]); }
            if (has_vel) { dmma884(a0, a1, gv[0], ctab[4 * 32]); dmma884(a0, a1, gv[1], ctab[5 * 32]); }
            if (has_acc) { dmma884(a0, a1, ga[0], ctab[6 * 32]); dmma884(a0, a1, ga[1], ctab[7 * 32]); }
            *reinterpret_cast<double2*>(Xs + 2 * lane) = make_double2(a0, a1);
        }
        __syncwarp();
        // a2 (Eq. 20a first bracket): c^ = (rho Pm^) R^ + c0^, rows lane, lane+4
#pragma unroll
        for (int b = 0; b < N2 / 2; ++b) {
            const double2 x2 = *reinterpret_cast<const double2*>(Xs + 2 * b);
#pragma unroll
            for (int h = 0; h < 2; ++h) { cacc[h] += pm[h][b].x * x2.x; cacc[h] += pm[h][b].y * x2.y; }
        }
        if (last_sweep && owned) {
#pragma unroll
            for (int h = 0; h < 2; ++h) static_cast<double*>(p.chat)[d * stride + gt[h]] = cacc[h];
        }
        __syncwarp();       // (Xs is read by every lane of the segment before the next sweep overwrites it)
        // a3: the lane's consensus rows of B = M c and its two samples of E0 c, E1 c, E2 c, this dim
        double Bnd[2];
        {
            double e0 = 0.0, e1 = 0.0;
            dmma884(e0, e1, cacc[0], ctab[8 * 32]); dmma884(e0, e1, cacc[1], ctab[12 * 32]);
            Bnd[0] = e0 * invTk[0]; Bnd[1] = e1 * invTk[1];
        }
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (isrow[h]) Bcur[own_off[h]] = Bnd[h];
            if (pub[h]) { if (clus) ll_store_cluster(cm_remote[right[h] ? 1 : 0] + cpar + pub_off[h], Bnd[h], seq); else ll_store(mpar + pub_off[h], Bnd[h], seq); }
        }
        LLRaw rr;
        if (need) { if (clus) ll_issue_smem(cm_local + cpar + need_off, rr); else ll_issue(mpar + need_off, rr); }
        {
            double Pv[2] = {0, 0}, Vv[2] = {0, 0}, Av[2] = {0, 0};
            if (has_vel) { double e0 = 0, e1 = 0; dmma884(e0, e1, cacc[0], ctab[10 * 32]); dmma884(e0, e1, cacc[1], ctab[14 * 32]); Vv[0] = e0; Vv[1] = e1; }
            if (has_acc) { double e0 = 0, e1 = 0; dmma884(e0, e1, cacc[0], ctab[11 * 32]); dmma884(e0, e1, cacc[1], ctab[15 * 32]); Av[0] = e0; Av[1] = e1; }
            if (has_box) { double e0 = 0, e1 = 0; dmma884(e0, e1, cacc[0], ctab[9 * 32]); dmma884(e0, e1, cacc[1], ctab[13 * 32]); Pv[0] = e0; Pv[1] = e1; }
            double2 w2[2], q2[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (has_vel || has_acc) w2[h] = ws[h * 3 * TS];
                if (has_box) q2[h] = qs[h * 3 * TS];
            }
            // a4 (Eq. 20f, 20g): y = A c + w; ||y|| runs over the three dims: the three warps exchange y_d (buffer of this
            // sweep's parity: the next sweep writes the other one, and nobody passes that sweep's barrier before everybody has
            // read this one)
            if (has_vel || has_acc) {
                double yv[2] = {0, 0}, ya[2] = {0, 0};
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    if (has_vel) yv[h] = Vv[h] * invT + w2[h].x;
                    if (has_acc) ya[h] = Av[h] * invT2 + w2[h].y;
                    nb[(h * 3 + d) * 32] = make_double2(yv[h], ya[h]);
                }
                asm volatile("bar.sync %0, 96;" ::"r"(ball_bar) : "memory");
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const double2 s0 = nb[(h * 3 + 0) * 32], s1 = nb[(h * 3 + 1) * 32], s2 = nb[(h * 3 + 2) * 32];
                    if (has_vel) {
                        const double y[3] = {s0.x, s1.x, s2.x};
                        const double scale = ball_scale(y, vmax);
                        const double ph = scale * yv[h];
                        w2[h].x = yv[h] - ph; gv[h] = (ph - w2[h].x) * invT;
                        if (SOLVE) phv_[h] = ph;
                        if (last_sweep && owned) static_cast<double*>(p.phv_out)[d * stride + gt[h]] = ph;
                    }
                    if (has_acc) {
                        const double y[3] = {s0.y, s1.y, s2.y};
                        const double scale = ball_scale(y, amax);
                        const double ph = scale * ya[h];
                        w2[h].y = ya[h] - ph; ga[h] = (ph - w2[h].y) * invT2;
                        if (SOLVE) pha_[h] = ph;
                        if (last_sweep && owned) static_cast<double*>(p.pha_out)[d * stride + gt[h]] = ph;
                    }
                    ws[h * 3 * TS] = w2[h];
                }
            }
            if (has_box) {      // a7 + a8 (Eq. 20d, 20e) as a Moreau pair
                const double lo = lohi[d * SA], hi = lohi[(3 + d) * SA];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const double qpn = (hi - Pv[h]) - neg_part(q2[h].x), qnn = (Pv[h] - lo) - neg_part(q2[h].y);
                    qs[h * 3 * TS] = make_double2(qpn, qnn);
                    A0[h] = (hi - fabs(qpn)) + (lo + fabs(qnn));
                }
            }
        }

        // ================= exchange: the next CTA's rows (mailbox), then the pair barrier with the octet in front
        {
            bool okk = !need || ll_ok(rr, seq);
            if (*abort_any) okk = true;
            if (!__all_sync(0xffffffffu, okk)) {
                const long long t0 = global_ns();
                unsigned spins = 0;
                bool failed = false;
                do {
                    if (!okk) { if (clus) ll_issue_smem(cm_local + cpar + need_off, rr); else ll_issue(mpar + need_off, rr); okk = ll_ok(rr, seq); }
                    bool bail = false;
                    if ((++spins & 255u) == 0) bail = *(volatile int*)p.abort_flag || global_ns() - t0 > WAIT_TIMEOUT_NS;
                    if (__any_sync(0xffffffffu, bail)) { if (!okk) { atomicExch(p.abort_flag, 1); failed = true; } break; }
                } while (!__all_sync(0xffffffffu, okk));
                if (failed) { *abort_any = 1; if (SOLVE) sv.abort_sh[it & 1] = 1; }
            }
        }
        if (SOLVE) {
            __syncthreads();
            if (sv.abort_sh[it & 1]) break;
        } else {
            if (use_first) asm volatile("bar.sync %0, %1;" ::"r"(bfirst), "r"(n_first) : "memory");
            if (use_second) asm volatile("bar.sync %0, %1;" ::"r"(bsecond), "r"(n_second) : "memory");
        }

        // ================= phase B: consensus, dual, residuals (this dim)
        double res_[2], own_[2], nb_[2], dz[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double own = Bnd[h];
            double nb = Bcur[nb_off[h]];
            if (need && need_h == h) nb = ll_value(rr);
            if (zshift[h]) nb += zoffs[((right[h] ? 3 : 0) + d) * SA];
            const double2 zu = zus[h * 3 * TS];
            const double avg = 0.5 * (own + nb);
            const double znew = (fixed[h] || !isrow[h]) ? zu.x : avg;            // a5: Eq. 6b / 20b
            dz[h] = znew - zu.x;
            const double res = isrow[h] ? own - znew : 0.0;
            const double unew = zu.y + res;                                        // a8: Eq. 6c / 20c
            zus[h * 3 * TS] = make_double2(znew, unew);
            gM[h] = (znew - unew) * invTk[h];
            res_[h] = res; own_[h] = own; nb_[h] = nb;
        }
        if (last_sweep) {
            // a6 (Eq. 21, 22; A7, A8): the three warps hand their terms to the dim-0 warp, which adds them in the order of the
            // unsplit lane (rows, then dims; then the 4 lanes)
            double x0 = 0, x1 = 0;
            dmma884(x0, x1, dz[0] * invTk[0], ctab[0 * 32]);
            dmma884(x0, x1, dz[1] * invTk[1], ctab[1 * 32]);
            double2* const rb = nbuf + (par ^ 1) * (2 * 3 * 32);      // (free: everybody is past this sweep's ball barrier, and the launch ends here)
            rb[(0 * 3 + d) * 32] = make_double2(res_[0], res_[1]);
            rb[(1 * 3 + d) * 32] = make_double2(rho_cur * x0, rho_cur * x1);
            asm volatile("bar.sync %0, 96;" ::"r"(ball_bar) : "memory");
            double2* const gb = nb;                     // own - nb of the gap rows (the ball exchange of this sweep is over)
            gb[d * 32] = make_double2(own_[0] - nb_[0], own_[1] - nb_[1]);
            asm volatile("bar.sync %0, 96;" ::"r"(ball_bar) : "memory");
            double rp2 = 0, rd2 = 0, rdn2 = 0, gap2 = 0;
            if (d == 0) {
                const double Tp0 = static_cast<const double*>(p.Tpow)[gseg * LANES + 2 * lane], Tp1 = static_cast<const double*>(p.Tpow)[gseg * LANES + 2 * lane + 1];
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int dd = 0; dd < 3; ++dd) {
                        const double2 r2 = rb[dd * 32], g2 = gb[dd * 32];
                        const double r = h ? r2.y : r2.x, g = h ? g2.y : g2.x;
                        rp2 = fma(r, r, rp2);
                        if (gaprow[h]) gap2 = fma(g, g, gap2);
                    }
#pragma unroll
                for (int dd = 0; dd < 3; ++dd) { const double2 x2 = rb[(3 + dd) * 32]; rd_accum(rd2, rdn2, x2.x, x2.y, Tp0, Tp1); }
#pragma unroll
                for (int m = 1; m < 4; m <<= 1) { rp2 += shfl_xor(rp2, m); rd2 += shfl_xor(rd2, m); rdn2 += shfl_xor(rdn2, m); gap2 += shfl_xor(gap2, m); }
                if (owned && lane == 0) { double* o = p.part + gseg * 4; o[0] = rp2; o[1] = rd2; o[2] = rdn2; o[3] = gap2; }
            }
            if (SOLVE && ce > 0) {
                // ---- octet partial (the dim-0 warp holds the per-segment sums), then the CTA-wide decision
                if (d == 0) {
                    double q4[4] = {rp2, rd2, rdn2, gap2};
                    if (!(owned && lane == 0)) { q4[0] = q4[1] = q4[2] = q4[3] = 0.0; }
#pragma unroll
                    for (int k = 0; k < 4; ++k) { q4[k] += shfl_xor(q4[k], 4); q4[k] += shfl_xor(q4[k], 8); q4[k] += shfl_xor(q4[k], 16); }
                    if (lane32 == 0) { for (int k = 0; k < 4; ++k) sv.wsum[oct][k] = q4[k]; }
                }
                double rho_new = rho_cur;
                if (solve_decide(p, seq, noct, sv.wsum, sv.allp, sv.tot, sv.cres, ncheck, rho_cur, rho_new, stopped)) { sweeps_done = it + 1; break; }
                if (rho_new != rho_cur) {      // Eq. 24 moved rho: scaled duals times rho_old / rho_new (A16), operands, operator rows
                    const double ratio = rho_cur / rho_new;
                    const double lo = has_box ? lohi[d * SA] : 0.0, hi = has_box ? lohi[(3 + d) * SA] : 0.0;
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        double2 zz = zus[h * 3 * TS];
                        zz.y *= ratio;
                        zus[h * 3 * TS] = zz;
                        gM[h] = (zz.x - zz.y) * invTk[h];
                        if (has_box) {
                            double2 q = qs[h * 3 * TS];
                            if (q.x < 0) q.x *= ratio;
                            if (q.y < 0) q.y *= ratio;
                            qs[h * 3 * TS] = q;
                            A0[h] = (hi - fabs(q.x)) + (lo + fabs(q.y));
                        }
                        if (has_vel || has_acc) {
                            double2 w2 = ws[h * 3 * TS];
                            w2.x *= ratio; w2.y *= ratio;
                            ws[h * 3 * TS] = w2;
                            if (has_vel) gv[h] = (phv_[h] - w2.x) * invT;
                            if (has_acc) ga[h] = (pha_[h] - w2.y) * invT2;
                        }
                        if (d == 0) refresh_operator_rows<N2, TS>(p, gseg, gt[h], jj[h], rho_new, Pms + h * 4 * TS, c0s + h * 3 * TS);
                    }
                    asm volatile("bar.sync %0, 96;" ::"r"(ball_bar) : "memory");      // the other two dims read the new operator rows
                    rho_cur = rho_new;
                }
            }
        }
    }
    if (SOLVE && ce > 0 && cta == 0 && threadIdx.x == 0) {
        double* o = p.solve_out;
        o[0] = (double)sweeps_done; o[1] = (double)stopped; o[2] = rho_cur;
        o[3] = sqrt(sv.tot[0]); o[4] = sqrt(sv.tot[1]); o[5] = sqrt(sv.tot[2]); o[6] = sqrt(sv.tot[3]);
    }

    if (clus) cluster_barrier();      // nobody leaves while a neighbour may still store into its mailbox
    // ---- write iterate k + k_sweeps back (phi went out on the last sweep)
    if (owned) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long i = d * stride + gt[h];
            const double2 zz = zus[h * 3 * TS];
            static_cast<double*>(p.zt_out)[i] = zz.x;
            static_cast<double*>(p.u_out)[i] = zz.y;
            if (has_box) { const double2 q = qs[h * 3 * TS]; static_cast<double*>(p.qp_out)[i] = q.x; static_cast<double*>(p.qn_out)[i] = q.y; }
            if (has_vel || has_acc) {
                const double2 w2 = ws[h * 3 * TS];
                if (has_vel) static_cast<double*>(p.wv_out)[i] = w2.x;
                if (has_acc) static_cast<double*>(p.wa_out)[i] = w2.y;
            }
            if (p.k_sweeps == 0) {
                if (has_vel) static_cast<double*>(p.phv_out)[i] = static_cast<const double*>(p.phv)[i];
                if (has_acc) static_cast<double*>(p.pha_out)[i] = static_cast<const double*>(p.pha)[i];
            }
        }
    }
}

template <typename Real, int S, int CM, int MAXT, bool SOLVE, bool POLY = false, bool WIDE = false, bool SPLIT = false>
// (SPLIT: MAXT + 64 threads are launched; the bound is rounded up to 12 warps so that ptxas sees what the hardware enforces -- three
// warps on a scheduler share its 16 K registers)
__global__ void __launch_bounds__(SPLIT ? (MAXT + 64 + 127) / 128 * 128 : MAXT, 1) cadmm_sweeps_mma_kernel(const KParams p) {
    constexpr int N2 = 2 * S;
    static_assert(!SPLIT || (sizeof(Real) == 8 && !POLY && !WIDE), "split octets: fp64, box / ball sets only");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    constexpr int MBS = WIDE ? 48 : 24;              // mailbox slots per CTA and parity: [2 sides][4 or 8 orders][3 dims]
    __shared__ int abort_any;
    __shared__ int abort_sh[2];
    __shared__ __align__(16) unsigned char cmbox[2 * MBS * 16];      // cluster exchange: this CTA's mailbox (see below)
    __shared__ double wsum_sh[SOLVE ? 32 : 1][4];      // in-kernel stop rule: per-octet partial sums, per-CTA partial sums, totals
    __shared__ double allp_sh[SOLVE ? 160 : 1][4];
    __shared__ double tot_sh[4];
    __shared__ __align__(16) unsigned char cresbox[SOLVE ? CRES_BYTES : 16];      // cluster exchange: this CTA's copy of the per-CTA residual sums
    // ---- CTA-wide prologue (before the split octets branch off): constant MMA operands, flags, cluster mailbox cleared
    {
        const SmemLayoutMma L0 = smem_layout_mma(CM != 0 || POLY, MAXT / 4, POLY, (int)sizeof(Real), WIDE);
        if (threadIdx.x < 32) fill_ctab<S, WIDE>(reinterpret_cast<double*>(smem_raw + L0.ctab) + threadIdx.x, (int)threadIdx.x);
        if (threadIdx.x < 2) abort_sh[threadIdx.x] = 0;
        if (threadIdx.x == 0) abort_any = 0;
        if (p.flags & KF_CLUSTER) {
            for (int i = threadIdx.x; i < 2 * MBS * 4; i += blockDim.x) reinterpret_cast<unsigned*>(cmbox)[i] = 0u;
            if (SOLVE) for (int i = threadIdx.x; i < CRES_BYTES / 4; i += blockDim.x) reinterpret_cast<unsigned*>(cresbox)[i] = 0u;
        }
    }
    if constexpr (SPLIT) {      // the last p.split_octets octets run on three warps each, one dim per warp
        // (SPLIT with the in-kernel stop rule: every octet is split, this is the whole kernel)
        if (SOLVE || (int)threadIdx.x >= (int)blockDim.x - 96 * p.split_octets) {
            const SolveShared sv = {abort_sh, wsum_sh, allp_sh, tot_sh, cresbox};
            split_tail_sweeps<S, (CM == 0 || CM == CM_RUNTIME) ? 7 : CM, MAXT, SOLVE>(p, smem_raw, &abort_any, cmbox, sv);
            return;
        }
    }
    if constexpr (!(SPLIT && SOLVE)) {
    // WIDE: the paper-literal consensus (reading A1): derivative orders 0..2s-2 at both boundaries.
    // Orders 0..s-1 are the first block (as always); orders s..2s-2 form a SECOND block of consensus rows with the same
    // lane <-> row map: lane t owns order s+t at the start boundary (item h = 0) and at the end boundary (h = 1), t <= s-2.
    // Rows that do not exist (t = s-1; the trajectory ends, where z_0 / z_N carry orders < s only) have 1/T^k = 0 in
    // invTk2: their operand, boundary value, residual and dual are identically 0.
    constexpr int LPS = 4;                         // lanes per segment
    constexpr bool CONS = CM != 0 || POLY;
    static_assert(!(SOLVE && POLY), "the in-kernel stop rule is not instantiated for polytope corridors (host loop)");
    static_assert(!POLY || sizeof(Real) == 8, "polytope corridors are fp64 only");
    // Real = double: everything in fp64.  Real = float (TOP_F32, mixed): state, projections, consensus and duals in fp32; the
    // two contractions stay on the fp64 tensor pipe (products of fp32-rounded operands, fp64 accumulation) and the operator
    // apply a2 stays fp64 (an fp32 operator loses Q against rho G): the fp64 pipe then carries the MMAs only.
    using R2 = typename Pair<Real>::type;

    const int T = SPLIT ? blockDim.x - 96 * p.split_octets : blockDim.x, tid = threadIdx.x, lane = tid & (LPS - 1), sl = tid >> 2;
    // Shared-memory arrays are laid out for the LARGEST CTA of this instantiation whatever the launched size (one CTA
    // per SM: the space is there), so every stride is a compile-time constant and every shared-memory address is one
    // per-thread base register plus an immediate (with run-time strides ptxas re-derived the offsets inside the loop).
    constexpr int TS = MAXT;                       // thread stride of the per-thread arrays
    constexpr int SA = MAXT / 4;                   // segment slots
    constexpr int BPAR = (SA + 2) * 24;            // doubles per parity of the boundary-row buffer
    const int SEGS = p.segs_per_cta;
    const int cta = blockIdx.x, nctas = gridDim.x;
    const uint32_t flags = p.flags;
    const bool has_box = POLY ? false : (CM == CM_RUNTIME ? (flags & KF_BOX) != 0 : (CM & (int)KF_BOX) != 0);
    const bool has_vel = CM == CM_RUNTIME ? (flags & KF_VEL) != 0 : (CM & (int)KF_VEL) != 0;
    const bool has_acc = CM == CM_RUNTIME ? (flags & KF_ACC) != 0 : (CM & (int)KF_ACC) != 0;
    const bool pin_pos = flags & KF_PIN_POS;
    const bool nb_sync = flags & KF_NEIGHBOUR_SYNC;

    const SmemLayoutMma L = smem_layout_mma(CONS, SA, POLY, (int)sizeof(Real), WIDE);
    R2* zus2 = reinterpret_cast<R2*>(smem_raw + L.zu2) + tid;        // [(h*3 + d) * TS]: (z~, u) of the second block
    Real* Bs2 = reinterpret_cast<Real*>(smem_raw + L.bs2);           // [2 parity][SA+2][2 sides][4][3]
    double2* Pms = reinterpret_cast<double2*>(smem_raw + L.pm) + tid;          // [((d*2 +) h*4 + b/2) * TS]   (d only with POLY)
    double* c0s = reinterpret_cast<double*>(smem_raw + L.c0) + tid;            // [(h*3 + d) * TS]
    R2* zus = reinterpret_cast<R2*>(smem_raw + L.zu) + tid;          // [(h*3 + d) * TS]: (z~, u)
    R2* qs = reinterpret_cast<R2*>(smem_raw + L.qs) + tid;           // [(h*3 + d) * TS]: (q+, q-)
    R2* ws = reinterpret_cast<R2*>(smem_raw + L.ws) + tid;           // [(h*3 + d) * TS]: (w_v, w_a)
    R2* phs = reinterpret_cast<R2*>(smem_raw + L.ph) + tid;          // [(h*3 + d) * TS]: (phi_v, phi_a)
    double* ctab = reinterpret_cast<double*>(smem_raw + L.ctab) + (tid & 31);  // [k * 32]: a1 k-step operands at k = 0..7, a3 operands at k = 8 + kstep*4 + block
    Real* lohi = reinterpret_cast<Real*>(smem_raw + L.lohi) + sl;          // [6 * SA]
    double* Xs = reinterpret_cast<double*>(smem_raw + L.xs) + (size_t)sl * XSTRIDE;
    Real* Bs = reinterpret_cast<Real*>(smem_raw + L.bs);                   // [2 parity][SA+2][8 rows][3]
    Real* zoffs = reinterpret_cast<Real*>(smem_raw + L.zoff) + sl;         // [(side*3 + d) * SA]
    double* qpls = reinterpret_cast<double*>(smem_raw + L.qpl) + tid;          // [(k*2 + h) * TS]
    double* pls = reinterpret_cast<double*>(smem_raw + L.pls) + (size_t)sl * PSTR;   // [k*4 + c]
    double* vs = reinterpret_cast<double*>(smem_raw + L.vs) + (size_t)sl * VSTR;     // V[d][e] at d*3 + e
    const int KP = POLY ? p.K : 0;

    const long long cta_first = p.seg_begin + (long long)cta * SEGS;
    const long long remaining = p.seg_end - cta_first;
    const int nact = remaining < SEGS ? (int)remaining : SEGS;
    const bool active = sl < nact;
    // inactive slots of a ragged CTA compute on a copy of the CTA's first segment (the MMAs need full warps) and never
    // write to global memory
    const long long gseg = active ? cta_first + sl : cta_first;
    const bool owned = active && gseg >= p.own_begin && gseg < p.own_end;
    const long long stride = p.stride;

    // the two items of this lane: sample / row index jj[h], global lane slot gt[h]
    // (s = 4: item 0 is always a left consensus row, item 1 a right one; s = 3: decided per lane)
    int jj[2]; long long gt[2]; bool isrow[2], right[2]; int korder[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        jj[h] = lane + 4 * h;
        gt[h] = gseg * LANES + jj[h];
        isrow[h] = S == 4 ? true : jj[h] < N2;
        right[h] = S == 4 ? h == 1 : jj[h] >= S;
        korder[h] = right[h] ? jj[h] - S : jj[h];
    }

    // B operand of a k-block: entries i0 (k-step of the lane's first item) and i1 (second item) of the constant table
    auto ldb = [&](int i0, int i1) {
        BOp b;
        b.b0 = ctab[i0 * 32]; b.b1 = ctab[i1 * 32];
        return b;
    };
    Real invTk[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
#pragma unroll
        for (int dd = 0; dd < (POLY ? 3 : 1); ++dd)
#pragma unroll
            for (int b = 0; b < 8; b += 2)
                Pms[((dd * 2 + h) * 4 + (b >> 1)) * TS] = make_double2(b < N2 ? p.Pm[((long long)dd * MAXN + b) * stride + gt[h]] : 0.0,
                                                                   b + 1 < N2 ? p.Pm[((long long)dd * MAXN + b + 1) * stride + gt[h]] : 0.0);
#pragma unroll
        for (int d = 0; d < 3; ++d) c0s[(h * 3 + d) * TS] = p.c0[d * stride + gt[h]];
        invTk[h] = static_cast<const Real*>(p.invTk)[gt[h]];
    }
    Real invTk2[2] = {0, 0};
    if (WIDE) { invTk2[0] = static_cast<const Real*>(p.invTk2)[gt[0]]; invTk2[1] = static_cast<const Real*>(p.invTk2)[gt[1]]; }
    const Real invT = static_cast<const Real*>(p.invT)[gseg], invT2 = static_cast<const Real*>(p.invT)[p.nseg_pad + gseg];
    if (CONS && !POLY) {
        lohi[lane * SA] = static_cast<const Real*>(p.lohi)[lane * p.nseg_pad + gseg];
        if (lane < 2) lohi[(lane + 4) * SA] = static_cast<const Real*>(p.lohi)[(lane + 4) * p.nseg_pad + gseg];
    }
    if (lane < 3) {        // frame shifts of the neighbours' position rows: left junction (row 0), right junction (row S)
        zoffs[lane * SA] = static_cast<const Real*>(p.zoff)[lane * stride + gseg * LANES + 0];
        zoffs[(3 + lane) * SA] = static_cast<const Real*>(p.zoff)[lane * stride + gseg * LANES + S];
    }
    if (POLY) {
        for (int i = lane; i < 9; i += LPS) vs[i] = p.rot[i * p.nseg_pad + gseg];
        for (int i = lane; i < KP * 4; i += LPS) pls[i] = p.planes[i * p.nseg_pad + gseg];
#pragma unroll
        for (int h = 0; h < 2; ++h)
            for (int k = 0; k < KP; ++k) qpls[(k * 2 + h) * TS] = static_cast<const double*>(p.qpl)[k * stride + gt[h]];
    }
    __syncwarp();
    const uint8_t sf = p.segflags[gseg];
    const bool open_l = (flags & KF_OPEN_LEFT) && gseg == p.seg_begin, open_r = (flags & KF_OPEN_RIGHT) && gseg == p.seg_end - 1;

    // ---- per-lane facts of the exchange, fixed for the launch
    // boundary-row buffer (doubles, relative to the parity base): my rows, and where the neighbour segment's matching rows are
    int own_off[2], nb_off[2];
    bool fixed[2], zshift[2], gaprow[2];
    // mailbox (bytes, relative to the parity base): where I publish, what I fetch.  A lane needs at most ONE of its two
    // rows from another CTA (a CTA with a neighbour on both sides owns >= 4 segments, so its left-edge and right-edge
    // segments differ): one prefetch buffer.
    int pub_off[2];
    bool pub[2];
    bool need = false;
    int need_h = 0, need_off = 0;
#pragma unroll
    for (int h = 0; h < 2; ++h) {
        own_off[h] = (sl + 1) * 24 + jj[h] * 3;
        nb_off[h] = right[h] ? (sl + 2) * 24 + korder[h] * 3 : sl * 24 + (korder[h] + S) * 3;
        fixed[h] = (right[h] ? (sf & SEG_LAST) : (sf & SEG_FIRST)) || (pin_pos && korder[h] == 0) ||
                   (right[h] ? open_r : open_l);      // outer end of a halo: no neighbour in this launch
        zshift[h] = isrow[h] && korder[h] == 0;       // position rows live in segment-local frames
        gaprow[h] = isrow[h] && right[h] && !(sf & SEG_LAST);
        const bool edge_l = active && isrow[h] && sl == 0 && !right[h] && cta > 0;
        const bool edge_r = active && isrow[h] && sl == nact - 1 && right[h] && cta + 1 < nctas;
        pub[h] = nctas > 1 && (edge_l || edge_r);
        pub_off[h] = (cta * MBS + (edge_r ? MBS / 2 : 0) + korder[h] * 3) * 16;
        if (edge_l || edge_r) {
            need = true; need_h = h;
            need_off = edge_l ? ((cta - 1) * MBS + MBS / 2 + korder[h] * 3) * 16 : ((cta + 1) * MBS + korder[h] * 3) * 16;
        }
    }
    // second consensus block (WIDE): item h = 0 is the start-boundary row of order S + lane, h = 1 the end-boundary row
    const bool isrow2 = WIDE && lane <= S - 2;
    int own2_off[2] = {0, 0}, nb2_off[2] = {0, 0}, pub2_off[2] = {0, 0};
    bool fixed2[2] = {true, true}, gaprow2[2] = {false, false}, pub2[2] = {false, false};
    bool need2 = false;
    int need2_h = 0, need2_off = 0;
    if (WIDE) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            own2_off[h] = (sl + 1) * 24 + (h * 4 + lane) * 3;
            nb2_off[h] = h ? (sl + 2) * 24 + lane * 3 : sl * 24 + (4 + lane) * 3;
            fixed2[h] = (h ? (sf & SEG_LAST) : (sf & SEG_FIRST)) || (h ? open_r : open_l);
            gaprow2[h] = isrow2 && h == 1 && !(sf & SEG_LAST);
            const bool edge_l = active && isrow2 && sl == 0 && h == 0 && cta > 0;
            const bool edge_r = active && isrow2 && sl == nact - 1 && h == 1 && cta + 1 < nctas;
            pub2[h] = nctas > 1 && (edge_l || edge_r);
            pub2_off[h] = (cta * MBS + (edge_r ? MBS / 2 : 0) + (S + lane) * 3) * 16;
            if (edge_l || edge_r) {
                need2 = true; need2_h = h;
                need2_off = edge_l ? ((cta - 1) * MBS + MBS / 2 + (S + lane) * 3) * 16 : ((cta + 1) * MBS + (S + lane) * 3) * 16;
            }
        }
    }

    // ---- state of iterate k.  Registers hold the a1 OPERANDS:
    //   gM = (z~ - u)/T^k      A0 = (hi - s+ - v+) + (lo + s- + v-)      gv = (phi_v - w_v)/T      ga = (phi_a - w_a)/T^2
    Real gM[2][3], A0[2][3], gv[2][3], ga[2][3];
    Real gM2[2][3] = {{0, 0, 0}, {0, 0, 0}};        // WIDE: operand of the second consensus block, (z~ - u)/T^k
    if (WIDE) {
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const long long i = d * stride + gt[h];
                const Real z0 = static_cast<const Real*>(p.zt2)[i], u0 = static_cast<const Real*>(p.u2)[i];
                zus2[(h * 3 + d) * TS] = make2(z0, u0);
                gM2[h][d] = (z0 - u0) * invTk2[h];
            }
    }
#pragma unroll
    for (int h = 0; h < 2; ++h)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const long long i = d * stride + gt[h];
            const Real z0 = static_cast<const Real*>(p.zt)[i], u0 = static_cast<const Real*>(p.u)[i];
            zus[(h * 3 + d) * TS] = make2(z0, u0);
            gM[h][d] = (z0 - u0) * invTk[h];
            A0[h][d] = gv[h][d] = ga[h][d] = 0;
            Real w_v = 0, w_a = 0, ph_v = 0, ph_a = 0;
            if (has_box) {
                const Real lo = static_cast<const Real*>(p.lohi)[d * p.nseg_pad + gseg], hi = static_cast<const Real*>(p.lohi)[(3 + d) * p.nseg_pad + gseg];
                const Real a = static_cast<const Real*>(p.qp)[i], b = static_cast<const Real*>(p.qn)[i];
                qs[(h * 3 + d) * TS] = make2(a, b);
                A0[h][d] = (hi - fabs(a)) + (lo + fabs(b));
            }
            if (has_vel) { w_v = static_cast<const Real*>(p.wv)[i]; ph_v = static_cast<const Real*>(p.phv)[i]; gv[h][d] = (ph_v - w_v) * invT; }
            if (has_acc) { w_a = static_cast<const Real*>(p.wa)[i]; ph_a = static_cast<const Real*>(p.pha)[i]; ga[h][d] = (ph_a - w_a) * invT2; }
            if (CONS) { ws[(h * 3 + d) * TS] = make2(w_v, w_a); if (!SPLIT) phs[(h * 3 + d) * TS] = make2(ph_v, ph_a); }
        }
    if constexpr (POLY) {      // consensus rows enter the segment's rotated frame; the E0 operand is sum_k (b_k - s_k - v_k) a_k
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            rot_in(vs, gM[h]);
            if (WIDE) rot_in(vs, gM2[h]);
            for (int k = 0; k < KP; ++k) {
                const double2 a01 = *reinterpret_cast<const double2*>(pls + k * 4), a2b = *reinterpret_cast<const double2*>(pls + k * 4 + 2);
                const double g = a2b.y - fabs(qpls[(k * 2 + h) * TS]);
                A0[h][0] += g * a01.x; A0[h][1] += g * a01.y; A0[h][2] += g * a2b.x;
            }
        }
    }

    const Real vmax = (Real)p.vmax, amax = (Real)p.amax;
    unsigned char* const mbox = static_cast<unsigned char*>(p.Bedge);
    const size_t mbox_par_stride = (size_t)p.max_ctas * MBS * 16;
    // cluster exchange (KF_CLUSTER: the grid is one thread-block cluster): the mailbox of a CTA lives in its own shared
    // memory, [2 parity][2 sides: 0 = from the left neighbour, 1 = from the right][MBS/2 slots]; the neighbours store into
    // it through distributed shared memory, this CTA polls it locally
    const bool clus = (flags & KF_CLUSTER) != 0;
    const unsigned cm_local = smem_u32(cmbox);
    unsigned cm_remote[2] = {0, 0};      // the mailbox of the CTA my item h publishes to
    if (clus) {
        cm_remote[0] = cta > 0 ? cluster_map(cm_local, (unsigned)(cta - 1)) : 0u;            // left neighbour
        cm_remote[1] = cta + 1 < nctas ? cluster_map(cm_local, (unsigned)(cta + 1)) : 0u;    // right neighbour
        cluster_barrier();      // every CTA of the cluster runs and has cleared its mailbox before anyone stores into it
        // offsets inside a mailbox (bytes, relative to the parity base): a row at my right edge goes to the right neighbour's
        // half 0, a row at my left edge to the left neighbour's half 1; what I need sits in my own half 0 (left edge) / 1
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const bool er = right[h];
            pub_off[h] = ((er ? 0 : 1) * (MBS / 2) + korder[h] * 3) * 16;
            if (need && need_h == h) need_off = ((er ? 1 : 0) * (MBS / 2) + korder[h] * 3) * 16;
            if (WIDE) {
                pub2_off[h] = ((h ? 0 : 1) * (MBS / 2) + (S + lane) * 3) * 16;
                if (need2 && need2_h == h) need2_off = ((h ? 1 : 0) * (MBS / 2) + (S + lane) * 3) * 16;
            }
        }
    }
    const size_t par_stride = clus ? (size_t)MBS * 16 : mbox_par_stride;
    const int warp = tid >> 5, nwarps = T >> 5;
    const bool pairwise = SPLIT || (nb_sync && nctas > 1 && nwarps <= 17 && (flags & KF_PAIRWISE));
    const int npair = nwarps + (SPLIT ? p.split_octets : 0);      // octets of the CTA (SPLIT: the last ones run on three warps each)
    // in-kernel solve: stop rule and Eq. 24 evaluated on the device (all CTAs all-gather their residual partial
    // sums through LL slots and take the same decision from the same numbers)
    const int ce = SOLVE ? p.check_every : 0;
    double rho_cur = p.rho;
    int ncheck = 0, sweeps_done = p.k_sweeps, stopped = 0, since_test = 0;
    __syncthreads();
    for (int it = 0; it < p.k_sweeps; ++it) {
        const unsigned seq = p.seq_base + (unsigned)it + 1u;
        const int par = (int)(seq & 1u);
        const bool final_sweep = (it == p.k_sweeps - 1);
        // sweeps on which residuals (and the coefficients) are materialised: the last one, and every test sweep
        bool test_sweep = false;
        if (SOLVE && ce > 0 && ++since_test == ce) { since_test = 0; test_sweep = true; }
        const bool last_sweep = final_sweep || test_sweep;
        Real* const Bcur = Bs + par * BPAR;
        Real* const Bcur2 = Bs2 + par * BPAR;
        unsigned char* const mpar = mbox + par * par_stride;     // (cluster exchange: only the offset part is used)
        const unsigned cpar = (unsigned)(par * MBS * 16);

        // ================= phase A: segment local =================
        // operator rows and c0 of this lane: issued first, they arrive while the MMAs of a1 run
        // (polytope corridor: one operator per rotated dim, read inside the dim loop of a2)
        double2 pm[2][4];
        double cacc[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (!POLY) {
#pragma unroll
                for (int b = 0; b < 4; ++b) pm[h][b] = Pms[(h * 4 + b) * TS];
            }
#pragma unroll
            for (int d = 0; d < 3; ++d) cacc[h][d] = c0s[(h * 3 + d) * TS];
        }
        // a1: right-hand side of Eq. 20a (second bracket; rho is folded into the operator, A3):
        // R^ = M^'[(z~ - u)/T^k] + E0'[(hi - s+ - v+) + (lo + s- + v-)] + E1'[(phi_v - w_v)/T] + E2'[(phi_a - w_a)/T^2].
        // Three accumulator tiles (one per dim), up to 8 k-steps each; the accumulator of lane t holds rows 2t, 2t+1.
        {
            Acc acc;
            acc.blk(make_aop(gM), ldb(0, 1));
            if (WIDE) acc.blk(make_aop(gM2), ldb(16, 17));
            if (has_box || POLY) acc.blk(make_aop(A0), ldb(2, 3));      // Ao'(b - s - v): box Ao = [E0; -E0], b = [hi; -lo], s + v = |q| (Moreau pair); polytope: kron(E0, a_k')
            if (has_vel) acc.blk(make_aop(gv), ldb(4, 5));
            if (has_acc) acc.blk(make_aop(ga), ldb(6, 7));
#pragma unroll
            for (int d = 0; d < 3; ++d) *reinterpret_cast<double2*>(Xs + d * 8 + 2 * lane) = make_double2((double)acc.get(d, 0), (double)acc.get(d, 1));
        }
        __syncwarp();
        // a2: x-update  c^ = (rho Pm^) R^ + c0^   (Eq. 20a first bracket, precomputed per segment): rows lane, lane+4
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            if (POLY) {
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int b = 0; b < 4; ++b) pm[h][b] = Pms[((d * 2 + h) * 4 + b) * TS];
            }
#pragma unroll
            for (int b = 0; b < N2 / 2; ++b) {
                const double2 x2 = *reinterpret_cast<const double2*>(Xs + d * 8 + 2 * b);
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    cacc[h][d] += pm[h][b].x * x2.x;
                    cacc[h][d] += pm[h][b].y * x2.y;
                }
            }
        }
        if (last_sweep && owned) {      // (every test sweep as well: the solve may stop there)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int d = 0; d < 3; ++d) static_cast<Real*>(p.chat)[d * stride + gt[h]] = (Real)cacc[h][d];
        }
        // a3: evaluate the new polynomial: consensus rows of B = M c (Eq. 20b), and the lane's two samples of E0 c, E1 c,
        // E2 c (Eq. 20d-g).  A operand = the lane's own coefficient rows; accumulator columns = the lane's own items.
        Real cf[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int d = 0; d < 3; ++d) cf[h][d] = (Real)cacc[h][d];
        const AOp cop = make_aop(cf);
        {
            Real Bnd[2][3];
            {
                Acc e;
                e.blk(cop, ldb(8, 12));
#pragma unroll
                for (int d = 0; d < 3; ++d) { Bnd[0][d] = (Real)e.get(d, 0) * invTk[0]; Bnd[1][d] = (Real)e.get(d, 1) * invTk[1]; }
            }
            if constexpr (POLY) { rot_out(vs, Bnd[0]); rot_out(vs, Bnd[1]); }      // consensus lives in the global frame
            // publish: shared memory for the neighbours in this CTA (and for this lane's own phase B), mailbox for the
            // neighbouring CTAs
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (isrow[h]) {
#pragma unroll
                    for (int d = 0; d < 3; ++d) Bcur[own_off[h] + d] = Bnd[h][d];
                }
                if (pub[h]) {
                    if (clus) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) ll_store_cluster(cm_remote[right[h] ? 1 : 0] + cpar + pub_off[h] + d * 16, (double)Bnd[h][d], seq);
                    } else {
#pragma unroll
                        for (int d = 0; d < 3; ++d) ll_store(mpar + pub_off[h] + d * 16, (double)Bnd[h][d], seq);
                    }
                }
            }
        }
        if (WIDE) {     // boundary derivatives of orders s..2s-2 (second block of B = M c)
            Real Bnd2[2][3];
            {
                Acc e;
                e.blk(cop, ldb(18, 19));
#pragma unroll
                for (int d = 0; d < 3; ++d) { Bnd2[0][d] = (Real)e.get(d, 0) * invTk2[0]; Bnd2[1][d] = (Real)e.get(d, 1) * invTk2[1]; }
            }
            if constexpr (POLY) { rot_out(vs, Bnd2[0]); rot_out(vs, Bnd2[1]); }      // consensus lives in the global frame
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (isrow2) {
#pragma unroll
                    for (int d = 0; d < 3; ++d) Bcur2[own2_off[h] + d] = Bnd2[h][d];
                }
                if (pub2[h]) {
                    if (clus) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) ll_store_cluster(cm_remote[h] + cpar + pub2_off[h] + d * 16, (double)Bnd2[h][d], seq);
                    } else {
#pragma unroll
                        for (int d = 0; d < 3; ++d) ll_store(mpar + pub2_off[h] + d * 16, (double)Bnd2[h][d], seq);
                    }
                }
            }
        }
        // prefetch the rows of the neighbouring CTA: the loads fly during the projections
        LLRaw rr[3], rr2[3];
        if (need) {
#pragma unroll
            for (int d = 0; d < 3; ++d) { if (clus) ll_issue_smem(cm_local + cpar + need_off + d * 16, rr[d]); else ll_issue(mpar + need_off + d * 16, rr[d]); }
        }
        if (WIDE && need2) {
#pragma unroll
            for (int d = 0; d < 3; ++d) { if (clus) ll_issue_smem(cm_local + cpar + need2_off + d * 16, rr2[d]); else ll_issue(mpar + need2_off + d * 16, rr2[d]); }
        }
        if (CONS) {
            // the three sample blocks of the evaluation back to back, then the projections of all blocks side by side:
            // independent dependency chains, no branch between them
            Real Pv[2][3], Vv[2][3], Av[2][3];
            Acc ev, ea, ep;
            if (has_vel) ev.blk(cop, ldb(10, 14));
            if (has_acc) ea.blk(cop, ldb(11, 15));
            if (has_box || POLY) ep.blk(cop, ldb(9, 13));
            if (has_vel) {
#pragma unroll
                for (int d = 0; d < 3; ++d) { Vv[0][d] = (Real)ev.get(d, 0); Vv[1][d] = (Real)ev.get(d, 1); }
            }
            if (has_acc) {
#pragma unroll
                for (int d = 0; d < 3; ++d) { Av[0][d] = (Real)ea.get(d, 0); Av[1][d] = (Real)ea.get(d, 1); }
            }
            if (has_box || POLY) {
#pragma unroll
                for (int d = 0; d < 3; ++d) { Pv[0][d] = (Real)ep.get(d, 0); Pv[1][d] = (Real)ep.get(d, 1); }
            }
            R2 w2[2][3], q2[2][3];
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    if (has_vel || has_acc) w2[h][d] = ws[(h * 3 + d) * TS];
                    if (has_box) q2[h][d] = qs[(h * 3 + d) * TS];
                }
            // a4: Eq. 20f, 20g;  y = A c + w,  phi = proj(y),  w <- y - phi;  next operand (phi - w)/T
            R2 ph2[2][3];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (has_vel) {
                    Real y[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) y[d] = Vv[h][d] * invT + w2[h][d].x;
                    const Real scale = ball_scale(y, vmax);
#pragma unroll
                    for (int d = 0; d < 3; ++d) { const Real ph = scale * y[d]; ph2[h][d].x = ph; w2[h][d].x = y[d] - ph; gv[h][d] = ((ph - w2[h][d].x) * invT); }
                } else {
#pragma unroll
                    for (int d = 0; d < 3; ++d) ph2[h][d].x = 0;
                }
                if (has_acc) {
                    Real y[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) y[d] = Av[h][d] * invT2 + w2[h][d].y;
                    const Real scale = ball_scale(y, amax);
#pragma unroll
                    for (int d = 0; d < 3; ++d) { const Real ph = scale * y[d]; ph2[h][d].y = ph; w2[h][d].y = y[d] - ph; ga[h][d] = ((ph - w2[h][d].y) * invT2); }
                } else {
#pragma unroll
                    for (int d = 0; d < 3; ++d) ph2[h][d].y = 0;
                }
            }
            if (has_vel || has_acc) {
#pragma unroll
                for (int h = 0; h < 2; ++h)
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        ws[(h * 3 + d) * TS] = w2[h][d];
                        // phi itself is only read back at the end of the launch and by the rho change of a test sweep (its
                        // effect on the next sweep is already in the operands gv, ga)
                        // (SPLIT: that slot of shared memory is the split octets' ball exchange; phi goes straight out)
                        if (last_sweep) {
                            if (!SPLIT) phs[(h * 3 + d) * TS] = ph2[h][d];
                            else if (owned) {
                                if (has_vel) static_cast<Real*>(p.phv_out)[d * stride + gt[h]] = ph2[h][d].x;
                                if (has_acc) static_cast<Real*>(p.pha_out)[d * stride + gt[h]] = ph2[h][d].y;
                            }
                        }
                    }
            }
            if constexpr (POLY) {         // a7 + a8 per (sample, plane): q = -(a_k'p - b_k + v);  next operand sum_k (b_k - |q_k|) a_k
#pragma unroll
                for (int h = 0; h < 2; ++h) A0[h][0] = A0[h][1] = A0[h][2] = 0.0;
                for (int k = 0; k < KP; ++k) {
                    const double2 a01 = *reinterpret_cast<const double2*>(pls + k * 4), a2b = *reinterpret_cast<const double2*>(pls + k * 4 + 2);
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const double val = a01.x * Pv[h][0] + a01.y * Pv[h][1] + a2b.x * Pv[h][2];
                        const double qn_ = (a2b.y - val) - neg_part(qpls[(k * 2 + h) * TS]);
                        qpls[(k * 2 + h) * TS] = qn_;
                        const double g = a2b.y - fabs(qn_);
                        A0[h][0] += g * a01.x; A0[h][1] += g * a01.y; A0[h][2] += g * a2b.x;
                    }
                }
            }
            if (has_box) {      // a7 + a8: Eq. 20d, 20e with q = -(A c - b + v):  s = max(0,q),  v <- max(0,-q);  next operand
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const Real lo = lohi[d * SA], hi = lohi[(3 + d) * SA];
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const Real qpn = (hi - Pv[h][d]) - neg_part(q2[h][d].x), qnn = (Pv[h][d] - lo) - neg_part(q2[h][d].y);
                        qs[(h * 3 + d) * TS] = make2(qpn, qnn);
                        A0[h][d] = ((hi - fabs(qpn)) + (lo + fabs(qnn)));
                    }
                }
            }
        }

        // ================= exchange of boundary rows =================
        int wait_failed = 0;
        {
            bool okk = !need || (ll_ok(rr[0], seq) && ll_ok(rr[1], seq) && ll_ok(rr[2], seq));
            bool okk2 = !(WIDE && need2) || (ll_ok(rr2[0], seq) && ll_ok(rr2[1], seq) && ll_ok(rr2[2], seq));
            if (pairwise && *(volatile int*)&abort_any) okk = okk2 = true;
            if (!__all_sync(0xffffffffu, okk && okk2)) {
                const long long t0 = global_ns();
                unsigned spins = 0;
                do {
                    if (!okk) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) { if (clus) ll_issue_smem(cm_local + cpar + need_off + d * 16, rr[d]); else ll_issue(mpar + need_off + d * 16, rr[d]); }
                        okk = ll_ok(rr[0], seq) && ll_ok(rr[1], seq) && ll_ok(rr[2], seq);
                    }
                    if (WIDE && !okk2) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) { if (clus) ll_issue_smem(cm_local + cpar + need2_off + d * 16, rr2[d]); else ll_issue(mpar + need2_off + d * 16, rr2[d]); }
                        okk2 = ll_ok(rr2[0], seq) && ll_ok(rr2[1], seq) && ll_ok(rr2[2], seq);
                    }
                    bool bail = false;
                    if ((++spins & 255u) == 0) bail = *(volatile int*)p.abort_flag || global_ns() - t0 > WAIT_TIMEOUT_NS;
                    if (__any_sync(0xffffffffu, bail)) { if (!(okk && okk2)) { atomicExch(p.abort_flag, 1); wait_failed = 1; } break; }
                } while (!__all_sync(0xffffffffu, okk && okk2));
            }
        }
        if (wait_failed) { abort_sh[it & 1] = 1; *(volatile int*)&abort_any = 1; }
        if (pairwise) {
            const int first = (warp & 1) ? warp - 1 : warp, second = (warp & 1) ? warp : warp - 1;
            if (first >= 0 && first + 1 < npair) asm volatile("bar.sync %0, %1;" ::"r"(first), "r"(SPLIT ? pair_threads(first, nwarps) : 64) : "memory");
            if (second >= 0 && second + 1 < npair) asm volatile("bar.sync %0, %1;" ::"r"(second), "r"(SPLIT ? pair_threads(second, nwarps) : 64) : "memory");
        } else if (nctas == 1) {
            __syncthreads();
        } else if (!nb_sync) {
            if (!grid_barrier(p.bar, (unsigned long long)(it + 1) * nctas, p.abort_flag)) break;
            if (abort_sh[it & 1]) break;
        } else {
            __syncthreads();
            if (abort_sh[it & 1]) break;
        }

        // ================= phase B: consensus, dual, residuals =================
        // everything is loaded first (own rows, neighbour rows, frame shifts, (z~, u)), then updated, then stored
        Real own[2][3], nb[2][3];
        R2 zu[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                own[h][d] = Bcur[own_off[h] + d];
                nb[h][d] = Bcur[nb_off[h] + d];
                zu[h][d] = zus[(h * 3 + d) * TS];
            }
        if (need) {
#pragma unroll
            for (int d = 0; d < 3; ++d) { const Real v = (Real)ll_value(rr[d]); if (need_h == 0) nb[0][d] = v; else nb[1][d] = v; }
        }
#pragma unroll
        for (int h = 0; h < 2; ++h)
            if (zshift[h]) {
#pragma unroll
                for (int d = 0; d < 3; ++d) nb[h][d] += zoffs[((right[h] ? 3 : 0) + d) * SA];
            }
        double rp2 = 0, rd2 = 0, rdn2 = 0, gap2 = 0;
        Real dz[2][3];
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const Real avg = (Real)0.5 * (own[h][d] + nb[h][d]);
                const Real znew = (fixed[h] || !isrow[h]) ? zu[h][d].x : avg;    // a5: Eq. 6b / 20b
                dz[h][d] = znew - zu[h][d].x;
                const Real res = isrow[h] ? own[h][d] - znew : (Real)0;
                const Real unew = zu[h][d].y + res;                               // a8: Eq. 6c / 20c (scaled dual, A5)
                zus[(h * 3 + d) * TS] = make2(znew, unew);
                gM[h][d] = ((znew - unew) * invTk[h]);                                // operand of the next sweep's a1
                if (last_sweep) rp_accum(rp2, gap2, (double)res, gaprow[h], (double)own[h][d], (double)nb[h][d]);
            }
        if constexpr (POLY) { rot_in(vs, gM[0]); rot_in(vs, gM[1]); }
        Real dz2[2][3] = {{0, 0, 0}, {0, 0, 0}};
        if (WIDE) {     // the same consensus / dual step on the rows of orders s..2s-2 (never position rows: no frame shift)
#pragma unroll
            for (int h = 0; h < 2; ++h)
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    const Real own2 = Bcur2[own2_off[h] + d];
                    Real nb2 = Bcur2[nb2_off[h] + d];
                    if (need2 && need2_h == h) nb2 = (Real)ll_value(rr2[d]);
                    const R2 zu2 = zus2[(h * 3 + d) * TS];
                    const Real avg = (Real)0.5 * (own2 + nb2);
                    const Real znew = (fixed2[h] || !isrow2) ? zu2.x : avg;             // a5: Eq. 6b / 20b
                    dz2[h][d] = znew - zu2.x;
                    const Real res = (isrow2 && !fixed2[h]) ? own2 - znew : (Real)0;    // rows at the trajectory ends do not exist (A1)
                    const Real unew = zu2.y + res;                                      // a8: Eq. 6c / 20c
                    zus2[(h * 3 + d) * TS] = make2(znew, unew);
                    gM2[h][d] = ((znew - unew) * invTk2[h]);
                    if (last_sweep) rp_accum(rp2, gap2, (double)res, gaprow2[h], (double)own2, (double)nb2);
                }
            if constexpr (POLY) { rot_in(vs, gM2[0]); rot_in(vs, gM2[1]); }
        }
        if (last_sweep) {
            // a6: dual residual rho M(T)'(z~^{k+1} - z~^k) in monomial physical-time coefficient space (Eq. 22, A8):
            // the consensus block of the a1 contraction applied to dz; lane t ends with coefficient rows 2t, 2t+1
            const double Tp0 = (double)static_cast<const Real*>(p.Tpow)[gseg * LANES + 2 * lane];
            const double Tp1 = (double)static_cast<const Real*>(p.Tpow)[gseg * LANES + 2 * lane + 1];
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                double x0 = 0, x1 = 0;
                dmma884(x0, x1, (double)(dz[0][d] * invTk[0]), ctab[0 * 32]);
                dmma884(x0, x1, (double)(dz[1][d] * invTk[1]), ctab[1 * 32]);
                if (WIDE) {
                    dmma884(x0, x1, (double)(dz2[0][d] * invTk2[0]), ctab[16 * 32]);
                    dmma884(x0, x1, (double)(dz2[1][d] * invTk2[1]), ctab[17 * 32]);
                }
                rd_accum(rd2, rdn2, rho_cur * x0, rho_cur * x1, Tp0, Tp1);
            }
#pragma unroll
            for (int m = 1; m < LPS; m <<= 1) {     // fixed-order tree over the 4 lanes of the segment
                rp2 += shfl_xor(rp2, m); rd2 += shfl_xor(rd2, m); rdn2 += shfl_xor(rdn2, m); gap2 += shfl_xor(gap2, m);
            }
            if (owned && lane == 0) {
                double* o = p.part + gseg * 4;
                o[0] = rp2; o[1] = rd2; o[2] = rdn2; o[3] = gap2;
            }
            if (SOLVE && ce > 0) {
                // ---- CTA partial (fixed order), all-gather over the CTAs, decision
                double q4[4] = {rp2, rd2, rdn2, gap2};
                if (!(owned && lane == 0)) { q4[0] = q4[1] = q4[2] = q4[3] = 0.0; }
#pragma unroll
                for (int k = 0; k < 4; ++k) { q4[k] += shfl_xor(q4[k], 4); q4[k] += shfl_xor(q4[k], 8); q4[k] += shfl_xor(q4[k], 16); }
                if ((tid & 31) == 0) { for (int k = 0; k < 4; ++k) wsum_sh[tid >> 5][k] = q4[k]; }
                double rho_new = rho_cur;
                if (solve_decide(p, seq, npair, wsum_sh, allp_sh, tot_sh, cresbox, ncheck, rho_cur, rho_new, stopped)) { sweeps_done = it + 1; break; }
                {
                    if (rho_new != rho_cur) {      // reading A16 for the scaled duals
                        const Real ratio = (Real)(rho_cur / rho_new);
                        // u, w, v = max(0,-q) are scaled duals: times rho_old/rho_new; then the operands that depend on them
#pragma unroll
                        for (int h = 0; h < 2; ++h) {
#pragma unroll
                            for (int d = 0; d < 3; ++d) {
                                R2 zz = zus[(h * 3 + d) * TS];
                                zz.y *= ratio;
                                zus[(h * 3 + d) * TS] = zz;
                                gM[h][d] = ((zz.x - zz.y) * invTk[h]);
                                if (WIDE) {
                                    R2 z2 = zus2[(h * 3 + d) * TS];
                                    z2.y *= ratio;
                                    zus2[(h * 3 + d) * TS] = z2;
                                    gM2[h][d] = ((z2.x - z2.y) * invTk2[h]);
                                }
                                if (has_box) {
                                    const Real lo = lohi[d * SA], hi = lohi[(3 + d) * SA];
                                    R2 q = qs[(h * 3 + d) * TS];
                                    if (q.x < 0) q.x *= ratio;
                                    if (q.y < 0) q.y *= ratio;
                                    qs[(h * 3 + d) * TS] = q;
                                    A0[h][d] = ((hi - fabs(q.x)) + (lo + fabs(q.y)));
                                }
                                if (has_vel || has_acc) {
                                    R2 w2 = ws[(h * 3 + d) * TS];
                                    const R2 ph = phs[(h * 3 + d) * TS];
                                    w2.x *= ratio; w2.y *= ratio;
                                    ws[(h * 3 + d) * TS] = w2;
                                    if (has_vel) gv[h][d] = ((ph.x - w2.x) * invT);
                                    if (has_acc) ga[h][d] = ((ph.y - w2.y) * invT2);
                                }
                            }
                            refresh_operator_rows<N2, TS>(p, gseg, gt[h], jj[h], rho_new, Pms + h * 4 * TS, c0s + h * 3 * TS);
                        }
                        rho_cur = rho_new;
                    }
                }
            }
        }
    }
    if (SOLVE && ce > 0 && cta == 0 && tid == 0) {
        double* o = p.solve_out;
        o[0] = (double)sweeps_done; o[1] = (double)stopped; o[2] = rho_cur;
        o[3] = sqrt(tot_sh[0]); o[4] = sqrt(tot_sh[1]); o[5] = sqrt(tot_sh[2]); o[6] = sqrt(tot_sh[3]);
    }

    if (clus) cluster_barrier();      // nobody leaves while a neighbour may still store into its mailbox
    // ---- write iterate k + k_sweeps back
    if (owned) {
#pragma unroll
        for (int h = 0; h < 2; ++h)
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const long long i = d * stride + gt[h];
                const R2 zz = zus[(h * 3 + d) * TS];
                static_cast<Real*>(p.zt_out)[i] = zz.x;
                static_cast<Real*>(p.u_out)[i] = zz.y;
                if (WIDE) { const R2 z2 = zus2[(h * 3 + d) * TS]; static_cast<Real*>(p.zt2)[i] = z2.x; static_cast<Real*>(p.u2)[i] = z2.y; }
                if (has_box) { const R2 q = qs[(h * 3 + d) * TS]; static_cast<Real*>(p.qp_out)[i] = q.x; static_cast<Real*>(p.qn_out)[i] = q.y; }
                if (POLY && d == 0) for (int k = 0; k < KP; ++k) static_cast<double*>(p.qpl_out)[k * stride + gt[h]] = qpls[(k * 2 + h) * TS];
                if (has_vel || has_acc) {
                    const R2 w2 = ws[(h * 3 + d) * TS];
                    R2 ph = make2((Real)0, (Real)0);
                    const bool ph_here = !SPLIT || p.k_sweeps == 0;      // (SPLIT: phi went out on the last sweep)
                    if (!SPLIT) ph = phs[(h * 3 + d) * TS];
                    else if (p.k_sweeps == 0) ph = make2(has_vel ? static_cast<const Real*>(p.phv)[i] : (Real)0, has_acc ? static_cast<const Real*>(p.pha)[i] : (Real)0);
                    if (has_vel) { static_cast<Real*>(p.wv_out)[i] = w2.x; if (ph_here) static_cast<Real*>(p.phv_out)[i] = ph.x; }
                    if (has_acc) { static_cast<Real*>(p.wa_out)[i] = w2.y; if (ph_here) static_cast<Real*>(p.pha_out)[i] = ph.y; }
                }
            }
    }
    }      // if constexpr (!(SPLIT && SOLVE))
}

// one launch: a single CTA plainly; KF_CLUSTER: the whole grid as ONE thread-block cluster (<= 16 CTAs, co-scheduled by
// the hardware); otherwise cooperatively (all CTAs co-resident: they wait for one another through the L2 mailbox)
template <typename K>
cudaError_t launch_any(K kern, const KParams& p, int ctas, int threads, size_t smem, cudaStream_t st) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    KParams pc = p;
    void* args[] = {&pc};
    if (ctas > 1 && (p.flags & KF_CLUSTER)) {
        if (ctas > 8 && (e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1)) != cudaSuccess) return e;
        cudaLaunchConfig_t cfg;
        memset(&cfg, 0, sizeof cfg);
        cfg.gridDim = dim3(ctas); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)ctas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        return cudaLaunchKernelExC(&cfg, (const void*)kern, args);
    }
    if (ctas > 1) return cudaLaunchCooperativeKernel((const void*)kern, dim3(ctas), dim3(threads), args, smem, st);
    return cudaLaunchKernel((const void*)kern, dim3(ctas), dim3(threads), args, smem, st);
}

template <typename Real, int S, int CM, int MAXT>
cudaError_t launch_mma(const KParams& p, int ctas, int threads, size_t smem, cudaStream_t st) {
    auto kern = p.check_every > 0 ? cadmm_sweeps_mma_kernel<Real, S, CM, MAXT, true> : cadmm_sweeps_mma_kernel<Real, S, CM, MAXT, false>;
    return launch_any(kern, p, ctas, threads, smem, st);
}

// can `ctas` CTAs of this size run as ONE thread-block cluster?  *nclusters = co-resident clusters (0: no)
template <typename K>
cudaError_t cluster_query(K kern, int ctas, int threads, size_t smem, int* nclusters) {
    *nclusters = 0;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (ctas > 8 && (e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1)) != cudaSuccess) return e;
    cudaLaunchConfig_t cfg;
    memset(&cfg, 0, sizeof cfg);
    cfg.gridDim = dim3(ctas); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)ctas; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaOccupancyMaxActiveClusters(nclusters, (const void*)kern, &cfg);
}
// SPLIT instantiations (fp64, box + velocity [+ acceleration], plain sweeps): `threads` counts one warp per octet as planned; the
// launch runs the last `nsplit` octets on three warps each
template <int S, int CM>
cudaError_t launch_mma_split(const KParams& p, int nsplit, int ctas, int threads, size_t smem, cudaStream_t st) {
    auto kern = p.check_every > 0 ? cadmm_sweeps_mma_kernel<double, S, CM, MAXT_MMA, true, false, false, true>
                                  : cadmm_sweeps_mma_kernel<double, S, CM, MAXT_MMA, false, false, false, true>;
    KParams ps = p;
    ps.split_octets = nsplit;
    return launch_any(kern, ps, ctas, threads + 64 * nsplit, smem, st);
}
template <int S, int CM>
cudaError_t cluster_mma_split(int ctas, int threads, size_t smem, int* nclusters) {
    int a = 0, b = 0;
    cudaError_t e = cluster_query(cadmm_sweeps_mma_kernel<double, S, CM, MAXT_MMA, true, false, false, true>, ctas, threads, smem, &a);
    if (e != cudaSuccess) return e;
    e = cluster_query(cadmm_sweeps_mma_kernel<double, S, CM, MAXT_MMA, false, false, false, true>, ctas, threads, smem, &b);
    *nclusters = a < b ? a : b;
    return e;
}

template <typename Real, int S, int CM, int MAXT>
cudaError_t cluster_mma(int ctas, int threads, size_t smem, int* nclusters) {
    int a = 0, b = 0;
    cudaError_t e = cluster_query(cadmm_sweeps_mma_kernel<Real, S, CM, MAXT, true>, ctas, threads, smem, &a);
    if (e != cudaSuccess) return e;
    e = cluster_query(cadmm_sweeps_mma_kernel<Real, S, CM, MAXT, false>, ctas, threads, smem, &b);
    *nclusters = a < b ? a : b;
    return e;
}

template <typename Real, int S, int CM, int MAXT>
cudaError_t limits_mma(int threads, size_t smem, int* per_sm) {
    auto kern = cadmm_sweeps_mma_kernel<Real, S, CM, MAXT, true>;     // the larger of the two instantiations
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, threads, smem);
}

template <int S>
cudaError_t launch_mma_wide(const KParams& p, int ctas, int threads, size_t smem, cudaStream_t st) {
    auto kern = p.check_every > 0 ? cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_WIDE, true, false, true>
                                  : cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_WIDE, false, false, true>;
    return launch_any(kern, p, ctas, threads, smem, st);
}
template <int S>
cudaError_t limits_mma_wide(int threads, size_t smem, int* per_sm) {
    auto kern = cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_WIDE, true, false, true>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, threads, smem);
}

template <int S>
cudaError_t launch_mma_poly(const KParams& p, int ctas, int threads, size_t smem, cudaStream_t st) {
    auto kern = cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_POLY, false, true>;
    return launch_any(kern, p, ctas, threads, smem, st);
}
template <int S>
cudaError_t launch_mma_poly_wide(const KParams& p, int ctas, int threads, size_t smem, cudaStream_t st) {
    auto kern = cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_POLY_WIDE, false, true, true>;
    return launch_any(kern, p, ctas, threads, smem, st);
}
template <int S>
cudaError_t limits_mma_poly_wide(int threads, size_t smem, int* per_sm) {
    auto kern = cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_POLY_WIDE, false, true, true>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, threads, smem);
}
template <int S>
cudaError_t limits_mma_poly(int threads, size_t smem, int* per_sm) {
    auto kern = cadmm_sweeps_mma_kernel<double, S, CM_RUNTIME, MAXT_MMA_POLY, false, true>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, threads, smem);
}

// constraint selection -> instantiation: none, box + velocity, box + velocity + acceleration; anything else at run time
int mma_mask(uint32_t kflags) {
    const int m = (int)(kflags & (KF_BOX | KF_VEL | KF_ACC));
    return (m == 0 || m == 3 || m == 7) ? m : CM_RUNTIME;
}

}  // namespace

// fp64: one instantiation of <= 288 threads.  fp32 (mixed): the state is half the size, <= 384 threads (12 warps of 8 segments:
// three warps on every scheduler, 168 registers)
#define TOP_DISPATCH_MMA(CALL)                                                                              \
    const int cm = mma_mask(kflags);                                                                        \
    if (dtype == 0) {                                                                                       \
        if (s == 3) { if (cm == 0) { CALL(double, 3, 0, MAXT_MMA) } else if (cm == 3) { CALL(double, 3, 3, MAXT_MMA) } else if (cm == 7) { CALL(double, 3, 7, MAXT_MMA) } else { CALL(double, 3, CM_RUNTIME, MAXT_MMA) } } \
        else        { if (cm == 0) { CALL(double, 4, 0, MAXT_MMA) } else if (cm == 3) { CALL(double, 4, 3, MAXT_MMA) } else if (cm == 7) { CALL(double, 4, 7, MAXT_MMA) } else { CALL(double, 4, CM_RUNTIME, MAXT_MMA) } } \
    } else {                                                                                                \
        if (s == 3) { if (cm == 0) { CALL(float, 3, 0, MAXT_MMA_F32) } else if (cm == 3) { CALL(float, 3, 3, MAXT_MMA_F32) } else if (cm == 7) { CALL(float, 3, 7, MAXT_MMA_F32) } else { CALL(float, 3, CM_RUNTIME, MAXT_MMA_F32) } } \
        else        { if (cm == 0) { CALL(float, 4, 0, MAXT_MMA_F32) } else if (cm == 3) { CALL(float, 4, 3, MAXT_MMA_F32) } else if (cm == 7) { CALL(float, 4, 7, MAXT_MMA_F32) } else { CALL(float, 4, CM_RUNTIME, MAXT_MMA_F32) } } \
    }

int max_threads_mma(int dtype, bool poly, bool wide) {
    return poly && wide ? MAXT_MMA_POLY_WIDE : wide ? MAXT_MMA_WIDE : poly ? MAXT_MMA_POLY : (dtype == 0 ? MAXT_MMA : MAXT_MMA_F32);
}

// Split tail (see split_tail_sweeps): a plain fp64 launch of several CTAs with warp-pair synchronisation over the L2 mailbox whose
// CTAs hold 4k+1 octets (5 or 9 warps) runs its last octet on three warps.  TOP_SPLIT_TAIL=0 in the environment keeps the
// unsplit launch (A/B measurements; the results are bit-identical).
bool split_supported(uint32_t f, int dtype) {
    const int cm = mma_mask(f);
    return dtype == 0 && !(f & (KF_POLY | KF_WIDE)) && (cm == 3 || cm == 7);
}

int split_octets_for(uint32_t f, int check_every, int dtype, int ctas, int threads) {
    // TOP_SPLIT_TAIL=0: never; =1: only the tail of 4k+1 octets; unset: also every octet of CTAs of <= 4 octets
    static const int mode = [] { const char* e = getenv("TOP_SPLIT_TAIL"); return !e ? 2 : (e[0] == '0' ? 0 : (e[0] == '1' ? 1 : 2)); }();
    const int warps = threads / 32;
    if (!split_supported(f, dtype) || mode == 0 || ctas < 2 || !(f & KF_NEIGHBOUR_SYNC) || threads % 32 != 0) return 0;
    // short chains run as one cluster: every octet on three warps (measured, us per sweep, box + velocity: 1 octet per CTA
    // 1.36 -> 1.02, 2 octets 1.35 -> 1.17, 3 octets 1.36 -> 1.28, 4 octets 1.39 -> 1.43; over the L2 mailbox it does not pay)
    // (with the in-kernel stop rule as well: config 2, a test every sweep 3.08 -> 2.74 us per sweep, every 8th 1.75 -> 1.34)
    if ((f & KF_CLUSTER) && warps <= SPLIT_MAX_ALL) return mode > 1 ? warps : 0;
    // long chains: the tail of 4k+1 octets (plain sweeps under warp-pair synchronisation)
    return check_every == 0 && (f & KF_PAIRWISE) && !(f & KF_CLUSTER) && (warps == 5 || warps == 9) ? 1 : 0;
}

cudaError_t launch_sweeps_mma(const KParams& p, int dtype, int s, int ctas, int threads, size_t smem, cudaStream_t st) {
    const uint32_t kflags = p.flags;
    if (kflags & KF_POLY) {
        if (p.check_every > 0 || dtype != 0) return cudaErrorInvalidValue;      // host loop only, fp64 only
        if (kflags & KF_WIDE) return s == 3 ? launch_mma_poly_wide<3>(p, ctas, threads, smem, st) : launch_mma_poly_wide<4>(p, ctas, threads, smem, st);
        return s == 3 ? launch_mma_poly<3>(p, ctas, threads, smem, st) : launch_mma_poly<4>(p, ctas, threads, smem, st);
    }
    if (kflags & KF_WIDE) {
        if (dtype != 0) return cudaErrorInvalidValue;      // fp64 only
        return s == 3 ? launch_mma_wide<3>(p, ctas, threads, smem, st) : launch_mma_wide<4>(p, ctas, threads, smem, st);
    }
    if (const int ns = split_octets_for(p.flags, p.check_every, dtype, ctas, threads)) {
        const int cm = mma_mask(kflags);
        if (s == 3) return cm == 3 ? launch_mma_split<3, 3>(p, ns, ctas, threads, smem, st) : launch_mma_split<3, 7>(p, ns, ctas, threads, smem, st);
        return cm == 3 ? launch_mma_split<4, 3>(p, ns, ctas, threads, smem, st) : launch_mma_split<4, 7>(p, ns, ctas, threads, smem, st);
    }
#define CALL(R_, S_, C_, M_) return launch_mma<R_, S_, C_, M_>(p, ctas, threads, smem, st);
    TOP_DISPATCH_MMA(CALL)
#undef CALL
    return cudaErrorInvalidValue;
}

cudaError_t sweep_kernel_limits_mma(int dtype, int s, uint32_t kflags, int threads, size_t smem, int* max_ctas_per_sm) {
    if ((kflags & KF_POLY) && (kflags & KF_WIDE)) return s == 3 ? limits_mma_poly_wide<3>(threads, smem, max_ctas_per_sm) : limits_mma_poly_wide<4>(threads, smem, max_ctas_per_sm);
    if (kflags & KF_POLY) return s == 3 ? limits_mma_poly<3>(threads, smem, max_ctas_per_sm) : limits_mma_poly<4>(threads, smem, max_ctas_per_sm);
    if (kflags & KF_WIDE) return s == 3 ? limits_mma_wide<3>(threads, smem, max_ctas_per_sm) : limits_mma_wide<4>(threads, smem, max_ctas_per_sm);
#define CALL(R_, S_, C_, M_) return limits_mma<R_, S_, C_, M_>(threads, smem, max_ctas_per_sm);
    TOP_DISPATCH_MMA(CALL)
#undef CALL
    return cudaErrorInvalidValue;
}

// 0 in *nclusters: the launch cannot run as one cluster (too many CTAs for a GPC at this shared-memory size): L2 mailbox then
cudaError_t sweep_cluster_limits_mma(int dtype, int s, uint32_t kflags, int ctas, int threads, size_t smem, int* nclusters) {
    *nclusters = 0;
    if (ctas < 2 || ctas > 16) return cudaSuccess;
    if ((kflags & KF_POLY) && (kflags & KF_WIDE))
        return s == 3 ? cluster_query(cadmm_sweeps_mma_kernel<double, 3, CM_RUNTIME, MAXT_MMA_POLY_WIDE, false, true, true>, ctas, threads, smem, nclusters)
                      : cluster_query(cadmm_sweeps_mma_kernel<double, 4, CM_RUNTIME, MAXT_MMA_POLY_WIDE, false, true, true>, ctas, threads, smem, nclusters);
    if (kflags & KF_POLY)
        return s == 3 ? cluster_query(cadmm_sweeps_mma_kernel<double, 3, CM_RUNTIME, MAXT_MMA_POLY, false, true>, ctas, threads, smem, nclusters)
                      : cluster_query(cadmm_sweeps_mma_kernel<double, 4, CM_RUNTIME, MAXT_MMA_POLY, false, true>, ctas, threads, smem, nclusters);
    if (kflags & KF_WIDE) {
        int a = 0, b = 0;
        cudaError_t e = s == 3 ? cluster_query(cadmm_sweeps_mma_kernel<double, 3, CM_RUNTIME, MAXT_MMA_WIDE, true, false, true>, ctas, threads, smem, &a)
                               : cluster_query(cadmm_sweeps_mma_kernel<double, 4, CM_RUNTIME, MAXT_MMA_WIDE, true, false, true>, ctas, threads, smem, &a);
        if (e != cudaSuccess) return e;
        e = s == 3 ? cluster_query(cadmm_sweeps_mma_kernel<double, 3, CM_RUNTIME, MAXT_MMA_WIDE, false, false, true>, ctas, threads, smem, &b)
                   : cluster_query(cadmm_sweeps_mma_kernel<double, 4, CM_RUNTIME, MAXT_MMA_WIDE, false, false, true>, ctas, threads, smem, &b);
        *nclusters = a < b ? a : b;
        return e;
    }
    if (const int ns = split_octets_for(kflags | KF_CLUSTER | KF_NEIGHBOUR_SYNC | KF_PAIRWISE, 0, dtype, ctas, threads)) {
        // plain sweeps of this plan run the SPLIT instantiation (more threads per CTA); the in-kernel solve the unsplit one: both must fit
        const int cmm = mma_mask(kflags);
        int a = 0;
        cudaError_t e = s == 3 ? (cmm == 3 ? cluster_mma_split<3, 3>(ctas, threads + 64 * ns, smem, &a) : cluster_mma_split<3, 7>(ctas, threads + 64 * ns, smem, &a))
                               : (cmm == 3 ? cluster_mma_split<4, 3>(ctas, threads + 64 * ns, smem, &a) : cluster_mma_split<4, 7>(ctas, threads + 64 * ns, smem, &a));
        if (e != cudaSuccess) return e;
        if (a < 1) return cudaSuccess;
    }
#define CALL(R_, S_, C_, M_) return cluster_mma<R_, S_, C_, M_>(ctas, threads, smem, nclusters);
    TOP_DISPATCH_MMA(CALL)
#undef CALL
    return cudaErrorInvalidValue;
}

size_t sweep_smem_bytes_mma(int dtype, bool constrained, bool poly, bool wide) {      // laid out for the largest CTA of the instantiation (see the kernel)
    if (wide && poly) return smem_layout_mma(true, MAXT_MMA_POLY_WIDE / 4, true, 8, true).total;
    if (wide) return smem_layout_mma(true, MAXT_MMA_WIDE / 4, false, 8, true).total;      // (run-time constraint mask: laid out with the constraint arrays)
    if (poly) return smem_layout_mma(true, MAXT_MMA_POLY / 4, true).total;
    return dtype == 0 ? smem_layout_mma(constrained, MAXT_MMA / 4).total : smem_layout_mma(constrained, MAXT_MMA_F32 / 4, false, 4).total;
}

}  // namespace top
