// top_kernels_numeric.cu -- the NumericSolve branch of Algorithm 1 (Eq. 15-17; Alg. 1 lines 6-7; L303).
//
// The linear sets keep their slack form; the quadratic sets (velocity / acceleration balls) are the "general convex
// inequality constraints" g0_j(c) = ||A_j c||^2 - bound^2 <= 0, replaced by g_j(c) = max{0, g0_j(c)}^2 = 0 (Eq. 15) with one
// scaled multiplier w_j each, and the x-update minimises the augmented Lagrangian (Eq. 17 on top of Eq. 5 and the slack penalty)
//     F(c) = c'Q~c + rho/2 ||M~c - z~ + u||^2 + rho/2 ||Ao c + s - b + v||^2 + rho/2 sum_j (g_j(c) + w_j)^2
// with L-BFGS (memory 6; initial inverse Hessian = the closed-form operator Pm of the quadratic part, which is exact while no
// ball is violated; Armijo backtracking), started at c^k; then w_j <- w_j + g_j(c^{k+1}).
// One sweep = two launches: numeric_xupdate_kernel (segment local: x-update, boundary rows, slack projection, multipliers)
// and numeric_consensus_kernel (z-update, u-update, residual partial sums; reads the neighbours' boundary rows).  The state
// lives in device memory in the per-lane layout of the other kernels and in the same normalised-time basis / segment-local
// frames, so top_get_coeffs / top_get_state / the init and operator kernels are shared.  Eight lanes per segment, all
// L-BFGS vectors in registers; the branch is an inner ITERATION whose length differs from segment to segment (the paper
// measures it 13x slower than the closed form).
// Product code: shares nothing with oracle/.
#include "top_device.cuh"

namespace top {

namespace {

constexpr int LB_MEM = 6;          // L-BFGS memory
constexpr int LB_MAXIT = 50;       // inner iterations per x-update
constexpr double LB_TOL = 1e-10;   // stop: step below this fraction of the coefficients (metres)
constexpr double LB_C1 = 1e-4;     // Armijo

struct NumTables {                 // constant rows in normalised time, built once per block in shared memory
    double Q1[MAXN][MAXN];         // int_0^1 beta^(s) beta^(s)'
    double Mh[MAXN][MAXN];         // consensus rows: orders 0..s-1 at tau = 0, then at tau = 1
    double E[3][MS][MAXN];         // sample rows of position / velocity / acceleration at tau_j = j/(Ms+1)
};

__device__ void build_tables(NumTables& t, int s) {
    const int n = 2 * s;
    for (int i = threadIdx.x; i < MAXN * MAXN; i += blockDim.x) {
        const int j = i / MAXN, l = i % MAXN;
        double q = 0.0, mh = 0.0;
        if (j >= s && l >= s && j < n && l < n) {
            double fj = 1.0, fl = 1.0;
            for (int k = 0; k < s; ++k) { fj *= (double)(j - k); fl *= (double)(l - k); }
            q = fj * fl / (double)(j + l - 2 * s + 1);
        }
        if (j < n && l < n) mh = beta_entry(j % s, l, j < s ? 0.0 : 1.0);
        t.Q1[j][l] = q; t.Mh[j][l] = mh;
        for (int k = 0; k < 3; ++k) t.E[k][j][l] = l < n ? beta_entry(k, l, (double)(j + 1) / (double)(MS + 1)) : 0.0;
    }
}

// ---- x-update of one segment by L-BFGS (Nocedal & Wright, Numerical Optimization, Alg. 7.4 / 7.5), then everything of the
// sweep that is local to the segment: boundary rows B = M c, slack projection of the box, multipliers of Eq. 17.
// ================================================================================================ 8 lanes per segment
// The x-update kernel proper.  Lane l of a segment owns coefficient row l (three dims) of every L-BFGS vector, consensus
// row l and inequality sample l -- the lane <-> item map of cadmm_sweeps_kernel.  Everything is in registers; the lanes of a
// segment talk through warp shuffles restricted to their own 8-lane group (the four segments of a warp run different
// numbers of inner iterations).  All decisions are taken from values that are bitwise identical in the 8 lanes.

struct LaneCtx {
    unsigned mask;                 // the 8 lanes of this segment
    int lane, base_lane, n, s;
    double rho, wq, it_row, invT, invT2, vmax2, amax2;
    bool has_box, has_vel, has_acc, hard, is_row;
    double zmu[3];                 // z~ - u of consensus row `lane`
    double bhi[3], blo[3];         // hi - |q+|, lo + |q-| of sample `lane`
    double wv, wa;                 // multipliers of sample `lane`
};

__device__ __forceinline__ double grp_sum(const LaneCtx& k, double v) {          // all-reduce over the 8 lanes (same bits everywhere)
    v += __shfl_xor_sync(k.mask, v, 1);
    v += __shfl_xor_sync(k.mask, v, 2);
    v += __shfl_xor_sync(k.mask, v, 4);
    return v;
}
__device__ __forceinline__ double grp_dot(const LaneCtx& k, const double (&a)[3], const double (&b)[3]) {
    return grp_sum(k, a[0] * b[0] + a[1] * b[1] + a[2] * b[2]);
}

// Everything F needs from a coefficient vector is LINEAR in it: the lane's row of Q(1)c, its consensus row of M^c and its
// sample of E0 c, E1 c / T, E2 c / T^2.  So along a search ray x + t d these values are vals(x) + t vals(d): a line-search
// trial costs a few FMAs and one 8-lane sum instead of an all-gather and five row products.
struct LaneVals { double qc[3], b[3], P[3], V[3], A[3]; };

__device__ __forceinline__ LaneVals lane_map(const NumTables& t, const LaneCtx& k, const double (&c)[3]) {
    double call[MAXN][3];
#pragma unroll
    for (int a = 0; a < MAXN; ++a)
#pragma unroll
        for (int d = 0; d < 3; ++d) call[a][d] = __shfl_sync(k.mask, c[d], k.base_lane + a);
    const int l = k.lane;
    LaneVals v;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double qc = 0.0, b = 0.0, P = 0.0, V = 0.0, A = 0.0;
#pragma unroll
        for (int a = 0; a < MAXN; ++a) {
            qc += t.Q1[l][a] * call[a][d]; b += t.Mh[l][a] * call[a][d];
            P += t.E[0][l][a] * call[a][d]; V += t.E[1][l][a] * call[a][d]; A += t.E[2][l][a] * call[a][d];
        }
        v.qc[d] = qc; v.b[d] = b * k.it_row; v.P[d] = P; v.V[d] = V * k.invT; v.A[d] = A * k.invT2;
    }
    return v;
}
__device__ __forceinline__ LaneVals vals_axpy(const LaneVals& x, double t, const LaneVals& d) {
    LaneVals r;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        r.qc[i] = x.qc[i] + t * d.qc[i]; r.b[i] = x.b[i] + t * d.b[i]; r.P[i] = x.P[i] + t * d.P[i];
        r.V[i] = x.V[i] + t * d.V[i]; r.A[i] = x.A[i] + t * d.A[i];
    }
    return r;
}

// F (Eq. 5 + slack penalty + Eq. 15/17), the same value in every lane of the segment; c = the lane's row of the coefficients
__device__ __forceinline__ double lane_F(const LaneCtx& k, const LaneVals& v, const double (&c)[3]) {
    double Fp = 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        Fp += k.wq * c[d] * v.qc[d];                                    // c'Q~c
        if (k.is_row) { const double e = v.b[d] - k.zmu[d]; Fp += 0.5 * k.rho * e * e; }
        if (k.has_box) { const double ep = v.P[d] - k.bhi[d], en = k.blo[d] - v.P[d]; Fp += 0.5 * k.rho * (ep * ep + en * en); }
    }
    if (k.has_vel) {
        const double g0 = v.V[0] * v.V[0] + v.V[1] * v.V[1] + v.V[2] * v.V[2] - k.vmax2, gp = g0 > 0.0 ? g0 : 0.0;
        Fp += 0.5 * k.rho * (gp * gp + k.wv) * (gp * gp + k.wv);
    }
    if (k.has_acc) {
        const double g0 = v.A[0] * v.A[0] + v.A[1] * v.A[1] + v.A[2] * v.A[2] - k.amax2, gp = g0 > 0.0 ? g0 : 0.0;
        Fp += 0.5 * k.rho * (gp * gp + k.wa) * (gp * gp + k.wa);
    }
    return grp_sum(k, Fp);
}

// the lane's row of the gradient of F: 2 T^(1-2s) Q(1)c + M^'we + E0'wb + E1'wv + E2'wa, tangent-projected in HARD mode
__device__ __forceinline__ void lane_grad(const NumTables& t, const LaneCtx& k, const LaneVals& v, double (&g)[3]) {
    const int l = k.lane;
    double we[3], wb[3], wv[3], wa[3];
    double kv = 0.0, ka = 0.0;
    if (k.has_vel) {
        const double g0 = v.V[0] * v.V[0] + v.V[1] * v.V[1] + v.V[2] * v.V[2] - k.vmax2, gp = g0 > 0.0 ? g0 : 0.0;
        kv = k.rho * (gp * gp + k.wv) * 2.0 * gp * 2.0 * k.invT;
    }
    if (k.has_acc) {
        const double g0 = v.A[0] * v.A[0] + v.A[1] * v.A[1] + v.A[2] * v.A[2] - k.amax2, gp = g0 > 0.0 ? g0 : 0.0;
        ka = k.rho * (gp * gp + k.wa) * 2.0 * gp * 2.0 * k.invT2;
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        g[d] = 2.0 * k.wq * v.qc[d];
        we[d] = k.is_row ? k.rho * k.it_row * (v.b[d] - k.zmu[d]) : 0.0;
        wb[d] = k.has_box ? k.rho * ((v.P[d] - k.bhi[d]) - (k.blo[d] - v.P[d])) : 0.0;
        wv[d] = kv * v.V[d]; wa[d] = ka * v.A[d];
    }
#pragma unroll
    for (int q = 0; q < MAXN; ++q) {      // the weights of every lane, times column l of the constant rows
        const double m = t.Mh[q][l], e0 = t.E[0][q][l], e1 = t.E[1][q][l], e2 = t.E[2][q][l];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double acc = m * __shfl_sync(k.mask, we[d], k.base_lane + q);
            if (k.has_box) acc += e0 * __shfl_sync(k.mask, wb[d], k.base_lane + q);
            if (k.has_vel) acc += e1 * __shfl_sync(k.mask, wv[d], k.base_lane + q);
            if (k.has_acc) acc += e2 * __shfl_sync(k.mask, wa[d], k.base_lane + q);
            g[d] += acc;
        }
    }
    if (k.hard) {       // remove the components along the two waypoint rows e_0 and (1,..,1) of every dimension: the L-BFGS
                        // iteration then stays in their null space up to rounding that nothing amplifies
        const double det = (double)(k.n - 1);
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const double b0 = __shfl_sync(k.mask, g[d], k.base_lane), b1 = grp_sum(k, g[d]);
            const double l0 = ((double)k.n * b0 - b1) / det, l1 = (b1 - b0) / det;
            if (l < k.n) g[d] -= l1;
            if (l == 0) g[d] -= l0;
        }
    }
}

__global__ void __launch_bounds__(128, 3) numeric_xupdate_kernel(const NumParams p) {
    __shared__ NumTables tab;
    build_tables(tab, p.s);
    __syncthreads();
    // Persistent 8-lane groups over a work queue: the inner iteration runs 1..50 times depending on the segment, so every
    // group fetches its next segment when it is done instead of idling until the slowest segment of a CTA wave finishes
    // (the shuffle masks are per group: the four groups of a warp loop independently).
    LaneCtx k;
    k.lane = threadIdx.x & 7; k.base_lane = (threadIdx.x & 31) & ~7; k.mask = 0xffu << k.base_lane;
    const int l = k.lane;
    const long long LS = p.stride, NP = p.nseg_pad;
    for (;;) {
        unsigned int gq = 0;
        if (l == 0) gq = atomicAdd(p.work_counter, 1u);
        const long long g = (long long)__shfl_sync(k.mask, gq, k.base_lane);
        if (g >= p.nseg) break;
        const long long base = g * LANES;
        k.s = p.s; k.n = 2 * p.s; k.rho = p.rho; k.hard = p.hard != 0;
        k.has_box = (p.flags & KF_BOX) != 0; k.has_vel = (p.flags & KF_VEL) != 0; k.has_acc = (p.flags & KF_ACC) != 0;
        k.invT = p.invT[g]; k.invT2 = p.invT[NP + g];
        const double invTk[4] = {1.0, k.invT, k.invT2, k.invT2 * k.invT};
        k.is_row = l < 2 * p.s; k.it_row = invTk[l % p.s];
        k.wq = 1.0;
        for (int q = 0; q < 2 * p.s - 1; ++q) k.wq *= k.invT;
        k.vmax2 = p.vmax * p.vmax; k.amax2 = p.amax * p.amax;
        const int n = k.n;
        double lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0}, x[3], org[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            k.zmu[d] = p.zt[d * LS + base + l] - p.u[d * LS + base + l];
            k.bhi[d] = k.blo[d] = 0.0;
            if (k.has_box) {
                lo[d] = p.lohi[d * NP + g]; hi[d] = p.lohi[(3 + d) * NP + g];
                k.bhi[d] = hi[d] - fabs(p.qp[d * LS + base + l]); k.blo[d] = lo[d] + fabs(p.qn[d * LS + base + l]);
            }
            x[d] = l < n ? p.chat[d * LS + base + l] : 0.0;
            org[d] = p.origin[d * NP + g];
        }
        k.wv = k.has_vel ? p.yv[base + l] : 0.0; k.wa = k.has_acc ? p.ya[base + l] : 0.0;
        double Pm_row[MAXN];                                   // row l of H0 = Pm^ (the array holds rho * Pm^)
#pragma unroll
        for (int b = 0; b < MAXN; ++b) Pm_row[b] = p.Pm[b * LS + base + l] / p.rho;

        double S[LB_MEM][3], Y[LB_MEM][3], rhoi[LB_MEM], alpha[LB_MEM];
        double gr[3], gn[3], xn[3], dir[3];
        int hist = 0, it = 0;
        LaneVals vx = lane_map(tab, k, x);
        double F = lane_F(k, vx, x);
        lane_grad(tab, k, vx, gr);
        for (; it < LB_MAXIT; ++it) {
            double qv[3] = {gr[0], gr[1], gr[2]};                                // two-loop recursion
#pragma unroll
            for (int h = LB_MEM - 1; h >= 0; --h)
                if (h < hist) {
                    alpha[h] = rhoi[h] * grp_dot(k, S[h], qv);
#pragma unroll
                    for (int d = 0; d < 3; ++d) qv[d] -= alpha[h] * Y[h][d];
                }
#pragma unroll
            for (int d = 0; d < 3; ++d) {                                        // r = H0 q: row l needs every row of q
                double acc = 0.0;
#pragma unroll
                for (int b = 0; b < MAXN; ++b) acc += Pm_row[b] * __shfl_sync(k.mask, qv[d], k.base_lane + b);
                dir[d] = acc;
            }
#pragma unroll
            for (int h = 0; h < LB_MEM; ++h)
                if (h < hist) {
                    const double beta = rhoi[h] * grp_dot(k, Y[h], dir);
#pragma unroll
                    for (int d = 0; d < 3; ++d) dir[d] += S[h][d] * (alpha[h] - beta);
                }
            double dm = 0.0, xm = 0.0;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                dir[d] = -dir[d];
                dm = fmax(dm, fabs(dir[d]));                                     // normalised-time coefficients are metres already
                xm = fmax(xm, fabs(x[d] + (l == 0 ? org[d] : 0.0)));             // (the tolerance is relative to the global-frame size)
            }
            const double slope = grp_dot(k, gr, dir);
#pragma unroll
            for (int m = 1; m < 8; m <<= 1) { dm = fmax(dm, __shfl_xor_sync(k.mask, dm, m)); xm = fmax(xm, __shfl_xor_sync(k.mask, xm, m)); }
            if (!(dm > LB_TOL * xm) || !(slope < 0.0)) break;
            const LaneVals vd = lane_map(tab, k, dir);
            LaneVals vn = vx;
            double t = 1.0, Fn = F;
            bool ok = false;
            for (int ls = 0; ls < 40; ++ls) {                                    // Armijo backtracking along the ray
#pragma unroll
                for (int d = 0; d < 3; ++d) xn[d] = x[d] + t * dir[d];
                vn = vals_axpy(vx, t, vd);
                Fn = lane_F(k, vn, xn);
                if (Fn <= F + LB_C1 * t * slope) { ok = true; break; }
                t *= 0.5;
            }
            if (!ok) break;
            vx = vn;
            lane_grad(tab, k, vx, gn);
            double sv[3], yv[3];
#pragma unroll
            for (int d = 0; d < 3; ++d) { sv[d] = t * dir[d]; yv[d] = gn[d] - gr[d]; }
            const double sy = grp_dot(k, sv, yv);
            if (sy > 0.0) {
                if (hist == LB_MEM) {
#pragma unroll
                    for (int h = 1; h < LB_MEM; ++h) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) { S[h - 1][d] = S[h][d]; Y[h - 1][d] = Y[h][d]; }
                        rhoi[h - 1] = rhoi[h];
                    }
                    hist = LB_MEM - 1;
                }
#pragma unroll
                for (int h = 0; h < LB_MEM; ++h)
                    if (h == hist) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) { S[h][d] = sv[d]; Y[h][d] = yv[d]; }
                        rhoi[h] = 1.0 / sy;
                    }
                ++hist;
            }
#pragma unroll
            for (int d = 0; d < 3; ++d) { x[d] = xn[d]; gr[d] = gn[d]; }
            F = Fn;
            if (!(t * dm > LB_TOL * xm)) { ++it; break; }                        // the step TAKEN is below tolerance: converged
        }
        if (l == 0) atomicAdd(p.inner_iters, (unsigned long long)it);

        // ---- c^{k+1}: coefficients, boundary rows, slack projection of the box (Eq. 10 / 20d-e as a Moreau pair), multipliers
        vx = lane_map(tab, k, x);                              // (recomputed from the final coefficients: no accumulated ray arithmetic in the state)
        double n2v = 0.0, n2a = 0.0;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            if (l < n) p.chat[d * LS + base + l] = x[d];
            if (k.is_row) p.bnd[d * LS + base + l] = vx.b[d];
            if (k.has_box) {                                  // q = -(A c - b + v_old): s = max(0,q), v_new = max(0,-q)
                const double qp0 = p.qp[d * LS + base + l], qn0 = p.qn[d * LS + base + l];
                p.qp[d * LS + base + l] = (hi[d] - vx.P[d]) - fmax(-qp0, 0.0);
                p.qn[d * LS + base + l] = (vx.P[d] - lo[d]) - fmax(-qn0, 0.0);
            }
            n2v += vx.V[d] * vx.V[d]; n2a += vx.A[d] * vx.A[d];
        }
        if (k.has_vel) { const double g0 = n2v - k.vmax2, gp = g0 > 0.0 ? g0 : 0.0; p.yv[base + l] = k.wv + gp * gp; }
        if (k.has_acc) { const double g0 = n2a - k.amax2, gp = g0 > 0.0 ? g0 : 0.0; p.ya[base + l] = k.wa + gp * gp; }
    }
}

// ---- consensus z-update (Eq. 6b / 20b), scaled dual (Eq. 6c / 20c), residual partial sums (Eq. 21-22; readings A7, A8):
// one thread per segment, reading the neighbours' boundary rows written by numeric_xupdate_kernel
__global__ void __launch_bounds__(128) numeric_consensus_kernel(const NumParams p) {
    __shared__ double Mh[MAXN][MAXN];
    for (int i = threadIdx.x; i < MAXN * MAXN; i += blockDim.x) {
        const int r = i / MAXN, a = i % MAXN;
        Mh[r][a] = (r < 2 * p.s && a < 2 * p.s) ? beta_entry(r % p.s, a, r < p.s ? 0.0 : 1.0) : 0.0;
    }
    __syncthreads();
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g == 0) *p.work_counter = 0u;                    // the x-update kernel of the next sweep starts its queue at segment 0
    if (g >= p.nseg) return;
    const long long LS = p.stride, NP = p.nseg_pad, base = g * LANES;
    const int s = p.s, n = 2 * s;
    const uint8_t sf = p.segflags[g];
    const bool pin_pos = p.flags & KF_PIN_POS;
    const double invT = p.invT[g], invT2 = p.invT[NP + g];
    const double invTk[4] = {1.0, invT, invT2, invT2 * invT};
    double rp2 = 0.0, gap2 = 0.0, rd2 = 0.0, rdn2 = 0.0;
    double dz[MAXN][3];
    for (int r = 0; r < n; ++r) {
        const bool right = r >= s;
        const int kord = r % s;
        const bool fixed = (right ? (sf & SEG_LAST) : (sf & SEG_FIRST)) || (pin_pos && kord == 0);
        const bool has_nb = right ? !(sf & SEG_LAST) : !(sf & SEG_FIRST);
        for (int d = 0; d < 3; ++d) {
            const double own = p.bnd[d * LS + base + r];
            double nb = 0.0;
            if (has_nb) {
                nb = right ? p.bnd[d * LS + base + LANES + kord] : p.bnd[d * LS + base - LANES + s + kord];
                if (kord == 0) nb += p.zoff[d * LS + base + r];           // position rows live in segment-local frames
            }
            const double zold = p.zt[d * LS + base + r];
            const double znew = fixed ? zold : 0.5 * (own + nb);
            const double res = own - znew;
            p.zt[d * LS + base + r] = znew;
            p.u[d * LS + base + r] += res;
            dz[r][d] = znew - zold;
            rp2 += res * res;
            if (right && has_nb) gap2 += (own - nb) * (own - nb);
        }
    }
    for (int a = 0; a < n; ++a) {                                         // rho M(T)'(z~^{k+1} - z~^k), Eq. 22
        const double Tp = p.Tpow[base + a];
        for (int d = 0; d < 3; ++d) {
            double xr = 0.0;
            for (int r = 0; r < n; ++r) xr += Mh[r][a] * dz[r][d] * invTk[r % s];
            xr *= p.rho;
            rdn2 += xr * xr;
            rd2 += (xr * Tp) * (xr * Tp);
        }
    }
    double* o = p.part + g * 4;
    o[0] = rp2; o[1] = rd2; o[2] = rdn2; o[3] = gap2;
}

}  // namespace

cudaError_t launch_numeric_sweep(const NumParams& p, cudaStream_t st) {
    if (p.nseg == 0) return cudaSuccess;
    const long long want = (p.nseg * LANES + 127) / 128;
    numeric_xupdate_kernel<<<(int)(want < p.max_blocks ? want : p.max_blocks), 128, 0, st>>>(p);
    numeric_consensus_kernel<<<(int)((p.nseg + 127) / 128), 128, 0, st>>>(p);
    return cudaGetLastError();
}

}  // namespace top
