/*
 * top_oracle.c -- plain, slow, obviously-correct CPU oracle of the CADMM sweep of
 * TOP (arXiv 2507.10290).  TEST INFRASTRUCTURE ONLY: nothing in the product path
 * (paper_2507_10290_b200/, the C ABI in include/top.h) includes, links or calls
 * this file; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may.  It shares no code, header, table or constant
 * generator with the CUDA path.
 *
 * What it computes: Algorithm 1 of the paper, closed-form
 * branch, one sweep k -> k+1 written in the paper's order and notation, raw
 * monomial basis in physical time, global frame (Eq. 18):
 *
 *   c_i   <- [2Q + rho(M'M + Ao'Ao + sum Av'Av)]^-1 rho[M'(z~-u) + Ao'(b-s-v) + sum Av'(phi-w)]
 *                                                   (Eq. 20a; rho on the RHS: reading A3)
 *   phi,w <- projection onto the ball and its dual   (Eq. 14/20f/20g)
 *   z_j   <- average of the two adjacent boundary-derivative vectors (Eq. 6b/20b)
 *   r_p, r_d                                         (Eq. 21-22; readings A7, A8)
 *   s     <- max(0, -(Ao c - b + v))                 (Eq. 10/20d)
 *   u,v   <- scaled dual updates                     (Eq. 6c/20c/20e)
 *
 * Readings of the paper taken here:
 *   A1  consensus carries derivative orders 0..n_c-1 at each boundary.  Default n_c = s (M is 2s x 2s).  The paper's
 *       literal choice (M(t) has rows beta^0..beta^(d-1), d = 2p-1; L257 "overdetermined", m x 2d
 *       continuity constraints on m(d+1) unknowns) is n_c = 2s-1 ("wide" consensus): M is 2(2s-1) x 2s.  z_0 and z_N
 *       are "initialized by sigma_0 and sigma_N" (L141), which carry orders 0..s-1 only (Eq. 2c: the boundary
 *       conditions go to order p-1, L261), so with n_c = 2s-1 the rows of orders s..2s-2 at the two trajectory ENDS do
 *       not exist: they are left out of M for the first / last segment (rowmask), nothing is fixed there.  Fixing them
 *       (e.g. at 0) would be a different problem from the one the paper's Optimality Conditions (L259-264) describe.
 *   A2  waypoint mode: HARD (default; sigma_i(0)=p_{i-1}, sigma_i(T_i)=p_i imposed as
 *       equalities inside each segment QP: Pm = H^-1 - K Ew H^-1, c0 = K [p_{i-1};p_i],
 *       K = H^-1 Ew'(Ew H^-1 Ew')^-1), PINNED_Z (Eq. 20a verbatim, position row of z_j held
 *       at p_j), FREE (paper's Alg. 1 verbatim, positions averaged too).
 *   A3  H c = rho * rhs.      A5  u is the scaled dual (never multiplied by rho).
 *   A7  r_p = || stack_i (M c_i - z~_i) ||_2 over ALL rows; Eq. 21 verbatim (junction gaps) is
 *       reported beside it.
 *   A8  r_d = rho || stack_i M(T_i)'(z~_i^{k+1} - z~_i^k) ||_2 in monomial physical-time
 *       coefficient space; the normalised variant divides component j by T_i^j.
 *   A9  Init: chord at constant speed; z0_j = (p_j, mean of adjacent chord velocities, 0..);
 *       duals 0; S = max(0,.) of the chord samples; Phi = projection of the chord velocity.
 *   A10 sample times t_ij = T_i * j/(Ms+1), j = 1..Ms.
 *   A11 box corridor: Ao = [E0; -E0] per axis, b = [hi; -lo].
 *   A11p general polytope corridor (Eq. 7-10): K half-spaces a_k'p <= b_k per
 *       segment, applied to the position at each of the Ms sample times: row (j,k) of Ao is
 *       kron(beta_0(t_ij)', a_k') (Ao is MK x m(d+1) as printed), one slack and one scaled dual per (sample, plane).
 *       The flat dimensions are then coupled: H is (n m) x (n m) and is formed and inverted as such (no
 *       per-dimension shortcut in the oracle).
 *   A20 NumericSolve (Eq. 15-17; Alg. 1 lines 6-7 "c, w <- NumericSolve(c, z, u, s, v, w)"; L303): the
 *       alternative x-update for "general convex inequality constraints".  Taken here: the LINEAR sets (box corridor) keep
 *       their slack form -- s and v are still arguments of NumericSolve and ProjectNonNeg / UpdateDual follow unchanged --
 *       and the QUADRATIC sets (velocity / acceleration balls) are the general constraints g0_j(c) = ||A(T_ij) c||^2 - bound^2
 *       <= 0, one per sample and ball, replaced by the equality g_j(c) = max{0, g0_j(c)}^2 = 0 (Eq. 15) with one multiplier
 *       each.  The x-update minimises the augmented Lagrangian (Eq. 17 on top of Eq. 5 and the slack penalty, scaled
 *       multiplier w_j = y_j / rho):
 *           F(c) = c'Q~c + rho/2 ||M~c - z~ + u||^2 + rho/2 ||Ao c + s - b + v||^2 + rho/2 sum_j (g_j(c) + w_j)^2   (+ const)
 *       with L-BFGS [21] started at c^k, and the multiplier follows "similarly to Eq. 6c": w_j <- w_j + g_j(c^{k+1}).
 *       The paper gives no L-BFGS parameters; taken: memory 6; initial inverse Hessian H0 = the closed-form operator of the
 *       quadratic part of F (Pm of reading A2 built WITHOUT the ball terms: exact when no ball is violated, and it keeps
 *       the iterates on the waypoint equalities in HARD mode, where the gradient is also projected onto the null space of
 *       the two waypoint rows so that the whole iteration lives in that subspace); Armijo backtracking (1e-4, halving from
 *       step 1); curvature pairs with s'y <= 0 are skipped; stop when the step (proposed, or taken after back-tracking) is below tol (default 1e-10)
 *       relative to the coefficients (in metres: component a times T^a), when the line search cannot decrease F any more,
 *       or after max_inner (default 50) iterations.  Pins: tests/test_oracle_numeric.py.
 *   A15 ball projection scale = min(1, bound/||y||), ||y|| = 0 -> scale 1.
 *   A18 a single rho for every penalty.   A19 cost c'Qc without 1/2  =>  2Q in H.
 *
 * Precision: the sweep is fp64 (real_t = double).  The one-off per-segment operator
 * (H, its inverse, K, Pm, c0) is formed and inverted in long double with Jacobi
 * equilibration and then rounded to real_t, so that the oracle's own conditioning
 * error (cond(H) up to 1e13 in the raw basis) does not consume the
 * 1e-9 parity budget.  Building with -DORACLE_LONG_DOUBLE makes the sweep long double
 * too (used by a test that bounds the fp64 oracle's own rounding error).
 *
 * Parity pins: tests/test_oracle_pins.py (closed forms, dense KKT, banded solve, SLSQP,
 * KKT certificate, per-iterate invariants); tests/test_oracle_residual_pins.py (r_p, r_d, r_d_norm,
 * r_p_gap recomputed from the iterates with numpy's polynomial calculus, Eq. 21-22, and shown to
 * catch a dropped rho / M for M' / a wrong power of T).  Finite-iteration iterates themselves depend on
 * readings A2/A9: PARITY UNPINNED for those (GPU-vs-oracle only), as DESIGN.md states.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifdef ORACLE_LONG_DOUBLE
typedef long double real_t;
#define R_SQRT sqrtl
#else
typedef double real_t;
#define R_SQRT sqrt
#endif
typedef long double pre_t; /* precision of the one-off operator precompute */

#define NMAX 8   /* n = 2s <= 8 */
#define RMAX 14  /* consensus rows per segment 2 n_c <= 2(2s-1) = 14 */
#define MODE_HARD 0
#define MODE_PINNED_Z 1
#define MODE_FREE 2

typedef struct {
    int N, s, n, m, Ms, mode;
    int nc;         /* consensus derivative orders per boundary: s (default) or 2s-1 (reading A1) */
    int has_box, has_vel, has_acc;
    real_t rho, vmax, amax;
    real_t *T;      /* [N] */
    real_t *p;      /* [N+1][m] waypoints */
    real_t *lo, *hi;/* [N][m] */
    /* per-segment matrices (Eq. 19 / L231) */
    real_t *Q;      /* [N][n][n]   */
    real_t *M;      /* [N][2nc][n]: rows beta_0(0)..beta_{nc-1}(0), beta_0(T)..beta_{nc-1}(T) */
    real_t *rowmask;/* [N][2nc]: 1 = the row takes part in the consensus, 0 = it does not exist (A1: ends, orders >= s) */
    real_t *E0, *E1, *E2; /* [N][Ms][n] : rows beta_k(t_ij) */
    real_t *Pm;     /* [N][n][n]   */
    real_t *c0;     /* [N][n][m]   */
    /* state */
    real_t *C;      /* [N][n][m]   */
    real_t *z, *zprev; /* [N+1][nc][m] */
    real_t *u;      /* [N][2nc][m]  */
    real_t *Sp, *Sn, *Vp, *Vn;   /* [N][Ms][m] slack / dual of the box, + and - side */
    real_t *PhiV, *WV, *PhiA, *WA; /* [N][Ms][m] */
    /* general polytope corridor (reading A11p): K planes per segment, coupled (n m) x (n m) operator */
    int K, has_poly;
    real_t *planes; /* [N][K][m+1]: normal a_k (m), offset b_k */
    real_t *PmF;    /* [N][nm][nm]  coupled operator, coefficient index a*m + d */
    real_t *c0F;    /* [N][nm]      */
    real_t *Spl, *Vpl; /* [N][Ms][K] slack / scaled dual per (sample, plane) */
    real_t *part;   /* [N][4] residual partial sums */
    /* NumericSolve branch (reading A20) */
    int numeric, lbfgs_m, lbfgs_maxit;
    double lbfgs_tol;
    real_t *Yv, *Ya;   /* [N][Ms] scaled multipliers w_j of Eq. 17, velocity / acceleration ball */
    int64_t inner_iters;   /* L-BFGS iterations so far, all segments */
    double rp, rd, rd_norm, rp_gap;
    int64_t iter;
} oracle_t;

/* [beta_k(t)]_j = j!/(j-k)! t^(j-k) for j >= k, else 0          (Eq. 18 differentiated) */
static void beta_row(int n, int k, pre_t t, pre_t *row) {
    for (int j = 0; j < n; ++j) {
        if (j < k) { row[j] = 0; continue; }
        pre_t f = 1;
        for (int q = 0; q < k; ++q) f *= (pre_t)(j - q);
        pre_t pw = 1;
        for (int q = 0; q < j - k; ++q) pw *= t;
        row[j] = f * pw;
    }
}

/* Q(T) = int_0^T beta^(s) beta^(s)' dt
 * Q_jl = j!/(j-s)! l!/(l-s)! T^(j+l-2s+1)/(j+l-2s+1), j,l >= s */
static void build_Q(int n, int s, pre_t T, pre_t *Q) {
    for (int j = 0; j < n; ++j)
        for (int l = 0; l < n; ++l) {
            if (j < s || l < s) { Q[j * n + l] = 0; continue; }
            pre_t fj = 1, fl = 1;
            for (int q = 0; q < s; ++q) { fj *= (pre_t)(j - q); fl *= (pre_t)(l - q); }
            int e = j + l - 2 * s + 1;
            pre_t pw = 1;
            for (int q = 0; q < e; ++q) pw *= T;
            Q[j * n + l] = fj * fl * pw / (pre_t)e;
        }
}

/* inverse of an SPD n x n matrix: Jacobi equilibration + Cholesky, all in pre_t. returns 0 on success */
static int spd_inverse(int n, const pre_t *A, pre_t *Ainv) {
    pre_t d[NMAX], L[NMAX * NMAX], X[NMAX * NMAX];
    for (int i = 0; i < n; ++i) {
        if (!(A[i * n + i] > 0)) return -1;
        d[i] = 1 / sqrtl(A[i * n + i]);
    }
    memset(L, 0, sizeof L);
    for (int i = 0; i < n; ++i)
        for (int j = 0; j <= i; ++j) {
            pre_t acc = A[i * n + j] * d[i] * d[j];
            for (int k = 0; k < j; ++k) acc -= L[i * n + k] * L[j * n + k];
            if (i == j) { if (!(acc > 0)) return -1; L[i * n + i] = sqrtl(acc); }
            else L[i * n + j] = acc / L[j * n + j];
        }
    /* solve (L L') X = I column by column */
    for (int c = 0; c < n; ++c) {
        pre_t y[NMAX];
        for (int i = 0; i < n; ++i) {
            pre_t acc = (i == c) ? 1 : 0;
            for (int k = 0; k < i; ++k) acc -= L[i * n + k] * y[k];
            y[i] = acc / L[i * n + i];
        }
        for (int i = n - 1; i >= 0; --i) {
            pre_t acc = y[i];
            for (int k = i + 1; k < n; ++k) acc -= L[k * n + i] * X[k * n + c];
            X[i * n + c] = acc / L[i * n + i];
        }
    }
    for (int i = 0; i < n; ++i)
        for (int j = 0; j < n; ++j) Ainv[i * n + j] = X[i * n + j] * d[i] * d[j];
    return 0;
}

#define FMAX 24  /* n*m <= 8*3 */
/* inverse of an SPD q x q matrix, q <= FMAX: Jacobi equilibration + Cholesky in pre_t. returns 0 on success */
static int spd_inverse_big(int q, const pre_t *A, pre_t *Ainv) {
    static __thread pre_t d[FMAX], L[FMAX * FMAX], X[FMAX * FMAX], y[FMAX];
    for (int i = 0; i < q; ++i) {
        if (!(A[i * q + i] > 0)) return -1;
        d[i] = 1 / sqrtl(A[i * q + i]);
    }
    memset(L, 0, sizeof L);
    for (int i = 0; i < q; ++i)
        for (int j = 0; j <= i; ++j) {
            pre_t acc = A[i * q + j] * d[i] * d[j];
            for (int k = 0; k < j; ++k) acc -= L[i * q + k] * L[j * q + k];
            if (i == j) { if (!(acc > 0)) return -1; L[i * q + i] = sqrtl(acc); }
            else L[i * q + j] = acc / L[j * q + j];
        }
    for (int c = 0; c < q; ++c) {
        for (int i = 0; i < q; ++i) {
            pre_t acc = (i == c) ? 1 : 0;
            for (int k = 0; k < i; ++k) acc -= L[i * q + k] * y[k];
            y[i] = acc / L[i * q + i];
        }
        for (int i = q - 1; i >= 0; --i) {
            pre_t acc = y[i];
            for (int k = i + 1; k < q; ++k) acc -= L[k * q + i] * X[k * q + c];
            X[i * q + c] = acc / L[i * q + i];
        }
    }
    for (int i = 0; i < q; ++i)
        for (int j = 0; j < q; ++j) Ainv[i * q + j] = X[i * q + j] * d[i] * d[j];
    return 0;
}

/* ------------------------------------------------------------------ create */

#define ALLOC(ptr, count) do { (ptr) = (real_t *)calloc((size_t)(count) > 0 ? (size_t)(count) : 1, sizeof(real_t)); \
                               if (!(ptr)) { oracle_destroy(o); return NULL; } } while (0)

void oracle_destroy(oracle_t *o) {
    if (!o) return;
    free(o->T); free(o->p); free(o->lo); free(o->hi);
    free(o->Q); free(o->M); free(o->rowmask); free(o->E0); free(o->E1); free(o->E2); free(o->Pm); free(o->c0);
    free(o->C); free(o->z); free(o->zprev); free(o->u);
    free(o->Sp); free(o->Sn); free(o->Vp); free(o->Vn);
    free(o->PhiV); free(o->WV); free(o->PhiA); free(o->WA); free(o->part);
    free(o->planes); free(o->PmF); free(o->c0F); free(o->Spl); free(o->Vpl); free(o->Yv); free(o->Ya);
    free(o);
}

/* project the m-vector y onto ||.|| <= bound (Eq. 14 / 20f; reading A15) */
static void proj_ball(int m, const real_t *y, real_t bound, real_t *phi) {
    real_t n2 = 0;
    for (int d = 0; d < m; ++d) n2 += y[d] * y[d];
    real_t scale = 1;
    if (n2 > bound * bound) scale = bound / R_SQRT(n2);
    for (int d = 0; d < m; ++d) phi[d] = scale * y[d];
}

/* per-segment operator Pm, c0 (reading A2) in long double, rounded to real_t */
static int build_operator(oracle_t *o, int i) {
    const int n = o->n, s = o->s, Ms = o->Ms, m = o->m;
    const pre_t T = (pre_t)o->T[i], rho = (pre_t)o->rho;
    pre_t Q[NMAX * NMAX], H[NMAX * NMAX], Hinv[NMAX * NMAX], row[NMAX];
    build_Q(n, s, T, Q);
    for (int a = 0; a < n * n; ++a) { o->Q[(size_t)i * n * n + a] = (real_t)Q[a]; H[a] = 2 * Q[a]; }
    /* M(T): rows beta_0(0)..beta_{nc-1}(0), beta_0(T)..beta_{nc-1}(T); rows that do not exist
     * (rowmask 0, reading A1) are stored but take no part in H */
    const int nc = o->nc;
    for (int r = 0; r < 2 * nc; ++r) {
        beta_row(n, r % nc, r < nc ? (pre_t)0 : T, row);
        for (int j = 0; j < n; ++j) o->M[((size_t)i * 2 * nc + r) * n + j] = (real_t)row[j];
        if (o->rowmask[(size_t)i * 2 * nc + r] == 0) continue;
        for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) H[a * n + b] += rho * row[a] * row[b];
    }
    /* sample rows (A10) and their Gram terms: 2 E0'E0 (two box sides, A11), E1'E1, E2'E2 */
    for (int j = 0; j < Ms; ++j) {
        pre_t t = T * (pre_t)(j + 1) / (pre_t)(Ms + 1);
        for (int k = 0; k < 3; ++k) {
            real_t *E = k == 0 ? o->E0 : (k == 1 ? o->E1 : o->E2);
            int on = k == 0 ? o->has_box : (k == 1 ? o->has_vel : o->has_acc);
            if (o->numeric && k > 0) on = 0;      /* A20: the balls are not part of the quadratic model */
            pre_t w = k == 0 ? 2 : 1;
            beta_row(n, k, t, row);
            for (int a = 0; a < n; ++a) E[((size_t)i * Ms + j) * n + a] = (real_t)row[a];
            if (!on) continue;
            for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) H[a * n + b] += rho * w * row[a] * row[b];
        }
    }
    if (spd_inverse(n, H, Hinv)) return -1;
    pre_t Pm[NMAX * NMAX], c0[NMAX * 3];
    memset(c0, 0, sizeof c0);
    if (o->mode == MODE_HARD) {
        /* Ew = [beta_0(0); beta_0(T)],  K = Hinv Ew'(Ew Hinv Ew')^-1,  Pm = Hinv - K Ew Hinv,  c0 = K [p_{i-1}; p_i] */
        pre_t Ew[2 * NMAX], HE[NMAX * 2], S[4], Si[4], K[NMAX * 2];
        beta_row(n, 0, 0, Ew); beta_row(n, 0, T, Ew + n);
        for (int a = 0; a < n; ++a) for (int c = 0; c < 2; ++c) {
            pre_t acc = 0; for (int b = 0; b < n; ++b) acc += Hinv[a * n + b] * Ew[c * n + b];
            HE[a * 2 + c] = acc;
        }
        for (int r = 0; r < 2; ++r) for (int c = 0; c < 2; ++c) {
            pre_t acc = 0; for (int b = 0; b < n; ++b) acc += Ew[r * n + b] * HE[b * 2 + c];
            S[r * 2 + c] = acc;
        }
        pre_t det = S[0] * S[3] - S[1] * S[2];
        if (!(det > 0)) return -1;
        Si[0] = S[3] / det; Si[1] = -S[1] / det; Si[2] = -S[2] / det; Si[3] = S[0] / det;
        for (int a = 0; a < n; ++a) for (int c = 0; c < 2; ++c)
            K[a * 2 + c] = HE[a * 2 + 0] * Si[0 * 2 + c] + HE[a * 2 + 1] * Si[1 * 2 + c];
        for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b)
            Pm[a * n + b] = Hinv[a * n + b] - (K[a * 2 + 0] * HE[b * 2 + 0] + K[a * 2 + 1] * HE[b * 2 + 1]);
        for (int a = 0; a < n; ++a) for (int d = 0; d < m; ++d)
            c0[a * 3 + d] = K[a * 2 + 0] * (pre_t)o->p[(size_t)i * m + d] + K[a * 2 + 1] * (pre_t)o->p[(size_t)(i + 1) * m + d];
    } else {
        memcpy(Pm, Hinv, sizeof(pre_t) * n * n);
    }
    for (int a = 0; a < n * n; ++a) o->Pm[(size_t)i * n * n + a] = (real_t)Pm[a];
    for (int a = 0; a < n; ++a) for (int d = 0; d < m; ++d) o->c0[((size_t)i * n + a) * m + d] = (real_t)c0[a * 3 + d];
    return 0;
}

/* Coupled operator of segment i with a polytope corridor (reading A11p), coefficient index a*m + d:
 *   H = kron(2Q + rho(M'M + E1'E1 + E2'E2), I_m) + rho sum_j sum_k kron(e0_j, a_k) kron(e0_j, a_k)'     (Eq. 20a)
 * HARD mode: the 2m waypoint equalities Ew (x) I_m are imposed inside the QP exactly as in build_operator. */
static int build_operator_poly(oracle_t *o, int i) {
    const int n = o->n, s = o->s, Ms = o->Ms, m = o->m, K = o->K, q = n * m;
    const pre_t T = (pre_t)o->T[i], rho = (pre_t)o->rho;
    static __thread pre_t H[FMAX * FMAX], Hinv[FMAX * FMAX], Pm[FMAX * FMAX], HE[FMAX * 6], Kg[FMAX * 6];
    pre_t Q[NMAX * NMAX], D[NMAX * NMAX], row[NMAX];
    build_Q(n, s, T, Q);
    for (int a = 0; a < n * n; ++a) { o->Q[(size_t)i * n * n + a] = (real_t)Q[a]; D[a] = 2 * Q[a]; }
    const int nc = o->nc;
    for (int r = 0; r < 2 * nc; ++r) {
        beta_row(n, r % nc, r < nc ? (pre_t)0 : T, row);
        for (int j = 0; j < n; ++j) o->M[((size_t)i * 2 * nc + r) * n + j] = (real_t)row[j];
        if (o->rowmask[(size_t)i * 2 * nc + r] == 0) continue;
        for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) D[a * n + b] += rho * row[a] * row[b];
    }
    memset(H, 0, sizeof(pre_t) * q * q);
    for (int j = 0; j < Ms; ++j) {
        pre_t t = T * (pre_t)(j + 1) / (pre_t)(Ms + 1);
        for (int k = 0; k < 3; ++k) {
            real_t *E = k == 0 ? o->E0 : (k == 1 ? o->E1 : o->E2);
            beta_row(n, k, t, row);
            for (int a = 0; a < n; ++a) E[((size_t)i * Ms + j) * n + a] = (real_t)row[a];
            if (k == 0) {
                /* rows kron(e0_j, a_k), k = 1..K */
                for (int kk = 0; kk < K; ++kk) {
                    const real_t *pl = o->planes + ((size_t)i * K + kk) * (m + 1);
                    for (int a = 0; a < n; ++a) for (int d = 0; d < m; ++d)
                        for (int b = 0; b < n; ++b) for (int e = 0; e < m; ++e)
                            H[(a * m + d) * q + (b * m + e)] += rho * (row[a] * (pre_t)pl[d]) * (row[b] * (pre_t)pl[e]);
                }
            } else if (k == 1 ? o->has_vel : o->has_acc) {
                for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) D[a * n + b] += rho * row[a] * row[b];
            }
        }
    }
    for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) for (int d = 0; d < m; ++d) H[(a * m + d) * q + (b * m + d)] += D[a * n + b];
    if (spd_inverse_big(q, H, Hinv)) return -1;
    real_t *PmF = o->PmF + (size_t)i * q * q, *c0F = o->c0F + (size_t)i * q;
    for (int a = 0; a < q; ++a) c0F[a] = 0;
    if (o->mode == MODE_HARD) {
        /* Ewf rows: (beta_0(0) (x) e_d), (beta_0(T) (x) e_d); 2m of them */
        pre_t Ew[2 * NMAX], S[36], Si[36];
        const int w = 2 * m;
        beta_row(n, 0, 0, Ew); beta_row(n, 0, T, Ew + n);
        /* HE = Hinv Ewf'  (q x 2m);  column c = (end e, dim d): Ewf row has Ew[e][b] at index b*m + d */
        for (int a = 0; a < q; ++a) for (int e = 0; e < 2; ++e) for (int d = 0; d < m; ++d) {
            pre_t acc = 0; for (int b = 0; b < n; ++b) acc += Hinv[a * q + b * m + d] * Ew[e * n + b];
            HE[a * w + e * m + d] = acc;
        }
        for (int e = 0; e < 2; ++e) for (int d = 0; d < m; ++d) for (int c = 0; c < w; ++c) {
            pre_t acc = 0; for (int b = 0; b < n; ++b) acc += Ew[e * n + b] * HE[(b * m + d) * w + c];
            S[(e * m + d) * w + c] = acc;
        }
        if (spd_inverse_big(w, S, Si)) return -1;
        for (int a = 0; a < q; ++a) for (int c = 0; c < w; ++c) {
            pre_t acc = 0; for (int r = 0; r < w; ++r) acc += HE[a * w + r] * Si[r * w + c];
            Kg[a * w + c] = acc;
        }
        for (int a = 0; a < q; ++a) for (int b = 0; b < q; ++b) {
            pre_t acc = Hinv[a * q + b];
            for (int c = 0; c < w; ++c) acc -= Kg[a * w + c] * HE[b * w + c];
            Pm[a * q + b] = acc;
        }
        for (int a = 0; a < q; ++a) {
            pre_t acc = 0;
            for (int d = 0; d < m; ++d)
                acc += Kg[a * w + 0 * m + d] * (pre_t)o->p[(size_t)i * m + d] + Kg[a * w + 1 * m + d] * (pre_t)o->p[(size_t)(i + 1) * m + d];
            c0F[a] = (real_t)acc;
        }
    } else {
        memcpy(Pm, Hinv, sizeof(pre_t) * q * q);
    }
    for (int a = 0; a < q * q; ++a) PmF[a] = (real_t)Pm[a];
    return 0;
}

/*
 * All inputs are host fp64.  waypoints [N+1][m]; durations [N]; start/end_derivs [s-1][m] (orders
 * 1..s-1) or NULL = rest; box_lo/hi [N][m] or NULL; vmax/amax <= 0 => off; Ms = samples per segment.
 */
static oracle_t *oracle_create_impl(int N, int s, int m, const double *waypoints, const double *durations,
                        const double *start_derivs, const double *end_derivs, int Ms,
                        const double *box_lo, const double *box_hi, double vmax, double amax,
                        double rho, int mode, int K, const double *planes, int nc) {
    if (N < 1 || (s != 3 && s != 4) || m < 1 || m > 3 || Ms < 0 || !(rho > 0) || mode < 0 || mode > 2) return NULL;
    if (nc != s && nc != 2 * s - 1) return NULL;
    if (K < 0 || (K > 0 && (!planes || Ms <= 0 || box_lo || box_hi))) return NULL;   /* a polytope replaces the box */
    oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
    if (!o) return NULL;
    const int n = 2 * s;
    o->N = N; o->s = s; o->n = n; o->m = m; o->Ms = Ms; o->mode = mode; o->nc = nc;
    o->rho = (real_t)rho; o->vmax = (real_t)vmax; o->amax = (real_t)amax;
    o->has_box = (Ms > 0 && box_lo && box_hi);
    o->has_vel = (Ms > 0 && vmax > 0);
    o->has_acc = (Ms > 0 && amax > 0);
    o->K = K; o->has_poly = K > 0;
    ALLOC(o->planes, (size_t)N * K * (m + 1)); ALLOC(o->PmF, o->has_poly ? (size_t)N * n * m * n * m : 0);
    ALLOC(o->c0F, o->has_poly ? (size_t)N * n * m : 0);
    ALLOC(o->Spl, (size_t)N * Ms * K); ALLOC(o->Vpl, (size_t)N * Ms * K);
    for (size_t a = 0; a < (size_t)N * K * (m + 1); ++a) o->planes[a] = (real_t)planes[a];
    ALLOC(o->T, N); ALLOC(o->p, (N + 1) * m); ALLOC(o->lo, N * m); ALLOC(o->hi, N * m);
    ALLOC(o->Q, (size_t)N * n * n); ALLOC(o->M, (size_t)N * 2 * nc * n); ALLOC(o->rowmask, (size_t)N * 2 * nc);
    ALLOC(o->E0, (size_t)N * Ms * n); ALLOC(o->E1, (size_t)N * Ms * n); ALLOC(o->E2, (size_t)N * Ms * n);
    ALLOC(o->Pm, (size_t)N * n * n); ALLOC(o->c0, (size_t)N * n * m);
    ALLOC(o->C, (size_t)N * n * m); ALLOC(o->z, (size_t)(N + 1) * nc * m); ALLOC(o->zprev, (size_t)(N + 1) * nc * m);
    ALLOC(o->u, (size_t)N * 2 * nc * m);
    ALLOC(o->Sp, (size_t)N * Ms * m); ALLOC(o->Sn, (size_t)N * Ms * m);
    ALLOC(o->Vp, (size_t)N * Ms * m); ALLOC(o->Vn, (size_t)N * Ms * m);
    ALLOC(o->PhiV, (size_t)N * Ms * m); ALLOC(o->WV, (size_t)N * Ms * m);
    ALLOC(o->PhiA, (size_t)N * Ms * m); ALLOC(o->WA, (size_t)N * Ms * m);
    ALLOC(o->part, (size_t)N * 4);
    ALLOC(o->Yv, (size_t)N * Ms); ALLOC(o->Ya, (size_t)N * Ms);
    for (int i = 0; i < N; ++i) { if (!(durations[i] > 0)) { oracle_destroy(o); return NULL; } o->T[i] = (real_t)durations[i]; }
    for (int a = 0; a < (N + 1) * m; ++a) o->p[a] = (real_t)waypoints[a];
    if (o->has_box) for (int a = 0; a < N * m; ++a) { o->lo[a] = (real_t)box_lo[a]; o->hi[a] = (real_t)box_hi[a]; }
    /* rows of M that exist (reading A1): all of them, except orders s..nc-1 at the start of the first segment and at the
     * end of the last one (z_0, z_N carry the given end state, orders 0..s-1, L141 / Eq. 2c) */
    for (int i = 0; i < N; ++i)
        for (int r = 0; r < 2 * nc; ++r) {
            const int k = r % nc, at_end = r >= nc;
            const int missing = k >= s && ((i == 0 && !at_end) || (i == N - 1 && at_end));
            o->rowmask[(size_t)i * 2 * nc + r] = missing ? 0 : 1;
        }
    for (int i = 0; i < N; ++i) if (o->has_poly ? build_operator_poly(o, i) : build_operator(o, i)) { oracle_destroy(o); return NULL; }

    /* ---- Init (Alg. 1 line 1; reading A9) ---- */
    for (int i = 0; i < N; ++i) {          /* C0 = chord at constant speed */
        for (int d = 0; d < m; ++d) {
            o->C[((size_t)i * n + 0) * m + d] = o->p[(size_t)i * m + d];
            o->C[((size_t)i * n + 1) * m + d] = (o->p[(size_t)(i + 1) * m + d] - o->p[(size_t)i * m + d]) / o->T[i];
        }
    }
    for (int j = 0; j <= N; ++j)           /* z0_j: position p_j, mean chord velocity, higher orders 0 */
        for (int d = 0; d < m; ++d) {
            o->z[((size_t)j * nc + 0) * m + d] = o->p[(size_t)j * m + d];
            if (j >= 1 && j <= N - 1)
                o->z[((size_t)j * nc + 1) * m + d] = (real_t)0.5 * (o->C[((size_t)(j - 1) * n + 1) * m + d] + o->C[((size_t)j * n + 1) * m + d]);
        }
    for (int k = 1; k < s; ++k)            /* z_0, z_N = given end states (Eq. 2c); rest if NULL */
        for (int d = 0; d < m; ++d) {
            o->z[((size_t)0 * nc + k) * m + d] = start_derivs ? (real_t)start_derivs[(k - 1) * m + d] : 0;
            o->z[((size_t)N * nc + k) * m + d] = end_derivs ? (real_t)end_derivs[(k - 1) * m + d] : 0;
        }
    memcpy(o->zprev, o->z, sizeof(real_t) * (size_t)(N + 1) * nc * m);
    for (int i = 0; i < N; ++i)            /* slacks / phi of the chord samples; all duals 0 */
        for (int j = 0; j < Ms; ++j) {
            real_t P[3] = {0, 0, 0}, V[3] = {0, 0, 0}, A[3] = {0, 0, 0};
            for (int d = 0; d < m; ++d)
                for (int a = 0; a < n; ++a) {
                    real_t c = o->C[((size_t)i * n + a) * m + d];
                    P[d] += o->E0[((size_t)i * Ms + j) * n + a] * c;
                    V[d] += o->E1[((size_t)i * Ms + j) * n + a] * c;
                    A[d] += o->E2[((size_t)i * Ms + j) * n + a] * c;
                }
            size_t q = ((size_t)i * Ms + j) * m;
            if (o->has_box) for (int d = 0; d < m; ++d) {
                real_t a = o->hi[(size_t)i * m + d] - P[d], b = P[d] - o->lo[(size_t)i * m + d];
                o->Sp[q + d] = a > 0 ? a : 0; o->Sn[q + d] = b > 0 ? b : 0;
            }
            if (o->has_vel) proj_ball(m, V, o->vmax, o->PhiV + q);
            if (o->has_acc) proj_ball(m, A, o->amax, o->PhiA + q);
            for (int k = 0; k < K; ++k) {          /* polytope slacks of the chord samples: s = max(0, b - a'p) */
                const real_t *pl = o->planes + ((size_t)i * K + k) * (m + 1);
                real_t val = 0;
                for (int d = 0; d < m; ++d) val += pl[d] * P[d];
                real_t sl = pl[m] - val;
                o->Spl[((size_t)i * Ms + j) * K + k] = sl > 0 ? sl : 0;
            }
        }
    o->iter = 0; o->rp = o->rd = o->rd_norm = o->rp_gap = NAN;
    return o;
}

oracle_t *oracle_create(int N, int s, int m, const double *waypoints, const double *durations,
                        const double *start_derivs, const double *end_derivs, int Ms,
                        const double *box_lo, const double *box_hi, double vmax, double amax,
                        double rho, int mode) {
    return oracle_create_impl(N, s, m, waypoints, durations, start_derivs, end_derivs, Ms, box_lo, box_hi, vmax, amax, rho, mode, 0, NULL, s);
}

/* the general entry: box (K = 0) or polytope corridor (K > 0, box_lo = box_hi = NULL), and the number n_c of consensus
 * derivative orders per boundary: s, or the paper-literal 2s-1 (reading A1) */
oracle_t *oracle_create_ex(int N, int s, int m, const double *waypoints, const double *durations,
                           const double *start_derivs, const double *end_derivs, int Ms,
                           const double *box_lo, const double *box_hi, int K, const double *planes,
                           double vmax, double amax, double rho, int mode, int nc) {
    return oracle_create_impl(N, s, m, waypoints, durations, start_derivs, end_derivs, Ms, box_lo, box_hi, vmax, amax, rho, mode, K, planes, nc);
}

/* the same with a general polytope corridor: planes [N][K][m+1] = (normal a_k, offset b_k), a_k'p <= b_k (A11p) */
oracle_t *oracle_create_poly(int N, int s, int m, const double *waypoints, const double *durations,
                             const double *start_derivs, const double *end_derivs, int Ms, int K, const double *planes,
                             double vmax, double amax, double rho, int mode) {
    return oracle_create_impl(N, s, m, waypoints, durations, start_derivs, end_derivs, Ms, NULL, NULL, vmax, amax, rho, mode, K, planes, s);
}

/* ------------------------------------------------------------------ NumericSolve (reading A20; Eq. 15-17) */

#define NVAR (NMAX * 3)   /* unknowns of one segment: c[a*m + d] */
#define LBFGS_MMAX 8

/* F(c) of segment i (see A20) and, if grad != NULL, its gradient, straight from the definition:
 *   F = sum_d c_d'Q c_d + rho/2 ||M c - z~ + u||^2 (rows that exist) + rho/2 ||Ao c + s - b + v||^2 (box, both sides)
 *       + rho/2 sum_j [ (g^v_j + w^v_j)^2 + (g^a_j + w^a_j)^2 ],   g_j = max(0, ||A_j c||^2 - bound^2)^2        (Eq. 15, 17) */
static real_t numeric_eval(const oracle_t *o, int i, const real_t *c, real_t *grad) {
    const int n = o->n, m = o->m, Ms = o->Ms, nc = o->nc;
    const real_t rho = o->rho;
    real_t F = 0;
    if (grad) for (int a = 0; a < n * m; ++a) grad[a] = 0;
    const real_t *Q = o->Q + (size_t)i * n * n;
    for (int d = 0; d < m; ++d)                       /* c'Q~c (no 1/2: A19) */
        for (int a = 0; a < n; ++a) {
            real_t qc = 0;
            for (int b = 0; b < n; ++b) qc += Q[a * n + b] * c[b * m + d];
            F += c[a * m + d] * qc;
            if (grad) grad[a * m + d] += 2 * qc;
        }
    const real_t *M = o->M + (size_t)i * 2 * nc * n;
    for (int r = 0; r < 2 * nc; ++r) {                /* consensus penalty of Eq. 5 */
        if (o->rowmask[(size_t)i * 2 * nc + r] == 0) continue;
        const real_t *zr = o->z + ((size_t)(i + (r >= nc)) * nc + (r % nc)) * m;
        const real_t *ur = o->u + ((size_t)i * 2 * nc + r) * m;
        for (int d = 0; d < m; ++d) {
            real_t e = -zr[d] + ur[d];
            for (int a = 0; a < n; ++a) e += M[r * n + a] * c[a * m + d];
            F += (rho / 2) * e * e;
            if (grad) for (int a = 0; a < n; ++a) grad[a * m + d] += rho * M[r * n + a] * e;
        }
    }
    for (int j = 0; j < Ms; ++j) {
        const real_t *e0 = o->E0 + ((size_t)i * Ms + j) * n, *e1 = o->E1 + ((size_t)i * Ms + j) * n, *e2 = o->E2 + ((size_t)i * Ms + j) * n;
        size_t q = ((size_t)i * Ms + j) * m;
        if (o->has_box)                                /* slack penalty of the linear set (Eq. 8), + and - side */
            for (int d = 0; d < m; ++d) {
                real_t P = 0;
                for (int a = 0; a < n; ++a) P += e0[a] * c[a * m + d];
                real_t ep = P + o->Sp[q + d] - o->hi[(size_t)i * m + d] + o->Vp[q + d];
                real_t en = -P + o->Sn[q + d] + o->lo[(size_t)i * m + d] + o->Vn[q + d];
                F += (rho / 2) * (ep * ep + en * en);
                if (grad) for (int a = 0; a < n; ++a) grad[a * m + d] += rho * e0[a] * (ep - en);
            }
        for (int kind = 1; kind <= 2; ++kind) {        /* general constraints: Eq. 15 inside Eq. 17 */
            if (kind == 1 ? !o->has_vel : !o->has_acc) continue;
            const real_t *e = kind == 1 ? e1 : e2;
            const real_t bound = kind == 1 ? o->vmax : o->amax;
            const real_t w = (kind == 1 ? o->Yv : o->Ya)[(size_t)i * Ms + j];
            real_t val[3] = {0, 0, 0}, n2 = 0;
            for (int d = 0; d < m; ++d) { for (int a = 0; a < n; ++a) val[d] += e[a] * c[a * m + d]; n2 += val[d] * val[d]; }
            const real_t g0 = n2 - bound * bound, gp = g0 > 0 ? g0 : 0, g = gp * gp;
            F += (rho / 2) * (g + w) * (g + w);
            if (grad && gp > 0) {                      /* d/dc: rho (g + w) * 2 gp * 2 A_j'(A_j c) */
                const real_t k = rho * (g + w) * 2 * gp * 2;
                for (int d = 0; d < m; ++d) for (int a = 0; a < n; ++a) grad[a * m + d] += k * e[a] * val[d];
            }
        }
    }
    return F;
}

/* g_j(c) = max(0, ||A_j c||^2 - bound^2)^2 of sample j (Eq. 15) */
static real_t numeric_g(const oracle_t *o, int i, int j, int kind, const real_t *c) {
    const int n = o->n, m = o->m, Ms = o->Ms;
    const real_t *e = (kind == 1 ? o->E1 : o->E2) + ((size_t)i * Ms + j) * n;
    const real_t bound = kind == 1 ? o->vmax : o->amax;
    real_t n2 = 0;
    for (int d = 0; d < m; ++d) { real_t v = 0; for (int a = 0; a < n; ++a) v += e[a] * c[a * m + d]; n2 += v * v; }
    const real_t g0 = n2 - bound * bound, gp = g0 > 0 ? g0 : 0;
    return gp * gp;
}

/* HARD waypoints: orthogonal projection of a gradient onto the null space of the two waypoint rows Ew = [beta_0(0); beta_0(T)]
 * of every dimension.  The L-BFGS iteration then lives in that subspace: H0 = Pm maps into it, and no rounding residue of
 * the steps can pick up the (large) constraint-normal part of the gradient. */
static void project_tangent(const oracle_t *o, int i, real_t *g) {
    if (o->mode != MODE_HARD) return;
    const int n = o->n, m = o->m;
    real_t r1[NMAX], g11 = 0;
    r1[0] = 1;
    for (int a = 1; a < n; ++a) r1[a] = r1[a - 1] * o->T[i];
    for (int a = 0; a < n; ++a) g11 += r1[a] * r1[a];
    /* Gram of (e_0, r1) = [[1, 1], [1, g11]] */
    const real_t det = g11 - 1;
    for (int d = 0; d < m; ++d) {
        real_t b0 = g[0 * m + d], b1 = 0;
        for (int a = 0; a < n; ++a) b1 += r1[a] * g[a * m + d];
        const real_t l0 = (g11 * b0 - b1) / det, l1 = (b1 - b0) / det;
        g[0 * m + d] -= l0;
        for (int a = 0; a < n; ++a) g[a * m + d] -= l1 * r1[a];
    }
}

/* x-update of segment i by L-BFGS (Nocedal & Wright, Numerical Optimization, Alg. 7.4 / 7.5) from c^k, in place.
 * H0 = Pm per dimension (A20).  Returns the iterations used. */
static int numeric_solve_segment(oracle_t *o, int i) {
    const int n = o->n, m = o->m, nv = n * m, mem = o->lbfgs_m;
    real_t *x = o->C + (size_t)i * nv;
    const real_t *Pm = o->Pm + (size_t)i * n * n;
    real_t g[NVAR], gn[NVAR], xn[NVAR], dir[NVAR], qv[NVAR];
    real_t S[LBFGS_MMAX][NVAR], Y[LBFGS_MMAX][NVAR], rhoi[LBFGS_MMAX], alpha[LBFGS_MMAX];
    int hist = 0, it = 0;
    real_t F = numeric_eval(o, i, x, g);
    project_tangent(o, i, g);
    real_t Tp[NMAX];
    Tp[0] = 1;
    for (int a = 1; a < n; ++a) Tp[a] = Tp[a - 1] * o->T[i];
    for (; it < o->lbfgs_maxit; ++it) {
        for (int a = 0; a < nv; ++a) qv[a] = g[a];                       /* two-loop recursion */
        for (int h = hist - 1; h >= 0; --h) {
            real_t sq = 0;
            for (int a = 0; a < nv; ++a) sq += S[h][a] * qv[a];
            alpha[h] = rhoi[h] * sq;
            for (int a = 0; a < nv; ++a) qv[a] -= alpha[h] * Y[h][a];
        }
        for (int a = 0; a < n; ++a) for (int d = 0; d < m; ++d) {        /* r = H0 q */
            real_t acc = 0;
            for (int b = 0; b < n; ++b) acc += Pm[a * n + b] * qv[b * m + d];
            dir[a * m + d] = acc;
        }
        for (int h = 0; h < hist; ++h) {
            real_t yr = 0;
            for (int a = 0; a < nv; ++a) yr += Y[h][a] * dir[a];
            const real_t beta = rhoi[h] * yr;
            for (int a = 0; a < nv; ++a) dir[a] += S[h][a] * (alpha[h] - beta);
        }
        real_t slope = 0, dmax = 0, xmax = 0;
        for (int a = 0; a < n; ++a) for (int d = 0; d < m; ++d) {
            dir[a * m + d] = -dir[a * m + d];
            slope += g[a * m + d] * dir[a * m + d];
            real_t da = fabsl((long double)(dir[a * m + d] * Tp[a])), xa = fabsl((long double)(x[a * m + d] * Tp[a]));
            if (da > dmax) dmax = da;
            if (xa > xmax) xmax = xa;
        }
        if (!(dmax > (real_t)o->lbfgs_tol * xmax) || !(slope < 0)) break;     /* converged (step below tolerance) */
        real_t t = 1, Fn = F;
        int ok = 0;
        for (int ls = 0; ls < 40; ++ls) {                                   /* Armijo backtracking */
            for (int a = 0; a < nv; ++a) xn[a] = x[a] + t * dir[a];
            Fn = numeric_eval(o, i, xn, NULL);
            if (Fn <= F + (real_t)1e-4 * t * slope) { ok = 1; break; }
            t *= (real_t)0.5;
        }
        if (!ok) break;                                                     /* no decrease possible: rounding floor */
        numeric_eval(o, i, xn, gn);
        project_tangent(o, i, gn);
        real_t sy = 0;
        real_t sv[NVAR], yv[NVAR];
        for (int a = 0; a < nv; ++a) { sv[a] = t * dir[a]; yv[a] = gn[a] - g[a]; sy += sv[a] * yv[a]; }
        if (sy > 0) {                                    /* curvature pair (F is convex: s'y >= 0; = 0 only at the rounding floor) */
            if (hist == mem) {
                for (int h = 1; h < mem; ++h) { memcpy(S[h - 1], S[h], sizeof(real_t) * nv); memcpy(Y[h - 1], Y[h], sizeof(real_t) * nv); rhoi[h - 1] = rhoi[h]; }
                hist = mem - 1;
            }
            memcpy(S[hist], sv, sizeof(real_t) * nv); memcpy(Y[hist], yv, sizeof(real_t) * nv); rhoi[hist] = 1 / sy;
            ++hist;
        }
        for (int a = 0; a < nv; ++a) { x[a] = xn[a]; g[a] = gn[a]; }
        F = Fn;
        if (!(t * dmax > (real_t)o->lbfgs_tol * xmax)) { ++it; break; }      /* the step TAKEN is below tolerance: converged */
    }
    return it;
}

/* ------------------------------------------------------------------ one sweep (Alg. 1 lines 3-13) */

static void sweep_once(oracle_t *o) {
    const int N = o->N, n = o->n, m = o->m, Ms = o->Ms, nc = o->nc;
    const real_t rho = o->rho;

    if (o->numeric) {      /* NumericSolve (Alg. 1 lines 6-7; reading A20) instead of ClosedFormSolve */
        int64_t inner = 0;
#pragma omp parallel for schedule(static) reduction(+ : inner)
        for (int i = 0; i < N; ++i) inner += numeric_solve_segment(o, i);
        o->inner_iters += inner;
    }
    /* ClosedFormSolve: Eq. 20a with rho on the right-hand side (A3) */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        if (o->numeric) continue;
        real_t R[NMAX * 3];
        for (int a = 0; a < n * m; ++a) R[a] = 0;
        const real_t *M = o->M + (size_t)i * 2 * nc * n;
        for (int r = 0; r < 2 * nc; ++r) {         /* M'(z~_i - u_i), z~_i = (z_{i-1}; z_i) */
            if (o->rowmask[(size_t)i * 2 * nc + r] == 0) continue;
            const real_t *zr = o->z + ((size_t)(i + (r >= nc)) * nc + (r % nc)) * m;
            const real_t *ur = o->u + ((size_t)i * 2 * nc + r) * m;
            for (int d = 0; d < m; ++d) {
                real_t g = zr[d] - ur[d];
                for (int a = 0; a < n; ++a) R[a * m + d] += M[r * n + a] * g;
            }
        }
        for (int j = 0; j < Ms; ++j) {
            size_t q = ((size_t)i * Ms + j) * m;
            const real_t *e0 = o->E0 + ((size_t)i * Ms + j) * n;
            const real_t *e1 = o->E1 + ((size_t)i * Ms + j) * n;
            const real_t *e2 = o->E2 + ((size_t)i * Ms + j) * n;
            for (int d = 0; d < m; ++d) {
                if (o->has_box) {                  /* Ao'(b - s - v) with Ao = [E0; -E0], b = [hi; -lo] */
                    real_t gp = o->hi[(size_t)i * m + d] - o->Sp[q + d] - o->Vp[q + d];
                    real_t gn = -o->lo[(size_t)i * m + d] - o->Sn[q + d] - o->Vn[q + d];
                    for (int a = 0; a < n; ++a) R[a * m + d] += e0[a] * gp + (-e0[a]) * gn;
                }
                if (o->has_vel) { real_t g = o->PhiV[q + d] - o->WV[q + d]; for (int a = 0; a < n; ++a) R[a * m + d] += e1[a] * g; }
                if (o->has_acc) { real_t g = o->PhiA[q + d] - o->WA[q + d]; for (int a = 0; a < n; ++a) R[a * m + d] += e2[a] * g; }
            }
            for (int k = 0; k < o->K; ++k) {       /* Ao'(b - s - v), row (j,k) of Ao = kron(e0_j, a_k)   (A11p) */
                const real_t *pl = o->planes + ((size_t)i * o->K + k) * (m + 1);
                size_t qk = ((size_t)i * Ms + j) * o->K + k;
                real_t g = pl[m] - o->Spl[qk] - o->Vpl[qk];
                for (int a = 0; a < n; ++a) for (int d = 0; d < m; ++d) R[a * m + d] += e0[a] * pl[d] * g;
            }
        }
        if (o->has_poly) {                         /* coupled dims: c = PmF (rho R) + c0F over the (n m)-vector */
            const int qd = n * m;
            const real_t *PmF = o->PmF + (size_t)i * qd * qd;
            for (int a = 0; a < qd; ++a) {
                real_t acc = 0;
                for (int b = 0; b < qd; ++b) acc += PmF[a * qd + b] * (rho * R[b]);
                o->C[(size_t)i * qd + a] = acc + o->c0F[(size_t)i * qd + a];
            }
            continue;
        }
        const real_t *Pm = o->Pm + (size_t)i * n * n;
        for (int a = 0; a < n; ++a)
            for (int d = 0; d < m; ++d) {
                real_t acc = 0;
                for (int b = 0; b < n; ++b) acc += Pm[a * n + b] * (rho * R[b * m + d]);
                o->C[((size_t)i * n + a) * m + d] = acc + o->c0[((size_t)i * n + a) * m + d];
            }
    }

    /* phi, w: Eq. 20f, 20g */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < Ms; ++j) {
            size_t q = ((size_t)i * Ms + j) * m;
            for (int kind = 1; kind <= 2; ++kind) {
                if (o->numeric) continue;                   /* A20: the balls are handled inside NumericSolve */
                if (kind == 1 ? !o->has_vel : !o->has_acc) continue;
                const real_t *e = (kind == 1 ? o->E1 : o->E2) + ((size_t)i * Ms + j) * n;
                real_t *Phi = (kind == 1 ? o->PhiV : o->PhiA) + q, *W = (kind == 1 ? o->WV : o->WA) + q;
                real_t Y[3];
                for (int d = 0; d < m; ++d) {
                    real_t acc = 0;
                    for (int a = 0; a < n; ++a) acc += e[a] * o->C[((size_t)i * n + a) * m + d];
                    Y[d] = acc + W[d];
                }
                proj_ball(m, Y, kind == 1 ? o->vmax : o->amax, Phi);
                for (int d = 0; d < m; ++d) W[d] = Y[d] - Phi[d];
            }
        }

    /* UpdateConsensus: Eq. 6b / 20b. z_0, z_N fixed (L141). */
    memcpy(o->zprev, o->z, sizeof(real_t) * (size_t)(N + 1) * nc * m);
#pragma omp parallel for schedule(static)
    for (int j = 1; j <= N - 1; ++j) {
        const real_t *Ml = o->M + (size_t)(j - 1) * 2 * nc * n, *Mr = o->M + (size_t)j * 2 * nc * n;
        for (int k = 0; k < nc; ++k) {
            if (k == 0 && o->mode == MODE_PINNED_Z) continue;   /* position row held at p_j */
            for (int d = 0; d < m; ++d) {
                real_t bl = 0, br = 0;
                for (int a = 0; a < n; ++a) {
                    bl += Ml[(nc + k) * n + a] * o->C[((size_t)(j - 1) * n + a) * m + d];
                    br += Mr[k * n + a] * o->C[((size_t)j * n + a) * m + d];
                }
                o->z[((size_t)j * nc + k) * m + d] = (real_t)0.5 * (bl + br);
            }
        }
    }

    /* UpdateResidual (Eq. 21, 22; A7, A8), ProjectNonNeg (20d), UpdateDual (20c, 20e) */
#pragma omp parallel for schedule(static)
    for (int i = 0; i < N; ++i) {
        const real_t *M = o->M + (size_t)i * 2 * nc * n;
        real_t rp2 = 0, rd2 = 0, rdn2 = 0, gap2 = 0;
        real_t dz[RMAX * 3];
        for (int r = 0; r < 2 * nc; ++r) {
            size_t zi = ((size_t)(i + (r >= nc)) * nc + (r % nc)) * m;
            for (int d = 0; d < m; ++d) {
                dz[r * m + d] = 0;
                if (o->rowmask[(size_t)i * 2 * nc + r] == 0) continue;  /* no such row (A1) */
                real_t b = 0;
                for (int a = 0; a < n; ++a) b += M[r * n + a] * o->C[((size_t)i * n + a) * m + d];
                real_t res = b - o->z[zi + d];
                rp2 += res * res;
                o->u[((size_t)i * 2 * nc + r) * m + d] += res;          /* Eq. 20c */
                dz[r * m + d] = o->z[zi + d] - o->zprev[zi + d];
                if (r >= nc && i < N - 1) {                             /* Eq. 21 verbatim: junction gap */
                    real_t br = 0;
                    const real_t *Mn = o->M + (size_t)(i + 1) * 2 * nc * n;
                    for (int a = 0; a < n; ++a) br += Mn[(r - nc) * n + a] * o->C[((size_t)(i + 1) * n + a) * m + d];
                    gap2 += (b - br) * (b - br);
                }
            }
        }
        real_t Tp = 1;
        for (int a = 0; a < n; ++a) {                                   /* rho M'(dz~): Eq. 22 */
            for (int d = 0; d < m; ++d) {
                real_t acc = 0;
                for (int r = 0; r < 2 * nc; ++r) acc += M[r * n + a] * dz[r * m + d];
                acc *= rho;
                rd2 += acc * acc;
                rdn2 += (acc / Tp) * (acc / Tp);
            }
            Tp *= o->T[i];
        }
        o->part[(size_t)i * 4 + 0] = rp2; o->part[(size_t)i * 4 + 1] = rd2;
        o->part[(size_t)i * 4 + 2] = rdn2; o->part[(size_t)i * 4 + 3] = gap2;

        if (o->numeric)                                  /* multiplier of Eq. 17, scaled: w_j <- w_j + g_j(c^{k+1})  (A20) */
            for (int j = 0; j < Ms; ++j) {
                if (o->has_vel) o->Yv[(size_t)i * Ms + j] += numeric_g(o, i, j, 1, o->C + (size_t)i * n * m);
                if (o->has_acc) o->Ya[(size_t)i * Ms + j] += numeric_g(o, i, j, 2, o->C + (size_t)i * n * m);
            }

        if (o->has_box)
            for (int j = 0; j < Ms; ++j) {
                const real_t *e0 = o->E0 + ((size_t)i * Ms + j) * n;
                size_t q = ((size_t)i * Ms + j) * m;
                for (int d = 0; d < m; ++d) {
                    real_t P = 0;
                    for (int a = 0; a < n; ++a) P += e0[a] * o->C[((size_t)i * n + a) * m + d];
                    real_t hi = o->hi[(size_t)i * m + d], lo = o->lo[(size_t)i * m + d];
                    real_t sp = -(P - hi + o->Vp[q + d]);            /* Eq. 20d, + side: A=E0,  b=hi  */
                    real_t sn = -(-P + lo + o->Vn[q + d]);           /*          - side: A=-E0, b=-lo */
                    o->Sp[q + d] = sp > 0 ? sp : 0;
                    o->Sn[q + d] = sn > 0 ? sn : 0;
                    o->Vp[q + d] += P + o->Sp[q + d] - hi;           /* Eq. 20e */
                    o->Vn[q + d] += -P + o->Sn[q + d] + lo;
                }
            }
    }
    if (o->has_poly) {                           /* Eq. 20d, 20e per (sample, plane): A = kron(e0_j, a_k), b = b_k */
#pragma omp parallel for schedule(static)
        for (int i = 0; i < N; ++i)
            for (int j = 0; j < Ms; ++j) {
                const real_t *e0 = o->E0 + ((size_t)i * Ms + j) * n;
                real_t P[3] = {0, 0, 0};
                for (int d = 0; d < m; ++d) for (int a = 0; a < n; ++a) P[d] += e0[a] * o->C[((size_t)i * n + a) * m + d];
                for (int k = 0; k < o->K; ++k) {
                    const real_t *pl = o->planes + ((size_t)i * o->K + k) * (m + 1);
                    size_t qk = ((size_t)i * Ms + j) * o->K + k;
                    real_t val = 0;
                    for (int d = 0; d < m; ++d) val += pl[d] * P[d];
                    real_t sl = -(val - pl[m] + o->Vpl[qk]);
                    o->Spl[qk] = sl > 0 ? sl : 0;
                    o->Vpl[qk] += val + o->Spl[qk] - pl[m];
                }
            }
    }
    real_t a0 = 0, a1 = 0, a2 = 0, a3 = 0;       /* fixed-order (serial) reduction */
    for (int i = 0; i < N; ++i) { a0 += o->part[(size_t)i * 4]; a1 += o->part[(size_t)i * 4 + 1];
                                  a2 += o->part[(size_t)i * 4 + 2]; a3 += o->part[(size_t)i * 4 + 3]; }
    o->rp = (double)R_SQRT(a0); o->rd = (double)R_SQRT(a1); o->rd_norm = (double)R_SQRT(a2); o->rp_gap = (double)R_SQRT(a3);
    o->iter += 1;
}

/* run k sweeps on `threads` OpenMP threads (<=0: leave the runtime default) */
void oracle_sweep(oracle_t *o, int64_t k, int threads) {
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
    for (int64_t it = 0; it < k; ++it) sweep_once(o);
}

int oracle_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* sweep until rp < eps and rd (or its normalised variant) < eps, or max_iter; returns sweeps done in this call */
int64_t oracle_solve(oracle_t *o, double eps, int64_t max_iter, int use_rd_norm, int threads) {
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
    int64_t it = 0;
    while (it < max_iter) {
        sweep_once(o); ++it;
        double rd = use_rd_norm ? o->rd_norm : o->rd;
        if (o->rp < eps && rd < eps) break;
    }
    return it;
}

/*
 * Adaptive rho (Eq. 24; Alg. 1 line 14).  Changing rho changes the x-update operator
 * (rebuilt from scratch) and -- reading A16, the paper is silent -- the SCALED duals u = y/rho, v, w are
 * multiplied by rho_old/rho_new so that the unscaled multipliers y = rho*u are unchanged (Boyd et al. [8] 3.4.1).
 * Returns 0 on success.
 */
int oracle_set_rho(oracle_t *o, double rho_new) {
    if (!(rho_new > 0)) return -1;
    const int N = o->N, m = o->m, Ms = o->Ms;
    const real_t r = o->rho / (real_t)rho_new;
    for (size_t a = 0; a < (size_t)N * 2 * o->nc * m; ++a) o->u[a] *= r;
    for (size_t a = 0; a < (size_t)N * Ms * m; ++a) { o->Vp[a] *= r; o->Vn[a] *= r; o->WV[a] *= r; o->WA[a] *= r; }
    for (size_t a = 0; a < (size_t)N * Ms * o->K; ++a) o->Vpl[a] *= r;
    for (size_t a = 0; a < (size_t)N * Ms; ++a) { o->Yv[a] *= r; o->Ya[a] *= r; }
    o->rho = (real_t)rho_new;
    for (int i = 0; i < N; ++i) if (o->has_poly ? build_operator_poly(o, i) : build_operator(o, i)) return -1;
    return 0;
}

double oracle_rho(const oracle_t *o) { return (double)o->rho; }

/* switch the solver to the NumericSolve branch (reading A20); call right after create (iterate 0).  Returns 0 on success. */
int oracle_set_numeric(oracle_t *o, int memory, int max_inner, double tol) {
    if (o->has_poly || o->iter != 0 || memory < 1 || memory > LBFGS_MMAX || max_inner < 1 || !(tol >= 0)) return -1;
    o->numeric = 1; o->lbfgs_m = memory; o->lbfgs_maxit = max_inner; o->lbfgs_tol = tol;
    for (int i = 0; i < o->N; ++i) if (build_operator(o, i)) return -1;      /* H0: the quadratic part only */
    return 0;
}
int64_t oracle_inner_iters(const oracle_t *o) { return o->inner_iters; }
/* F and its gradient for segment i at coefficients c [n][m] (the current z, u, s, v, w): exposed for the pins */
double oracle_numeric_eval(const oracle_t *o, int i, const double *c, double *grad) {
    real_t cc[NVAR], gg[NVAR];
    for (int a = 0; a < o->n * o->m; ++a) cc[a] = (real_t)c[a];
    real_t F = numeric_eval(o, i, cc, grad ? gg : NULL);
    if (grad) for (int a = 0; a < o->n * o->m; ++a) grad[a] = (double)gg[a];
    return (double)F;
}

/* Alg. 1 with line 14: sweep; test the stop rule (Eq. 23); every `every` sweeps apply Eq. 24 with the residuals of
 * that sweep:  rho <- tau_incr*rho if r_p > mu r_d;  rho <- rho/tau_decr if r_d > mu r_p.  Returns sweeps done. */
int64_t oracle_solve_adaptive(oracle_t *o, double eps, int64_t max_iter, int use_rd_norm, double mu, double tau_incr,
                              double tau_decr, int every, int threads) {
#ifdef _OPENMP
    if (threads > 0) omp_set_num_threads(threads);
#else
    (void)threads;
#endif
    int64_t it = 0;
    while (it < max_iter) {
        sweep_once(o); ++it;
        double rd = use_rd_norm ? o->rd_norm : o->rd;
        if (o->rp < eps && rd < eps) break;
        if (every > 0 && it % every == 0) {
            if (o->rp > mu * rd) oracle_set_rho(o, (double)o->rho * tau_incr);
            else if (rd > mu * o->rp) oracle_set_rho(o, (double)o->rho / tau_decr);
        }
    }
    return it;
}

/* out[0..3] = r_p (A7), r_d (Eq. 22, A8), r_d normalised, r_p of Eq. 21 verbatim (junction gaps) */
void oracle_residuals(const oracle_t *o, double *out) {
    out[0] = o->rp; out[1] = o->rd; out[2] = o->rd_norm; out[3] = o->rp_gap;
}

/* J = sum_i tr(C_i' Q(T_i) C_i)   (Eq. 2a with W = I, A19) */
double oracle_objective(const oracle_t *o) {
    real_t J = 0;
    for (int i = 0; i < o->N; ++i)
        for (int d = 0; d < o->m; ++d)
            for (int a = 0; a < o->n; ++a)
                for (int b = 0; b < o->n; ++b)
                    J += o->C[((size_t)i * o->n + a) * o->m + d] * o->Q[((size_t)i * o->n + a) * o->n + b]
                       * o->C[((size_t)i * o->n + b) * o->m + d];
    return (double)J;
}

int64_t oracle_iter(const oracle_t *o) { return o->iter; }

/* copy a field as doubles. returns the element count, or -1 for an unknown name.
 * "coeffs" is [N][m][n] (dim-major per segment, the paper's squeezed c_i); every other field is in its
 * native layout: C [N][n][m], z [N+1][nc][m], u [N][2nc][m], sample fields [N][Ms][m], Pm [N][n][n] ... */
int64_t oracle_get(const oracle_t *o, const char *name, double *out) {
    const int N = o->N, n = o->n, m = o->m, Ms = o->Ms, nc = o->nc;
    const real_t *src = NULL; size_t cnt = 0;
    if (!strcmp(name, "coeffs")) {
        for (int i = 0; i < N; ++i) for (int d = 0; d < m; ++d) for (int a = 0; a < n; ++a)
            out[((size_t)i * m + d) * n + a] = (double)o->C[((size_t)i * n + a) * m + d];
        return (int64_t)N * m * n;
    }
#define FIELD(nm, ptr, count) else if (!strcmp(name, nm)) { src = (ptr); cnt = (size_t)(count); }
    if (0) {}
    FIELD("C", o->C, (size_t)N * n * m) FIELD("z", o->z, (size_t)(N + 1) * nc * m) FIELD("u", o->u, (size_t)N * 2 * nc * m)
    FIELD("s_pos", o->Sp, (size_t)N * Ms * m) FIELD("s_neg", o->Sn, (size_t)N * Ms * m)
    FIELD("v_pos", o->Vp, (size_t)N * Ms * m) FIELD("v_neg", o->Vn, (size_t)N * Ms * m)
    FIELD("phi_v", o->PhiV, (size_t)N * Ms * m) FIELD("w_v", o->WV, (size_t)N * Ms * m)
    FIELD("phi_a", o->PhiA, (size_t)N * Ms * m) FIELD("w_a", o->WA, (size_t)N * Ms * m)
    FIELD("y_v", o->Yv, (size_t)N * Ms) FIELD("y_a", o->Ya, (size_t)N * Ms)
    FIELD("s_poly", o->Spl, (size_t)N * Ms * o->K) FIELD("v_poly", o->Vpl, (size_t)N * Ms * o->K)
    FIELD("Pm", o->Pm, (size_t)N * n * n) FIELD("c0", o->c0, (size_t)N * n * m) FIELD("Q", o->Q, (size_t)N * n * n)
    FIELD("M", o->M, (size_t)N * 2 * nc * n) FIELD("rowmask", o->rowmask, (size_t)N * 2 * nc) FIELD("E0", o->E0, (size_t)N * Ms * n) FIELD("E1", o->E1, (size_t)N * Ms * n)
    FIELD("E2", o->E2, (size_t)N * Ms * n)
    else return -1;
#undef FIELD
    for (size_t a = 0; a < cnt; ++a) out[a] = (double)src[a];
    return (int64_t)cnt;
}
