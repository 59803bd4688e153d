// top_api.cpp -- host side of the C ABI in include/top.h: validation, the one-off per-segment precompute of
// the x-update operator (Eq. 20a), SoA packing, launch planning and the calls themselves.
// Product code: shares nothing with oracle/.  Every sweep step runs in top_kernels.cu; there is no CPU path.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <chrono>
#include <cstdlib>
#include <thread>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <memory>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/top.h"
#include "top_internal.h"

using namespace top;

namespace {

typedef long double xreal;   // precision of the one-off operator precompute (cond(H) reaches 1e13, R6)

thread_local std::string g_create_error;

// phase timer of top_create / top_reset (stderr, enabled by the environment variable TOP_TRACE_CREATE=1)
struct PhaseTimer {
    bool on;
    std::chrono::steady_clock::time_point t0;
    PhaseTimer() : on(std::getenv("TOP_TRACE_CREATE") != nullptr), t0(std::chrono::steady_clock::now()) {}
    void mark(const char* what) {
        if (!on) return;
        const auto t1 = std::chrono::steady_clock::now();
        std::fprintf(stderr, "[top_create] %-28s %8.3f ms\n", what, std::chrono::duration<double, std::milli>(t1 - t0).count());
        t0 = t1;
    }
};

}  // namespace

namespace {
// One private memory pool per device for the solvers' arenas.  Freed arenas stay in the pool (up to 1 GiB; beyond that the
// driver releases them at the next synchronisation), so top_destroy followed by top_create of a similar size costs no driver
// allocation.  nullptr: pools unavailable on this device -> plain cudaMalloc / cudaFree.
cudaMemPool_t arena_pool(int device) {
    constexpr int MAXDEV = 64;
    static std::mutex mu;
    static cudaMemPool_t pools[MAXDEV] = {};
    static bool tried[MAXDEV] = {};
    if (device < 0 || device >= MAXDEV) return nullptr;
    std::lock_guard<std::mutex> lk(mu);
    if (!tried[device]) {
        tried[device] = true;
        int supported = 0;
        if (cudaDeviceGetAttribute(&supported, cudaDevAttrMemoryPoolsSupported, device) == cudaSuccess && supported) {
            cudaMemPoolProps props;
            std::memset(&props, 0, sizeof props);
            props.allocType = cudaMemAllocationTypePinned;
            props.handleTypes = cudaMemHandleTypeNone;
            props.location.type = cudaMemLocationTypeDevice;
            props.location.id = device;
            cudaMemPool_t pool = nullptr;
            unsigned long long keep = 1ull << 30;
            if (cudaMemPoolCreate(&pool, &props) == cudaSuccess &&
                cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep) == cudaSuccess)
                pools[device] = pool;
        }
        cudaGetLastError();
    }
    return pools[device];
}
}  // namespace

struct top_solver {
    int batch = 0, N = 0, s = 0, dims = 0, dtype = 0, n = 0;
    uint32_t opt_flags = 0, kflags = 0;
    bool constrained = false, has_box = false, has_vel = false, has_acc = false;
    double rho = 0, vmax = 0, amax = 0;
    int check_every = 32;
    int64_t max_iter = 1000000;
    int device = 0;
    cudaStream_t stream = nullptr;
    long long nseg = 0, nseg_pad = 0, stride = 0;
    int num_sms = 0, max_ctas = 0, user_segs = 0, lanes = 8;
    bool mma = false;                  // fp64, 4 lanes per segment: the tensor-core (DMMA) kernel of top_kernels_mma.cu
    bool wide = false;                 // paper-literal consensus n_c = 2s-1 (reading A1): second block of consensus rows
    int nc = 0;                        // consensus derivative orders per boundary: s, or 2s-1
    void *d_zt2 = nullptr, *d_u2 = nullptr, *d_invTk2 = nullptr;
    // NumericSolve branch (TOP_XUPDATE_NUMERIC; top_kernels_numeric.cu): state in device memory, two launches per sweep
    bool numeric = false;
    double *d_yv = nullptr, *d_ya = nullptr, *d_bnd = nullptr;
    unsigned long long* d_inner = nullptr;
    struct Wave { long long seg_begin, seg_end, own_begin, own_end; uint32_t kflags; int segs_per_cta, ctas, threads; size_t smem;
                  bool cluster;      // the wave can run as ONE thread-block cluster (<= 16 CTAs): exchange through distributed shared memory
    };
    // streaming (temporal blocking) for chains longer than the on-chip capacity: pieces with `halo` extra segments on
    // each open side run `halo` sweeps per launch (the dependency radius of a sweep is one segment), reading iterate
    // k from one set of state buffers and writing iterate k + halo of their own segments to the other set
    bool streaming = false;
    int halo = 0;
    void* alt[8] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    std::vector<Wave> waves;
    // device buffers: ONE arena allocation carved into the arrays below (one cudaMalloc / cudaFree per solver)
    unsigned char* arena = nullptr;
    size_t arena_bytes = 0;
    bool arena_pooled = false;      // allocated from arena_pool(device) with cudaMallocFromPoolAsync (else plain cudaMalloc)
    unsigned char* d_upload = nullptr;     // region that mirrors the host staging buffer: [rho Pm^ rows | the caller's arrays]
    size_t off_gram = 0;                   // double-double Gram tables for the device-side operator precompute (first byte of what is uploaded then)
    size_t upload_bytes = 0, off_wp = 0, off_T = 0, off_lo = 0, off_hi = 0, off_sd = 0, off_ed = 0;
    bool have_sd = false, have_ed = false;
    unsigned char* zero_begin = nullptr;   // arrays that top_reset sets to zero again (duals, partial sums)
    size_t zero_bytes = 0;
    std::unique_ptr<unsigned char[]> stage;   // host staging buffer (kept: top_reset re-uses it)
    std::vector<double> h_wp, h_T;         // host copies of waypoints / durations (local-frame origins, lazy spectral form)
    bool have_spectral = false;            // W, lambda on the device (built on first use: top_set_rho, Eq. 24)
    // general polytope corridor (reading A11p): K planes per segment; per-segment rotated frame
    bool has_poly = false;
    int K = 0;
    double *d_rot = nullptr, *d_planes = nullptr, *d_lam3 = nullptr, *d_qpl = nullptr;
    size_t off_rot = 0, off_planes = 0, off_lam3 = 0, pm_dims = 1;
    std::vector<double> h_rot;             // [9][nseg_pad] host copy of the rotations (top_get_state)
    std::vector<double> h_planes;          // host copy of the caller's planes (a new rho rebuilds the operators)
    double *d_Pm = nullptr, *d_c0 = nullptr, *d_part = nullptr, *d_res = nullptr;
    double *d_W = nullptr, *d_lam = nullptr, *d_g0 = nullptr, *d_dp = nullptr;   // spectral operator data (rho-independent)
    void *d_invTk = nullptr, *d_Tpow = nullptr, *d_invT = nullptr, *d_lohi = nullptr, *d_zoff = nullptr;
    double* d_origin = nullptr;        // [3][nseg_pad] origin o_i = p_{i-1} of each segment's local frame
    uint32_t wp_mode = 0;
    double adapt_mu = 10.0, adapt_incr = 1.1, adapt_decr = 1.1;
    uint8_t* d_segflags = nullptr;
    void *d_zt = nullptr, *d_u = nullptr, *d_qp = nullptr, *d_qn = nullptr, *d_phv = nullptr, *d_wv = nullptr,
         *d_pha = nullptr, *d_wa = nullptr, *d_chat = nullptr, *d_Bedge = nullptr, *d_coef = nullptr;
    unsigned char* d_sync = nullptr;   // u64 grid-barrier counter
    int* d_abort = nullptr;
    std::vector<double> h_res;         // [batch][4]   (small results come back into pageable memory: every fetch
    int h_abort[4] = {0, 0, 0, 0};     //                synchronises the stream anyway, and pinned allocations cost ms)
    void* d_resbox = nullptr;          // in-kernel solve: LL slots of the per-CTA residual partial sums
    double* d_solve = nullptr;         // in-kernel solve result [8]
    double h_solve[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    bool have_residuals = false;
    int64_t iter = 0, launches = 0;
    unsigned long long seq_counter = 0;   // sweeps launched so far over all waves (mailbox sequence space; the slots carry its low 32 bits)
    size_t bedge_bytes = 0, resbox_bytes = 0;   // sizes of the two mailboxes (cleared when the sequence space starts a new epoch)
    std::string err;
};

namespace {

size_t real_bytes(const top_solver* h) { return h->dtype == TOP_F64 ? 8 : 4; }

top_status fail(top_solver* h, top_status st, const std::string& msg) {
    if (h) h->err = msg; else g_create_error = msg;
    return st;
}
top_status cuda_fail(top_solver* h, cudaError_t e, const char* what) {
    return fail(h, TOP_E_CUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define CU(call, what) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(h, e_, what); } while (0)

// ---------------------------------------------------------------------------------- small dense linear algebra

// [beta_k(tau)]_a = a!/(a-k)! tau^(a-k)   (Eq. 18 differentiated, normalised time)
xreal beta_hat(int k, int a, xreal tau) {
    if (a < k) return 0;
    xreal f = 1;
    for (int q = 0; q < k; ++q) f *= (xreal)(a - q);
    return f * std::pow(tau, (xreal)(a - k));
}

// In-place inverse of a symmetric positive definite q x q matrix: symmetric diagonal scaling, then
// Gauss-Jordan elimination without pivoting (safe for SPD), in extended precision.  false if not SPD.
bool spd_invert(int q, xreal* A) {
    xreal sc[MAXN], W[MAXN * 2 * MAXN];
    for (int i = 0; i < q; ++i) {
        if (!(A[i * q + i] > 0)) return false;
        sc[i] = 1 / std::sqrt(A[i * q + i]);
    }
    for (int i = 0; i < q; ++i) {
        for (int j = 0; j < 2 * q; ++j) W[i * 2 * q + j] = 0;
        for (int j = 0; j < q; ++j) W[i * 2 * q + j] = A[i * q + j] * sc[i] * sc[j];
        W[i * 2 * q + q + i] = 1;
    }
    for (int c = 0; c < q; ++c) {
        const xreal piv = W[c * 2 * q + c];
        if (!(piv > 0)) return false;
        for (int j = 0; j < 2 * q; ++j) W[c * 2 * q + j] /= piv;
        for (int r = 0; r < q; ++r) {
            if (r == c) continue;
            const xreal f = W[r * 2 * q + c];
            if (f == 0) continue;
            for (int j = 0; j < 2 * q; ++j) W[r * 2 * q + j] -= f * W[c * 2 * q + j];
        }
    }
    for (int i = 0; i < q; ++i)
        for (int j = 0; j < q; ++j) A[i * q + j] = W[i * 2 * q + q + j] * sc[i] * sc[j];
    for (int i = 0; i < q; ++i)          // symmetrise the rounding
        for (int j = 0; j < i; ++j) { const xreal m = (A[i * q + j] + A[j * q + i]) / 2; A[i * q + j] = A[j * q + i] = m; }
    return true;
}

// Per-segment operator in the normalised-time basis c^_a = c_a T^a:
//   H^ = 2 T^(1-2s) Q(1) + rho [ sum_r m^_r m^_r' + 2 sum_j e0_j e0_j' + sum_j e1_j e1_j'/T^2 + sum_j e2_j e2_j'/T^4 ]
// (Eq. 20a first bracket; Q, M, Ao, Av of PAPER.md:L231; cost without 1/2 => 2Q, reading A19).
// HARD waypoint mode (reading A2): the two equalities c^_0 = p_{i-1}, sum_a c^_a = p_i are eliminated with the
// null-space basis Z = {e_a - e_1, a >= 2}:  Pm^ = Z (Z'H^Z)^-1 Z',  c0^ = (I - Pm^ H^) c_chord.
// Other modes: Pm^ = H^^-1, c0^ = 0.
// Gram matrices of the constant (normalised-time) rows, built once per s: H^ is a T-weighted sum of them.
struct GramTables {
    xreal Q1[MAXN * MAXN];        // int_0^1 beta^(s) beta^(s)'
    xreal Gc[4][MAXN * MAXN];     // consensus rows of derivative order k: beta_k(0)beta_k(0)' + beta_k(1)beta_k(1)'
    xreal Ge[3][MAXN * MAXN];     // sample rows of E_0, E_1, E_2: sum_j beta_k(tau_j) beta_k(tau_j)'
    xreal Gw[2][3][MAXN * MAXN];  // wide consensus (n_c = 2s-1): order s + j at tau = 0 ([0][j]) and at tau = 1 ([1][j]), j <= s-2
};
void build_gram_tables(int s, GramTables& G) {
    const int n = 2 * s;
    std::memset(&G, 0, sizeof G);
    for (int j = s; j < n; ++j)
        for (int l = s; l < n; ++l) {
            xreal fj = 1, fl = 1;
            for (int q = 0; q < s; ++q) { fj *= (xreal)(j - q); fl *= (xreal)(l - q); }
            G.Q1[j * MAXN + l] = fj * fl / (xreal)(j + l - 2 * s + 1);
        }
    auto add = [&](xreal* M, int k, xreal tau) {
        xreal row[MAXN];
        for (int a = 0; a < n; ++a) row[a] = beta_hat(k, a, tau);
        for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) M[a * MAXN + b] += row[a] * row[b];
    };
    for (int k = 0; k < s; ++k) { add(G.Gc[k], k, 0); add(G.Gc[k], k, 1); }
    for (int j = 0; j <= s - 2; ++j) { add(G.Gw[0][j], s + j, 0); add(G.Gw[1][j], s + j, 1); }
    for (int j = 1; j <= MS; ++j)
        for (int k = 0; k < 3; ++k) add(G.Ge[k], k, (xreal)j / (xreal)(MS + 1));     // reading A10
}
const GramTables& gram_tables(int s) {       // built once per s, whatever thread comes first (concurrent top_create calls)
    static GramTables tab[2];
    static std::once_flag once[2];
    std::call_once(once[s - 3], [s] { build_gram_tables(s, tab[s - 3]); });
    return tab[s - 3];
}

bool build_operator(int s, xreal T, xreal rho, bool box, bool vel, bool acc, int mode,
                    const xreal* p0, const xreal* p1, xreal* Pm /*[8][8]*/, xreal* c0 /*[8][3]*/, xreal box_weight = 2,
                    int wide_mask = 0 /* bit 0 / 1: the consensus rows of orders s..2s-2 exist at the start / end boundary */) {
    const int n = 2 * s;
    const GramTables& G = gram_tables(s);
    xreal iT[14];                      // T^-k
    iT[0] = 1;
    for (int k = 1; k < 14; ++k) iT[k] = iT[k - 1] / T;
    const xreal wq = 2 * T * iT[2 * s - 1] * iT[1];             // 2 T^(1-2s)
    const xreal wb = box ? box_weight * rho : 0;               // box: its two sides (A11); polytope: eigenvalue of sum_k a_k a_k' (A11p)
    const xreal wv = vel ? rho * iT[2] : 0, wa = acc ? rho * iT[4] : 0;
    xreal H[MAXN * MAXN];
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b) {
            const int i = a * MAXN + b;
            xreal v = wq * G.Q1[i] + wb * G.Ge[0][i] + wv * G.Ge[1][i] + wa * G.Ge[2][i];
            for (int k = 0; k < s; ++k) v += rho * iT[2 * k] * G.Gc[k][i];
            for (int side = 0; side < 2; ++side)
                if (wide_mask & (1 << side)) for (int j = 0; j <= s - 2; ++j) v += rho * iT[2 * (s + j)] * G.Gw[side][j][i];
            H[a * n + b] = v;
        }
    for (int i = 0; i < MAXN * MAXN; ++i) Pm[i] = 0;
    if (c0) for (int i = 0; i < MAXN * 3; ++i) c0[i] = 0;
    if (mode == (int)TOP_WAYPOINT_HARD) {
        const int q = n - 2;
        xreal A[MAXN * MAXN];
        auto Hz = [&](int a, int b) { return H[a * n + b]; };
        for (int i = 0; i < q; ++i)
            for (int j = 0; j < q; ++j) {
                const int a = i + 2, b = j + 2;            // Z column i = e_a - e_1
                A[i * q + j] = Hz(a, b) - Hz(a, 1) - Hz(1, b) + Hz(1, 1);
            }
        if (!spd_invert(q, A)) return false;
        // Pm^ = Z A^-1 Z'
        for (int i = 0; i < q; ++i)
            for (int j = 0; j < q; ++j) {
                const xreal v = A[i * q + j];
                Pm[(i + 2) * MAXN + (j + 2)] += v;
                Pm[1 * MAXN + (j + 2)] -= v;
                Pm[(i + 2) * MAXN + 1] -= v;
                Pm[1 * MAXN + 1] += v;
            }
        for (int d = 0; c0 && d < 3; ++d) {
            xreal cp[MAXN] = {0}, Hc[MAXN] = {0};
            cp[0] = p0[d]; cp[1] = p1[d] - p0[d];
            for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) Hc[a] += H[a * n + b] * cp[b];
            for (int a = 0; a < n; ++a) {
                xreal acc2 = 0;
                for (int b = 0; b < n; ++b) acc2 += Pm[a * MAXN + b] * Hc[b];
                c0[a * 3 + d] = cp[a] - acc2;
            }
        }
    } else {
        xreal A[MAXN * MAXN];
        for (int i = 0; i < n * n; ++i) A[i] = H[i];
        if (!spd_invert(n, A)) return false;
        for (int a = 0; a < n; ++a) for (int b = 0; b < n; ++b) Pm[a * MAXN + b] = A[a * n + b];
    }
    return true;
}

// ---- rho-independent (spectral) form of the same operator, so that rho is a run-time parameter on the device.
// H^(rho) = Q2 + rho G with Q2 = 2 T^(1-2s) Q(1) and G the Gram matrix of all penalty rows (Eq. 20a first bracket).
// In the reduced basis Z (HARD: polynomials vanishing at both ends; else Z = I):  A_Q = Z'Q2 Z, A_G = Z'G Z (SPD).
// Generalised symmetric eigenproblem A_Q v = lambda A_G v with V'A_G V = I, V'A_Q V = Lambda gives
//     (A_Q + rho A_G)^-1 = V diag(1/(lambda_i + rho)) V'      =>     rho Pm^ = W diag(rho/(lambda_i + rho)) W',  W = Z V,
// and, because the chord (degree 1 < s) is in the null space of Q2,  c0^ = c_chord - (rho Pm^) (G c_chord).
// Everything below is done once per segment in extended precision (diagonal scaling, Cholesky of A_G, cyclic Jacobi
// on L^-1 A_Q L^-T); the device only evaluates the two formulas above (refresh_operator_kernel).
struct Spectral {
    xreal W[MAXN * MAXN];     // [a][i], zero padded
    xreal lam[MAXN];
    xreal g0[MAXN * 3];       // G c_chord, [a][d]   (HARD mode; else 0)
    xreal gcol0[MAXN];        // G e_0 (only top_precompute_operator needs it: a frame other than the local one)
    xreal gcol1[MAXN];        // G e_1: g0 = gcol1 * dp (kept so that segments of equal duration can share the rest)
    int q;
};

bool jacobi_eigen(int q, std::vector<xreal>& C, std::vector<xreal>& U) {       // C symmetric -> diag; U its eigenvectors
    U.assign(q * q, 0);
    for (int i = 0; i < q; ++i) U[i * q + i] = 1;
    for (int sweep = 0; sweep < 60; ++sweep) {
        xreal off = 0, diag = 0;
        for (int i = 0; i < q; ++i) for (int j = 0; j < q; ++j) (i == j ? diag : off) += C[i * q + j] * C[i * q + j];
        if (off <= diag * (xreal)1e-37 || off == 0) return true;   // off-diagonal mass below the rounding of long double
        for (int pp = 0; pp < q; ++pp)
            for (int r = pp + 1; r < q; ++r) {
                const xreal apq = C[pp * q + r];
                if (apq == 0) continue;
                const xreal theta = (C[r * q + r] - C[pp * q + pp]) / (2 * apq);
                const xreal t = (theta >= 0 ? 1 : -1) / (std::fabs(theta) + std::sqrt(theta * theta + 1));
                const xreal c = 1 / std::sqrt(t * t + 1), sn = t * c;
                for (int k = 0; k < q; ++k) {       // columns
                    const xreal a = C[k * q + pp], b = C[k * q + r];
                    C[k * q + pp] = c * a - sn * b; C[k * q + r] = sn * a + c * b;
                }
                for (int k = 0; k < q; ++k) {       // rows
                    const xreal a = C[pp * q + k], b = C[r * q + k];
                    C[pp * q + k] = c * a - sn * b; C[r * q + k] = sn * a + c * b;
                }
                for (int k = 0; k < q; ++k) {
                    const xreal a = U[k * q + pp], b = U[k * q + r];
                    U[k * q + pp] = c * a - sn * b; U[k * q + r] = sn * a + c * b;
                }
            }
    }
    return true;
}

bool build_spectral(int s, xreal T, bool box, bool vel, bool acc, int mode, const xreal* dp, Spectral& S, int wide_mask = 0) {
    const int n = 2 * s;
    const GramTables& G = gram_tables(s);
    xreal iT[14];
    iT[0] = 1;
    for (int k = 1; k < 14; ++k) iT[k] = iT[k - 1] / T;
    const xreal wq = 2 * T * iT[2 * s - 1] * iT[1];             // 2 T^(1-2s)
    std::vector<xreal> Q2(n * n), Gm(n * n);
    for (int a = 0; a < n; ++a)
        for (int b = 0; b < n; ++b) {
            const int i = a * MAXN + b;
            Q2[a * n + b] = wq * G.Q1[i];
            xreal v = (box ? 2 * G.Ge[0][i] : 0) + (vel ? iT[2] * G.Ge[1][i] : 0) + (acc ? iT[4] * G.Ge[2][i] : 0);
            for (int k = 0; k < s; ++k) v += iT[2 * k] * G.Gc[k][i];
            for (int side = 0; side < 2; ++side)
                if (wide_mask & (1 << side)) for (int j = 0; j <= s - 2; ++j) v += iT[2 * (s + j)] * G.Gw[side][j][i];
            Gm[a * n + b] = v;
        }
    const bool hard = mode == (int)TOP_WAYPOINT_HARD;
    const int q = hard ? n - 2 : n;
    std::vector<xreal> AQ(q * q), AG(q * q);
    auto red = [&](const std::vector<xreal>& M, int i, int j) -> xreal {
        if (!hard) return M[i * n + j];
        const int a = i + 2, b = j + 2;                         // Z column i = e_a - e_1
        return M[a * n + b] - M[a * n + 1] - M[1 * n + b] + M[1 * n + 1];
    };
    for (int i = 0; i < q; ++i) for (int j = 0; j < q; ++j) { AQ[i * q + j] = red(Q2, i, j); AG[i * q + j] = red(Gm, i, j); }
    std::vector<xreal> sc(q);
    for (int i = 0; i < q; ++i) { if (!(AG[i * q + i] > 0)) return false; sc[i] = 1 / std::sqrt(AG[i * q + i]); }
    for (int i = 0; i < q; ++i) for (int j = 0; j < q; ++j) { AQ[i * q + j] *= sc[i] * sc[j]; AG[i * q + j] *= sc[i] * sc[j]; }
    // Cholesky A_G = L L'
    std::vector<xreal> Lm(q * q, 0);
    for (int i = 0; i < q; ++i)
        for (int j = 0; j <= i; ++j) {
            xreal v = AG[i * q + j];
            for (int k = 0; k < j; ++k) v -= Lm[i * q + k] * Lm[j * q + k];
            if (i == j) { if (!(v > 0)) return false; Lm[i * q + i] = std::sqrt(v); }
            else Lm[i * q + j] = v / Lm[j * q + j];
        }
    // C = L^-1 A_Q L^-T  (two triangular solves)
    std::vector<xreal> Y(q * q), C(q * q), U;
    for (int c = 0; c < q; ++c)                                   // Y = L^-1 A_Q
        for (int i = 0; i < q; ++i) {
            xreal v = AQ[i * q + c];
            for (int k = 0; k < i; ++k) v -= Lm[i * q + k] * Y[k * q + c];
            Y[i * q + c] = v / Lm[i * q + i];
        }
    for (int r = 0; r < q; ++r)                                   // C = Y L^-T  <=>  C L' = Y, row by row
        for (int j = 0; j < q; ++j) {
            xreal v = Y[r * q + j];
            for (int k = 0; k < j; ++k) v -= C[r * q + k] * Lm[j * q + k];
            C[r * q + j] = v / Lm[j * q + j];
        }
    for (int i = 0; i < q; ++i) for (int j = 0; j < i; ++j) { const xreal m = (C[i * q + j] + C[j * q + i]) / 2; C[i * q + j] = C[j * q + i] = m; }
    if (!jacobi_eigen(q, C, U)) return false;
    // V = S L^-T U
    std::vector<xreal> V(q * q);
    for (int c = 0; c < q; ++c)
        for (int i = q - 1; i >= 0; --i) {
            xreal v = U[i * q + c];
            for (int k = i + 1; k < q; ++k) v -= Lm[k * q + i] * V[k * q + c];
            V[i * q + c] = v / Lm[i * q + i];
        }
    for (int i = 0; i < q; ++i) for (int c = 0; c < q; ++c) V[i * q + c] *= sc[i];
    std::memset(&S, 0, sizeof S);
    S.q = q;
    for (int i = 0; i < q; ++i) S.lam[i] = C[i * q + i] > 0 ? C[i * q + i] : 0;
    for (int i = 0; i < q; ++i) {
        if (hard) {
            xreal sum = 0;
            for (int a = 2; a < n; ++a) { S.W[a * MAXN + i] = V[(a - 2) * q + i]; sum += V[(a - 2) * q + i]; }
            S.W[1 * MAXN + i] = -sum;
        } else {
            for (int a = 0; a < n; ++a) S.W[a * MAXN + i] = V[a * q + i];
        }
    }
    if (hard) for (int a = 0; a < n; ++a) for (int d = 0; d < 3; ++d) S.g0[a * 3 + d] = Gm[a * n + 1] * dp[d];
    for (int a = 0; a < n; ++a) { S.gcol0[a] = Gm[a * n + 0]; S.gcol1[a] = Gm[a * n + 1]; }
    return true;
}

// host twin of refresh_operator_kernel (extended precision): rho Pm^ and c0^ from the spectral form
void spectral_operator(const Spectral& S, int n, bool hard, xreal rho, const xreal* dp, xreal* rhoPm /*[8][8]*/, xreal* c0 /*[8][3]*/) {
    for (int a = 0; a < MAXN; ++a)
        for (int b = 0; b < MAXN; ++b) {
            xreal v = 0;
            for (int i = 0; i < S.q; ++i) v += S.W[a * MAXN + i] * S.W[b * MAXN + i] * (rho / (S.lam[i] + rho));
            rhoPm[a * MAXN + b] = v;
        }
    for (int a = 0; a < MAXN; ++a)
        for (int d = 0; d < 3; ++d) {
            xreal v = (hard && a == 1) ? dp[d] : 0;
            for (int b = 0; b < n; ++b) v -= rhoPm[a * MAXN + b] * S.g0[b * 3 + d];
            c0[a * 3 + d] = v;
        }
}

top_status download_real(top_solver* h, const void* src, std::vector<double>& dst, size_t count) {
    dst.resize(count);
    if (h->dtype == TOP_F64) {
        CU(cudaMemcpyAsync(dst.data(), src, count * 8, cudaMemcpyDeviceToHost, h->stream), "D2H");
        CU(cudaStreamSynchronize(h->stream), "sync");
    } else {
        std::vector<float> f(count);
        CU(cudaMemcpyAsync(f.data(), src, count * 4, cudaMemcpyDeviceToHost, h->stream), "D2H");
        CU(cudaStreamSynchronize(h->stream), "sync");
        for (size_t i = 0; i < count; ++i) dst[i] = (double)f[i];
    }
    return TOP_OK;
}

int round_up(int x, int m) { return (x + m - 1) / m * m; }

// the sweep kernel family of a solver: 8 lanes, 4 lanes (shuffle form), or 4 lanes with fp64 tensor-core contractions
size_t kernel_smem(int dtype, int s, bool constrained, int lanes, bool mma, int segs, bool poly = false, bool wide = false) {
    return mma ? sweep_smem_bytes_mma(dtype, constrained, poly, wide) : sweep_smem_bytes(dtype, s, constrained, lanes, segs);
}
int kernel_max_threads(int dtype, int lanes, bool mma, bool poly = false, bool wide = false) {
    return mma ? max_threads_mma(dtype, poly, wide) : max_threads_for(dtype, lanes);
}

// largest segments-per-CTA (multiple of 4) whose threads and shared memory fit one CTA
int max_segs_per_cta(int dtype, int s, bool constrained, int lanes, bool mma, size_t smem_limit, bool poly = false, bool wide = false) {
    int best = 0;
    for (int segs = 4; (segs * lanes + 31) / 32 * 32 <= kernel_max_threads(dtype, lanes, mma, poly, wide); segs += 4)
        if (kernel_smem(dtype, s, constrained, lanes, mma, segs, poly, wide) <= smem_limit) best = segs;
    return best;
}

}  // namespace

// Host helpers for top_operator_rows_static (top_static_scratch.cu), which lives in a .cu file beside its static device array.
namespace top {
void gram_tables_dd(int s, GramDD* out) {       // the tables of gram_tables(s), each entry split into a double-double
    const GramTables& G = gram_tables(s);
    const xreal* tabs[GRAM_TABLES] = {G.Q1, G.Gc[0], G.Gc[1], G.Gc[2], G.Gc[3], G.Ge[0], G.Ge[1], G.Ge[2],
                                      G.Gw[0][0], G.Gw[0][1], G.Gw[0][2], G.Gw[1][0], G.Gw[1][1], G.Gw[1][2]};
    for (int t = 0; t < GRAM_TABLES; ++t)
        for (int i = 0; i < MAXN * MAXN; ++i) {
            const double hi = (double)tabs[t][i];
            out->hi[t][i] = hi; out->lo[t][i] = (double)(tabs[t][i] - (xreal)hi);
        }
}
int report_error(int status, const char* msg) { return (int)fail(nullptr, (top_status)status, msg); }
}  // namespace top

namespace {
// (re)build rho*Pm^ and c0^ on the device for `rho` from the spectral data
cudaError_t refresh_operator(top_solver* h, double rho) {
    RefreshParams r;
    r.W = h->d_W; r.lam = h->d_lam; r.g0 = h->d_g0; r.dp = h->d_dp; r.Pm = h->d_Pm; r.c0 = h->d_c0;
    r.stride = h->stride; r.nseg_pad = h->nseg_pad; r.nseg = h->nseg;
    r.q = h->wp_mode == TOP_WAYPOINT_HARD ? h->n - 2 : h->n;
    r.rho = rho;
    h->launches += 1;
    return launch_refresh_operator(r, h->stream);
}
// run fn(g0, g1) over [0, n) on the host cores (segments are independent).  A chunk whose thread cannot be started runs
// on the calling thread; fn must not throw (the callers catch inside).
template <typename F> void parallel_segments(long long n, F fn) {
    unsigned nt = std::thread::hardware_concurrency();
    nt = std::max(1u, std::min(nt, 32u));
    if (n < 2048) nt = 1;
    std::vector<std::thread> pool;
    const long long chunk = (n + nt - 1) / nt;
    for (unsigned t = 1; t < nt; ++t) {
        const long long lo = (long long)t * chunk, hi = std::min(n, (long long)(t + 1) * chunk);
        if (lo >= n) break;
        try { pool.emplace_back(fn, lo, hi); } catch (...) { fn(lo, hi); }
    }
    fn(0, std::min(n, chunk));
    for (auto& th : pool) th.join();
}
}  // namespace

namespace {

// symmetric 3x3 eigen-decomposition A = V diag(lam) V' (cyclic Jacobi, extended precision); V row-major, columns = axes
void eigen3(const xreal* A, xreal* V, xreal* lam) {
    xreal C[9];
    for (int i = 0; i < 9; ++i) { C[i] = A[i]; V[i] = (i % 4 == 0) ? 1 : 0; }
    for (int sweep = 0; sweep < 60; ++sweep) {
        const xreal off = C[1] * C[1] + C[2] * C[2] + C[5] * C[5], diag = C[0] * C[0] + C[4] * C[4] + C[8] * C[8];
        if (off <= diag * (xreal)1e-40 || off == 0) break;
        for (int pp = 0; pp < 3; ++pp)
            for (int r = pp + 1; r < 3; ++r) {
                const xreal apq = C[pp * 3 + r];
                if (apq == 0) continue;
                const xreal theta = (C[r * 3 + r] - C[pp * 3 + pp]) / (2 * apq);
                const xreal tt = (theta >= 0 ? 1 : -1) / (std::fabs(theta) + std::sqrt(theta * theta + 1));
                const xreal c = 1 / std::sqrt(tt * tt + 1), sn = tt * c;
                for (int k = 0; k < 3; ++k) { const xreal x = C[k * 3 + pp], y = C[k * 3 + r]; C[k * 3 + pp] = c * x - sn * y; C[k * 3 + r] = sn * x + c * y; }
                for (int k = 0; k < 3; ++k) { const xreal x = C[pp * 3 + k], y = C[r * 3 + k]; C[pp * 3 + k] = c * x - sn * y; C[r * 3 + k] = sn * x + c * y; }
                for (int k = 0; k < 3; ++k) { const xreal x = V[k * 3 + pp], y = V[k * 3 + r]; V[k * 3 + pp] = c * x - sn * y; V[k * 3 + r] = sn * x + c * y; }
            }
    }
    for (int d = 0; d < 3; ++d) lam[d] = C[d * 3 + d] > 0 ? C[d * 3 + d] : 0;
}
void fill_init_params(top_solver* h, InitParams& ip) {
    const GramTables& G = gram_tables(h->s);
    unsigned char* D = h->d_upload;
    ip.waypoints = (const double*)(D + h->off_wp); ip.durations = (const double*)(D + h->off_T);
    ip.box_lo = h->has_box ? (const double*)(D + h->off_lo) : nullptr; ip.box_hi = h->has_box ? (const double*)(D + h->off_hi) : nullptr;
    ip.start_derivs = h->have_sd ? (const double*)(D + h->off_sd) : nullptr;
    ip.end_derivs = h->have_ed ? (const double*)(D + h->off_ed) : nullptr;
    for (int a = 0; a < MAXN; ++a) {
        for (int k = 0; k < 4; ++k) ip.gc1[k][a] = (double)G.Gc[k][a * MAXN + 1];
        for (int k = 0; k < 3; ++k) ip.ge1[k][a] = (double)G.Ge[k][a * MAXN + 1];
    }
    ip.Pm = h->d_Pm; ip.c0 = h->d_c0; ip.g0 = h->d_g0; ip.dp = h->d_dp; ip.origin = h->d_origin;
    ip.invTk = h->d_invTk; ip.Tpow = h->d_Tpow; ip.invT = h->d_invT; ip.lohi = h->d_lohi; ip.zoff = h->d_zoff;
    ip.invTk2 = h->d_invTk2;
    ip.zt = h->d_zt; ip.chat = h->d_chat; ip.qp = h->d_qp; ip.qn = h->d_qn; ip.phv = h->d_phv; ip.segflags = h->d_segflags;
    ip.stride = h->stride; ip.nseg_pad = h->nseg_pad; ip.nseg = h->nseg; ip.N = h->N; ip.batch = h->batch; ip.s = h->s; ip.dims = h->dims;
    ip.hard = h->wp_mode == TOP_WAYPOINT_HARD; ip.has_box = h->has_box;
    ip.has_vel = h->has_vel && !h->numeric; ip.has_acc = h->has_acc && !h->numeric;
    ip.vmax = h->vmax;
    ip.rot = h->d_rot; ip.planes = h->d_planes; ip.lam3 = h->d_lam3; ip.qpl = h->d_qpl; ip.K = h->K; ip.has_poly = h->has_poly;
}

// rho Pm^ of every segment for the current rho into the staging buffer, by the direct (null-space) inverse in extended
// precision; segments of equal duration (config 3: all of them) share one factorisation.  The rho-independent spectral
// form is only built when rho is going to change.  Polytope corridor (reading A11p): with N_i = sum_k a_k a_k' = V L V'
// the coupled (n m)^2 operator of Eq. 20a splits, in the rotated frame y = V'(p - o_i), into one n x n operator per
// rotated dim with box weight L_d; also staged: V, L and the planes in that frame.
top_status stage_operators(top_solver* h) {
    const int N = h->N, s = h->s, dims = h->dims, n = 2 * s, K = h->K;
    const long long nseg = h->nseg;
    const size_t LS = (size_t)h->stride, NP = (size_t)h->nseg_pad;
    unsigned char* S = h->stage.get();
    double* Pm_st = reinterpret_cast<double*>(S);
    double* rot_st = reinterpret_cast<double*>(S + h->off_rot);
    double* pl_st = reinterpret_cast<double*>(S + h->off_planes);
    double* lam_st = reinterpret_cast<double*>(S + h->off_lam3);
    const double* durations = h->h_T.data();
    gram_tables(s);     // built before the worker threads start
    std::atomic<int> bad_operator(0);
    const bool box = h->has_box, vel = h->has_vel, acc = h->has_acc, poly = h->has_poly;
    const int mode = (int)h->wp_mode;
    const xreal rho = (xreal)h->rho;
    auto do_segments = [&](long long g0, long long g1) {
        try {
            xreal Pm[MAXN * MAXN];
            double cached_T = -1.0;
            int cached_mask = -1;
            for (long long g = g0; g < g1; ++g) {
                const double Td = durations[g];
                // wide consensus: the rows of orders >= s exist at every boundary except the two trajectory ends (A1)
                const int wmask = h->wide ? ((g % N != 0 ? 1 : 0) | (g % N != N - 1 ? 2 : 0)) : 0;
                if (!poly) {
                    if (Td != cached_T || wmask != cached_mask) {
                        if (!build_operator(s, (xreal)Td, rho, box, vel, acc, mode, nullptr, nullptr, Pm, nullptr, 2, wmask)) { bad_operator.store(1); return; }
                        cached_T = Td; cached_mask = wmask;
                    }
                    for (int lane = 0; lane < n; ++lane)
                        for (int b = 0; b < n; ++b) Pm_st[(size_t)b * LS + (size_t)g * LANES + lane] = (double)(rho * Pm[lane * MAXN + b]);
                    continue;
                }
                const double* pl = h->h_planes.data() + (size_t)g * K * (dims + 1);
                xreal Nm[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0}, V[9], lam[3];
                for (int k = 0; k < K; ++k)
                    for (int d = 0; d < dims; ++d) for (int e = 0; e < dims; ++e) Nm[d * 3 + e] += (xreal)pl[k * (dims + 1) + d] * (xreal)pl[k * (dims + 1) + e];
                eigen3(Nm, V, lam);
                const long long b_ = g / N, i_ = g % N;
                const double* o = h->h_wp.data() + ((size_t)b_ * (N + 1) + i_) * dims;      // origin of the local frame
                for (int q = 0; q < 9; ++q) rot_st[(size_t)q * NP + g] = (double)V[q];
                for (int d = 0; d < 3; ++d) {
                    lam_st[(size_t)d * NP + g] = (double)lam[d];
                    if (!build_operator(s, (xreal)Td, rho, true, vel, acc, mode, nullptr, nullptr, Pm, nullptr, lam[d], wmask)) { bad_operator.store(1); return; }
                    for (int lane = 0; lane < n; ++lane)
                        for (int b = 0; b < n; ++b)
                            Pm_st[((size_t)d * MAXN + b) * LS + (size_t)g * LANES + lane] = (double)(rho * Pm[lane * MAXN + b]);
                }
                for (int k = 0; k < K; ++k) {
                    xreal ao = 0;
                    for (int d = 0; d < dims; ++d) ao += (xreal)pl[k * (dims + 1) + d] * (xreal)o[d];
                    for (int e = 0; e < 3; ++e) {
                        xreal v = 0;
                        for (int d = 0; d < dims; ++d) v += V[d * 3 + e] * (xreal)pl[k * (dims + 1) + d];
                        pl_st[((size_t)k * 4 + e) * NP + g] = (double)v;                    // a'_k = V'a_k
                    }
                    pl_st[((size_t)k * 4 + 3) * NP + g] = (double)((xreal)pl[k * (dims + 1) + dims] - ao);   // b'_k = b_k - a_k'o_i
                }
            }
        } catch (...) { bad_operator.store(2); }
    };
    parallel_segments(nseg, do_segments);
    if (bad_operator.load() == 2) return fail(h, TOP_E_NOMEM, "host precompute failed");
    if (bad_operator.load()) return fail(h, TOP_E_INVALID, "x-update operator is not positive definite (check durations / rho)");
    if (poly) h->h_rot.assign(rot_st, rot_st + 9 * NP);
    return TOP_OK;
}

// The per-problem part of top_create, shared with top_reset: host precompute of the x-update operator (Eq. 20a first
// bracket; per segment, extended precision, for the current rho), ONE host-to-device copy of the operator rows and of
// the caller's arrays, then the init kernel (per-lane constants and iterate 0, reading A9).  Asynchronous.
top_status fill_problem(top_solver* h, const double* waypoints, const double* durations, const double* start_derivs,
                        const double* end_derivs, const top_constraints* cons, PhaseTimer* pt) {
    const int N = h->N, s = h->s, dims = h->dims, batch = h->batch;
    const long long nseg = h->nseg;
    unsigned char* S = h->stage.get();
    std::memcpy(S + h->off_wp, waypoints, (size_t)batch * (N + 1) * dims * 8);
    std::memcpy(S + h->off_T, durations, (size_t)nseg * 8);
    if (h->has_box) {
        std::memcpy(S + h->off_lo, cons->box_lo, (size_t)nseg * dims * 8);
        std::memcpy(S + h->off_hi, cons->box_hi, (size_t)nseg * dims * 8);
    }
    h->have_sd = start_derivs != nullptr; h->have_ed = end_derivs != nullptr;
    if (start_derivs) std::memcpy(S + h->off_sd, start_derivs, (size_t)batch * (s - 1) * dims * 8);
    if (end_derivs) std::memcpy(S + h->off_ed, end_derivs, (size_t)batch * (s - 1) * dims * 8);
    h->h_wp.assign(waypoints, waypoints + (size_t)batch * (N + 1) * dims);
    h->h_T.assign(durations, durations + nseg);
    if (h->has_poly) h->h_planes.assign(cons->planes, cons->planes + (size_t)nseg * h->K * (dims + 1));
    const GramTables& G = gram_tables(s);
    if (pt) pt->mark("staging copies");

    if (h->has_poly) {       // three operators per segment in a rotated frame: host precompute (stage_operators)
        top_status so = stage_operators(h);
        if (pt) pt->mark("host precompute");
        if (so != TOP_OK) return so;
        CU(cudaMemcpyAsync(h->d_upload, S, h->upload_bytes, cudaMemcpyHostToDevice, h->stream), "H2D problem data");
    } else {
        // the operator is computed on the device (precompute_operator_kernel, double-double): what goes up is the caller's
        // arrays and 14 KB of Gram tables -- not 8 operator rows per lane
        GramDD* gd = reinterpret_cast<GramDD*>(S + h->off_gram);
        const xreal* tabs[GRAM_TABLES] = {G.Q1, G.Gc[0], G.Gc[1], G.Gc[2], G.Gc[3], G.Ge[0], G.Ge[1], G.Ge[2],
                                          G.Gw[0][0], G.Gw[0][1], G.Gw[0][2], G.Gw[1][0], G.Gw[1][1], G.Gw[1][2]};
        for (int t = 0; t < GRAM_TABLES; ++t)
            for (int i = 0; i < MAXN * MAXN; ++i) {
                const double hi = (double)tabs[t][i];
                gd->hi[t][i] = hi; gd->lo[t][i] = (double)(tabs[t][i] - (xreal)hi);
            }
        CU(cudaMemcpyAsync(h->d_upload + h->off_gram, S + h->off_gram, h->upload_bytes - h->off_gram, cudaMemcpyHostToDevice, h->stream), "H2D problem data");
        PrecompParams pp;
        std::memset(&pp, 0, sizeof pp);
        pp.gram = reinterpret_cast<const GramDD*>(h->d_upload + h->off_gram);
        pp.durations = reinterpret_cast<const double*>(h->d_upload + h->off_T);
        pp.Pm = h->d_Pm; pp.stride = h->stride; pp.nseg = h->nseg; pp.N = h->N; pp.s = h->s;
        pp.hard = h->wp_mode == TOP_WAYPOINT_HARD; pp.box = h->has_box; pp.wide = h->wide;
        pp.vel = h->has_vel && !h->numeric; pp.acc = h->has_acc && !h->numeric;      // NumericSolve: H0 is the quadratic part only
        pp.rho = h->rho; pp.bad = h->d_abort + 1;
        CU(launch_precompute_operator(pp, h->stream), "operator precompute launch");
        h->launches += 1;
        if (pt) pt->mark("operator kernel launch");
    }
    InitParams ip;
    std::memset(&ip, 0, sizeof ip);
    fill_init_params(h, ip);
    CU(launch_init(ip, h->dtype, h->stream), "init kernel launch");
    h->launches += 1;
    h->have_spectral = false;
    h->have_residuals = false;
    std::fill(h->h_res.begin(), h->h_res.end(), std::numeric_limits<double>::quiet_NaN());
    h->iter = 0;
    if (pt) pt->mark("upload + init kernel");
    return TOP_OK;
}

// W, lambda of the rho-independent spectral form (build_spectral) on the device: needed only when rho changes
// (top_set_rho, Eq. 24, a snapshot with another rho).  Host eigen-solves in extended precision; synchronises.
top_status ensure_spectral(top_solver* h) {
    if (h->have_spectral) return TOP_OK;
    const int s = h->s, n = 2 * s;
    const size_t LS = (size_t)h->stride, NP = (size_t)h->nseg_pad;
    std::vector<double> Wv, lamv;
    try { Wv.assign(MAXN * LS, 0.0); lamv.assign(MAXN * NP, 0.0); } catch (...) { return fail(h, TOP_E_NOMEM, "host allocation failed"); }
    gram_tables(s);
    std::atomic<int> bad(0);
    const double* durations = h->h_T.data();
    auto work = [&](long long g0, long long g1) {
        try {
            Spectral SP;
            double cached_T = -1.0;
            int cached_mask = -1;
            const xreal zero3[3] = {0, 0, 0};
            for (long long g = g0; g < g1; ++g) {
                const int wmask = h->wide ? ((g % h->N != 0 ? 1 : 0) | (g % h->N != h->N - 1 ? 2 : 0)) : 0;
                if (durations[g] != cached_T || wmask != cached_mask) {
                    // (NumericSolve branch: the operator is the quadratic part only, the balls are not in it)
                    if (!build_spectral(s, (xreal)durations[g], h->has_box, h->has_vel && !h->numeric, h->has_acc && !h->numeric, (int)h->wp_mode, zero3, SP, wmask)) { bad.store(1); return; }
                    cached_T = durations[g]; cached_mask = wmask;
                }
                for (int i = 0; i < MAXN; ++i) lamv[(size_t)i * NP + g] = i < SP.q ? (double)SP.lam[i] : 0.0;
                for (int lane = 0; lane < n; ++lane)
                    for (int i = 0; i < MAXN; ++i) Wv[(size_t)i * LS + (size_t)g * LANES + lane] = (double)SP.W[lane * MAXN + i];
            }
        } catch (...) { bad.store(2); }
    };
    parallel_segments(h->nseg, work);
    if (bad.load()) return fail(h, bad.load() == 2 ? TOP_E_NOMEM : TOP_E_INVALID, "spectral form of the x-update operator failed");
    CU(cudaMemcpyAsync(h->d_W, Wv.data(), MAXN * LS * 8, cudaMemcpyHostToDevice, h->stream), "H2D spectral form");
    CU(cudaMemcpyAsync(h->d_lam, lamv.data(), MAXN * NP * 8, cudaMemcpyHostToDevice, h->stream), "H2D spectral form");
    CU(cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
    h->have_spectral = true;
    return TOP_OK;
}

}  // namespace

namespace {
// argument checks common to top_create and top_reset (messages go to the handle, or to the thread-local slot)
top_status validate_problem(top_solver* h, int batch, int N, int s, int dims, const double* waypoints, const double* durations,
                            const double* start_derivs, const double* end_derivs, const top_constraints* cons, double rho,
                            bool* has_box, bool* has_vel, bool* has_acc, int* num_planes = nullptr) {
    if (num_planes) *num_planes = 0;
    if (!waypoints || !durations) return fail(h, TOP_E_INVALID, "waypoints and durations are required");
    if (!(rho > 0) || !std::isfinite(rho)) return fail(h, TOP_E_INVALID, "rho must be finite and > 0");
    const long long nseg = (long long)batch * N;
    for (long long i = 0; i < (long long)batch * (N + 1) * dims; ++i)
        if (!std::isfinite(waypoints[i])) return fail(h, TOP_E_INVALID, "non-finite waypoint");
    for (long long i = 0; i < nseg; ++i)
        if (!(durations[i] > 0) || !std::isfinite(durations[i])) return fail(h, TOP_E_INVALID, "durations must be finite and > 0");
    for (int e = 0; e < 2; ++e) {
        const double* dv = e ? end_derivs : start_derivs;
        if (dv) for (long long i = 0; i < (long long)batch * (s - 1) * dims; ++i)
            if (!std::isfinite(dv[i])) return fail(h, TOP_E_INVALID, "non-finite end state");
    }
    *has_box = *has_vel = *has_acc = false;
    if (cons && cons->samples != 0) {
        if (cons->samples < 0) return fail(h, TOP_E_INVALID, "constraints.samples must be >= 0");
        if (cons->samples != MS) return fail(h, TOP_E_UNSUPPORTED, "constraints.samples: this build evaluates the inequality sets at 8 samples per segment");
        if ((cons->box_lo == nullptr) != (cons->box_hi == nullptr)) return fail(h, TOP_E_INVALID, "box_lo and box_hi go together");
        *has_box = cons->box_lo != nullptr;
        if (*has_box) for (long long i = 0; i < nseg * dims; ++i) {
            if (!std::isfinite(cons->box_lo[i]) || !std::isfinite(cons->box_hi[i]) || !(cons->box_lo[i] < cons->box_hi[i]))
                return fail(h, TOP_E_INVALID, "box needs finite lo < hi");
        }
        if (std::isnan(cons->vmax) || std::isnan(cons->amax) || std::isinf(cons->vmax) || std::isinf(cons->amax))
            return fail(h, TOP_E_INVALID, "vmax/amax must be finite");
        *has_vel = cons->vmax > 0;
        *has_acc = cons->amax > 0;
        if (cons->num_planes != 0) {       // general polytope corridor (reading A11p)
            if (cons->num_planes < 0 || !cons->planes) return fail(h, TOP_E_INVALID, "num_planes must be >= 0 and planes non-NULL");
            if (*has_box) return fail(h, TOP_E_INVALID, "a polytope corridor replaces the box: box_lo / box_hi must be NULL");
            if (cons->num_planes > KMAX) return fail(h, TOP_E_UNSUPPORTED, "more than 16 planes per segment");
            const long long cnt = nseg * cons->num_planes;
            for (long long i = 0; i < cnt; ++i) {
                const double* pl = cons->planes + i * (dims + 1);
                double n2 = 0;
                for (int d = 0; d <= dims; ++d) { if (!std::isfinite(pl[d])) return fail(h, TOP_E_INVALID, "non-finite plane"); if (d < dims) n2 += pl[d] * pl[d]; }
                if (!(n2 > 0)) return fail(h, TOP_E_INVALID, "a plane normal is zero");
            }
            if (num_planes) *num_planes = cons->num_planes;
            else return fail(h, TOP_E_INVALID, "polytope corridor not expected here");
        }
    }
    return TOP_OK;
}

}  // namespace

// =================================================================================== top_create

namespace {
struct HandleGuard {        // destroys a half-built solver on every early return / exception of top_create
    top_solver* h = nullptr;
    ~HandleGuard() { if (h) top_destroy(h); }
};

top_status create_impl(top_solver** out, int32_t batch, int32_t N, int32_t s, int32_t dims, top_dtype dtype,
                       const double* waypoints, const double* durations, const double* start_derivs,
                       const double* end_derivs, const top_constraints* cons, double rho, const top_options* opt) {
    top_solver* h = nullptr;   // errors before the handle exists go to the thread-local message
    HandleGuard guard;
    PhaseTimer pt;
    if (!out) return fail(h, TOP_E_INVALID, "out is NULL");
    *out = nullptr;
    if (batch < 1 || N < 1) return fail(h, TOP_E_INVALID, "batch and N must be >= 1");
    if (s != 3 && s != 4) return fail(h, TOP_E_INVALID, "s must be 3 (jerk) or 4 (snap)");
    if (dims < 1 || dims > 3) return fail(h, TOP_E_INVALID, "dims must be 1..3");
    if (dtype != TOP_F64 && dtype != TOP_F32) return fail(h, TOP_E_INVALID, "unknown dtype");
    const long long nseg = (long long)batch * N;
    if (nseg > (1ll << 28)) return fail(h, TOP_E_UNSUPPORTED, "more than 2^28 segments");
    bool has_box = false, has_vel = false, has_acc = false;
    int num_planes = 0;
    {
        top_status vs = validate_problem(nullptr, batch, N, s, dims, waypoints, durations, start_derivs, end_derivs, cons, rho,
                                         &has_box, &has_vel, &has_acc, &num_planes);
        if (vs != TOP_OK) return vs;
    }
    top_options o;
    std::memset(&o, 0, sizeof o);
    o.check_every = 32; o.device = -1; o.max_iter = 1000000;
    if (opt) {
        if (opt->struct_size < 8 || opt->struct_size > sizeof(top_options)) return fail(h, TOP_E_INVALID, "options.struct_size");
        top_options in;
        std::memset(&in, 0, sizeof in);
        std::memcpy(&in, opt, opt->struct_size);
        o.flags = in.flags;
        if (opt->struct_size >= offsetof(top_options, device)) if (in.check_every > 0) o.check_every = in.check_every;
        if (opt->struct_size >= offsetof(top_options, max_iter)) o.device = in.device;
        if (opt->struct_size >= offsetof(top_options, cuda_stream)) if (in.max_iter > 0) o.max_iter = in.max_iter;
        if (opt->struct_size >= offsetof(top_options, segs_per_cta)) o.cuda_stream = in.cuda_stream;
        if (opt->struct_size >= offsetof(top_options, lanes_per_segment)) o.segs_per_cta = in.segs_per_cta;
        if (opt->struct_size >= offsetof(top_options, adapt_mu)) o.lanes_per_segment = in.lanes_per_segment;
        if (opt->struct_size >= sizeof(top_options)) {
            o.adapt_mu = in.adapt_mu; o.adapt_tau_incr = in.adapt_tau_incr; o.adapt_tau_decr = in.adapt_tau_decr;
        }
    }
    const uint32_t mode = o.flags & TOP_WAYPOINT_MASK;
    if (mode > TOP_WAYPOINT_FREE) return fail(h, TOP_E_INVALID, "unknown waypoint mode");
    if (o.segs_per_cta < 0 || (o.segs_per_cta % 4) != 0) return fail(h, TOP_E_INVALID, "segs_per_cta must be a multiple of 4");
    if (o.lanes_per_segment != 0 && o.lanes_per_segment != 4 && o.lanes_per_segment != 8)
        return fail(h, TOP_E_INVALID, "lanes_per_segment must be 0 (choose), 4 or 8");
    for (double v : {o.adapt_mu, o.adapt_tau_incr, o.adapt_tau_decr})
        if (v != 0 && !(v > 1 && std::isfinite(v))) return fail(h, TOP_E_INVALID, "adapt_mu / adapt_tau_* must be > 1 (or 0 = default)");

    pt.mark("validation");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(h, TOP_E_CUDA, "no CUDA device: this library has no CPU path");
    }
    int dev = o.device;
    if (dev < 0) { if (cudaGetDevice(&dev) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaGetDevice failed"); }
    if (dev >= ndev) return fail(h, TOP_E_INVALID, "device ordinal out of range");
    if (cudaSetDevice(dev) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");

    h = new (std::nothrow) top_solver();
    if (!h) return fail(nullptr, TOP_E_NOMEM, "host allocation failed");
    guard.h = h;
    // from here on errors are reported through the thread-local message and the guard destroys the handle
#define CREATE_FAIL(st_) do { top_status s__ = (st_); g_create_error = h->err; return s__; } while (0)
    h->batch = batch; h->N = N; h->s = s; h->n = 2 * s; h->dims = dims; h->dtype = (int)dtype;
    h->opt_flags = o.flags; h->rho = rho; h->check_every = o.check_every; h->max_iter = o.max_iter;
    h->device = dev; h->stream = (cudaStream_t)o.cuda_stream; h->user_segs = o.segs_per_cta;
    h->has_box = has_box; h->has_vel = has_vel; h->has_acc = has_acc;
    h->has_poly = num_planes > 0; h->K = num_planes; h->pm_dims = h->has_poly ? 3 : 1;
    h->constrained = has_box || has_vel || has_acc || h->has_poly;
    h->vmax = has_vel ? cons->vmax : 0; h->amax = has_acc ? cons->amax : 0;
    h->wp_mode = mode;
    h->wide = (o.flags & TOP_CONSENSUS_WIDE) != 0;
    // test hook (include/top.h, "Environment variables"): start the mailbox sequence counter near the end of its 32-bit space
    if (const char* e = std::getenv("TOP_TEST_SEQ_START")) h->seq_counter = std::strtoull(e, nullptr, 0);
    h->numeric = (o.flags & TOP_XUPDATE_NUMERIC) != 0;
    if (h->numeric && (dtype != TOP_F64 || h->has_poly || h->wide))
        CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "TOP_XUPDATE_NUMERIC: TOP_F64 only, no polytope corridor, no TOP_CONSENSUS_WIDE"));
    h->nc = h->wide ? 2 * s - 1 : s;
    if (o.adapt_mu > 0) h->adapt_mu = o.adapt_mu;
    if (o.adapt_tau_incr > 0) h->adapt_incr = o.adapt_tau_incr;
    if (o.adapt_tau_decr > 0) h->adapt_decr = o.adapt_tau_decr;
    h->kflags = (has_box ? KF_BOX : 0) | (has_vel ? KF_VEL : 0) | (has_acc ? KF_ACC : 0) |
                (mode == TOP_WAYPOINT_PINNED_Z ? KF_PIN_POS : 0) | (h->has_poly ? KF_POLY : 0) | (h->wide ? KF_WIDE : 0);
    h->nseg = nseg; h->nseg_pad = (nseg + 31) / 32 * 32; h->stride = h->nseg_pad * LANES;

    // ---- launch plan: waves of whole trajectories, each wave resident on chip for all its sweeps
    int smem_optin = 0;
    if (cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
        CREATE_FAIL(fail(h, TOP_E_CUDA, "cudaDeviceGetAttribute failed"));
    int coop = 0;
    cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev);
    if (!coop) CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "device lacks cooperative launch"));
    if (h->numeric) {
        // NumericSolve branch: the state lives in device memory and a sweep is two plain launches (no on-chip capacity,
        // no cooperative grid): one "wave" that only describes the x-update launch for top_launch_info
        top_solver::Wave w;
        w.seg_begin = 0; w.seg_end = nseg; w.own_begin = 0; w.own_end = nseg; w.kflags = 0;
        w.segs_per_cta = 64; w.ctas = (int)((nseg + 63) / 64); w.threads = 64; w.smem = 0; w.cluster = false;
        h->waves.push_back(w);
        h->lanes = 8; h->mma = false; h->max_ctas = h->num_sms;
    } else {
    // fp32: 8 lanes per segment unless told otherwise; 4 lanes (twice the registers per thread, two samples per lane) win
    // once every SM is full of segments (measured on config 5: 4.1e9 vs 3.3e9 segment-iterations/s)
    h->lanes = o.lanes_per_segment ? o.lanes_per_segment : 8;
    if (!o.lanes_per_segment && dtype == TOP_F32 && nseg >= (long long)h->num_sms * 96) h->lanes = 4;
    // fp64: the 4-lane kernel runs its constant-matrix contractions on the tensor cores (top_kernels_mma.cu); it wins
    // whenever there are inequality constraints (config 2: 1.55 vs 1.74 us per sweep, config 4: 3.0 vs 4.6) and for
    // unconstrained chains once an SM holds more than a few warps (N = 10^4: 1.6 vs 2.1-2.3); short unconstrained chains
    // (configs 1, 3) stay on the 8-lane kernel (0.64 vs 0.85, 1.42 vs 1.57)
    if (!o.lanes_per_segment && dtype == TOP_F64 && ((has_box || has_vel || has_acc) || nseg >= (long long)h->num_sms * 32)) h->lanes = 4;
    if (!o.lanes_per_segment && (h->has_poly || h->wide)) h->lanes = 4;
    // short chains (the paper's regime, tens to a thousand segments): at most 16 CTAs run as ONE thread-block cluster and
    // exchange their boundary rows through distributed shared memory, which costs 0-0.25 us per sweep instead of the
    // 0.45-0.8 us of the L2 mailbox between 25-125 small CTAs (profiles/r2_small_configs_latency.md: config 2 1.60 -> 1.38 us,
    // config 3 1.41 -> 1.24 us; fp32: config 3 1.30 -> 1.16 us).  It pays as long as the per-CTA share stays small: <= 32 segments per CTA with inequality
    // sets, <= 64 without.  Chains of <= 16 segments stay on one CTA.
    int plan_segs = 0;
    if (!o.lanes_per_segment && !o.segs_per_cta && (o.flags & TOP_SYNC_MASK) == TOP_SYNC_AUTO &&
        !(o.flags & TOP_KERNEL_NO_MMA) && !h->has_poly) {
        const bool cons_any = has_box || has_vel || has_acc;
        // (chains that the SPLIT instantiation can take run best at ONE octet per CTA, three warps each: config 2 1.35 -> 1.02 us)
        const long long per_cta_max = cons_any ? 32 : 64, per_cta_min = cons_any ? (split_supported(h->kflags, dtype) ? 8 : 16) : 32;
        if (nseg > 16 && nseg <= 16 * per_cta_max) {
            h->lanes = 4;
            plan_segs = (int)std::max<long long>(per_cta_min, round_up((int)((nseg + 15) / 16), 8));
        }
    }
    if (h->lanes == 4 && (o.flags & TOP_KERNEL_NO_MMA))
        CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "TOP_KERNEL_NO_MMA: the shuffle form of the 4-lane kernel was removed (use lanes_per_segment = 8 for a kernel without tensor-core contractions)"));
    h->mma = h->lanes == 4;
    if (h->wide && !(h->mma && dtype == TOP_F64))
        CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "TOP_CONSENSUS_WIDE runs on the fp64 tensor-core kernel only (TOP_F64, lanes_per_segment 0 or 4, no TOP_KERNEL_NO_MMA)"));
    if (h->has_poly && !(h->mma && dtype == TOP_F64))
        CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "polytope corridors run on the fp64 tensor-core kernel only (TOP_F64, lanes_per_segment 0 or 4, no TOP_KERNEL_NO_MMA)"));
    const int segs_max = max_segs_per_cta(h->dtype, s, h->constrained, h->lanes, h->mma, (size_t)smem_optin - 8192, h->has_poly, h->wide);
    if (segs_max < 4) CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "shared memory too small for one warp of segments"));
    h->max_ctas = h->num_sms;
    if (plan_segs > segs_max) plan_segs = 0;
    const long long capacity = (long long)h->max_ctas * std::min(segs_max, h->user_segs ? h->user_segs : segs_max);
    auto make_wave = [&](long long r0, long long r1, long long o0, long long o1, uint32_t kf) -> bool {
        top_solver::Wave w;
        w.seg_begin = r0; w.seg_end = r1; w.own_begin = o0; w.own_end = o1; w.kflags = kf;
        const long long cnt = r1 - r0;
        int segs = h->user_segs ? h->user_segs : plan_segs ? plan_segs : round_up((int)((cnt + h->max_ctas - 1) / h->max_ctas), 4);
        segs = std::max(4, std::min(segs, segs_max));
        w.segs_per_cta = segs;
        w.ctas = (int)((cnt + segs - 1) / segs);
        w.threads = (segs * h->lanes + 31) / 32 * 32;
        w.smem = kernel_smem(h->dtype, s, h->constrained, h->lanes, h->mma, segs, h->has_poly, h->wide);
        w.cluster = false;
        if (w.ctas > h->max_ctas) return false;
        h->waves.push_back(w);
        return true;
    };
    if ((long long)N > capacity && (h->has_poly || h->wide))
        CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "a trajectory with a polytope corridor or with TOP_CONSENSUS_WIDE must fit on chip (streaming is not built for it)"));
    if ((long long)N > capacity) {
        // one trajectory does not fit on chip: stream the whole segment index space in pieces with halos
        h->streaming = true;
        h->halo = (int)std::min<long long>(64, std::max<long long>(1, capacity / 8));
        const long long own_max = capacity - 2 * h->halo;
        if (own_max < 4) CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "on-chip capacity too small to stream this trajectory"));
        const long long npieces = (nseg + own_max - 1) / own_max;
        const long long own = (nseg + npieces - 1) / npieces;
        for (long long o0 = 0; o0 < nseg; o0 += own) {
            const long long o1 = std::min(nseg, o0 + own);
            const long long r0 = std::max<long long>(0, o0 - h->halo), r1 = std::min(nseg, o1 + h->halo);
            if (!make_wave(r0, r1, o0, o1, (r0 > 0 ? KF_OPEN_LEFT : 0) | (r1 < nseg ? KF_OPEN_RIGHT : 0)))
                CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "launch plan exceeds one CTA per SM"));
        }
    } else {
        const long long traj_cap = capacity / N;
        const long long nwaves = (batch + traj_cap - 1) / traj_cap;
        const long long per_wave = (batch + nwaves - 1) / nwaves;
        for (long long b0 = 0; b0 < batch; b0 += per_wave) {
            const long long b1 = std::min<long long>(batch, b0 + per_wave);
            if (!make_wave(b0 * N, b1 * N, b0 * N, b1 * N, 0))
                CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "launch plan exceeds one CTA per SM"));
        }
    }
    for (const auto& w : h->waves) {
        int per_sm = 0;
        cudaError_t e = h->mma ? sweep_kernel_limits_mma(h->dtype, s, h->kflags, w.threads, w.smem, &per_sm)
                               : sweep_kernel_limits(h->dtype, s, h->constrained, h->lanes, w.threads, w.smem, &per_sm);
        if (e != cudaSuccess) CREATE_FAIL(cuda_fail(h, e, "occupancy query"));
        if (per_sm < 1) CREATE_FAIL(fail(h, TOP_E_UNSUPPORTED, "sweep kernel does not fit an SM"));
    }
    // short chains (the paper's regime: tens to a few hundred segments): when a wave is at most 16 CTAs it runs as ONE
    // thread-block cluster and the boundary rows travel through distributed shared memory instead of the L2 mailbox
    // (TOP_SYNC_AUTO only; the explicit sync modes keep the mailbox so that the two can be compared)
    if (h->mma && !h->streaming && (o.flags & TOP_SYNC_MASK) == TOP_SYNC_AUTO)
        for (auto& w : h->waves) {
            int ncl = 0;
            if (w.ctas >= 2 && w.ctas <= 16 &&
                sweep_cluster_limits_mma(h->dtype, s, h->kflags, w.ctas, w.threads, w.smem, &ncl) == cudaSuccess && ncl >= 1)
                w.cluster = true;
            cudaGetLastError();
        }

    }
    pt.mark("launch plan");

    // ---- memory: one device arena, one host staging buffer
    const size_t LS = (size_t)h->stride, NP = (size_t)h->nseg_pad;
    const size_t rb = real_bytes(h);
    const int n = 2 * s;
    struct Carve { size_t off = 0; size_t take(size_t bytes) { const size_t o = off; off = (off + bytes + 255) & ~(size_t)255; return o; } } cv;
    // (a) the region that mirrors the staging buffer: operator rows, then the caller's arrays as they are
    const size_t o_Pm = cv.take(h->pm_dims * MAXN * LS * 8);
    h->off_rot = cv.take(h->has_poly ? 9 * NP * 8 : 0);
    h->off_planes = cv.take(h->has_poly ? (size_t)h->K * 4 * NP * 8 : 0);
    h->off_lam3 = cv.take(h->has_poly ? 3 * NP * 8 : 0);
    h->off_gram = cv.take(h->has_poly ? 0 : sizeof(GramDD));
    h->off_wp = cv.take((size_t)batch * (N + 1) * dims * 8);
    h->off_T = cv.take((size_t)nseg * 8);
    h->off_lo = cv.take(has_box ? (size_t)nseg * dims * 8 : 0);
    h->off_hi = cv.take(has_box ? (size_t)nseg * dims * 8 : 0);
    h->off_sd = cv.take((size_t)batch * (s - 1) * dims * 8);
    h->off_ed = cv.take((size_t)batch * (s - 1) * dims * 8);
    h->upload_bytes = cv.off;
    // (b) constants written by the init kernel
    const size_t o_c0 = cv.take(3 * LS * 8), o_W = cv.take(MAXN * LS * 8), o_g0 = cv.take(3 * LS * 8), o_lam = cv.take(MAXN * NP * 8),
                 o_dp = cv.take(3 * NP * 8), o_invTk = cv.take(LS * rb), o_Tpow = cv.take(LS * rb), o_invT = cv.take(2 * NP * rb),
                 o_lohi = cv.take(6 * NP * rb), o_segf = cv.take(NP), o_zoff = cv.take(3 * LS * rb), o_origin = cv.take(3 * NP * 8),
                 o_coef = cv.take((size_t)nseg * dims * n * rb), o_invTk2 = cv.take(h->wide ? LS * rb : 0);
    // (c) iterate: written by the init kernel ...
    const size_t o_zt = cv.take(3 * LS * rb), o_chat = cv.take(3 * LS * rb), o_qp = cv.take(has_box ? 3 * LS * rb : 0),
                 o_qn = cv.take(has_box ? 3 * LS * rb : 0), o_phv = cv.take(has_vel ? 3 * LS * rb : 0),
                 o_qpl = cv.take(h->has_poly ? (size_t)h->K * LS * 8 : 0);
    // ... or zero at iterate 0 (duals), together with the reduction buffers: one memset, repeated by top_reset
    const size_t o_zero = cv.off;
    const size_t o_u = cv.take(3 * LS * rb), o_wv = cv.take(has_vel ? 3 * LS * rb : 0), o_pha = cv.take(has_acc ? 3 * LS * rb : 0),
                 o_wa = cv.take(has_acc ? 3 * LS * rb : 0), o_part = cv.take(NP * 4 * 8), o_res = cv.take((size_t)batch * 4 * 8),
                 o_solve = cv.take(64), o_zt2 = cv.take(h->wide ? 3 * LS * rb : 0), o_u2 = cv.take(h->wide ? 3 * LS * rb : 0),
                 o_yv = cv.take(h->numeric ? LS * 8 : 0), o_ya = cv.take(h->numeric ? LS * 8 : 0), o_bnd = cv.take(h->numeric ? 3 * LS * 8 : 0),
                 o_inner = cv.take(h->numeric ? 16 : 0);      // u64 iteration count + u32 work-queue counter
    size_t o_alt[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    if (h->streaming) {
        const bool on[8] = {true, true, has_box, has_box, has_vel, has_vel, has_acc, has_acc};
        for (int i = 0; i < 8; ++i) o_alt[i] = cv.take(on[i] ? 3 * LS * rb : 0);
    }
    h->zero_bytes = cv.off - o_zero;
    // (d) exchange buffers (zero once; sequence numbers keep growing over the life of the solver)
    const size_t o_Bedge = cv.take((size_t)2 * h->max_ctas * (h->wide ? 48 : 24) * 16), o_resbox = cv.take((size_t)2 * h->max_ctas * 4 * 16),
                 o_sync = cv.take(16), o_abort = cv.take(16);
    h->arena_bytes = cv.off;
    {
        // stream-ordered allocation from the library's pool of this device: a re-planning loop that creates and destroys solvers
        // of the same shape gets its arena back without a trip to the driver (cudaMalloc + cudaFree: 0.8 ms at config 4)
        void* pa = nullptr;
        cudaError_t e = cudaErrorNotSupported;
        if (cudaMemPool_t pool = arena_pool(h->device)) {
            e = cudaMallocFromPoolAsync(&pa, h->arena_bytes, pool, h->stream);
            if (e == cudaSuccess) h->arena_pooled = true; else cudaGetLastError();
        }
        if (e != cudaSuccess) e = cudaMalloc(&pa, h->arena_bytes);
        if (e != cudaSuccess) CREATE_FAIL(fail(h, e == cudaErrorMemoryAllocation ? TOP_E_NOMEM : TOP_E_CUDA, std::string("cudaMalloc: ") + cudaGetErrorString(e)));
        h->arena = static_cast<unsigned char*>(pa);
        if ((e = cudaMemsetAsync(h->arena, 0, h->arena_bytes, h->stream)) != cudaSuccess) CREATE_FAIL(cuda_fail(h, e, "cudaMemsetAsync"));
    }
    unsigned char* A = h->arena;
    h->d_upload = A; h->zero_begin = A + o_zero;
    h->d_Pm = (double*)(A + o_Pm); h->d_c0 = (double*)(A + o_c0); h->d_W = (double*)(A + o_W); h->d_g0 = (double*)(A + o_g0);
    h->d_lam = (double*)(A + o_lam); h->d_dp = (double*)(A + o_dp); h->d_invTk = A + o_invTk; h->d_Tpow = A + o_Tpow;
    h->d_invT = A + o_invT; h->d_lohi = A + o_lohi; h->d_segflags = A + o_segf; h->d_zoff = A + o_zoff;
    h->d_origin = (double*)(A + o_origin); h->d_coef = A + o_coef; h->d_zt = A + o_zt; h->d_chat = A + o_chat;
    h->d_u = A + o_u; h->d_part = (double*)(A + o_part); h->d_res = (double*)(A + o_res); h->d_solve = (double*)(A + o_solve);
    if (has_box) { h->d_qp = A + o_qp; h->d_qn = A + o_qn; }
    if (h->wide) { h->d_invTk2 = A + o_invTk2; h->d_zt2 = A + o_zt2; h->d_u2 = A + o_u2; }
    if (h->numeric) { h->d_yv = (double*)(A + o_yv); h->d_ya = (double*)(A + o_ya); h->d_bnd = (double*)(A + o_bnd); h->d_inner = (unsigned long long*)(A + o_inner); }
    if (h->has_poly) {
        h->d_rot = (double*)(A + h->off_rot); h->d_planes = (double*)(A + h->off_planes); h->d_lam3 = (double*)(A + h->off_lam3);
        h->d_qpl = (double*)(A + o_qpl);
    }
    if (has_vel) { h->d_phv = A + o_phv; h->d_wv = A + o_wv; }
    if (has_acc) { h->d_pha = A + o_pha; h->d_wa = A + o_wa; }
    if (h->streaming) {
        void* cur[8] = {h->d_zt, h->d_u, h->d_qp, h->d_qn, h->d_phv, h->d_wv, h->d_pha, h->d_wa};
        for (int i = 0; i < 8; ++i) if (cur[i]) h->alt[i] = A + o_alt[i];
    }
    h->bedge_bytes = (size_t)2 * h->max_ctas * (h->wide ? 48 : 24) * 16; h->resbox_bytes = (size_t)2 * h->max_ctas * 4 * 16;
    h->d_Bedge = A + o_Bedge; h->d_resbox = A + o_resbox; h->d_sync = A + o_sync; h->d_abort = (int*)(A + o_abort);
    h->stage.reset(new (std::nothrow) unsigned char[h->upload_bytes]);
    if (!h->stage) CREATE_FAIL(fail(h, TOP_E_NOMEM, "host allocation failed"));
    if (h->has_poly) std::memset(h->stage.get(), 0, h->off_wp);      // padded operator rows (and rotation / plane tables) stay zero
    // (without a polytope corridor the operator rows are computed on the device and that part of the buffer is never touched)
    h->h_res.assign((size_t)batch * 4, std::numeric_limits<double>::quiet_NaN());
    pt.mark("memory (1 cudaMalloc)");

    top_status st = fill_problem(h, waypoints, durations, start_derivs, end_derivs, cons, &pt);
    if (st != TOP_OK) CREATE_FAIL(st);
    if (o.flags & TOP_RHO_ADAPTIVE) {        // Eq. 24 will change rho: have the rho-independent form ready
        st = ensure_spectral(h);
        if (st != TOP_OK) CREATE_FAIL(st);
        pt.mark("spectral form");
    }
#undef CREATE_FAIL
    guard.h = nullptr;
    *out = h;
    return TOP_OK;
}
}  // namespace

// Nothing throws across the ABI: allocation failures and anything unexpected come back as a status.
#define TOP_GUARDED(handle, ...)                                                                          \
    try { __VA_ARGS__ }                                                                                   \
    catch (const std::bad_alloc&) { return fail(handle, TOP_E_NOMEM, "out of host memory"); }             \
    catch (const std::exception& e) { return fail(handle, TOP_E_INVALID, std::string("internal error: ") + e.what()); } \
    catch (...) { return fail(handle, TOP_E_INVALID, "internal error"); }

extern "C" TOP_API top_status top_create(top_solver** out, int32_t batch, int32_t N, int32_t s, int32_t dims, top_dtype dtype,
                                 const double* waypoints, const double* durations, const double* start_derivs,
                                 const double* end_derivs, const top_constraints* cons, double rho,
                                 const top_options* opt) {
    if (out) *out = nullptr;
    TOP_GUARDED(nullptr, return create_impl(out, batch, N, s, dims, dtype, waypoints, durations, start_derivs, end_derivs, cons, rho, opt);)
}

// top_reset: a new problem of the same shape on an existing handle (re-planning): same batch,
// N, s, dims, dtype, options and constraint SELECTION; new waypoints, durations, end states, bounds and rho.  No
// allocation, one host-to-device copy, iterate 0 again.
extern "C" TOP_API top_status top_reset(top_solver* h, const double* waypoints, const double* durations, const double* start_derivs,
                                const double* end_derivs, const top_constraints* cons, double rho) {
    if (!h) return TOP_E_INVALID;
    TOP_GUARDED(h,
        bool hb, hv, ha;
        int kp = 0;
        top_status st = validate_problem(h, h->batch, h->N, h->s, h->dims, waypoints, durations, start_derivs, end_derivs, cons, rho, &hb, &hv, &ha, &kp);
        if (st != TOP_OK) return st;
        if (hb != h->has_box || hv != h->has_vel || ha != h->has_acc || kp != h->K)
            return fail(h, TOP_E_INVALID, "top_reset: the constraint selection (box / velocity / acceleration) must be the one the solver was created with");
        if (cudaSetDevice(h->device) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");
        PhaseTimer pt;
        h->rho = rho;
        h->vmax = hv ? cons->vmax : 0; h->amax = ha ? cons->amax : 0;
        CU(cudaMemsetAsync(h->zero_begin, 0, h->zero_bytes, h->stream), "cudaMemsetAsync");
        CU(cudaMemsetAsync(h->d_abort, 0, 2 * sizeof(int), h->stream), "cudaMemsetAsync");
        st = fill_problem(h, waypoints, durations, start_derivs, end_derivs, cons, &pt);
        if (st != TOP_OK) return st;
        if (h->opt_flags & TOP_RHO_ADAPTIVE) st = ensure_spectral(h);
        return st;
    )
}

// =================================================================================== sweeps

namespace {

top_status check_abort(top_solver* h) {
    CU(cudaMemcpyAsync(h->h_abort, h->d_abort, 2 * sizeof(int), cudaMemcpyDeviceToHost, h->stream), "D2H abort flag");
    CU(cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
    if (h->h_abort[1]) return fail(h, TOP_E_INVALID, "x-update operator is not positive definite (check durations / rho)");
    if (h->h_abort[0]) return fail(h, TOP_E_CUDA, "inter-CTA barrier timed out inside the sweep kernel");
    return TOP_OK;
}

uint32_t sync_flag(const top_solver* h) {
    const uint32_t m = h->opt_flags & TOP_SYNC_MASK;
    if (m == TOP_SYNC_GRID) return 0;
    if (m == TOP_SYNC_NEIGHBOUR) return KF_NEIGHBOUR_SYNC;            // CTA barrier + mailbox
    return KF_NEIGHBOUR_SYNC | KF_PAIRWISE;   // TOP_SYNC_AUTO / TOP_SYNC_PAIRWISE: warp-pair barriers + mailbox
}

// k sweeps on every wave, then the per-trajectory residual reduction.  Asynchronous.
struct InKernelSolve { int check_every; int rd_sel; int adaptive; double tol; };

top_status run_sweeps(top_solver* h, int64_t k, const InKernelSolve* iks = nullptr) {
    if (cudaSetDevice(h->device) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");
    if (h->numeric) {      // NumericSolve branch: x-update kernel + consensus kernel per sweep, state in device memory
        NumParams np;
        std::memset(&np, 0, sizeof np);
        np.Pm = h->d_Pm; np.invT = (const double*)h->d_invT; np.lohi = (const double*)h->d_lohi; np.origin = h->d_origin;
        np.segflags = h->d_segflags; np.zoff = (const double*)h->d_zoff; np.Tpow = (const double*)h->d_Tpow;
        np.zt = (double*)h->d_zt; np.u = (double*)h->d_u; np.qp = (double*)h->d_qp; np.qn = (double*)h->d_qn; np.chat = (double*)h->d_chat;
        np.yv = h->d_yv; np.ya = h->d_ya; np.bnd = h->d_bnd; np.part = h->d_part; np.inner_iters = h->d_inner;
        np.work_counter = reinterpret_cast<unsigned int*>(h->d_inner + 1); np.max_blocks = 3 * h->num_sms;
        np.stride = h->stride; np.nseg_pad = h->nseg_pad; np.nseg = h->nseg; np.s = h->s; np.hard = h->wp_mode == TOP_WAYPOINT_HARD;
        np.flags = h->kflags & (KF_BOX | KF_VEL | KF_ACC | KF_PIN_POS); np.rho = h->rho; np.vmax = h->vmax; np.amax = h->amax;
        for (int64_t i = 0; i < k; ++i) CU(launch_numeric_sweep(np, h->stream), "numeric sweep launch");
        h->launches += 2 * k;
        h->iter += k;
        CU(launch_residual_reduce(h->d_part, h->d_res, h->N, h->batch, h->stream), "residual reduction launch");
        h->launches += 1;
        h->have_residuals = true;
        return TOP_OK;
    }
    while (k > 0) {
        // streaming: at most `halo` sweeps per launch (that is how far a piece can run before the staleness of
        // its halo reaches the segments it owns)
        const int kk = (int)std::min<int64_t>(k, h->streaming ? h->halo : (1 << 30));
        for (const auto& w : h->waves) {
            KParams p;
            std::memset(&p, 0, sizeof p);
            p.Pm = h->d_Pm; p.c0 = h->d_c0; p.invTk = h->d_invTk; p.Tpow = h->d_Tpow; p.invT = h->d_invT;
            p.lohi = h->d_lohi; p.segflags = h->d_segflags; p.zoff = h->d_zoff;
            p.zt = h->d_zt; p.u = h->d_u; p.qp = h->d_qp; p.qn = h->d_qn; p.phv = h->d_phv; p.wv = h->d_wv;
            p.pha = h->d_pha; p.wa = h->d_wa; p.chat = h->d_chat;
            if (h->streaming) {
                p.zt_out = h->alt[0]; p.u_out = h->alt[1]; p.qp_out = h->alt[2]; p.qn_out = h->alt[3];
                p.phv_out = h->alt[4]; p.wv_out = h->alt[5]; p.pha_out = h->alt[6]; p.wa_out = h->alt[7];
            } else {
                p.zt_out = p.zt; p.u_out = p.u; p.qp_out = p.qp; p.qn_out = p.qn;
                p.phv_out = p.phv; p.wv_out = p.wv; p.pha_out = p.pha; p.wa_out = p.wa;
            }
            p.own_begin = w.own_begin; p.own_end = w.own_end;
            p.Bedge = h->d_Bedge; p.part = h->d_part;
            p.bar = reinterpret_cast<unsigned long long*>(h->d_sync);
            p.abort_flag = h->d_abort;
            p.stride = h->stride; p.nseg_pad = h->nseg_pad; p.seg_begin = w.seg_begin; p.seg_end = w.seg_end;
            p.segs_per_cta = w.segs_per_cta; p.k_sweeps = kk; p.flags = h->kflags | sync_flag(h) | w.kflags | (w.cluster ? KF_CLUSTER : 0);
            if (iks) {      // device-side stop rule / Eq. 24 (one CTA-wide barrier per sweep: no warp-pair barriers)
                p.flags &= ~KF_PAIRWISE;
                p.check_every = iks->check_every; p.rd_sel = iks->rd_sel; p.adaptive = iks->adaptive; p.tol = iks->tol;
                p.mu = h->adapt_mu; p.tau_incr = h->adapt_incr; p.tau_decr = h->adapt_decr;
                p.q = h->wp_mode == TOP_WAYPOINT_HARD ? h->n - 2 : h->n;
                p.resbox = h->d_resbox; p.solve_out = h->d_solve;
                p.W = h->d_W; p.lam = h->d_lam; p.g0 = h->d_g0; p.dp = h->d_dp;
            }
            p.max_ctas = h->max_ctas; p.rho = h->rho; p.vmax = h->vmax; p.amax = h->amax;
            p.rot = h->d_rot; p.planes = h->d_planes; p.qpl = h->d_qpl; p.qpl_out = h->d_qpl; p.K = h->K;
            p.invTk2 = h->d_invTk2; p.zt2 = h->d_zt2; p.u2 = h->d_u2;
            // mailbox sequence numbers are the low 32 bits of seq_counter + 1 .. + kk.  A slot is valid when it carries the
            // reader's number, and cleared slots carry 0: a launch must never issue 0 nor a number that a slot may still hold
            // from 2^32 sweeps ago, so a launch that would run past 2^32 - 1 starts a new epoch on cleared mailboxes
            if ((h->seq_counter & 0xffffffffull) + (unsigned long long)kk > 0xffffffffull) {
                h->seq_counter = (h->seq_counter | 0xffffffffull) + 1ull;
                CU(cudaMemsetAsync(h->d_Bedge, 0, h->bedge_bytes, h->stream), "cudaMemsetAsync");
                CU(cudaMemsetAsync(h->d_resbox, 0, h->resbox_bytes, h->stream), "cudaMemsetAsync");
            }
            p.seq_base = (unsigned int)(h->seq_counter & 0xffffffffull);
            h->seq_counter += (unsigned long long)kk;
            if (w.ctas > 1 && !(p.flags & KF_NEIGHBOUR_SYNC))
                CU(cudaMemsetAsync(h->d_sync, 0, 8, h->stream), "cudaMemsetAsync");
            CU(h->mma ? launch_sweeps_mma(p, h->dtype, h->s, w.ctas, w.threads, w.smem, h->stream)
                      : launch_sweeps(p, h->dtype, h->s, h->constrained, h->lanes, w.ctas, w.threads, w.smem, h->stream), "sweep kernel launch");
            h->launches += 1;
        }
        if (h->streaming) {       // every piece has written iterate k + kk of its own segments: swap the buffer sets
            std::swap(h->d_zt, h->alt[0]); std::swap(h->d_u, h->alt[1]); std::swap(h->d_qp, h->alt[2]);
            std::swap(h->d_qn, h->alt[3]); std::swap(h->d_phv, h->alt[4]); std::swap(h->d_wv, h->alt[5]);
            std::swap(h->d_pha, h->alt[6]); std::swap(h->d_wa, h->alt[7]);
        }
        k -= kk;
        if (iks) {
            // how far did the kernel get, and with which rho?
            CU(cudaMemcpyAsync(h->h_solve, h->d_solve, 64, cudaMemcpyDeviceToHost, h->stream), "D2H solve result");
            CU(cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
            const int64_t done = (int64_t)h->h_solve[0];
            h->iter += done;
            // the sequence space advances by the sweeps that ran, not by the cap (one wave on this path): a default top_solve
            // reserves max_iter numbers, and a re-planning loop would otherwise walk through 2^32 in a few thousand calls
            if (done >= 0 && done < kk) h->seq_counter -= (unsigned long long)(kk - done);
            if (h->h_solve[2] != h->rho) {      // the kernel refreshed its on-chip operator only: bring the arrays along
                h->rho = h->h_solve[2];
                CU(refresh_operator(h, h->rho), "operator refresh launch");      // (Eq. 24 ran: the spectral form is there)
            }
            if (h->h_solve[1] != 0.0 || done < kk) break;
        } else {
            h->iter += kk;
        }
    }
    CU(launch_residual_reduce(h->d_part, h->d_res, h->N, h->batch, h->stream), "residual reduction launch");
    h->launches += 1;
    h->have_residuals = true;
    return TOP_OK;
}

top_status fetch_residuals(top_solver* h) {
    if (!h->have_residuals) return TOP_OK;
    CU(cudaMemcpyAsync(h->h_res.data(), h->d_res, (size_t)h->batch * 4 * 8, cudaMemcpyDeviceToHost, h->stream), "D2H residuals");
    return check_abort(h);   // synchronises
}

}  // namespace

extern "C" TOP_API top_status top_iterate(top_solver* h, int64_t k) {
    if (!h) return TOP_E_INVALID;
    if (k < 0) return fail(h, TOP_E_INVALID, "k must be >= 0");
    if (k == 0) return TOP_OK;
    return run_sweeps(h, k);
}

namespace { top_status set_rho_impl(top_solver* h, double rho); }
static top_status solve_impl(top_solver* h, double eps, int64_t* iters) {
    if (!h) return TOP_E_INVALID;
    if (!(eps > 0)) return fail(h, TOP_E_INVALID, "eps must be > 0");
    const double tol = (h->opt_flags & TOP_EPS_N_SCALED) ? eps * h->N : eps;
    const int rd_idx = (h->opt_flags & TOP_RD_NORMALISED) ? 2 : 1;
    // (large CTAs run the plain kernel faster than the solve instantiation -- 96-register cap -- so with a sparse
    // test cadence they keep the host loop below)
    if (h->batch == 1 && h->waves.size() == 1 && !h->streaming && !h->has_poly && !h->numeric && (h->lanes == 8 || h->mma) && h->waves[0].ctas <= 160 &&
        (h->waves[0].threads <= 256 || h->check_every < 16)) {
        // one resident trajectory: the stop rule (and Eq. 24) runs inside the kernel, one launch for the whole solve
        InKernelSolve iks;
        iks.check_every = h->check_every; iks.rd_sel = rd_idx; iks.adaptive = (h->opt_flags & TOP_RHO_ADAPTIVE) ? 1 : 0;
        iks.tol = tol;
        if (iks.adaptive) { top_status se = ensure_spectral(h); if (se != TOP_OK) return se; }
        const int64_t it0 = h->iter;
        top_status st = run_sweeps(h, h->max_iter, &iks);
        if (st != TOP_OK) return st;
        st = fetch_residuals(h);
        if (st != TOP_OK) return st;
        if (iters) iters[0] = h->iter - it0;
        const double rp = h->h_res[0], rd = h->h_res[rd_idx];
        if (!std::isfinite(rp) || !std::isfinite(rd)) return fail(h, TOP_E_NONFINITE, "non-finite residual");
        return h->h_solve[1] != 0.0 ? TOP_OK : TOP_NOT_CONVERGED;
    }
    std::vector<int64_t> first(h->batch, -1);
    int64_t done = 0;
    bool all = false;
    while (done < h->max_iter && !all) {
        const int64_t k = std::min<int64_t>(h->check_every, h->max_iter - done);
        top_status st = run_sweeps(h, k);
        if (st != TOP_OK) return st;
        done += k;
        st = fetch_residuals(h);
        if (st != TOP_OK) return st;
        all = true;
        for (int b = 0; b < h->batch; ++b) {
            const double rp = h->h_res[b * 4 + 0], rd = h->h_res[b * 4 + rd_idx];
            if (!std::isfinite(rp) || !std::isfinite(rd)) return fail(h, TOP_E_NONFINITE, "non-finite residual");
            if (rp < tol && rd < tol) { if (first[b] < 0) first[b] = done; }
            else { all = false; first[b] = -1; }     // a trajectory counts as converged only while it stays below
        }
        if (!all && (h->opt_flags & TOP_RHO_ADAPTIVE)) {
            // Eq. 24 with the residuals of this check; one rho for the whole batch: the norms are
            // taken over all trajectories
            double rp2 = 0, rd2 = 0;
            for (int b = 0; b < h->batch; ++b) {
                rp2 += h->h_res[b * 4 + 0] * h->h_res[b * 4 + 0];
                rd2 += h->h_res[b * 4 + rd_idx] * h->h_res[b * 4 + rd_idx];
            }
            const double rp = std::sqrt(rp2), rd = std::sqrt(rd2);
            double rho_new = h->rho;
            if (rp > h->adapt_mu * rd) rho_new = h->rho * h->adapt_incr;
            else if (rd > h->adapt_mu * rp) rho_new = h->rho / h->adapt_decr;
            if (rho_new != h->rho) { st = set_rho_impl(h, rho_new); if (st != TOP_OK) return st; }
        }
    }
    if (iters) for (int b = 0; b < h->batch; ++b) iters[b] = first[b] >= 0 ? first[b] : done;
    return all ? TOP_OK : TOP_NOT_CONVERGED;
}

namespace {
top_status set_rho_impl(top_solver* h, double rho) {
    if (!h) return TOP_E_INVALID;
    if (!(rho > 0) || !std::isfinite(rho)) return fail(h, TOP_E_INVALID, "rho must be finite and > 0");
    if (rho == h->rho) return TOP_OK;
    if (cudaSetDevice(h->device) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");
    const size_t LS = (size_t)h->stride;
    if (h->has_poly) {
        // polytope corridor: three operators per segment; they are rebuilt on the host for the new rho (no spectral form),
        // uploaded, c0^ follows on the device, and the scaled duals (u, w, and v = max(0,-q) of every plane) are rescaled
        const double old = h->rho;
        h->rho = rho;            // (stage_operators builds for h->rho; put back below if anything fails)
        auto enqueue = [&]() -> top_status {
            top_status so = stage_operators(h);
            if (so != TOP_OK) return so;
            CU(cudaMemcpyAsync(h->d_upload, h->stage.get(), h->off_wp, cudaMemcpyHostToDevice, h->stream), "H2D operators");
            InitParams ip;
            std::memset(&ip, 0, sizeof ip);
            fill_init_params(h, ip);
            ip.c0_only = 1;
            CU(launch_init(ip, h->dtype, h->stream), "init kernel launch");
            RescaleParams r;
            r.u = h->d_u; r.qp = nullptr; r.qn = nullptr; r.wv = h->d_wv; r.wa = h->d_wa;
            r.count = 3 * (long long)LS; r.ratio = old / rho; r.qpl = h->d_qpl; r.qpl_count = (long long)h->K * (long long)LS;
            r.u2 = h->d_u2;      // wide consensus: the scaled duals of the second row block as well (null otherwise)
            r.yv = r.ya = nullptr; r.y_count = 0;
            CU(launch_rescale_duals(r, h->dtype, h->stream), "dual rescale launch");
            return TOP_OK;
        };
        const top_status st = enqueue();
        if (st != TOP_OK) { h->rho = old; return st; }      // the handle keeps reporting the rho its device operator has
        h->launches += 2;
        return TOP_OK;
    }
    { top_status se = ensure_spectral(h); if (se != TOP_OK) return se; }      // first change of rho: build W, lambda (host, once)
    CU(refresh_operator(h, rho), "operator refresh launch");      // on the device, from the spectral data
    RescaleParams r;
    r.yv = r.ya = nullptr; r.y_count = 0;
    r.u = h->d_u; r.qp = h->d_qp; r.qn = h->d_qn; r.wv = h->d_wv; r.wa = h->d_wa;
    r.count = 3 * (long long)LS; r.ratio = h->rho / rho; r.qpl = nullptr; r.qpl_count = 0; r.u2 = h->d_u2;
    if (h->numeric) { r.wv = nullptr; r.wa = nullptr; r.yv = h->d_yv; r.ya = h->d_ya; r.y_count = (long long)LS; }      // multipliers of Eq. 17 are scaled duals too
    CU(launch_rescale_duals(r, h->dtype, h->stream), "dual rescale launch");
    h->launches += 1;
    h->rho = rho;
    return TOP_OK;
}
}  // namespace

extern "C" TOP_API double top_get_rho(const top_solver* h) { return h ? h->rho : std::numeric_limits<double>::quiet_NaN(); }

extern "C" TOP_API top_status top_get_residuals(top_solver* h, double* r_primal, double* r_dual, double* r_dual_norm,
                                        double* r_primal_gap) {
    if (!h) return TOP_E_INVALID;
    top_status st = fetch_residuals(h);
    if (st != TOP_OK) return st;
    for (int b = 0; b < h->batch; ++b) {
        if (r_primal) r_primal[b] = h->h_res[b * 4 + 0];
        if (r_dual) r_dual[b] = h->h_res[b * 4 + 1];
        if (r_dual_norm) r_dual_norm[b] = h->h_res[b * 4 + 2];
        if (r_primal_gap) r_primal_gap[b] = h->h_res[b * 4 + 3];
    }
    return TOP_OK;
}

extern "C" TOP_API top_status top_get_coeffs(top_solver* h, void* out, int32_t out_is_device) {
    if (!h) return TOP_E_INVALID;
    if (!out) return fail(h, TOP_E_INVALID, "out is NULL");
    if (cudaSetDevice(h->device) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");
    ConvParams p;
    p.rot = h->d_rot;
    p.chat = h->d_chat; p.invT = h->d_invT; p.origin = h->d_origin; p.out = out_is_device ? out : h->d_coef;
    p.nseg_pad = h->nseg_pad;
    p.stride = h->stride; p.nseg = h->nseg; p.s = h->s; p.dims = h->dims;
    CU(launch_convert(p, h->dtype, h->stream), "coefficient conversion launch");
    h->launches += 1;
    if (!out_is_device) {
        CU(cudaMemcpyAsync(out, h->d_coef, (size_t)h->nseg * h->dims * h->n * real_bytes(h), cudaMemcpyDeviceToHost, h->stream), "D2H coefficients");
        return check_abort(h);
    }
    return TOP_OK;
}

static top_status get_state_impl(top_solver* h, const char* field, double* out, size_t count) {
    if (!h) return TOP_E_INVALID;
    if (!field || !out) return fail(h, TOP_E_INVALID, "field and out are required");
    const std::string f(field);
    const int s = h->s, dims = h->dims, N = h->N, batch = h->batch;
    const size_t LS = (size_t)h->stride;
    std::vector<double> buf;
    top_status st;
    if (f == "z" || f == "u") {
        // consensus rows per boundary: nc = s, or 2s-1 with TOP_CONSENSUS_WIDE (the orders >= s live in the second row block:
        // slot t = start-boundary row of order s + t, slot 4 + t = end-boundary row; rows that do not exist read 0)
        const int nc = h->nc;
        const size_t want = f == "z" ? (size_t)batch * (N + 1) * nc * dims : (size_t)batch * N * 2 * nc * dims;
        if (count != want) return fail(h, TOP_E_INVALID, "top_get_state: count does not match the field");
        if ((st = download_real(h, f == "z" ? h->d_zt : h->d_u, buf, 3 * LS)) != TOP_OK) return st;
        std::vector<double> buf2;
        if (h->wide && (st = download_real(h, f == "z" ? h->d_zt2 : h->d_u2, buf2, 3 * LS)) != TOP_OK) return st;
        for (int b = 0; b < batch; ++b)
            for (int i = 0; i < N; ++i) {
                const size_t g = (size_t)b * N + i;
                for (int side = 0; side < 2; ++side)
                    for (int k = 0; k < nc; ++k)
                        for (int d = 0; d < dims; ++d) {
                            double v = k < s ? buf[(size_t)d * LS + g * LANES + side * s + k]
                                             : buf2[(size_t)d * LS + g * LANES + side * 4 + (k - s)];
                            if (f == "z" && k == 0) v += h->h_wp[((size_t)b * (N + 1) + i) * dims + d];   // local frame (origin p_{i-1}) -> global
                            if (f == "u") out[((g * 2 * nc) + side * nc + k) * dims + d] = v;
                            else if (side == 0) out[(((size_t)b * (N + 1) + i) * nc + k) * dims + d] = v;
                            else if (i == N - 1) out[(((size_t)b * (N + 1) + N) * nc + k) * dims + d] = v;
                        }
            }
        return check_abort(h);
    }
    if (f == "y_v" || f == "y_a") {       // scaled multipliers of Eq. 17 (NumericSolve branch), [batch][N][Ms]
        const size_t want = (size_t)batch * N * MS;
        if (!h->numeric || count != want) return fail(h, TOP_E_INVALID, "top_get_state: count does not match the field (or not a TOP_XUPDATE_NUMERIC solver)");
        buf.resize(LS);
        CU(cudaMemcpyAsync(buf.data(), f == "y_v" ? h->d_yv : h->d_ya, LS * 8, cudaMemcpyDeviceToHost, h->stream), "D2H");
        CU(cudaStreamSynchronize(h->stream), "sync");
        for (size_t g = 0; g < (size_t)batch * N; ++g) for (int j = 0; j < MS; ++j) out[g * MS + j] = buf[g * LANES + j];
        return check_abort(h);
    }
    if (f == "s_poly" || f == "v_poly") {
        const size_t want = (size_t)batch * N * MS * (size_t)h->K;
        if (!h->has_poly || count != want) return fail(h, TOP_E_INVALID, "top_get_state: count does not match the field (or no polytope corridor)");
        buf.resize((size_t)h->K * LS);
        CU(cudaMemcpyAsync(buf.data(), h->d_qpl, buf.size() * 8, cudaMemcpyDeviceToHost, h->stream), "D2H");
        CU(cudaStreamSynchronize(h->stream), "sync");
        for (size_t g = 0; g < (size_t)batch * N; ++g)
            for (int j = 0; j < MS; ++j)
                for (int k = 0; k < h->K; ++k) {
                    const double v = buf[(size_t)k * LS + g * LANES + j];      // Moreau pair: s = max(0,q), v = max(0,-q)
                    out[(g * MS + j) * h->K + k] = f == "s_poly" ? std::max(0.0, v) : std::max(0.0, -v);
                }
        return check_abort(h);
    }
    struct { const char* name; void* ptr; int how; bool on; } tab[] = {
        {"s_pos", h->d_qp, 1, h->has_box}, {"v_pos", h->d_qp, 2, h->has_box},
        {"s_neg", h->d_qn, 1, h->has_box}, {"v_neg", h->d_qn, 2, h->has_box},
        {"phi_v", h->d_phv, 0, h->has_vel}, {"w_v", h->d_wv, 0, h->has_vel},
        {"phi_a", h->d_pha, 0, h->has_acc}, {"w_a", h->d_wa, 0, h->has_acc}};
    for (auto& t : tab) {
        if (f != t.name) continue;
        const size_t want = (size_t)batch * N * MS * dims;
        if (count != want) return fail(h, TOP_E_INVALID, "top_get_state: count does not match the field");
        if (!t.on) { std::fill(out, out + count, 0.0); return TOP_OK; }
        if ((st = download_real(h, t.ptr, buf, 3 * LS)) != TOP_OK) return st;
        for (size_t g = 0; g < (size_t)batch * N; ++g)
            for (int j = 0; j < MS; ++j) {
                double v3[3];
                for (int d = 0; d < 3; ++d) v3[d] = buf[(size_t)d * LS + g * LANES + j];
                if (h->has_poly) {      // ball variables live in the segment's rotated frame: x = V y
                    const double a0 = v3[0], a1 = v3[1], a2 = v3[2];
                    const double* R = h->h_rot.data();
                    const size_t NPp = (size_t)h->nseg_pad;
                    for (int d = 0; d < 3; ++d) v3[d] = R[(d * 3 + 0) * NPp + g] * a0 + R[(d * 3 + 1) * NPp + g] * a1 + R[(d * 3 + 2) * NPp + g] * a2;
                }
                for (int d = 0; d < dims; ++d) {
                    const double v = v3[d];
                    // Moreau pair of the slack projection (Eq. 10 / 20d-e): s = max(0,q), v = max(0,-q)
                    out[(g * MS + j) * dims + d] = t.how == 0 ? v : (t.how == 1 ? std::max(0.0, v) : std::max(0.0, -v));
                }
            }
        return check_abort(h);
    }
    return fail(h, TOP_E_INVALID, "top_get_state: unknown field '" + f + "'");
}

namespace {
struct SnapshotHeader {
    uint64_t magic;
    int64_t nseg, stride, iter;
    int32_t s, dims, dtype, batch;
    uint32_t kflags, have_residuals;
    uint32_t wp_mode, N;
    double rho;
};
constexpr uint64_t SNAP_MAGIC = 0x544f50534e415032ull;     // "TOPSNAP2"
// the device arrays that make up an iterate, in snapshot order (null ones are skipped)
int snapshot_fields(top_solver* h, void** out) {
    void* all[] = {h->d_zt, h->d_u, h->d_qp, h->d_qn, h->d_phv, h->d_wv, h->d_pha, h->d_wa, h->d_chat, h->d_zt2, h->d_u2};
    int n = 0;
    for (void* p : all) if (p) out[n++] = p;
    return n;
}
}  // namespace

extern "C" TOP_API size_t top_snapshot_bytes(const top_solver* hc) {
    if (!hc || hc->numeric) return 0;      // (snapshots are not built for TOP_XUPDATE_NUMERIC: save / restore then reject every size)
    top_solver* h = const_cast<top_solver*>(hc);
    void* f[11];
    const int n = snapshot_fields(h, f);
    return sizeof(SnapshotHeader) + (size_t)n * 3 * (size_t)h->stride * real_bytes(h) + (size_t)h->batch * 4 * 8 +
           (h->has_poly ? (size_t)h->K * (size_t)h->stride * 8 : 0);
}

extern "C" TOP_API top_status top_snapshot_save(top_solver* h, void* host_buf, size_t bytes) {
    if (!h) return TOP_E_INVALID;
    if (h->numeric) return fail(h, TOP_E_UNSUPPORTED, "snapshots are not built for TOP_XUPDATE_NUMERIC");
    if (!host_buf || bytes != top_snapshot_bytes(h)) return fail(h, TOP_E_INVALID, "top_snapshot_save: buffer size must be top_snapshot_bytes()");
    if (cudaSetDevice(h->device) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");
    SnapshotHeader hd;
    std::memset(&hd, 0, sizeof hd);
    hd.magic = SNAP_MAGIC; hd.nseg = h->nseg; hd.stride = h->stride; hd.iter = h->iter; hd.s = h->s; hd.dims = h->dims;
    hd.dtype = h->dtype; hd.batch = h->batch; hd.kflags = h->kflags; hd.have_residuals = h->have_residuals ? 1u : 0u; hd.rho = h->rho;
    hd.wp_mode = h->wp_mode; hd.N = (uint32_t)h->N;
    unsigned char* o = static_cast<unsigned char*>(host_buf);
    std::memcpy(o, &hd, sizeof hd); o += sizeof hd;
    void* f[11];
    const int n = snapshot_fields(h, f);
    const size_t fb = 3 * (size_t)h->stride * real_bytes(h);
    for (int i = 0; i < n; ++i) { CU(cudaMemcpyAsync(o, f[i], fb, cudaMemcpyDeviceToHost, h->stream), "D2H snapshot"); o += fb; }
    CU(cudaMemcpyAsync(o, h->d_res, (size_t)h->batch * 4 * 8, cudaMemcpyDeviceToHost, h->stream), "D2H snapshot");
    o += (size_t)h->batch * 4 * 8;
    if (h->has_poly) CU(cudaMemcpyAsync(o, h->d_qpl, (size_t)h->K * (size_t)h->stride * 8, cudaMemcpyDeviceToHost, h->stream), "D2H snapshot");
    return check_abort(h);
}

static top_status snapshot_restore_impl(top_solver* h, const void* host_buf, size_t bytes) {
    if (!h) return TOP_E_INVALID;
    if (h->numeric) return fail(h, TOP_E_UNSUPPORTED, "snapshots are not built for TOP_XUPDATE_NUMERIC");
    if (!host_buf || bytes != top_snapshot_bytes(h)) return fail(h, TOP_E_INVALID, "top_snapshot_restore: buffer size does not match this solver");
    SnapshotHeader hd;
    std::memcpy(&hd, host_buf, sizeof hd);
    if (hd.magic != SNAP_MAGIC || hd.nseg != h->nseg || hd.stride != h->stride || hd.s != h->s || hd.dims != h->dims ||
        hd.dtype != h->dtype || hd.batch != h->batch || hd.kflags != h->kflags || hd.wp_mode != h->wp_mode ||
        hd.N != (uint32_t)h->N || !(hd.rho > 0))
        return fail(h, TOP_E_INVALID, "top_snapshot_restore: the snapshot belongs to a different problem");
    if (cudaSetDevice(h->device) != cudaSuccess) return fail(h, TOP_E_CUDA, "cudaSetDevice failed");
    const unsigned char* o = static_cast<const unsigned char*>(host_buf) + sizeof hd;
    void* f[11];
    const int n = snapshot_fields(h, f);
    const size_t fb = 3 * (size_t)h->stride * real_bytes(h);
    for (int i = 0; i < n; ++i) { CU(cudaMemcpyAsync(f[i], o, fb, cudaMemcpyHostToDevice, h->stream), "H2D snapshot"); o += fb; }
    CU(cudaMemcpyAsync(h->d_res, o, (size_t)h->batch * 4 * 8, cudaMemcpyHostToDevice, h->stream), "H2D snapshot");
    o += (size_t)h->batch * 4 * 8;
    if (h->has_poly) CU(cudaMemcpyAsync(h->d_qpl, o, (size_t)h->K * (size_t)h->stride * 8, cudaMemcpyHostToDevice, h->stream), "H2D snapshot");
    if (hd.rho != h->rho && h->has_poly) {
        const double old = h->rho;
        h->rho = hd.rho;         // (stage_operators builds for h->rho; put back if anything fails)
        auto enqueue = [&]() -> top_status {
            top_status so = stage_operators(h);
            if (so != TOP_OK) return so;
            CU(cudaMemcpyAsync(h->d_upload, h->stage.get(), h->off_wp, cudaMemcpyHostToDevice, h->stream), "H2D operators");
            InitParams ip;
            std::memset(&ip, 0, sizeof ip);
            fill_init_params(h, ip);
            ip.c0_only = 1;
            CU(launch_init(ip, h->dtype, h->stream), "init kernel launch");
            return TOP_OK;
        };
        const top_status so = enqueue();
        if (so != TOP_OK) { h->rho = old; return so; }
    } else if (hd.rho != h->rho) {
        top_status se = ensure_spectral(h);
        if (se != TOP_OK) return se;
        CU(refresh_operator(h, hd.rho), "operator refresh launch");
        h->rho = hd.rho;
    }
    CU(cudaMemsetAsync(h->d_abort, 0, sizeof(int), h->stream), "cudaMemsetAsync");      // a restored iterate starts with a clean abort flag
    CU(cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
    h->iter = hd.iter;
    h->have_residuals = hd.have_residuals != 0;
    if (!h->have_residuals) std::fill(h->h_res.begin(), h->h_res.end(), std::numeric_limits<double>::quiet_NaN());
    return TOP_OK;
}

extern "C" TOP_API int64_t top_iteration(const top_solver* h) { return h ? h->iter : -1; }

extern "C" TOP_API top_status top_numeric_info(top_solver* h, int64_t* inner_iterations) {
    if (!h) return TOP_E_INVALID;
    if (!h->numeric) return fail(h, TOP_E_INVALID, "top_numeric_info: not a TOP_XUPDATE_NUMERIC solver");
    unsigned long long v = 0;
    CU(cudaMemcpyAsync(&v, h->d_inner, 8, cudaMemcpyDeviceToHost, h->stream), "D2H");
    CU(cudaStreamSynchronize(h->stream), "cudaStreamSynchronize");
    if (inner_iterations) *inner_iterations = (int64_t)v;
    return TOP_OK;
}

extern "C" TOP_API top_status top_launch_info(const top_solver* h, int32_t* ctas, int32_t* threads, int32_t* segs_per_cta,
                                      int32_t* smem_bytes, int32_t* waves, int64_t* launches) {
    if (!h || h->waves.empty()) return TOP_E_INVALID;
    const auto& w = h->waves[0];
    if (ctas) *ctas = w.ctas;
    if (threads) {      // as top_iterate launches it (the fp64 tensor-core kernel may run its last octet on three warps)
        const uint32_t f = h->kflags | sync_flag(h) | w.kflags | (w.cluster ? KF_CLUSTER : 0);
        *threads = w.threads + (h->mma && !h->numeric ? 64 * split_octets_for(f, 0, h->dtype, w.ctas, w.threads) : 0);
    }
    if (segs_per_cta) *segs_per_cta = w.segs_per_cta;
    if (smem_bytes) *smem_bytes = (int32_t)w.smem;
    if (waves) *waves = (int32_t)h->waves.size();
    if (launches) *launches = h->launches;
    return TOP_OK;
}

extern "C" TOP_API top_status top_memory_info(const top_solver* h, int64_t* device_bytes, int64_t* h2d_bytes_per_problem) {
    if (!h) return TOP_E_INVALID;
    if (device_bytes) *device_bytes = (int64_t)h->arena_bytes;
    if (h2d_bytes_per_problem) *h2d_bytes_per_problem = (int64_t)(h->has_poly ? h->upload_bytes : h->upload_bytes - h->off_gram);
    return TOP_OK;
}

extern "C" TOP_API int64_t top_capacity(int32_t device, int32_t s, top_dtype dtype, int32_t constrained) {
    if ((s != 3 && s != 4) || (dtype != TOP_F64 && dtype != TOP_F32)) return -1;
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return -1; }
    int sms = 0, smem = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) { cudaGetLastError(); return -1; }
    // the same rule top_create applies (kernel family of a long chain, shared-memory reserve)
    const int lanes = 4;
    const bool mma = true;
    return (int64_t)sms * max_segs_per_cta((int)dtype, s, constrained != 0, lanes, mma, (size_t)smem - 8192);
}

extern "C" TOP_API double top_fma_peak(int32_t device, top_dtype dtype, int32_t reps, void* cuda_stream) {
    int dev = device;
    if (dev < 0 && cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return -1; }
    if (cudaSetDevice(dev) != cudaSuccess) return -1;
    int sms = 0;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    float* sink = nullptr;
    if (cudaMalloc(&sink, 16) != cudaSuccess) return -1;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms * 4, threads = 512;
    const long long iters = dtype == TOP_F64 ? 4000 : 8000;
    double best = -1;
    launch_fma_peak((int)dtype, blocks, threads, 100, sink, st);   // warm-up
    for (int r = 0; r < std::max(1, reps); ++r) {
        cudaEventRecord(e0, st);
        if (launch_fma_peak((int)dtype, blocks, threads, iters, sink, st) != cudaSuccess) { best = -1; break; }
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1; break; }
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flops = 2.0 * 32.0 * (double)iters * blocks * threads;
        if (ms > 0) best = std::max(best, flops / (ms * 1e-3));
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    return best;
}

extern "C" TOP_API top_status top_precompute_operator(int32_t s, double T, double rho, int32_t box, int32_t vel,
                                                      int32_t acc, uint32_t flags, const double* p0, const double* p1,
                                                      double* Pm_hat, double* c0_hat) {
    if ((s != 3 && s != 4) || !(T > 0) || !(rho > 0) || !p0 || !p1 || !Pm_hat || !c0_hat ||
        (flags & TOP_WAYPOINT_MASK) > TOP_WAYPOINT_FREE)
        return fail(nullptr, TOP_E_INVALID, "top_precompute_operator: bad argument");
    xreal a[3], b[3], PmX[MAXN * MAXN], c0X[MAXN * 3];
    for (int d = 0; d < 3; ++d) { a[d] = p0[d]; b[d] = p1[d]; }
    {
        // the spectral path top_create and top_set_rho use (local frame: p0 is the origin); the direct inverse
        // build_operator() is kept as an in-library cross-check of it
        const int mode = (int)(flags & TOP_WAYPOINT_MASK);
        xreal dp[3] = {b[0] - a[0], b[1] - a[1], b[2] - a[2]}, zero[3] = {0, 0, 0}, PmD[MAXN * MAXN], c0D[MAXN * 3], rPm[MAXN * MAXN];
        Spectral S;
        if (!build_spectral(s, (xreal)T, box != 0, vel != 0, acc != 0, mode, dp, S))
            return fail(nullptr, TOP_E_INVALID, "operator is not positive definite");
        spectral_operator(S, 2 * s, mode == (int)TOP_WAYPOINT_HARD, (xreal)rho, dp, rPm, c0X);
        if (!build_operator(s, (xreal)T, (xreal)rho, box != 0, vel != 0, acc != 0, mode, zero, dp, PmD, c0D))
            return fail(nullptr, TOP_E_INVALID, "operator is not positive definite");
        xreal worst = 0, scale = 0;
        for (int i = 0; i < MAXN * MAXN; ++i) { PmX[i] = rPm[i] / (xreal)rho; worst = std::max(worst, std::fabs(PmX[i] - PmD[i])); scale = std::max(scale, std::fabs(PmD[i])); }
        if (worst > (xreal)1e-13 * scale) return fail(nullptr, TOP_E_INVALID, "spectral and direct operators disagree");
        if (mode == (int)TOP_WAYPOINT_HARD)     // the caller's frame: the chord also carries p0 in c^_0
            for (int r = 0; r < MAXN; ++r)
                for (int d = 0; d < 3; ++d) {
                    xreal v = (r == 0) ? a[d] : 0;
                    for (int c = 0; c < 2 * s; ++c) v -= rPm[r * MAXN + c] * S.gcol0[c] * a[d];
                    c0X[r * 3 + d] += v;
                }
    }
    for (int i = 0; i < MAXN * MAXN; ++i) Pm_hat[i] = (double)PmX[i];
    for (int i = 0; i < MAXN * 3; ++i) c0_hat[i] = (double)c0X[i];
    return TOP_OK;
}

extern "C" TOP_API top_status top_solve(top_solver* h, double eps, int64_t* iters) {
    if (!h) return TOP_E_INVALID;
    TOP_GUARDED(h, return solve_impl(h, eps, iters);)
}
extern "C" TOP_API top_status top_set_rho(top_solver* h, double rho) {
    if (!h) return TOP_E_INVALID;
    TOP_GUARDED(h, return set_rho_impl(h, rho);)
}
extern "C" TOP_API top_status top_get_state(top_solver* h, const char* field, double* out, size_t count) {
    if (!h) return TOP_E_INVALID;
    TOP_GUARDED(h, return get_state_impl(h, field, out, count);)
}
extern "C" TOP_API top_status top_snapshot_restore(top_solver* h, const void* host_buf, size_t bytes) {
    if (!h) return TOP_E_INVALID;
    TOP_GUARDED(h, return snapshot_restore_impl(h, host_buf, bytes);)
}

extern "C" TOP_API top_status top_destroy(top_solver* h) {
    if (!h) return TOP_OK;
    cudaSetDevice(h->device);
    cudaStreamSynchronize(h->stream);
    // a pooled arena goes back to the pool in stream order; if that fails (the caller destroyed the stream first, or it is
    // being captured) cudaFree -- legal for pool allocations, synchronises -- so that the arena is never left allocated
    if (h->arena && (!h->arena_pooled || cudaFreeAsync(h->arena, h->stream) != cudaSuccess)) { cudaGetLastError(); cudaFree(h->arena); }
    cudaGetLastError();
    delete h;
    return TOP_OK;
}

extern "C" TOP_API const char* top_last_error(const top_solver* h) { return h ? h->err.c_str() : g_create_error.c_str(); }
