// top_kernels.cu -- the CADMM segment sweep of TOP (arXiv 2507.10290) as a persistent sm_100a kernel.
//
// One launch runs k sweeps of Algorithm 1 (closed-form branch) over a contiguous range of
// segments.  Mapping:
//   * one CTA owns `segs_per_cta` consecutive segments for the whole launch; their state stays in shared
//     memory / registers across all k sweeps (HBM is touched at launch start and end only);
//   * 8 lanes per segment: lane j owns inequality sample j (its box slack pair and velocity / acceleration
//     ball variables, 3 dims), lane a owns coefficient row a and consensus row a (u, z~);
//   * the internal basis is normalised time, c^_a = c_a T^a (an exact change of variable of Eq. 18), so the
//     evaluation matrices M, E_0, E_1, E_2 of Eq. 19 are the same constants for every
//     segment, scaled by 1/T^k per derivative order k;
//   * a sweep is split at its only cross-segment dependency (the neighbour read of Eq. 20b):
//       phase A (segment local):  x-update (20a), phi/w (20f,g), slack + its dual (20d,e), boundary B = M c
//       exchange: neighbours inside the CTA through shared memory, across CTAs through an L2 mailbox
//       phase B:                  z-update (20b), u-update (20c), residual partial sums (Eq. 21-22)
//   * CTAs synchronise once per sweep: either a grid-wide barrier or release/acquire flags with the two
//     neighbouring CTAs only (the dependency radius of a sweep is exactly one segment).
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <math.h>

#include "top_internal.h"

namespace top {

namespace {

// ------------------------------------------------------------------------------------------------ helpers

template <typename Real> struct Traits;
template <> struct Traits<double> { static constexpr int GSTRIDE = 98; };   // Reals of per-segment scratch (padded:
template <> struct Traits<float>  { static constexpr int GSTRIDE = 100; };  //  4 segments of a warp hit distinct banks)

constexpr int GSLOT = 12;  // per lane: gM[3], g0[3], g1[3], g2[3]

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned int ld_acquire_u32(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u32(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ long long global_ns() {
    long long t;
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t));
    return t;
}
constexpr long long WAIT_TIMEOUT_NS = 2000000000ll;  // a barrier wait longer than 2 s aborts the launch

// Grid-wide barrier on a monotonically increasing counter (reset to 0 before the launch).  All CTAs are
// co-resident (cooperative launch).  Returns false on time-out / abort.
__device__ __forceinline__ bool grid_barrier(unsigned long long* bar, unsigned long long target, int* abort_flag) {
    __shared__ int ok_sh;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(bar, 1ull);
        int ok = 1;
        if (ld_acquire_u64(bar) < target) {
            const long long t0 = global_ns();
            unsigned spins = 0;
            while (ld_acquire_u64(bar) < target) {
                if ((++spins & 1023u) == 0) {
                    if (*(volatile int*)abort_flag || global_ns() - t0 > WAIT_TIMEOUT_NS) {
                        atomicExch(abort_flag, 1);
                        ok = 0;
                        break;
                    }
                }
            }
        }
        ok_sh = ok;
    }
    __syncthreads();
    return ok_sh != 0;
}

// wait until CTA `who` has published sweep `want` (neighbour synchronisation)
__device__ __forceinline__ bool wait_flag(const unsigned int* flag, unsigned int want, int* abort_flag) {
    if (ld_acquire_u32(flag) >= want) return true;
    const long long t0 = global_ns();
    unsigned spins = 0;
    while (ld_acquire_u32(flag) < want) {
        if ((++spins & 1023u) == 0) {
            if (*(volatile int*)abort_flag || global_ns() - t0 > WAIT_TIMEOUT_NS) {
                atomicExch(abort_flag, 1);
                return false;
            }
        }
    }
    return true;
}

template <typename Real> __device__ __forceinline__ Real ldcg(const Real* p) { return __ldcg(p); }
template <typename Real> __device__ __forceinline__ void stcg(Real* p, Real v) { __stcg(p, v); }

// [beta_k(tau)]_a = a!/(a-k)! tau^(a-k), a >= k   (Eq. 18 differentiated k times, normalised time)
__device__ __forceinline__ double beta_entry(int k, int a, double tau) {
    if (a < k) return 0.0;
    double f = 1.0;
    for (int q = 0; q < k; ++q) f *= (double)(a - q);
    double pw = 1.0;
    for (int q = 0; q < a - k; ++q) pw *= tau;
    return f * pw;
}

// table entry (row r, coefficient a, kind): kind 0 = consensus row r of M (derivative r%S at tau = 0 for r < S,
// at tau = 1 for S <= r < 2S); kind 1..3 = sample r of E_0, E_1, E_2 at tau_r = (r+1)/(MS+1)  (reading A10)
template <int S> __device__ __forceinline__ double table_entry(int r, int a, int kind) {
    if (a >= 2 * S) return 0.0;
    if (kind == 0) {
        if (r >= 2 * S) return 0.0;
        return beta_entry(r % S, a, r < S ? 0.0 : 1.0);
    }
    return beta_entry(kind - 1, a, (double)(r + 1) / (double)(MS + 1));
}

// projection onto the Euclidean ball ||y|| <= bound  (Eq. 14 / 20f; reading A15: y = 0 -> scale 1)
template <typename Real>
__device__ __forceinline__ void project_ball(const Real (&y)[3], Real bound, Real (&phi)[3]) {
    const Real n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
    Real scale = (Real)1;
    if (n2 > bound * bound) scale = bound / sqrt(n2);
    phi[0] = scale * y[0]; phi[1] = scale * y[1]; phi[2] = scale * y[2];
}

template <typename Real> __device__ __forceinline__ Real shfl_xor(Real v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

}  // namespace

// ------------------------------------------------------------------------------------------------ the sweep kernel

namespace {

// shared-memory carve-up, identical on host (size) and device (pointers)
struct SmemLayout {
    size_t pm, tabA, tabJ, gs, bs, segc, sst, total;
    int nsample_fields;
};
__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }
__host__ __device__ inline SmemLayout smem_layout(int real_bytes, int S, bool cons, uint32_t flags, int segs, int gstride) {
    SmemLayout L;
    const int T = segs * LANES;
    size_t off = 0;
    L.pm = off;   off = align16(off + (size_t)2 * S * T * sizeof(double));
    L.tabA = off; off = align16(off + (size_t)8 * 8 * 4 * real_bytes);
    L.tabJ = off; off = align16(off + (size_t)8 * 8 * 4 * real_bytes);
    L.gs = off;   off = align16(off + (size_t)segs * gstride * real_bytes);
    L.bs = off;   off = align16(off + (size_t)2 * (segs + 2) * 24 * real_bytes);
    L.segc = off; off = align16(off + (size_t)8 * segs * real_bytes);
    int nf = 0;
    if (cons) nf = ((flags & KF_BOX) ? 6 : 0) + ((flags & KF_VEL) ? 6 : 0) + ((flags & KF_ACC) ? 6 : 0);
    L.nsample_fields = nf;
    L.sst = off;  off = align16(off + (size_t)nf * T * real_bytes);
    L.total = off;
    return L;
}

template <typename Real, int S, bool CONS, int MAXT>
__global__ void __launch_bounds__(MAXT, 1) cadmm_sweeps_kernel(const KParams p) {
    constexpr int N2 = 2 * S;                      // n = 2s coefficients = 2s consensus rows per segment
    constexpr int GST = Traits<Real>::GSTRIDE;
    extern __shared__ __align__(16) unsigned char smem_raw[];

    const int T = blockDim.x, tid = threadIdx.x, lane = tid & (LANES - 1), sl = tid >> 3;
    const int SEGS = p.segs_per_cta;
    const int cta = blockIdx.x, nctas = gridDim.x;
    const uint32_t flags = p.flags;
    const bool has_box = CONS && (flags & KF_BOX), has_vel = CONS && (flags & KF_VEL), has_acc = CONS && (flags & KF_ACC);
    const bool pin_pos = flags & KF_PIN_POS;
    const bool nb_sync = flags & KF_NEIGHBOUR_SYNC;

    const SmemLayout L = smem_layout((int)sizeof(Real), S, CONS, flags, SEGS, GST);
    double* Pms = reinterpret_cast<double*>(smem_raw + L.pm);
    Real* tabA = reinterpret_cast<Real*>(smem_raw + L.tabA);   // [row/sample j][coef a][kind]
    Real* tabJ = reinterpret_cast<Real*>(smem_raw + L.tabJ);   // [coef b][row/sample j][kind]
    Real* Gs = reinterpret_cast<Real*>(smem_raw + L.gs);
    Real* Bs = reinterpret_cast<Real*>(smem_raw + L.bs);       // [2 parity][SEGS+2][8 rows][3]
    Real* segc = reinterpret_cast<Real*>(smem_raw + L.segc);   // [8][SEGS]: 1/T, 1/T^2, lo[3], hi[3]
    Real* sst = reinterpret_cast<Real*>(smem_raw + L.sst);     // [field][T] per-lane sample state
    // sample-state field offsets (in units of T)
    const int F_QP = 0, F_QN = 3;
    const int F_PHV = has_box ? 6 : 0, F_WV = F_PHV + 3;
    const int F_PHA = F_PHV + (has_vel ? 6 : 0), F_WA = F_PHA + 3;

    const long long cta_first = p.seg_begin + (long long)cta * SEGS;
    const long long remaining = p.seg_end - cta_first;
    const int nact = remaining < SEGS ? (int)remaining : SEGS;     // active segments of this CTA (>= 1)
    const bool active = sl < nact;
    const long long gseg = active ? cta_first + sl : cta_first;     // inactive threads alias a valid segment (loads only)
    const long long gt = gseg * LANES + lane;
    const long long stride = p.stride;
    const bool isrow = lane < N2;
    const bool right = lane >= S;
    const int korder = right ? lane - S : lane;

    // ---- tables (same for every segment: normalised time)
    for (int idx = tid; idx < 8 * 8 * 4; idx += T) {
        const int kind = idx & 3, a = (idx >> 2) & 7, r = idx >> 5;
        const Real v = (Real)table_entry<S>(r, a, kind);
        tabA[(r * 8 + a) * 4 + kind] = v;
        tabJ[(a * 8 + r) * 4 + kind] = v;
    }
    // ---- constants
#pragma unroll
    for (int b = 0; b < N2; ++b) Pms[b * T + tid] = p.Pm[b * stride + gt];
    double c0[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) c0[d] = p.c0[d * stride + gt];
    const Real invTk = static_cast<const Real*>(p.invTk)[gt];
    if (active) {
        Real v;
        if (lane < 2) v = static_cast<const Real*>(p.invT)[lane * p.nseg_pad + gseg];
        else v = static_cast<const Real*>(p.lohi)[(lane - 2) * p.nseg_pad + gseg];
        segc[lane * SEGS + sl] = v;
    }
    const uint8_t sf = p.segflags[gseg];
    // ---- state of iterate k
    Real zt[3], u[3], chat[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        zt[d] = static_cast<const Real*>(p.zt)[d * stride + gt];
        u[d] = static_cast<const Real*>(p.u)[d * stride + gt];
        chat[d] = static_cast<const Real*>(p.chat)[d * stride + gt];
    }
    if (CONS) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            if (has_box) {
                sst[(F_QP + d) * T + tid] = static_cast<const Real*>(p.qp)[d * stride + gt];
                sst[(F_QN + d) * T + tid] = static_cast<const Real*>(p.qn)[d * stride + gt];
            }
            if (has_vel) {
                sst[(F_PHV + d) * T + tid] = static_cast<const Real*>(p.phv)[d * stride + gt];
                sst[(F_WV + d) * T + tid] = static_cast<const Real*>(p.wv)[d * stride + gt];
            }
            if (has_acc) {
                sst[(F_PHA + d) * T + tid] = static_cast<const Real*>(p.pha)[d * stride + gt];
                sst[(F_WA + d) * T + tid] = static_cast<const Real*>(p.wa)[d * stride + gt];
            }
        }
    }
    __syncthreads();

    const Real invT = segc[0 * SEGS + (active ? sl : 0)], invT2 = segc[1 * SEGS + (active ? sl : 0)];
    const Real rho = (Real)p.rho, vmax = (Real)p.vmax, amax = (Real)p.amax;
    Real* const G = Gs + (size_t)sl * GST;                 // this segment's scratch
    double* const X = reinterpret_cast<double*>(G);         // [8][3] rhs rows (aliases the g slots)
    Real* const Cs = G + 48;                                // [8][3] coefficient rows
    Real* const Bedge = static_cast<Real*>(p.Bedge);
    const size_t edge_par_stride = (size_t)p.max_ctas * 2 * 4 * 3;

    int wait_failed = 0;
    for (int it = 0; it < p.k_sweeps; ++it) {
        const int par = it & 1;
        const bool last_sweep = (it == p.k_sweeps - 1);
        Real* const Bcur = Bs + (size_t)par * (SEGS + 2) * 24;

        // ================= phase A: segment local =================
        // right-hand side of Eq. 20a (second bracket; rho is applied with the operator, reading A3)
        if (active) {
            Real* g = G + lane * GSLOT;
#pragma unroll
            for (int d = 0; d < 3; ++d) g[d] = isrow ? (zt[d] - u[d]) * invTk : (Real)0;   // M'(z~ - u)
            if (CONS) {
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    Real g0 = 0, g1 = 0, g2 = 0;
                    if (has_box) {      // Ao'(b - s - v), Ao = [E0; -E0], b = [hi; -lo];  s + v = |q| (Moreau pair)
                        const Real lo = segc[(2 + d) * SEGS + sl], hi = segc[(5 + d) * SEGS + sl];
                        g0 = (hi - fabs(sst[(F_QP + d) * T + tid])) + (lo + fabs(sst[(F_QN + d) * T + tid]));
                    }
                    if (has_vel) g1 = (sst[(F_PHV + d) * T + tid] - sst[(F_WV + d) * T + tid]) * invT;    // Av'(phi - w)
                    if (has_acc) g2 = (sst[(F_PHA + d) * T + tid] - sst[(F_WA + d) * T + tid]) * invT2;
                    g[3 + d] = g0; g[6 + d] = g1; g[9 + d] = g2;
                }
            }
        }
        __syncwarp();
        Real R[3] = {0, 0, 0};
        if (active) {
#pragma unroll
            for (int j = 0; j < (CONS ? 8 : N2); ++j) {
                const Real* gj = G + j * GSLOT;
                const Real* t = tabA + (j * 8 + lane) * 4;
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    if (CONS) R[d] += t[0] * gj[d] + t[1] * gj[3 + d] + t[2] * gj[6 + d] + t[3] * gj[9 + d];
                    else R[d] += t[0] * gj[d];
                }
            }
        }
        __syncwarp();
        if (active) {
#pragma unroll
            for (int d = 0; d < 3; ++d) X[lane * 3 + d] = (double)R[d];
        }
        __syncwarp();
        // x-update: c^ = (rho Pm^) R^ + c0^   (Eq. 20a, first bracket precomputed per segment from T_i; fp64 always)
        if (active) {
            double c[3] = {c0[0], c0[1], c0[2]};
#pragma unroll
            for (int b = 0; b < N2; ++b) {
                const double pm = Pms[b * T + tid];
#pragma unroll
                for (int d = 0; d < 3; ++d) c[d] += pm * X[b * 3 + d];
            }
#pragma unroll
            for (int d = 0; d < 3; ++d) { chat[d] = (Real)c[d]; Cs[lane * 3 + d] = chat[d]; }
        }
        __syncwarp();
        Real Bnd[3] = {0, 0, 0};
        if (active) {
            Real C[N2][3];
#pragma unroll
            for (int b = 0; b < N2; ++b)
#pragma unroll
                for (int d = 0; d < 3; ++d) C[b][d] = Cs[b * 3 + d];
            // boundary derivative row `lane` of B = M c  (Eq. 20b's sigma~)
            if (isrow) {
                Real acc[3] = {0, 0, 0};
#pragma unroll
                for (int b = 0; b < N2; ++b) {
                    const Real m = tabJ[(b * 8 + lane) * 4 + 0];
#pragma unroll
                    for (int d = 0; d < 3; ++d) acc[d] += m * C[b][d];
                }
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    Bnd[d] = acc[d] * invTk;
                    Bcur[(sl + 1) * 24 + lane * 3 + d] = Bnd[d];
                }
                if (nctas > 1) {
                    Real* e = Bedge + par * edge_par_stride + (size_t)cta * 24;
                    if (sl == 0 && !right) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) stcg(e + 0 * 12 + korder * 3 + d, Bnd[d]);
                    }
                    if (sl == nact - 1 && right) {
#pragma unroll
                        for (int d = 0; d < 3; ++d) stcg(e + 1 * 12 + korder * 3 + d, Bnd[d]);
                    }
                }
            }
            if (CONS) {
                Real P[3] = {0, 0, 0}, V[3] = {0, 0, 0}, A[3] = {0, 0, 0};
#pragma unroll
                for (int b = 0; b < N2; ++b) {
                    const Real* t = tabJ + (b * 8 + lane) * 4;
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        if (has_box) P[d] += t[1] * C[b][d];
                        if (has_vel) V[d] += t[2] * C[b][d];
                        if (has_acc) A[d] += t[3] * C[b][d];
                    }
                }
                if (has_vel) {      // Eq. 20f, 20g: y = Av c + w;  phi = proj(y);  w = y - phi
                    Real Y[3], phi[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) Y[d] = V[d] * invT + sst[(F_WV + d) * T + tid];
                    project_ball(Y, vmax, phi);
#pragma unroll
                    for (int d = 0; d < 3; ++d) { sst[(F_PHV + d) * T + tid] = phi[d]; sst[(F_WV + d) * T + tid] = Y[d] - phi[d]; }
                }
                if (has_acc) {
                    Real Y[3], phi[3];
#pragma unroll
                    for (int d = 0; d < 3; ++d) Y[d] = A[d] * invT2 + sst[(F_WA + d) * T + tid];
                    project_ball(Y, amax, phi);
#pragma unroll
                    for (int d = 0; d < 3; ++d) { sst[(F_PHA + d) * T + tid] = phi[d]; sst[(F_WA + d) * T + tid] = Y[d] - phi[d]; }
                }
                if (has_box) {      // Eq. 20d, 20e with q = -(A c - b + v):  s = max(0,q),  v <- max(0,-q)
#pragma unroll
                    for (int d = 0; d < 3; ++d) {
                        const Real lo = segc[(2 + d) * SEGS + sl], hi = segc[(5 + d) * SEGS + sl];
                        const Real qp = sst[(F_QP + d) * T + tid], qn = sst[(F_QN + d) * T + tid];
                        const Real vp = qp < 0 ? -qp : (Real)0, vn = qn < 0 ? -qn : (Real)0;
                        sst[(F_QP + d) * T + tid] = (hi - P[d]) - vp;
                        sst[(F_QN + d) * T + tid] = (P[d] - lo) - vn;
                    }
                }
            }
        }

        // ================= exchange of boundary rows =================
        if (nctas == 1) {
            __syncthreads();
        } else if (!nb_sync) {
            if (!grid_barrier(p.bar, (unsigned long long)(it + 1) * nctas, p.abort_flag)) break;   // uniform per CTA
        } else {
            if (__syncthreads_or(wait_failed)) break;       // a wait of the previous sweep timed out: give up together
            if (tid == 0) { __threadfence(); st_release_u32(p.nflag + cta, (unsigned)(it + 1)); }
            if (active && isrow) {
                if (sl == 0 && !right && cta > 0)
                    wait_failed |= !wait_flag(p.nflag + cta - 1, (unsigned)(it + 1), p.abort_flag);
                if (sl == nact - 1 && right && cta + 1 < nctas)
                    wait_failed |= !wait_flag(p.nflag + cta + 1, (unsigned)(it + 1), p.abort_flag);
            }
        }

        // ================= phase B: consensus, dual, residuals =================
        double rp2 = 0, rd2 = 0, rdn2 = 0, gap2 = 0;
        Real dz[3] = {0, 0, 0};
        if (active && isrow) {
            Real nb[3];
            if (nctas > 1 && sl == 0 && !right) {             // left neighbour lives in the previous CTA
                const Real* e = Bedge + par * edge_par_stride + (size_t)(cta > 0 ? cta - 1 : 0) * 24 + 1 * 12 + korder * 3;
#pragma unroll
                for (int d = 0; d < 3; ++d) nb[d] = ldcg(e + d);
            } else if (nctas > 1 && sl == nact - 1 && right) { // right neighbour lives in the next CTA
                const Real* e = Bedge + par * edge_par_stride + (size_t)(cta + 1 < nctas ? cta + 1 : cta) * 24 + 0 * 12 + korder * 3;
#pragma unroll
                for (int d = 0; d < 3; ++d) nb[d] = ldcg(e + d);
            } else {
                const Real* e = right ? Bcur + (sl + 2) * 24 + korder * 3 : Bcur + sl * 24 + (korder + S) * 3;
#pragma unroll
                for (int d = 0; d < 3; ++d) nb[d] = e[d];
            }
            const bool fixed = (right ? (sf & SEG_LAST) : (sf & SEG_FIRST)) || (pin_pos && korder == 0);
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                const Real bl = right ? Bnd[d] : nb[d], br = right ? nb[d] : Bnd[d];
                const Real znew = fixed ? zt[d] : (Real)0.5 * (bl + br);      // Eq. 6b / 20b
                dz[d] = znew - zt[d];
                zt[d] = znew;
                const Real res = Bnd[d] - znew;
                u[d] += res;                                                 // Eq. 6c / 20c (scaled dual, A5)
                rp2 += (double)res * (double)res;
                if (right && !(sf & SEG_LAST)) { const double gp = (double)Bnd[d] - (double)nb[d]; gap2 += gp * gp; }   // Eq. 21
            }
        }
        if (last_sweep) {
            // dual residual rho M(T)'(z~^{k+1} - z~^k) in monomial physical-time coefficient space (Eq. 22, A8)
            __syncwarp();
            if (active) {
#pragma unroll
                for (int d = 0; d < 3; ++d) G[lane * GSLOT + d] = isrow ? dz[d] * invTk : (Real)0;
            }
            __syncwarp();
            if (active && isrow) {
                const double Tp = (double)static_cast<const Real*>(p.Tpow)[gt];
#pragma unroll
                for (int d = 0; d < 3; ++d) {
                    Real x = 0;
#pragma unroll
                    for (int r = 0; r < N2; ++r) x += tabA[(r * 8 + lane) * 4 + 0] * G[r * GSLOT + d];
                    const double xr = p.rho * (double)x;
                    rdn2 += xr * xr;
                    rd2 += (xr * Tp) * (xr * Tp);
                }
            }
#pragma unroll
            for (int m = 1; m < LANES; m <<= 1) {     // fixed-order tree over the 8 lanes of the segment
                rp2 += shfl_xor(rp2, m); rd2 += shfl_xor(rd2, m); rdn2 += shfl_xor(rdn2, m); gap2 += shfl_xor(gap2, m);
            }
            if (active && lane == 0) {
                double* o = p.part + gseg * 4;
                o[0] = rp2; o[1] = rd2; o[2] = rdn2; o[3] = gap2;
            }
            __syncwarp();
        }
    }

    // ---- write iterate k + k_sweeps back
    if (active) {
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            static_cast<Real*>(p.zt)[d * stride + gt] = zt[d];
            static_cast<Real*>(p.u)[d * stride + gt] = u[d];
            static_cast<Real*>(p.chat)[d * stride + gt] = chat[d];
            if (has_box) {
                static_cast<Real*>(p.qp)[d * stride + gt] = sst[(F_QP + d) * T + tid];
                static_cast<Real*>(p.qn)[d * stride + gt] = sst[(F_QN + d) * T + tid];
            }
            if (has_vel) {
                static_cast<Real*>(p.phv)[d * stride + gt] = sst[(F_PHV + d) * T + tid];
                static_cast<Real*>(p.wv)[d * stride + gt] = sst[(F_WV + d) * T + tid];
            }
            if (has_acc) {
                static_cast<Real*>(p.pha)[d * stride + gt] = sst[(F_PHA + d) * T + tid];
                static_cast<Real*>(p.wa)[d * stride + gt] = sst[(F_WA + d) * T + tid];
            }
        }
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------ small kernels

namespace {

// c_a = c^_a / T^a, layout [seg][dim][a]  (Eq. 18; dim-major "squeezed" c_i)
template <typename Real>
__global__ void convert_coeffs_kernel(const ConvParams p) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // one thread per (segment, lane)
    if (idx >= p.nseg * LANES) return;
    const long long seg = idx / LANES;
    const int a = (int)(idx % LANES);
    if (a >= 2 * p.s) return;
    const Real invT = static_cast<const Real*>(p.invT)[seg];
    Real sc = 1;
    for (int q = 0; q < a; ++q) sc *= invT;
    Real* out = static_cast<Real*>(p.out);
    for (int d = 0; d < p.dims; ++d)
        out[(seg * p.dims + d) * (2 * p.s) + a] = static_cast<const Real*>(p.chat)[d * p.stride + idx] * sc;
}

// res[b][q] = sqrt(sum_i part[b*N+i][q]) with a fixed-order tree (deterministic; no atomics)
__global__ void residual_reduce_kernel(const double* __restrict__ part, double* __restrict__ res, long long N) {
    __shared__ double sh[4][256];
    const int b = blockIdx.x, t = threadIdx.x;
    double acc[4] = {0, 0, 0, 0};
    for (long long i = t; i < N; i += 256) {
        const double* q = part + ((long long)b * N + i) * 4;
        acc[0] += q[0]; acc[1] += q[1]; acc[2] += q[2]; acc[3] += q[3];
    }
    for (int q = 0; q < 4; ++q) sh[q][t] = acc[q];
    __syncthreads();
    for (int w = 128; w > 0; w >>= 1) {
        if (t < w) for (int q = 0; q < 4; ++q) sh[q][t] += sh[q][t + w];
        __syncthreads();
    }
    if (t < 4) res[b * 4 + t] = sqrt(sh[t][0]);
}

// dependent-chain-free FMA loop: 8 independent accumulators per thread; 2 flops per FMA
template <typename Real>
__global__ void fma_peak_kernel(long long iters, float* sink) {
    Real a[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) a[i] = (Real)(threadIdx.x + i) * (Real)1e-3;
    const Real x = (Real)0.999, y = (Real)1e-4;
    for (long long it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep)
#pragma unroll
            for (int i = 0; i < 8; ++i) a[i] = a[i] * x + y;
    }
    Real s = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += a[i];
    if (s == (Real)123456.789) sink[0] = (float)s;
}

template <typename Real, int S, bool CONS, int MAXT>
cudaError_t launch_one(const KParams& p, int ctas, int threads, size_t smem, cudaStream_t st) {
    auto kern = cadmm_sweeps_kernel<Real, S, CONS, MAXT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    KParams pc = p;
    void* args[] = {&pc};
    if (ctas > 1) return cudaLaunchCooperativeKernel((const void*)kern, dim3(ctas), dim3(threads), args, smem, st);
    return cudaLaunchKernel((const void*)kern, dim3(ctas), dim3(threads), args, smem, st);
}

template <typename Real, int S, bool CONS, int MAXT>
cudaError_t limits_one(int threads, size_t smem, int* per_sm) {
    auto kern = cadmm_sweeps_kernel<Real, S, CONS, MAXT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(per_sm, kern, threads, smem);
}

// f64 kernels are compiled for <= 576 threads (112 registers per thread); f32 for <= 1024 (64 registers)
constexpr int MAXT_F64 = 576, MAXT_F32 = 1024;

}  // namespace

#define TOP_DISPATCH(CALL_F64, CALL_F32)                                           \
    if (dtype == 0) {                                                              \
        if (s == 3) { if (constrained) { CALL_F64(3, true) } else { CALL_F64(3, false) } } \
        else        { if (constrained) { CALL_F64(4, true) } else { CALL_F64(4, false) } } \
    } else {                                                                       \
        if (s == 3) { if (constrained) { CALL_F32(3, true) } else { CALL_F32(3, false) } } \
        else        { if (constrained) { CALL_F32(4, true) } else { CALL_F32(4, false) } } \
    }

int max_threads_for(int dtype) { return dtype == 0 ? MAXT_F64 : MAXT_F32; }

cudaError_t launch_sweeps(const KParams& p, int dtype, int s, bool constrained, int ctas, int threads,
                          size_t smem, cudaStream_t st) {
#define F64(S_, C_) return launch_one<double, S_, C_, MAXT_F64>(p, ctas, threads, smem, st);
#define F32(S_, C_) return launch_one<float, S_, C_, MAXT_F32>(p, ctas, threads, smem, st);
    TOP_DISPATCH(F64, F32)
#undef F64
#undef F32
    return cudaErrorInvalidValue;
}

cudaError_t sweep_kernel_limits(int dtype, int s, bool constrained, int threads, size_t smem, int* max_ctas_per_sm) {
#define F64(S_, C_) return limits_one<double, S_, C_, MAXT_F64>(threads, smem, max_ctas_per_sm);
#define F32(S_, C_) return limits_one<float, S_, C_, MAXT_F32>(threads, smem, max_ctas_per_sm);
    TOP_DISPATCH(F64, F32)
#undef F64
#undef F32
    return cudaErrorInvalidValue;
}

size_t sweep_smem_bytes(int dtype, int s, bool constrained, uint32_t flags, int segs_per_cta) {
    const int rb = dtype == 0 ? 8 : 4;
    const int gst = dtype == 0 ? Traits<double>::GSTRIDE : Traits<float>::GSTRIDE;
    return smem_layout(rb, s, constrained, flags, segs_per_cta, gst).total;
}

cudaError_t launch_convert(const ConvParams& p, int dtype, cudaStream_t st) {
    const long long n = p.nseg * LANES;
    if (n == 0) return cudaSuccess;
    const int blocks = (int)((n + 255) / 256);
    if (dtype == 0) convert_coeffs_kernel<double><<<blocks, 256, 0, st>>>(p);
    else convert_coeffs_kernel<float><<<blocks, 256, 0, st>>>(p);
    return cudaGetLastError();
}

cudaError_t launch_residual_reduce(const double* part, double* res, long long N, int batch, cudaStream_t st) {
    residual_reduce_kernel<<<batch, 256, 0, st>>>(part, res, N);
    return cudaGetLastError();
}

cudaError_t launch_fma_peak(int dtype, int blocks, int threads, long long iters, float* sink, cudaStream_t st) {
    if (dtype == 0) fma_peak_kernel<double><<<blocks, threads, 0, st>>>(iters, sink);
    else fma_peak_kernel<float><<<blocks, threads, 0, st>>>(iters, sink);
    return cudaGetLastError();
}

}  // namespace top
