// top_device.cuh -- device helpers shared by the sweep kernels (top_kernels.cu, top_kernels_mma.cu).
// Product code: shares nothing with oracle/.
#pragma once
#include <cooperative_groups.h>
#include <cuda_runtime.h>
#include <math.h>

#include "top_internal.h"

namespace top {

namespace {

// ------------------------------------------------------------------------------------------------ helpers

// per-segment strides of the all-gather buffers (24 values used; padded so that the four segments of a warp
// read distinct 16-byte bank groups): rhs rows in doubles; coefficient rows 26 doubles / 28 floats
constexpr int XSTRIDE = 26;

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
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

// ---- inter-CTA mailbox: "LL" slots.  One 16-byte slot carries one fp64 value as {lo32, seq, hi32, seq}, written
// with a single 128-bit store and read with a single 128-bit load; each aligned 8-byte half is atomic, so a
// reader that sees `seq` in both halves has the whole value.  No fence, no separate flag: the data is the flag,
// and neither side invalidates L1 (an acquire/fence at gpu scope would: CCTL.IVALL).
__device__ __forceinline__ void ll_store(void* slot, double v, unsigned seq) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    asm volatile("st.relaxed.gpu.global.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(slot), "r"((unsigned)b), "r"(seq),
                 "r"((unsigned)(b >> 32)), "r"(seq) : "memory");
}
struct LLRaw { unsigned a, f0, b, f1; };
__device__ __forceinline__ void ll_issue(const void* slot, LLRaw& r) {      // the load is issued here, consumed later
    asm volatile("ld.relaxed.gpu.global.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.a), "=r"(r.f0), "=r"(r.b), "=r"(r.f1) : "l"(slot) : "memory");
}
__device__ __forceinline__ bool ll_ok(const LLRaw& r, unsigned seq) { return r.f0 == seq && r.f1 == seq; }
__device__ __forceinline__ double ll_value(const LLRaw& r) {
    return __longlong_as_double((long long)(((unsigned long long)r.b << 32) | r.a));
}

// ---- the same LL slots in DISTRIBUTED SHARED MEMORY (thread-block cluster): the producer stores straight into the
// consumer CTA's shared memory (st.shared::cluster, ~215 cycles one way), the consumer polls its OWN shared memory
// (~40 cycles per look) -- no L2 round trip.  Used when the whole chain fits one cluster (<= 16 CTAs).
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ unsigned cluster_map(unsigned local_addr, unsigned cta_rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(cta_rank));
    return r;
}
__device__ __forceinline__ void ll_store_cluster(unsigned remote_addr, double v, unsigned seq) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v);
    asm volatile("st.shared::cluster.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(remote_addr), "r"((unsigned)b), "r"(seq),
                 "r"((unsigned)(b >> 32)), "r"(seq) : "memory");
}
__device__ __forceinline__ void ll_issue_smem(unsigned local_addr, LLRaw& r) {
    asm volatile("ld.volatile.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(r.a), "=r"(r.f0), "=r"(r.b), "=r"(r.f1) : "r"(local_addr) : "memory");
}
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// [beta_k(tau)]_a = a!/(a-k)! tau^(a-k), a >= k   (Eq. 18 differentiated k times, normalised time)
__device__ __forceinline__ double beta_entry(int k, int a, double tau) {
    if (a < k) return 0.0;
    double f = 1.0;
    for (int q = 0; q < k; ++q) f *= (double)(a - q);
    double pw = 1.0;
    for (int q = 0; q < a - k; ++q) pw *= tau;
    return f * pw;
}

template <typename Real> __device__ __forceinline__ Real shfl_xor(Real v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

template <typename Real> __device__ __forceinline__ Real rsqrt_real(Real x);
template <> __device__ __forceinline__ double rsqrt_real<double>(double x) { return rsqrt(x); }
template <> __device__ __forceinline__ float rsqrt_real<float>(float x) { return rsqrtf(x); }

// Eq. 20f, 20g: y = A c + w;  phi = projection of y onto ||.|| <= bound (reading A15);  w = y - phi
template <typename Real>
__device__ __forceinline__ void ball_update(const Real (&val)[3], Real bound, Real (&phi)[3], Real (&w)[3]) {
    Real y[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) y[d] = val[d] + w[d];
    const Real n2 = y[0] * y[0] + y[1] * y[1] + y[2] * y[2];
    Real scale = (Real)1;
    if (n2 > bound * bound) scale = bound * rsqrt_real<Real>(n2);
#pragma unroll
    for (int d = 0; d < 3; ++d) { phi[d] = scale * y[d]; w[d] = y[d] - phi[d]; }
}

}  // namespace

}  // namespace top
