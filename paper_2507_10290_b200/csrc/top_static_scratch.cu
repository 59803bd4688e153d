// top_static_scratch.cu -- top_operator_rows_static (include/top.h): the per-segment x-update operator of Eq. 20a
// computed by the library's own precompute kernel, for callers that must not allocate device memory.
//
// Who that is.  A planner that runs inside somebody else's process is often handed its buffers and nothing else: a
// flight-stack or simulator plug-in whose host reserved the whole device heap at start-up, a re-planning loop with a hard
// period (cudaMalloc / cudaFree may synchronise the device and take an unbounded time), a thread that runs while another
// thread of the process records a CUDA graph (an allocation call then breaks the recording), or a process whose memory
// budget is fixed by its container.  Such a caller can pass pointers it already owns, but it cannot let us create a solver
// (top_create takes an arena from a memory pool).  For it the kernel's working memory -- the double-double Gram tables, the
// device copy of the durations, the status word -- lives in the file-scope array below instead: part of the library image,
// present on every GPU that loads libtop.so from the moment the module is loaded until the process exits (SCRATCH_BYTES
// per GPU, whether the entry point is ever called or not).
//
// The array's name is a host-side stand-in in host code, not a device address; its address on the current device comes from
// cudaGetSymbolAddress, once per device (static_scratch_on_current_device), and that pointer is what the kernel is given.
// Product code: shares nothing with oracle/.
#include <cuda_runtime.h>

#include <cmath>
#include <cstddef>
#include <cstdio>
#include <mutex>

#include "../../include/top.h"
#include "top_internal.h"

using namespace top;

namespace {

// Everything precompute_operator_kernel touches besides the caller's output buffer.
struct StaticScratch {
    GramDD gram[2];                                  // Gram tables of s = 3 and s = 4 (written once per device, read only afterwards)
    int status[64];                                  // [0]: the kernel sets it when a segment's operator is not positive definite
    double durations[TOP_STATIC_MAX_SEGMENTS];       // device copy of the caller's host array (this call's)
};
constexpr size_t SCRATCH_BYTES = sizeof(StaticScratch);
static_assert(SCRATCH_BYTES <= 192 * 1024, "the static scratch array is meant to stay modest");

static __device__ __align__(256) unsigned char g_static_scratch[SCRATCH_BYTES];

// The array keeps whatever the previous call left in it: the status word is the one thing that must start at zero.
// (Device code may name the array directly; only host code needs the looked-up address.)
__global__ void static_scratch_clear_status_kernel() {
    reinterpret_cast<StaticScratch*>(g_static_scratch)->status[0] = 0;
}

constexpr int MAXDEV = 64;
struct DeviceSlot {
    std::mutex mu;                   // held for a whole call: calls on one device share the one array
    StaticScratch* ptr = nullptr;    // device address of g_static_scratch on this device (nullptr: not set up yet)
};
DeviceSlot g_slots[MAXDEV];

// Set-up, once per device, with that device current: look the array's device address up and fill the Gram tables
// (a synchronous 28 KB copy -- the reason the first call on a device should not come while a stream is being captured).
cudaError_t static_scratch_on_current_device(DeviceSlot& slot) {
    if (slot.ptr) return cudaSuccess;
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    GramDD host_tables[2];                   // 28 KB on the stack; identical for every device
    gram_tables_dd(3, &host_tables[0]);
    gram_tables_dd(4, &host_tables[1]);
    e = cudaMemcpy(static_cast<unsigned char*>(p) + offsetof(StaticScratch, gram), host_tables, sizeof host_tables, cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
    slot.ptr = static_cast<StaticScratch*>(p);
    return cudaSuccess;
}

struct DeviceGuard {                 // makes `device` current for the call and puts the caller's device back afterwards
    int prev = -1;
    bool switched = false;
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
};

top_status fail_static(top_status st, const char* msg) { return static_cast<top_status>(report_error((int)st, msg)); }

top_status cuda_error(cudaError_t e, const char* what) {
    char msg[256];
    std::snprintf(msg, sizeof msg, "top_operator_rows_static: %s: %s", what, cudaGetErrorString(e));
    return fail_static(TOP_E_CUDA, msg);
}

}  // namespace

extern "C" TOP_API top_status top_operator_rows_static(int32_t device, int32_t nseg, int32_t s, const double* durations,
                                                       double rho, int32_t box, int32_t vel, int32_t acc, uint32_t flags,
                                                       double* rows_out, void* cuda_stream) {
    if ((s != 3 && s != 4) || nseg < 1 || !durations || !rows_out || !(rho > 0) || !std::isfinite(rho) ||
        (flags & TOP_WAYPOINT_MASK) > TOP_WAYPOINT_FREE)
        return fail_static(TOP_E_INVALID, "top_operator_rows_static: bad argument (s in {3,4}, nseg >= 1, rho > 0, flags = one TOP_WAYPOINT_*, non-null pointers)");
    if (nseg > TOP_STATIC_MAX_SEGMENTS) {
        char msg[256];
        std::snprintf(msg, sizeof msg, "top_operator_rows_static: nseg = %d is more than TOP_STATIC_MAX_SEGMENTS = %d, all that the "
                      "static scratch array holds; split the segments over several calls", (int)nseg, (int)TOP_STATIC_MAX_SEGMENTS);
        return fail_static(TOP_E_UNSUPPORTED, msg);
    }
    for (int32_t g = 0; g < nseg; ++g)
        if (!(durations[g] > 0) || !std::isfinite(durations[g]))
            return fail_static(TOP_E_INVALID, "top_operator_rows_static: durations must be finite and > 0");

    DeviceGuard guard;
    cudaError_t e = cudaGetDevice(&guard.prev);
    if (e != cudaSuccess) return cuda_error(e, "no CUDA device");
    if (device < 0) device = guard.prev;
    if (device >= MAXDEV) return fail_static(TOP_E_INVALID, "top_operator_rows_static: device ordinal out of range");
    if (device != guard.prev) {
        if ((e = cudaSetDevice(device)) != cudaSuccess) return cuda_error(e, "cudaSetDevice");
        guard.switched = true;
    }
    cudaPointerAttributes attr;
    if (cudaPointerGetAttributes(&attr, rows_out) != cudaSuccess || (attr.type != cudaMemoryTypeDevice && attr.type != cudaMemoryTypeManaged) ||
        (attr.type == cudaMemoryTypeDevice && attr.device != device)) {
        cudaGetLastError();
        return fail_static(TOP_E_INVALID, "top_operator_rows_static: rows_out must be device memory of the selected device");
    }

    DeviceSlot& slot = g_slots[device];
    std::lock_guard<std::mutex> lock(slot.mu);
    if ((e = static_scratch_on_current_device(slot)) != cudaSuccess) return cuda_error(e, "set-up of the static scratch array");
    StaticScratch* sc = slot.ptr;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    if ((e = cudaMemcpyAsync(sc->durations, durations, sizeof(double) * (size_t)nseg, cudaMemcpyHostToDevice, st)) != cudaSuccess)
        return cuda_error(e, "copy of the durations");
    static_scratch_clear_status_kernel<<<1, 1, 0, st>>>();
    if ((e = cudaGetLastError()) != cudaSuccess) return cuda_error(e, "status clear launch");
    // the kernel writes the 2s x 2s block of every segment; the zero padding up to 8 x 8 is written here
    if ((e = cudaMemsetAsync(rows_out, 0, sizeof(double) * MAXN * LANES * (size_t)nseg, st)) != cudaSuccess)
        return cuda_error(e, "clearing rows_out");
    PrecompParams pp = {};
    pp.gram = &sc->gram[s - 3];
    pp.durations = sc->durations;
    pp.Pm = rows_out;
    pp.stride = (long long)nseg * LANES;
    pp.nseg = nseg;
    pp.N = nseg;
    pp.s = s;
    pp.hard = (flags & TOP_WAYPOINT_MASK) == TOP_WAYPOINT_HARD;
    pp.box = box != 0; pp.vel = vel != 0; pp.acc = acc != 0;
    pp.wide = 0;
    pp.rho = rho;
    pp.bad = &sc->status[0];
    if ((e = launch_precompute_operator(pp, st)) != cudaSuccess) return cuda_error(e, "operator kernel launch");
    int status = 0;
    if ((e = cudaMemcpyAsync(&status, &sc->status[0], sizeof status, cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_error(e, "status read-back");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_error(e, "cudaStreamSynchronize");
    if (status != 0)
        return fail_static(TOP_E_INVALID, "top_operator_rows_static: the operator of at least one segment is not positive definite (extreme duration or rho)");
    return TOP_OK;
}
