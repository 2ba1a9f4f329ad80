// bg_eval_static: the one entry point of libbg.so that allocates nothing - for callers that cannot call cudaMalloc
// (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
//
// What it computes: |A_{i1 j1 .. in jn}|^2 of the colour-dressed recursion, Eq. 28-32 closed with Eq. 22
// (PAPER.md:L187-213), exactly as bg_eval does for a BG_CDBG_GIVEN context with BG_OPT_KERNEL = 1: the
// thread-per-event kernel of bg_generic.cu (plain FP64, no conditioning flag, no class programs and therefore no
// device tables).  That kernel keeps every sub-current, subset momentum and colour type of an event in global scratch;
// here the scratch is NOT the context's cudaMalloc'ed buffer but the file-scope array below, BG_STATIC_SCRATCH_BYTES
// of device memory that every GPU which loads the library holds until the process exits.
//
// In host code the array's name is a host-side stand-in, not a device address; the address comes from
// cudaGetSymbolAddress, once per device with that device current (static_scratch()), and is what the kernel gets.
// Nothing in the scratch has to start at zero: the kernel writes the type byte and the momentum of every subset of an
// event before it reads them, and reads a current slot only where the type byte says it was written - so the previous
// call's contents are harmless.  All calls share the one array: calls that overlap on the GPU (different streams, or
// different host threads without a common stream) race.
#include <mutex>

#include "bg_internal.h"

namespace {

static __device__ __align__(256) unsigned char g_static_scratch[BG_STATIC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
void* g_scratch_addr[kMaxDevices];   // device address of g_static_scratch on device d (0 = not resolved yet)
std::mutex g_scratch_mutex;

// device address of the scratch array on the CURRENT device
int static_scratch(void** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { cudaGetLastError(); return BG_ECUDA; }
    if (dev < 0 || dev >= kMaxDevices) return BG_EUNSUPPORTED;
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        if (cudaGetSymbolAddress(&p, g_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return BG_ECUDA; }
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return BG_OK;
}

}  // namespace

extern "C" {

long long bg_static_max_events(int n) {
    if (n < 4 || n > 12) return BG_EINVAL;
    return (long long)((size_t)BG_STATIC_SCRATCH_BYTES / bg::cdbg_generic_scratch_per_event(n));
}

int bg_static_setup(void) {
    void* p = nullptr;
    return static_scratch(&p);
}

int bg_eval_static(void* cuda_stream, int n, long long N, const double* mom, const signed char* hel, const signed char* col,
                   double* out) {
    if (n < 4 || n > 12 || N < 0) return BG_EINVAL;
    if (N == 0) return BG_OK;
    if (!mom || !hel || !col || !out) return BG_EINVAL;
    if (N > bg_static_max_events(n)) return BG_ELIMIT;
    void* scratch = nullptr;
    const int rc = static_scratch(&scratch);
    if (rc != BG_OK) return rc;
    const cudaError_t err = bg::cdbg_generic_launch((cudaStream_t)cuda_stream, n, false, N, 0, N, mom, hel, col, out, scratch);
    if (err != cudaSuccess) { cudaGetLastError(); return BG_ECUDA; }
    return BG_OK;
}

}  // extern "C"
