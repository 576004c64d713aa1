// static_scratch.cu -- the device side of ttc_execute_host_static (include/ttc.h): Eq. 1 on HOST
// buffers without any device allocation.  ttc_execute_host stages A and B through device buffers it gets from
// cudaMalloc; callers that may not allocate (code under stream capture set-up rules, serving loops, harnesses that
// forbid cudaMalloc) get the same staging inside ONE file-scope device array of TTC_STATIC_SCRATCH_BYTES, which
// every device that loads this module holds until the process exits:
//
//     [0, 256)                the work counter of the atomic tile distribution (WorkSched mode 2), cleared per call
//     [256, 256 + |A|)        A as the caller laid it out (span_a elements), 256-byte aligned
//     [.., .. + |B|)          B (span_b elements), 256-byte aligned
//
// In host code `g_static_scratch` is only the host-side stand-in of the symbol, not a device address: the address
// the kernels get comes from cudaGetSymbolAddress, looked up once per device with that device current.
// Nothing here (or in what it calls: cudaMemsetAsync, cudaMemcpyAsync, cudaLaunchKernelExC,
// cudaStreamSynchronize) allocates.  This file owns no arithmetic of the method: the kernels are the library's.
#include <cuda_runtime.h>

#include <mutex>

#include "ttc_internal.h"

namespace ttc {

namespace {

constexpr size_t kCounterBytes = 256;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_static_scratch[TTC_STATIC_SCRATCH_BYTES];

std::mutex g_mu;                       // guards g_base and serialises the calls (they share the array)
void* g_base[kMaxDevices] = {};        // device address of g_static_scratch on device d, once looked up

size_t round256(size_t x) { return (x + 255) & ~(size_t)255; }

// Device address of the array on the CURRENT device (cudaError_t as int; 0 = ok).  Caller holds g_mu.
int scratch_base_locked(unsigned char** base) {
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (int)e;
    if (dev < 0 || dev >= kMaxDevices) return (int)cudaErrorInvalidDevice;
    if (!g_base[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return (int)e;
        if (!p || ((uintptr_t)p & 255) != 0) return (int)cudaErrorInvalidSymbol;
        g_base[dev] = p;
    }
    *base = static_cast<unsigned char*>(g_base[dev]);
    return 0;
}

}  // namespace

bool static_scratch_fits(size_t bytes_a, size_t bytes_b) {
    const size_t cap = (size_t)TTC_STATIC_SCRATCH_BYTES - kCounterBytes;
    const size_t a = round256(bytes_a), b = round256(bytes_b);
    return a <= cap && b <= cap - a;
}

// Copies A (and B when `b_in`) into the array, launches `cand` on the copies, copies B back and waits.
// Returns a cudaError_t as int.  The caller has checked static_scratch_fits and prepared the candidate.
int static_scratch_run(const Candidate& cand, ttc_dtype dtype, ttc_dtype dtype_a, const Scalar& alpha, const Scalar& beta,
                       const void* A_host, size_t bytes_a, void* B_host, size_t bytes_b, bool b_in, void* stream) {
    if (!static_scratch_fits(bytes_a, bytes_b)) return (int)cudaErrorInvalidValue;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    std::lock_guard<std::mutex> lk(g_mu);
    unsigned char* base = nullptr;
    int rc = scratch_base_locked(&base);
    if (rc != 0) return rc;
    unsigned char* dev_a = base + kCounterBytes;
    unsigned char* dev_b = dev_a + round256(bytes_a);
    // the array keeps what the last call left: the counter has to start at zero; A's region is overwritten whole;
    // B's region is overwritten whole by the copy (b_in) or, when B has no padding and beta == 0, by the kernel
    cudaError_t e = cudaMemsetAsync(base, 0, kCounterBytes, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dev_a, A_host, bytes_a, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && b_in) e = cudaMemcpyAsync(dev_b, B_host, bytes_b, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        rc = launch_candidate(cand, dtype, dtype_a, alpha, beta, dev_a, dev_b, stream, reinterpret_cast<uint32_t*>(base));
        e = (cudaError_t)rc;
    }
    if (e != cudaSuccess) {             // nothing of this call may still use the array once the lock is released
        cudaStreamSynchronize(st);
        return (int)e;
    }
    e = cudaMemcpyAsync(B_host, dev_b, bytes_b, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    return (int)e;
}

}  // namespace ttc
