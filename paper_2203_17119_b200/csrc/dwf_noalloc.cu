// dwf_norm2_static: the squared norm of a device array, computed without asking the CUDA runtime for any memory.
//
// Who this is for.  dwf_norm2 (and every solver in this library) keeps its per-block partial sums in a buffer that the
// context obtains with cudaMalloc.  Some programs that would like to call us cannot afford that:
//   - lattice codes and tensor frameworks that take (nearly) the whole device into their own pool at start-up, so that a
//     cudaMalloc coming from a library finds no memory left, or takes it from under the pool;
//   - code on a latency-critical path, where the implicit device-wide synchronisation of cudaMalloc / cudaFree would stall
//     the work the application has in flight on its other streams;
//   - plug-ins that run under a host which forbids allocation inside its callbacks altogether.
// For them the partial sums live here, in a fixed array that is part of the library image: 512 KiB of global memory on
// every GPU that loads libdwf_b200.so, held until the process exits.  The caller brings the input and the 8 bytes of
// output; nothing else is touched, no context is needed and no cudaMalloc, cudaFree or allocating library routine is called.
//
// What the fixed size costs.  One partial per 256-thread block, one block per 65536 input bytes, 65536 slots: arrays of up
// to DWF_NORM2_STATIC_MAX_BYTES = 4 GiB (2^29 doubles or 2^30 floats; a native fp64 half field of two 32^4 x 16 domains
// is 3.2 GB).  Larger inputs are refused with DWF_EINVAL before anything is launched.
//
// Sharing.  There is ONE array per device and every call on that device uses it.  A call overwrites the slots it is going to
// read before it reads them, so whatever an earlier call left behind never enters a result and nothing has to be cleared.
// Two calls that can overlap on the GPU (different streams, or different host threads on the same device without ordering
// between them) would write the same slots: that is a data race and either result may be wrong.  Order such calls on one
// stream or with events.
//
// Set-up.  Host code cannot use the array's name as a pointer (on the host the name only stands for the symbol), so the
// first call on each device asks the runtime once for the array's device address (cudaGetSymbolAddress, with that device
// current) and remembers it; later calls on that device only launch.  Make that first call outside any stream capture.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/dwf.h"

// The scratch memory of this entry point: one partial sum per block, 65536 slots = 512 KiB.  It lives in the library image,
// one copy on every device; in host code below the name is only a handle for cudaGetSymbolAddress.
static __device__ __align__(256) double ns_partials[65536];

namespace {

constexpr int NS_THREADS = 256;                       // threads per block
constexpr int NS_VEC_PER_THREAD = 16;                 // 16-byte vectors per thread
constexpr size_t NS_BLOCK_BYTES = (size_t)NS_THREADS * NS_VEC_PER_THREAD * 16;   // 65536 input bytes per block
constexpr int NS_MAX_PARTIALS = 65536;                // slots of the fixed array = blocks of the largest input
constexpr int NS_MAX_DEVICES = 64;
static_assert(NS_BLOCK_BYTES * NS_MAX_PARTIALS == DWF_NORM2_STATIC_MAX_BYTES, "header and kernel disagree on the limit");
static_assert(sizeof(ns_partials) == sizeof(double) * NS_MAX_PARTIALS, "scratch array and slot count disagree");

__device__ __forceinline__ double ns_sq(const double2& a) { return a.x * a.x + a.y * a.y; }
__device__ __forceinline__ double ns_sq(const float4& a) {
    return (double)a.x * a.x + (double)a.y * a.y + (double)a.z * a.z + (double)a.w * a.w;
}

// sum over the block, fixed tree (shuffles inside a warp, then the warp leaders): the same inputs give the same bits
template <int NT>
__device__ __forceinline__ double ns_block_sum(double v) {
    __shared__ double warp_sum[NT / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    if ((threadIdx.x & 31) == 0) warp_sum[threadIdx.x >> 5] = v;
    __syncthreads();
    v = (threadIdx.x < NT / 32) ? warp_sum[threadIdx.x] : 0.0;
    if (threadIdx.x < 32) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    }
    return v;
}

// block b sums vectors [b * 4096, (b + 1) * 4096) of the input, coalesced 16-byte loads, and writes slot b.
// The block -> data assignment depends on the input length only, never on the GPU's SM count.
template <typename V>
__global__ void __launch_bounds__(NS_THREADS) norm2_static_kernel(const V* __restrict__ v, size_t nvec,
                                                                  double* __restrict__ partials) {
    const size_t base = (size_t)blockIdx.x * (NS_THREADS * NS_VEC_PER_THREAD);
    double acc = 0.0;
#pragma unroll 4
    for (int k = 0; k < NS_VEC_PER_THREAD; ++k) {
        const size_t i = base + (size_t)k * NS_THREADS + threadIdx.x;
        if (i < nvec) acc += ns_sq(v[i]);
    }
    const double tot = ns_block_sum<NS_THREADS>(acc);
    if (threadIdx.x == 0) partials[blockIdx.x] = tot;
}

// one block: slots [0, n) -> *result.  Reads only slots the launch before it has just written.
__global__ void __launch_bounds__(1024) norm2_static_final_kernel(const double* __restrict__ partials, int n,
                                                                  double* __restrict__ result) {
    double v = 0.0;
    for (int i = threadIdx.x; i < n; i += 1024) v += partials[i];
    const double tot = ns_block_sum<1024>(v);
    if (threadIdx.x == 0) *result = tot;
}

std::mutex ns_mutex;
double* ns_scratch_addr[NS_MAX_DEVICES] = {};         // device address of ns_partials on each device, filled on first use

int ns_fail(char* errbuf, size_t errbuf_len, int status, const char* what, const char* detail = nullptr) {
    if (errbuf && errbuf_len) {
        if (detail) snprintf(errbuf, errbuf_len, "dwf_norm2_static: %s (%s)", what, detail);
        else snprintf(errbuf, errbuf_len, "dwf_norm2_static: %s", what);
    }
    return status;
}

}  // namespace

extern "C" dwf_status dwf_norm2_static(const void* v_dev, size_t nreal, dwf_prec prec, double* result_dev, void* cuda_stream,
                                       char* errbuf, size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (prec != DWF_F64 && prec != DWF_F32) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_EINVAL, "prec must be DWF_F32 or DWF_F64");
    const size_t per_vec = (prec == DWF_F64) ? 2 : 4;            // reals in 16 bytes
    if (!result_dev || ((uintptr_t)result_dev & 7)) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_EINVAL, "result_dev is null or not 8-byte aligned");
    if (nreal && (!v_dev || ((uintptr_t)v_dev & 15))) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_EINVAL, "v_dev is null or not 16-byte aligned");
    if (nreal % per_vec) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_EINVAL, "nreal must be a whole number of 16-byte vectors (2 doubles / 4 floats)");
    const size_t nvec = nreal / per_vec;
    if (nvec > DWF_NORM2_STATIC_MAX_BYTES / 16) {
        char detail[160];
        snprintf(detail, sizeof detail, "%zu reals of %d bytes asked for, the fixed scratch array serves at most %llu bytes", nreal,
                 prec == DWF_F64 ? 8 : 4, (unsigned long long)DWF_NORM2_STATIC_MAX_BYTES);
        return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_EINVAL, "input larger than DWF_NORM2_STATIC_MAX_BYTES", detail);
    }

    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_ECUDA, "cudaGetDevice failed", cudaGetErrorString(e));
    if (dev < 0 || dev >= NS_MAX_DEVICES) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_EINVAL, "device ordinal above 63");
    double* scratch = nullptr;
    {
        // once per device, with that device current: the DEVICE address of the array (its name is not one in host code)
        std::lock_guard<std::mutex> lock(ns_mutex);
        if (!ns_scratch_addr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, ns_partials);
            if (e != cudaSuccess || !p) {
                cudaGetLastError();
                return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_ECUDA, "cudaGetSymbolAddress(scratch) failed", cudaGetErrorString(e));
            }
            ns_scratch_addr[dev] = (double*)p;
        }
        scratch = ns_scratch_addr[dev];
    }

    cudaStream_t stream = (cudaStream_t)cuda_stream;
    const int nblocks = (int)((nvec + NS_THREADS * NS_VEC_PER_THREAD - 1) / (NS_THREADS * NS_VEC_PER_THREAD));   // <= 65536
    if (nblocks > 0) {
        if (prec == DWF_F64) norm2_static_kernel<double2><<<nblocks, NS_THREADS, 0, stream>>>((const double2*)v_dev, nvec, scratch);
        else norm2_static_kernel<float4><<<nblocks, NS_THREADS, 0, stream>>>((const float4*)v_dev, nvec, scratch);
        e = cudaGetLastError();
        if (e != cudaSuccess) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_ECUDA, "launch of the partial-sum kernel failed", cudaGetErrorString(e));
    }
    norm2_static_final_kernel<<<1, 1024, 0, stream>>>(scratch, nblocks, result_dev);   // nblocks == 0: writes 0.0
    e = cudaGetLastError();
    if (e != cudaSuccess) return (dwf_status)ns_fail(errbuf, errbuf_len, DWF_ECUDA, "launch of the final-sum kernel failed", cudaGetErrorString(e));
    return DWF_OK;
}
