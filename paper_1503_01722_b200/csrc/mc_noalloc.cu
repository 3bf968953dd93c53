// mc_edep_total_static (include/mc.h) — the deposited-energy total of the per-batch grids for callers that must not
// allocate device memory.
//
// Who that is.  A dose engine is often a guest in somebody else's process: a planning service whose tensor framework has
// already taken nearly all of the GPU's memory into its own caching allocator (a plain cudaMalloc then fails although the
// framework could still hand out the same bytes); a host thread that runs while another thread is recording a CUDA graph in
// the global capture mode, where any cudaMalloc / cudaFree in the process is illegal and invalidates the recording; a
// delivery-time QA loop that checks the energy ledger between beam segments and cannot afford cudaMalloc / cudaFree, both of
// which stall every stream of the device.  Such callers own their buffers and can pass pointers, but every other compute
// call of this library creates device state (the context's tables, queues and counters).  This one creates nothing.
//
// What it computes.  The same quantity as the ledger's sum_kernel (mc_kernels.cuh: fp64 total of a float array, i.e.
// mc_stats.e_deposited_MeV when given the [n_batches][nvox] grids), with a different reduction: sum_kernel adds one
// partial per CTA into a context-owned ledger word with an fp64 atomic, this variant writes one fp64 partial per fixed
// chunk of kChunk floats into the scratch array below and the CTA that finishes last adds the partials in a fixed order.
// The result therefore does not depend on the grid size or on the order in which CTAs finish: two calls on the same data
// return the same bits (the atomic version is reproducible only to fp64 rounding order).
//
// The scratch.  g_scratch is a file-scope __device__ array: every GPU on which this library's module gets loaded carries
// its kScratchBytes (256 B header + 64 Ki partials x 8 B = 512.25 KiB) from load until the process exits, whether or not
// this entry point is ever called.  That bounds the input: at most kMaxChunks x kChunk = 2^28 floats (1 GiB of grids; the
// largest paper workload, 128^3 voxels x 10 batches, is 2.1e7).  Larger inputs are refused, never truncated.
//   * In HOST code the name g_scratch is only a stand-in the runtime uses to look the symbol up — it is not a device
//     address, and a kernel handed &g_scratch[0] from the host would fault (or, on a system where the GPU can reach host
//     memory, quietly scribble on the wrong bytes).  The device address comes from cudaGetSymbolAddress, asked once per
//     device with that device current and cached in g_dev_ptr[]; only that pointer is passed to the kernel.
//   * All calls on one device share the array and it keeps whatever the previous call left there.  The only word that has
//     to start at zero is the finished-CTA ticket; the entry point clears it on the caller's stream before every launch
//     (so an earlier call that died half-way cannot poison the next one).  Partials are always written before they are
//     read, and only the first n_chunks of them are read, so stale partials of a larger earlier call are never seen.
//   * Nothing serialises two calls against each other: calls on the same device that overlap on the GPU (two host threads,
//     or two streams) race on the ticket and the partials and return garbage.  Callers serialise them.
#include "../../include/mc.h"

#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

namespace {

constexpr int kSumThreads = 256;
constexpr int kPerThread = 16;
constexpr int kChunk = kSumThreads * kPerThread;  // floats per partial
constexpr uint32_t kMaxChunks = 1u << 16;         // partials the scratch holds
constexpr size_t kHeaderBytes = 256;              // word 0: finished-CTA ticket; bytes 8..15: the total (fp64)
constexpr size_t kScratchBytes = kHeaderBytes + (size_t)kMaxChunks * sizeof(double);
constexpr uint64_t kMaxFloats = (uint64_t)kMaxChunks * kChunk;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

// sum of v over the CTA in a fixed order (xor tree inside a warp, warps in index order); the result is valid in thread 0
__device__ __forceinline__ double cta_sum_fixed_order(double v, double* s_part) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();  // s_part may still be read from the previous use
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = v;
    __syncthreads();
    double t = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < kSumThreads / 32; ++w) t += s_part[w];
    return t;
}

// Variant of sum_kernel with its partial sums in the static scratch (see the file header).  `scratch` is the DEVICE
// address of g_scratch as returned by cudaGetSymbolAddress.
__global__ void __launch_bounds__(kSumThreads) sum_static_kernel(const float* __restrict__ a, unsigned long long n, uint32_t n_chunks,
                                                                 unsigned char* scratch) {
    __shared__ double s_part[kSumThreads / 32];
    __shared__ bool s_last;
    unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
    double* total = reinterpret_cast<double*>(scratch + 8);
    double* part = reinterpret_cast<double*>(scratch + kHeaderBytes);
    for (uint32_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const unsigned long long base = (unsigned long long)c * kChunk + threadIdx.x;
        double s = 0.0;
#pragma unroll
        for (int k = 0; k < kPerThread; ++k) {
            const unsigned long long i = base + (unsigned long long)k * kSumThreads;
            s += i < n ? (double)a[i] : 0.0;
        }
        const double t = cta_sum_fixed_order(s, s_part);
        if (threadIdx.x == 0) part[c] = t;
    }
    // the CTA that takes the last ticket sees every partial (each writer fenced before it took its ticket)
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double s = 0.0;
    for (uint32_t c = threadIdx.x; c < n_chunks; c += kSumThreads) s += __ldcg(part + c);  // L2, never a stale L1 line
    const double t = cta_sum_fixed_order(s, s_part);
    if (threadIdx.x == 0) *total = t;
}

std::mutex g_mu;
unsigned char* g_dev_ptr[kMaxDevices];  // device address of g_scratch per device ordinal (nullptr = not asked yet)

mc_status refuse(char* err, int32_t err_len, mc_status st, const char* what, const char* detail = "") {
    if (err && err_len > 0) snprintf(err, (size_t)err_len, "mc_edep_total_static: %s%s", what, detail);
    return st;
}

}  // namespace

extern "C" {

uint64_t mc_edep_total_static_max(void) { return kMaxFloats; }

mc_status mc_edep_total_static(const float* edep_dev, uint64_t n, double* total_out, void* cuda_stream, char* err, int32_t err_len) {
    if (err && err_len > 0) err[0] = '\0';
    if (!edep_dev || !total_out) return refuse(err, err_len, MC_ERR_INVALID_ARG, "edep_dev / total_out is null");
    if (n == 0) return refuse(err, err_len, MC_ERR_INVALID_ARG, "n must be at least 1");
    if (n > kMaxFloats) {
        char lim[96];
        snprintf(lim, sizeof lim, "%llu floats asked, the static scratch covers %llu", (unsigned long long)n, (unsigned long long)kMaxFloats);
        return refuse(err, err_len, MC_ERR_INVALID_ARG, "input larger than the fixed scratch allows: ", lim);
    }
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return refuse(err, err_len, MC_ERR_CUDA, "no CUDA device (this library has no CPU path): ", cudaGetErrorString(e)); }
    if (dev < 0 || dev >= kMaxDevices) return refuse(err, err_len, MC_ERR_CUDA, "device ordinal beyond 63");
    cudaPointerAttributes at;
    e = cudaPointerGetAttributes(&at, edep_dev);
    if (e != cudaSuccess || (at.type != cudaMemoryTypeDevice && at.type != cudaMemoryTypeManaged)) {
        cudaGetLastError();
        return refuse(err, err_len, MC_ERR_INVALID_ARG, "edep_dev is not device memory");
    }
    unsigned char* scratch = nullptr;
    {
        // set-up, once per device and with that device current: the device address of the static array (this is the call
        // that loads the module on the device, which is why the first call belongs before any stream capture)
        std::lock_guard<std::mutex> lock(g_mu);
        if (!g_dev_ptr[dev]) {
            void* p = nullptr;
            e = cudaGetSymbolAddress(&p, g_scratch);
            if (e != cudaSuccess || !p) { cudaGetLastError(); return refuse(err, err_len, MC_ERR_CUDA, "cudaGetSymbolAddress: ", cudaGetErrorString(e)); }
            g_dev_ptr[dev] = static_cast<unsigned char*>(p);
        }
        scratch = g_dev_ptr[dev];
    }
    cudaStream_t s = (cudaStream_t)cuda_stream;
    const uint32_t n_chunks = (uint32_t)((n + kChunk - 1) / kChunk);
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess || sms <= 0) { cudaGetLastError(); return refuse(err, err_len, MC_ERR_CUDA, "cudaDeviceGetAttribute: ", cudaGetErrorString(e)); }
    const uint32_t grid = n_chunks < (uint32_t)sms * 8u ? n_chunks : (uint32_t)sms * 8u;
    e = cudaMemsetAsync(scratch, 0, 16, s);  // ticket (and the previous total): the one thing that must start at zero
    if (e == cudaSuccess) {
        sum_static_kernel<<<grid, kSumThreads, 0, s>>>(edep_dev, (unsigned long long)n, n_chunks, scratch);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpyAsync(total_out, scratch + 8, sizeof(double), cudaMemcpyDefault, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) { cudaGetLastError(); return refuse(err, err_len, MC_ERR_CUDA, "CUDA error: ", cudaGetErrorString(e)); }
    return MC_OK;
}

}  // extern "C"
