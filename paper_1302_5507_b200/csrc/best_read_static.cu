// best_read_static.cu -- sdp_best_per_read_static: the per-read choice of sdp_best_per_read (SURVEY.md 8(f1),
// PAPER.md:240, 390-392; rule of DESIGN.md R16) for callers that must not allocate device memory.
//
// Who that is: a host program that handed the GPU's memory to an allocator of its own at start-up (an aligner that
// sizes its index and batch buffers to fill the card, a framework with a caching pool), so that a later cudaMalloc
// can fail or fragment the pool; and a program that keeps several streams busy, where cudaMalloc / cudaFree stall the
// whole device while they run. sdp_best_per_read needs a context (sdp_create allocates) and grows five device arrays
// on demand. This entry point needs neither: the caller passes every input and output array, and the one piece of
// working memory the method needs -- a 64-bit (score, window) key per read -- lives in the fixed array below, which
// is part of the library image. Every GPU that loads libsdp.so holds those 8 MiB from the moment the library's module
// is loaded on it until the process exits, whether or not this entry point is ever called.
//
// The kernels are copies of best_read.cu's four passes (the existing path is untouched); integer atomics only, so the
// outputs are the same whatever the order of the threads.
#include <cuda_runtime.h>
#include <limits.h>
#include <stdio.h>

#include <mutex>

#include "../../include/sdp.h"

namespace {

// The key of read r. The host code below must never hand this NAME to a kernel: on the host it is only a stand-in
// object of the runtime's symbol table, not the array's device address (a kernel given it would fault, or scribble
// over host memory where the GPU can reach it). The address comes from cudaGetSymbolAddress, once per device.
static __device__ __align__(256) unsigned long long g_static_key[SDP_STATIC_MAX_READS];

constexpr int kMaxDevices = 64;
std::mutex g_setup_lock;
unsigned long long* g_key_addr[kMaxDevices];       // device address of g_static_key on device d, null until set up
thread_local char g_static_err[256];

int fail_static(int code, const char* what, cudaError_t ce = cudaSuccess)
{
    if (ce != cudaSuccess) snprintf(g_static_err, sizeof g_static_err, "%s: %s", what, cudaGetErrorString(ce));
    else snprintf(g_static_err, sizeof g_static_err, "%s", what);
    return code;
}

__device__ __forceinline__ unsigned long long static_key(int32_t score, uint32_t win)
{
    // higher score first, then lower window index, as two unsigned fields of one comparable word
    return ((unsigned long long)((uint32_t)score ^ 0x80000000u) << 32) | (unsigned long long)(0xFFFFFFFFu - win);
}

// The array keeps whatever the previous call left in it, so every call starts by zeroing the keys it will use.
__global__ void k_static_init(uint32_t n_reads, unsigned long long* __restrict__ key, uint32_t* __restrict__ best_pair,
                              int32_t* __restrict__ best_score, int32_t* __restrict__ second, uint32_t* __restrict__ ncand)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_reads) return;
    key[r] = 0ull; best_pair[r] = SDP_NO_PAIR; best_score[r] = INT_MIN; second[r] = INT_MIN; ncand[r] = 0u;
}

// A pair that names a read outside [0, n_reads) is skipped in every pass (there is no context to report it to, and
// it must not reach past the array).
__global__ void k_static_key(uint64_t n_pairs, uint32_t n_reads, const uint32_t* __restrict__ pairs,
                             const int32_t* __restrict__ score, unsigned long long* __restrict__ key,
                             uint32_t* __restrict__ ncand)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t r = pairs[2 * p], w = pairs[2 * p + 1];
    if (r >= n_reads) return;
    atomicMax(key + r, static_key(score[p], w));
    atomicAdd(ncand + r, 1u);
}

__global__ void k_static_pair(uint64_t n_pairs, uint32_t n_reads, const uint32_t* __restrict__ pairs,
                              const int32_t* __restrict__ score, const unsigned long long* __restrict__ key,
                              uint32_t* __restrict__ best_pair, int32_t* __restrict__ best_score)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t r = pairs[2 * p], w = pairs[2 * p + 1];
    if (r >= n_reads) return;
    if (static_key(score[p], w) == key[r]) { atomicMin(best_pair + r, (uint32_t)p); best_score[r] = score[p]; }
}

__global__ void k_static_second(uint64_t n_pairs, uint32_t n_reads, const uint32_t* __restrict__ pairs,
                                const int32_t* __restrict__ score, const uint32_t* __restrict__ best_pair,
                                int32_t* __restrict__ second)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t r = pairs[2 * p];
    if (r >= n_reads) return;
    if (best_pair[r] != (uint32_t)p) atomicMax(second + r, score[p]);
}

// Once per device, with that device current: ask the runtime where g_static_key lives there.
int key_address(int dev, unsigned long long** out)
{
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_key_addr[dev]) {
        void* p = nullptr;
        const cudaError_t ce = cudaGetSymbolAddress(&p, g_static_key);
        if (ce != cudaSuccess || !p) return fail_static(SDP_ECUDA, "cudaGetSymbolAddress(g_static_key)", ce);
        g_key_addr[dev] = (unsigned long long*)p;
    }
    *out = g_key_addr[dev];
    return SDP_OK;
}

}  // namespace

extern "C" const char* sdp_static_last_error(void) { return g_static_err; }

extern "C" int sdp_best_per_read_static(int cuda_device, const uint32_t* pairs, const int32_t* score, uint64_t n_pairs,
                                        uint32_t n_reads, void* cuda_stream, uint32_t* best_pair, int32_t* best_score,
                                        int32_t* second_score, uint32_t* n_candidates)
{
    g_static_err[0] = 0;
    if (cuda_device < 0 || cuda_device >= kMaxDevices) return fail_static(SDP_EINVAL, "cuda_device outside 0..63");
    if (n_reads > SDP_STATIC_MAX_READS) {
        snprintf(g_static_err, sizeof g_static_err,
                 "n_reads = %u is beyond SDP_STATIC_MAX_READS = %u, the size of the library's fixed key array "
                 "(split the batch by read, or use sdp_best_per_read)", n_reads, (unsigned)SDP_STATIC_MAX_READS);
        return SDP_ERANGE;
    }
    if (n_pairs > 0xFFFFFFF0ull) return fail_static(SDP_ERANGE, "n_pairs does not fit the 32-bit pair index of best_pair");
    if (n_reads && (!best_pair || !best_score || !second_score || !n_candidates)) return fail_static(SDP_EINVAL, "null output array");
    if (n_pairs && (!pairs || !score)) return fail_static(SDP_EINVAL, "null input array");
    if (!n_reads) return SDP_OK;                             // nothing to write (pairs, if any, name no valid read)

    int prev = -1;
    cudaError_t ce = cudaGetDevice(&prev);
    if (ce != cudaSuccess) return fail_static(SDP_ECUDA, "cudaGetDevice", ce);
    if (prev != cuda_device && (ce = cudaSetDevice(cuda_device)) != cudaSuccess) return fail_static(SDP_ECUDA, "cudaSetDevice", ce);
    unsigned long long* key = nullptr;
    int rc = key_address(cuda_device, &key);
    if (rc == SDP_OK) {
        cudaStream_t st = (cudaStream_t)cuda_stream;
        k_static_init<<<(n_reads + 255) / 256, 256, 0, st>>>(n_reads, key, best_pair, best_score, second_score, n_candidates);
        if (n_pairs) {
            const uint32_t grid = (uint32_t)((n_pairs + 255) / 256);
            k_static_key<<<grid, 256, 0, st>>>(n_pairs, n_reads, pairs, score, key, n_candidates);
            k_static_pair<<<grid, 256, 0, st>>>(n_pairs, n_reads, pairs, score, key, best_pair, best_score);
            k_static_second<<<grid, 256, 0, st>>>(n_pairs, n_reads, pairs, score, best_pair, second_score);
        }
        if ((ce = cudaGetLastError()) != cudaSuccess) rc = fail_static(SDP_ECUDA, "kernel launch", ce);
    }
    if (prev != cuda_device) cudaSetDevice(prev);
    return rc;
}
