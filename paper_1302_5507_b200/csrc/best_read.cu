// best_read.cu -- SURVEY.md 8(f1): per-read arg-max over its candidate windows (the paper's step 3,
// PAPER.md:240, 390-392). Three passes of one thread per pair over the results of sdp_align_batch:
//   1. key[read] = max over its pairs of (score, lowest window index) packed into 64 bits; count the pairs
//   2. best_pair[read] = the lowest pair index among the pairs that reach the key
//   3. second_score[read] = max score over the read's other pairs
// HBM-trivial (20 bytes per pair); integer atomics only, so the result does not depend on the order.
#include <limits.h>

#include "sdp_host.cuh"

namespace sdp {

__device__ __forceinline__ unsigned long long best_key(int32_t score, uint32_t win) {
    // higher score first, then lower window index: both as unsigned fields of one comparable word
    return ((unsigned long long)((uint32_t)score ^ 0x80000000u) << 32) | (unsigned long long)(0xFFFFFFFFu - win);
}

__global__ void k_best_init(uint32_t n_reads, unsigned long long* __restrict__ key, uint32_t* __restrict__ best_pair,
                            int32_t* __restrict__ best_score, int32_t* __restrict__ second, uint32_t* __restrict__ ncand)
{
    const uint32_t r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n_reads) return;
    key[r] = 0ull; best_pair[r] = SDP_NO_PAIR; best_score[r] = INT_MIN; second[r] = INT_MIN; ncand[r] = 0u;
}

__global__ void k_best_key(uint64_t n_pairs, const uint32_t* __restrict__ pairs, const int32_t* __restrict__ score,
                           unsigned long long* __restrict__ key, uint32_t* __restrict__ ncand)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t r = pairs[2 * p], w = pairs[2 * p + 1];
    atomicMax(key + r, best_key(score[p], w));
    atomicAdd(ncand + r, 1u);
}

__global__ void k_best_pair(uint64_t n_pairs, const uint32_t* __restrict__ pairs, const int32_t* __restrict__ score,
                            const unsigned long long* __restrict__ key, uint32_t* __restrict__ best_pair,
                            int32_t* __restrict__ best_score)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t r = pairs[2 * p], w = pairs[2 * p + 1];
    if (best_key(score[p], w) == key[r]) { atomicMin(best_pair + r, (uint32_t)p); best_score[r] = score[p]; }
}

__global__ void k_best_second(uint64_t n_pairs, const uint32_t* __restrict__ pairs, const int32_t* __restrict__ score,
                              const uint32_t* __restrict__ best_pair, int32_t* __restrict__ second)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t r = pairs[2 * p];
    if (best_pair[r] != (uint32_t)p) atomicMax(second + r, score[p]);
}

void launch_best_per_read(uint64_t n_pairs, uint32_t n_reads, const uint32_t* pairs, const int32_t* score,
                          unsigned long long* key, uint32_t* best_pair, int32_t* best_score, int32_t* second,
                          uint32_t* ncand, cudaStream_t st)
{
    if (n_reads) k_best_init<<<(n_reads + 255) / 256, 256, 0, st>>>(n_reads, key, best_pair, best_score, second, ncand);
    if (!n_pairs) return;
    const uint32_t grid = (uint32_t)((n_pairs + 255) / 256);
    k_best_key<<<grid, 256, 0, st>>>(n_pairs, pairs, score, key, ncand);
    k_best_pair<<<grid, 256, 0, st>>>(n_pairs, pairs, score, key, best_pair, best_score);
    k_best_second<<<grid, 256, 0, st>>>(n_pairs, pairs, score, best_pair, second);
}

}  // namespace sdp
