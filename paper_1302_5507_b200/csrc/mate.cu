// mate.cu -- SURVEY.md 8(f4): the thin layer just above the path for the paper's step 2 (mate rescue,
// PAPER.md:240, 394-396): candidate window from the mapped end and the fragment-length bounds, and the
// "properly paired" test after the alignment. Integer arithmetic, one thread per rescue; definitions in sdp.h.
#include "sdp_host.cuh"

namespace sdp {

__global__ void k_mate_windows(const sdp_mates mt, uint32_t min_ins, uint32_t max_ins, uint64_t ref_bases,
                               uint64_t* __restrict__ win_off, uint32_t* __restrict__ win_len)
{
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= mt.n) return;
    const long long p = (long long)mt.mate_pos[k], L = (long long)mt.mate_len[k], n = (long long)mt.read_len[k];
    long long lo, hi;                                      // the other end lies in [lo, hi)
    if (mt.mate_reverse[k] == 0) { lo = p + (long long)min_ins - n; hi = p + (long long)max_ins; }
    else                         { lo = p + L - (long long)max_ins; hi = p + L - (long long)min_ins + n; }
    lo = max(lo, 0LL);
    hi = min(hi, (long long)ref_bases);
    const bool ok = hi > lo && hi - lo <= 0xFFFFFFFFLL;
    win_off[k] = ok ? (uint64_t)lo : 0ull;
    win_len[k] = ok ? (uint32_t)(hi - lo) : 0u;
}

__global__ void k_proper_pairs(const sdp_mates mt, uint32_t min_ins, uint32_t max_ins, const uint64_t* __restrict__ win_off,
                               const uint32_t* __restrict__ win_len, const uint32_t* __restrict__ pair_of_rescue,
                               const int32_t* __restrict__ ref_start, const int32_t* __restrict__ ref_end,
                               const uint8_t* __restrict__ pass, uint8_t* __restrict__ proper)
{
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= mt.n) return;
    uint8_t ok = 0;
    const uint64_t q = pair_of_rescue ? (uint64_t)pair_of_rescue[k] : k;      // where rescue k sits in the aligned pair list
    if (win_len[k] > 0 && q != (uint64_t)SDP_NO_PAIR && pass[q]) {
        const long long p = (long long)mt.mate_pos[k], L = (long long)mt.mate_len[k], w = (long long)win_off[k];
        const long long ins = mt.mate_reverse[k] == 0 ? (w + ref_end[q] + 1) - p : (p + L) - (w + ref_start[q]);
        ok = (ins >= (long long)min_ins && ins <= (long long)max_ins) ? 1 : 0;
    }
    proper[k] = ok;
}

// pair list of a rescue batch: rescues with a non-empty window, in rescue order (off = exclusive scan of the flags)
__global__ void k_mate_flags(const uint32_t* __restrict__ win_len, uint64_t n, uint32_t* __restrict__ flag)
{
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) flag[k] = win_len[k] > 0 ? 1u : 0u;
}
__global__ void k_mate_pairs(const uint32_t* __restrict__ flag, const uint64_t* __restrict__ off, uint64_t n,
                             uint32_t* __restrict__ pairs, uint32_t* __restrict__ pair_of_rescue)
{
    const uint64_t k = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    if (flag[k]) {
        const uint64_t q = off[k];
        pairs[2 * q] = (uint32_t)k; pairs[2 * q + 1] = (uint32_t)k;
        pair_of_rescue[k] = (uint32_t)q;
    } else pair_of_rescue[k] = SDP_NO_PAIR;
}

void launch_mate_windows(const sdp_mates& mt, uint32_t min_ins, uint32_t max_ins, uint64_t ref_bases, uint64_t* win_off,
                         uint32_t* win_len, cudaStream_t st)
{
    if (mt.n) k_mate_windows<<<(uint32_t)((mt.n + 255) / 256), 256, 0, st>>>(mt, min_ins, max_ins, ref_bases, win_off, win_len);
}

void launch_proper_pairs(const sdp_mates& mt, uint32_t min_ins, uint32_t max_ins, const uint64_t* win_off,
                         const uint32_t* win_len, const uint32_t* pair_of_rescue, const int32_t* ref_start,
                         const int32_t* ref_end, const uint8_t* pass, uint8_t* proper, cudaStream_t st)
{
    if (mt.n) k_proper_pairs<<<(uint32_t)((mt.n + 255) / 256), 256, 0, st>>>(mt, min_ins, max_ins, win_off, win_len,
                                                                              pair_of_rescue, ref_start, ref_end, pass, proper);
}

void launch_mate_flags(const uint32_t* win_len, uint64_t n, uint32_t* flag, cudaStream_t st)
{
    if (n) k_mate_flags<<<(uint32_t)((n + 255) / 256), 256, 0, st>>>(win_len, n, flag);
}

void launch_mate_pairs(const uint32_t* flag, const uint64_t* off, uint64_t n, uint32_t* pairs, uint32_t* pair_of_rescue,
                       cudaStream_t st)
{
    if (n) k_mate_pairs<<<(uint32_t)((n + 255) / 256), 256, 0, st>>>(flag, off, n, pairs, pair_of_rescue);
}

}  // namespace sdp
