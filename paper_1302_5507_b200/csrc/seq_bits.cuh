// seq_bits.cuh -- word-parallel helpers on the 2-bit packed sequences and their N bitmaps, shared by the
// narrow-band traceback (thin_kernel.cu) and the post-forward classification (traceback.cu).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sdp {

// 16 consecutive 2-bit bases starting at base position pos; words outside [0, nwords) read as 0
__device__ __forceinline__ uint32_t bases16(const uint32_t* __restrict__ packed, long long pos, long long nwords) {
    const long long w = pos >> 4;
    const uint32_t sh = ((uint32_t)pos & 15u) * 2u;
    const uint32_t lo = (w >= 0 && w < nwords) ? __ldg(packed + w) : 0u;
    const uint32_t hi = (sh != 0u && w + 1 >= 0 && w + 1 < nwords) ? __ldg(packed + w + 1) : 0u;
    return __funnelshift_r(lo, hi, sh);
}
// 16 consecutive mask bits starting at bit position pos, spread to the even bit positions
__device__ __forceinline__ uint32_t nbits16_spread(const uint32_t* __restrict__ bits, long long pos, long long nwords) {
    if (bits == nullptr) return 0u;
    const long long w = pos >> 5;
    const uint32_t sh = (uint32_t)pos & 31u;
    const uint32_t lo = (w >= 0 && w < nwords) ? __ldg(bits + w) : 0u;
    const uint32_t hi = (sh > 16u && w + 1 >= 0 && w + 1 < nwords) ? __ldg(bits + w + 1) : 0u;
    uint32_t x = __funnelshift_r(lo, hi, sh) & 0xFFFFu;
    x = (x | (x << 8)) & 0x00FF00FFu;
    x = (x | (x << 4)) & 0x0F0F0F0Fu;
    x = (x | (x << 2)) & 0x33333333u;
    x = (x | (x << 1)) & 0x55555555u;
    return x;
}
// even bit 2k set iff base k of a and of b are equal (N never equal)
__device__ __forceinline__ uint32_t eq16(uint32_t a, uint32_t b, uint32_t nmask_spread) {
    const uint32_t x = a ^ b;
    return ~(x | (x >> 1) | nmask_spread) & 0x55555555u;
}


// matches (N never matches) between n read bases from base position rpos and n window bases from wpos
__device__ __forceinline__ int count_equal_bases(const uint32_t* __restrict__ reads, const uint32_t* __restrict__ read_nmask,
                                                 long long rpos, long long rwords, long long rnwords,
                                                 const uint32_t* __restrict__ wins, const uint32_t* __restrict__ win_nmask,
                                                 long long wpos, long long wwords, long long wnwords, int n)
{
    int eqc = 0;
    for (int j0 = 0; j0 < n; j0 += 16) {
        const uint32_t r = bases16(reads, rpos + j0, rwords);
        const uint32_t t = bases16(wins, wpos + j0, wwords);
        const uint32_t nm = nbits16_spread(read_nmask, rpos + j0, rnwords) | nbits16_spread(win_nmask, wpos + j0, wnwords);
        uint32_t eq = eq16(r, t, nm);
        if (n - j0 < 16) eq &= (1u << (2 * (n - j0))) - 1u;
        eqc += __popc(eq);
    }
    return eqc;
}

}  // namespace sdp
