// slow_lane.cu -- the int32 lane and the local / soft-clipping variant (8(f2)).
//
// The int16x2 DPX kernels take pairs inside the int16 range rule of sdp.h with reads up to SDP_MAX_READ_LEN. Every
// other pair -- longer reads, windows past the rule (the paper enforces no maximum read length) -- and
// every pair of a context in SDP_MODE_LOCAL is scored here with the paper's recurrences in plain
// int32, one thread per pair, row arrays of M and D in global scratch: slow, exact, never clamped. The traceback of
// these pairs is k_traceback_dyn (traceback.cu).
//
// Local variant (R18; the paper names Smith-Waterman, and soft-clipped alignments,
// PAPER.md:228): M(i,0) = M(0,j) = 0, M(i,j) = max(0, ...), S = max over all cells, lowest row then lowest column.
#include "sdp_host.cuh"

namespace sdp {

namespace {

constexpr int SNEG = -(1 << 29);

__device__ __forceinline__ uint32_t code_at(const uint32_t* __restrict__ packed, const uint32_t* __restrict__ nmask,
                                            uint64_t pos, uint32_t ncode) {
    uint32_t c = (__ldg(packed + (pos >> 4)) >> (2u * ((uint32_t)pos & 15u))) & 3u;
    if (nmask != nullptr && ((__ldg(nmask + (pos >> 5)) >> ((uint32_t)pos & 31u)) & 1u)) c = ncode;
    return c;
}

}  // namespace

// one thread per pair of the batch; pairs with slow_off[p + 1] == slow_off[p] (not routed here) return at once
__global__ void __launch_bounds__(64) k_forward_i32(const sdp_batch b, const Scoring sc, int local, uint64_t n_pairs,
                                                    const uint32_t* __restrict__ slow_words,
                                                    const uint64_t* __restrict__ slow_off, int32_t* __restrict__ rows,
                                                    int32_t* __restrict__ score, int32_t* __restrict__ ref_end,
                                                    int32_t* __restrict__ end_col)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs || slow_words[p] == 0) return;
    const uint32_t ri = b.pairs[2 * p], wi = b.pairs[2 * p + 1];
    const int n = (int)b.read_len[ri], m = (int)b.win_len[wi];
    const uint64_t roff = b.read_off[ri], woff = b.win_off[wi];
    int32_t* Hr = rows + slow_off[p];                      // M(i-1, 0..n) -> M(i, 0..n) in place
    int32_t* Dr = Hr + (n + 1);                            // D(i-1, .)   -> D(i, .)
    const int oe = sc.gap_open + sc.gap_extend, e = sc.gap_extend;
    // row 0 (local: zeros)
    Hr[0] = 0; Dr[0] = SNEG;
    for (int j = 1; j <= n; ++j) { Hr[j] = local ? 0 : -(sc.gap_open + e * j); Dr[j] = SNEG; }
    int best = local ? 0 : SNEG, bi = 0, bj = local ? 0 : n;
    for (int i = 1; i <= m; ++i) {
        const uint32_t t = code_at(b.wins_packed, b.win_nmask, woff + (uint64_t)(i - 1), SDP_CODE_WIN_N);
        int diag = Hr[0];                                  // M(i-1, 0) = 0
        int left = 0, ileft = SNEG;                        // M(i, 0) = 0, I(i, 0) = -inf
        for (int j = 1; j <= n; ++j) {
            const uint32_t r = code_at(b.reads_packed, b.read_nmask, roff + (uint64_t)(j - 1), SDP_CODE_READ_N);
            const int up = Hr[j];
            const int vd = max(up - oe, Dr[j] - e);
            const int vi = max(left - oe, ileft - e);
            int h = max(diag + (r == t ? sc.match : sc.mismatch), max(vd, vi));
            if (local) h = max(h, 0);
            diag = up;
            Hr[j] = h; Dr[j] = vd; left = h; ileft = vi;
            if (local && h > best) { best = h; bi = i; bj = j; }       // row-major: lowest row, then lowest column
        }
        if (!local && left > best) { best = left; bi = i; }             // max over 1 <= i <= m of M(i,n), lowest row
    }
    score[p] = best;
    ref_end[p] = bi - 1;                                   // local with S == 0: -1
    end_col[p] = bj;                                       // local: column of the end cell (0 when S == 0); else n
}

void launch_forward_i32(const sdp_batch& b, const Scoring& sc, int local, const uint32_t* slow_words, const uint64_t* slow_off,
                        int32_t* rows, int32_t* score, int32_t* ref_end, int32_t* end_col, cudaStream_t st)
{
    if (b.n_pairs)
        k_forward_i32<<<(uint32_t)((b.n_pairs + 63) / 64), 64, 0, st>>>(b, sc, local, b.n_pairs, slow_words, slow_off, rows, score,
                                                                       ref_end, end_col);
}

}  // namespace sdp
