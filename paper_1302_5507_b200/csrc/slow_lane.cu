// slow_lane.cu -- the int32 lane and the local / soft-clipping variant (8(f2)).
//
// The int16x2 DPX kernels take pairs inside the int16 range rule of sdp.h with reads up to SDP_MAX_READ_LEN. Every
// other pair -- longer reads, windows past the rule (the paper enforces no maximum read length) -- and
// every pair of a context in SDP_MODE_LOCAL is scored here with the paper's recurrences in plain
// int32: one WARP per pair with the row state in registers for reads up to 1,024 bases (k_forward_i32_warp), one thread
// per pair with the row arrays of M and D in global scratch beyond that (k_forward_i32). Exact, never clamped. The
// traceback of these pairs is k_traceback<0, .> (traceback.cu).
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
    if (n <= 1024) return;                                 // k_forward_i32_warp takes these
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

// One WARP per pair, for reads up to 32 * 32 bases: lane l owns KC consecutive read columns (H and D of the previous
// row in registers), the window streams by as rows, lane l works on row s - l at step s (anti-diagonal wavefront) and
// hands M(i, last column), I(i, last column) and the row's window base to lane l + 1 with three shuffles per row.
// Same recurrences, same int32 arithmetic and the same tie rules as k_forward_i32 (lowest row, then lowest column),
// about twelve times its throughput: no row array ever goes to memory.
template <int KC>
__device__ __forceinline__ void forward_i32_warp(const sdp_batch& b, const Scoring& sc, const int local, const uint64_t p,
                                                 int32_t* __restrict__ score, int32_t* __restrict__ ref_end,
                                                 int32_t* __restrict__ end_col)
{
    const int lane = threadIdx.x & 31;
    const uint32_t ri = b.pairs[2 * p], wi = b.pairs[2 * p + 1];
    const int n = (int)b.read_len[ri], m = (int)b.win_len[wi];
    const uint64_t roff = b.read_off[ri], woff = b.win_off[wi];
    const int oe = sc.gap_open + sc.gap_extend, e = sc.gap_extend;
    const int j0 = lane * KC;                              // this lane owns columns j0 + 1 .. j0 + KC
    int H[KC], D[KC];
    uint32_t rc[KC];
#pragma unroll
    for (int k = 0; k < KC; ++k) {
        const int j = j0 + k + 1;
        rc[k] = j <= n ? code_at(b.reads_packed, b.read_nmask, roff + (uint64_t)(j - 1), SDP_CODE_READ_N) : 7u;   // 7: matches nothing
        H[k] = local ? 0 : -(sc.gap_open + e * j);         // row 0 (local: zeros)
        D[k] = SNEG;
    }
    int best = local ? 0 : SNEG, bi = 0, bj = local ? 0 : n;
    int h_out = 0, i_out = SNEG;                           // M(i, last column), I(i, last column) of the row just done
    int diag = lane == 0 ? 0 : (local ? 0 : -(sc.gap_open + e * j0));   // M(i-1, j0)
    uint32_t t_out = 0;
    const int steps = m + 31;
    for (int s = 1; s <= steps; ++s) {
        int left = __shfl_up_sync(0xffffffffu, h_out, 1);
        int ileft = __shfl_up_sync(0xffffffffu, i_out, 1);
        uint32_t t = __shfl_up_sync(0xffffffffu, t_out, 1);
        const int i = s - lane;
        if (lane == 0) {
            left = 0; ileft = SNEG;                        // M(i, 0) = 0, I(i, 0) = -inf
            t = i <= m ? code_at(b.wins_packed, b.win_nmask, woff + (uint64_t)(i - 1), SDP_CODE_WIN_N) : 0u;
        }
        if (i >= 1 && i <= m) {
            const int left_in = left;
#pragma unroll
            for (int k = 0; k < KC; ++k) {
                const int j = j0 + k + 1;
                const int up = H[k];
                const int vd = max(up - oe, D[k] - e);
                const int vi = max(left - oe, ileft - e);
                int h = max(diag + (rc[k] == t ? sc.match : sc.mismatch), max(vd, vi));
                if (local) h = max(h, 0);
                diag = up;
                H[k] = h; D[k] = vd; left = h; ileft = vi;
                if (local) { if (j <= n && h > best) { best = h; bi = i; bj = j; } }   // this lane's cells in row-major order
                else if (j == n && h > best) { best = h; bi = i; }                     // max over i of M(i,n), lowest row
            }
            diag = left_in;                                // M(i, j0) is the next row's diagonal neighbour
        }
        h_out = left; i_out = ileft; t_out = t;
    }
    // over the lanes: highest score, then lowest row, then lowest column
    for (int o = 16; o > 0; o >>= 1) {
        const int ob = __shfl_down_sync(0xffffffffu, best, o);
        const int oi = __shfl_down_sync(0xffffffffu, bi, o);
        const int oj = __shfl_down_sync(0xffffffffu, bj, o);
        if (ob > best || (ob == best && (oi < bi || (oi == bi && oj < bj)))) { best = ob; bi = oi; bj = oj; }
    }
    if (lane == 0) {
        score[p] = best;
        ref_end[p] = bi - 1;                               // local with S == 0: -1
        end_col[p] = bj;                                   // local: column of the end cell (0 when S == 0); else n
    }
}

// LARGE = false: reads up to 256 bases (4 or 8 columns per lane); true: up to 1,024 (16 or 32). Two kernels because
// their register budgets differ by a factor of three.
template <bool LARGE>
__global__ void __launch_bounds__(256) k_forward_i32_warp(const sdp_batch b, const Scoring sc, int local, uint64_t n_pairs,
                                                          const uint32_t* __restrict__ slow_words,
                                                          int32_t* __restrict__ score, int32_t* __restrict__ ref_end,
                                                          int32_t* __restrict__ end_col)
{
    const uint64_t p = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (p >= n_pairs || slow_words[p] == 0) return;        // warp-uniform
    const int n = (int)b.read_len[b.pairs[2 * p]];
    if (LARGE) {
        if (n <= 256 || n > 1024) return;                  // (longer reads: k_forward_i32)
        if (n <= 512) forward_i32_warp<16>(b, sc, local, p, score, ref_end, end_col);
        else          forward_i32_warp<32>(b, sc, local, p, score, ref_end, end_col);
    } else {
        if (n > 256) return;
        if (n <= 128) forward_i32_warp<4>(b, sc, local, p, score, ref_end, end_col);
        else          forward_i32_warp<8>(b, sc, local, p, score, ref_end, end_col);
    }
}

void launch_forward_i32(const sdp_batch& b, const Scoring& sc, int local, const uint32_t* slow_words, const uint64_t* slow_off,
                        int32_t* rows, int32_t* score, int32_t* ref_end, int32_t* end_col, cudaStream_t st)
{
    if (b.n_pairs) {
        const uint32_t wgrid = (uint32_t)((b.n_pairs * 32 + 255) / 256);
        k_forward_i32_warp<false><<<wgrid, 256, 0, st>>>(b, sc, local, b.n_pairs, slow_words, score, ref_end, end_col);
        k_forward_i32_warp<true><<<wgrid, 256, 0, st>>>(b, sc, local, b.n_pairs, slow_words, score, ref_end, end_col);
        k_forward_i32<<<(uint32_t)((b.n_pairs + 63) / 64), 64, 0, st>>>(b, sc, local, b.n_pairs, slow_words, slow_off, rows, score,
                                                                       ref_end, end_col);
    }
}

}  // namespace sdp
