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
#include "score_kernel.cuh"      // the fp16-pipe delta helpers (hsub2_u, hfma2_relu_negsq, read_code_half, prmt_raw)

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

// ---------------------------------------------------------------------------------------------------------------------
// Local mode, int16x2: one warp scores TWO pairs (pair 2w in the low halves, pair 2w + 1 in the high halves) with the DPX
// max/add instructions, for reads up to 256 bases inside the value rule below. Same recurrences, same results as the
// int32 kernels (every quantity is exact in 16 bits under the rule); about 2.5 times their throughput.
//
// Per cell of two pairs, six ALU-pipe instructions. With beta = |mismatch|, every H carries +beta (the zero floor is the
// constant beta), D carries + e*i and I + e*(column within the lane), so that extending a gap needs no add:
//     D~ = max(S(i-1,j) + (e*i - oe - mismatch), D~(i-1,j))        S = H + beta + mismatch, the stored row
//     I~ = max(H^(i,j-1) + (e*jr - oe), I~(i,j-1))
//     a  = max(D~ - e*i, beta)         b = max(I~ - e*jr, a)         H^ = max(S(i-1,j-1) + q, b)
//     best = max(best, H^)
// q = match - mismatch or 0 comes from the FMA pipe (score_kernel.cuh: HADD2 + HFMA2.RELU on fp16 base codes), and so
// does S = H^ - beta as one 32-bit integer subtraction (no borrow between the halves: H^ >= beta in both).
// The position of the best cell: when a row raises the lane's best in one half, the lane notes the row number and keeps
// that half of the row's values (one LOP3 per column); the column is read off the kept row after the last step. Cells of padded read columns (a shorter partner, columns past n) and padded window rows hold
// N codes, which match nothing: such a cell never exceeds its real ancestors, all of which have a lower row or column,
// so it can tie but never win under the rule "highest score, then lowest row, then lowest column".
__device__ __forceinline__ uint32_t pack2(int v) { return ((uint32_t)v & 0xFFFFu) * 0x00010001u; }
// bitwise (mask ? b : a) in one LOP3
__device__ __forceinline__ uint32_t lop3_pick(uint32_t a, uint32_t b, uint32_t mask) {
    uint32_t r; asm("lop3.b32 %0, %1, %2, %3, 0xD8;" : "=r"(r) : "r"(a), "r"(b), "r"(mask)); return r;
}

// value rule of the int16x2 local kernel: largest stored magnitude match*n + beta + e*rows, and -(oe + e*rows) below
__device__ __forceinline__ bool local_i16_rule(const Scoring& sc, int n, int m) {
    const long long oe = (long long)sc.gap_open + sc.gap_extend;
    return n <= 256 && sc.match - sc.mismatch < 0x3C00 &&
           (long long)sc.match * n + (long long)sc.gap_extend * (m + 48) + 2 * oe - 2LL * sc.mismatch <= 32000;
}
// Does the int16x2 kernel score pair p (local mode)? Pairs 2w and 2w + 1 share a warp there when both reads fit and
// the rule holds for the larger of their lengths; a pair whose partner is absent or too long runs alone. Evaluated the
// same way by k_forward_local_i16 and by the int32 kernels, which skip what it takes.
__device__ __forceinline__ bool local_i16_taken(const sdp_batch& b, const Scoring& sc, uint64_t p, uint64_t n_pairs,
                                                const uint32_t* __restrict__ slow_words)
{
    const int n = (int)b.read_len[b.pairs[2 * p]], m = (int)b.win_len[b.pairs[2 * p + 1]];
    if (n > 256) return false;
    const uint64_t q = p ^ 1ull;
    if (q < n_pairs && slow_words[q] != 0) {
        const int nq = (int)b.read_len[b.pairs[2 * q]], mq = (int)b.win_len[b.pairs[2 * q + 1]];
        if (nq <= 256) return local_i16_rule(sc, max(n, nq), max(m, mq));
    }
    return local_i16_rule(sc, n, m);
}

// LANES = 32: the warp is one group (reads up to 256 bases); LANES = 16: two groups of 16 lanes, each with its own two
// pairs (reads up to 128 bases): the per-row work that does not depend on the column count (shuffles, row constants,
// selector expansion, best-cell bookkeeping) is then shared by four pairs instead of two.
template <int KC, int LANES>
__device__ __forceinline__ void forward_local_i16x2_warp(const sdp_batch& b, const Scoring& sc, const uint64_t pA,
                                                         const uint64_t pB, const bool hasA, const bool hasB,
                                                         int32_t* __restrict__ score, int32_t* __restrict__ ref_end,
                                                         int32_t* __restrict__ end_col)
{
    const int gl = (threadIdx.x & 31) & (LANES - 1);       // lane within the group
    int nA = 0, mA = 0, nB = 0, mB = 0;
    uint64_t roffA = 0, woffA = 0, roffB = 0, woffB = 0;
    if (hasA) {
        const uint32_t riA = b.pairs[2 * pA], wiA = b.pairs[2 * pA + 1];
        nA = (int)b.read_len[riA]; mA = (int)b.win_len[wiA];
        roffA = b.read_off[riA]; woffA = b.win_off[wiA];
    }
    if (hasB) {
        const uint32_t riB = b.pairs[2 * pB], wiB = b.pairs[2 * pB + 1];
        nB = (int)b.read_len[riB]; mB = (int)b.win_len[wiB];
        roffB = b.read_off[riB]; woffB = b.win_off[wiB];
    }
    const int e = sc.gap_extend, oe = sc.gap_open + sc.gap_extend, beta = -sc.mismatch;
    const int mmax = max(mA, mB);                          // rows of this group
    const int mwarp = LANES == 32 ? mmax : __reduce_max_sync(0xffffffffu, mmax);
    const int j0 = gl * KC;                                // this lane owns columns j0 + 1 .. j0 + KC of both pairs
    uint32_t S[KC], Dt[KC], rh[KC], ck[KC], negek[KC], snap[KC];
#pragma unroll
    for (int k = 0; k < KC; ++k) {
        const int j = j0 + k + 1;
        snap[k] = 0u;
        const uint32_t cA = j <= nA ? code_at(b.reads_packed, b.read_nmask, roffA + (uint64_t)(j - 1), SDP_CODE_READ_N) : SDP_CODE_READ_N;
        const uint32_t cB = j <= nB ? code_at(b.reads_packed, b.read_nmask, roffB + (uint64_t)(j - 1), SDP_CODE_READ_N) : SDP_CODE_READ_N;
        rh[k] = read_code_half(cA) | (read_code_half(cB) << 16);
        S[k] = 0u;                                         // M(0,j) = 0: S = 0 + beta + mismatch
        Dt[k] = pack2(beta - oe);                          // D(0,j): anything <= -oe + e acts as minus infinity under the zero floor
        ck[k] = pack2(e * (k + 1) - oe);
        negek[k] = pack2(-e * (k + 1));
    }
    const uint32_t BETA2 = pack2(beta), E2 = pack2(e), NEGE2 = pack2(-e), NEG2 = 0x80008000u, NEGEK2 = pack2(-e * KC);
    const uint32_t MISABS2 = (uint32_t)beta * 0x00010001u, Cd = pack2(sc.match - sc.mismatch);
    const uint32_t EDGE_I = pack2(beta - oe);              // I(i,0), in the frame of column 0
    const uint32_t one = opaque_u32(1u), NEGMIS2 = 0u - MISABS2;           // (a multiplier the compiler cannot fold: the add stays an IMAD)
    uint32_t ci = pack2(-e * gl - oe - sc.mismatch);       // e*i - oe - mismatch for the row before this lane's first step
    uint32_t negei = pack2(e * gl);
    uint32_t best = BETA2;
    int biA = 0, bjA = 0, biB = 0, bjB = 0;
    uint32_t h_out = BETA2, i_out = EDGE_I, sel_out = 0u;
    uint32_t diag = 0u;                                    // S(i-1, j0); row 0 is all zeros
    uint32_t wsel = 0u;
    const int steps = mwarp + LANES - 1;
    for (int s = 1; s <= steps; ++s) {
        if (((s - 1) & (LANES - 1)) == 0) {                // window codes of the next LANES rows, one row per lane, as PRMT selectors
            const int r = s + gl;
            const uint32_t cA = r <= mA ? code_at(b.wins_packed, b.win_nmask, woffA + (uint64_t)(r - 1), SDP_CODE_WIN_N) : SDP_CODE_WIN_N;
            const uint32_t cB = r <= mB ? code_at(b.wins_packed, b.win_nmask, woffB + (uint64_t)(r - 1), SDP_CODE_WIN_N) : SDP_CODE_WIN_N;
            wsel = cA * 0x11u | cB * 0x1100u;
        }
        const uint32_t sel0 = __shfl_sync(0xffffffffu, wsel, (s - 1) & (LANES - 1), LANES);
        uint32_t left = __shfl_up_sync(0xffffffffu, h_out, 1, LANES);
        uint32_t ileft = __shfl_up_sync(0xffffffffu, i_out, 1, LANES);
        uint32_t sel = __shfl_up_sync(0xffffffffu, sel_out, 1, LANES);
        ci = __viaddmax_s16x2(ci, E2, NEG2);               // packed add (max with the most negative value)
        negei = __viaddmax_s16x2(negei, NEGE2, NEG2);
        const int i = s - gl;
        if (gl == 0) { left = BETA2; ileft = EDGE_I; sel = sel0; }        // M(i,0) = 0, I(i,0) = -inf
        else ileft = __viaddmax_s16x2(ileft, NEGEK2, NEG2);               // from the left lane's column frame into this one
        if (i >= 1 && i <= mmax) {
            const uint32_t left_in = left, bprev = best;
            const uint32_t nt = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, sel);
#pragma unroll
            for (int k = 0; k < KC; ++k) {
                const uint32_t up = S[k];
                const uint32_t dt = __viaddmax_s16x2(up, ci, Dt[k]);
                const uint32_t it = __viaddmax_s16x2(left, ck[k], ileft);
                const uint32_t q = hfma2_relu_negsq(hsub2_u(nt, rh[k]), Cd);
                const uint32_t a = __viaddmax_s16x2(dt, negei, BETA2);
                const uint32_t bb = __viaddmax_s16x2(it, negek[k], a);
                const uint32_t h = __viaddmax_s16x2(diag, q, bb);
                diag = up;
                S[k] = imad_sel(h, one, NEGMIS2);          // h - beta per half, on the FMA pipe
                Dt[k] = dt; left = h; ileft = it;
                best = __vmaxs2(best, h);
            }
            if (best != bprev) {                           // this row raised the lane's best in one half or both:
                const uint32_t d = best ^ bprev;           // keep the row's values of that half; the column is read off at the end
                const uint32_t mask = ((d & 0xFFFFu) ? 0x0000FFFFu : 0u) | ((d >> 16) ? 0xFFFF0000u : 0u);
                if (mask & 0x0000FFFFu) biA = i;
                if (mask & 0xFFFF0000u) biB = i;
#pragma unroll
                for (int k = 0; k < KC; ++k) snap[k] = lop3_pick(snap[k], S[k], mask);
            }
            diag = left_in - MISABS2;                      // S(i, j0): the next row's diagonal neighbour
        }
        h_out = left; i_out = ileft; sel_out = sel;
    }
    int bA = (int)(int16_t)(best & 0xFFFFu) - beta, bB = (int)(int16_t)(best >> 16) - beta;
    {   // lowest column of the lane's best cell: the first entry of the kept row that equals the best (bi == 0: none)
        const uint32_t target = best - MISABS2;
#pragma unroll
        for (int k = KC - 1; k >= 0; --k) {
            if (biA && ((snap[k] ^ target) & 0xFFFFu) == 0u) bjA = j0 + k + 1;
            if (biB && ((snap[k] ^ target) >> 16) == 0u) bjB = j0 + k + 1;
        }
    }
    // over the lanes of the group, per pair: highest score, then lowest row, then lowest column
    for (int o = LANES / 2; o > 0; o >>= 1) {
        int ob = __shfl_down_sync(0xffffffffu, bA, o, LANES), oi = __shfl_down_sync(0xffffffffu, biA, o, LANES),
            oj = __shfl_down_sync(0xffffffffu, bjA, o, LANES);
        if (ob > bA || (ob == bA && (oi < biA || (oi == biA && oj < bjA)))) { bA = ob; biA = oi; bjA = oj; }
        ob = __shfl_down_sync(0xffffffffu, bB, o, LANES); oi = __shfl_down_sync(0xffffffffu, biB, o, LANES);
        oj = __shfl_down_sync(0xffffffffu, bjB, o, LANES);
        if (ob > bB || (ob == bB && (oi < biB || (oi == biB && oj < bjB)))) { bB = ob; biB = oi; bjB = oj; }
    }
    if (gl == 0) {
        if (hasA) { score[pA] = bA; ref_end[pA] = biA - 1; end_col[pA] = bjA; }        // S == 0: row 0, column 0 -> ref_end -1
        if (hasB) { score[pB] = bB; ref_end[pB] = biB - 1; end_col[pB] = bjB; }
    }
}

// Four consecutive pairs q0 .. q0 + 3 share one warp (two groups of 16 lanes) when every one of them that exists goes to
// the int16x2 kernel and has a read of at most 128 bases. *nmax receives the longest read.
__device__ __forceinline__ bool local_i16_quad(const sdp_batch& b, const Scoring& sc, uint64_t q0, uint64_t n_pairs,
                                               const uint32_t* __restrict__ slow_words, int* nmax)
{
    int nm = 0;
    for (int t = 0; t < 4; ++t) {
        const uint64_t p = q0 + (uint64_t)t;
        if (p >= n_pairs) break;
        if (slow_words[p] == 0) return false;
        const int n = (int)b.read_len[b.pairs[2 * p]];
        if (n > 128 || !local_i16_taken(b, sc, p, n_pairs, slow_words)) return false;
        nm = max(nm, n);
    }
    *nmax = nm;
    return true;
}

#define SDP_LOCAL_I16_DISPATCH(KEXPR, LANES_, ...)                                                      \
    switch (KEXPR) {                                                                                    \
    case 1: forward_local_i16x2_warp<1, LANES_>(__VA_ARGS__); break;                                    \
    case 2: forward_local_i16x2_warp<2, LANES_>(__VA_ARGS__); break;                                    \
    case 3: forward_local_i16x2_warp<3, LANES_>(__VA_ARGS__); break;                                    \
    case 4: forward_local_i16x2_warp<4, LANES_>(__VA_ARGS__); break;                                    \
    case 5: forward_local_i16x2_warp<5, LANES_>(__VA_ARGS__); break;                                    \
    case 6: forward_local_i16x2_warp<6, LANES_>(__VA_ARGS__); break;                                    \
    case 7: forward_local_i16x2_warp<7, LANES_>(__VA_ARGS__); break;                                    \
    default: forward_local_i16x2_warp<8, LANES_>(__VA_ARGS__); break;                                   \
    }

// QUAD = true: warp w takes pairs 4w .. 4w + 3 if local_i16_quad says so; QUAD = false: warp w takes pairs 2w, 2w + 1
// unless their quad went to the other kernel. Every decision is warp-uniform.
template <bool QUAD>
__global__ void __launch_bounds__(256) k_forward_local_i16(const sdp_batch b, const Scoring sc, uint64_t n_pairs,
                                                           const uint32_t* __restrict__ slow_words,
                                                           int32_t* __restrict__ score, int32_t* __restrict__ ref_end,
                                                           int32_t* __restrict__ end_col)
{
    const uint64_t w = ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    int nmax = 0;
    if (QUAD) {
        const uint64_t q0 = 4ull * w;
        if (q0 >= n_pairs || !local_i16_quad(b, sc, q0, n_pairs, slow_words, &nmax)) return;
        const uint64_t pA = q0 + 2ull * (uint64_t)((threadIdx.x & 31) >> 4), pB = pA + 1;
        const bool hasA = pA < n_pairs, hasB = pB < n_pairs;
        SDP_LOCAL_I16_DISPATCH((nmax + 15) >> 4, 16, b, sc, pA, pB, hasA, hasB, score, ref_end, end_col)
    } else {
        const uint64_t p0 = 2ull * w;
        if (p0 >= n_pairs) return;
        if (local_i16_quad(b, sc, p0 & ~3ull, n_pairs, slow_words, &nmax)) return;
        const bool runA = slow_words[p0] != 0 && local_i16_taken(b, sc, p0, n_pairs, slow_words);
        const bool runB = p0 + 1 < n_pairs && slow_words[p0 + 1] != 0 && local_i16_taken(b, sc, p0 + 1, n_pairs, slow_words);
        if (!runA && !runB) return;
        nmax = max(runA ? (int)b.read_len[b.pairs[2 * p0]] : 0, runB ? (int)b.read_len[b.pairs[2 * (p0 + 1)]] : 0);
        SDP_LOCAL_I16_DISPATCH((nmax + 31) >> 5, 32, b, sc, p0, p0 + 1, runA, runB, score, ref_end, end_col)
    }
}
#undef SDP_LOCAL_I16_DISPATCH

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
        if (local && local_i16_taken(b, sc, p, n_pairs, slow_words)) return;      // k_forward_local_i16 scores it
        if (n <= 128) forward_i32_warp<4>(b, sc, local, p, score, ref_end, end_col);
        else          forward_i32_warp<8>(b, sc, local, p, score, ref_end, end_col);
    }
}

void launch_forward_i32(const sdp_batch& b, const Scoring& sc, int local, const uint32_t* slow_words, const uint64_t* slow_off,
                        int32_t* rows, int32_t* score, int32_t* ref_end, int32_t* end_col, cudaStream_t st)
{
    if (b.n_pairs) {
        const uint32_t wgrid = (uint32_t)((b.n_pairs * 32 + 255) / 256);
        if (local) {    // int16x2 DPX instructions where the reads and the values fit: four or two pairs per warp
            k_forward_local_i16<true><<<(uint32_t)(((b.n_pairs + 3) / 4 * 32 + 255) / 256), 256, 0, st>>>(b, sc, b.n_pairs, slow_words,
                                                                                                        score, ref_end, end_col);
            k_forward_local_i16<false><<<(uint32_t)(((b.n_pairs + 1) / 2 * 32 + 255) / 256), 256, 0, st>>>(b, sc, b.n_pairs, slow_words,
                                                                                                         score, ref_end, end_col);
        }
        k_forward_i32_warp<false><<<wgrid, 256, 0, st>>>(b, sc, local, b.n_pairs, slow_words, score, ref_end, end_col);
        k_forward_i32_warp<true><<<wgrid, 256, 0, st>>>(b, sc, local, b.n_pairs, slow_words, score, ref_end, end_col);
        k_forward_i32<<<(uint32_t)((b.n_pairs + 63) / 64), 64, 0, st>>>(b, sc, local, b.n_pairs, slow_words, slow_off, rows, score,
                                                                       ref_end, end_col);
    }
}

}  // namespace sdp
