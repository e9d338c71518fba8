// thin_kernel.cu -- a5/a6 for pairs whose score leaves room for few gap bases: one thread per pair.
//
// The forward score S bounds the gap content of every co-optimal alignment,
// W = floor((n*match - S - o) / e), so every co-optimal path lies in the
// band |i - j - (i_end - n)| <= W of rows (i_end - n - W, i_end]. For W = 0 the alignment is
// gapless: CIGAR nM, n_match from the score alone. For 1 <= W < THIN_NW (24) the band
// (2W+1 <= 47 columns) is recomputed with the paper's recurrences in the same
// x8 tagged integer domain as trace_kernel.cuh -- scalar int32 here, band cells in registers, the
// row loop fully unrolled over the band -- and leaves four direction bits per cell in a per-thread
// (hardware-interleaved, hence coalesced) local-memory array; the walk of PAPER.md:353 /
// DESIGN.md R6 then reads them back. Nothing of this uses the reverse pass.
#include "sdp_host.cuh"
#include "seq_bits.cuh"

namespace sdp {

namespace {

constexpr int TNEG = -(1 << 28);                  // "minus infinity", a multiple of 8

__device__ __forceinline__ int base_at(const uint32_t* __restrict__ packed, const uint32_t* __restrict__ nmask,
                                       uint64_t pos, int ncode) {
    int c = (int)((__ldg(packed + (pos >> 4)) >> (2u * ((uint32_t)pos & 15u))) & 3u);
    if (nmask != nullptr && ((__ldg(nmask + (pos >> 5)) >> ((uint32_t)pos & 31u)) & 1u)) c = ncode;
    return c;
}

}  // namespace

struct ThinConsts {
    int negOe;      // 8 * (-o) + 1
    int negOf;      // 8 * (-o) + 6
    int qm, qx;     // 8 * (2e + match) + 7, 8 * (2e + mismatch) + 7
    int e8;         // 8 * e
};

// W_ = gap-content bound of every pair of the launch (0 = gapless). MAXROWS bounds the rows of the
// band (n + W); pairs beyond it are classified onto the other paths by k_post_forward.
template <int W_, int MAXROWS>
__device__ __forceinline__ void thin_body(const TraceParams& tp, const ThinConsts& tc, const uint32_t first,
                                          const uint32_t count, const uint32_t k)
{
    constexpr int BW = 2 * W_ + 1;                 // band columns
    constexpr int WPR = (BW + 7) / 8;              // 32-bit words of direction nibbles per row
    if (k >= count) return;
    const uint32_t p = tp.order[first + k];
    const sdp_batch& b = tp.b;
    const uint32_t ri = b.pairs[2 * (uint64_t)p], wi = b.pairs[2 * (uint64_t)p + 1];
    const int n = (int)b.read_len[ri];
    const uint64_t roff = b.read_off[ri], woff = b.win_off[wi];
    const int i_end = tp.ref_end[p] + 1;
    const long long rwords = (long long)((b.reads_bases + 15) / 16), wwords = (long long)((b.wins_bases + 15) / 16);
    const long long rnwords = (long long)((b.reads_bases + 31) / 32), wnwords = (long long)((b.wins_bases + 31) / 32);
    uint32_t* ops = tp.ops_rev + tp.ops_off[p];
    constexpr uint32_t cap = 2u * (uint32_t)W_ + 3u;

    int n_match = 0, n_cols = 0, ref_start = 0;
    uint32_t nops = 0;
    int cur_op = -1; uint32_t cur_len = 0;
    bool bad = false;
    int gap_runs = 0, gap_bases = 0;
    auto emit = [&](int op, uint32_t len) {
        if (op == cur_op) { cur_len += len; return; }
        if (cur_op >= 0) {
            if (nops < cap) ops[nops] = (cur_len << 4) | (uint32_t)cur_op; else bad = true;
            ++nops;
            if (cur_op > 0) { ++gap_runs; gap_bases += (int)cur_len; }
        }
        cur_op = op; cur_len = len;
    };

    if constexpr (W_ == 0) {
        // gapless: every co-optimal alignment is ungapped, so the CIGAR is nM
        ref_start = i_end - n;
        if (ref_start < 0) { bad = true; ref_start = 0; }
        n_cols = n;
        emit(0, (uint32_t)n);
    } else {
        const int c = i_end - n;
        const int i_lo = max(0, c - W_);
        const int R = i_end - i_lo;
        uint32_t lbits[MAXROWS * WPR];
        int Hc[BW + 1], Fc[BW + 1];
        {   // row i_lo of the restricted problem: M(i_lo, 0) = 0, M(i_lo, j) = -(o + e j) (drift form: -o)
            const int jb0 = i_lo - c - W_;
#pragma unroll
            for (int jj = 0; jj <= BW; ++jj) {
                const int j = jj + jb0;
                Hc[jj] = (jj == BW || j < 0 || j > n) ? TNEG : (j == 0 ? 0 : tc.negOe - 1);
                Fc[jj] = TNEG + 2;
            }
        }
        // sliding buffer of the read: NSEG + 1 words of 16 bases (and their spread N bits) starting at read
        // position q0; row ir looks at the BW bases from position q0 + roffs on. Refilled every 16 rows.
        constexpr int NSEG = (BW + 15) / 16;
        long long q0 = (long long)(i_lo + 1 - c - W_) - 1;            // read position of segment bit 0 at row i_lo+1
        uint32_t rw[NSEG + 1], rnw[NSEG + 1];
#pragma unroll
        for (int sgm = 0; sgm <= NSEG; ++sgm) {
            rw[sgm] = bases16(b.reads_packed, (long long)roff + q0 + 16 * sgm, rwords);
            rnw[sgm] = nbits16_spread(b.read_nmask, (long long)roff + q0 + 16 * sgm, rnwords);
        }
        int roffs = 0;                                                // bases consumed from the buffer
        uint32_t tw = 0, twn = 0;
        int finH = TNEG;

        auto row = [&](const int ir, auto check_tag) {
            constexpr bool CHECK = decltype(check_tag)::value;
            const int i = i_lo + ir;
            const int jb = i - c - W_;
            const uint64_t tpos = woff + (uint64_t)(i - 1);
            if (ir == 1 || (tpos & 15u) == 0) tw = __ldg(b.wins_packed + (tpos >> 4));
            const uint32_t t = (tw >> (2u * ((uint32_t)tpos & 15u))) & 3u;
            uint32_t nm = 0;
            if (b.win_nmask != nullptr) {
                if (ir == 1 || (tpos & 31u) == 0) twn = __ldg(b.win_nmask + (tpos >> 5));
                if ((twn >> ((uint32_t)tpos & 31u)) & 1u) nm = 0x55555555u;
            }
            if (roffs == 16) {
                q0 += 16; roffs = 0;
#pragma unroll
                for (int sgm = 0; sgm < NSEG; ++sgm) { rw[sgm] = rw[sgm + 1]; rnw[sgm] = rnw[sgm + 1]; }
                rw[NSEG] = bases16(b.reads_packed, (long long)roff + q0 + 16 * NSEG, rwords);
                rnw[NSEG] = nbits16_spread(b.read_nmask, (long long)roff + q0 + 16 * NSEG, rnwords);
            }
            uint32_t eqw[NSEG];
#pragma unroll
            for (int sgm = 0; sgm < NSEG; ++sgm)
                eqw[sgm] = eq16(__funnelshift_r(rw[sgm], rw[sgm + 1], 2 * roffs), t * 0x55555555u,
                                nm | __funnelshift_r(rnw[sgm], rnw[sgm + 1], 2 * roffs));
            ++roffs;

            int Hl = TNEG, El = TNEG;
            uint32_t acc[WPR];
#pragma unroll
            for (int w = 0; w < WPR; ++w) acc[w] = 0u;
#pragma unroll
            for (int jj = 0; jj < BW; ++jj) {
                int Ft = __viaddmax_s32(Hc[jj + 1], tc.negOf, Fc[jj + 1]);
                int Et = __viaddmax_s32(Hl, tc.negOe, El);
                const int q = ((eqw[jj >> 4] >> (2 * (jj & 15))) & 1u) ? tc.qm : tc.qx;
                int Ht = __vimax3_s32(Hc[jj] + q, Ft, Et);
                if (CHECK) {
                    const int j = jb + jj;
                    if (j < 1 || j > n) { Ht = (j == 0) ? tc.e8 * ir : TNEG; Ft = TNEG + 2; Et = TNEG; }
                }
                const int Hn = Ht & ~7, Fn = Ft & ~4, En = Et & ~1;
                const uint32_t nib = (uint32_t)(((Ht & 3) | (Ft & 4)) + 8 * (Et - En));
                acc[jj >> 3] |= nib << (4 * (jj & 7));
                Hc[jj] = Hn; Fc[jj] = Fn; Hl = Hn; El = En;
                if (CHECK) { if (jb + jj == n) finH = Hn; }
            }
#pragma unroll
            for (int w = 0; w < WPR; ++w) lbits[(ir - 1) * WPR + w] = acc[w];
        };

        // rows whose band touches column 0 or column n+1 take the checked variant
        const int ir_a = min(R, max(0, c + W_ + 1 - i_lo - 1));        // last row with jb < 1
        const int ir_b = max(ir_a, min(R, c - W_ + n - i_lo));         // last row with jb + BW - 1 <= n
        int ir = 1;
        for (; ir <= ir_a; ++ir) row(ir, std::true_type{});
        for (; ir <= ir_b; ++ir) row(ir, std::false_type{});
        for (; ir <= R; ++ir) row(ir, std::true_type{});
        // the band DP must end on the forward score: H'(R, n) = 8 (S + e (R + n))
        if ((finH >> 3) - (tc.e8 >> 3) * (R + n) != tp.score[p]) bad = true;

        // walk back from (i_end, n)
        int i = i_end, j = n, st = 0;                                  // 0 = H, 1 = D, 2 = I
        while (j > 0) {
            if (i == i_lo) { emit(1, (uint32_t)j); n_cols += j; j = 0; break; }
            const int jj = j - (i - c - W_);
            if (jj < 0 || jj >= BW) { bad = true; break; }
            const uint32_t f = (lbits[(i - i_lo - 1) * WPR + (jj >> 3)] >> (4 * (jj & 7))) & 15u;
            if (st == 0) {
                if ((f & 3u) == 3u) {
                    emit(0, 1u); ++n_cols;
                    --i; --j;
                } else if ((f & 3u) == 2u) st = 1;
                else st = 2;
            } else if (st == 1) {
                emit(2, 1u); ++n_cols;
                if (f & 4u) st = 0;
                --i;
            } else {
                emit(1, 1u); ++n_cols;
                if (f & 8u) st = 0;
                --j;
            }
        }
        ref_start = i;
    }
    emit(-2, 0u);                                          // flush the last run
    {   // The path scores exactly S = match*n_match + mismatch*(M columns - n_match) - sum over gap runs of
        // (o + e*len), so n_match follows from the score without touching the sequences again
        // (N columns score mismatch and are not matches, consistently). A remainder means the walk is wrong.
        const int num = tp.score[p] + tp.sc.gap_open * gap_runs + tp.sc.gap_extend * gap_bases -
                        tp.sc.mismatch * (n_cols - gap_bases);
        const int den = tp.sc.match - tp.sc.mismatch;
        n_match = num / den;
        if (num < 0 || n_match * den != num || n_match > n_cols - gap_bases) bad = true;
    }
    if (bad) { atomicOr(tp.err_flag, SDP_ERRF_TRACE); nops = min(nops, cap); }
    tp.ref_start[p] = ref_start;
    tp.read_start[p] = 0;
    tp.read_end[p] = n - 1;
    tp.n_match[p] = n_match;
    tp.n_cols[p] = n_cols;
    tp.cigar_len[p] = nops;
    tp.pass[p] = ((long long)n_match * 1000000LL >= tp.sc.min_sim_q * (long long)n_cols) ? 1 : 0;
}

// Gap bounds LO..HI-1 in ONE launch: block b serves class w with
// r.block_start[w] <= b < r.block_start[w+1] (one small launch per class left the GPU mostly idle).
struct ThinRanges { uint32_t first[THIN_NW], count[THIN_NW], block_start[THIN_NW + 1]; };

template <int W_, int HI>
__device__ __forceinline__ void thin_dispatch(const int w, const TraceParams& tp, const ThinConsts& tc,
                                              const ThinRanges& r, const uint32_t k)
{
    if (w == W_) thin_body<W_, THIN_MAXROWS>(tp, tc, r.first[W_], r.count[W_], k);
    else if constexpr (W_ + 1 < HI) thin_dispatch<W_ + 1, HI>(w, tp, tc, r, k);
}

template <int LO, int HI>
__global__ void __launch_bounds__(128) k_thin_range(const TraceParams tp, const ThinConsts tc, const ThinRanges r)
{
    const uint32_t b = blockIdx.x + r.block_start[LO];
    int w = LO;
#pragma unroll
    for (int c = LO + 1; c < HI; ++c) w += (b >= r.block_start[c]) ? 1 : 0;
    const uint32_t k = (b - r.block_start[w]) * blockDim.x + threadIdx.x;
    thin_dispatch<LO, HI>(w, tp, tc, r, k);                // w is block-uniform
}

// bounds[w] .. bounds[w+1]: range of tp.order that holds the pairs with gap bound w
int launch_thin_all(const uint32_t* bounds, const TraceParams& tp, cudaStream_t st, cudaStream_t st_hi)
{
    ThinConsts tc;
    const int o = tp.sc.gap_open, e = tp.sc.gap_extend;
    tc.negOe = -8 * o + 1; tc.negOf = -8 * o + 6;
    tc.qm = 8 * (2 * e + tp.sc.match) + 7; tc.qx = 8 * (2 * e + tp.sc.mismatch) + 7; tc.e8 = 8 * e;
    ThinRanges r;
    uint32_t blocks = 0;
    for (int w = 0; w < THIN_NW; ++w) {
        r.first[w] = bounds[w]; r.count[w] = bounds[w + 1] - bounds[w];
        r.block_start[w] = blocks;
        blocks += (r.count[w] + 127) / 128;
    }
    r.block_start[THIN_NW] = blocks;
    int launched = 0;
    const uint32_t lo_blocks = r.block_start[THIN_SPLIT], hi_blocks = blocks - lo_blocks;
    // the wider bands on their own stream: few blocks that run long
    if (hi_blocks) { k_thin_range<THIN_SPLIT, THIN_NW><<<hi_blocks, 128, 0, st_hi>>>(tp, tc, r); ++launched; }
    if (lo_blocks) { k_thin_range<0, THIN_SPLIT><<<lo_blocks, 128, 0, st>>>(tp, tc, r); ++launched; }
    return launched;
}

}  // namespace sdp
