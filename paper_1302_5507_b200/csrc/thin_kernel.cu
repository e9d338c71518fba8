// thin_kernel.cu -- a5/a6 for pairs whose score leaves room for few gap bases.
//
// The forward score S bounds the gap content of every co-optimal alignment,
// W = floor((n*match - S - o) / e), so every co-optimal path lies in the
// band |i - j - (i_end - n)| <= W of rows (i_end - n - W, i_end]. For W = 0 the alignment is
// gapless: CIGAR nM, n_match from the score alone, one thread per pair. For 1 <= W < THIN_NW (24) the band
// (2W+1 <= 47 columns) is recomputed with the paper's recurrences in the x8 tagged
// int16x2 domain of trace_kernel.cuh: ONE THREAD OWNS TWO PAIRS (the two 16-bit lanes of every register), the
// band cells of H and F stay in registers in band coordinates (cell jj of row i is read column
// j = i - (i_end - n) - W + jj, so "up" is slot jj+1 and "diagonal" is slot jj of the previous row and nothing is
// ever moved), the row body is fully unrolled over the band, and each cell leaves four direction bits in a
// per-thread (hardware-interleaved, hence coalesced) local-memory array that the walk of PAPER.md:353 /
// DESIGN.md R6 reads back. Nothing of this uses the reverse pass.
//
// Per cell and per TWO pairs the ALU pipe sees 4 DPX + 4 LOP3 (c = 2e + mismatch, q' = delta - mismatch,
// tags diag 7 > D opened 6 > D extended 2 > I opened 1 > I extended 0 in the low three bits, every value x8):
//     Ft = max(H7(i-1,j) + 8(-o-c) - 1, Fc(i-1,j))      VIADDMNMX    Fc = Ft & ~4   (F~ = F' - c, tag 2)
//     u  = max(H7(i-1,j-1) + 8q', Ft)                   VIADDMNMX    H7 = H | 7: the diagonal tag rides on H itself
//     Et = max(H7(i,j-1) - 8o - 6, Ec(i,j-1))           VIADDMNMX    Ec = Et & ~1
//     Ht = max(u + 8c, Et)                              VIADDMNMX    H7 = Ht | 7
// and the fp16/FMA pipe delivers q' (HADD2 + HFMA2.RELU on fp16 base codes, exact: score_kernel.cuh) and packs
// the nibble (7 - (Ht&3 | Ft&4)) + 8 (Et&1) of four cells into 16 bits per lane with integer and denormal-fp16
// multiply-adds. The scalar int32 version this replaces spent about 14 ALU instructions per cell of ONE pair.
#include "sdp_host.cuh"
#include "seq_bits.cuh"
#include "score_kernel.cuh"

namespace sdp {

namespace {

__device__ __forceinline__ uint32_t t_imad(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r; asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c)); return r;
}
// bitwise (mask ? b : a) in one LOP3
__device__ __forceinline__ uint32_t t_select(uint32_t a, uint32_t b, uint32_t mask) {
    uint32_t r; asm("lop3.b32 %0, %1, %2, %3, 0xD8;" : "=r"(r) : "r"(a), "r"(b), "r"(mask)); return r;
}
// 16 consecutive mask bits starting at bit position pos (0 when there is no mask)
__device__ __forceinline__ uint32_t nbits16(const uint32_t* __restrict__ bits, long long pos, long long nwords) {
    if (bits == nullptr) return 0u;
    const long long w = pos >> 5;
    const uint32_t sh = (uint32_t)pos & 31u;
    const uint32_t lo = (w >= 0 && w < nwords) ? __ldg(bits + w) : 0u;
    const uint32_t hi = (sh > 16u && w + 1 >= 0 && w + 1 < nwords) ? __ldg(bits + w + 1) : 0u;
    return __funnelshift_r(lo, hi, sh) & 0xFFFFu;
}
// 16 bases of lane A (word a) and lane B (word b), N bits na / nb, -> sixteen 16-bit PRMT selectors
// (index of A doubled in the low byte, of B in the high byte), two per output word; N takes table index ncode.
__device__ __forceinline__ void expand16(uint32_t a, uint32_t b, uint32_t na, uint32_t nb, uint32_t ncode, uint32_t (&out)[8]) {
#pragma unroll
    for (int tt = 0; tt < 8; ++tt) {
        const uint32_t x = (a >> (4 * tt)) & 0xFu, y = (b >> (4 * tt)) & 0xFu;
        uint32_t w = ((x * 0x44011u) & 0x00330033u) | (((y * 0x44011u) << 8) & 0x33003300u);
        if (na | nb) {
            const uint32_t ma = (na >> (2 * tt)) & 3u, mb = (nb >> (2 * tt)) & 3u, nn = ncode * 0x11u;
            if (ma & 1u) w = (w & 0xFFFFFF00u) | nn;
            if (ma & 2u) w = (w & 0xFF00FFFFu) | (nn << 16);
            if (mb & 1u) w = (w & 0xFFFF00FFu) | (nn << 8);
            if (mb & 2u) w = (w & 0x00FFFFFFu) | (nn << 24);
        }
        out[tt] = w;
    }
}

}  // namespace

struct ThinConsts {
    uint32_t negOf;     // packed 8 (-o - c) - 1 : H7 -> "D opened here" candidate, tag 6
    uint32_t negOe;     // packed -8 o - 6      : H7 -> "I opened here" candidate, tag 1
    uint32_t c8;        // packed 8 c, c = 2e + mismatch
    uint32_t Cd8;       // packed 8 (match - mismatch), read as an fp16 pair (< 1.0)
    uint32_t e8;        // packed 8 e
    uint32_t hb0;       // packed 8 beta + 7          : H7(i_lo, 0)
    uint32_t hrow0;     // packed 8 (beta - o) + 7    : H7(i_lo, j >= 1)
    int beta, e;
};

// per pair geometry: j = ir - off - W + jj for row ir (1-based from i_lo) and band slot jj; rows R = n + off
struct ThinPair {
    uint32_t p;
    int n, i_end, off, R;
    uint64_t roff, woff;
};

template <int W_>
__device__ __forceinline__ ThinPair thin_pair(const TraceParams& tp, uint32_t p) {
    const sdp_batch& b = tp.b;
    const uint32_t ri = b.pairs[2 * (uint64_t)p], wi = b.pairs[2 * (uint64_t)p + 1];
    ThinPair t;
    t.p = p;
    t.n = (int)b.read_len[ri];
    t.roff = b.read_off[ri]; t.woff = b.win_off[wi];
    t.i_end = tp.ref_end[p] + 1;
    const int c = t.i_end - t.n;
    const int i_lo = max(0, c - W_);
    t.off = c - i_lo;
    t.R = t.i_end - i_lo;
    return t;
}

// W_ = 0: gapless, one pair per thread
__device__ __forceinline__ void thin_gapless(const TraceParams& tp, const uint32_t p) {
    const sdp_batch& b = tp.b;
    const uint32_t ri = b.pairs[2 * (uint64_t)p];
    const int n = (int)b.read_len[ri];
    const int i_end = tp.ref_end[p] + 1;
    bool bad = false;
    int ref_start = i_end - n;
    if (ref_start < 0) { bad = true; ref_start = 0; }
    tp.ops_rev[tp.ops_off[p]] = ((uint32_t)n << 4);
    // S = match*n_match + mismatch*(n - n_match)
    const int num = tp.score[p] - tp.sc.mismatch * n, den = tp.sc.match - tp.sc.mismatch;
    const int n_match = num / den;
    if (num < 0 || n_match * den != num || n_match > n) bad = true;
    if (bad) atomicOr(tp.err_flag, SDP_ERRF_TRACE);
    tp.ref_start[p] = ref_start;
    tp.read_start[p] = 0;
    tp.read_end[p] = n - 1;
    tp.n_match[p] = n_match;
    tp.n_cols[p] = n;
    tp.cigar_len[p] = 1;
    tp.pass[p] = ((long long)n_match * 1000000LL >= tp.sc.min_sim_q * (long long)n) ? 1 : 0;
}

// ---- the two walks back from (i_end, n), interleaved, then the per-pair results: ONE copy of this code serves every
// band width (the band DP above is instantiated per W; this is not, which keeps the kernels' code small).
// The nibbles sit in local memory (an L2 round trip per dependent load), so each walk fetches the words of EIGHT rows
// at once -- the rows above the current cell in the same band-slot word, which is where a diagonal step, the common
// one, stays -- and the two walks' loads are in flight together.
constexpr int WALK_ROWS = 8;      // (16: measured no faster)
__device__ __noinline__ void thin_walks(const TraceParams& tp, const ThinConsts& tc, const ThinPair& A, const ThinPair& B,
                                        const bool writeB, const uint32_t* lbits, const int W, const uint32_t finH)
{
    const int BW = 2 * W + 1, WPR = (BW + 3) / 4;
    const int n = A.n, off = A.off, R = A.R;
    struct Walk {
        int i, j, st, n_cols, gap_runs, gap_bases, cur_op, c_row, c_wc;
        uint32_t cur_len, nops;
        bool bad, live;
        uint32_t c[WALK_ROWS];
        uint32_t* ops;
    };
    const uint32_t cap = 2u * (uint32_t)W + 3u;
    Walk w[2];
#pragma unroll
    for (int lane = 0; lane < 2; ++lane) {
        const ThinPair& T = lane ? B : A;
        Walk& x = w[lane];
        x.i = R; x.j = n; x.st = 0; x.n_cols = 0; x.gap_runs = 0; x.gap_bases = 0; x.cur_op = -1; x.cur_len = 0; x.nops = 0;
        x.c_row = -100; x.c_wc = -1;
        x.live = lane == 0 || writeB;
        x.ops = tp.ops_rev + tp.ops_off[T.p];
        // the band DP must end on the forward score: H'(R, n) = 8 (S + e (R + n) + beta) + 7
        const int f = (int)((finH >> (16 * lane)) & 0xFFFFu) >> 3;
        x.bad = (f - tc.beta - tc.e * (R + n) != tp.score[T.p]);
#pragma unroll
        for (int k = 0; k < WALK_ROWS; ++k) x.c[k] = 0u;
    }
    auto emit = [&](Walk& x, int op, uint32_t len) {
        if (op == x.cur_op) { x.cur_len += len; return; }
        if (x.cur_op >= 0) {
            if (x.nops < cap) x.ops[x.nops] = (x.cur_len << 4) | (uint32_t)x.cur_op; else x.bad = true;
            ++x.nops;
            if (x.cur_op > 0) { ++x.gap_runs; x.gap_bases += (int)x.cur_len; }
        }
        x.cur_op = op; x.cur_len = len;
    };
#pragma unroll 1
    while (w[0].live || w[1].live) {
#pragma unroll
        for (int lane = 0; lane < 2; ++lane) {             // make sure the cached rows cover the current cell
            Walk& x = w[lane];
            if (!x.live) continue;
            if (x.i == 0) { emit(x, 1, (uint32_t)x.j); x.n_cols += x.j; x.j = 0; x.live = false; continue; }   // row i_lo: all insertions
            const int jj = x.j - (x.i - off - W);
            if (jj < 0 || jj >= BW) { x.bad = true; x.live = false; continue; }
            const int wc = jj >> 2, d = x.c_row - (x.i - 1);
            if (wc != x.c_wc || d < 0 || d >= WALK_ROWS) {
                x.c_row = x.i - 1; x.c_wc = wc;
#pragma unroll
                for (int k = 0; k < WALK_ROWS; ++k) {
                    const int r = x.i - 1 - k;
                    x.c[k] = r >= 0 ? lbits[r * WPR + wc] : 0u;
                }
            }
        }
#pragma unroll
        for (int lane = 0; lane < 2; ++lane) {             // one step of the walk (R6)
            Walk& x = w[lane];
            if (!x.live) continue;
            const int jj = x.j - (x.i - off - W);
            const int d = x.c_row - (x.i - 1);
            uint32_t word = x.c[0];
#pragma unroll
            for (int k = 1; k < WALK_ROWS; ++k) word = (d == k) ? x.c[k] : word;
            const uint32_t f = ((word >> (16u * (uint32_t)lane + 4u * (uint32_t)(3 - (jj & 3)))) & 15u) ^ 7u;
            if (x.st == 0) {
                if ((f & 3u) == 3u) {
                    emit(x, 0, 1u); ++x.n_cols;
                    --x.i; --x.j;
                } else if ((f & 3u) == 2u) x.st = 1;
                else x.st = 2;
            } else if (x.st == 1) {
                emit(x, 2, 1u); ++x.n_cols;
                if (f & 4u) x.st = 0;
                --x.i;
            } else {
                emit(x, 1, 1u); ++x.n_cols;
                if (f & 8u) x.st = 0;
                --x.j;
            }
            if (x.j == 0) x.live = false;
        }
    }
#pragma unroll
    for (int lane = 0; lane < 2; ++lane) {
        if (lane == 1 && !writeB) continue;
        const ThinPair& T = lane ? B : A;
        Walk& x = w[lane];
        const uint32_t p = T.p;
        const int ref_start = T.i_end - R + x.i;
        emit(x, -2, 0u);                           // flush the last run
        int n_match;
        {   // The path scores exactly S = match*n_match + mismatch*(M columns - n_match) - sum over gap runs of
            // (o + e*len), so n_match follows from the score without touching the sequences again
            // (N columns score mismatch and are not matches, consistently). A remainder means the walk is wrong.
            const int num = tp.score[p] + tp.sc.gap_open * x.gap_runs + tp.sc.gap_extend * x.gap_bases -
                            tp.sc.mismatch * (x.n_cols - x.gap_bases);
            const int den = tp.sc.match - tp.sc.mismatch;
            n_match = num / den;
            if (num < 0 || n_match * den != num || n_match > x.n_cols - x.gap_bases) x.bad = true;
        }
        if (x.bad) { atomicOr(tp.err_flag, SDP_ERRF_TRACE); x.nops = min(x.nops, cap); }
        tp.ref_start[p] = ref_start;
        tp.read_start[p] = 0;
        tp.read_end[p] = n - 1;
        tp.n_match[p] = n_match;
        tp.n_cols[p] = x.n_cols;
        tp.cigar_len[p] = x.nops;
        tp.pass[p] = ((long long)n_match * 1000000LL >= tp.sc.min_sim_q * (long long)x.n_cols) ? 1 : 0;
    }
}

// The band DP of two pairs with the SAME geometry (n, off) and the two walks. nB == 0 pairs: pass A twice, write once.
template <int W_, int MAXROWS>
__device__ __forceinline__ void thin_body2(const TraceParams& tp, const ThinConsts& tc, const ThinPair& A, const ThinPair& B,
                                           const bool writeB)
{
    constexpr int BW = 2 * W_ + 1;                 // band columns
    constexpr int WPR = (BW + 3) / 4;              // 32-bit words of direction nibbles per row (4 cells x 2 lanes)
    const sdp_batch& b = tp.b;
    const long long rwords = (long long)((b.reads_bases + 15) / 16), wwords = (long long)((b.wins_bases + 15) / 16);
    const long long rnwords = (long long)((b.reads_bases + 31) / 32), wnwords = (long long)((b.wins_bases + 31) / 32);
    const int n = A.n, off = A.off, R = A.R;
    const long long wposA = (long long)A.woff + (A.i_end - R), wposB = (long long)B.woff + (B.i_end - R);   // window base of row 1

    uint32_t lbits[MAXROWS * WPR];
    uint32_t wsel[8], rsel[8];                     // selectors of 16 rows: window base of the row, read base entering the band
    uint32_t Hc[BW + 1], Fc[BW + 1], rc[BW];
    {   // row i_lo of the restricted problem: M(i_lo, 0) = 0, M(i_lo, j) = -(o + e j) (drift form: beta - o)
        const int jb0 = -off - W_;
#pragma unroll
        for (int jj = 0; jj <= BW; ++jj) {
            const int j = jj + jb0;
            Hc[jj] = (jj == BW || j < 0 || j > n) ? 0x00070007u : (j == 0 ? tc.hb0 : tc.hrow0);
            Fc[jj] = 0x00020002u;
        }
    }
    {   // read codes of row 1's band slots 0 .. BW-2, held one slot to the right (every row shifts them left by one)
        constexpr int NSEG = (BW + 15) / 16;
        const long long q0 = (long long)(-off - W_);                   // read position (0-based) of slot 0 at row 1
#pragma unroll
        for (int sg = 0; sg < NSEG; ++sg) {
            const uint32_t a = bases16(b.reads_packed, (long long)A.roff + q0 + 16 * sg, rwords);
            const uint32_t bb = bases16(b.reads_packed, (long long)B.roff + q0 + 16 * sg, rwords);
            const uint32_t na = nbits16(b.read_nmask, (long long)A.roff + q0 + 16 * sg, rnwords);
            const uint32_t nb = nbits16(b.read_nmask, (long long)B.roff + q0 + 16 * sg, rnwords);
            uint32_t ex[8];
            expand16(a, bb, na, nb, SDP_CODE_READ_N, ex);
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const int slot = 16 * sg + k;
                if (slot < BW - 1) rc[slot + 1] = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, (ex[k >> 1] >> (16 * (k & 1))) & 0xFFFFu);
            }
        }
        rc[0] = 0u;
    }
    uint32_t hb = tc.hb0;                          // H7(ir, 0) = 8 (beta + e ir) + 7
    uint32_t finH = 0u;

    auto refill = [&](const int ir) {              // selectors of rows ir .. ir + 15
        {
            const uint32_t a = bases16(b.wins_packed, wposA + (ir - 1), wwords);
            const uint32_t bb = bases16(b.wins_packed, wposB + (ir - 1), wwords);
            const uint32_t na = nbits16(b.win_nmask, wposA + (ir - 1), wnwords);
            const uint32_t nb = nbits16(b.win_nmask, wposB + (ir - 1), wnwords);
            expand16(a, bb, na, nb, SDP_CODE_WIN_N, wsel);
        }
        {   // the read column that enters the band at row ir is j = ir - off + W_, 0-based position j - 1
            const long long q = (long long)(ir - off + W_ - 1);
            const uint32_t a = bases16(b.reads_packed, (long long)A.roff + q, rwords);
            const uint32_t bb = bases16(b.reads_packed, (long long)B.roff + q, rwords);
            const uint32_t na = nbits16(b.read_nmask, (long long)A.roff + q, rnwords);
            const uint32_t nb = nbits16(b.read_nmask, (long long)B.roff + q, rnwords);
            expand16(a, bb, na, nb, SDP_CODE_READ_N, rsel);
        }
    };

    auto row = [&](const int ir, auto check_tag) {
        constexpr bool CHECK = decltype(check_tag)::value;
        const int r16 = (ir - 1) & 15;
        if (r16 == 0) refill(ir);
        const uint32_t nt = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, reinterpret_cast<const uint16_t*>(wsel)[r16]);
#pragma unroll
        for (int k = 0; k < BW - 1; ++k) rc[k] = rc[k + 1];
        rc[BW - 1] = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, reinterpret_cast<const uint16_t*>(rsel)[r16]);
        hb = __vadd2(hb, tc.e8);
        const int jj0 = off + W_ - ir;             // band slot of read column 0 (CHECK rows only)

        uint32_t Hl = 0x00070007u, El = 0u;        // left of the band: -inf
        uint32_t b0 = 0u, b1 = 0u, t0 = 0u;
        constexpr uint32_t H2_8 = 0x48004800u, H2_16 = 0x4C004C00u;    // fp16 8.0 and 16.0, both lanes
#pragma unroll
        for (int jj = 0; jj < BW; ++jj) {
            const uint32_t q = hfma2_relu_negsq(hsub2_u(nt, rc[jj]), tc.Cd8);
            const uint32_t Ft = __viaddmax_s16x2(Hc[jj + 1], tc.negOf, Fc[jj + 1]);
            const uint32_t u = __viaddmax_s16x2(Hc[jj], q, Ft);
            uint32_t Et = __viaddmax_s16x2(Hl, tc.negOe, El);
            uint32_t Ht = __viaddmax_s16x2(u, tc.c8, Et);
            if (CHECK) { if (jj == jj0) { Ht = hb; Et = 0u; } }        // column 0: M(i,0) = 0, I(i,0) = -inf
            Fc[jj] = Ft & 0xFFFBFFFBu;
            El = Et & 0xFFFEFFFEu;
            Hl = Ht | 0x00070007u;
            Hc[jj] = Hl;
            const uint32_t v = t_select(Ht, Ft, 0x00040004u);
            const uint32_t x = t_imad(v, 0xFFFFFFFFu, Hl);             // 7 - (Ht&3 | Ft&4) per lane, no borrow
            const uint32_t eb = t_imad(El, 0xFFFFFFFFu, Et);           // Et & 1 per lane
            const uint32_t t = hfma2_u(eb, H2_8, x);                   // x + 8 eb as fp16 denormals: exact
            if ((jj & 1) == 0) t0 = t;
            if ((jj & 1) == 1 || jj == BW - 1) {
                const uint32_t byte = (jj & 1) ? hfma2_u(t0, H2_16, t) : hfma2_u(t0, H2_16, 0u);
                if ((jj & 3) < 2) b0 = byte; else b1 = byte;
            }
            if ((jj & 3) == 3 || jj == BW - 1) {
                if ((jj & 3) < 2) b1 = 0u;
                lbits[(ir - 1) * WPR + (jj >> 2)] = __byte_perm(b1, b0, 0x6240);
            }
        }
        if (ir == R) finH = Hc[W_];                // column n sits in the middle slot of the last row
    };

    // rows whose band holds read column 0 take the checked variant
    const int ir_a = min(R, max(0, off + W_));
    int ir = 1;
#pragma unroll 1
    for (; ir <= ir_a; ++ir) row(ir, std::true_type{});
#pragma unroll 1
    for (; ir <= R; ++ir) row(ir, std::false_type{});

    thin_walks(tp, tc, A, B, writeB, lbits, W_, finH);
}

// thread k of class W_ takes pairs 2k and 2k+1 of the class's range of tp.order (sorted by rows, so neighbours nearly
// always share their geometry); a pair of pairs whose geometries differ runs the body once per pair
template <int W_, int MAXROWS>
__device__ __forceinline__ void thin_two(const TraceParams& tp, const ThinConsts& tc, const uint32_t first,
                                         const uint32_t count, const uint32_t k)
{
    if (2 * k >= count) return;
    const ThinPair A = thin_pair<W_>(tp, tp.order[first + 2 * k]);
    const bool hasB = 2 * k + 1 < count;
    const ThinPair B = hasB ? thin_pair<W_>(tp, tp.order[first + 2 * k + 1]) : A;
    const bool same = hasB && A.n == B.n && A.off == B.off;
    const int passes = (hasB && !same) ? 2 : 1;
#pragma unroll 1
    for (int h = 0; h < passes; ++h) {             // (A, B) together, or A alone and then B alone
        const ThinPair X = h ? B : A;
        const ThinPair Y = same ? B : X;
        thin_body2<W_, MAXROWS>(tp, tc, X, Y, same);
    }
}

// Gap bounds LO..HI-1 in ONE launch: block b serves class w with
// r.block_start[w] <= b < r.block_start[w+1] (one small launch per class left the GPU mostly idle).
struct ThinRanges { uint32_t first[THIN_NW], count[THIN_NW], block_start[THIN_NW + 1]; };

template <int W_, int HI>
__device__ __forceinline__ void thin_dispatch(const int w, const TraceParams& tp, const ThinConsts& tc,
                                              const ThinRanges& r, const uint32_t k)
{
    if (w == W_) {
        if constexpr (W_ == 0) { if (k < r.count[0]) thin_gapless(tp, tp.order[r.first[0] + k]); }
        else thin_two<W_, THIN_MAXROWS>(tp, tc, r.first[W_], r.count[W_], k);
    } else if constexpr (W_ + 1 < HI) thin_dispatch<W_ + 1, HI>(w, tp, tc, r, k);
}

template <int LO, int HI>
__global__ void __launch_bounds__(128) k_thin_range(const TraceParams tp, const ThinConsts tc, const ThinRanges r)
{
    // widest bands and longest rows first (blocks are dispatched in index order): the cheap classes fill the tail
    const uint32_t b = (gridDim.x - 1u - blockIdx.x) + r.block_start[LO];
    int w = LO;
#pragma unroll
    for (int c = LO + 1; c < HI; ++c) w += (b >= r.block_start[c]) ? 1 : 0;
    const uint32_t k = (b - r.block_start[w]) * blockDim.x + threadIdx.x;
    thin_dispatch<LO, HI>(w, tp, tc, r, k);                // w is block-uniform
}

// bounds[w] .. bounds[w+1]: range of tp.order that holds the pairs with gap bound w
int launch_thin_all(const uint32_t* bounds, const TraceParams& tp, cudaStream_t st, cudaStream_t st_mid, cudaStream_t st_hi)
{
    ThinConsts tc;
    const int o = tp.sc.gap_open, e = tp.sc.gap_extend, c = 2 * e + tp.sc.mismatch;
    const int beta = 3 * o + 8 + (c > 0 ? c : 0);
    tc.negOf = sdp_pack2(8 * (-o - c) - 1); tc.negOe = sdp_pack2(-8 * o - 6);
    tc.c8 = sdp_pack2(8 * c); tc.Cd8 = sdp_pack2(8 * (tp.sc.match - tp.sc.mismatch)); tc.e8 = sdp_pack2(8 * e);
    tc.hb0 = sdp_pack2(8 * beta + 7); tc.hrow0 = sdp_pack2(8 * (beta - o) + 7);
    tc.beta = beta; tc.e = e;
    ThinRanges r;
    uint32_t blocks = 0;
    for (int w = 0; w < THIN_NW; ++w) {
        r.first[w] = bounds[w]; r.count[w] = bounds[w + 1] - bounds[w];
        r.block_start[w] = blocks;
        blocks += (r.count[w] + (w ? 255 : 127)) / (w ? 256 : 128);     // two pairs per thread from W = 1 on
    }
    r.block_start[THIN_NW] = blocks;
    int launched = 0;
    const uint32_t lo_blocks = r.block_start[THIN_SPLIT];
    const uint32_t mid_blocks = r.block_start[THIN_SPLIT2] - lo_blocks, hi_blocks = blocks - r.block_start[THIN_SPLIT2];
    // the wider bands on their own stream: few blocks that run long (and three register budgets)
    if (hi_blocks) { k_thin_range<THIN_SPLIT2, THIN_NW><<<hi_blocks, 128, 0, st_hi>>>(tp, tc, r); ++launched; }
    if (mid_blocks) { k_thin_range<THIN_SPLIT, THIN_SPLIT2><<<mid_blocks, 128, 0, st_mid>>>(tp, tc, r); ++launched; }
    if (lo_blocks) { k_thin_range<0, THIN_SPLIT><<<lo_blocks, 128, 0, st>>>(tp, tc, r); ++launched; }
    return launched;
}

}  // namespace sdp
