// traceback.cu -- a5 (banded traceback + CIGAR), a6 (similarity filter), a7 (CIGAR compaction).
//
// The paper backtracks through full tables D and M kept in global memory. Here
// the forward pass keeps no table; instead the score S bounds the gap content of every
// co-optimal alignment, W = floor((n*match - S - o) / e) (0 when negative), so all co-optimal
// paths lie in the band |i - j - (i_end - n)| <= W and in rows >= i_lo = max(s_lo, i_end-n-W).
// The DP restricted to that band equals the full DP on every co-optimal cell, so the equality
// tests of the walk (diagonal first, then deletion, then insertion; "opened here" before
// "extended") resolve exactly as in the full-table oracle.
// W == 0 means the alignment is gapless: CIGAR nM, no DP at all.
#include "sdp_host.cuh"
#include "seq_bits.cuh"

namespace sdp {

constexpr int NEG = -(1 << 28);

// sequential reader of a 2-bit packed sequence with optional N bitmap
struct SeqReader {
    const uint32_t* packed; const uint32_t* nmask; uint32_t ncode;
    __device__ __forceinline__ uint32_t at(uint64_t pos) const {
        uint32_t c = (__ldg(packed + (pos >> 4)) >> (2u * ((uint32_t)pos & 15u))) & 3u;
        if (nmask != nullptr && ((__ldg(nmask + (pos >> 5)) >> ((uint32_t)pos & 31u)) & 1u)) c = ncode;
        return c;
    }
};

// ---------------------------------------------------------------------------------------------
// after the forward pass: gap-content bound, bucket keys of the reverse and traceback passes,
// scratch sizes. One thread per pair.
__device__ __forceinline__ int tb_class_of(int bw) {
    static_assert(TB_NCLASS == 5, "update tb_class_of");
    return bw > 1032 ? 4 : (bw > 256 ? 3 : (bw > 64 ? 2 : (bw > 16 ? 1 : 0)));
}
static_assert((THIN_NW + TB_NCLASS) * TB_KEY_STRIDE <= SDP_NBINS && SDP_MAX_READ_LEN < TB_KEY_STRIDE, "thin keys must fit the bucket-sort key space");

// Histogram add for every thread of the block (call from uniform control flow). The key of the block's first thread
// is counted once per block -- half of a typical batch shares one key (the gapless class), and one atomic per warp
// would serialise on that bin -- every other key once per warp.
__device__ __forceinline__ void hist_add(uint32_t* hist, uint32_t key, bool valid) {
    __shared__ uint32_t s_key;
    __syncthreads();
    if (threadIdx.x == 0) s_key = valid ? key : SDP_KEY_SKIP;
    __syncthreads();
    const uint32_t bkey = s_key;
    const bool same = valid && key == bkey;
    const int n_same = __syncthreads_count(same ? 1 : 0);
    if (threadIdx.x == 0 && n_same) atomicAdd(hist + bkey, (uint32_t)n_same);
    const bool other = valid && !same;
    const uint32_t active = __ballot_sync(0xffffffffu, other);
    if (other) {
        const uint32_t peers = __match_any_sync(active, key);
        if ((threadIdx.x & 31) == (uint32_t)(__ffs(peers) - 1)) atomicAdd(hist + key, (uint32_t)__popc(peers));
    }
}

__global__ void k_post_forward(const PostParams pp)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = p < pp.n_pairs;
    uint32_t ktb = SDP_KEY_SKIP, kwide = SDP_KEY_SKIP;
    unsigned long long c_tb = 0;
    bool too_big = false;
    if (valid) {
        // slow = the int32 lane (slow_lane.cu): pairs outside the int16 kernels' domain, and every pair in local mode,
        // where only the first end_col read columns matter (the alignment ends in column end_col)
        const bool slow = pp.slow_words[p] != 0;
        const int n = pp.local ? pp.end_col[p] : (int)pp.pn[p];
        const int S = pp.score[p], i_end = pp.ref_end[p] + 1;
        const long long slack = (long long)n * pp.sc.match - S - pp.sc.gap_open;
        int W = slack >= pp.sc.gap_extend ? (int)min(slack / pp.sc.gap_extend, (long long)(1 << 29)) : 0;
        W = min(W, n + i_end);
        if (W > 0 && i_end >= n && !slow) {
            // Ungapped shortcut. If the gap-free alignment on the end cell's diagonal already scores S, it is the
            // alignment the traceback reports: every prefix of an optimal path is optimal for its end cell, so
            // the walk's first test (diagonal) succeeds at every step of it. Such a pair is gapless (W = 0):
            // CIGAR nM, no band to recompute. Costs one XOR + popcount pass over ~n/16 words.
            const sdp_batch& b = pp.b;
            const uint32_t ri = b.pairs[2 * p], wi = b.pairs[2 * p + 1];
            const long long rpos = (long long)b.read_off[ri], wpos = (long long)b.win_off[wi] + (i_end - n);
            const int eq = count_equal_bases(b.reads_packed, b.read_nmask, rpos, (long long)((b.reads_bases + 15) / 16),
                                             (long long)((b.reads_bases + 31) / 32), b.wins_packed, b.win_nmask, wpos,
                                             (long long)((b.wins_bases + 15) / 16), (long long)((b.wins_bases + 31) / 32), n);
            if (pp.sc.match * eq + pp.sc.mismatch * (n - eq) == S) W = 0;
        }
        pp.tbW[p] = W;
        uint32_t words = 0;
        int bw = 1, rows = 0;
        if (W > 0) {
            rows = min(i_end, n + W);
            bw = min(2 * W + 1, n + 1);
        }
        pp.tb_rows[p] = rows;
        // Three paths. Narrow: W < THIN_NW and a real band -> one thread per pair,
        // band in registers (thin_kernel.cu). Wide: the register-resident wavefront recomputes the
        // whole rectangle rows x n (trace_kernel.cuh) when its x8 scaled values fit 16 bits; the
        // reverse pass first trims the rectangle's rows. Anything else: the generic band kernel.
        const long long vmax = (long long)pp.sc.match * n + (long long)pp.sc.gap_extend * (n + rows) +
                               3LL * pp.sc.gap_open + 8;
        if (slow && W == 0) { rows = min(i_end, n); bw = 1; }      // (the dynamic kernel walks a gapless pair through its band too)
        const int c_shift = 2 * pp.sc.gap_extend + pp.sc.mismatch;
        const bool thin_fits = pp.thin_ok && vmax + (c_shift > 0 ? c_shift : 0) <= SDP_TB_MAX_VALUE;      // x8 tagged int16 lanes
        const bool narrow = !slow && (W == 0 || (W < THIN_NW && 2 * W + 1 < n + 1 && rows <= THIN_MAXROWS && thin_fits && !pp.no_thin));
        const bool wide = !slow && !narrow && pp.wide_ok && vmax + (c_shift > 0 ? c_shift : 0) <= SDP_TB_MAX_VALUE;
        if (narrow) {
            ktb = (uint32_t)W * TB_KEY_STRIDE + (uint32_t)min((int)TB_KEY_STRIDE - 1, W ? rows : n);
            c_tb = (unsigned long long)bw * rows;
        } else if (wide) {
            // 64 row classes per read length, scaled to the rows a read of this length can need (rows <= 2.5 n),
            // so that the pairs of one warp walk nearly the same number of rows
            const uint32_t rbin = (uint32_t)min(63, (rows * 64) / (5 * n / 2 + 1));
            kwide = (uint32_t)(n - 1) * 64u + rbin;         // the reverse pass and the traceback DP share this order
            c_tb = (unsigned long long)n * rows;            // (whether the pair takes the reverse pass: k_fill_desc_rev)
        } else {
            // int32-lane pairs keep their row arrays in global scratch (any width); in local mode a read of up to 1,024
            // bases has a band of at most 1,025 cells, which fits the local-memory classes
            const bool any_width = slow && !(pp.local && pp.pn[p] <= 1024u);
            const int cls = any_width ? TB_NCLASS - 1 : tb_class_of(bw);
            const unsigned long long w64 = (unsigned long long)rows * (unsigned long long)((bw + 7) / 8) +
                                           (cls == TB_NCLASS - 1 ? 2ull * (unsigned long long)(bw + 2) : 0ull);   // + the two row arrays
            if (w64 > 0xFFFFFFFFull) { words = 0; too_big = true; } else words = (uint32_t)w64;
            c_tb = (unsigned long long)bw * rows;
            ktb = (uint32_t)(THIN_NW + cls) * TB_KEY_STRIDE + (uint32_t)min(bw, (int)TB_KEY_STRIDE - 1);
        }
        pp.keys_wide[p] = kwide;
        pp.keys_tb[p] = ktb;
        pp.bits_words[p] = words;
        pp.ops_cap[p] = 2u * (uint32_t)W + 5u;            // runs of a path with <= W gap bases, + flush slot + two soft clips
        if (too_big) atomicOr(pp.err_flag, SDP_ERRF_RANGE);
    }
    hist_add(pp.hist_tb, ktb, ktb != SDP_KEY_SKIP);
    hist_add(pp.hist_wide, kwide, kwide != SDP_KEY_SKIP);
    for (int o = 16; o > 0; o >>= 1) c_tb += __shfl_down_sync(0xffffffffu, c_tb, o);
    if ((threadIdx.x & 31) == 0 && c_tb) atomicAdd(pp.counters + 1, c_tb);
}

void launch_post_forward(const PostParams& pp, cudaStream_t st)
{
    if (pp.n_pairs) k_post_forward<<<(uint32_t)((pp.n_pairs + 255) / 256), 256, 0, st>>>(pp);
}

// descriptors of the reverse pass, in its bucket order: DP row 1 is window base ref_end, the
// read is walked from its last base, rows = min(ref_end + 1, n + W).
// a4 WHERE IT PAYS. The pass costs `rows` score-kernel rows and trims the traceback rectangle from `rows` to the
// alignment's span (about n) rows, each worth ~2.2 score-kernel rows (measured on config 4: DESIGN.md "Traceback").
// With enough wide pairs to fill the GPU many times over, that is worth it only when the bound exceeds ratio10/10
// read lengths (2.4 by measurement); such a pair gets m = 0 here (the kernel skips it) and rev_rows = rows, i.e. its
// rectangle is the whole bound. With few wide pairs the kernels' time is set by the longest task, not by the total
// work, and the host passes ratio10 = 0: every wide pair takes the pass.
__global__ void k_fill_desc_rev(const sdp_batch b, const uint32_t* __restrict__ order, uint32_t count,
                                const int32_t* __restrict__ score, const int32_t* __restrict__ ref_end,
                                const int32_t* __restrict__ tbW, int ratio10, int32_t* __restrict__ rev_rows,
                                unsigned long long* __restrict__ counters, PairDesc* __restrict__ desc)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    unsigned long long c_rev = 0, n_rev = 0;
    if (k < count) {
        const uint32_t p = order[k];
        const uint32_t ri = b.pairs[2 * (uint64_t)p], wi = b.pairs[2 * (uint64_t)p + 1];
        PairDesc d;
        d.n = b.read_len[ri];
        d.roff = b.read_off[ri];
        d.woff = b.win_off[wi] + (uint64_t)ref_end[p];
        const int rows = min(ref_end[p] + 1, (int)d.n + tbW[p]);
        const bool use_rev = 10 * rows > ratio10 * (int)d.n + 80 || ratio10 == 0;
        d.m = use_rev ? (uint32_t)rows : 0u;
        rev_rows[p] = use_rev ? 0 : rows;                   // (the kernel overwrites the 0)
        d.pid = p; d.aux = score[p];
        desc[k] = d;
        if (use_rev) { c_rev = (unsigned long long)d.n * rows; n_rev = 1; }
    }
    for (int o = 16; o > 0; o >>= 1) {
        c_rev += __shfl_down_sync(0xffffffffu, c_rev, o);
        n_rev += __shfl_down_sync(0xffffffffu, n_rev, o);
    }
    if ((threadIdx.x & 31) == 0 && n_rev) { atomicAdd(counters + 0, c_rev); atomicAdd(counters + 2, n_rev); }
}

void launch_fill_desc_rev(const sdp_batch& b, const uint32_t* order, uint32_t count, const int32_t* score,
                          const int32_t* ref_end, const int32_t* tbW, int ratio10, int32_t* rev_rows,
                          unsigned long long* counters, PairDesc* desc, cudaStream_t st)
{
    if (count) k_fill_desc_rev<<<(count + 255) / 256, 256, 0, st>>>(b, order, count, score, ref_end, tbW, ratio10, rev_rows,
                                                                    counters, desc);
}

// ---------------------------------------------------------------------------------------------
// traceback: one thread per pair, row arrays of the band in local memory (MAXBW + 2 entries).
// Direction bits per cell: 1 = H came from the diagonal, 2 = H equals D, 4 = D was opened here,
// 8 = I was opened here. Rows i_lo+1 .. i_end each take wpr = ceil(bw / 8) words.
// MAXBW == 0: any band width, the two row arrays sit in global scratch behind the pair's direction bits (the int32 lane:
// reads beyond SDP_MAX_READ_LEN, windows beyond the int16 range rule). LOCAL: the soft-clipping variant (R18):
// zero floor, walk from (i_end, end_col), stops where the remaining score is 0, clips as CIGAR op 4.
template <int MAXBW, bool LOCAL>
__global__ void __launch_bounds__(128) k_traceback(const TraceParams tp)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= tp.count) return;
    const uint32_t p = tp.order[tp.first + k];
    const sdp_batch& b = tp.b;
    const uint32_t ri = b.pairs[2 * (uint64_t)p], wi = b.pairs[2 * (uint64_t)p + 1];
    const int n_full = (int)b.read_len[ri];
    const int n = LOCAL ? tp.end_col[p] : n_full;          // local: the alignment ends in read column end_col
    const uint64_t roff = b.read_off[ri], woff = b.win_off[wi];
    const SeqReader RD{b.reads_packed, b.read_nmask, SDP_CODE_READ_N};
    const SeqReader WN{b.wins_packed, b.win_nmask, SDP_CODE_WIN_N};
    const int i_end = tp.ref_end[p] + 1;
    const int W = tp.tbW[p];
    const int o = tp.sc.gap_open, e = tp.sc.gap_extend, oe = o + e;
    uint32_t* ops = tp.ops_rev + tp.ops_off[p];
    const uint32_t cap = 2u * (uint32_t)W + 5u;

    int n_match = 0, n_cols = 0, ref_start = 0, read_start = 0;
    uint32_t nops = 0;
    int cur_op = -1; uint32_t cur_len = 0;
    bool bad = false;
    auto emit = [&](int op, uint32_t len) {
        if (op == cur_op) { cur_len += len; return; }
        if (cur_op >= 0) { if (nops < cap) ops[nops] = (cur_len << 4) | (uint32_t)cur_op; else bad = true; ++nops; }
        cur_op = op; cur_len = len;
    };
    if (LOCAL && n_full > n && tp.score[p] > 0) emit(4, (uint32_t)(n_full - n));   // trailing soft clip (runs are stored end -> start)

    if (LOCAL && tp.score[p] == 0) {
        emit(4, (uint32_t)n_full);                        // no alignment: everything is clipped
    } else if (W == 0 && MAXBW != 0 && !LOCAL) {
        // gapless: the only co-optimal alignments are ungapped, so the CIGAR is nM
        ref_start = i_end - n;
        if (ref_start < 0) { bad = true; ref_start = 0; }
        for (int j = 0; j < n; ++j) {
            const uint32_t r = RD.at(roff + (uint64_t)j), t = WN.at(woff + (uint64_t)(ref_start + j));
            n_match += (r == t);
        }
        n_cols = n;
        emit(0, (uint32_t)n);
    } else {
        const int c = i_end - n;
        const int s_lo = 0;                               // thin pairs skip the reverse pass
        const int i_lo = max(0, max(s_lo, i_end - n - W));
        const bool banded = (2 * W + 1 < n + 1);
        const int bw = banded ? 2 * W + 1 : n + 1;
        const int shift = banded ? 1 : 0;
        const int wpr = (bw + 7) / 8;
        uint32_t* bits = tp.bits + tp.bits_off[p];
        if (MAXBW != 0 && bw > MAXBW) { bad = true; }
        else {
            int Hloc[MAXBW + 2], Dloc[MAXBW + 2];
            int* const Hr = MAXBW != 0 ? Hloc : reinterpret_cast<int*>(bits + (size_t)(i_end - i_lo) * wpr);
            int* const Dr = MAXBW != 0 ? Dloc : Hr + (bw + 2);
            // row i_lo is the restricted problem's row 0: H = -(o + e j) via insertions, H(.,0) = 0 (local: all zero)
            {
                const int jb = banded ? (i_lo - c - W) : 0;
                for (int jj = 0; jj <= bw; ++jj) {
                    const int j = jj + jb;
                    Hr[jj] = (jj == bw || j < 0 || j > n) ? NEG : ((j == 0 || LOCAL) ? 0 : -(o + e * j));
                    Dr[jj] = NEG;
                }
            }
            for (int i = i_lo + 1; i <= i_end; ++i) {
                const uint32_t t = WN.at(woff + (uint64_t)(i - 1));
                const int jb = banded ? (i - c - W) : 0;
                int Hleft = NEG, Ileft = NEG, saved_old = NEG;
                uint32_t word = 0;
                uint32_t* brow = bits + (size_t)(i - i_lo - 1) * wpr;
                for (int jj = 0; jj < bw; ++jj) {
                    const int j = jj + jb;
                    const int oldH = Hr[jj];
                    const int upH = shift ? Hr[jj + 1] : oldH;
                    const int upD = shift ? Dr[jj + 1] : Dr[jj];
                    const int dgH = shift ? oldH : saved_old;
                    saved_old = oldH;
                    int Hn, Dn, In;
                    uint32_t f = 0;
                    if (j < 0 || j > n) { Hn = NEG; Dn = NEG; In = NEG; }
                    else if (j == 0) { Hn = 0; Dn = NEG; In = NEG; }
                    else {
                        const uint32_t r = RD.at(roff + (uint64_t)(j - 1));
                        In = max(Hleft - oe, Ileft - e);
                        Dn = max(upH - oe, upD - e);
                        const int dg = dgH + ((r == t) ? tp.sc.match : tp.sc.mismatch);
                        Hn = max(dg, max(Dn, In));
                        if (LOCAL) Hn = max(Hn, 0);
                        f = (Hn == dg ? 1u : 0u) | (Hn == Dn ? 2u : 0u) | (Dn == upH - oe ? 4u : 0u) |
                            (In == Hleft - oe ? 8u : 0u);
                    }
                    Hr[jj] = Hn; Dr[jj] = Dn; Hleft = Hn; Ileft = In;
                    word |= f << (4 * (jj & 7));
                    if ((jj & 7) == 7 || jj == bw - 1) { brow[jj >> 3] = word; word = 0; }
                }
            }
            if (Hr[n - (banded ? (i_end - c - W) : 0)] != tp.score[p]) bad = true;   // band DP must end on S
            // walk back from (i_end, n). Local: `rem` is the score still to be explained, i.e. M(i,j) while in state H;
            // the walk stops where it reaches 0 (R18), and what is left of the read is a soft clip.
            int i = i_end, j = n, st = 0;                  // 0 = H, 1 = D, 2 = I
            int rem = tp.score[p], run = 0;
            while (j > 0) {
                if (LOCAL && st == 0 && rem == 0) break;
                if (i == i_lo) {
                    if (LOCAL) { bad = true; break; }      // a local alignment never starts with a gap
                    emit(1, (uint32_t)j); n_cols += j; j = 0; break;
                }
                const int jj = j - (banded ? (i - c - W) : 0);
                if (jj < 0 || jj >= bw) { bad = true; break; }
                const uint32_t f = (bits[(size_t)(i - i_lo - 1) * wpr + (jj >> 3)] >> (4 * (jj & 7))) & 15u;
                if (st == 0) {
                    if (f & 1u) {
                        emit(0, 1u); ++n_cols;
                        const bool eq = RD.at(roff + (uint64_t)(j - 1)) == WN.at(woff + (uint64_t)(i - 1));
                        n_match += eq;
                        rem -= eq ? tp.sc.match : tp.sc.mismatch;
                        --i; --j;
                    } else if (f & 2u) { st = 1; run = 0; }
                    else { st = 2; run = 0; }
                } else if (st == 1) {
                    emit(2, 1u); ++n_cols; ++run;
                    if (f & 4u) { st = 0; rem += o + e * run; }
                    --i;
                } else {
                    emit(1, 1u); ++n_cols; ++run;
                    if (f & 8u) { st = 0; rem += o + e * run; }
                    --j;
                }
            }
            if (LOCAL && (rem != 0 || st != 0)) bad = true;
            ref_start = i;
            read_start = j;
            if (LOCAL && j > 0) emit(4, (uint32_t)j);       // leading soft clip
        }
    }
    emit(-2, 0u);                                          // flush the last run
    if (bad) { atomicOr(tp.err_flag, SDP_ERRF_TRACE); nops = min(nops, cap); }
    const bool none = LOCAL && tp.score[p] == 0;
    tp.ref_start[p] = none ? 0 : ref_start;
    tp.read_start[p] = none ? 0 : read_start;
    tp.read_end[p] = none ? -1 : n - 1;
    tp.n_match[p] = n_match;
    tp.n_cols[p] = n_cols;
    tp.cigar_len[p] = nops;
    // local: soft-clipped read bases count as columns that do not match, and an empty alignment never passes (R18)
    const long long cols = LOCAL ? (long long)n_cols + (none ? n_full : read_start + (n_full - n)) : (long long)n_cols;
    tp.pass[p] = ((!LOCAL || n_cols > 0) && (long long)n_match * 1000000LL >= tp.sc.min_sim_q * cols) ? 1 : 0;
}

void launch_traceback(int cls, bool local, const TraceParams& tp, cudaStream_t st)
{
    if (tp.count == 0) return;
    const uint32_t grid = (tp.count + 127) / 128;
    if (local) {
        switch (cls) {
            case 0: k_traceback<16, true><<<grid, 128, 0, st>>>(tp); break;
            case 1: k_traceback<64, true><<<grid, 128, 0, st>>>(tp); break;
            case 2: k_traceback<256, true><<<grid, 128, 0, st>>>(tp); break;
            case 3: k_traceback<1032, true><<<grid, 128, 0, st>>>(tp); break;
            default: k_traceback<0, true><<<grid, 128, 0, st>>>(tp); break;
        }
        return;
    }
    switch (cls) {
        case 0: k_traceback<16, false><<<grid, 128, 0, st>>>(tp); break;
        case 1: k_traceback<64, false><<<grid, 128, 0, st>>>(tp); break;
        case 2: k_traceback<256, false><<<grid, 128, 0, st>>>(tp); break;
        case 3: k_traceback<1032, false><<<grid, 128, 0, st>>>(tp); break;
        default: k_traceback<0, false><<<grid, 128, 0, st>>>(tp); break;
    }
}

// ---------------------------------------------------------------------------------------------
// wide pairs (trace_kernel.cuh). Sorted by (n, rows) into `order`; the pairs of one warp task share
// one region of direction nibbles, laid out so that a warp's store of one word per lane is contiguous.
__global__ void k_wide_regions(const uint32_t* __restrict__ order, uint32_t max_count,
                               const uint32_t* __restrict__ count_dev, const uint32_t* __restrict__ pn,
                               const int32_t* __restrict__ tb_rows, const uint16_t* __restrict__ slot_of_n,
                               const SlotInfo* __restrict__ slots, uint32_t* __restrict__ words)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= max_count || k >= *count_dev) return;       // the number of wide pairs is only known on the device
    const uint32_t p = order[k];
    const SlotInfo si = slots[slot_of_n[pn[p] - 1]];
    const uint32_t local = k - si.first;
    const uint32_t ppw = 2u * (32u / si.G);               // pairs per warp task
    uint32_t w = 0;
    if (local % ppw == 0) {                               // first pair of a task owns the task's region
        int rows = 0;
        for (uint32_t t = 0; t < ppw && local + t < si.count; ++t) rows = max(rows, tb_rows[order[k + t]]);
        // one line set per wavefront step, steps in pairs (+ one pair: a pass may store its second row past the last)
        w = (uint32_t)((rows + SDP_SCORE_SKEW * (si.G - 1) + 3) / 2) * 64u * (uint32_t)((si.K + 3) / 4);
    }
    words[k] = w;
}

void launch_wide_regions(const uint32_t* order, uint32_t max_count, const uint32_t* count_dev, const uint32_t* pn,
                         const int32_t* tb_rows, const uint16_t* slot_of_n, const SlotInfo* slots, uint32_t* words,
                         cudaStream_t st)
{
    if (max_count)
        k_wide_regions<<<(max_count + 255) / 256, 256, 0, st>>>(order, max_count, count_dev, pn, tb_rows, slot_of_n,
                                                                 slots, words);
}

// descriptors of the traceback DP: rows (i_lo, i_end] with i_lo = i_end - R, R = rows the reverse
// pass found the longest co-optimal alignment to span (at least 1, so that the DP has a row)
__global__ void k_fill_desc_tb(const sdp_batch b, const uint32_t* __restrict__ order, uint32_t count,
                               const int32_t* __restrict__ score, const int32_t* __restrict__ ref_end,
                               const int32_t* __restrict__ rev_rows, PairDesc* __restrict__ desc)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= count) return;
    const uint32_t p = order[k];
    const uint32_t ri = b.pairs[2 * (uint64_t)p], wi = b.pairs[2 * (uint64_t)p + 1];
    const int i_end = ref_end[p] + 1;
    const int R = min(i_end, max(1, rev_rows[p]));
    PairDesc d;
    d.n = b.read_len[ri];
    d.roff = b.read_off[ri];
    d.woff = b.win_off[wi] + (uint64_t)(i_end - R);
    d.m = (uint32_t)R;
    d.pid = p; d.aux = score[p];
    desc[k] = d;
}

void launch_fill_desc_tb(const sdp_batch& b, const uint32_t* order, uint32_t count, const int32_t* score,
                         const int32_t* ref_end, const int32_t* rev_rows, PairDesc* desc, cudaStream_t st)
{
    if (count) k_fill_desc_tb<<<(count + 255) / 256, 256, 0, st>>>(b, order, count, score, ref_end, rev_rows, desc);
}

// the walk (R6) over the nibbles trace_kernel left: one thread per pair
__global__ void __launch_bounds__(128) k_walk(const WalkParams wp)
{
    const uint32_t k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= wp.count) return;
    const PairDesc d = wp.desc[k];
    const uint32_t p = d.pid;
    const int n = (int)d.n, R = (int)d.m;
    const SlotInfo si = wp.slots[wp.slot_of_n[n - 1]];
    const uint32_t local = k - si.first;
    const int G = si.G, K = si.K, NW = (K + 3) / 4;
    const int pad = G * K - n;
    const uint32_t ppw = 2u * (32u / (uint32_t)G);
    const uint32_t in_task = local % ppw;
    const uint32_t* region = wp.bits + wp.bits_off[k - in_task];
    const uint32_t lane0 = (in_task >> 1) * (uint32_t)G;  // lane of the group's first thread
    const uint32_t lane_shift = (local & 1u) * 16u;
    const uint32_t cap = 2u * (uint32_t)wp.tbW[p] + 3u;
    uint32_t* ops = wp.ops_rev + wp.ops_off[p];

    int n_match = 0, n_cols = 0;
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
    int i = R, j = n, st = 0;                              // 0 = H, 1 = D, 2 = I
    const int split = pad * (K - 1);                       // columns owned by the threads that skip one
    while (j > 0) {
        if (i == 0) { emit(1, (uint32_t)j); n_cols += j; j = 0; break; }   // row i_lo: all insertions
        const int j0 = j - 1;
        int g, kk;
        if (j0 < split) { g = j0 / (K - 1); kk = j0 - g * (K - 1); }
        else { const int j1 = j0 - split; const int t = j1 / K; g = pad + t; kk = j1 - t * K; }
        const int w = kk >> 2;
        const int t = i - 1 + SDP_SCORE_SKEW * g;          // 0-based step of row i in thread g (trace_kernel.cuh layout)
        const uint32_t word = __ldg(region + (((size_t)(t >> 1) * NW + w) * 32u + lane0 + (uint32_t)g) * 2u + (uint32_t)(t & 1));
        const uint32_t f = ((word >> (lane_shift + 4u * (uint32_t)(3 - (kk & 3)))) & 15u) ^ 7u;   // low three bits are stored complemented
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
    emit(-2, 0u);
    {   // n_match from the score (see thin_kernel.cu): S = match*n_match + mismatch*(M columns - n_match) - gap costs
        const int num = d.aux + wp.sc.gap_open * gap_runs + wp.sc.gap_extend * gap_bases -
                        wp.sc.mismatch * (n_cols - gap_bases);
        const int den = wp.sc.match - wp.sc.mismatch;
        n_match = num / den;
        if (num < 0 || n_match * den != num || n_match > n_cols - gap_bases) bad = true;
    }
    if (bad) { atomicOr(wp.err_flag, SDP_ERRF_TRACE); nops = min(nops, cap); }
    wp.ref_start[p] = wp.ref_end[p] + 1 - R + i;
    wp.read_start[p] = 0;
    wp.read_end[p] = n - 1;
    wp.n_match[p] = n_match;
    wp.n_cols[p] = n_cols;
    wp.cigar_len[p] = nops;
    wp.pass[p] = ((long long)n_match * 1000000LL >= wp.sc.min_sim_q * (long long)n_cols) ? 1 : 0;
}

void launch_walk(const WalkParams& wp, cudaStream_t st)
{
    if (wp.count) k_walk<<<(wp.count + 127) / 128, 128, 0, st>>>(wp);
}

// a7: copy each pair's runs (stored end -> start) into the dense buffer in alignment order
__global__ void k_compact(uint64_t n_pairs, const uint64_t* __restrict__ ops_off, const uint32_t* __restrict__ ops_rev,
                          const uint32_t* __restrict__ cigar_len, const uint64_t* __restrict__ cigar_off,
                          uint32_t* __restrict__ cigar_ops)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n_pairs) return;
    const uint32_t len = cigar_len[p];
    const uint32_t* src = ops_rev + ops_off[p];
    uint32_t* dst = cigar_ops + cigar_off[p];
    for (uint32_t k = 0; k < len; ++k) dst[k] = src[len - 1 - k];
}

void launch_compact(uint64_t n_pairs, const uint64_t* ops_off, const uint32_t* ops_rev, const uint32_t* cigar_len,
                    const uint64_t* cigar_off, uint32_t* cigar_ops, cudaStream_t st)
{
    if (n_pairs) k_compact<<<(uint32_t)((n_pairs + 255) / 256), 256, 0, st>>>(n_pairs, ops_off, ops_rev, cigar_len,
                                                                             cigar_off, cigar_ops);
}

}  // namespace sdp
