// score_kernel.cuh -- forward score pass (a3) and reverse pass (a4) of the hot path.
//
// What it computes: for each pair, over window rows i = 1..m and
// read columns j = 1..n,
//     I(i,j) = max(M(i,j-1) + S_GO, I(i,j-1) + S_GE)
//     D(i,j) = max(M(i-1,j) + S_GO, D(i-1,j) + S_GE)
//     M(i,j) = max(M(i-1,j-1) + delta(T[i], R[j]), I(i,j), D(i,j))
// and S = max_{1<=i<=m} M(i,n) with the lowest maximising row (forward), or the highest row of
// the reversed, start-anchored problem whose M(i,n) equals S (reverse).
//
// How: nothing like the paper's global-memory tables survives.
//  * int16x2 lanes hold TWO pairs; a group of G threads owns the read's n columns, K per thread,
//    H/F columns live in registers, the window streams by as rows, and thread g works on row
//    s - g at step s (anti-diagonal wavefront); H and E of the chunk's last column cross to the
//    right neighbour with one warp shuffle each per row.
//  * drift form: stored values are H + e*(i+j) + beta, so gap extension needs no add:
//        E' = max(H'(i,j-1) - o, E'(i,j-1))          1 VIADDMNMX.S16x2
//        F' = max(H'(i-1,j) - o, F'(i-1,j))          1 VIADDMNMX.S16x2
//        t  = max(H'(i-1,j-1) + (2e+mismatch), E')   1 VIADDMNMX.S16x2
//        H' = max3(H'(i-1,j-1) + q, t, F')           1 VIMNMX3.S16x2
//    where q = (2e+match) when the bases are equal and a large negative number otherwise. q comes
//    from the otherwise idle FMA pipe: base codes are fp16 values (1 + c/4), d = r - t (HADD2),
//    q = fma(d, -d, C) (HFMA2) with C the fp16 DENORMAL whose bit pattern is the integer 2e+match;
//    d == 0 gives exactly C, d != 0 gives a negative half whose bit pattern read as int16 is below
//    -12000. The add H' + q is a 32-bit IMAD (no carry crosses the lanes because every stored
//    value is in [0, 16000]). Four ALU-pipe instructions per two cells.
//  * reads whose length is not G*K: the first G*K-n threads treat their last column as absent
//    (pass the previous column's H/E through), per int16 lane.
#pragma once
#include "sdp_internal.cuh"

namespace sdp {

__device__ __forceinline__ uint32_t hadd2_u(uint32_t a, uint32_t b) {
    uint32_t d; asm("add.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b)); return d;
}
// fma(d, -d, c) per fp16 lane; non-ftz so the denormal addend survives
__device__ __forceinline__ uint32_t hfma2_negsq(uint32_t d, uint32_t c) {
    uint32_t r;
    asm("{.reg .b32 nd; neg.f16x2 nd, %1; fma.rn.f16x2 %0, %1, nd, %2;}" : "=r"(r) : "r"(d), "r"(c));
    return r;
}
__device__ __forceinline__ uint32_t imad_add(uint32_t one, uint32_t a, uint32_t b) {
    uint32_t r; asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(one), "r"(a), "r"(b)); return r;
}
// max per int16 lane plus, per lane, whether a >= b. Same PTX as CUDA's __vibmax_s16x2 but with an
// early-clobber output: the header's "=r" lets the result share a's register, which turns the
// predicates into constants when the caller writes `a = vibmax(a, b)`.
__device__ __forceinline__ uint32_t vibmax_s16x2(uint32_t a, uint32_t b, bool* a_ge_b_hi, bool* a_ge_b_lo) {
    uint32_t val, phi, plo;
    asm("{.reg .pred pu, pv; \n\t"
        ".reg .s16 rs0, rs1, rs2, rs3; \n\t"
        "max.s16x2 %0, %3, %4; \n\t"
        "mov.b32 {rs0, rs1}, %0; \n\t"
        "mov.b32 {rs2, rs3}, %3; \n\t"
        "setp.eq.s16 pv, rs0, rs2; \n\t"
        "setp.eq.s16 pu, rs1, rs3; \n\t"
        "selp.b32 %1, 1, 0, pu; \n\t"
        "selp.b32 %2, 1, 0, pv;} \n\t"
        : "=&r"(val), "=&r"(phi), "=&r"(plo) : "r"(a), "r"(b));
    *a_ge_b_hi = (phi != 0); *a_ge_b_lo = (plo != 0);
    return val;
}
__device__ __forceinline__ uint32_t blend(uint32_t mask, uint32_t a, uint32_t b) {  // mask ? a : b
    return (a & mask) | (b & ~mask);
}

// base `idx` (signed, relative to word pointer `base`) of a 2-bit packed buffer, N-mask aware
__device__ __forceinline__ uint32_t fetch_code(const uint32_t* __restrict__ packed,
                                               const uint32_t* __restrict__ nmask,
                                               uint64_t pos, uint32_t ncode) {
    uint32_t w = __ldg(packed + (pos >> 4));
    uint32_t c = (w >> (2u * ((uint32_t)pos & 15u))) & 3u;
    if (nmask != nullptr) {
        uint32_t mw = __ldg(nmask + (pos >> 5));
        if ((mw >> ((uint32_t)pos & 31u)) & 1u) c = ncode;
    }
    return c;
}

template <int K, bool REV>
__global__ void __launch_bounds__(SDP_SCORE_THREADS)
score_kernel(const ScoreParams P)
{
    const int lane = threadIdx.x & 31;
    const uint32_t task = P.task_begin + blockIdx.x * SDP_WARPS_PER_CTA + (threadIdx.x >> 5);
    if (task >= P.task_end) return;                       // warp-uniform

    // ---- which slot (read length) does this warp's task belong to
    uint32_t lo = P.slot_lo, hi = P.slot_hi;
    while (hi - lo > 1) {
        uint32_t mid = (lo + hi) >> 1;
        if (task >= __ldg(P.task_prefix + mid)) lo = mid; else hi = mid;
    }
    const SlotInfo si = P.slots[lo];
    const uint32_t local = task - __ldg(P.task_prefix + lo);
    const int G = si.G;
    const int ngroups = 32 / G;
    const int ppw = 2 * ngroups;
    const uint32_t first = si.first + local * ppw;
    const int cnt = min((uint32_t)ppw, si.count - local * ppw);

    int q = lane / G;
    int g = lane - q * G;
    const bool in_group = q < ngroups;
    if (!in_group) { q = 0; g = (G > 2) ? 1 : 0; }        // spare lanes shadow group 0, write nothing
    const bool hasA = in_group && (2 * q < cnt);
    const bool hasB = in_group && (2 * q + 1 < cnt);
    const PairDesc dA = P.desc[first + (hasA ? 2 * q : 0)];
    const PairDesc dB = hasB ? P.desc[first + 2 * q + 1] : dA;
    const bool is_first = (g == 0);
    const bool is_last = in_group && (g == G - 1);

    const int nA = (int)dA.n, nB = (int)dB.n;
    const int mA = (int)dA.m, mB = (int)dB.m;
    const int Mmin = __reduce_min_sync(0xffffffffu, min(mA, mB));
    const int Mmax = __reduce_max_sync(0xffffffffu, max(mA, mB));

    // ---- columns of this thread: the first pad = G*K - n threads skip their last column
    const int padA = G * K - nA, padB = G * K - nB;
    const bool skipA = g < padA, skipB = g < padB;
    const int startA = g * K - min(g, padA), startB = g * K - min(g, padB);
    const int realA = K - (skipA ? 1 : 0), realB = K - (skipB ? 1 : 0);
    const uint32_t skipmask = (skipA ? 0x0000FFFFu : 0u) | (skipB ? 0xFFFF0000u : 0u);

    uint32_t rh[K], H[K], F[K];
    const uint32_t h_row0 = P.c.betaMinusO2;              // H'(0,j) = -o + beta for j >= 1
#pragma unroll
    for (int k = 0; k < K; ++k) {
        uint32_t cA = SDP_CODE_READ_N, cB = SDP_CODE_READ_N;
        if (k < realA) {
            int r = startA + k;
            cA = fetch_code(P.reads_packed, P.read_nmask, dA.roff + (uint64_t)(REV ? nA - 1 - r : r), SDP_CODE_READ_N);
        }
        if (k < realB) {
            int r = startB + k;
            cB = fetch_code(P.reads_packed, P.read_nmask, dB.roff + (uint64_t)(REV ? nB - 1 - r : r), SDP_CODE_READ_N);
        }
        rh[k] = (0x3C00u + (cA << 8)) | ((0x3C00u + (cB << 8)) << 16);
        H[k] = h_row0;
        F[k] = 0u;                                        // F'(0,j) = -inf: 0 <= beta - 2o
    }

    const uint32_t one = P.c.one, negO = P.c.negO, cmis = P.c.cmis, Cf = P.c.Cf;
    uint32_t hout = h_row0, eout = 0u;
    uint32_t hdiag = is_first ? P.c.beta2 : h_row0;       // H'(0, left boundary column)
    uint32_t drift = 0u;                                  // packed e*i of the row this thread is on
    uint32_t best = REV ? h_row0 : 0x80008000u;           // reverse: row 0 (all-insertion) counts
    int idxA = 0, idxB = 0;

    auto row_step = [&](const int i, auto slow_tag) {
        constexpr bool SLOW = decltype(slow_tag)::value;
        uint32_t hin = __shfl_up_sync(0xffffffffu, hout, 1);
        uint32_t ein = __shfl_up_sync(0xffffffffu, eout, 1);
        if (SLOW && i < 1) return;                        // this thread has not reached row 1 yet
        drift = __vadd2(drift, P.c.e2);
        if (is_first) {
            hin = REV ? P.c.betaMinusO2 : __vadd2(P.c.beta2, drift);
            ein = 0u;
        }
        // window bases of row i for both lanes -> negated fp16 codes
        const int iA = min(i, mA), iB = min(i, mB);
        const uint32_t tA = fetch_code(P.wins_packed, P.win_nmask,
                                       REV ? dA.woff - (uint64_t)(iA - 1) : dA.woff + (uint64_t)(iA - 1), SDP_CODE_WIN_N);
        const uint32_t tB = fetch_code(P.wins_packed, P.win_nmask,
                                       REV ? dB.woff - (uint64_t)(iB - 1) : dB.woff + (uint64_t)(iB - 1), SDP_CODE_WIN_N);
        const uint32_t nt = (0xBC00u + (tA << 8)) | ((0xBC00u + (tB << 8)) << 16);

        uint32_t Hd = hdiag, Hl = hin, E = ein;
        uint32_t Hsk = hin, Esk = ein;                    // outputs if the last column is skipped
        hdiag = hin;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t d = hadd2_u(rh[k], nt);
            const uint32_t qv = hfma2_negsq(d, Cf);
            const uint32_t dg = imad_add(one, Hd, qv);
            E = __viaddmax_s16x2(Hl, negO, E);
            F[k] = __viaddmax_s16x2(H[k], negO, F[k]);
            const uint32_t t1 = __viaddmax_s16x2(Hd, cmis, E);
            const uint32_t Hn = __vimax3_s16x2(dg, t1, F[k]);
            Hd = H[k]; H[k] = Hn; Hl = Hn;
            if (k == K - 2) { Hsk = Hn; Esk = E; }
        }
        hout = blend(skipmask, Hsk, Hl);
        eout = blend(skipmask, Esk, E);

        if (is_last) {
            // running maximum of H(i,n) = H'(i,n) - e*i - (beta + e*n); strict > keeps the lowest
            // row (forward), >= keeps the highest (reverse)
            uint32_t cmp = __vsub2(Hl, drift);
            if (SLOW) {
                const uint32_t ok = (i <= mA ? 0x0000FFFFu : 0u) | (i <= mB ? 0xFFFF0000u : 0u);
                cmp = blend(ok, cmp, 0x80008000u);
            }
            bool p_hi, p_lo;
            if (REV) {
                best = vibmax_s16x2(cmp, best, &p_hi, &p_lo);       // p = cmp >= best
                if (p_lo) idxA = i;
                if (p_hi) idxB = i;
            } else {
                best = vibmax_s16x2(best, cmp, &p_hi, &p_lo);       // p = best >= cmp
                if (!p_lo) idxA = i;
                if (!p_hi) idxB = i;
            }
        }
    };

    int s = 1;
    for (; s < G; ++s) row_step(s - g, std::true_type{});                   // fill: some threads idle
    const int fast_end = Mmin + G - 1;
    for (; s <= fast_end; ++s) row_step(s - g, std::false_type{});          // steady state
    const int all_end = Mmax + G - 1;
    for (; s <= all_end; ++s) row_step(s - g, std::true_type{});            // lanes with fewer rows done

    if (is_last) {
        const int bA = (int)(int16_t)(best & 0xFFFFu), bB = (int)(int16_t)(best >> 16);
        const int sA = bA - P.c.beta - P.c.e * nA, sB = bB - P.c.beta - P.c.e * nB;
        if (REV) {
            // idx = rows of the reversed window consumed by the longest alignment scoring S;
            // the lowest co-optimal start is s_lo = ref_end + 1 - idx
            if (hasA) { P.rev_rows[dA.pid] = idxA; if (sA != dA.aux) atomicOr(P.err_flag, SDP_ERRF_REVERSE); }
            if (hasB) { P.rev_rows[dB.pid] = idxB; if (sB != dB.aux) atomicOr(P.err_flag, SDP_ERRF_REVERSE); }
        } else {
            if (hasA) { P.score[dA.pid] = sA; P.ref_end[dA.pid] = idxA - 1; }
            if (hasB) { P.score[dB.pid] = sB; P.ref_end[dB.pid] = idxB - 1; }
        }
    }
}

template <int K>
static void launch_score_K(bool rev, const ScoreParams& p, cudaStream_t st) {
    const uint32_t ntasks = p.task_end - p.task_begin;
    if (ntasks == 0) return;
    const uint32_t grid = (ntasks + SDP_WARPS_PER_CTA - 1) / SDP_WARPS_PER_CTA;
    if (rev) score_kernel<K, true><<<grid, SDP_SCORE_THREADS, 0, st>>>(p);
    else     score_kernel<K, false><<<grid, SDP_SCORE_THREADS, 0, st>>>(p);
}

}  // namespace sdp
