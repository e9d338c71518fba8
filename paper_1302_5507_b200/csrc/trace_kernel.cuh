// trace_kernel.cuh -- a5, wide pairs: the DP half of the traceback.
//
// The paper backtracks through tables D and M kept in global memory. Here no table
// survives the forward pass; instead the rectangle of window rows (i_lo, i_end] x all n read
// columns that contains every co-optimal path is recomputed with the same register-resident
// anti-diagonal wavefront as the score kernel (score_kernel.cuh), and each cell leaves FOUR BITS
// behind instead of two table entries:
//     bits 1..0  where M(i,j) came from: 3 = diagonal, 2 = D(i,j), 0/1 = I(i,j)   (diag > D > I)
//     bit  2     D(i,j) was opened from M(i-1,j)   (else extended from D(i-1,j))
//     bit  3     I(i,j) was opened from M(i,j-1)   (else extended from I(i,j-1))
// which is all the walk of PAPER.md:353 / DESIGN.md R6 ever asks of a cell.
//
// The bits are free by-products of the max instructions: every value is stored x8 and the three
// low bits of a candidate are a tag chosen so that (a) ties between candidates of equal value are
// won by the candidate the tie rule prefers (diag 7 > D opened 6 > D extended 2 > I opened 1 >
// I extended 0) and (b) the winner's tag survives in the low bits of the result:
//     Et = max(Hc(i,j-1) - 8o + 1, Ec(i,j-1))             VIADDMNMX   tag bit 0 = opened
//     Ft = max(Hc(i-1,j) - 8o + 6, Fc(i-1,j) [= 8v+2])    VIADDMNMX   tag bit 2 = opened
//     u  = max(Hc(i-1,j-1) + q8, Ft)                      VIADDMNMX   q8 = 8(2e+delta)+7, exact (fp16 pipe,
//     Ht = max(u, Et)                                     VIMNMX           as in score_kernel.cuh)
//     Ec = Et & ~1, Fc = Ft & ~4, Hc = Ht & ~7            3 LOP3      clean values for the next cell
//     v  = Ht & ~4 | Ft & 4                               1 LOP3
// Eight ALU-pipe instructions per two cells (two pairs share the int16x2 lanes) against four in
// the score kernel. The nibble (v - Hc) + 8 (Et - Ec) and its packing run on the FMA pipe: the two
// subtractions are 32-bit IMADs (an IMAD costs two HFMA2 slots on sm_100a, but masking the tags out with
// two more LOP3 instead loads the ALU pipe, which is this kernel's bottleneck: measured 6 % slower), then fp16
// FMAs on the small integers as DENORMALS (t = eb*8 + nib, byte = t0*16 + t1: exact below 2048),
// and one PRMT per four cells joins two bytes. Nibbles are left-aligned, four cells per 16-bit
// lane (cell kk of a word in bits 4*(3 - kk)), and stored row by row:
//     word((i, w, lane)) = task region + ((s-1) * ceil(K/4) + w) * 32 + lane,   low half = first pair of the two,
// where s = i + g is the STEP at which thread g of its group works on row i: the threads of a warp are on
// different rows at any one time (anti-diagonal wavefront), so only a step-major layout makes a warp-wide
// store one 128-byte line. One region of (rows + G - 1) steps per warp task.
#pragma once
#include "score_kernel.cuh"

namespace sdp {

// bitwise (mask ? b : a) in one LOP3 (mask kept in a register: a LOP3 takes one immediate at most)
__device__ __forceinline__ uint32_t imad_u(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r; asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c)); return r;
}
__device__ __forceinline__ uint32_t lop3_select(uint32_t a, uint32_t b, uint32_t mask) {
    uint32_t r; asm("lop3.b32 %0, %1, %2, %3, 0xD8;" : "=r"(r) : "r"(a), "r"(b), "r"(mask)); return r;
}

template <int K, bool PAD>
__global__ void __launch_bounds__(SDP_SCORE_THREADS, SDP_SCORE_MIN_CTAS(K))
trace_kernel(const ScoreParams P, const TraceDP T)
{
    __shared__ uint32_t ring_mem[SDP_WARPS_PER_CTA][SDP_RING_WORDS];
    constexpr int NW = (K + 3) / 4;
    const int lane = threadIdx.x & 31;
    const uint32_t task = P.task_begin + blockIdx.x * SDP_WARPS_PER_CTA + (threadIdx.x >> 5);
    if (task >= P.task_end) return;                       // warp-uniform

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
    if (!in_group) { q = 0; g = 1; }                      // spare lanes shadow group 0, write nothing
    const bool hasA = in_group && (2 * q < cnt);
    const bool hasB = in_group && (2 * q + 1 < cnt);
    const PairDesc dA = P.desc[first + (hasA ? 2 * q : 0)];
    const PairDesc dB = hasB ? P.desc[first + 2 * q + 1] : dA;
    const bool is_first = in_group && (g == 0);
    const bool is_last = in_group && (g == G - 1);

    const int nA = (int)dA.n, nB = (int)dB.n;
    const int mA = (int)dA.m, mB = (int)dB.m;
    const int Rpp = max(mA, mB);                          // rows of this group's region
    const int Mmin = __reduce_min_sync(0xffffffffu, min(mA, mB));
    const int Mmax = __reduce_max_sync(0xffffffffu, Rpp);

    const int padA = PAD ? G * K - nA : 0, padB = PAD ? G * K - nB : 0;
    const bool skipA = g < padA, skipB = g < padB;
    const int startA = g * K - min(g, padA), startB = g * K - min(g, padB);
    const int realA = K - (skipA ? 1 : 0), realB = K - (skipB ? 1 : 0);
    const uint32_t skipmask = (skipA ? 0x0000FFFFu : 0u) | (skipB ? 0xFFFF0000u : 0u);

    uint32_t rh[K], H[K], F[K];
    const uint32_t h_row0 = T.c.betaMinusO2;              // 8 (H'(0,j)) = 8 (beta - o) for j >= 1
#pragma unroll
    for (int k = 0; k < K; ++k) {
        uint32_t cA = SDP_CODE_READ_N, cB = SDP_CODE_READ_N;
        if (k < realA) cA = fetch_code(P.reads_packed, P.read_nmask, dA.roff + (uint64_t)(startA + k), SDP_CODE_READ_N);
        if (k < realB) cB = fetch_code(P.reads_packed, P.read_nmask, dB.roff + (uint64_t)(startB + k), SDP_CODE_READ_N);
        rh[k] = read_code_half(cA) | (read_code_half(cB) << 16);
        H[k] = h_row0;
        F[k] = 0x00020002u;                               // D(0,j) = -inf, carrying the "extended" tag
    }

    const RingGeom rg = ring_geometry(G, ngroups, 1);
    uint32_t* const ring_w = ring_mem[threadIdx.x >> 5] + q * rg.stride_w;
    const uint16_t* const rp0 = reinterpret_cast<const uint16_t*>(ring_w) + rg.mirror - g;

    const bool st_ok = hasA;                              // hasB implies hasA
    constexpr uint32_t rowstride = 32u * NW;              // word (step, w, lane): a warp-wide store is one 128-byte line
    uint32_t* wp = T.bits + T.bits_off[first] + (uint32_t)lane;

    const uint32_t m4 = T.c.m4, Cd8 = T.c.Cd8, cm1 = T.c.cm1;
    const uint32_t negOe = T.c.negO_e, negOf = T.c.negO_f, qx = T.c.qx, e2 = T.c.e2;
    constexpr uint32_t H2_8 = 0x48004800u, H2_16 = 0x4C004C00u;        // fp16 8.0 and 16.0, both lanes
    const uint32_t notfirst = opaque_u32(is_first ? 0u : 0xFFFFFFFFu);   // a mask, not a predicate: one LOP3 per use
    uint32_t fv = is_first ? T.c.beta2 : 0u;              // 8 H'(i,0) = 8 (beta + e i): free start
    const uint32_t fstep = is_first ? e2 : 0u;
    uint32_t hout = h_row0, eout = 0u;
    uint32_t hdiag = is_first ? T.c.beta2 : h_row0;
    uint32_t fin = 0u;                                    // 8 H'(m, n) per lane, caught on the lane's last row

    auto row_step = [&](const int i, const uint16_t* rp, auto slow_tag, const uint32_t (&Hs)[K], uint32_t (&Hn)[K]) {
        constexpr bool SLOW = decltype(slow_tag)::value;
        uint32_t hin = __shfl_up_sync(0xffffffffu, hout, 1);
        uint32_t ein = __shfl_up_sync(0xffffffffu, eout, 1);
        if (SLOW && i < 1) {
#pragma unroll
            for (int k = 0; k < K; ++k) Hn[k] = Hs[k];
            wp += rowstride;                              // wp follows the STEP, not the row (see the layout above)
            return;
        }
        fv = __vadd2(fv, fstep);
        hin = (hin & notfirst) | fv;
        ein = ein & notfirst;
        const uint32_t nt = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, (uint32_t)*rp);
        // (thread g runs G-1-g rows past Mmin inside the steady-state loop: always test the row)
        const bool do_store = st_ok && i <= Rpp;

        uint32_t Hl = hin, E = ein;
        uint32_t Hsk = hin, Esk = ein;
        uint32_t hd = hdiag;
        hdiag = hin;
        uint32_t b0 = 0u, b1 = 0u, t0 = 0u;              // high byte, low byte of the current word; first nibble of a byte
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t q8 = hfma2_u(hfma2_is_zero(hsub2_u(nt, rh[k])), Cd8, qx);
            const uint32_t Ft = __viaddmax_s16x2(Hs[k], negOf, F[k]);
            F[k] = Ft & 0xFFFBFFFBu;
            const uint32_t u = __viaddmax_s16x2(hd, q8, Ft);
            hd = Hs[k];
            const uint32_t Et = __viaddmax_s16x2(Hl, negOe, E);
            E = Et & 0xFFFEFFFEu;
            const uint32_t Ht = __vmaxs2(u, Et);
            Hl = Ht & 0xFFF8FFF8u;
            Hn[k] = Hl;
            const uint32_t v = lop3_select(Ht, Ft, m4);
            // v - Hc and Et - Ec as 32-bit IMADs (no borrow crosses the lanes: Hc <= v, Ec <= Et per lane). An IMAD
            // costs two FMA-pipe slots, but the ALU pipe is this kernel's bottleneck and the FMA pipe has room.
            const uint32_t nib = imad_u(Hl, cm1, v);      // bits 2..0
            const uint32_t eb = imad_u(E, cm1, Et);       // 0 or 1
            const uint32_t t = hfma2_u(eb, H2_8, nib);    // nib + 8 eb as fp16 denormals: exact
            if ((k & 1) == 0) t0 = t;
            if ((k & 1) == 1 || k == K - 1) {
                const uint32_t byte = (k & 1) ? hfma2_u(t0, H2_16, t) : hfma2_u(t0, H2_16, 0u);
                if ((k & 3) < 2) b0 = byte; else b1 = byte;
            }
            if ((k & 3) == 3 || k == K - 1) {
                if ((k & 3) < 2) b1 = 0u;
                if (do_store) wp[(k >> 2) * 32] = __byte_perm(b1, b0, 0x6240);
            }
            if (PAD && k == K - 2) { Hsk = Hl; Esk = E; }
        }
        wp += rowstride;
        if (PAD) { hout = blend(skipmask, Hsk, Hl); eout = blend(skipmask, Esk, E); }
        else     { hout = Hl; eout = E; }
        if (is_last) {
            if (i == mA) fin = (fin & 0xFFFF0000u) | (Hl & 0x0000FFFFu);
            if (i == mB) fin = (fin & 0x0000FFFFu) | (Hl & 0xFFFF0000u);
        }
    };
    auto row_step1 = [&](const int i, const uint16_t* rp, auto slow_tag) {
        uint32_t H2[K];
        row_step(i, rp, slow_tag, H, H2);
#pragma unroll
        for (int k = 0; k < K; ++k) H[k] = H2[k];
    };

    const int fast_end = Mmin + G - 1, all_end = Mmax + G - 1;
    for (int s0 = 0; s0 < all_end; s0 += rg.chunk) {
        if (in_group) fill_ring_rows<false>(P, rg, ring_w, g, G, s0, dA.woff, mA, dB.woff, mB);
        __syncwarp();
        const int send = min(s0 + rg.chunk, all_end);
        const uint16_t* rp = rp0 + (s0 & (rg.ring - 1));
        int s = s0 + 1;
#pragma unroll 1
        for (; s <= min(send, G - 1); ++s, ++rp) row_step1(s - g, rp, std::true_type{});
        const int fe = min(send, fast_end);
#pragma unroll 1
        for (; s + 1 <= fe; s += 2, rp += 2) {
            uint32_t H2[K];
            row_step(s - g, rp, std::false_type{}, H, H2);
            row_step(s + 1 - g, rp + 1, std::false_type{}, H2, H);
        }
        if (s <= fe) { row_step1(s - g, rp, std::false_type{}); ++s; ++rp; }
#pragma unroll 1
        for (; s <= send; ++s, ++rp) row_step1(s - g, rp, std::true_type{});
    }

    if (is_last) {
        // the restricted DP must end on the forward score: 8 H'(m,n) = 8 (S + e (m + n) + beta)
        const int fA = (int)(fin & 0xFFFFu) >> 3, fB = (int)(fin >> 16) >> 3;
        if (hasA && fA - T.c.beta - T.c.e * (nA + mA) != dA.aux) atomicOr(P.err_flag, SDP_ERRF_TRACE);
        if (hasB && fB - T.c.beta - T.c.e * (nB + mB) != dB.aux) atomicOr(P.err_flag, SDP_ERRF_TRACE);
    }
}

template <int K>
static void launch_trace_K(bool pad, const ScoreParams& p, const TraceDP& t, cudaStream_t st) {
    const uint32_t ntasks = p.task_end - p.task_begin;
    if (ntasks == 0) return;
    const uint32_t grid = (ntasks + SDP_WARPS_PER_CTA - 1) / SDP_WARPS_PER_CTA;
    if (pad) trace_kernel<K, true><<<grid, SDP_SCORE_THREADS, 0, st>>>(p, t);
    else     trace_kernel<K, false><<<grid, SDP_SCORE_THREADS, 0, st>>>(p, t);
}

}  // namespace sdp
