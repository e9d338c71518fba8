// trace_kernel.cuh -- a5, wide pairs: the DP half of the traceback.
//
// The paper backtracks through tables D and M kept in global memory. Here no table
// survives the forward pass; instead the rectangle of window rows (i_lo, i_end] x all n read
// columns that contains every co-optimal path is recomputed with the same register-resident
// anti-diagonal wavefront as the score kernel (score_kernel.cuh: two rows of skew per thread, two rows per pass,
// scoring constants as patched instruction immediates), and each cell leaves FOUR BITS behind instead of two
// table entries:
//     bits 1..0  where M(i,j) came from: 3 = diagonal, 2 = D(i,j), 0/1 = I(i,j)   (diag > D > I)
//     bit  2     D(i,j) was opened from M(i-1,j)   (else extended from D(i-1,j))
//     bit  3     I(i,j) was opened from M(i,j-1)   (else extended from I(i,j-1))
// which is all the walk of PAPER.md:353 / DESIGN.md R6 ever asks of a cell.
//
// The bits are free by-products of the max instructions: every value is stored x8 and the three
// low bits of a candidate are a tag chosen so that (a) ties between candidates of equal value are
// won by the candidate the tie rule prefers (diag 7 > D opened 6 > D extended 2 > I opened 1 >
// I extended 0) and (b) the winner's tag survives in the low bits of the result. With c = 2e + mismatch,
// q' = delta - mismatch, F~ = F' - c as in the score kernel, and H kept as H7 = H | 7 (the diagonal tag rides on it):
//     Ft = max(H7(i-1,j) + 8(-o-c) - 1, Fc(i-1,j))      VIADDMNMX    Fc = Ft & ~4 (tag 2)       LOP3
//     u  = max(H7(i-1,j-1) + 8q', Ft)                   VIADDMNMX    8q' exact from the fp16 pipe (HADD2 + HFMA2.RELU)
//     Et = max(H7(i,j-1) - 8o - 6, Ec(i,j-1))           VIADDMNMX    Ec = Et & ~1               LOP3
//     Ht = max(u + 8c, Et)                              VIADDMNMX    H7 = Ht | 7                LOP3
//     v  = Ht & ~4 | Ft & 4                                                                     LOP3
// Eight ALU-pipe instructions per two cells (two pairs share the int16x2 lanes) against four in
// the score kernel. The nibble (H7 - v) + 8 (Et - Ec) -- the three low bits COMPLEMENTED, the walk undoes that -- and
// its packing run on the FMA pipe: two integer subtractions, then fp16 FMAs on the small integers as DENORMALS
// (t = eb*8 + x, byte = t0*16 + t1: exact below 2048), and one PRMT per four cells joins two bytes. Nibbles are
// left-aligned, four cells per 16-bit lane (cell kk of a word in bits 4*(3 - kk)), and stored step by step:
//     word((i, w, lane)) = task region + (((s-1)/2 * ceil(K/4) + w) * 32 + lane) * 2 + (s-1)%2,   low half = first pair,
// where s = i + SDP_SCORE_SKEW*g is the STEP at which thread g of its group works on row i: the threads of a warp are
// on different rows at any one time (anti-diagonal wavefront), so only a step-major layout makes a warp-wide
// store whole 128-byte lines; the two steps of one pass sit side by side, so a pass stores 8 bytes per thread and the
// walk gets two steps per 32-byte sector. One region of (rows + SKEW*(G - 1)) steps, rounded up to pairs, per warp task.
#pragma once
#include "score_kernel.cuh"

namespace sdp {

// sentinel immediates of the traceback DP kernels (patched like the score kernels', score_modules.cu)
#define SDP_SENT_T_NEGOF 0x4E2B7D13u    // packed 8 (-o - c) - 1
#define SDP_SENT_T_NEGOE 0x2D9C51E6u    // packed -8 o - 6
#define SDP_SENT_T_C8    0x35A8C6F1u    // packed 8 c
#define SDP_SENT_T_CD8   0x3B5E92A7u    // packed 8 (match - mismatch), read as an fp16 pair

__device__ __forceinline__ uint32_t sub_u32(uint32_t a, uint32_t b) {
    uint32_t r; asm("sub.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b)); return r;
}
// bitwise (mask ? b : a) in one LOP3
__device__ __forceinline__ uint32_t lop3_select(uint32_t a, uint32_t b, uint32_t mask) {
    uint32_t r; asm("lop3.b32 %0, %1, %2, %3, 0xD8;" : "=r"(r) : "r"(a), "r"(b), "r"(mask)); return r;
}

// nibble packer of one row: four cells -> one 32-bit word (16 bits per int16 lane)
struct NibblePack {
    uint32_t t0, b0, b1;
    __device__ __forceinline__ void reset() { t0 = 0u; b0 = 0u; b1 = 0u; }
    // returns true when `word` is complete (after cell k with k % 4 == 3 or k == last)
    template <int K>
    __device__ __forceinline__ bool add(const int k, const uint32_t t, uint32_t& word) {
        constexpr uint32_t H2_16 = 0x4C004C00u;            // fp16 16.0, both lanes
        if ((k & 1) == 0) t0 = t;
        if ((k & 1) == 1 || k == K - 1) {
            const uint32_t byte = (k & 1) ? hfma2_u(t0, H2_16, t) : hfma2_u(t0, H2_16, 0u);
            if ((k & 3) < 2) b0 = byte; else b1 = byte;
        }
        if ((k & 3) == 3 || k == K - 1) {
            if ((k & 3) < 2) b1 = 0u;
            word = __byte_perm(b1, b0, 0x6240);
            return true;
        }
        return false;
    }
};

template <int K, bool PAD>
__device__ __forceinline__ void trace_body(const ScoreParams& P, const TraceDP& T, uint32_t (*ring_mem)[SDP_RING_WORDS])
{
    constexpr int NW = (K + 3) / 4;
    constexpr int SKEW = SDP_SCORE_SKEW;
    static_assert(SKEW == 2, "the row-pair pass below assumes two rows of skew");
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
    const uint32_t h_row0 = T.c.betaMinusO2;              // H7(0,j) = 8 (beta - o) + 7 for j >= 1
#pragma unroll
    for (int k = 0; k < K; ++k) {
        uint32_t cA = SDP_CODE_READ_N, cB = SDP_CODE_READ_N;
        if (k < realA) cA = fetch_code(P.reads_packed, P.read_nmask, dA.roff + (uint64_t)(startA + k), SDP_CODE_READ_N);
        if (k < realB) cB = fetch_code(P.reads_packed, P.read_nmask, dB.roff + (uint64_t)(startB + k), SDP_CODE_READ_N);
        rh[k] = read_code_half(cA) | (read_code_half(cB) << 16);
        H[k] = h_row0;
        F[k] = 0x00020002u;                               // D(0,j) = -inf, carrying the "extended" tag
    }

    const RingGeom rg = ring_geometry(G, ngroups, SKEW);
    uint32_t* const ring_w = ring_mem[threadIdx.x >> 5] + q * rg.stride_w;
    const uint16_t* const rp0 = reinterpret_cast<const uint16_t*>(ring_w) + rg.mirror - SKEW * g;

    const bool st_ok = hasA;                              // hasB implies hasA
    // word (step pair, w, lane, step parity): the two rows of one pass go out as ONE 8-byte store per thread (a warp-wide
    // store is two full lines), and the walk finds two consecutive steps of a column group in one 32-byte sector
    constexpr uint32_t pairstride = 64u * NW;
    uint32_t* const wbase = T.bits + T.bits_off[first] + 2u * (uint32_t)lane;
    int tstep = 0;                                        // steps done by this warp (0-based step of the next row)

    constexpr uint32_t negOf = SDP_SENT_T_NEGOF, negOe = SDP_SENT_T_NEGOE, c8 = SDP_SENT_T_C8, Cd8 = SDP_SENT_T_CD8;
    constexpr uint32_t H2_8 = 0x48004800u;                // fp16 8.0, both lanes
    const uint32_t notfirst = opaque_u32(is_first ? 0u : 1u);            // multiplier: the select stays on the FMA pipe
    uint32_t fv = is_first ? T.c.beta2 : 0u;              // H7(i,0) = 8 (beta + e i) + 7: free start
    const uint32_t fstep = is_first ? T.c.e2 : 0u;
    uint32_t houtA = h_row0, eoutA = 0u, houtB = h_row0, eoutB = 0u;     // the two rows in flight towards the right neighbour
    uint32_t hdiag = is_first ? T.c.beta2 : h_row0;
    uint32_t fin = 0u;                                    // H7(m, n) per lane, caught on the lane's last row

    // one cell of two pairs: updates F (tag 2), E (tag 0), Hl (H7); returns the packed nibble value as an fp16 denormal
    auto cell = [&](const uint32_t hd, const uint32_t hup, uint32_t& Fk, const uint32_t nt, const uint32_t rcode,
                    uint32_t& Hl, uint32_t& E) -> uint32_t {
        const uint32_t qv = hfma2_relu_negsq(hsub2_u(nt, rcode), Cd8);
        const uint32_t Ft = __viaddmax_s16x2(hup, negOf, Fk);
        const uint32_t u = __viaddmax_s16x2(hd, qv, Ft);
        const uint32_t Et = __viaddmax_s16x2(Hl, negOe, E);
        const uint32_t Ht = __viaddmax_s16x2(u, c8, Et);
        Fk = Ft & 0xFFFBFFFBu;
        E = Et & 0xFFFEFFFEu;
        Hl = Ht | 0x00070007u;
        const uint32_t v = lop3_select(Ht, Ft, 0x00040004u);
        const uint32_t x = sub_u32(Hl, v);                // 7 - (Ht&3 | Ft&4) per lane, no borrow (Hl >= v per lane)
        const uint32_t eb = sub_u32(Et, E);               // Et & 1 per lane
        return hfma2_u(eb, H2_8, x);                      // x + 8 eb as fp16 denormals: exact
    };

    // One DP row of this thread's K columns (fill, drain and odd rows). Hs = H7(i-1, .) is only read, Hn receives H7(i, .).
    auto row_step = [&](const int i, const uint16_t* rp, auto slow_tag, const uint32_t (&Hs)[K], uint32_t (&Hn)[K],
                        uint32_t& hout, uint32_t& eout) {
        constexpr bool SLOW = decltype(slow_tag)::value;
        uint32_t hin = __shfl_up_sync(0xffffffffu, hout, 1);
        uint32_t ein = __shfl_up_sync(0xffffffffu, eout, 1);
        if (SLOW && i < 1) {
#pragma unroll
            for (int k = 0; k < K; ++k) Hn[k] = Hs[k];
            ++tstep;                                      // the layout follows the STEP, not the row (see above)
            return;
        }
        fv = __vadd2(fv, fstep);
        hin = imad_sel(hin, notfirst, fv);
        ein = imad_sel(ein, notfirst, 0u);
        const uint32_t nt = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, (uint32_t)*rp);
        // (thread g runs SKEW*(G-1-g) rows past Mmin inside the steady-state loop: always test the row)
        const bool do_store = st_ok && i <= Rpp;

        uint32_t Hl = hin, E = ein;
        uint32_t Hsk = hin, Esk = ein;
        uint32_t hd = hdiag;
        hdiag = hin;
        NibblePack np; np.reset();
        uint32_t* const wp = wbase + (uint32_t)(tstep >> 1) * pairstride + (uint32_t)(tstep & 1);
        ++tstep;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint32_t t = cell(hd, Hs[k], F[k], nt, rh[k], Hl, E);
            hd = Hs[k];
            Hn[k] = Hl;
            uint32_t word;
            if (np.template add<K>(k, t, word)) { if (do_store) wp[(k >> 2) * 64] = word; }
            if (PAD && k == K - 2) { Hsk = Hl; Esk = E; }
        }
        if (PAD) { hout = blend(skipmask, Hsk, Hl); eout = blend(skipmask, Esk, E); }
        else     { hout = Hl; eout = E; }
        if (is_last) {
            if (i == mA) fin = (fin & 0xFFFF0000u) | (Hl & 0x0000FFFFu);
            if (i == mB) fin = (fin & 0x0000FFFFu) | (Hl & 0xFFFF0000u);
        }
    };
    // Two consecutive steps of the steady state (rows ia and ia + 1 of this thread) as ONE skewed pass, as in the score
    // kernel: column k of the first row, then column k-1 of the second, whose "row above" is the first row's chain value.
    auto row_pair = [&](const int ia, const uint16_t* rp) {
        uint32_t hinA = __shfl_up_sync(0xffffffffu, houtA, 1);
        uint32_t einA = __shfl_up_sync(0xffffffffu, eoutA, 1);
        uint32_t hinB = __shfl_up_sync(0xffffffffu, houtB, 1);
        uint32_t einB = __shfl_up_sync(0xffffffffu, eoutB, 1);
        fv = __vadd2(fv, fstep);
        hinA = imad_sel(hinA, notfirst, fv);
        einA = imad_sel(einA, notfirst, 0u);
        fv = __vadd2(fv, fstep);
        hinB = imad_sel(hinB, notfirst, fv);
        einB = imad_sel(einB, notfirst, 0u);
        const uint32_t ntA = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, (uint32_t)rp[0]);
        const uint32_t ntB = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, (uint32_t)rp[1]);
        const bool storeA = st_ok && ia <= Rpp;           // (the region has room for the pass's second row past Rpp)
        uint2* const wp2 = reinterpret_cast<uint2*>(wbase + (uint32_t)(tstep >> 1) * pairstride);   // tstep is even here
        tstep += 2;

        uint32_t HlA = hinA, EA = einA, HlB = hinB, EB = einB;
        uint32_t hdA = hdiag, hdB = hinA;                 // H7(ia-1, left), H7(ia, left)
        hdiag = hinB;
        uint32_t HskA = hinA, EskA = einA, HskB = hinB, EskB = einB;
        uint32_t prevA = hinA;                            // H7(ia, k-1)
        NibblePack npA, npB; npA.reset(); npB.reset();
        uint32_t pendA = 0u;                              // the first row's word, until the second row's word of the same cells
#pragma unroll
        for (int k = 0; k <= K; ++k) {
            const uint32_t upB = prevA;                   // H7(ia, k-1): the second row's "row above" at column k-1
            const uint32_t pendB = pendA;                 // (the first row may finish its LAST word in this very iteration)
            if (k < K) {                                  // first row, column k
                const uint32_t t = cell(hdA, H[k], F[k], ntA, rh[k], HlA, EA);
                hdA = H[k];
                prevA = HlA;
                uint32_t word;
                if (npA.template add<K>(k, t, word)) pendA = word;
                if (PAD && k == K - 2) { HskA = HlA; EskA = EA; }
            }
            if (k >= 1) {                                 // second row, column k-1
                const uint32_t t = cell(hdB, upB, F[k - 1], ntB, rh[k - 1], HlB, EB);
                hdB = upB;
                H[k - 1] = HlB;
                uint32_t word;
                if (npB.template add<K>(k - 1, t, word)) { if (storeA) wp2[((k - 1) >> 2) * 32] = make_uint2(pendB, word); }
                if (PAD && k - 1 == K - 2) { HskB = HlB; EskB = EB; }
            }
        }
        if (PAD) {
            houtA = blend(skipmask, HskA, HlA); eoutA = blend(skipmask, EskA, EA);
            houtB = blend(skipmask, HskB, HlB); eoutB = blend(skipmask, EskB, EB);
        } else { houtA = HlA; eoutA = EA; houtB = HlB; eoutB = EB; }
        if (is_last) {
            if (ia == mA) fin = (fin & 0xFFFF0000u) | (HlA & 0x0000FFFFu);
            if (ia == mB) fin = (fin & 0x0000FFFFu) | (HlA & 0xFFFF0000u);
            if (ia + 1 == mA) fin = (fin & 0xFFFF0000u) | (HlB & 0x0000FFFFu);
            if (ia + 1 == mB) fin = (fin & 0x0000FFFFu) | (HlB & 0xFFFF0000u);
        }
    };
    // one step outside the paired loop; the two output sets trade places afterwards
    auto row_step1 = [&](const int i, const uint16_t* rp, auto slow_tag) {
        uint32_t H2[K];
        row_step(i, rp, slow_tag, H, H2, houtA, eoutA);
#pragma unroll
        for (int k = 0; k < K; ++k) H[k] = H2[k];
        const uint32_t th = houtA, te = eoutA;
        houtA = houtB; eoutA = eoutB; houtB = th; eoutB = te;
    };

    const int lead = SKEW * (G - 1);
    const int fast_end = Mmin + lead, all_end = Mmax + lead;
    for (int s0 = 0; s0 < all_end; s0 += rg.chunk) {
        if (in_group) fill_ring_rows<false>(P, rg, ring_w, g, G, s0, dA.woff, mA, dB.woff, mB);
        __syncwarp();
        const int send = min(s0 + rg.chunk, all_end);
        const uint16_t* rp = rp0 + (s0 & (rg.ring - 1));
        int s = s0 + 1;
#pragma unroll 1
        for (; s <= min(send, lead); ++s, ++rp) row_step1(s - SKEW * g, rp, std::true_type{});
        const int fe = min(send, fast_end);
#pragma unroll 1
        for (; s + 1 <= fe; s += 2, rp += 2) row_pair(s - SKEW * g, rp);     // (four rows per iteration: measured slower)
#pragma unroll 1
        for (; s <= fe; ++s, ++rp) row_step1(s - SKEW * g, rp, std::false_type{});
#pragma unroll 1
        for (; s <= send; ++s, ++rp) row_step1(s - SKEW * g, rp, std::true_type{});
    }

    if (is_last) {
        // the restricted DP must end on the forward score: H7(m, n) = 8 (S + e (m + n) + beta) + 7
        const int fA = (int)(fin & 0xFFFFu) >> 3, fB = (int)(fin >> 16) >> 3;
        if (hasA && fA - T.c.beta - T.c.e * (nA + mA) != dA.aux) atomicOr(P.err_flag, SDP_ERRF_TRACE);
        if (hasB && fB - T.c.beta - T.c.e * (nB + mB) != dB.aux) atomicOr(P.err_flag, SDP_ERRF_TRACE);
    }
}

}  // namespace sdp
