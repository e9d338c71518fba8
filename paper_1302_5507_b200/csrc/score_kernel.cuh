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
//    s - 2g at step s (anti-diagonal wavefront, two rows of skew per thread: SDP_SCORE_SKEW); H and E of the
//    chunk's last column cross to the right neighbour with one warp shuffle each per row.
//  * drift form: stored values are H + e*(i+j) + beta, so gap extension needs no add. With
//    c = 2e + mismatch (any sign) and q' = delta - mismatch = (match - mismatch) or 0:
//        F~ = max(H'(i-1,j) - (o + c), F~(i-1,j))      VIADDMNMX.S16x2   F~ = F' - c         (off the chain)
//        u~ = max(H'(i-1,j-1) + q', F~)                VIADDMNMX.S16x2   u~ = u - c          (off the chain)
//        E' = max(H'(i,j-1) - o, E'(i,j-1))            VIADDMNMX.S16x2                       (the row's serial chain)
//        H' = max(u~ + c, E')                          VIADDMNMX.S16x2                       (the row's serial chain)
//    Four ALU-pipe instructions per two cells, for EVERY scoring. q' comes from the FMA pipe, which runs beside the ALU pipe (measured: DESIGN.md "Pipes"), in
//    two instructions: base codes are fp16 values at least 1 apart, d = t - r (HADD2) and
//    q' = relu(Cd - d*d) (HFMA2.RELU) with Cd the fp16 DENORMAL whose bit pattern is the integer match - mismatch:
//    d == 0 gives exactly Cd (the FMA is not flush-to-zero), |d| >= 1 a negative value that relu turns into +0,
//    so the result's bit pattern IS the integer q'. Shifting F and u by c moves the constant part of the
//    diagonal increment into the add of the H' update, which a plain max left unused.
//    No integer multiply-add and no register move is wanted in the column loop: IMAD and IMAD.MOV cost two
//    FMA-pipe slots on sm_100a (measured).
//  * window rows: the 2-bit window bases of both lanes are expanded once per chunk of rows into
//    a per-group shared-memory ring of 16-bit PRMT selectors; a row then costs one LDS.U16 and one
//    PRMT to obtain the fp16 codes of both lanes (instead of two address computations, two global
//    loads and the bit extraction per row and thread).
//  * reads whose length is not G*K (PAD variant): the first G*K-n threads treat their last column
//    as absent (pass the previous column's H/E through), per int16 lane.
#pragma once
#include "sdp_internal.cuh"

namespace sdp {

// fp16 codes: the half whose two bytes both equal B[c], for c = A,C,G,T, read-N (4), window-N (5):
// 0x3C3C = 1.059, 0x4040 = 2.125, 0x4242 = 3.129, 0x4444 = 4.266, 0x4545 = 5.270, 0x4646 = 6.273.
// Any two differ by more than 1 and every difference is exact in fp16, so d*d >= 1 unless the
// bases are equal. Read-N and window-N have different codes: N never matches, not even N.
#define SDP_TBL_LO 0x4442403Cu      // PRMT source a: bytes 0..3 = A C G T
#define SDP_TBL_HI 0x00004645u      // PRMT source b: byte 4 = read N, byte 5 = window N

__device__ __forceinline__ uint32_t read_code_half(uint32_t c) {      // c in 0..4
    const uint32_t t = __byte_perm(SDP_TBL_LO, SDP_TBL_HI, c);
    return (t & 0xFFu) * 0x0101u;
}

// value the optimiser cannot see through (keeps masks from being turned back into predicates + SEL)
__device__ __forceinline__ uint32_t opaque_u32(uint32_t x) {
    uint32_t r; asm("mov.b32 %0, %1;" : "=r"(r) : "r"(x)); return r;
}
// PRMT without the selector masking __byte_perm adds (every selector nibble here is <= 5)
__device__ __forceinline__ uint32_t prmt_raw(uint32_t a, uint32_t b, uint32_t sel) {
    uint32_t r; asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel)); return r;
}
__device__ __forceinline__ uint32_t hsub2_u(uint32_t a, uint32_t b) {
    uint32_t d; asm("sub.rn.f16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b)); return d;
}
// relu(c - d*d) per fp16 lane; non-ftz so a denormal c survives: c when d == 0, +0 when d*d > c
__device__ __forceinline__ uint32_t hfma2_relu_negsq(uint32_t d, uint32_t c) {
    uint32_t r;
    asm("{.reg .b32 nd; neg.f16x2 nd, %1; fma.rn.relu.f16x2 %0, %1, nd, %2;}" : "=r"(r) : "r"(d), "r"(c));
    return r;
}
// a * m + c as a 32-bit integer multiply-add (FMA pipe): with m in {0, 1} a select that stays off the ALU pipe
__device__ __forceinline__ uint32_t imad_sel(uint32_t a, uint32_t m, uint32_t c) {
    uint32_t r; asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(m), "r"(c)); return r;
}
// sat(1 - d*d) per fp16 lane: 1.0 when d == 0, 0.0 when |d| >= 1
__device__ __forceinline__ uint32_t hfma2_is_zero(uint32_t d) {
    uint32_t r;
    asm("{.reg .b32 nd, on; neg.f16x2 nd, %1; mov.b32 on, 0x3C003C00; fma.rn.sat.f16x2 %0, %1, nd, on;}"
        : "=r"(r) : "r"(d));
    return r;
}
__device__ __forceinline__ uint32_t hfma2_u(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t r; asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c)); return r;
}
__device__ __forceinline__ uint32_t add_s16x2(uint32_t a, uint32_t b) {
    uint32_t r; asm("add.s16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b)); return r;
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
// running maximum with its row: val = max(a, b) per int16 lane; a lane's index becomes i when the lane of `a` LOST
// (KEEP_A_ON_TIE) or when the lane of `a` won or tied (!KEEP_A_ON_TIE ... see callers). One VIMNMX.S16x2 that also
// writes the two "a >= b" predicates, and two predicated moves.
template <bool MOVE_IF_A_WINS>
__device__ __forceinline__ uint32_t vibmax_track(uint32_t a, uint32_t b, int i, int& idx_lo, int& idx_hi) {
    uint32_t val;
    if (MOVE_IF_A_WINS)
        asm("{.reg .pred pu, pv; \n\t"
            ".reg .s16 rs0, rs1, rs2, rs3; \n\t"
            "max.s16x2 %0, %3, %4; \n\t"
            "mov.b32 {rs0, rs1}, %0; \n\t"
            "mov.b32 {rs2, rs3}, %3; \n\t"
            "setp.eq.s16 pv, rs0, rs2; \n\t"
            "setp.eq.s16 pu, rs1, rs3; \n\t"
            "@pv mov.b32 %1, %5; \n\t"
            "@pu mov.b32 %2, %5;} \n\t"
            : "=&r"(val), "+r"(idx_lo), "+r"(idx_hi) : "r"(a), "r"(b), "r"(i));
    else
        asm("{.reg .pred pu, pv; \n\t"
            ".reg .s16 rs0, rs1, rs2, rs3; \n\t"
            "max.s16x2 %0, %3, %4; \n\t"
            "mov.b32 {rs0, rs1}, %0; \n\t"
            "mov.b32 {rs2, rs3}, %3; \n\t"
            "setp.eq.s16 pv, rs0, rs2; \n\t"
            "setp.eq.s16 pu, rs1, rs3; \n\t"
            "@!pv mov.b32 %1, %5; \n\t"
            "@!pu mov.b32 %2, %5;} \n\t"
            : "=&r"(val), "+r"(idx_lo), "+r"(idx_hi) : "r"(a), "r"(b), "r"(i));
    return val;
}
__device__ __forceinline__ uint32_t blend(uint32_t mask, uint32_t a, uint32_t b) {  // mask ? a : b
    return (a & mask) | (b & ~mask);
}

// base at position `pos` of a 2-bit packed buffer, N-mask aware
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

// 16 consecutive bases starting at base position `pos` (may lie partly outside [0, 16*nwords));
// words outside the buffer read as 0
__device__ __forceinline__ uint32_t load_bases16(const uint32_t* __restrict__ packed, long long pos, long long nwords) {
    const long long w = pos >> 4;
    const uint32_t sh = ((uint32_t)pos & 15u) * 2u;
    const uint32_t lo = (w >= 0 && w < nwords) ? __ldg(packed + w) : 0u;
    const uint32_t hi = (sh != 0u && w + 1 >= 0 && w + 1 < nwords) ? __ldg(packed + w + 1) : 0u;
    return __funnelshift_r(lo, hi, sh);
}
// 16 consecutive mask bits starting at bit position `pos`
__device__ __forceinline__ uint32_t load_bits16(const uint32_t* __restrict__ bits, long long pos, long long nwords) {
    const long long w = pos >> 5;
    const uint32_t sh = (uint32_t)pos & 31u;
    const uint32_t lo = (w >= 0 && w < nwords) ? __ldg(bits + w) : 0u;
    const uint32_t hi = (sh > 16u && w + 1 >= 0 && w + 1 < nwords) ? __ldg(bits + w + 1) : 0u;
    return __funnelshift_r(lo, hi, sh) & 0xFFFFu;
}
// reverse the order of the sixteen 2-bit fields / of the low sixteen bits
__device__ __forceinline__ uint32_t reverse_fields2(uint32_t x) {
    x = __brev(x);
    return ((x & 0x55555555u) << 1) | ((x >> 1) & 0x55555555u);
}
__device__ __forceinline__ uint32_t reverse_bits16(uint32_t x) { return __brev(x) >> 16; }

// Shared-memory ring of window-row selectors: per warp SDP_RING_WORDS 32-bit words, carved into one
// region per group. A region holds `ring` 16-bit entries (row i at slot (i-1) & (ring-1), stored at
// position slot + mirror) plus a `mirror`-entry copy of the ring's tail in front of it, so that thread g
// can read row s - skew*g at position ((s-1) & (ring-1)) + mirror - skew*g without a wrap test.
struct RingGeom {
    int chunk, ring, stride_w, mirror;
};
__device__ __forceinline__ RingGeom ring_geometry(int G, int ngroups, int skew, bool short_chunks = false) {
    RingGeom r;
    r.mirror = skew * (G - 1) > 32 ? 64 : 32;             // (64 only when one group fills the warp)
    if (G == 1)      { r.chunk = 32; r.stride_w = 49; }
    else if (G == 2) { r.chunk = 32; r.stride_w = 50; }
    else {
        // short_chunks (reverse pass): its early-exit test runs once per chunk. A chunk must still cover the
        // skew * (G - 1) <= 62 rows the group's last thread trails behind (the ring keeps one chunk of history).
        r.chunk = short_chunks ? 64 : 128;
        const int want = (32 / ngroups) & 31;             // bank offset between neighbouring groups
        const int base = r.chunk + 16;                    // >= (2 * chunk + 32) / 2 words
        r.stride_w = base + ((want - base) & 31);         // == want (mod 32)
    }
    r.ring = 2 * r.chunk;
    return r;
}


// Expand window rows s0+1 .. s0+chunk of both int16 lanes into the group's selector ring (thread g
// of G takes every G-th unit of 16 rows). REV walks the window backwards from woff.
template <bool REV>
__device__ __forceinline__ void fill_ring_rows(const ScoreParams& P, const RingGeom& rg, uint32_t* ring_w,
                                               int g, int G, int s0, uint64_t woffA, int mA, uint64_t woffB, int mB)
{
    const long long win_words = (long long)P.wins_words, nm_words = (long long)P.win_nmask_words;
    for (int u = g; u < rg.chunk / 16; u += G) {
        const int r0 = s0 + 16 * u;                       // 0-based row of the unit's first entry
        uint32_t a = 0u, b = 0u, na = 0u, nb = 0u;
        if (r0 < mA) {
            a = REV ? reverse_fields2(load_bases16(P.wins_packed, (long long)woffA - r0 - 15, win_words))
                    : load_bases16(P.wins_packed, (long long)woffA + r0, win_words);
            if (P.win_nmask != nullptr)
                na = REV ? reverse_bits16(load_bits16(P.win_nmask, (long long)woffA - r0 - 15, nm_words))
                         : load_bits16(P.win_nmask, (long long)woffA + r0, nm_words);
        }
        if (r0 < mB) {
            b = REV ? reverse_fields2(load_bases16(P.wins_packed, (long long)woffB - r0 - 15, win_words))
                    : load_bases16(P.wins_packed, (long long)woffB + r0, win_words);
            if (P.win_nmask != nullptr)
                nb = REV ? reverse_bits16(load_bits16(P.win_nmask, (long long)woffB - r0 - 15, nm_words))
                         : load_bits16(P.win_nmask, (long long)woffB + r0, nm_words);
        }
        const int slot0 = r0 & (rg.ring - 1);
        uint32_t* dst = ring_w + ((rg.mirror + slot0) >> 1);
        uint32_t* mir = (slot0 >= rg.ring - rg.mirror) ? ring_w + ((slot0 - (rg.ring - rg.mirror)) >> 1) : nullptr;
        uint32_t ww[8];
#pragma unroll
        for (int tt = 0; tt < 8; ++tt) {
            // two rows -> two 16-bit selectors (idxA * 0x11 | idxB * 0x1100)
            const uint32_t x = (a >> (4 * tt)) & 0xFu, y = (b >> (4 * tt)) & 0xFu;
            uint32_t w = ((x * 0x44011u) & 0x00330033u) | (((y * 0x44011u) << 8) & 0x33003300u);
            if (na | nb) {                                // window N -> table index 5
                const uint32_t ma = (na >> (2 * tt)) & 3u, mb = (nb >> (2 * tt)) & 3u;
                if (ma & 1u) w = (w & 0xFFFFFF00u) | 0x00000055u;
                if (ma & 2u) w = (w & 0xFF00FFFFu) | 0x00550000u;
                if (mb & 1u) w = (w & 0xFFFF00FFu) | 0x00005500u;
                if (mb & 2u) w = (w & 0x00FFFFFFu) | 0x55000000u;
            }
            ww[tt] = w;
        }
        // The unit's 8 words. With G = 4 word-wide stores put the warp's lanes on 8 banks (groups 4 banks apart, units 8
        // words apart): a four-way conflict; two 128-bit stores per lane are conflict-free there (a quarter-warp covers
        // all 32 banks; the regions are 16-byte aligned). Measured: config 2 forward 6.72 -> 6.68 ms; with G = 8 the
        // same change is 1 % slower, so it stays with G = 4.
        if (G == 4) {
            reinterpret_cast<uint4*>(dst)[0] = make_uint4(ww[0], ww[1], ww[2], ww[3]);
            reinterpret_cast<uint4*>(dst)[1] = make_uint4(ww[4], ww[5], ww[6], ww[7]);
            if (mir != nullptr) {
                reinterpret_cast<uint4*>(mir)[0] = make_uint4(ww[0], ww[1], ww[2], ww[3]);
                reinterpret_cast<uint4*>(mir)[1] = make_uint4(ww[4], ww[5], ww[6], ww[7]);
            }
        } else {
#pragma unroll
            for (int tt = 0; tt < 8; ++tt) { dst[tt] = ww[tt]; if (mir != nullptr) mir[tt] = ww[tt]; }
        }
    }
}

// Rows per iteration of the steady-state loop (even). ptxas pays ~45 register moves per loop
// iteration to bring the loop-carried H/F registers back to their entry assignment, and a move
// (IMAD.MOV) costs as much FMA-pipe time as two HFMA2: unrolling amortises them.
#ifndef SDP_ROWS_UNROLL
#define SDP_ROWS_UNROLL 8
#endif

// resident CTAs per SM the register budget is sized for: 128 registers up to K = 21, 168 above
#ifndef SDP_SCORE_MIN_CTAS
#define SDP_SCORE_MIN_CTAS(K) ((K) <= 21 ? 4 : 3)
#endif

// The scoring constants of the column loop are INSTRUCTION IMMEDIATES, not registers. Each VIADDMNMX then reads two
// registers instead of three, which matters because the register file delivers one operand per bank per cycle to
// BOTH pipes: with three-register DPX instructions the fp16 instructions of the FMA pipe no longer fit beside them
// (measured on B200: 10.1 against 9.0 cycles per column for the same instruction mix; the forward pass of config 2
// went from 7.4 to 6.7 ms). The scoring is a run-time argument of sdp_create, so the kernels are compiled to a cubin
// with the SENTINEL values below as immediates, and score_modules.cu rewrites those immediates in a copy of the
// cubin with the context's scoring before loading it. Sentinels are arbitrary
// 32-bit patterns (both halves finite fp16 values) that occur nowhere else in the code.
#define SDP_SENT_NEGOC 0x5D1A37C2u      // packed -(o + c)
#define SDP_SENT_NEGO  0x2B6E4A91u      // packed -o
#define SDP_SENT_C2    0x63C5195Du      // packed c = 2e + mismatch
#define SDP_SENT_CD    0x39E2746Bu      // packed match - mismatch (bit pattern of an fp16 pair)
#define SDP_SENT_E2    0x1F83528Eu      // packed e

template <int K, bool REV, bool PAD>
__device__ __forceinline__ void score_body(const ScoreParams& P, uint32_t (*ring_mem)[SDP_RING_WORDS])
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
    if (!in_group) { q = 0; g = 1; }                      // spare lanes (G >= 3) shadow group 0, write nothing
    const bool hasA = in_group && (2 * q < cnt);
    const bool hasB = in_group && (2 * q + 1 < cnt);
    const PairDesc dA = P.desc[first + (hasA ? 2 * q : 0)];
    const PairDesc dB = hasB ? P.desc[first + 2 * q + 1] : dA;
    const bool is_first = in_group && (g == 0);
    const bool is_last = in_group && (g == G - 1);

    const int nA = (int)dA.n, nB = (int)dB.n;
    const int mA = (int)dA.m, mB = (int)dB.m;
    // (reverse pass: a descriptor with m == 0 is a pair whose rectangle the reverse pass would not pay for; it keeps
    // its place in the task but takes no part: not in the row bounds, no output, no check)
    const int Mmin = __reduce_min_sync(0xffffffffu, REV ? min(mA > 0 ? mA : 0x7fffffff, mB > 0 ? mB : 0x7fffffff) : min(mA, mB));
    const int Mmax = __reduce_max_sync(0xffffffffu, max(mA, mB));
    if (REV && Mmax == 0) return;                         // warp-uniform: nothing to do for this task

    // ---- columns of this thread: the first pad = G*K - n threads skip their last column
    const int padA = PAD ? G * K - nA : 0, padB = PAD ? G * K - nB : 0;
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
        rh[k] = read_code_half(cA) | (read_code_half(cB) << 16);
        H[k] = h_row0;
        F[k] = 0u;                                        // F~(0,j) = -inf: 0 <= beta - 2o - c
    }

    // ---- window-row selector ring of this group
    constexpr int SKEW = SDP_SCORE_SKEW;
    const RingGeom rg = ring_geometry(G, ngroups, SKEW, REV);
    uint32_t* const ring_w = ring_mem[threadIdx.x >> 5] + q * rg.stride_w;
    const uint16_t* const rp0 = reinterpret_cast<const uint16_t*>(ring_w) + rg.mirror - SKEW * g;

    auto fill_ring = [&](const int s0) {                  // rows s0+1 .. s0+chunk
        if (in_group) fill_ring_rows<REV>(P, rg, ring_w, g, G, s0, dA.woff, mA, dB.woff, mB);
    };

    constexpr uint32_t negOc = SDP_SENT_NEGOC, negO = SDP_SENT_NEGO, c2 = SDP_SENT_C2, Cd = SDP_SENT_CD, e2 = SDP_SENT_E2;
    // 1 for every thread but the group's first: hin * notfirst + fv is a select on the FMA pipe (kept opaque so
    // that it stays a multiplier instead of becoming a predicate and an ALU-pipe SEL)
    const uint32_t notfirst = opaque_u32(is_first ? 0u : 1u);
    // boundary column 0 as seen by the group's first thread: H'(i,0) = beta + e*i (forward, free start) or
    // beta - o (reverse, start anchored: a leading deletion of i bases costs o + e*i)
    uint32_t fv = is_first ? (REV ? P.c.betaMinusO2 : P.c.beta2) : 0u;
    const uint32_t fstep = (is_first && !REV) ? e2 : 0u;
    // what the right neighbour fetches: H'(i, last column), E'(i, last column). With a skew of two rows the values of
    // two steps are in flight, alternating between the two sets.
    uint32_t houtA = h_row0, eoutA = 0u, houtB = h_row0, eoutB = 0u;
    uint32_t hdiag = is_first ? P.c.beta2 : h_row0;       // H'(0, left boundary column)
    // running maximum of H(i,n) in the drift frame of the current row: best += e per row, so that
    // H'(i,n) can be compared with it directly. Reverse: row 0 (all-insertion) counts.
    uint32_t best = REV ? h_row0 : 0x80008000u;
    int idxA = 0, idxB = 0;

    // One DP row of this thread's K columns. Hs = H'(i-1, .) is only read, Hn receives H'(i, .):
    // two register sets that swap roles from row to row, so that no H' value is ever copied.
    auto row_step = [&](const int i, const uint16_t* rp, auto slow_tag, const uint32_t (&Hs)[K], uint32_t (&Hn)[K],
                        uint32_t& hout, uint32_t& eout) {
        constexpr bool SLOW = decltype(slow_tag)::value;
        uint32_t hin = __shfl_up_sync(0xffffffffu, hout, 1);
        uint32_t ein = __shfl_up_sync(0xffffffffu, eout, 1);
        if (SLOW && i < 1) {                              // this thread has not reached row 1 yet
#pragma unroll
            for (int k = 0; k < K; ++k) Hn[k] = Hs[k];
            return;
        }
        fv = __vadd2(fv, fstep);
        hin = imad_sel(hin, notfirst, fv);
        ein = imad_sel(ein, notfirst, 0u);                // E'(i,0) = -inf
        // fp16 codes of the window bases of row i, both lanes
        const uint32_t nt = prmt_raw(SDP_TBL_LO, SDP_TBL_HI, (uint32_t)*rp);

        uint32_t Hl = hin, E = ein;
        uint32_t Hsk = hin, Esk = ein;                    // outputs if the last column is skipped
        // u~[k] = max(H'(i-1,k-1) + q', F~(i,k)): everything of column k that does not wait for the chain
        auto off_chain = [&](const int k, const uint32_t hd) -> uint32_t {
            const uint32_t d = hsub2_u(nt, rh[k]);
            F[k] = __viaddmax_s16x2(Hs[k], negOc, F[k]);
            return __viaddmax_s16x2(hd, hfma2_relu_negsq(d, Cd), F[k]);
        };
        Hn[0] = off_chain(0, hdiag);
        hdiag = hin;
#pragma unroll
        for (int k = 0; k < K; ++k) {
            if (k + 1 < K) Hn[k + 1] = off_chain(k + 1, Hs[k]);
            E = __viaddmax_s16x2(Hl, negO, E);            // E'(i,k)
            Hl = __viaddmax_s16x2(Hn[k], c2, E);          // H'(i,k) = max(u~ + c, E')
            Hn[k] = Hl;
            if (PAD && k == K - 2) { Hsk = Hl; Esk = E; }
        }
        if (PAD) { hout = blend(skipmask, Hsk, Hl); eout = blend(skipmask, Esk, E); }
        else     { hout = Hl; eout = E; }

        {   // Running maximum of the thread's last column; only the group's last thread holds H'(i,n) there, the other
            // threads' copies are never read. Unconditional on purpose: under a predicate ptxas computes into
            // temporaries and pays a conditional register move per value.
            // strict > keeps the lowest row (forward), >= keeps the highest (reverse)
            best = __vadd2(best, e2);
            uint32_t cmp = Hl;
            if (SLOW) {
                const uint32_t ok = (i <= mA ? 0x0000FFFFu : 0u) | (i <= mB ? 0xFFFF0000u : 0u);
                cmp = blend(ok, cmp, 0x80008000u);
            }
            if (REV) best = vibmax_track<true>(cmp, best, i, idxA, idxB);     // row i takes over when cmp >= best
            else     best = vibmax_track<false>(best, cmp, i, idxA, idxB);    // ... when not (best >= cmp)
        }
    };
    // Two consecutive steps of the steady state (rows ia and ia + 1 of this thread) as ONE skewed pass: column k of
    // the first row, then column k-1 of the second, which needs nothing of the first row beyond column k-1. The two
    // rows' serial chains are independent (SKEW == 2: both rows' inputs were shuffled in before the pass), so each
    // chain instruction has the other row's work between itself and its successor, and no second H' register set
    // is needed: the second row takes H'(ia, k-1) straight from the first row's chain.
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

        uint32_t HlA = hinA, EA = einA, HlB = hinB, EB = einB;
        uint32_t hdA = hdiag, hdB = hinA;                 // H'(ia-1, left), H'(ia, left)
        hdiag = hinB;
        uint32_t HskA = hinA, EskA = einA, HskB = hinB, EskB = einB;
        uint32_t prevA = hinA;                            // H'(ia, k-1)
#pragma unroll
        for (int k = 0; k <= K; ++k) {
            const uint32_t upB = prevA;                   // H'(ia, k-1): the second row's "row above" at column k-1
            if (k < K) {                                  // first row, column k
                const uint32_t d = hsub2_u(ntA, rh[k]);
                F[k] = __viaddmax_s16x2(H[k], negOc, F[k]);
                const uint32_t u = __viaddmax_s16x2(hdA, hfma2_relu_negsq(d, Cd), F[k]);
                hdA = H[k];
                EA = __viaddmax_s16x2(HlA, negO, EA);
                HlA = __viaddmax_s16x2(u, c2, EA);
                prevA = HlA;
                if (PAD && k == K - 2) { HskA = HlA; EskA = EA; }
            }
            if (k >= 1) {                                 // second row, column k-1
                const uint32_t d = hsub2_u(ntB, rh[k - 1]);
                F[k - 1] = __viaddmax_s16x2(upB, negOc, F[k - 1]);
                const uint32_t u = __viaddmax_s16x2(hdB, hfma2_relu_negsq(d, Cd), F[k - 1]);
                hdB = upB;
                EB = __viaddmax_s16x2(HlB, negO, EB);
                HlB = __viaddmax_s16x2(u, c2, EB);
                H[k - 1] = HlB;
                if (PAD && k - 1 == K - 2) { HskB = HlB; EskB = EB; }
            }
        }
        if (PAD) {
            houtA = blend(skipmask, HskA, HlA); eoutA = blend(skipmask, EskA, EA);
            houtB = blend(skipmask, HskB, HlB); eoutB = blend(skipmask, EskB, EB);
        } else { houtA = HlA; eoutA = EA; houtB = HlB; eoutB = EB; }
        best = __vadd2(best, e2);
        if (REV) best = vibmax_track<true>(HlA, best, ia, idxA, idxB);
        else     best = vibmax_track<false>(best, HlA, ia, idxA, idxB);
        best = __vadd2(best, e2);
        if (REV) best = vibmax_track<true>(HlB, best, ia + 1, idxA, idxB);
        else     best = vibmax_track<false>(best, HlB, ia + 1, idxA, idxB);
    };
    // one step outside the unrolled loop; the two output sets trade places afterwards
    auto row_step1 = [&](const int i, const uint16_t* rp, auto slow_tag) {
        uint32_t H2[K];
        row_step(i, rp, slow_tag, H, H2, houtA, eoutA);
#pragma unroll
        for (int k = 0; k < K; ++k) H[k] = H2[k];
        if (SKEW == 2) {
            const uint32_t th = houtA, te = eoutA;
            houtA = houtB; eoutA = eoutB; houtB = th; eoutB = te;
        }
    };

    // step s: thread g works on row s - SKEW*g. Steps 1..SKEW*(G-1) fill the wavefront, steps up to
    // Mmin+SKEW*(G-1) are the steady state (SDP_ROWS_UNROLL rows per iteration), the rest drain lanes whose
    // window is longer.
    const int lead = SKEW * (G - 1);
    const int fast_end = Mmin + lead, all_end = Mmax + lead;
    int rows_done = Mmax;
    // (the exit test adds up to n*match + e*SKEW*G to a stored value: only where that still fits 16 bits)
    const bool can_exit = REV && 2 * P.c.match * max(nA, nB) + P.c.e * (max(nA, nB) + Mmax + SKEW * G + 2) + P.c.beta <= 32000;
    for (int s0 = 0; s0 < all_end; s0 += rg.chunk) {
        fill_ring(s0);
        __syncwarp();
        const int send = min(s0 + rg.chunk, all_end);
        const uint16_t* rp = rp0 + (s0 & (rg.ring - 1));
        int s = s0 + 1;
#pragma unroll 1
        for (; s <= min(send, lead); ++s, ++rp) row_step1(s - SKEW * g, rp, std::true_type{});
        const int fe = min(send, fast_end);
#pragma unroll 1
        for (; s + SDP_ROWS_UNROLL - 1 <= fe; s += SDP_ROWS_UNROLL, rp += SDP_ROWS_UNROLL) {
            if (SKEW == 2) {
#pragma unroll
                for (int r = 0; r < SDP_ROWS_UNROLL; r += 2) row_pair(s + r - SKEW * g, rp + r);
            } else {
                uint32_t H2[K];
#pragma unroll
                for (int r = 0; r < SDP_ROWS_UNROLL; r += 2) {
                    row_step(s + r - SKEW * g, rp + r, std::false_type{}, H, H2, houtA, eoutA);
                    row_step(s + r + 1 - SKEW * g, rp + r + 1, std::false_type{}, H2, H, houtA, eoutA);
                }
            }
        }
#pragma unroll 1
        for (; s <= fe; ++s, ++rp) row_step1(s - SKEW * g, rp, std::false_type{});
#pragma unroll 1
        for (; s <= send; ++s, ++rp) row_step1(s - SKEW * g, rp, std::true_type{});
        if (REV) rows_done = send - lead;
        if (REV && can_exit && send < all_end) {
            // Early exit of the reverse pass. The pass looks for the LAST row whose M(i,n) equals the forward score S
            // (dA.aux), so it may stop as soon as no later row can reach S. Any path to a later cell of column n leaves
            // the cells computed so far through a cell on their staircase frontier -- a thread's current row, the cell left
            // of it that the thread's next row takes as its diagonal neighbour, the last column of one of its two most
            // recent rows (the right neighbour trails by SKEW rows), or the closed-form boundary column 0 -- and gains at
            // most `match` per read base it still has to consume:
            //     M(i2, n) <= max over frontier cells (i,j) of  M(i,j) + (n - j) * match.
            // In drift form (stored X' = X + e(i+j) + beta, this thread at row s - SKEW*g):
            //     alive  <=>  X' + (n-j)*match - e*j + e*SKEW*g  >=  S + beta + e*s.
            const int M = P.c.match, e = P.c.e;
            const int jA = startA + 1, jB = startB + 1;             // 1-based column of H[0]
            uint32_t c = sdp_pack_lo_hi((nA - jA) * M - e * jA + e * SKEW * g, (nB - jB) * M - e * jB + e * SKEW * g);
            const uint32_t dstep = sdp_pack2(-(M + e));
            uint32_t acc = 0x80008000u;
#pragma unroll
            for (int k = 0; k < K; ++k) { acc = __viaddmax_s16x2(H[k], c, acc); c = __vadd2(c, dstep); }
            {   // the lane's true last column, one row back: one more e of allowance covers both rows in flight
                const int lA = startA + realA, lB = startB + realB;
                const uint32_t cl = sdp_pack_lo_hi((nA - lA) * M - e * lA + e * SKEW * g + e, (nB - lB) * M - e * lB + e * SKEW * g + e);
                acc = __viaddmax_s16x2(houtA, cl, acc);
                if (SKEW == 2) acc = __viaddmax_s16x2(houtB, cl, acc);
            }
            if (is_first) acc = __viaddmax_s16x2(fv, sdp_pack_lo_hi(nA * M, nB * M), acc);   // boundary column 0
            else {
                // the diagonal neighbour of this thread's next cell: M(current row, column left of H[0]), still to be used
                acc = __viaddmax_s16x2(hdiag, sdp_pack_lo_hi((nA - jA + 1) * M - e * (jA - 1) + e * SKEW * g,
                                                             (nB - jB + 1) * M - e * (jB - 1) + e * SKEW * g), acc);
            }
            const int tA = dA.aux + P.c.beta + e * send, tB = dB.aux + P.c.beta + e * send;
            const bool alive = (hasA && mA > 0 && (int)(int16_t)(acc & 0xFFFFu) >= tA) ||
                               (hasB && mB > 0 && (int)(int16_t)(acc >> 16) >= tB);
            if (!__any_sync(0xffffffffu, alive)) break;
        }
    }

    if (is_last) {
        // best = H'(idx,n) + e*(rows_done - idx) = H(idx,n) + e*(n + rows_done) + beta, rows_done = rows this thread
        // went through (Mmax unless the reverse pass stopped early)
        const int bA = (int)(int16_t)(best & 0xFFFFu), bB = (int)(int16_t)(best >> 16);
        const int sA = bA - P.c.beta - P.c.e * (nA + rows_done), sB = bB - P.c.beta - P.c.e * (nB + rows_done);
        if (REV) {
            // idx = rows of the reversed window consumed by the longest alignment scoring S;
            // the lowest co-optimal start is s_lo = ref_end + 1 - idx
            if (hasA && mA > 0) { P.rev_rows[dA.pid] = idxA; if (sA != dA.aux) atomicOr(P.err_flag, SDP_ERRF_REVERSE); }
            if (hasB && mB > 0) { P.rev_rows[dB.pid] = idxB; if (sB != dB.aux) atomicOr(P.err_flag, SDP_ERRF_REVERSE); }
        } else {
            if (hasA) { P.score[dA.pid] = sA; P.ref_end[dA.pid] = idxA - 1; }
            if (hasB) { P.score[dB.pid] = sB; P.ref_end[dB.pid] = idxB - 1; }
        }
    }
}

}  // namespace sdp
