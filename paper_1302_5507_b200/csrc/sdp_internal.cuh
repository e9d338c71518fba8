// sdp_internal.cuh -- structures shared by the kernels and the host-side driver of libsdp.
// Not part of the ABI (include/sdp.h is). Notation follows the paper:
// window T[1..m] indexed by i (rows), read R[1..n] indexed by j (columns).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define SDP_WARPS_PER_CTA 4
#define SDP_SCORE_THREADS (32 * SDP_WARPS_PER_CTA)
#define SDP_MAX_K 32            // columns of the read one thread keeps in registers
#define SDP_NBINS 65536         // bucket-sort key space: (n-1) * 64 + min(63, rows >> 6)
#define SDP_BIN_SCRATCH 60      // words behind bin_start[SDP_NBINS] the bin scan may use
#define SDP_NSLOTS 1024         // one slot per read length 1..SDP_MAX_READ_LEN
#define SDP_RING_WORDS 1792     // shared-memory words per warp for the window-row selector rings
#define SDP_KEY_SKIP 0xFFFFFFFFu

// device-side error flag bits
#define SDP_ERRF_INDEX   1u     // pair index / offset out of range, empty sequence
#define SDP_ERRF_REVERSE 2u     // reverse pass did not reproduce the forward score (internal)
#define SDP_ERRF_RANGE   4u     // int16 range rule or SDP_MAX_READ_LEN broken
#define SDP_ERRF_TRACE   8u     // traceback left its band or overflowed its run buffer (internal)

// code index of the two N kinds (0..3 = ACGT); fp16 values in score_kernel.cuh
#define SDP_CODE_READ_N 4u
#define SDP_CODE_WIN_N 5u

// One pair as the score kernel sees it, stored in bucket order.
struct PairDesc {
    uint64_t roff;     // first read base (in bases) -- forward orientation for both passes
    uint64_t woff;     // window base of DP row 1: win_off (forward) or win_off + ref_end (reverse)
    uint32_t n;        // read length (columns)
    uint32_t m;        // DP rows: window length (forward) or min(ref_end + 1, n + W) (reverse)
    uint32_t pid;      // caller pair index
    int32_t  aux;      // reverse pass: forward score S
};

// One read length in the task table. Tasks (one per warp) of slot s are
// task_prefix[s] .. task_prefix[s+1]; task t of the slot takes pairs first + t*ppw ..
struct SlotInfo {
    uint32_t first;    // index of the slot's first pair in bucket order
    uint32_t count;    // pairs in the slot
    uint32_t n;        // read length
    uint16_t G;        // threads per pair-of-pairs (anti-diagonal group)
    uint16_t K;        // columns per thread; G*K - n in [0, G)
};

struct ScoreConsts {           // what the score kernels take as arguments; the constants of their column loop are
                               // instruction immediates (ScorePatch in sdp_host.cuh, score_kernel.cuh)
    uint32_t beta2;            // packed int16x2 beta
    uint32_t betaMinusO2;      // packed beta - o
    int32_t  e, beta;          // scalars
    int32_t  match;            // reverse pass: early-exit bound
};

struct ScoreParams {
    const uint32_t* reads_packed; const uint32_t* read_nmask;
    const uint32_t* wins_packed;  const uint32_t* win_nmask;
    uint64_t wins_words;           // 32-bit words addressable in wins_packed / win_nmask (loads outside
    uint64_t win_nmask_words;      // read as 0)
    const PairDesc* desc;
    const uint32_t* task_prefix;   // [SDP_NSLOTS + 1], slots in (K, padded) order
    const SlotInfo* slots;         // [SDP_NSLOTS]
    uint32_t slot_lo, slot_hi;     // slots of this launch's (K, padded) class
    uint32_t task_begin, task_end; // == task_prefix[slot_lo], task_prefix[slot_hi]
    ScoreConsts c;
    int32_t* score;                // forward outputs, caller order
    int32_t* ref_end;
    int32_t* rev_rows;             // reverse output: window rows consumed by the longest alignment
                                   // that scores S (lowest co-optimal start = ref_end + 1 - rows)
    uint32_t* err_flag;            // reverse: SDP_ERRF_REVERSE when max != S
};

// Traceback DP (trace_kernel.cuh): the same wavefront in a x8 scaled domain whose low three bits
// carry "which operand won" tags. All fields are packed int16x2 unless noted.
#define SDP_TB_SCALE 8
#define SDP_TB_MAX_VALUE 4090   // largest unscaled drift-form value: 8 * 4090 + 7 <= 32767
struct TraceConsts {
    uint32_t cm1;                  // 0xFFFFFFFF (-1), opaque multiplier: subtractions as IMAD on the FMA pipe
    uint32_t m4;                   // 0x00040004, opaque so that the tag select stays one LOP3
    uint32_t negO_e;               // 8 * (-o) + 1 : "I opened here" candidate (tag bit 0)
    uint32_t negO_f;               // 8 * (-o) + 6 : "D opened here" candidate (tag bit 2); D extended carries tag 2
    uint32_t qx;                   // 8 * (2e + mismatch) + 7 : diagonal increment of a mismatch, tag 7
    uint32_t Cd8;                  // fp16 denormal whose bits are 8 * (match - mismatch)
    uint32_t e2, beta2, betaMinusO2;   // 8e, 8 beta, 8 (beta - o)
    int32_t  e, beta;              // unscaled
};

struct TraceDP {
    TraceConsts c;
    uint32_t* bits;                // direction nibbles, one region per pair of pairs
    const uint64_t* bits_off;      // [desc index of the region's first pair] word offset of the region
};

// packed helpers
__host__ __device__ constexpr static inline uint32_t sdp_pack_lo_hi(int lo, int hi) {
    return ((uint32_t)(uint16_t)(int16_t)lo) | (((uint32_t)(uint16_t)(int16_t)hi) << 16);
}
__host__ __device__ constexpr static inline uint32_t sdp_pack2(int v) {
    return ((uint32_t)(uint16_t)(int16_t)v) | (((uint32_t)(uint16_t)(int16_t)v) << 16);
}
