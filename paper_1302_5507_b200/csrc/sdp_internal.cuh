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

// Rows between neighbouring threads of a group: thread g works on row s - SDP_SCORE_SKEW*g at step s. With 1 the
// H'/E' a thread receives at step s were finished by its left neighbour at the very end of step s-1, so the serial
// chains of consecutive steps cannot overlap and a warp waits out the ALU latency between dependent chain
// instructions (measured: a third of the issue slots idle). With 2 they were finished at step s-2: the chains of two
// consecutive steps are independent (row i+1 only trails row i by a column inside the thread) and ptxas interleaves them.
#ifndef SDP_SCORE_SKEW
#define SDP_SCORE_SKEW 2
#endif


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
struct TraceConsts {            // arguments of the traceback DP kernels; the constants of their column loop are patched
                                // instruction immediates like the score kernels' (trace_kernel.cuh, ScorePatch)
    uint32_t e2;                   // packed 8 e
    uint32_t beta2;                // packed 8 beta + 7          : H7(i_lo, 0)
    uint32_t betaMinusO2;          // packed 8 (beta - o) + 7    : H7(i_lo, j >= 1)
    int32_t  e, beta;              // unscaled; beta = 3o + 8 + max(2e + mismatch, 0)
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
