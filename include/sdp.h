/*
 * sdp.h -- C ABI of libsdp: batched semi-global affine-gap (Gotoh) alignment on one B200.
 *
 * The operation is the gapped-alignment stage of SOAP3-dp (arXiv 1302.5507, Methods section 3):
 * "Given a candidate region T (of length m) and a read R (of length n), the aim is to find a
 * sub-region T' inside T such that the alignment score between R and T' is maximum"
 * (PAPER.md:267), with the recurrences of PAPER.md:289-293, the base cases of PAPER.md:303-310
 * and the result max_{1<=i<=m} M(i,n) of PAPER.md:269, followed by backtracking.
 * Tie rules, the similarity filter and every other point the paper leaves open are fixed in
 * DESIGN.md ("Readings"). All arithmetic runs in hand-written sm_100a kernels; there is no CPU
 * fallback.
 *
 * Sequence layout (both reads and windows)
 *   2 bits per base, A=0 C=1 G=2 T=3; base k of a buffer sits in bits 2*(k mod 16) (LSB first)
 *   of little-endian uint32 word k/16. Offsets are in BASES, so windows may be overlapping views
 *   into one packed reference and a read may appear in many pairs. *_nmask (nullable) holds one
 *   bit per base on the same base offsets (bit k mod 32 of word k/32); a set bit makes the
 *   position N, which scores as a mismatch against everything including N. Buffers must be
 *   readable up to the next multiple of 16 bytes past the last word used.
 *
 * Coordinates are 0-based, inclusive, relative to the window. The whole read is aligned
 * (read_start = 0, read_end = n-1; SDP_MODE_LOCAL differs, see sdp_set_mode). ref_end - ref_start + 1 is the number of window bases the
 * CIGAR consumes and may be 0 (an all-insertion alignment reports ref_start = ref_end + 1).
 * CIGAR runs use the BAM encoding (len << 4) | op with M=0, I=1, D=2; runs of one pair are
 * contiguous, in alignment order, at cigar_ops[cigar_off[p] .. cigar_off[p] + cigar_len[p]).
 */
#ifndef SDP_H_
#define SDP_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SDP_OK       0
#define SDP_EINVAL  (-1)  /* null pointer, bad scoring, empty sequence, index / offset out of range  */
#define SDP_ERANGE  (-2)  /* a pair is beyond even the int32 lane (see the range rule below)                 */
#define SDP_ECUDA   (-3)  /* a CUDA call failed; sdp_last_error() has the CUDA message                */
#define SDP_ENOMEM  (-4)  /* host or device allocation failed                                         */

/* Longest read the register-resident int16 kernels take (32 lanes x 32 columns). */
#define SDP_MAX_READ_LEN 1024
/*
 * int16 range rule (per pair, n = read length, m = window length):
 *     match*n + gap_extend*(n + m + 32) + 3*gap_open + 8 + |2*gap_extend + mismatch| <= SDP_MAX_CELL_VALUE
 * The int16 kernels store H + gap_extend*(i+j) + bias in 16-bit lanes; the left side bounds every stored value and
 * every intermediate sum (R13). A pair that breaks the rule, or whose read is longer than SDP_MAX_READ_LEN,
 * is never clamped and never rejected for that: it takes the int32 lane (one thread per pair, much slower, same
 * results). SDP_ERANGE is left for what that lane cannot hold either: a sequence longer than SDP_MAX_SEQ_LEN, a pair
 * outside the int32 range rule below, or traceback scratch of one pair beyond 16 GiB.
 */
#define SDP_MAX_CELL_VALUE 32000
#define SDP_MAX_SEQ_LEN 1000000
/*
 * int32 range rule (per pair): match*n + gap_extend*(n + 2) + 2*gap_open + |mismatch| < SDP_MAX_CELL_VALUE_I32.
 * The int32 lane and the band traceback mark cells outside the table with -2^28; the rule keeps that mark, even after
 * n matches were added to it, below every real cell value. It only binds for scorings far from the default: with
 * 1/-3/5/2 a read of SDP_MAX_SEQ_LEN bases is inside it, with all four parameters at SDP_MAX_SCORE_PARAM reads up to
 * about 33,000 bases are. A pair that breaks it makes the call return SDP_ERANGE (nothing is clamped).
 */
#define SDP_MAX_CELL_VALUE_I32 (1 << 28)
/* Largest magnitude of match, mismatch, gap_open and gap_extend sdp_create accepts. */
#define SDP_MAX_SCORE_PARAM 4000

typedef struct sdp_ctx sdp_ctx;   /* opaque; owns device scratch, result buffers, pinned staging */

/* Scoring of PAPER.md:283: S_MA = match, S_MI = mismatch, S_GO = -(gap_open + gap_extend),
 * S_GE = -gap_extend, i.e. a gap of k bases costs gap_open + k*gap_extend. */
typedef struct sdp_scoring {
    int32_t match;           /* 0 .. SDP_MAX_SCORE_PARAM, and match - mismatch > 0              */
    int32_t mismatch;        /* -SDP_MAX_SCORE_PARAM .. 0                                       */
    int32_t gap_open;        /* 0 .. SDP_MAX_SCORE_PARAM                                        */
    int32_t gap_extend;      /* 1 .. SDP_MAX_SCORE_PARAM                                        */
    double  min_similarity;  /* in [0,1]; quantised once as q = llround(x * 1e6); a pair passes  */
                             /* iff n_match * 1e6 >= q * n_cols (n_cols = CIGAR columns)         */
} sdp_scoring;

/* Inputs of one call. Every pointer is caller-owned and read-only: DEVICE memory for
 * sdp_align_batch, HOST memory for sdp_align_batch_host. */
typedef struct sdp_batch {
    const uint32_t* reads_packed;  /* 2-bit packed read bases                                   */
    const uint64_t* read_off;      /* [n_reads] first base of read r, in bases                  */
    const uint32_t* read_len;      /* [n_reads] length in bases, 1..SDP_MAX_SEQ_LEN             */
    const uint32_t* read_nmask;    /* nullable N bitmap over reads_packed's base offsets        */
    uint32_t        n_reads;
    uint64_t        reads_bases;   /* bases addressable in reads_packed (for bounds checks)     */
    const uint32_t* wins_packed;   /* 2-bit packed windows or one packed reference              */
    const uint64_t* win_off;       /* [n_wins]                                                  */
    const uint32_t* win_len;       /* [n_wins] >= 1                                             */
    const uint32_t* win_nmask;     /* nullable                                                  */
    uint32_t        n_wins;
    uint64_t        wins_bases;
    const uint32_t* pairs;         /* [2*n_pairs] (read_idx, win_idx) per pair                  */
    uint64_t        n_pairs;       /* 0 is allowed: every result array is then empty            */
} sdp_batch;

/* Outputs, in caller pair order. Pointers are owned by the ctx and stay valid until the next
 * align call on it or sdp_destroy: DEVICE memory from sdp_align_batch, pinned HOST memory from
 * sdp_align_batch_host. */
typedef struct sdp_result {
    const int32_t*  score;        /* max_{1<=i<=m} M(i,n)                          */
    const int32_t*  ref_start;    /* first consumed window base (where the traceback stops)     */
    const int32_t*  ref_end;      /* (lowest maximising row i) - 1                               */
    const int32_t*  read_start;   /* 0 (first aligned read base in SDP_MODE_LOCAL)               */
    const int32_t*  read_end;     /* n-1 (last aligned read base in SDP_MODE_LOCAL)              */
    const uint8_t*  pass;         /* similarity filter, 1 = pass                                 */
    const int32_t*  n_match;      /* M columns whose two bases are equal and not N               */
    const int32_t*  n_cols;       /* alignment columns = M + I + D bases                         */
    const uint64_t* cigar_off;    /* exclusive scan of cigar_len in caller pair order            */
    const uint32_t* cigar_len;    /* runs of pair p                                              */
    const uint32_t* cigar_ops;    /* [n_cigar_ops] compacted runs                                */
    uint64_t        n_cigar_ops;
    uint64_t        n_pairs;
} sdp_result;

/* Per-call counters; times are CUDA-event milliseconds on the library's streams and are only
 * filled when timing was switched on with sdp_set_timing(ctx, 1). With more than one lane (sdp_set_chunks) the
 * per-stage times are summed over the lanes, whose stages overlap: only ms_total is wall time then. */
typedef struct sdp_stats {
    uint64_t n_pairs;
    uint64_t cells_forward;       /* sum n*m: the CUPS numerator                                 */
    uint64_t cells_reverse;       /* cells of the reverse pass                                   */
    uint64_t cells_traceback;     /* band cells of the traceback pass                            */
    uint64_t n_reverse_pairs;     /* pairs that took the reverse pass (a4)                       */
    uint32_t kernel_launches;     /* kernels of this library launched by the call                */
    uint32_t forward_launches;    /* launches of the forward score kernel                        */
    float ms_total;               /* whole call, first kernel to last                            */
    float ms_bucket;              /* a1 + a2 validate, histogram, scan, scatter, task build      */
    float ms_forward;             /* a3 forward score kernels                                    */
    float ms_reverse;             /* post-forward bookkeeping (gap bounds, bucket sorts, one host round trip) + a4 */
    float ms_traceback;           /* a5 + a6                                                     */
    float ms_compact;             /* a7 + a8                                                     */
    uint64_t cells_prefiltered;   /* sum n*m of the pairs the ungapped pre-pass settled (sdp_set_prefilter);
                                     cells_forward counts only the pairs that went through the DP   */
    uint64_t n_slow_words;        /* int32 scratch words of the pairs that took the int32 lane: 2*(n+1) per read over
                                     SDP_MAX_READ_LEN bases, 1 per shorter read (0 = no pair took that lane)        */
} sdp_stats;

/* Create a context on CUDA device `cuda_device`. SDP_EINVAL for bad scoring or null arguments,
 * SDP_ECUDA / SDP_ENOMEM otherwise; *out is written only on success. Not thread-safe: use one
 * ctx per thread; separate ctxs are independent. */
int sdp_create(const sdp_scoring* scoring, int cuda_device, sdp_ctx** out);
/* Test and tuning hook; results never depend on it (tests/test_gpu_parity.py routes the same pairs through every
 * traceback kernel and requires identical output). flags = OR of the SDP_ROUTE_* bits and SDP_ROUTE_FORCE_G(g):
 *   SDP_ROUTE_NO_THIN      pairs with gap bound W >= 1 go to the wide / generic traceback instead of the narrow-band kernels
 *   SDP_ROUTE_NO_WIDE      wide pairs go to the generic scalar band kernel instead of the wavefront traceback kernel
 *   SDP_ROUTE_ALWAYS_REVERSE  every wide pair takes the reverse pass (by default only those whose row bound exceeds about
 *                          twice the read length, where trimming the traceback rectangle pays for the pass)
 *   SDP_ROUTE_FORCE_G(g)   g threads per pair group for every read length that admits it (geometry experiments), 0 = off
 * 0 restores the default routing. SDP_EINVAL for unknown bits. */
#define SDP_ROUTE_NO_THIN 1u
#define SDP_ROUTE_NO_WIDE 2u
#define SDP_ROUTE_ALWAYS_REVERSE 4u
#define SDP_ROUTE_FORCE_G(g) (((uint32_t)(g) & 0x3Fu) << 8)
int sdp_set_debug_route(sdp_ctx* ctx, uint32_t flags);

/* Align every pair of `batch` (DEVICE pointers). The call is ordered after everything already enqueued on
 * `cuda_stream` (a cudaStream_t; NULL = default stream), runs on the ctx's own streams, and returns after all of it
 * has completed (the host needs sizes from the device between stages, and n_cigar_ops at the end), so errors are
 * synchronous and the results are visible to any stream afterwards.
 * On error `out` is untouched. A CIGAR is produced for every pair, passing the filter or not. */
int sdp_align_batch(sdp_ctx* ctx, const sdp_batch* batch, void* cuda_stream, sdp_result* out);

/* Tuning hook; results never depend on it. A call splits its pair list into `chunks` contiguous ranges ("lanes") that
 * run the path one after the other through the forward score kernel, while everything a lane does after its forward
 * pass (bookkeeping, reverse pass, traceback) runs on higher-priority streams under the next lane's forward kernel.
 * 0 (default) = the library's choice, which is 1 (no pipelining: on B200 the overlap costs the forward kernel more than
 * it hides); at most 8. SDP_EINVAL outside 0..8. */
int sdp_set_chunks(sdp_ctx* ctx, int chunks);

/* Same operation with HOST pointers in `batch`: copies the inputs into device buffers owned by the ctx
 * (cudaMemcpyAsync on internal streams, straight from the caller's arrays: pass page-locked memory for full PCIe
 * speed; pageable memory is accepted, the driver then stages the copies and they run synchronously), runs
 * sdp_align_batch's pipeline, and copies every result array back into pinned memory; `out` then holds pinned HOST
 * pointers owned by the ctx, valid until the next call on this ctx. The offsets, lengths and the pair list go first,
 * so that validation and bucketing run while the sequences are still uploading; score and ref_end are downloaded as
 * soon as the forward pass is done. To hide the remaining copies, drive two contexts from two host threads. */
int sdp_align_batch_host(sdp_ctx* ctx, const sdp_batch* batch, sdp_result* out);

/*
 * Step-3 shape ("enumerates candidate regions to be aligned to the whole read using dynamic
 * programming"; up to a ceiling of candidate regions per read): after sdp_align_batch
 * has aligned a pair list in which a read appears with several candidate windows, pick per read the best
 * candidate. The paper does not say how the winner is chosen; the rule here (R16):
 * highest score; among equal scores the lowest window index; among equal windows the lowest pair index.
 * DEVICE pointers owned by the ctx, one entry per read of the batch, valid until the next call on the ctx.
 */
typedef struct sdp_read_best {
    const uint32_t* best_pair;      /* index into the pair list, SDP_NO_PAIR if the read is in no pair      */
    const int32_t*  best_score;     /* score of best_pair (undefined when SDP_NO_PAIR)                      */
    const int32_t*  second_score;   /* best score among the read's OTHER pairs, INT32_MIN if it has none    */
    const uint32_t* n_candidates;   /* pairs of the batch that name the read                                */
    uint32_t        n_reads;
} sdp_read_best;
#define SDP_NO_PAIR 0xFFFFFFFFu

/* `batch` (DEVICE pointers) and `result` must be the arguments / output of the last successful
 * sdp_align_batch on this ctx (sdp_align_batch_host results are host pointers: not accepted). Enqueued on
 * `cuda_stream`, returns after completion. SDP_EINVAL for null arguments or a result of another batch. */
int sdp_best_per_read(sdp_ctx* ctx, const sdp_batch* batch, const sdp_result* result, void* cuda_stream,
                      sdp_read_best* out);

/*
 * The same per-read choice (same rule, same four outputs, bit for bit) for callers that must not allocate device
 * memory: programs that gave the whole card to their own pool at start-up (a later cudaMalloc may fail or fragment
 * it), and programs with several busy streams, which cudaMalloc / cudaFree would stall device-wide. It takes no
 * sdp_ctx (sdp_create allocates) and calls no cudaMalloc, cudaFree or allocating library routine. `pairs` [2*n_pairs]
 * and `score` [n_pairs] are DEVICE inputs (for instance sdp_batch.pairs and sdp_result.score of an earlier
 * sdp_align_batch); best_pair, best_score, second_score and n_candidates are caller-owned DEVICE arrays of n_reads
 * entries, filled as sdp_read_best describes. A pair whose read index is >= n_reads is ignored.
 *
 * The method's working memory, one 64-bit key per read, is a fixed array inside the library:
 * SDP_STATIC_MAX_READS * 8 bytes = 8 MiB, held by every GPU that loads libsdp.so until the process exits. That array
 * is the limit: n_reads > SDP_STATIC_MAX_READS returns SDP_ERANGE and does nothing (split the batch by read, or use
 * sdp_best_per_read). Every call on a device uses the same array and clears the part it needs first, so calls run
 * one after another in any mix of sizes; two calls that can overlap on one GPU (different streams with no ordering
 * between them, or two host threads) race on it and give garbage: order them yourself.
 *
 * The work is enqueued on `cuda_stream` (NULL = default stream) of device `cuda_device` and the call returns without
 * waiting; the outputs are complete when the stream reaches that point. The first call on each device also looks up
 * the array's device address (cudaGetSymbolAddress, which loads the library's device code there if nothing has yet):
 * make that first call during start-up, before any stream capture begins. The caller's current device is restored.
 * Returns SDP_OK, SDP_EINVAL (null array, device outside 0..63), SDP_ERANGE (n_reads as above, or n_pairs beyond
 * 32 bits), SDP_ECUDA. sdp_static_last_error() gives the message of the calling thread's last failure ("" if none).
 */
#define SDP_STATIC_MAX_READS (1u << 20)
int sdp_best_per_read_static(int cuda_device, const uint32_t* pairs, const int32_t* score, uint64_t n_pairs,
                             uint32_t n_reads, void* cuda_stream, uint32_t* best_pair, int32_t* best_score,
                             int32_t* second_score, uint32_t* n_candidates);
const char* sdp_static_last_error(void);

/*
 * Alignment mode. SDP_MODE_SEMIGLOBAL (default) is the paper's formulation: the whole read against any sub-region of
 * the window. SDP_MODE_LOCAL is the soft-clipping variant (the paper names
 * Smith-Waterman, and soft-clipped alignments; R18): M(i,0) = M(0,j) = 0,
 * M(i,j) = max(0, ...), score = max over all cells (lowest row, then lowest column), the walk stops at the first cell
 * with M = 0. Then read_start / read_end are the first / last aligned read base, unaligned read ends appear in the
 * CIGAR as soft clips (BAM op 4), n_cols counts aligned columns only, and the filter counts clipped bases as columns
 * that do not match: pass iff n_cols > 0 and n_match * 1e6 >= q * (n_cols + clipped). A pair without any positive-
 * scoring alignment reports score 0, ref_start 0, ref_end -1, read_start 0, read_end -1, CIGAR <n>S, pass 0.
 * Local mode has its own forward kernels (an int16x2 one for reads up to 256 bases, the int32 lane beyond) and the generic
 * traceback: exact, about one fifth of the default mode's throughput on 100-base reads.
 * SDP_EINVAL for an unknown mode.
 */
#define SDP_MODE_SEMIGLOBAL 0
#define SDP_MODE_LOCAL 1
int sdp_set_mode(sdp_ctx* ctx, int mode);

/* Candidate screening for the step-3 shape: with score-only on (1), sdp_align_batch / sdp_align_batch_host stop
 * after the forward score pass (a1-a3): `score` and `ref_end` are as always, `ref_start` and `read_end` are -1,
 * `read_start`, `n_match`, `n_cols`, `pass`, `cigar_len`, `cigar_off` are 0 and n_cigar_ops is 0. A caller scores every
 * candidate this way, picks winners with sdp_best_per_read and aligns only those with score-only off (0, default). */
int sdp_set_score_only(sdp_ctx* ctx, int enabled);

/* Optional ungapped pre-pass (off by default; the analogue of the paper's step 1, inside one window).
 * A gapped alignment scores at most n*match - (gap_open + gap_extend). With the pre-pass on (1), a pair whose best
 * gap-free placement in the window has x mismatches with x*(match - mismatch) < gap_open + gap_extend gets its score and
 * lowest ref_end from a word-parallel Hamming scan and skips the forward DP; every other pair, and every later stage,
 * is unchanged, and so is every output (tests/test_gpu_parity.py::test_prefilter_changes_nothing). */
int sdp_set_prefilter(sdp_ctx* ctx, int enabled);

/*
 * Mate-rescue wrapper (step 2: "a candidate region flanking the mapped end is aligned to the unmapped
 * end"; expected minimum and maximum fragment lengths -v / -u and the orientation of the ends).
 * The paper does not say how the region follows from the bounds; reading taken (R17), forward-reverse
 * orientation: a fragment is the reference interval [f, f + ins) with min_insert <= ins <= max_insert, its forward-strand
 * end starts at f and its reverse-strand end stops at f + ins.
 *   mate on the forward strand at [p, p + L):  the other end lies in  [p + min_insert - n, p + max_insert)
 *   mate on the reverse strand at [p, p + L):  the other end lies in  [p + L - max_insert, p + L - min_insert + n)
 * clipped to [0, ref_bases); n = length of the unmapped read. win_len is 0 when nothing is left; sdp_align_batch rejects
 * empty windows, so such a rescue must stay out of the pair list: sdp_mate_pairs builds that list. All pointers are DEVICE
 * pointers; outputs are caller-owned.
 */
typedef struct sdp_mates {
    const uint64_t* mate_pos;      /* leftmost reference base of the mapped end                 */
    const uint32_t* mate_len;      /* reference bases the mapped end covers                      */
    const uint8_t*  mate_reverse;  /* 0 = mapped end on the forward strand, 1 = reverse          */
    const uint32_t* read_len;      /* length n of the unmapped end                               */
    uint64_t        n;             /* number of rescues                                          */
} sdp_mates;
int sdp_mate_windows(sdp_ctx* ctx, const sdp_mates* mates, uint32_t min_insert, uint32_t max_insert, uint64_t ref_bases,
                     void* cuda_stream, uint64_t* win_off, uint32_t* win_len);
/* Pair list of a rescue batch in which read k and window k belong to rescue k: the rescues with win_len[k] > 0, in rescue
 * order, as pairs (k, k). pairs receives 2 * (*n_pairs) entries (capacity 2 * n), pair_of_rescue[k] the index of rescue k
 * in that list or SDP_NO_PAIR when its window is empty; *n_pairs is a HOST pointer. The other pointers are DEVICE memory. */
int sdp_mate_pairs(sdp_ctx* ctx, const uint32_t* win_len, uint64_t n, void* cuda_stream, uint32_t* pairs,
                   uint32_t* pair_of_rescue, uint64_t* n_pairs);
/* After aligning the rescue batch: proper[k] = 1 iff rescue k was aligned (win_len[k] > 0 and, when pair_of_rescue is given,
 * pair_of_rescue[k] != SDP_NO_PAIR), passed the similarity filter, and the implied fragment length is within the bounds:
 * mate forward: (win_off + ref_end + 1) - p;  mate reverse: (p + L) - (win_off + ref_start). `ref_start`, `ref_end`,
 * `pass` are the arrays of the sdp_result of that alignment (device pointers), read at index pair_of_rescue[k]; a NULL
 * pair_of_rescue means pair k = rescue k (only valid when no window is empty). */
int sdp_proper_pairs(sdp_ctx* ctx, const sdp_mates* mates, uint32_t min_insert, uint32_t max_insert, const uint64_t* win_off,
                     const uint32_t* win_len, const uint32_t* pair_of_rescue, const int32_t* ref_start, const int32_t* ref_end,
                     const uint8_t* pass, void* cuda_stream, uint8_t* proper);

/* Counters of the last align call on this ctx. */
int sdp_get_stats(const sdp_ctx* ctx, sdp_stats* out);

/* Switch per-stage CUDA-event timing on (1) or off (0, the default). */
int sdp_set_timing(sdp_ctx* ctx, int enabled);

/* Message of the last error on this ctx ("" if none). Never NULL; valid until the next call. */
const char* sdp_last_error(const sdp_ctx* ctx);

/* Release everything the ctx owns. NULL is ignored. */
void sdp_destroy(sdp_ctx* ctx);

/*
 * Roofline helper: runs an issue-rate microbenchmark of the int16x2
 * DPX instructions the score kernel is built from (VIADDMNMX.S16x2 / VIMNMX3.S16x2, 50:50,
 * 8 independent chains per thread, full occupancy) on `cuda_device` and reports
 * thread-instructions per clock per SM (thread-instructions per second per SM from the CUDA-event
 * time of the launches, divided by the device's maximum SM clock), the SM count and that clock in MHz.
 */
int sdp_measure_dpx_rate(int cuda_device, double* instr_per_clk_per_sm, int32_t* sm_count, double* sm_mhz);

/* Library version, e.g. "sdp 0.1 (sm_100a)". */
const char* sdp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SDP_H_ */
