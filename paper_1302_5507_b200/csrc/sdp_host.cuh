// sdp_host.cuh -- host-side declarations shared by the translation units of libsdp.
#pragma once
#include "../../include/sdp.h"
#include "sdp_internal.cuh"

namespace sdp {

struct Scoring {
    int32_t match, mismatch, gap_open, gap_extend;
    long long min_sim_q;            // llround(min_similarity * 1e6)
};

// ---- bucket.cu
void launch_validate_key(const sdp_batch& b, const Scoring& sc, uint32_t* keys, uint32_t* pn, uint32_t* pm,
                         uint32_t* hist, uint32_t* err_flag, unsigned long long* cells, int prefilter, int32_t* score,
                         int32_t* ref_end, unsigned long long* cells_skipped, int local, uint32_t* slow_words,
                         unsigned long long* slow_total, cudaStream_t st);
// scan bins, scatter into `order` (or, with b_desc != nullptr, write the forward descriptors of *b_desc straight into
// `desc` in bucket order), and (if slots != nullptr) build the per-read-length task table
void launch_sort_tail(const uint32_t* keys, uint64_t n, uint32_t* hist, uint32_t* bin_start, uint32_t* order,
                      const uint16_t* slot_n, const uint16_t* slot_G, const uint16_t* slot_K,
                      SlotInfo* slots, uint32_t* task_prefix, uint32_t* host_prefix, uint32_t* host_total, cudaStream_t st,
                      const sdp_batch* b_desc = nullptr, PairDesc* desc = nullptr);
void launch_mailbox(const uint32_t* tb_bin_start, uint32_t stride, uint32_t nbounds, const uint64_t* totals,
                    const unsigned long long* counters, uint32_t* host_bounds, uint64_t* host_totals,
                    unsigned long long* host_counters, cudaStream_t st);
// exclusive scan of n 32-bit values into 64-bit offsets starting at *base_dev (0 when null); *total_dev = base + sum
void exclusive_scan_u32_u64(const uint32_t* in, uint64_t n, uint64_t* out, uint64_t* total_dev, const uint64_t* base_dev,
                            uint32_t* tmp_local, uint32_t* tmp_tiles, uint64_t* tmp_tile_base,
                            cudaStream_t st, uint32_t* launches);

// ---- score_modules.cu: the score kernels, loaded per context with the scoring patched into their immediates
constexpr int SDP_SCORE_UNITS_N = 16;     // cubins, two column counts each (K = 2r+1, 2r+2)
constexpr int SDP_N_SENTINELS = 9;
struct ScorePatch {                                            // packed int16x2 values
    uint32_t negOc, negO, c2, Cd, e2;                          // score kernels, see score_kernel.cuh
    uint32_t t_negOf, t_negOe, t_c8, t_Cd8;                    // traceback DP kernels, see trace_kernel.cuh
};
struct ScoreModules {
    cudaLibrary_t lib[SDP_SCORE_UNITS_N];
    unsigned char loaded[SDP_SCORE_UNITS_N];
    cudaKernel_t kern[SDP_MAX_K + 1][2][2];                     // [K][reverse][padded]
    cudaKernel_t kern_trace[SDP_MAX_K + 1][2];                  // [K][padded]
};
void score_modules_init(ScoreModules* m);
void score_modules_destroy(ScoreModules* m);
bool patch_score_image(unsigned char* img, size_t len, const ScorePatch& pv, uint32_t hits[SDP_N_SENTINELS]);
// td == nullptr: the score kernel (forward, or reverse with rev); else the traceback DP kernel
int score_modules_launch(ScoreModules* m, const ScorePatch& pv, int K, bool pad, bool rev, const ScoreParams& p,
                         const TraceDP* td, cudaStream_t st, char* err, size_t errlen);

// ---- traceback.cu
struct PostParams {
    sdp_batch b;                 // sequences, for the ungapped shortcut
    uint64_t n_pairs;
    Scoring sc;
    const uint32_t* pn; const uint32_t* pm;      // per pair read / window length
    const int32_t* score; const int32_t* ref_end;
    int32_t* tbW;                // gap-content bound W per pair
    int32_t* tb_rows;            // rows the traceback may need: min(i_end, n + W), 0 when W == 0
    uint32_t* keys_wide;         // bucket key of the reverse pass and the traceback DP kernel (wide pairs only, else SKIP)
    uint32_t* keys_tb;           // bucket key of the one-thread-per-pair traceback (everything else)
    int wide_ok;                 // scoring fits the x8 tagged domain of trace_kernel.cuh
    int no_thin;                 // debugging: keep W >= 1 pairs off the narrow-band kernel
    int thin_ok;                 // scoring fits the x8 tagged int16 domain of thin_kernel.cu
    int local;                   // SDP_MODE_LOCAL
    const uint32_t* slow_words;  // != 0: the pair went through the int32 lane
    const int32_t* end_col;      // local: read column of the end cell
    uint32_t* err_flag;
    uint32_t* bits_words;        // direction-bit words the pair needs
    uint32_t* ops_cap;           // CIGAR run capacity the pair needs (2W + 1)
    uint32_t* hist_tb; uint32_t* hist_wide;
    unsigned long long* counters;   // [0] reverse cells, [1] traceback cells, [2] reverse pairs
};
void launch_post_forward(const PostParams& pp, cudaStream_t st);
// ratio10: the pair takes the reverse pass when its row bound exceeds ratio10 / 10 read lengths (0 = always)
void launch_fill_desc_rev(const sdp_batch& b, const uint32_t* order, uint32_t count, const int32_t* score,
                          const int32_t* ref_end, const int32_t* tbW, int ratio10, int32_t* rev_rows,
                          unsigned long long* counters, PairDesc* desc, cudaStream_t st);

struct TraceParams {
    sdp_batch b;
    Scoring sc;
    const uint32_t* order;       // traceback bucket order
    uint32_t first, count;       // range of `order` this launch covers
    const int32_t* score; const int32_t* ref_end; const int32_t* tbW; const int32_t* rev_rows;
    const int32_t* end_col;      // local variant: read column of the end cell
    const uint64_t* bits_off; uint32_t* bits;     // direction bits scratch
    const uint64_t* ops_off;  uint32_t* ops_rev;  // per-pair runs, end -> start order
    int32_t* ref_start; int32_t* read_start; int32_t* read_end; uint8_t* pass;
    int32_t* n_match; int32_t* n_cols; uint32_t* cigar_len;
    uint32_t* err_flag;
};
void launch_wide_regions(const uint32_t* order, uint32_t max_count, const uint32_t* count_dev, const uint32_t* pn,
                         const int32_t* tb_rows, const uint16_t* slot_of_n, const SlotInfo* slots, uint32_t* words,
                         cudaStream_t st);
void launch_fill_desc_tb(const sdp_batch& b, const uint32_t* order, uint32_t count, const int32_t* score,
                         const int32_t* ref_end, const int32_t* rev_rows, PairDesc* desc, cudaStream_t st);
struct WalkParams {
    sdp_batch b;
    Scoring sc;
    const PairDesc* desc; uint32_t count;         // traceback-DP descriptors (wide order)
    const SlotInfo* slots; const uint16_t* slot_of_n;
    const uint32_t* bits; const uint64_t* bits_off;
    const int32_t* ref_end; const int32_t* tbW;
    const uint64_t* ops_off; uint32_t* ops_rev;
    int32_t* ref_start; int32_t* read_start; int32_t* read_end; uint8_t* pass;
    int32_t* n_match; int32_t* n_cols; uint32_t* cigar_len;
    uint32_t* err_flag;
};
void launch_walk(const WalkParams& wp, cudaStream_t st);
// band-width classes of the traceback kernel (local-memory row arrays)
constexpr int TB_NCLASS = 5;               // row arrays of 16 / 64 / 256 / 1032 entries in local memory; the last class keeps
                                           // them in global scratch (any width: the int32 lane and the local variant)
void launch_traceback(int cls, bool local, const TraceParams& tp, cudaStream_t st);

// ---- slow_lane.cu: int32 forward pass, one thread per pair (pairs with slow_words[p] != 0)
void launch_forward_i32(const sdp_batch& b, const Scoring& sc, int local, const uint32_t* slow_words, const uint64_t* slow_off,
                        int32_t* rows, int32_t* score, int32_t* ref_end, int32_t* end_col, cudaStream_t st);
// narrow bands (thin_kernel.cu): gap bound W in 0..THIN_NW-1, band rows <= THIN_MAXROWS
constexpr int THIN_NW = 24;
constexpr int THIN_SPLIT = 8;             // classes [0, SPLIT), [SPLIT, SPLIT2), [SPLIT2, NW) run in three launches
constexpr int THIN_SPLIT2 = 16;           // (register budgets differ)
constexpr uint32_t TB_KEY_STRIDE = 2048;  // traceback bucket key = class * TB_KEY_STRIDE + rows (rows, n < 2048)
constexpr int THIN_MAXROWS = 336;
int launch_thin_all(const uint32_t* bounds, const TraceParams& tp, cudaStream_t st, cudaStream_t st_mid, cudaStream_t st_hi);   // returns kernels launched
void launch_compact(uint64_t n_pairs, const uint64_t* ops_off, const uint32_t* ops_rev, const uint32_t* cigar_len,
                    const uint64_t* cigar_off, uint32_t* cigar_ops, cudaStream_t st);

// ---- best_read.cu
void launch_best_per_read(uint64_t n_pairs, uint32_t n_reads, const uint32_t* pairs, const int32_t* score,
                          unsigned long long* key, uint32_t* best_pair, int32_t* best_score, int32_t* second,
                          uint32_t* ncand, cudaStream_t st);

// ---- mate.cu
void launch_mate_windows(const sdp_mates& mt, uint32_t min_ins, uint32_t max_ins, uint64_t ref_bases, uint64_t* win_off,
                         uint32_t* win_len, cudaStream_t st);
void launch_proper_pairs(const sdp_mates& mt, uint32_t min_ins, uint32_t max_ins, const uint64_t* win_off,
                         const uint32_t* win_len, const uint32_t* pair_of_rescue, const int32_t* ref_start,
                         const int32_t* ref_end, const uint8_t* pass, uint8_t* proper, cudaStream_t st);
void launch_mate_flags(const uint32_t* win_len, uint64_t n, uint32_t* flag, cudaStream_t st);
void launch_mate_pairs(const uint32_t* flag, const uint64_t* off, uint64_t n, uint32_t* pairs, uint32_t* pair_of_rescue,
                       cudaStream_t st);

// ---- microbench.cu
int measure_dpx_rate(int device, double* rate, int32_t* sms, double* mhz);

}  // namespace sdp
