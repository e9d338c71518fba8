// sdp_api.cu -- the C ABI of include/sdp.h: context, stage orchestration, host-buffer entry.
// Stage order per call:
//   a1 validate + key -> a2 bucket (hist, scan, scatter, task table) -> a3 forward score kernels
//   -> W, keys -> bucket (reverse), bucket (traceback) -> a4 reverse kernels -> a5/a6 traceback
//   -> a7 scan + compaction. a8 (un-permute) is implicit: every kernel writes its per-pair
//   results at the caller's pair index.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "sdp_host.cuh"

using namespace sdp;

namespace {

struct DevBuf {
    void* p = nullptr; size_t cap = 0;
    template <class T> T* as() const { return (T*)p; }
};

struct Mailbox {                    // pinned host memory the device results land in
    uint32_t task_prefix[3][SDP_NSLOTS + 1];   // forward, (unused), traceback DP + reverse pass
    uint32_t bin_total[4];                     // forward, (unused), thin traceback, wide traceback
    uint32_t tb_bounds[THIN_NW + TB_NCLASS + 1];   // narrow-band launches (one per W), then the generic band classes
    uint32_t err_flag;
    uint64_t totals[4];             // [0] thin direction-bit words, [1] run capacity, [2] CIGAR runs, [3] wide nibble words
    uint64_t slow_total;            // words of int32 row arrays the slow lane needs
    unsigned long long counters[8]; // [0] reverse cells [1] traceback cells [2] reverse pairs [3] forward cells
                                    // [4] cells of pairs the ungapped pre-pass settled
};

constexpr int SDP_FAN_STREAMS = 4;
constexpr int SDP_MAX_LANES = 8;

enum { LEV_A0, LEV_A1, LEV_F0, LEV_F1, LEV_REV, LEV_TRACE, LEV_END, LEV_COUNT };

// One chunk of a call's pair list (a "lane"): a contiguous range of caller pairs that runs the whole path a1..a7 with
// its own scratch. Lanes are software-pipelined (sdp_align_batch): all forward kernels go back to back on one
// low-priority stream, and everything a lane does after its forward pass -- latency-bound bookkeeping, two host
// round trips, the reverse pass and the traceback kernels -- runs on higher-priority streams UNDER the next lane's
// forward kernel instead of after it.
struct Lane {
    Mailbox* mb = nullptr;
    cudaStream_t st = nullptr;       // this lane's stream (high priority): everything but the forward kernels
    cudaEvent_t evA = nullptr, evB = nullptr, evC = nullptr, evD = nullptr;   // end of the four phases
    cudaEvent_t ev_desc = nullptr, ev_fwd = nullptr;
    cudaEvent_t fan_fork = nullptr, fan_join[SDP_FAN_STREAMS] = {};
    cudaEvent_t side_done[3] = {};
    cudaEvent_t tev[LEV_COUNT] = {};
    // what every call starts from zero sits in ONE block (one memset): counters, err_flag, the three histograms
    void* zero_block = nullptr; size_t zero_bytes = 0;
    uint32_t* hist[4] = {};          // forward, (unused), thin traceback, wide traceback + reverse pass
    uint32_t* bin_start[4] = {};
    SlotInfo* slots[3] = {};         // forward, (unused), wide traceback + reverse pass
    uint32_t* task_prefix[3] = {};
    uint32_t* err_flag = nullptr;
    unsigned long long* counters = nullptr;
    uint64_t* totals = nullptr;
    // per-pair device buffers (grow only), indexed by the pair's position inside the lane
    DevBuf keys, pn, pm, order, desc, desc_rev, order_tb, keys_tb, tbW, rev_rows,
        tb_rows, keys_wide, order_wide, desc_wide, wide_words, wide_off, wide_bits,
        bits_words, ops_cap, bits_off, ops_off, bits, ops_rev;
    DevBuf scan_local[3], scan_tiles[3], scan_tile_base[3];   // one set per concurrent scan
    DevBuf slow_words, slow_off, slow_rows;   // int32 lane (slow_lane.cu): per-pair row-array words, their offsets, the arrays
    // this call
    uint64_t p0 = 0, P = 0;          // caller pair range [p0, p0 + P)
    sdp_batch b{};                   // the caller's batch restricted to that range
    uint32_t nl = 0, fwd_launches = 0;
    uint32_t n_wide = 0;
};

}  // namespace

struct sdp_ctx {
    int device = 0;
    sdp_scoring user_sc{};
    Scoring sc{};
    ScoreConsts consts{};
    TraceConsts tconsts{};
    ScorePatch patch{};              // the scoring as the score kernels' immediates (score_modules.cu)
    ScoreModules modules;            // score kernels loaded so far, patched with `patch`
    int wide_ok = 0;                 // scoring fits the x8 tagged domain of the traceback DP kernel
    int wide_fits = 0;               // wide_ok before sdp_set_debug_route masked it
    int no_thin = 0;                 // sdp_set_debug_route: keep W >= 1 pairs off the narrow-band kernel
    int thin_ok = 0;                 // scoring fits the x8 tagged int16 domain of thin_kernel.cu
    int force_rev = 0;               // sdp_set_debug_route: the reverse pass for every wide pair, not only where it pays
    uint32_t resident_warps = 1776;  // SMs x warps of the score kernels resident per SM (12 at 168 registers)
    char err[512] = {0};
    bool timing = false;
    bool prefilter = false;          // sdp_set_prefilter: ungapped pre-pass before the forward DP
    bool score_only = false;         // sdp_set_score_only: stop after the forward pass
    int mode = SDP_MODE_SEMIGLOBAL;  // sdp_set_mode
    int chunks = 0;                  // sdp_set_chunks: lanes per call, 0 = chosen from the pair count
    sdp_stats stats{};
    uint16_t h_slot_n[SDP_NSLOTS], h_slot_G[SDP_NSLOTS], h_slot_K[SDP_NSLOTS];
    uint32_t cls_begin[2 * SDP_MAX_K + 3];   // first slot of class c = 2K + padded; [c+1] ends it
    uint16_t h_slot_of_n[SDP_NSLOTS];        // read length - 1 -> slot
    uint16_t *d_slot_n = nullptr, *d_slot_G = nullptr, *d_slot_K = nullptr, *d_slot_of_n = nullptr;
    int prio_lo = 0, prio_hi = 0;
    Lane lane[SDP_MAX_LANES];
    int lanes_ready = 0;                  // lanes whose streams, events and fixed-size buffers exist
    cudaStream_t own_stream = nullptr;    // sdp_align_batch_host
    cudaStream_t copy_stream = nullptr;   // sdp_align_batch_host: sequence upload beside the bucket stage, early result download
    cudaEvent_t ev_seq_ready = nullptr;   // ... the sequences have arrived
    bool wait_seq = false;                // this call's forward pass (and pre-pass) must wait for ev_seq_ready
    int32_t* h_early_score = nullptr;     // host arrays score / ref_end go to as soon as a lane's forward pass is done
    int32_t* h_early_ref_end = nullptr;
    cudaStream_t fwd_stream = nullptr;    // every lane's forward score kernels, lowest priority
    cudaStream_t fan_fwd[SDP_FAN_STREAMS] = {};    // [0] unused; forward / reverse / trace launches of several K classes
    cudaStream_t fan_post[SDP_FAN_STREAMS] = {};   // [0] unused; the short sort and scan chains after the forward pass
    cudaStream_t side_stream[3] = {};     // narrow-band traceback (three register classes), beside the wide path
    cudaEvent_t ev_start = nullptr, ev_end = nullptr, ev_cig[SDP_MAX_LANES] = {};
    uint64_t* cig_total = nullptr;        // [SDP_MAX_LANES + 1] running CIGAR run totals across lanes; [0] = 0
    // results, caller pair order, shared by the lanes
    DevBuf score, ref_start, ref_end, read_start, read_end, pass, n_match, n_cols, cigar_off, cigar_len, cigar_ops;
    // sdp_align_batch_host: device copies of the inputs and pinned host copies of the outputs
    DevBuf in_reads, in_read_off, in_read_len, in_read_nmask, in_wins, in_win_off, in_win_len, in_win_nmask, in_pairs;
    DevBuf h_out, h_ops;             // pinned: the per-pair result arrays (one slab, carved per call) and the CIGAR runs
    // sdp_best_per_read
    DevBuf rb_key, rb_pair, rb_score, rb_second, rb_ncand;
    DevBuf mp_flag, mp_off;          // sdp_mate_pairs
    const uint32_t* last_pairs = nullptr;   // pair list of the last successful align call (to match results to it)
    uint64_t last_n_pairs = 0;
    uint32_t last_n_reads = 0;
};

namespace {

int fail(sdp_ctx* c, int code, const char* fmt, ...) {
    if (c) {
        va_list ap; va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

#define CU(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(ctx, e_ == cudaErrorMemoryAllocation ? SDP_ENOMEM : SDP_ECUDA,        \
                        "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__); \
    } while (0)

int ensure(sdp_ctx* ctx, DevBuf& b, size_t bytes) {
    if (bytes <= b.cap) return SDP_OK;
    if (b.p) { cudaFree(b.p); b.p = nullptr; b.cap = 0; }
    size_t want = bytes + bytes / 8 + 256;
    CU(cudaMalloc(&b.p, want));
    b.cap = want;
    return SDP_OK;
}

int ensure_pinned(sdp_ctx* ctx, DevBuf& b, size_t bytes) {
    if (bytes <= b.cap) return SDP_OK;
    if (b.p) { cudaFreeHost(b.p); b.p = nullptr; b.cap = 0; }
    size_t want = bytes + bytes / 8 + 256;
    CU(cudaMallocHost(&b.p, want));
    b.cap = want;
    return SDP_OK;
}

#define EN(buf, bytes)                                         \
    do {                                                       \
        int rc_ = ensure(ctx, ctx->buf, (size_t)(bytes));      \
        if (rc_ != SDP_OK) return rc_;                         \
    } while (0)
#define LEN(buf, bytes)                                        \
    do {                                                       \
        int rc_ = ensure(ctx, L.buf, (size_t)(bytes));         \
        if (rc_ != SDP_OK) return rc_;                         \
    } while (0)

// streams, events and fixed-size buffers of lanes [ctx->lanes_ready, want)
int lanes_init(sdp_ctx* ctx, int want)
{
    for (int li = ctx->lanes_ready; li < want; ++li) {
        Lane& L = ctx->lane[li];
        CU(cudaMallocHost(&L.mb, sizeof(Mailbox)));
        memset(L.mb, 0, sizeof(Mailbox));
        CU(cudaStreamCreateWithPriority(&L.st, cudaStreamNonBlocking, ctx->prio_hi));
        cudaEvent_t* evs[] = {&L.evA, &L.evB, &L.evC, &L.evD, &L.ev_desc, &L.ev_fwd, &L.fan_fork, &L.side_done[0],
                              &L.side_done[1], &L.side_done[2]};
        for (cudaEvent_t* e : evs) CU(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
        for (int k = 1; k < SDP_FAN_STREAMS; ++k) CU(cudaEventCreateWithFlags(&L.fan_join[k], cudaEventDisableTiming));
        for (int k = 0; k < LEV_COUNT; ++k) CU(cudaEventCreate(&L.tev[k]));
        {
            const size_t hist_words = ((SDP_NBINS + 1 + 3) / 4) * 4;
            L.zero_bytes = 8 * 8 + 16 + 3 * hist_words * 4;
            CU(cudaMalloc(&L.zero_block, L.zero_bytes));
            char* z = (char*)L.zero_block;
            L.counters = (unsigned long long*)z;
            L.err_flag = (uint32_t*)(z + 64);
            uint32_t* h = (uint32_t*)(z + 80);
            L.hist[0] = h; L.hist[2] = h + hist_words; L.hist[3] = h + 2 * hist_words;
        }
        for (int i = 0; i < 4; ++i) {
            if (i == 1) continue;
            CU(cudaMalloc(&L.bin_start[i], (SDP_NBINS + 4 + SDP_BIN_SCRATCH) * 4));
        }
        for (int i = 0; i < 3; ++i) {
            if (i == 1) continue;
            CU(cudaMalloc(&L.slots[i], SDP_NSLOTS * sizeof(SlotInfo)));
            CU(cudaMalloc(&L.task_prefix[i], (SDP_NSLOTS + 1) * 4));
        }
        CU(cudaMalloc(&L.totals, 4 * 8));
        ctx->lanes_ready = li + 1;
    }
    return SDP_OK;
}

void lane_destroy(Lane& L)
{
    DevBuf* bufs[] = {&L.keys, &L.pn, &L.pm, &L.order, &L.desc, &L.desc_rev, &L.order_tb, &L.keys_tb, &L.tbW, &L.rev_rows,
                      &L.tb_rows, &L.keys_wide, &L.order_wide, &L.desc_wide, &L.wide_words, &L.wide_off, &L.wide_bits,
                      &L.bits_words, &L.ops_cap, &L.bits_off, &L.ops_off, &L.bits, &L.ops_rev, &L.scan_local[0],
                      &L.scan_local[1], &L.scan_local[2], &L.scan_tiles[0], &L.scan_tiles[1], &L.scan_tiles[2],
                      &L.scan_tile_base[0], &L.scan_tile_base[1], &L.scan_tile_base[2], &L.slow_words, &L.slow_off,
                      &L.slow_rows};
    for (DevBuf* b : bufs) if (b->p) cudaFree(b->p);
    for (int i = 0; i < 4; ++i) cudaFree(L.bin_start[i]);
    for (int i = 0; i < 3; ++i) { cudaFree(L.slots[i]); cudaFree(L.task_prefix[i]); }
    cudaFree(L.zero_block); cudaFree(L.totals);
    if (L.mb) cudaFreeHost(L.mb);
    if (L.st) cudaStreamDestroy(L.st);
    cudaEvent_t evs[] = {L.evA, L.evB, L.evC, L.evD, L.ev_desc, L.ev_fwd, L.fan_fork, L.side_done[0], L.side_done[1],
                         L.side_done[2]};
    for (cudaEvent_t e : evs) if (e) cudaEventDestroy(e);
    for (int k = 1; k < SDP_FAN_STREAMS; ++k) if (L.fan_join[k]) cudaEventDestroy(L.fan_join[k]);
    for (int k = 0; k < LEV_COUNT; ++k) if (L.tev[k]) cudaEventDestroy(L.tev[k]);
}

// (G, K) per read length: G threads share the read, K = ceil(n / G) columns each. A warp runs 2*floor(32/G) pairs
// for (m + G - 1) steps, and a step costs what the (K, padded) kernel variant was MEASURED to cost on B200
// (200,000 pairs, m = n + 300, G = 4; relative units; re-measured in round 2 for the two-row-skew, immediate-operand
// kernel, whose cost is close to 0.24 + 0.103 K: the per-K irregularities of the round-1 kernel are gone).
// A table, not a formula, so that it can follow ptxas's register allocation per K; DESIGN.md "Score kernel".
static const double kStepCostExact[SDP_MAX_K] = {3.49, 4.5, 5.37, 6.48, 7.47, 8.4, 9.46, 10.54, 11.39, 12.37, 13.52, 14.63, 15.56, 16.46, 17.57, 18.49, 19.65, 20.48, 21.6, 22.87, 23.79, 24.95, 26.21, 26.9, 28.09, 29.27, 30.13, 30.86, 32.22, 33.02, 33.24, 35.01};
static const double kStepCostPadded[SDP_MAX_K] = {3.91, 4.97, 5.97, 6.82, 7.75, 8.78, 9.97, 10.81, 11.85, 12.73, 13.85, 14.93, 16.17, 17.29, 17.78, 19.11, 19.97, 21.1, 22.09, 23.51, 24.22, 25.32, 26.67, 27.58, 28.59, 29.44, 30.79, 31.82, 32.64, 33.59, 34.75, 35.57};

void choose_geometry(sdp_ctx* c, int force_g) {      // force_g: sdp_set_debug_route (geometry experiments), 0 = off
    struct Ent { uint16_t n, G, K, pad; };
    Ent ents[SDP_NSLOTS];
    for (int n = 1; n <= SDP_NSLOTS; ++n) {
        double best = -1; int bG = 32, bK = (n + 31) / 32;
        for (int G = 1; G <= 32; ++G) {
            int K = (n + G - 1) / G;
            if (K > SDP_MAX_K) continue;
            if (G * K - n >= G) continue;
            if (force_g && G != force_g && (n + force_g - 1) / force_g <= SDP_MAX_K &&
                force_g * ((n + force_g - 1) / force_g) - n < force_g) continue;
            double ppw = 2.0 * (32 / G);
            double rows = (double)n + 300.0 + 2.0 * (G - 1);        // two rows of skew per thread
            double thr = ppw / (rows * (G * K != n ? kStepCostPadded[K - 1] : kStepCostExact[K - 1]));
            if (thr > best) { best = thr; bG = G; bK = K; }
        }
        ents[n - 1] = Ent{(uint16_t)n, (uint16_t)bG, (uint16_t)bK, (uint16_t)(bG * bK != n ? 1 : 0)};
    }
    auto cls = [](const Ent& a) { return 2 * (int)a.K + (int)a.pad; };
    std::stable_sort(ents, ents + SDP_NSLOTS, [&](const Ent& a, const Ent& b) { return cls(a) < cls(b); });
    const int NC = 2 * SDP_MAX_K + 2;
    for (int k = 0; k <= NC; ++k) c->cls_begin[k] = SDP_NSLOTS;
    for (int t = SDP_NSLOTS - 1; t >= 0; --t) {
        c->h_slot_n[t] = ents[t].n; c->h_slot_G[t] = ents[t].G; c->h_slot_K[t] = ents[t].K;
        c->h_slot_of_n[ents[t].n - 1] = (uint16_t)t;
        c->cls_begin[cls(ents[t])] = (uint32_t)t;
    }
    // classes that no read length uses start where the next used class starts
    for (int k = NC - 1; k >= 0; --k)
        if (c->cls_begin[k] == SDP_NSLOTS) c->cls_begin[k] = c->cls_begin[k + 1];
    c->cls_begin[0] = 0;
}

}  // namespace

extern "C" {

const char* sdp_version(void) { return "sdp 0.1 (sm_100a)"; }

const char* sdp_last_error(const sdp_ctx* ctx) { return ctx ? ctx->err : "null context"; }

int sdp_create(const sdp_scoring* s, int cuda_device, sdp_ctx** out)
{
    if (!s || !out) return SDP_EINVAL;
    if (s->match < 0 || s->mismatch > 0 || s->match - s->mismatch <= 0 || s->gap_open < 0 || s->gap_extend < 1 ||
        !(s->min_similarity >= 0.0 && s->min_similarity <= 1.0))
        return SDP_EINVAL;
    // limits of the int16 kernels (documented at sdp_scoring in sdp.h): match - mismatch must read as an fp16 value
    // below 1.0 (bit pattern < 0x3C00), and no constant may come near the 16-bit range by itself
    if (s->match > SDP_MAX_SCORE_PARAM || s->mismatch < -SDP_MAX_SCORE_PARAM || s->gap_open > SDP_MAX_SCORE_PARAM ||
        s->gap_extend > SDP_MAX_SCORE_PARAM)
        return SDP_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || cuda_device < 0 || cuda_device >= ndev) return SDP_ECUDA;
    sdp_ctx* ctx = new (std::nothrow) sdp_ctx();
    if (!ctx) return SDP_ENOMEM;
    ctx->device = cuda_device;
    ctx->user_sc = *s;
    ctx->sc = Scoring{s->match, s->mismatch, s->gap_open, s->gap_extend, llround(s->min_similarity * 1e6)};
    const int o = s->gap_open, e = s->gap_extend, beta = 3 * o + 8;      // beta: traceback DP kernel
    {   // score kernel (score_kernel.cuh): c = 2e + mismatch; F~ = F' - c starts at 0 = "minus infinity", which needs
        // beta >= 2o + c
        const int c = 2 * e + s->mismatch, beta_s = 3 * o + 8 + (c > 0 ? c : 0);
        ctx->patch.negOc = sdp_pack2(-(o + c)); ctx->patch.negO = sdp_pack2(-o); ctx->patch.c2 = sdp_pack2(c);
        ctx->patch.Cd = sdp_pack2(s->match - s->mismatch); ctx->patch.e2 = sdp_pack2(e);
        score_modules_init(&ctx->modules);
        ctx->consts.beta2 = sdp_pack2(beta_s);
        ctx->consts.betaMinusO2 = sdp_pack2(beta_s - o);
        ctx->consts.e = e; ctx->consts.beta = beta_s; ctx->consts.match = s->match;
    }
    {   // traceback DP kernels (trace_kernel.cuh, thin_kernel.cu): x8 scaled values with tags in the low three bits,
        // F and u shifted by c = 2e + mismatch as in the score kernel
        const int sc8 = SDP_TB_SCALE, c = 2 * e + s->mismatch, beta_t = 3 * o + 8 + (c > 0 ? c : 0);
        TraceConsts& t = ctx->tconsts;
        t.e2 = sdp_pack2(sc8 * e);
        t.beta2 = sdp_pack2(sc8 * beta_t + 7);
        t.betaMinusO2 = sdp_pack2(sc8 * (beta_t - o) + 7);
        t.e = e; t.beta = beta_t;
        ctx->patch.t_negOf = sdp_pack2(sc8 * (-o - c) - 1);
        ctx->patch.t_negOe = sdp_pack2(-sc8 * o - 6);
        ctx->patch.t_c8 = sdp_pack2(sc8 * c);
        ctx->patch.t_Cd8 = sdp_pack2(sc8 * (s->match - s->mismatch));
        // 8 (match - mismatch) must read as an fp16 value below 1.0, and 8 beta must leave room in 16 bits
        ctx->thin_ok = (sc8 * (s->match - s->mismatch) < 0x3C00 && sc8 * beta_t <= 32000) ? 1 : 0;
        ctx->wide_ok = ctx->thin_ok;
        ctx->wide_fits = ctx->wide_ok;
    }
    choose_geometry(ctx, 0);

    auto init = [&]() -> int {
        CU(cudaSetDevice(cuda_device));
        CU(cudaMalloc(&ctx->d_slot_n, SDP_NSLOTS * 2));
        CU(cudaMalloc(&ctx->d_slot_G, SDP_NSLOTS * 2));
        CU(cudaMalloc(&ctx->d_slot_K, SDP_NSLOTS * 2));
        CU(cudaMemcpy(ctx->d_slot_n, ctx->h_slot_n, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->d_slot_G, ctx->h_slot_G, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
        CU(cudaMemcpy(ctx->d_slot_K, ctx->h_slot_K, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
        CU(cudaMalloc(&ctx->d_slot_of_n, SDP_NSLOTS * 2));
        CU(cudaMemcpy(ctx->d_slot_of_n, ctx->h_slot_of_n, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
        CU(cudaStreamCreateWithFlags(&ctx->own_stream, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
        CU(cudaEventCreateWithFlags(&ctx->ev_seq_ready, cudaEventDisableTiming));
        // Three priority levels (numerically lower = higher priority): the forward kernels of all lanes at the lowest,
        // the narrow-band traceback kernels in the middle, each lane's own stream (bookkeeping, reverse pass, wide
        // traceback: the lane's critical path) at the highest, so that a lane's tail runs under the next lane's
        // forward kernel instead of queueing behind its thousands of CTAs.
        CU(cudaDeviceGetStreamPriorityRange(&ctx->prio_lo, &ctx->prio_hi));
        const int prio_mid = (ctx->prio_lo + ctx->prio_hi) / 2;
        CU(cudaStreamCreateWithPriority(&ctx->fwd_stream, cudaStreamNonBlocking, ctx->prio_lo));
        for (int k = 0; k < 3; ++k) CU(cudaStreamCreateWithPriority(&ctx->side_stream[k], cudaStreamNonBlocking, prio_mid));
        for (int k = 1; k < SDP_FAN_STREAMS; ++k) {
            CU(cudaStreamCreateWithPriority(&ctx->fan_fwd[k], cudaStreamNonBlocking, ctx->prio_lo));
            CU(cudaStreamCreateWithPriority(&ctx->fan_post[k], cudaStreamNonBlocking, ctx->prio_hi));
        }
        CU(cudaEventCreate(&ctx->ev_start));
        CU(cudaEventCreate(&ctx->ev_end));
        for (int k = 0; k < SDP_MAX_LANES; ++k) CU(cudaEventCreateWithFlags(&ctx->ev_cig[k], cudaEventDisableTiming));
        {
            int sms = 148;
            CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, cuda_device));
            ctx->resident_warps = (uint32_t)sms * 12u;
        }
        CU(cudaMalloc(&ctx->cig_total, (SDP_MAX_LANES + 1) * 8));
        CU(cudaMemset(ctx->cig_total, 0, (SDP_MAX_LANES + 1) * 8));
        return lanes_init(ctx, 1);
    };
    int rc = init();
    if (rc != SDP_OK) { sdp_destroy(ctx); return rc; }
    *out = ctx;
    return SDP_OK;
}

void sdp_destroy(sdp_ctx* ctx)
{
    if (!ctx) return;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    score_modules_destroy(&ctx->modules);
    for (int li = 0; li < SDP_MAX_LANES; ++li) if (ctx->lane[li].mb) lane_destroy(ctx->lane[li]);
    DevBuf* bufs[] = {&ctx->score, &ctx->ref_start, &ctx->ref_end, &ctx->read_start, &ctx->read_end, &ctx->pass, &ctx->n_match,
                      &ctx->n_cols, &ctx->cigar_off, &ctx->cigar_len, &ctx->cigar_ops, &ctx->in_reads, &ctx->in_read_off,
                      &ctx->in_read_len, &ctx->in_read_nmask, &ctx->in_wins, &ctx->in_win_off, &ctx->in_win_len,
                      &ctx->in_win_nmask, &ctx->in_pairs, &ctx->rb_key, &ctx->rb_pair, &ctx->rb_score, &ctx->rb_second,
                      &ctx->rb_ncand, &ctx->mp_flag, &ctx->mp_off};
    for (DevBuf* b : bufs) if (b->p) cudaFree(b->p);
    if (ctx->h_out.p) cudaFreeHost(ctx->h_out.p);
    if (ctx->h_ops.p) cudaFreeHost(ctx->h_ops.p);
    if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
    if (ctx->ev_seq_ready) cudaEventDestroy(ctx->ev_seq_ready);
    cudaFree(ctx->cig_total);
    cudaFree(ctx->d_slot_n); cudaFree(ctx->d_slot_G); cudaFree(ctx->d_slot_K); cudaFree(ctx->d_slot_of_n);
    if (ctx->own_stream) cudaStreamDestroy(ctx->own_stream);
    if (ctx->fwd_stream) cudaStreamDestroy(ctx->fwd_stream);
    for (int k = 0; k < 3; ++k) if (ctx->side_stream[k]) cudaStreamDestroy(ctx->side_stream[k]);
    for (int k = 1; k < SDP_FAN_STREAMS; ++k) {
        if (ctx->fan_fwd[k]) cudaStreamDestroy(ctx->fan_fwd[k]);
        if (ctx->fan_post[k]) cudaStreamDestroy(ctx->fan_post[k]);
    }
    if (ctx->ev_start) cudaEventDestroy(ctx->ev_start);
    if (ctx->ev_end) cudaEventDestroy(ctx->ev_end);
    for (int k = 0; k < SDP_MAX_LANES; ++k) if (ctx->ev_cig[k]) cudaEventDestroy(ctx->ev_cig[k]);
    delete ctx;
}

int sdp_set_timing(sdp_ctx* ctx, int enabled)
{
    if (!ctx) return SDP_EINVAL;
    ctx->timing = enabled != 0;
    return SDP_OK;
}

int sdp_set_debug_route(sdp_ctx* ctx, uint32_t flags)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    const int force_g = (int)((flags >> 8) & 0x3Fu);
    if ((flags & ~(SDP_ROUTE_NO_THIN | SDP_ROUTE_NO_WIDE | SDP_ROUTE_ALWAYS_REVERSE | 0x3F00u)) || force_g > 32)
        return fail(ctx, SDP_EINVAL, "unknown route flags");
    ctx->no_thin = (flags & SDP_ROUTE_NO_THIN) ? 1 : 0;
    ctx->force_rev = (flags & SDP_ROUTE_ALWAYS_REVERSE) ? 1 : 0;
    ctx->wide_ok = (flags & SDP_ROUTE_NO_WIDE) ? 0 : ctx->wide_fits;
    choose_geometry(ctx, force_g);
    CU(cudaSetDevice(ctx->device));
    CU(cudaMemcpy(ctx->d_slot_n, ctx->h_slot_n, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_slot_G, ctx->h_slot_G, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_slot_K, ctx->h_slot_K, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
    CU(cudaMemcpy(ctx->d_slot_of_n, ctx->h_slot_of_n, SDP_NSLOTS * 2, cudaMemcpyHostToDevice));
    return SDP_OK;
}

int sdp_set_prefilter(sdp_ctx* ctx, int enabled)
{
    if (!ctx) return SDP_EINVAL;
    ctx->prefilter = enabled != 0;
    return SDP_OK;
}

int sdp_set_mode(sdp_ctx* ctx, int mode)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (mode != SDP_MODE_SEMIGLOBAL && mode != SDP_MODE_LOCAL) return fail(ctx, SDP_EINVAL, "unknown alignment mode %d", mode);
    ctx->mode = mode;
    return SDP_OK;
}

int sdp_set_score_only(sdp_ctx* ctx, int enabled)
{
    if (!ctx) return SDP_EINVAL;
    ctx->score_only = enabled != 0;
    return SDP_OK;
}

int sdp_get_stats(const sdp_ctx* ctx, sdp_stats* out)
{
    if (!ctx || !out) return SDP_EINVAL;
    *out = ctx->stats;
    return SDP_OK;
}

int sdp_measure_dpx_rate(int cuda_device, double* rate, int32_t* sms, double* mhz)
{
    return measure_dpx_rate(cuda_device, rate, sms, mhz);
}

int sdp_set_chunks(sdp_ctx* ctx, int chunks)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (chunks < 0 || chunks > SDP_MAX_LANES) return fail(ctx, SDP_EINVAL, "chunks must be 0 (automatic) .. %d", SDP_MAX_LANES);
    ctx->chunks = chunks;
    return SDP_OK;
}

// which: 0 forward, 1 reverse, 2 traceback DP (trace_kernel). Launches on `st`; with several column-count classes
// (mixed read lengths) the launches go round-robin over `st` and the helper streams fan[1..], forked from and
// joined back into `st` with the lane's events, so that one class's tail overlaps the next class's start.
static int launch_score_stage(sdp_ctx* ctx, Lane& L, int which, const PairDesc* desc, cudaStream_t st,
                              cudaStream_t* fan, uint32_t* nlaunch)
{
    const bool rev = which == 1;
    const int ti = which == 0 ? 0 : 2;                    // task table: the reverse pass runs on the wide-traceback buckets
    const sdp_batch& b = L.b;
    TraceDP td{};
    td.c = ctx->tconsts; td.bits = L.wide_bits.as<uint32_t>(); td.bits_off = L.wide_off.as<uint64_t>();
    const uint32_t* tp = L.mb->task_prefix[ti];
    ScoreParams sp{};
    sp.reads_packed = b.reads_packed; sp.read_nmask = b.read_nmask;
    sp.wins_packed = b.wins_packed; sp.win_nmask = b.win_nmask;
    sp.wins_words = (b.wins_bases + 15) / 16; sp.win_nmask_words = (b.wins_bases + 31) / 32;
    sp.desc = desc;
    sp.task_prefix = L.task_prefix[ti];
    sp.slots = L.slots[ti];
    sp.c = ctx->consts;
    sp.score = ctx->score.as<int32_t>() + L.p0; sp.ref_end = ctx->ref_end.as<int32_t>() + L.p0;
    sp.rev_rows = L.rev_rows.as<int32_t>(); sp.err_flag = L.err_flag;
    int classes = 0;
    for (int cls = 2; cls <= 2 * SDP_MAX_K + 1; ++cls) {
        const uint32_t s0 = ctx->cls_begin[cls], s1 = ctx->cls_begin[cls + 1];
        if (s1 > s0 && tp[s1] > tp[s0]) ++classes;
    }
    const bool do_fan = classes > 1;
    if (do_fan) {
        CU(cudaEventRecord(L.fan_fork, st));
        for (int k = 1; k < SDP_FAN_STREAMS; ++k) CU(cudaStreamWaitEvent(fan[k], L.fan_fork, 0));
    }
    int turn = 0;
    for (int cls = 2 * SDP_MAX_K + 1; cls >= 2; --cls) {                 // largest K (longest reads) first
        const uint32_t s0 = ctx->cls_begin[cls], s1 = ctx->cls_begin[cls + 1];
        if (s1 <= s0) continue;
        const uint32_t t0 = tp[s0], t1 = tp[s1];
        if (t1 <= t0) continue;
        sp.slot_lo = s0; sp.slot_hi = s1; sp.task_begin = t0; sp.task_end = t1;
        cudaStream_t ls = (do_fan && (turn % SDP_FAN_STREAMS)) ? fan[turn % SDP_FAN_STREAMS] : st;
        ++turn;
        {
            const int rc = score_modules_launch(&ctx->modules, ctx->patch, cls >> 1, (cls & 1) != 0, rev, sp,
                                                which == 2 ? &td : nullptr, ls, ctx->err, sizeof(ctx->err));
            if (rc != SDP_OK) return rc;
        }
        ++*nlaunch;
    }
    if (do_fan) {
        for (int k = 1; k < SDP_FAN_STREAMS; ++k) {
            CU(cudaEventRecord(L.fan_join[k], fan[k]));
            CU(cudaStreamWaitEvent(st, L.fan_join[k], 0));
        }
    }
    CU(cudaGetLastError());
    return SDP_OK;
}

namespace {

// wait until nothing of this ctx is in flight any more (error paths: a later call must not meet leftover work)
void drain(sdp_ctx* ctx)
{
    cudaStreamSynchronize(ctx->fwd_stream);
    for (int k = 0; k < 3; ++k) cudaStreamSynchronize(ctx->side_stream[k]);
    for (int k = 1; k < SDP_FAN_STREAMS; ++k) { cudaStreamSynchronize(ctx->fan_fwd[k]); cudaStreamSynchronize(ctx->fan_post[k]); }
    for (int li = 0; li < ctx->lanes_ready; ++li) cudaStreamSynchronize(ctx->lane[li].st);
}

// ---- phase A: a1 + a2 of one lane (validate, key, histogram, scan, scatter, task table), enqueued on the lane's stream
int lane_phase_a(sdp_ctx* ctx, Lane& L, const int local)
{
    const sdp_batch& b = L.b;
    const uint64_t P = L.P;
    const size_t Pp = (size_t)(P ? P : 1);
    LEN(keys, Pp * 4); LEN(pn, Pp * 4); LEN(pm, Pp * 4); LEN(order, Pp * 4); LEN(desc, Pp * sizeof(PairDesc));
    LEN(desc_rev, Pp * sizeof(PairDesc)); LEN(order_tb, Pp * 4);
    LEN(keys_tb, Pp * 4); LEN(tbW, Pp * 4); LEN(rev_rows, Pp * 4);
    LEN(tb_rows, Pp * 4); LEN(keys_wide, Pp * 4); LEN(order_wide, Pp * 4); LEN(desc_wide, Pp * sizeof(PairDesc));
    LEN(wide_words, Pp * 4); LEN(wide_off, Pp * 8);
    LEN(bits_words, Pp * 4); LEN(ops_cap, Pp * 4); LEN(bits_off, Pp * 8); LEN(ops_off, Pp * 8);
    for (int k = 0; k < 3; ++k) { LEN(scan_local[k], Pp * 4); LEN(scan_tiles[k], (Pp / 4096 + 2) * 4); LEN(scan_tile_base[k], (Pp / 4096 + 2) * 8); }
    LEN(slow_words, Pp * 4); LEN(slow_off, Pp * 8);
    cudaStream_t st = L.st;
    L.nl = 0; L.fwd_launches = 0; L.n_wide = 0;
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_A0], st));
    if (ctx->wait_seq && ctx->prefilter) CU(cudaStreamWaitEvent(st, ctx->ev_seq_ready, 0));   // the pre-pass reads sequences
    CU(cudaMemsetAsync(L.zero_block, 0, L.zero_bytes, st));
    CU(cudaMemsetAsync(L.wide_words.p, 0, P * 4, st));       // region sizes of the wide traceback (filled after the forward pass)
    launch_validate_key(b, ctx->sc, L.keys.as<uint32_t>(), L.pn.as<uint32_t>(), L.pm.as<uint32_t>(),
                        L.hist[0], L.err_flag, L.counters + 3, (ctx->prefilter && !local) ? 1 : 0,
                        ctx->score.as<int32_t>() + L.p0, ctx->ref_end.as<int32_t>() + L.p0, L.counters + 4, local,
                        L.slow_words.as<uint32_t>(), L.counters + 5, st);
    // (row arrays of the int32 lane: the host learns their total here; their offsets are scanned in phase B, and only
    // when there are any)
    CU(cudaMemcpyAsync(&L.mb->slow_total, L.counters + 5, 8, cudaMemcpyDeviceToHost, st));
    // bucket sort; the scatter writes the forward descriptors straight into bucket order
    launch_sort_tail(L.keys.as<uint32_t>(), P, L.hist[0], L.bin_start[0], L.order.as<uint32_t>(),
                     ctx->d_slot_n, ctx->d_slot_G, ctx->d_slot_K, L.slots[0], L.task_prefix[0],
                     L.mb->task_prefix[0], &L.mb->bin_total[0], st, &L.b, L.desc.as<PairDesc>());
    L.nl += 5;
    CU(cudaMemcpyAsync(&L.mb->err_flag, L.err_flag, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaEventRecord(L.evA, st));
    return SDP_OK;
}

// ---- phase B: a3 on the shared forward stream, then (on the lane's stream) the gap bound W, the keys of the later
// stages, their bucket sorts and the scratch-size scans
int lane_phase_b(sdp_ctx* ctx, Lane& L, const int local)
{
    const sdp_batch& b = L.b;
    const uint64_t P = L.P;
    cudaStream_t st = L.st, fs = ctx->fwd_stream;
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_A1], st));
    CU(cudaEventRecord(L.ev_desc, st));
    CU(cudaStreamWaitEvent(fs, L.ev_desc, 0));
    if (ctx->wait_seq) CU(cudaStreamWaitEvent(fs, ctx->ev_seq_ready, 0));     // host path: sequences upload beside a1/a2
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_F0], fs));
    {
        uint32_t before = L.nl;
        int rc = launch_score_stage(ctx, L, 0, L.desc.as<PairDesc>(), fs, ctx->fan_fwd, &L.nl);
        if (rc != SDP_OK) return rc;
        L.fwd_launches = L.nl - before;
    }
    if (L.mb->slow_total) {
        // the int32 lane: pairs outside the int16 kernels' domain, and every pair in local mode (slow_lane.cu)
        LEN(slow_rows, (L.mb->slow_total + 4) * 4);
        exclusive_scan_u32_u64(L.slow_words.as<uint32_t>(), P, L.slow_off.as<uint64_t>(), L.totals + 0, nullptr,
                               L.scan_local[0].as<uint32_t>(), L.scan_tiles[0].as<uint32_t>(),
                               L.scan_tile_base[0].as<uint64_t>(), fs, &L.nl);
        launch_forward_i32(b, ctx->sc, local, L.slow_words.as<uint32_t>(), L.slow_off.as<uint64_t>(),
                           L.slow_rows.as<int32_t>(), ctx->score.as<int32_t>() + L.p0, ctx->ref_end.as<int32_t>() + L.p0,
                           L.rev_rows.as<int32_t>(), fs);
        L.nl += local ? 5 : 3;
    }
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_F1], fs));
    CU(cudaEventRecord(L.ev_fwd, fs));
    CU(cudaStreamWaitEvent(st, L.ev_fwd, 0));
    if (ctx->h_early_score) {
        // host path: score and ref_end are final now; their download runs under the rest of the path
        CU(cudaStreamWaitEvent(ctx->copy_stream, L.ev_fwd, 0));
        CU(cudaMemcpyAsync(ctx->h_early_score + L.p0, ctx->score.as<int32_t>() + L.p0, P * 4, cudaMemcpyDeviceToHost, ctx->copy_stream));
        CU(cudaMemcpyAsync(ctx->h_early_ref_end + L.p0, ctx->ref_end.as<int32_t>() + L.p0, P * 4, cudaMemcpyDeviceToHost, ctx->copy_stream));
    }

    if (ctx->score_only) {
        // candidate screening (step-3 shape): score and ref_end only; everything the traceback would fill reads
        // as "no alignment" (ref_start -1, no CIGAR, pass 0)
        CU(cudaMemsetAsync(ctx->ref_start.as<int32_t>() + L.p0, 0xFF, P * 4, st));
        CU(cudaMemsetAsync(ctx->read_start.as<int32_t>() + L.p0, 0, P * 4, st));
        CU(cudaMemsetAsync(ctx->read_end.as<int32_t>() + L.p0, 0xFF, P * 4, st));
        CU(cudaMemsetAsync(ctx->pass.as<uint8_t>() + L.p0, 0, P, st));
        CU(cudaMemsetAsync(ctx->n_match.as<int32_t>() + L.p0, 0, P * 4, st));
        CU(cudaMemsetAsync(ctx->n_cols.as<int32_t>() + L.p0, 0, P * 4, st));
        CU(cudaMemsetAsync(ctx->cigar_off.as<uint64_t>() + L.p0, 0, P * 8, st));
        CU(cudaMemsetAsync(ctx->cigar_len.as<uint32_t>() + L.p0, 0, P * 4, st));
        CU(cudaMemcpyAsync(L.mb->counters + 3, L.counters + 3, 16, cudaMemcpyDeviceToHost, st));
        if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_END], st));
        CU(cudaEventRecord(L.evB, st));
        return SDP_OK;
    }

    PostParams pp{};
    pp.b = b; pp.n_pairs = P; pp.sc = ctx->sc; pp.pn = L.pn.as<uint32_t>(); pp.pm = L.pm.as<uint32_t>();
    pp.score = ctx->score.as<int32_t>() + L.p0; pp.ref_end = ctx->ref_end.as<int32_t>() + L.p0;
    pp.tbW = L.tbW.as<int32_t>(); pp.tb_rows = L.tb_rows.as<int32_t>();
    pp.keys_tb = L.keys_tb.as<uint32_t>();
    pp.keys_wide = L.keys_wide.as<uint32_t>();
    pp.wide_ok = ctx->wide_ok; pp.no_thin = ctx->no_thin; pp.thin_ok = ctx->thin_ok;
    pp.local = local; pp.slow_words = L.slow_words.as<uint32_t>(); pp.end_col = L.rev_rows.as<int32_t>();

    pp.err_flag = L.err_flag;
    pp.bits_words = L.bits_words.as<uint32_t>(); pp.ops_cap = L.ops_cap.as<uint32_t>();
    pp.hist_tb = L.hist[2]; pp.hist_wide = L.hist[3]; pp.counters = L.counters;
    launch_post_forward(pp, st);
    // The two bucket sorts and the three scratch-offset scans are short, latency-bound launch chains that
    // depend only on k_post_forward: they fan out over the helper streams and join before the mailbox kernel.
    // (The reverse pass and the wide traceback serve the same pairs with the same key: one sort, one task table.)
    cudaStream_t f2 = ctx->fan_post[2], f3 = ctx->fan_post[3];
    CU(cudaEventRecord(L.fan_fork, st));
    for (int k = 2; k < SDP_FAN_STREAMS; ++k) CU(cudaStreamWaitEvent(ctx->fan_post[k], L.fan_fork, 0));
    launch_sort_tail(L.keys_tb.as<uint32_t>(), P, L.hist[2], L.bin_start[2], L.order_tb.as<uint32_t>(),
                     nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, f2);
    launch_sort_tail(L.keys_wide.as<uint32_t>(), P, L.hist[3], L.bin_start[3], L.order_wide.as<uint32_t>(),
                     ctx->d_slot_n, ctx->d_slot_G, ctx->d_slot_K, L.slots[2], L.task_prefix[2],
                     L.mb->task_prefix[2], &L.mb->bin_total[3], st);
    L.nl += 8;
    // one region of direction nibbles per warp task of wide pairs (every slot of order_wide beyond the wide
    // pairs reads as a zero-size region)
    launch_wide_regions(L.order_wide.as<uint32_t>(), (uint32_t)P, L.bin_start[3] + SDP_NBINS, L.pn.as<uint32_t>(),
                        L.tb_rows.as<int32_t>(), ctx->d_slot_of_n, L.slots[2], L.wide_words.as<uint32_t>(), st);
    ++L.nl;
    exclusive_scan_u32_u64(L.wide_words.as<uint32_t>(), P, L.wide_off.as<uint64_t>(), L.totals + 3, nullptr,
                           L.scan_local[0].as<uint32_t>(), L.scan_tiles[0].as<uint32_t>(),
                           L.scan_tile_base[0].as<uint64_t>(), st, &L.nl);
    exclusive_scan_u32_u64(L.bits_words.as<uint32_t>(), P, L.bits_off.as<uint64_t>(), L.totals + 0, nullptr,
                           L.scan_local[1].as<uint32_t>(), L.scan_tiles[1].as<uint32_t>(),
                           L.scan_tile_base[1].as<uint64_t>(), f2, &L.nl);
    exclusive_scan_u32_u64(L.ops_cap.as<uint32_t>(), P, L.ops_off.as<uint64_t>(), L.totals + 1, nullptr,
                           L.scan_local[2].as<uint32_t>(), L.scan_tiles[2].as<uint32_t>(),
                           L.scan_tile_base[2].as<uint64_t>(), f3, &L.nl);
    for (int k = 2; k < SDP_FAN_STREAMS; ++k) {
        CU(cudaEventRecord(L.fan_join[k], ctx->fan_post[k]));
        CU(cudaStreamWaitEvent(st, L.fan_join[k], 0));
    }
    launch_mailbox(L.bin_start[2], TB_KEY_STRIDE, THIN_NW + TB_NCLASS + 1, L.totals, L.counters,
                   L.mb->tb_bounds, L.mb->totals, L.mb->counters, st);
    ++L.nl;
    CU(cudaEventRecord(L.evB, st));
    return SDP_OK;
}

// ---- phase C: a4 reverse pass, a5 + a6 traceback (wide path on the lane's stream, narrow bands on the side streams)
int lane_phase_c(sdp_ctx* ctx, Lane& L, const int local)
{
    const sdp_batch& b = L.b;
    cudaStream_t st = L.st;
    const uint32_t n_wide = L.mb->bin_total[3];
    L.n_wide = n_wide;
    LEN(bits, (L.mb->totals[0] + 4) * 4);
    LEN(ops_rev, (L.mb->totals[1] + 4) * 4);
    LEN(wide_bits, (L.mb->totals[3] + 4) * 4);
    int32_t* score = ctx->score.as<int32_t>() + L.p0;
    int32_t* ref_end = ctx->ref_end.as<int32_t>() + L.p0;

    // ---- a4 reverse pass over the wide pairs (same buckets and task table as their traceback DP)
    // a4 where it pays (k_fill_desc_rev): with fewer wide-pair tasks than four waves of resident warps the kernels'
    // time follows the longest task, not the total work, and every wide pair takes the pass
    const uint32_t wide_tasks = L.mb->task_prefix[2][SDP_NSLOTS];
    const int ratio10 = (ctx->force_rev || wide_tasks < 4u * ctx->resident_warps) ? 0 : 24;
    launch_fill_desc_rev(b, L.order_wide.as<uint32_t>(), n_wide, score, ref_end, L.tbW.as<int32_t>(), ratio10,
                         L.rev_rows.as<int32_t>(), L.counters, L.desc_rev.as<PairDesc>(), st);
    ++L.nl;
    {
        int rc = launch_score_stage(ctx, L, 1, L.desc_rev.as<PairDesc>(), st, ctx->fan_post, &L.nl);
        if (rc != SDP_OK) return rc;
    }
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_REV], st));

    // ---- a5 + a6: wide pairs: rectangle DP that leaves four direction bits per cell, then the walk
    if (n_wide) {
        launch_fill_desc_tb(b, L.order_wide.as<uint32_t>(), n_wide, score, ref_end, L.rev_rows.as<int32_t>(),
                            L.desc_wide.as<PairDesc>(), st);
        ++L.nl;
        int rc = launch_score_stage(ctx, L, 2, L.desc_wide.as<PairDesc>(), st, ctx->fan_post, &L.nl);
        if (rc != SDP_OK) return rc;
        WalkParams wp{};
        wp.b = b; wp.sc = ctx->sc; wp.desc = L.desc_wide.as<PairDesc>(); wp.count = n_wide;
        wp.slots = L.slots[2]; wp.slot_of_n = ctx->d_slot_of_n;
        wp.bits = L.wide_bits.as<uint32_t>(); wp.bits_off = L.wide_off.as<uint64_t>();
        wp.ref_end = ref_end; wp.tbW = L.tbW.as<int32_t>();
        wp.ops_off = L.ops_off.as<uint64_t>(); wp.ops_rev = L.ops_rev.as<uint32_t>();
        wp.ref_start = ctx->ref_start.as<int32_t>() + L.p0; wp.read_start = ctx->read_start.as<int32_t>() + L.p0;
        wp.read_end = ctx->read_end.as<int32_t>() + L.p0; wp.pass = ctx->pass.as<uint8_t>() + L.p0;
        wp.n_match = ctx->n_match.as<int32_t>() + L.p0; wp.n_cols = ctx->n_cols.as<int32_t>() + L.p0;
        wp.cigar_len = ctx->cigar_len.as<uint32_t>() + L.p0; wp.err_flag = L.err_flag;
        launch_walk(wp, st);
        ++L.nl;
    }
    // ---- a5 + a6, narrow bands (W < THIN_NW: two pairs per thread, band in registers) and the generic band kernel.
    // They need nothing from the reverse pass and touch other pairs than the wide path, so they run on side streams
    // beside it (the host has waited for the lane's phase B, which produced everything they read).
    TraceParams tp{};
    tp.b = b; tp.sc = ctx->sc; tp.order = L.order_tb.as<uint32_t>();
    tp.score = score; tp.ref_end = ref_end; tp.tbW = L.tbW.as<int32_t>();
    tp.rev_rows = nullptr; tp.end_col = L.rev_rows.as<int32_t>();
    tp.bits_off = L.bits_off.as<uint64_t>(); tp.bits = L.bits.as<uint32_t>();
    tp.ops_off = L.ops_off.as<uint64_t>(); tp.ops_rev = L.ops_rev.as<uint32_t>();
    tp.ref_start = ctx->ref_start.as<int32_t>() + L.p0; tp.read_start = ctx->read_start.as<int32_t>() + L.p0;
    tp.read_end = ctx->read_end.as<int32_t>() + L.p0; tp.pass = ctx->pass.as<uint8_t>() + L.p0;
    tp.n_match = ctx->n_match.as<int32_t>() + L.p0; tp.n_cols = ctx->n_cols.as<int32_t>() + L.p0;
    tp.cigar_len = ctx->cigar_len.as<uint32_t>() + L.p0; tp.err_flag = L.err_flag;
    L.nl += (uint32_t)launch_thin_all(L.mb->tb_bounds, tp, ctx->side_stream[0], ctx->side_stream[1], ctx->side_stream[2]);
    for (int c = THIN_NW; c < THIN_NW + TB_NCLASS; ++c) {
        tp.first = L.mb->tb_bounds[c];
        tp.count = L.mb->tb_bounds[c + 1] - tp.first;
        if (!tp.count) continue;
        launch_traceback(c - THIN_NW, local != 0, tp, ctx->side_stream[0]);
        ++L.nl;
    }
    for (int k = 0; k < 3; ++k) {
        CU(cudaEventRecord(L.side_done[k], ctx->side_stream[k]));
        CU(cudaStreamWaitEvent(st, L.side_done[k], 0));
    }
    CU(cudaGetLastError());
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_TRACE], st));
    CU(cudaEventRecord(L.evC, st));
    return SDP_OK;
}

// ---- phase D: a7 compaction in caller pair order; the lane's run offsets start at the previous lanes' total
int lane_phase_d(sdp_ctx* ctx, Lane& L, const int li)
{
    cudaStream_t st = L.st;
    const uint64_t P = L.P;
    if (li > 0) CU(cudaStreamWaitEvent(st, ctx->ev_cig[li - 1], 0));
    exclusive_scan_u32_u64(ctx->cigar_len.as<uint32_t>() + L.p0, P, ctx->cigar_off.as<uint64_t>() + L.p0, ctx->cig_total + li + 1,
                           ctx->cig_total + li, L.scan_local[0].as<uint32_t>(), L.scan_tiles[0].as<uint32_t>(),
                           L.scan_tile_base[0].as<uint64_t>(), st, &L.nl);
    CU(cudaEventRecord(ctx->ev_cig[li], st));
    launch_compact(P, L.ops_off.as<uint64_t>(), L.ops_rev.as<uint32_t>(), ctx->cigar_len.as<uint32_t>() + L.p0,
                   ctx->cigar_off.as<uint64_t>() + L.p0, ctx->cigar_ops.as<uint32_t>(), st);
    ++L.nl;
    CU(cudaMemcpyAsync(&L.mb->totals[2], ctx->cig_total + li + 1, 8, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(&L.mb->err_flag, L.err_flag, 4, cudaMemcpyDeviceToHost, st));
    CU(cudaMemcpyAsync(L.mb->counters, L.counters, 3 * 8, cudaMemcpyDeviceToHost, st));   // reverse counters: k_fill_desc_rev
    if (ctx->timing) CU(cudaEventRecord(L.tev[LEV_END], st));
    CU(cudaEventRecord(L.evD, st));
    return SDP_OK;
}

}  // namespace

int sdp_align_batch(sdp_ctx* ctx, const sdp_batch* batch, void* cuda_stream, sdp_result* out)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (!batch || !out) return fail(ctx, SDP_EINVAL, "null batch or result");
    const sdp_batch& b = *batch;
    const uint64_t P = b.n_pairs;
    if (P > 0 && (!b.reads_packed || !b.read_off || !b.read_len || !b.wins_packed || !b.win_off || !b.win_len ||
                  !b.pairs || b.n_reads == 0 || b.n_wins == 0))
        return fail(ctx, SDP_EINVAL, "null input array");
    if (P > 0xFFFFFFF0ull) return fail(ctx, SDP_EINVAL, "too many pairs");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->device));
    // a failed call may already have overwritten result buffers: its batch must not pass for the "last aligned" one
    ctx->last_pairs = nullptr; ctx->last_n_pairs = 0; ctx->last_n_reads = 0;
    sdp_stats stats{};
    stats.n_pairs = P;

    const size_t Pp = (size_t)(P ? P : 1);
    EN(score, Pp * 4); EN(ref_start, Pp * 4); EN(ref_end, Pp * 4); EN(read_start, Pp * 4); EN(read_end, Pp * 4);
    EN(pass, Pp); EN(n_match, Pp * 4); EN(n_cols, Pp * 4); EN(cigar_off, Pp * 8); EN(cigar_len, Pp * 4);
    const int local = ctx->mode == SDP_MODE_LOCAL ? 1 : 0;

    auto finish = [&](uint64_t n_ops) {
        out->score = ctx->score.as<int32_t>(); out->ref_start = ctx->ref_start.as<int32_t>();
        out->ref_end = ctx->ref_end.as<int32_t>(); out->read_start = ctx->read_start.as<int32_t>();
        out->read_end = ctx->read_end.as<int32_t>(); out->pass = ctx->pass.as<uint8_t>();
        out->n_match = ctx->n_match.as<int32_t>(); out->n_cols = ctx->n_cols.as<int32_t>();
        out->cigar_off = ctx->cigar_off.as<uint64_t>(); out->cigar_len = ctx->cigar_len.as<uint32_t>();
        out->cigar_ops = ctx->cigar_ops.as<uint32_t>(); out->n_cigar_ops = n_ops; out->n_pairs = P;
    };
    if (P == 0) {
        EN(cigar_ops, 16);
        ctx->stats = stats;
        ctx->last_pairs = b.pairs; ctx->last_n_pairs = 0; ctx->last_n_reads = b.n_reads;
        finish(0);
        return SDP_OK;
    }

    // ---- lanes: contiguous ranges of the pair list, software-pipelined (see Lane)
    int NL = ctx->chunks;
    if (NL <= 0) NL = 1;      // measured on B200: a lane's latency-bound tail under the next forward kernel costs that kernel
                              // more than it hides, so pipelining stays opt-in
    if ((uint64_t)NL > P) NL = (int)P;
    {
        const int rc = lanes_init(ctx, NL);
        if (rc != SDP_OK) return rc;
    }
    // from here on work is in flight on the ctx's streams: every failure leaves through bail(), which waits for all of
    // it, so that a later call (or a reallocation's cudaFree) never meets leftover kernels
    auto bail = [&](int rc) { drain(ctx); return rc; };
#define CUB(call)                                                                                        \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return bail(fail(ctx, e_ == cudaErrorMemoryAllocation ? SDP_ENOMEM : SDP_ECUDA,              \
                             "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__));      \
    } while (0)
    CUB(cudaEventRecord(ctx->ev_start, st));
    CUB(cudaStreamWaitEvent(ctx->fwd_stream, ctx->ev_start, 0));
    for (int li = 0; li < NL; ++li) {
        Lane& L = ctx->lane[li];
        L.p0 = P * (uint64_t)li / (uint64_t)NL;
        L.P = P * (uint64_t)(li + 1) / (uint64_t)NL - L.p0;
        L.b = b; L.b.pairs = b.pairs + 2 * L.p0; L.b.n_pairs = L.P;
        CUB(cudaStreamWaitEvent(L.st, ctx->ev_start, 0));
    }

    for (int li = 0; li < NL; ++li) {
        const int rc = lane_phase_a(ctx, ctx->lane[li], local);
        if (rc != SDP_OK) return bail(rc);
    }
    for (int li = 0; li < NL; ++li) {
        Lane& L = ctx->lane[li];
        CUB(cudaEventSynchronize(L.evA));
        if (L.mb->err_flag & SDP_ERRF_INDEX)
            return bail(fail(ctx, SDP_EINVAL, "pair index, offset or length out of range (or empty sequence)"));
        if (L.mb->err_flag & SDP_ERRF_RANGE)
            return bail(fail(ctx, SDP_ERANGE, "a sequence is longer than SDP_MAX_SEQ_LEN, or a pair is outside the int32 "
                             "range rule (see sdp.h)"));
    }
    for (int li = 0; li < NL; ++li) {
        const int rc = lane_phase_b(ctx, ctx->lane[li], local);
        if (rc != SDP_OK) return bail(rc);
    }
    uint64_t n_ops = 0;
    if (!ctx->score_only) {
        uint64_t ops_capacity = 0;
        for (int li = 0; li < NL; ++li) {
            Lane& L = ctx->lane[li];
            CUB(cudaEventSynchronize(L.evB));
            ops_capacity += L.mb->totals[1];
            const int rc = lane_phase_c(ctx, L, local);
            if (rc != SDP_OK) return bail(rc);
        }
        {
            const int rc = ensure(ctx, ctx->cigar_ops, (ops_capacity + 4) * 4);
            if (rc != SDP_OK) return bail(rc);
        }
        for (int li = 0; li < NL; ++li) {
            const int rc = lane_phase_d(ctx, ctx->lane[li], li);
            if (rc != SDP_OK) return bail(rc);
        }
        for (int li = 0; li < NL; ++li) CUB(cudaStreamWaitEvent(st, ctx->lane[li].evD, 0));
    } else {
        const int rc = ensure(ctx, ctx->cigar_ops, 16);
        if (rc != SDP_OK) return bail(rc);
        for (int li = 0; li < NL; ++li) CUB(cudaStreamWaitEvent(st, ctx->lane[li].evB, 0));
    }
    CUB(cudaEventRecord(ctx->ev_end, st));
    CUB(cudaStreamSynchronize(st));
    CUB(cudaGetLastError());
    uint32_t errf = 0;
    for (int li = 0; li < NL; ++li) errf |= ctx->lane[li].mb->err_flag;
    if (!ctx->score_only) {
        if (errf & SDP_ERRF_RANGE)
            return bail(fail(ctx, SDP_ERANGE, "the traceback scratch of one pair exceeds 16 GiB (see sdp.h)"));
        if (errf & (SDP_ERRF_REVERSE | SDP_ERRF_TRACE))
            return bail(fail(ctx, SDP_ECUDA, "internal consistency check failed (flags 0x%x): reverse pass or traceback "
                             "disagrees with the forward score", errf));
        n_ops = ctx->lane[NL - 1].mb->totals[2];
    }

#undef CUB
    if (ctx->timing) cudaEventElapsedTime(&stats.ms_total, ctx->ev_start, ctx->ev_end);
    for (int li = 0; li < NL; ++li) {
        Lane& L = ctx->lane[li];
        stats.cells_forward += L.mb->counters[3];
        stats.cells_prefiltered += L.mb->counters[4];
        stats.n_slow_words += L.mb->slow_total;
        stats.kernel_launches += L.nl;
        stats.forward_launches += L.fwd_launches;
        if (!ctx->score_only) {
            stats.cells_reverse += L.mb->counters[0];
            stats.cells_traceback += L.mb->counters[1];
            stats.n_reverse_pairs += L.mb->counters[2];
        }
        if (ctx->timing) {
            // per-stage times are summed over the lanes; with more than one lane the stages of different lanes overlap,
            // so the sum of the parts exceeds ms_total (ms_forward: the forward kernels run back to back on one stream)
            float t = 0.f;
            cudaEventElapsedTime(&t, L.tev[LEV_A0], L.tev[LEV_A1]); stats.ms_bucket += t;
            cudaEventElapsedTime(&t, L.tev[LEV_F0], L.tev[LEV_F1]); stats.ms_forward += t;
            if (!ctx->score_only) {
                cudaEventElapsedTime(&t, L.tev[LEV_F1], L.tev[LEV_REV]); stats.ms_reverse += t;
                cudaEventElapsedTime(&t, L.tev[LEV_REV], L.tev[LEV_TRACE]); stats.ms_traceback += t;
                cudaEventElapsedTime(&t, L.tev[LEV_TRACE], L.tev[LEV_END]); stats.ms_compact += t;
            }
        }
    }
    ctx->stats = stats;
    ctx->last_pairs = b.pairs; ctx->last_n_pairs = P; ctx->last_n_reads = b.n_reads;
    finish(n_ops);
    return SDP_OK;
}

int sdp_best_per_read(sdp_ctx* ctx, const sdp_batch* batch, const sdp_result* result, void* cuda_stream,
                      sdp_read_best* out)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (!batch || !result || !out) return fail(ctx, SDP_EINVAL, "null batch, result or output");
    if (result->score != ctx->score.as<int32_t>() || result->n_pairs != batch->n_pairs ||
        batch->pairs != ctx->last_pairs || batch->n_pairs != ctx->last_n_pairs || batch->n_reads != ctx->last_n_reads)
        return fail(ctx, SDP_EINVAL, "result does not belong to the last sdp_align_batch of this ctx on this batch");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->device));
    const size_t R = batch->n_reads ? batch->n_reads : 1;
    EN(rb_key, R * 8); EN(rb_pair, R * 4); EN(rb_score, R * 4); EN(rb_second, R * 4); EN(rb_ncand, R * 4);
    launch_best_per_read(batch->n_pairs, batch->n_reads, batch->pairs, result->score,
                         ctx->rb_key.as<unsigned long long>(), ctx->rb_pair.as<uint32_t>(), ctx->rb_score.as<int32_t>(),
                         ctx->rb_second.as<int32_t>(), ctx->rb_ncand.as<uint32_t>(), st);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
    out->best_pair = ctx->rb_pair.as<uint32_t>(); out->best_score = ctx->rb_score.as<int32_t>();
    out->second_score = ctx->rb_second.as<int32_t>(); out->n_candidates = ctx->rb_ncand.as<uint32_t>();
    out->n_reads = batch->n_reads;
    return SDP_OK;
}

int sdp_mate_windows(sdp_ctx* ctx, const sdp_mates* mates, uint32_t min_insert, uint32_t max_insert, uint64_t ref_bases,
                     void* cuda_stream, uint64_t* win_off, uint32_t* win_len)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (!mates || !win_off || !win_len || min_insert > max_insert) return fail(ctx, SDP_EINVAL, "null argument or min_insert > max_insert");
    if (mates->n && (!mates->mate_pos || !mates->mate_len || !mates->mate_reverse || !mates->read_len))
        return fail(ctx, SDP_EINVAL, "null input array");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->device));
    launch_mate_windows(*mates, min_insert, max_insert, ref_bases, win_off, win_len, st);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
    return SDP_OK;
}

int sdp_mate_pairs(sdp_ctx* ctx, const uint32_t* win_len, uint64_t n, void* cuda_stream, uint32_t* pairs,
                   uint32_t* pair_of_rescue, uint64_t* n_pairs)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (!n_pairs || (n && (!win_len || !pairs || !pair_of_rescue))) return fail(ctx, SDP_EINVAL, "null argument");
    if (n > 0xFFFFFFF0ull) return fail(ctx, SDP_EINVAL, "too many rescues");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->device));
    const size_t N = (size_t)(n ? n : 1);
    Lane& L = ctx->lane[0];                    // scan scratch and mailbox of the first lane (no align call is in flight)
    EN(mp_flag, N * 4); EN(mp_off, N * 8);
    LEN(scan_local[0], N * 4); LEN(scan_tiles[0], (N / 4096 + 2) * 4); LEN(scan_tile_base[0], (N / 4096 + 2) * 8);
    uint32_t nl = 0;
    launch_mate_flags(win_len, n, ctx->mp_flag.as<uint32_t>(), st);
    exclusive_scan_u32_u64(ctx->mp_flag.as<uint32_t>(), n, ctx->mp_off.as<uint64_t>(), L.totals + 2, nullptr,
                           L.scan_local[0].as<uint32_t>(), L.scan_tiles[0].as<uint32_t>(),
                           L.scan_tile_base[0].as<uint64_t>(), st, &nl);
    launch_mate_pairs(ctx->mp_flag.as<uint32_t>(), ctx->mp_off.as<uint64_t>(), n, pairs, pair_of_rescue, st);
    CU(cudaMemcpyAsync(&L.mb->totals[2], L.totals + 2, 8, cudaMemcpyDeviceToHost, st));
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
    *n_pairs = L.mb->totals[2];
    return SDP_OK;
}

int sdp_proper_pairs(sdp_ctx* ctx, const sdp_mates* mates, uint32_t min_insert, uint32_t max_insert, const uint64_t* win_off,
                     const uint32_t* win_len, const uint32_t* pair_of_rescue, const int32_t* ref_start, const int32_t* ref_end,
                     const uint8_t* pass, void* cuda_stream, uint8_t* proper)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (!mates || !win_off || !win_len || !ref_start || !ref_end || !pass || !proper || min_insert > max_insert)
        return fail(ctx, SDP_EINVAL, "null argument or min_insert > max_insert");
    if (mates->n && (!mates->mate_pos || !mates->mate_len || !mates->mate_reverse))
        return fail(ctx, SDP_EINVAL, "null input array");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    CU(cudaSetDevice(ctx->device));
    launch_proper_pairs(*mates, min_insert, max_insert, win_off, win_len, pair_of_rescue, ref_start, ref_end, pass, proper, st);
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
    return SDP_OK;
}

int sdp_align_batch_host(sdp_ctx* ctx, const sdp_batch* hb, sdp_result* out)
{
    if (!ctx) return SDP_EINVAL;
    ctx->err[0] = 0;
    if (!hb || !out) return fail(ctx, SDP_EINVAL, "null batch or result");
    const uint64_t P = hb->n_pairs;
    if (P > 0 && (!hb->reads_packed || !hb->read_off || !hb->read_len || !hb->wins_packed || !hb->win_off ||
                  !hb->win_len || !hb->pairs))
        return fail(ctx, SDP_EINVAL, "null input array");
    CU(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->own_stream;
    sdp_batch d = *hb;
    struct Cp { DevBuf* buf; const void* src; size_t bytes; const void** dst; };
    // the caller's buffers are only guaranteed readable to the end of the last word in use
    const size_t rb = (size_t)((hb->reads_bases + 15) / 16) * 4, wb = (size_t)((hb->wins_bases + 15) / 16) * 4;
    const size_t rnb = (size_t)((hb->reads_bases + 31) / 32) * 4, wnb = (size_t)((hb->wins_bases + 31) / 32) * 4;
    // The small arrays (all the bucket stage needs) go first on the call's stream; the sequences follow on the copy
    // stream, so that they upload beside a1/a2, and the forward pass waits for them.
    Cp cps[] = {
        {&ctx->in_pairs, hb->pairs, (size_t)P * 8, (const void**)&d.pairs},
        {&ctx->in_read_off, hb->read_off, (size_t)hb->n_reads * 8, (const void**)&d.read_off},
        {&ctx->in_read_len, hb->read_len, (size_t)hb->n_reads * 4, (const void**)&d.read_len},
        {&ctx->in_win_off, hb->win_off, (size_t)hb->n_wins * 8, (const void**)&d.win_off},
        {&ctx->in_win_len, hb->win_len, (size_t)hb->n_wins * 4, (const void**)&d.win_len},
        {&ctx->in_reads, hb->reads_packed, rb, (const void**)&d.reads_packed},
        {&ctx->in_read_nmask, hb->read_nmask, rnb, (const void**)&d.read_nmask},
        {&ctx->in_wins, hb->wins_packed, wb, (const void**)&d.wins_packed},
        {&ctx->in_win_nmask, hb->win_nmask, wnb, (const void**)&d.win_nmask},
    };
    // uploads and downloads are in flight from here on: a failure waits for them (and for whatever the pipeline left
    // behind) before it returns, so that the caller may free its buffers and a later call finds the streams idle
    auto hbail = [&](int rc_) { cudaStreamSynchronize(st); cudaStreamSynchronize(ctx->copy_stream); drain(ctx); return rc_; };
#define CUH(call)                                                                                        \
    do {                                                                                                 \
        cudaError_t e_ = (call);                                                                         \
        if (e_ != cudaSuccess)                                                                           \
            return hbail(fail(ctx, e_ == cudaErrorMemoryAllocation ? SDP_ENOMEM : SDP_ECUDA,             \
                              "%s: %s (%s:%d)", #call, cudaGetErrorString(e_), __FILE__, __LINE__));     \
    } while (0)
    int ci = 0;
    for (Cp& c : cps) {
        const cudaStream_t cs = ci++ < 5 ? st : ctx->copy_stream;
        if (!c.src) { *c.dst = nullptr; continue; }
        int rc = ensure(ctx, *c.buf, c.bytes + 64);
        if (rc != SDP_OK) return hbail(rc);
        if (c.bytes) CUH(cudaMemcpyAsync(c.buf->p, c.src, c.bytes, cudaMemcpyHostToDevice, cs));
        *c.dst = c.buf->p;
    }
    CUH(cudaEventRecord(ctx->ev_seq_ready, ctx->copy_stream));
    // per-pair results go into one pinned slab (sized before the call: score and ref_end leave early), the runs into another
    const size_t Pp = (size_t)(P ? P : 1);
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off += (bytes + 63) / 64 * 64; return o; };
    const size_t o_score = carve(Pp * 4), o_rs = carve(Pp * 4), o_re = carve(Pp * 4), o_qs = carve(Pp * 4),
                 o_qe = carve(Pp * 4), o_pass = carve(Pp), o_nm = carve(Pp * 4), o_nc = carve(Pp * 4),
                 o_coff = carve(Pp * 8), o_clen = carve(Pp * 4);
    int rc = ensure_pinned(ctx, ctx->h_out, off);
    if (rc != SDP_OK) return hbail(rc);
    char* h = (char*)ctx->h_out.p;
    sdp_result dr{};
    ctx->wait_seq = true;
    ctx->h_early_score = (int32_t*)(h + o_score); ctx->h_early_ref_end = (int32_t*)(h + o_re);
    rc = sdp_align_batch(ctx, &d, st, &dr);
    ctx->wait_seq = false; ctx->h_early_score = nullptr; ctx->h_early_ref_end = nullptr;
    if (rc != SDP_OK) return hbail(rc);
    const size_t n_ops = (size_t)dr.n_cigar_ops;
    rc = ensure_pinned(ctx, ctx->h_ops, (n_ops + 1) * 4);
    if (rc != SDP_OK) return hbail(rc);
    char* hops = (char*)ctx->h_ops.p;
    if (P) {
        CUH(cudaMemcpyAsync(h + o_rs, dr.ref_start, P * 4, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_qs, dr.read_start, P * 4, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_qe, dr.read_end, P * 4, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_pass, dr.pass, P, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_nm, dr.n_match, P * 4, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_nc, dr.n_cols, P * 4, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_coff, dr.cigar_off, P * 8, cudaMemcpyDeviceToHost, st));
        CUH(cudaMemcpyAsync(h + o_clen, dr.cigar_len, P * 4, cudaMemcpyDeviceToHost, st));
        if (n_ops) CUH(cudaMemcpyAsync(hops, dr.cigar_ops, n_ops * 4, cudaMemcpyDeviceToHost, st));
        CUH(cudaStreamSynchronize(st));
    }
    CUH(cudaStreamSynchronize(ctx->copy_stream));
#undef CUH
    out->score = (const int32_t*)(h + o_score); out->ref_start = (const int32_t*)(h + o_rs);
    out->ref_end = (const int32_t*)(h + o_re); out->read_start = (const int32_t*)(h + o_qs);
    out->read_end = (const int32_t*)(h + o_qe); out->pass = (const uint8_t*)(h + o_pass);
    out->n_match = (const int32_t*)(h + o_nm); out->n_cols = (const int32_t*)(h + o_nc);
    out->cigar_off = (const uint64_t*)(h + o_coff); out->cigar_len = (const uint32_t*)(h + o_clen);
    out->cigar_ops = (const uint32_t*)hops; out->n_cigar_ops = n_ops; out->n_pairs = P;
    return SDP_OK;
}

}  // extern "C"
