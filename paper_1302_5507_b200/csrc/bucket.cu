// bucket.cu -- a1 (ingest + validate) and a2 (device-side length bucketing) of the hot path, plus
// the generic pieces the later stages reuse: key histogram, bin scan, scatter into bucket order,
// per-read-length task table, and a large exclusive scan.
//
// The paper's analogue is grouping reads by 32 so warp loads coalesce and running
// work of different complexity classes separately; here pairs are binned by
// (read length, rows >> 6) so that the lanes of one warp walk the same number of DP rows.
#include "sdp_host.cuh"
#include "seq_bits.cuh"

namespace sdp {

// ---------------------------------------------------------------------------------------------
// Optional ungapped pre-pass (sdp_set_prefilter; the analogue of the paper's step 1, for one window).
// A gapped alignment scores at most n*match - (o + e). If the best gap-free placement of the read in the window
// has x mismatches with x*(match - mismatch) < o + e, its score n*match - x*(match - mismatch) beats every gapped
// alignment, so it is the optimum, and the lowest offset reaching x is the lowest maximising end row: score and
// ref_end without any DP. Word-parallel Hamming scan over all m - n + 1 offsets with early exit. Returns false
// when no placement has few enough mismatches (the pair then takes the DP).
__device__ bool ungapped_optimum(const sdp_batch& b, const Scoring& sc, uint64_t ro, uint64_t wo, int n, int m,
                                 int32_t* score, int32_t* ref_end)
{
    const int delta = sc.match - sc.mismatch;
    const int xmax = (sc.gap_open + sc.gap_extend + delta - 1) / delta - 1;     // largest x with x*delta < o + e
    if (xmax < 0 || n > m) return false;
    const long long rwords = (long long)((b.reads_bases + 15) / 16), wwords = (long long)((b.wins_bases + 15) / 16);
    const long long rnwords = (long long)((b.reads_bases + 31) / 32), wnwords = (long long)((b.wins_bases + 31) / 32);
    int best_x = xmax + 1, best_s = -1;
    // first 16 read bases in a register, the window as a sliding 32-base buffer: one shift, XOR and popcount per
    // offset reject almost every placement; only the survivors look at the rest of the read
    const int cnt0 = min(16, n);
    const uint32_t mask0 = cnt0 < 16 ? (1u << (2 * cnt0)) - 1u : 0xFFFFFFFFu;
    const uint32_t r0 = bases16(b.reads_packed, (long long)ro, rwords);
    const uint32_t rn0 = nbits16_spread(b.read_nmask, (long long)ro, rnwords);
    uint64_t wb = 0, wnb = 0;
    for (int s = 0; s + n <= m; ++s) {
        const int k = s & 15;
        if (k == 0) {
            wb = (uint64_t)bases16(b.wins_packed, (long long)wo + s, wwords) |
                 ((uint64_t)bases16(b.wins_packed, (long long)wo + s + 16, wwords) << 32);
            if (b.win_nmask != nullptr)
                wnb = (uint64_t)nbits16_spread(b.win_nmask, (long long)wo + s, wnwords) |
                      ((uint64_t)nbits16_spread(b.win_nmask, (long long)wo + s + 16, wnwords) << 32);
        }
        const int limit = best_x - 1;                     // only a strictly better placement replaces an earlier one
        int x = cnt0 - __popc(eq16(r0, (uint32_t)(wb >> (2 * k)), rn0 | (uint32_t)(wnb >> (2 * k))) & mask0);
        for (int j0 = 16; j0 < n && x <= limit; j0 += 16) {
            const uint32_t r = bases16(b.reads_packed, (long long)ro + j0, rwords);
            const uint32_t t = bases16(b.wins_packed, (long long)wo + s + j0, wwords);
            const uint32_t nm = nbits16_spread(b.read_nmask, (long long)ro + j0, rnwords) |
                                nbits16_spread(b.win_nmask, (long long)wo + s + j0, wnwords);
            uint32_t eq = eq16(r, t, nm);
            const int cnt = min(16, n - j0);
            if (cnt < 16) eq &= (1u << (2 * cnt)) - 1u;
            x += cnt - __popc(eq);
        }
        if (x <= limit) { best_x = x; best_s = s; if (x == 0) break; }
    }
    if (best_s < 0) return false;
    *score = sc.match * n - best_x * delta;
    *ref_end = best_s + n - 1;
    return true;
}

// ---------------------------------------------------------------------------------------------
// a1: validate every pair and emit its bucket key. One thread per pair.
__global__ void k_validate_key(const sdp_batch b, const Scoring sc, uint32_t* __restrict__ keys,
                               uint32_t* __restrict__ pn, uint32_t* __restrict__ pm,
                               uint32_t* __restrict__ hist, uint32_t* __restrict__ err_flag,
                               unsigned long long* __restrict__ cells, int prefilter,
                               int32_t* __restrict__ score, int32_t* __restrict__ ref_end,
                               unsigned long long* __restrict__ cells_skipped, int local,
                               uint32_t* __restrict__ slow_words, unsigned long long* __restrict__ slow_total)
{
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t key = SDP_KEY_SKIP, err = 0, slow = 0;
    unsigned long long my_cells = 0;
    if (p < b.n_pairs) {
        const uint32_t ri = b.pairs[2 * p], wi = b.pairs[2 * p + 1];
        if (ri >= b.n_reads || wi >= b.n_wins) err = SDP_ERRF_INDEX;
        else {
            const uint32_t n = b.read_len[ri], m = b.win_len[wi];
            const uint64_t ro = b.read_off[ri], wo = b.win_off[wi];
            if (n < 1 || m < 1 || ro + n > b.reads_bases || wo + m > b.wins_bases || ro + n < ro || wo + m < wo)
                err = SDP_ERRF_INDEX;
            else if (n > SDP_MAX_SEQ_LEN || m > SDP_MAX_SEQ_LEN)
                err = SDP_ERRF_RANGE;                      // beyond even the int32 lane
            else if ((long long)sc.match * n + (long long)sc.gap_extend * ((long long)n + 2) + 2LL * sc.gap_open -
                             (long long)sc.mismatch >= SDP_MAX_CELL_VALUE_I32)
                // the int32 lane's minus infinity is -2^28 (traceback) / -2^29 (forward): every real cell value lies
                // in [-(2*gap_open + gap_extend*(n+1)), match*n], and a sentinel plus up to n matches must stay below
                // that range, or an out-of-band cell would beat a real one (sdp.h, int32 range rule)
                err = SDP_ERRF_RANGE;
            else if (local || n > SDP_MAX_READ_LEN ||
                     (long long)sc.match * n + (long long)sc.gap_extend * ((long long)n + m + 32) + 3LL * sc.gap_open + 8 +
                             llabs(2LL * sc.gap_extend + sc.mismatch) > SDP_MAX_CELL_VALUE) {
                // outside the int16 kernels' domain (or local mode): the int32 lane (slow_lane.cu) takes the pair; it
                // never enters the forward buckets. slow_words = its two row arrays of n + 1 entries when the read is
                // longer than SDP_MAX_READ_LEN (k_forward_i32); up to that length the warp kernels keep the rows in
                // registers and the word is only the "took the int32 lane" flag (local mode on a full batch would
                // otherwise reserve gigabytes nobody touches).
                pn[p] = n; pm[p] = m;
                my_cells = (unsigned long long)n * m;
                slow = n > SDP_MAX_READ_LEN ? 2u * (n + 1u) : 1u;
            } else {
                key = (n - 1) * 64u + min(63u, m >> 6);
                pn[p] = n; pm[p] = m;
                my_cells = (unsigned long long)n * m;
                int32_t s_u, e_u;
                if (prefilter && ungapped_optimum(b, sc, ro, wo, (int)n, (int)m, &s_u, &e_u)) {
                    score[p] = s_u; ref_end[p] = e_u;     // no DP for this pair: it never enters the forward buckets
                    key = SDP_KEY_SKIP;
                    atomicAdd(cells_skipped, my_cells);
                    my_cells = 0;
                }
            }
        }
        keys[p] = key;
        slow_words[p] = slow;
    }
    if (err) atomicOr(err_flag, err);
    // histogram: the key of the block's first thread is counted per block (a uniform batch would otherwise serialise
    // one atomic per warp on a single bin, see k_scatter), every other key per warp
    {
        __shared__ uint32_t s_key;
        if (threadIdx.x == 0) s_key = key;
        __syncthreads();
        const uint32_t bkey = s_key;
        const bool same = key == bkey && key != SDP_KEY_SKIP;
        const int n_same = __syncthreads_count(same ? 1 : 0);
        if (threadIdx.x == 0 && n_same) atomicAdd(hist + bkey, (uint32_t)n_same);
        const bool other = !same && key != SDP_KEY_SKIP;
        const uint32_t active = __ballot_sync(0xffffffffu, other);
        if (other) {
            const uint32_t peers = __match_any_sync(active, key);
            if ((threadIdx.x & 31) == (uint32_t)(__ffs(peers) - 1)) atomicAdd(hist + key, (uint32_t)__popc(peers));
        }
    }
    // cells and int32-lane words: one atomic each per block
    {
        __shared__ unsigned long long s_cells[8], s_slow[8];
        unsigned long long my_slow = slow;
        for (int o = 16; o > 0; o >>= 1) {
            my_cells += __shfl_down_sync(0xffffffffu, my_cells, o);
            my_slow += __shfl_down_sync(0xffffffffu, my_slow, o);
        }
        if ((threadIdx.x & 31) == 0) { s_cells[threadIdx.x >> 5] = my_cells; s_slow[threadIdx.x >> 5] = my_slow; }
        __syncthreads();
        if (threadIdx.x == 0) {
            unsigned long long t = 0, u = 0;
            for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { t += s_cells[k]; u += s_slow[k]; }
            if (t) atomicAdd(cells, t);
            if (u) atomicAdd(slow_total, u);
        }
    }
}

// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t block_exclusive_scan_1024(uint32_t v, uint32_t* total)
{
    __shared__ uint32_t warp_sums[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint32_t x = v;
    for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) warp_sums[w] = x;
    __syncthreads();
    if (w == 0) {
        uint32_t s = warp_sums[lane];
        for (int o = 1; o < 32; o <<= 1) { uint32_t y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        warp_sums[lane] = s;
    }
    __syncthreads();
    const uint32_t base = w ? warp_sums[w - 1] : 0u;
    if (total) *total = warp_sums[31];
    __syncthreads();
    return base + x - v;
}

// exclusive scan of the SDP_NBINS histogram in two launches of SDP_NBINS / 4096 blocks (a single
// block took 115 us per sort, four sorts per call). Phase 1: every block scans 4096 bins (one
// coalesced uint4 per thread) and leaves its total in tile_sums. Phase 2: every block adds the
// totals of the tiles before it; bin_start[SDP_NBINS] = grand total; hist is left holding a copy
// of bin_start (the scatter cursors).
constexpr int BIN_TILE = 4096;
constexpr int BIN_TILES = SDP_NBINS / BIN_TILE;
static_assert(SDP_NBINS % BIN_TILE == 0 && BIN_TILES <= SDP_BIN_SCRATCH, "bin scan tiling");

__global__ void __launch_bounds__(1024) k_scan_bins_tiles(const uint32_t* __restrict__ hist,
                                                          uint32_t* __restrict__ bin_start,
                                                          uint32_t* __restrict__ tile_sums)
{
    const uint32_t base = blockIdx.x * BIN_TILE + threadIdx.x * 4;
    const uint4 v = *reinterpret_cast<const uint4*>(hist + base);
    uint32_t total;
    const uint32_t run = block_exclusive_scan_1024(v.x + v.y + v.z + v.w, &total);
    *reinterpret_cast<uint4*>(bin_start + base) = make_uint4(run, run + v.x, run + v.x + v.y, run + v.x + v.y + v.z);
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(1024) k_scan_bins_finish(uint32_t* __restrict__ hist, uint32_t* __restrict__ bin_start,
                                                           const uint32_t* __restrict__ tile_sums)
{
    uint32_t before = 0, all = 0;
#pragma unroll
    for (int t = 0; t < BIN_TILES; ++t) { const uint32_t x = tile_sums[t]; all += x; if (t < (int)blockIdx.x) before += x; }
    const uint32_t base = blockIdx.x * BIN_TILE + threadIdx.x * 4;
    uint4 v = *reinterpret_cast<const uint4*>(bin_start + base);
    v.x += before; v.y += before; v.z += before; v.w += before;
    *reinterpret_cast<uint4*>(bin_start + base) = v;
    *reinterpret_cast<uint4*>(hist + base) = v;
    if (blockIdx.x == 0 && threadIdx.x == 0) bin_start[SDP_NBINS] = all;
}

// scatter pair indices into bucket order (order inside one bin is not deterministic; no result
// depends on it because every pair is aligned independently and written back by caller index)
// A batch of one read length and one window length puts every pair into ONE bin: a warp-aggregated atomic per warp
// then serialises on that bin's cursor (31,250 atomics on one address for a million pairs: 75 us). So the key of the
// block's first thread is handled per BLOCK (one atomic for all threads that share it, positions from a ballot /
// warp-count scan); every other key takes the warp-aggregated path.
// DESC: the forward sort. Instead of the pair's index the thread writes the pair's forward descriptor straight to its
// place in bucket order (one kernel and one pass over `order` less than scatter + gather).
template <bool DESC>
__global__ void __launch_bounds__(256) k_scatter(const uint32_t* __restrict__ keys, uint64_t n, uint32_t* __restrict__ cursor,
                                                 uint32_t* __restrict__ order, const sdp_batch b, PairDesc* __restrict__ desc)
{
    auto put = [&](const uint32_t pos, const uint64_t pp) {
        if (DESC) {
            const uint32_t ri = b.pairs[2 * pp], wi = b.pairs[2 * pp + 1];
            PairDesc d;
            d.roff = b.read_off[ri]; d.woff = b.win_off[wi];
            d.n = b.read_len[ri]; d.m = b.win_len[wi]; d.pid = (uint32_t)pp; d.aux = 0;
            desc[pos] = d;
        } else order[pos] = (uint32_t)pp;
    };
    __shared__ uint32_t s_key, s_base, s_wcnt[8];
    const uint64_t p = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t key = p < n ? keys[p] : SDP_KEY_SKIP;
    const uint32_t lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) s_key = key;
    __syncthreads();
    const uint32_t bkey = s_key;
    const bool same = key == bkey && key != SDP_KEY_SKIP;
    const uint32_t same_mask = __ballot_sync(0xffffffffu, same);
    if (lane == 0) s_wcnt[w] = (uint32_t)__popc(same_mask);
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t total = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) total += s_wcnt[k];
        s_base = total ? atomicAdd(cursor + bkey, total) : 0u;
    }
    __syncthreads();
    if (same) {
        uint32_t pre = 0;
#pragma unroll
        for (int k = 0; k < 8; ++k) pre += (k < (int)w) ? s_wcnt[k] : 0u;
        put(s_base + pre + (uint32_t)__popc(same_mask & ((1u << lane) - 1u)), p);
    }
    const bool other = !same && key != SDP_KEY_SKIP;
    const uint32_t active = __ballot_sync(0xffffffffu, other);
    if (other) {
        const uint32_t peers = __match_any_sync(active, key);
        const int leader = __ffs(peers) - 1;
        uint32_t base = 0;
        if (lane == (uint32_t)leader) base = atomicAdd(cursor + key, (uint32_t)__popc(peers));
        base = __shfl_sync(peers, base, leader);
        put(base + (uint32_t)__popc(peers & ((1u << lane) - 1u)), p);
    }
}

// ---------------------------------------------------------------------------------------------
// task table: slot t (K-major order, host-built table slot_n/slot_G/slot_K) -> its pairs and the
// running number of warp tasks. One 1024-thread block.
__global__ void __launch_bounds__(1024) k_tasks(const uint32_t* __restrict__ bin_start,
                                                const uint16_t* __restrict__ slot_n,
                                                const uint16_t* __restrict__ slot_G,
                                                const uint16_t* __restrict__ slot_K,
                                                SlotInfo* __restrict__ slots, uint32_t* __restrict__ task_prefix,
                                                uint32_t* __restrict__ host_prefix, uint32_t* __restrict__ host_total)
{
    const int t = threadIdx.x;
    const uint32_t n = slot_n[t];
    const uint32_t first = bin_start[(n - 1) * 64u];
    const uint32_t count = bin_start[n * 64u] - first;
    const uint32_t G = slot_G[t];
    const uint32_t ppw = 2u * (32u / G);
    const uint32_t ntasks = (count + ppw - 1) / ppw;
    uint32_t total;
    const uint32_t pre = block_exclusive_scan_1024(ntasks, &total);
    SlotInfo si; si.first = first; si.count = count; si.n = n; si.G = (uint16_t)G; si.K = slot_K[t];
    slots[t] = si;
    task_prefix[t] = pre;
    host_prefix[t] = pre;                                 // pinned host mailbox: the host sizes the launches from it
    if (t == 0) { task_prefix[SDP_NSLOTS] = total; host_prefix[SDP_NSLOTS] = total; *host_total = bin_start[SDP_NBINS]; }
}

// ---------------------------------------------------------------------------------------------
// large exclusive scan uint32 -> uint64 (cigar offsets, scratch offsets): 3 phases
constexpr int SCAN_PER = 4;                       // elements per thread
constexpr int SCAN_TILE = 1024 * SCAN_PER;

__global__ void __launch_bounds__(1024) k_scan_tiles(const uint32_t* __restrict__ in, uint64_t n,
                                                     uint32_t* __restrict__ local_out, uint32_t* __restrict__ tile_sums)
{
    const uint64_t base = (uint64_t)blockIdx.x * SCAN_TILE + (uint64_t)threadIdx.x * SCAN_PER;
    uint32_t v[SCAN_PER], sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_PER; ++k) { v[k] = (base + k < n) ? in[base + k] : 0u; sum += v[k]; }
    uint32_t total;
    uint32_t run = block_exclusive_scan_1024(sum, &total);
#pragma unroll
    for (int k = 0; k < SCAN_PER; ++k) { if (base + k < n) local_out[base + k] = run; run += v[k]; }
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = total;
}

// 64-bit variant for the tile sums (1024 tile sums of up to 2^32 - 1 each do not fit 32 bits)
__device__ __forceinline__ uint64_t block_exclusive_scan_1024_u64(uint64_t v, uint64_t* total)
{
    __shared__ uint64_t warp_sums64[32];
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    uint64_t x = v;
    for (int o = 1; o < 32; o <<= 1) { uint64_t y = __shfl_up_sync(0xffffffffu, x, o); if (lane >= o) x += y; }
    if (lane == 31) warp_sums64[w] = x;
    __syncthreads();
    if (w == 0) {
        uint64_t s = warp_sums64[lane];
        for (int o = 1; o < 32; o <<= 1) { uint64_t y = __shfl_up_sync(0xffffffffu, s, o); if (lane >= o) s += y; }
        warp_sums64[lane] = s;
    }
    __syncthreads();
    const uint64_t base = w ? warp_sums64[w - 1] : 0ull;
    if (total) *total = warp_sums64[31];
    __syncthreads();
    return base + x - v;
}

// base_in (may be null): the scan starts from *base_in instead of 0, and the total includes it
__global__ void __launch_bounds__(1024) k_scan_tile_sums(const uint32_t* __restrict__ tile_sums, uint32_t ntiles,
                                                         uint64_t* __restrict__ tile_base, uint64_t* __restrict__ total_out,
                                                         const uint64_t* __restrict__ base_in)
{
    __shared__ uint64_t carry;
    if (threadIdx.x == 0) carry = base_in ? *base_in : 0ull;
    __syncthreads();
    for (uint32_t start = 0; start < ntiles; start += 1024) {
        const uint32_t idx = start + threadIdx.x;
        const uint64_t v = idx < ntiles ? (uint64_t)tile_sums[idx] : 0ull;
        uint64_t total;
        const uint64_t pre = block_exclusive_scan_1024_u64(v, &total);
        if (idx < ntiles) tile_base[idx] = carry + pre;
        __syncthreads();
        if (threadIdx.x == 0) carry += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) *total_out = carry;
}

__global__ void k_scan_add(const uint32_t* __restrict__ local, const uint64_t* __restrict__ tile_base, uint64_t n,
                           uint64_t* __restrict__ out)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = tile_base[i / SCAN_TILE] + local[i];
}

// n <= SCAN_TILE: the three phases in one block, 64-bit throughout (small batches are launch-bound: one launch
// instead of three)
__global__ void __launch_bounds__(1024) k_scan_small(const uint32_t* __restrict__ in, uint32_t n, uint64_t* __restrict__ out,
                                                     uint64_t* __restrict__ total_out, const uint64_t* __restrict__ base_in)
{
    const uint32_t base = threadIdx.x * SCAN_PER;
    uint32_t v[SCAN_PER];
    uint64_t sum = 0;
#pragma unroll
    for (int k = 0; k < SCAN_PER; ++k) { v[k] = (base + k < n) ? in[base + k] : 0u; sum += v[k]; }
    uint64_t total;
    uint64_t run = block_exclusive_scan_1024_u64(sum, &total) + (base_in ? *base_in : 0ull);
#pragma unroll
    for (int k = 0; k < SCAN_PER; ++k) { if (base + k < n) out[base + k] = run; run += v[k]; }
    if (threadIdx.x == 0) *total_out = total + (base_in ? *base_in : 0ull);
}

void exclusive_scan_u32_u64(const uint32_t* in, uint64_t n, uint64_t* out, uint64_t* total_dev, const uint64_t* base_dev,
                            uint32_t* tmp_local, uint32_t* tmp_tiles, uint64_t* tmp_tile_base,
                            cudaStream_t st, uint32_t* launches)
{
    if (n <= (uint64_t)SCAN_TILE) {
        k_scan_small<<<1, 1024, 0, st>>>(in, (uint32_t)n, out, total_dev, base_dev);
        *launches += 1;
        return;
    }
    const uint32_t ntiles = (uint32_t)((n + SCAN_TILE - 1) / SCAN_TILE);
    if (n) k_scan_tiles<<<ntiles, 1024, 0, st>>>(in, n, tmp_local, tmp_tiles);
    k_scan_tile_sums<<<1, 1024, 0, st>>>(tmp_tiles, ntiles, tmp_tile_base, total_dev, base_dev);
    if (n) k_scan_add<<<(uint32_t)((n + 255) / 256), 256, 0, st>>>(tmp_local, tmp_tile_base, n, out);
    *launches += n ? 3 : 1;
}

// ---------------------------------------------------------------------------------------------
// everything else the host needs after the post-forward bookkeeping, written straight into the pinned
// mailbox by one small kernel (instead of some twenty 4-byte copies)
__global__ void k_mailbox(const uint32_t* __restrict__ tb_bin_start, uint32_t stride, uint32_t nbounds,
                          const uint64_t* __restrict__ totals, const unsigned long long* __restrict__ counters,
                          uint32_t* __restrict__ host_bounds, uint64_t* __restrict__ host_totals,
                          unsigned long long* __restrict__ host_counters)
{
    const uint32_t t = threadIdx.x;
    if (t < nbounds) host_bounds[t] = tb_bin_start[(size_t)t * stride];
    if (t < 4) host_totals[t] = totals[t];
    if (t < 8) host_counters[t] = counters[t];
}

void launch_mailbox(const uint32_t* tb_bin_start, uint32_t stride, uint32_t nbounds, const uint64_t* totals,
                    const unsigned long long* counters, uint32_t* host_bounds, uint64_t* host_totals,
                    unsigned long long* host_counters, cudaStream_t st)
{
    k_mailbox<<<1, 64, 0, st>>>(tb_bin_start, stride, nbounds, totals, counters, host_bounds, host_totals, host_counters);
}

// ---------------------------------------------------------------------------------------------
// host wrappers
void launch_validate_key(const sdp_batch& b, const Scoring& sc, uint32_t* keys, uint32_t* pn, uint32_t* pm,
                         uint32_t* hist, uint32_t* err_flag, unsigned long long* cells, int prefilter, int32_t* score,
                         int32_t* ref_end, unsigned long long* cells_skipped, int local, uint32_t* slow_words,
                         unsigned long long* slow_total, cudaStream_t st)
{
    const uint32_t grid = (uint32_t)((b.n_pairs + 255) / 256);
    k_validate_key<<<grid, 256, 0, st>>>(b, sc, keys, pn, pm, hist, err_flag, cells, prefilter, score, ref_end, cells_skipped,
                                         local, slow_words, slow_total);
}

void launch_sort_tail(const uint32_t* keys, uint64_t n, uint32_t* hist, uint32_t* bin_start, uint32_t* order,
                      const uint16_t* slot_n, const uint16_t* slot_G, const uint16_t* slot_K,
                      SlotInfo* slots, uint32_t* task_prefix, uint32_t* host_prefix, uint32_t* host_total, cudaStream_t st,
                      const sdp_batch* b_desc, PairDesc* desc)
{
    uint32_t* tile_sums = bin_start + SDP_NBINS + 4;        // scratch behind the total (SDP_BIN_SCRATCH words)
    k_scan_bins_tiles<<<BIN_TILES, 1024, 0, st>>>(hist, bin_start, tile_sums);
    k_scan_bins_finish<<<BIN_TILES, 1024, 0, st>>>(hist, bin_start, tile_sums);
    if (b_desc) k_scatter<true><<<(uint32_t)((n + 255) / 256), 256, 0, st>>>(keys, n, hist, order, *b_desc, desc);
    else        k_scatter<false><<<(uint32_t)((n + 255) / 256), 256, 0, st>>>(keys, n, hist, order, sdp_batch{}, nullptr);
    if (slots) k_tasks<<<1, 1024, 0, st>>>(bin_start, slot_n, slot_G, slot_K, slots, task_prefix, host_prefix, host_total);
}

}  // namespace sdp
