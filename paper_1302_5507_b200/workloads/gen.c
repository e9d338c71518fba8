/*
 * gen.c -- seeded synthetic workload generator (inputs only; none of the method's arithmetic).
 *
 * Serves both the CPU oracle and the CUDA path: it writes the packed arrays of the C ABI
 * (include/sdp.h) on the host. The five shapes stand in for the paper's Illumina 100/150 bp
 * paired-end lanes and Mason-simulated 50-250 bp pairs with 500 bp inserts (PAPER.md:79, 85,
 * 452-460), none of which is available; recipes are BASELINE.json "configs" as detailed in
 * DESIGN.md "Input recipe".
 *
 * RNG: xoshiro256** seeded through splitmix64; every pair draws from its own sub-stream
 * splitmix64(seed ^ golden*pair_idx) so generation is independent of order and thread count.
 * Packing: A=0 C=1 G=2 T=3; base k sits in bits 2*(k mod 16) of little-endian uint32 word k/16.
 * N-mask: 1 bit per base (bit k mod 32 of word k/32), set = N.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { uint64_t s[4]; } rng_t;

static inline uint64_t splitmix64(uint64_t* x) {
    uint64_t z = (*x += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
static inline void rng_seed(rng_t* r, uint64_t seed) {
    for (int i = 0; i < 4; ++i) r->s[i] = splitmix64(&seed);
}
static inline uint64_t rotl(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }
static inline uint64_t rng_next(rng_t* r) {
    uint64_t* s = r->s;
    uint64_t result = rotl(s[1] * 5, 7) * 9, t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3]; s[2] ^= t; s[3] = rotl(s[3], 45);
    return result;
}
static inline double rng_unif(rng_t* r) { return (double)(rng_next(r) >> 11) * (1.0 / 9007199254740992.0); }
static inline uint64_t rng_below(rng_t* r, uint64_t n) { return (uint64_t)(rng_unif(r) * (double)n); }
static inline double rng_normal(rng_t* r) {
    double u1 = rng_unif(r), u2 = rng_unif(r);
    if (u1 < 1e-300) u1 = 1e-300;
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586 * u2);
}

static inline unsigned get2(const uint32_t* p, uint64_t k) { return (p[k >> 4] >> (2 * (k & 15))) & 3u; }
static inline void put2(uint32_t* p, uint64_t k, unsigned v) {
    p[k >> 4] = (p[k >> 4] & ~(3u << (2 * (k & 15)))) | ((v & 3u) << (2 * (k & 15)));
}
static inline unsigned getbit(const uint32_t* p, uint64_t k) { return (p[k >> 5] >> (k & 31)) & 1u; }

/*
 * Reference: n_bases i.i.d. uniform ACGT. If nmask != NULL, alternate clean stretches
 * (geometric, mean n_clean_mean) and N runs (geometric, mean n_run_mean) and set mask bits
 * (config 5: about 10 % N with 4500 / 500). packed has ceil(n_bases/16)+4 words, nmask
 * ceil(n_bases/32)+4 words, both zero-initialised by the caller.
 */
void sdpgen_reference(uint64_t seed, uint64_t n_bases, uint32_t* packed, uint32_t* nmask,
                      double n_clean_mean, double n_run_mean)
{
    rng_t r; rng_seed(&r, seed ^ 0xA5A5A5A5DEADBEEFULL);
    uint64_t words = (n_bases + 15) / 16;
    for (uint64_t w = 0; w + 1 < words; w += 2) {
        uint64_t x = rng_next(&r);
        packed[w] = (uint32_t)x; packed[w + 1] = (uint32_t)(x >> 32);
    }
    if (words & 1) packed[words - 1] = (uint32_t)rng_next(&r);
    if (n_bases & 15) packed[words - 1] &= (1u << (2 * (n_bases & 15))) - 1u;
    if (nmask) {
        uint64_t pos = 0; int in_n = 0;
        while (pos < n_bases) {
            double mean = in_n ? n_run_mean : n_clean_mean;
            double u = rng_unif(&r); if (u < 1e-300) u = 1e-300;
            uint64_t len = 1 + (uint64_t)(-log(u) * mean);
            if (pos + len > n_bases) len = n_bases - pos;
            if (in_n) for (uint64_t k = pos; k < pos + len; ++k) nmask[k >> 5] |= 1u << (k & 31);
            pos += len; in_n = !in_n;
        }
    }
}

typedef struct {
    int32_t  cfg;              /* 1..5: BASELINE.json config number                              */
    uint64_t seed;
    uint64_t n_pairs;
    uint64_t ref_bases;
    int32_t  read_len_min, read_len_max;  /* n ~ U{min..max}                                      */
    int32_t  win_len;          /* m when > 0; otherwise m = n + win_extra                         */
    int32_t  win_extra;
    int32_t  private_windows;  /* 1: windows are copied into wins_out (config 3)                  */
    double   random_frac;      /* fraction of uniform random ("unplaceable") reads                */
    double   sub_lo, sub_hi;   /* substitution rate at read position 0 and n-1 (linear between)   */
    double   indel_rate;       /* indel starts per base; insertion / deletion 50:50               */
    double   indel_geom_p;     /* > 0: length ~ geometric(p) capped at indel_max; 0: U{1..max}    */
    int32_t  indel_max;
    int32_t  start_mode;       /* 0: uniform in [0, m-n]; 1: start_center + round(N(0, start_sd)) */
    int32_t  start_center;     /*    clipped to [0, m-n]                                          */
    double   start_sd;
    double   tandem_frac;      /* fraction of windows given a tandem-repeat block (config 3)      */
    int32_t  divergence_mode;  /* 1: per-read d ~ U(div_lo, div_hi); sub = .8 d; indel = .2 d/15.5 */
    double   div_lo, div_hi;
} sdpgen_params;

static int draw_indel_len(rng_t* r, const sdpgen_params* P) {
    if (P->indel_geom_p > 0.0) {
        int len = 1;
        while (len < P->indel_max && rng_unif(r) >= P->indel_geom_p) ++len;
        return len;
    }
    return 1 + (int)rng_below(r, (uint64_t)P->indel_max);
}

/*
 * Outputs (caller allocates, zero-initialised):
 *   read_len[P], read_off[P] (bases, dense back to back), reads_packed (enough words for the
 *   total, see sdpgen_read_bases), win_off[P], win_len[P]; for private windows wins_out
 *   receives dense copies, otherwise windows are views into ref_packed (win_off = position).
 * Lengths must be drawn first (sdpgen_lengths) so offsets are known; this keeps generation
 * order-independent.
 */
void sdpgen_lengths(const sdpgen_params* P, uint32_t* read_len, uint64_t* read_off,
                    uint32_t* win_len, uint64_t* win_off_private, uint64_t* total_read_bases,
                    uint64_t* total_win_bases)
{
    uint64_t ro = 0, wo = 0;
    for (uint64_t p = 0; p < P->n_pairs; ++p) {
        uint64_t s = P->seed ^ (0x9E3779B97F4A7C15ULL * (p + 1));
        rng_t r; rng_seed(&r, s);
        int n = P->read_len_min + (int)rng_below(&r, (uint64_t)(P->read_len_max - P->read_len_min + 1));
        int m = P->win_len > 0 ? P->win_len : n + P->win_extra;
        read_len[p] = (uint32_t)n; read_off[p] = ro; ro += (uint64_t)n;
        win_len[p] = (uint32_t)m;
        if (win_off_private) { win_off_private[p] = wo; }
        wo += (uint64_t)m;
    }
    *total_read_bases = ro; *total_win_bases = wo;
}

void sdpgen_pairs(const sdpgen_params* P, const uint32_t* ref_packed, const uint32_t* ref_nmask,
                  const uint32_t* read_len, const uint64_t* read_off, uint32_t* reads_packed,
                  const uint32_t* win_len, uint64_t* win_off, uint32_t* wins_out)
{
    /* reads are dense, so two pairs can share a 32-bit word: generate into private byte
     * buffers in parallel, pack serially afterwards in chunks */
    const uint64_t CH = 1u << 16;
    uint8_t* rbuf = NULL; uint8_t* wbuf = NULL;
    int nmax = P->read_len_max, mmax = P->win_len > 0 ? P->win_len : P->read_len_max + P->win_extra;
    rbuf = (uint8_t*)malloc((size_t)CH * (size_t)nmax);
    if (P->private_windows) wbuf = (uint8_t*)malloc((size_t)CH * (size_t)mmax);
    for (uint64_t base = 0; base < P->n_pairs; base += CH) {
        uint64_t cnt = P->n_pairs - base < CH ? P->n_pairs - base : CH;
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
        for (int64_t q = 0; q < (int64_t)cnt; ++q) {
            uint64_t p = base + (uint64_t)q;
            uint64_t s = P->seed ^ (0x9E3779B97F4A7C15ULL * (p + 1));
            rng_t r; rng_seed(&r, s);
            (void)rng_next(&r);                       /* the draw sdpgen_lengths used */
            int n = (int)read_len[p], m = (int)win_len[p];
            uint8_t* R = rbuf + (size_t)q * (size_t)nmax;
            uint8_t* Wp = wbuf ? wbuf + (size_t)q * (size_t)mmax : NULL;
            uint64_t w0 = rng_below(&r, P->ref_bases - (uint64_t)m + 1);
            if (!P->private_windows) win_off[p] = w0;
            if (Wp) {
                for (int k = 0; k < m; ++k) Wp[k] = (uint8_t)get2(ref_packed, w0 + (uint64_t)k);
                if (rng_unif(&r) < P->tandem_frac) {      /* tandem-repeat block, period 2..6 */
                    int blen = 20 + (int)rng_below(&r, 41), per = 2 + (int)rng_below(&r, 5);
                    int bpos = (int)rng_below(&r, (uint64_t)(m - blen + 1));
                    uint8_t unit[6];
                    for (int k = 0; k < per; ++k) unit[k] = (uint8_t)rng_below(&r, 4);
                    for (int k = 0; k < blen; ++k) Wp[bpos + k] = unit[k % per];
                }
            }
            int is_random = rng_unif(&r) < P->random_frac;
            int start;
            if (P->start_mode == 1) {
                double x = (double)P->start_center + floor(rng_normal(&r) * P->start_sd + 0.5);
                start = (int)x;
                if (start < 0) start = 0;
                if (start > m - n) start = m - n;
                if (start < 0) start = 0;
            } else {
                start = m > n ? (int)rng_below(&r, (uint64_t)(m - n + 1)) : 0;
            }
            double sub_lo = P->sub_lo, sub_hi = P->sub_hi, indel = P->indel_rate;
            if (P->divergence_mode) {
                double d = P->div_lo + (P->div_hi - P->div_lo) * rng_unif(&r);
                sub_lo = sub_hi = 0.8 * d; indel = 0.2 * d / 15.5;
            }
            if (is_random) {
                for (int k = 0; k < n; ++k) R[k] = (uint8_t)rng_below(&r, 4);
            } else {
                /* walk the source (window copy, then the reference after it) from `start` */
                int64_t src = start; int j = 0;
                while (j < n) {
                    if (rng_unif(&r) < indel) {
                        int len = draw_indel_len(&r, P);
                        if (rng_unif(&r) < 0.5) {          /* insertion into the read */
                            for (int k = 0; k < len && j < n; ++k) R[j++] = (uint8_t)rng_below(&r, 4);
                        } else {                            /* deletion from the read */
                            src += len;
                        }
                        continue;
                    }
                    unsigned b; int isn = 0;
                    uint64_t gpos = w0 + (uint64_t)src;
                    if (Wp && src < m) b = Wp[src];
                    else if (gpos < P->ref_bases) { b = get2(ref_packed, gpos); isn = ref_nmask ? (int)getbit(ref_nmask, gpos) : 0; }
                    else b = (unsigned)rng_below(&r, 4);
                    if (isn) b = (unsigned)rng_below(&r, 4);   /* a sequencer never emits the reference's N */
                    double ps = n > 1 ? sub_lo + (sub_hi - sub_lo) * (double)j / (double)(n - 1) : sub_lo;
                    if (rng_unif(&r) < ps) b = (b + 1 + (unsigned)rng_below(&r, 3)) & 3u;
                    R[j++] = (uint8_t)b; ++src;
                }
            }
        }
        for (uint64_t q = 0; q < cnt; ++q) {
            uint64_t p = base + q;
            const uint8_t* R = rbuf + (size_t)q * (size_t)nmax;
            for (uint32_t k = 0; k < read_len[p]; ++k) put2(reads_packed, read_off[p] + k, R[k]);
            if (wbuf) {
                const uint8_t* Wp = wbuf + (size_t)q * (size_t)mmax;
                for (uint32_t k = 0; k < win_len[p]; ++k) put2(wins_out, win_off[p] + k, Wp[k]);
            }
        }
    }
    free(rbuf); free(wbuf);
}
