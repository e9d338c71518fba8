// score_cubin.cu -- DEVICE CODE ONLY: the forward / reverse score kernels (score_kernel.cuh) for K in
// [SDP_K_LO, SDP_K_HI], compiled to a cubin (nvcc -cubin) once per K range. The scoring constants of the column
// loop are sentinel immediates; score_modules.cu patches them with a context's scoring and loads the image
// (DESIGN.md "Immediate patching"). Kernel names are plain C so that the loader can ask for them by name:
//     sdp_score_k<K>_<f|r><e|p>     f = forward, r = reverse;  e = read length == G*K, p = padded
//     sdp_trace_k<K>_<e|p>          the traceback DP kernel (trace_kernel.cuh), same treatment
#include "trace_kernel.cuh"

#if !defined(SDP_K_LO) || !defined(SDP_K_HI)
#error "define SDP_K_LO and SDP_K_HI"
#endif

#define SDP_CAT3_(a, b, c) a##b##c
#define SDP_CAT3(a, b, c) SDP_CAT3_(a, b, c)
#define SDP_DEFINE_SCORE(K, SUFFIX, REV, PAD)                                                              \
    extern "C" __global__ void __launch_bounds__(SDP_SCORE_THREADS, SDP_SCORE_MIN_CTAS(K))                 \
    SDP_CAT3(sdp_score_k, K, SUFFIX)(const ScoreParams P)                                                  \
    {                                                                                                      \
        __shared__ __align__(16) uint32_t ring_mem[SDP_WARPS_PER_CTA][SDP_RING_WORDS];                                 \
        sdp::score_body<K, REV, PAD>(P, ring_mem);                                                         \
    }
#define SDP_DEFINE_TRACE(K, SUFFIX, PAD)                                                                   \
    extern "C" __global__ void __launch_bounds__(SDP_SCORE_THREADS, SDP_SCORE_MIN_CTAS(K))                 \
    SDP_CAT3(sdp_trace_k, K, SUFFIX)(const ScoreParams P, const TraceDP T)                                 \
    {                                                                                                      \
        __shared__ __align__(16) uint32_t ring_mem[SDP_WARPS_PER_CTA][SDP_RING_WORDS];                                 \
        sdp::trace_body<K, PAD>(P, T, ring_mem);                                                           \
    }
#define SDP_DEFINE_SCORE_ALL(K)         \
    SDP_DEFINE_SCORE(K, _fe, false, false) \
    SDP_DEFINE_SCORE(K, _fp, false, true)  \
    SDP_DEFINE_SCORE(K, _re, true, false)  \
    SDP_DEFINE_SCORE(K, _rp, true, true)   \
    SDP_DEFINE_TRACE(K, _e, false)         \
    SDP_DEFINE_TRACE(K, _p, true)

SDP_DEFINE_SCORE_ALL(SDP_K_LO)
#if SDP_K_HI != SDP_K_LO
SDP_DEFINE_SCORE_ALL(SDP_K_HI)
#endif
#if SDP_K_HI > SDP_K_LO + 1
#error "a unit holds at most two column counts"
#endif
