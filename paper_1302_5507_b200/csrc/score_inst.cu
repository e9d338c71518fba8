// score_inst.cu -- instantiations of the score kernel and of the traceback DP kernel for K in
// [SDP_K_LO, SDP_K_HI]. The build compiles this file once per K range (-DSDP_K_LO=.. -DSDP_K_HI=..
// -DSDP_K_FN=.. -DSDP_T_FN=..) so the 192 kernels (32 column counts x {forward, reverse, traceback}
// x {exact, padded read length}) compile in parallel.
#include "trace_kernel.cuh"

#if !defined(SDP_K_LO) || !defined(SDP_K_HI) || !defined(SDP_K_FN) || !defined(SDP_T_FN)
#error "define SDP_K_LO, SDP_K_HI, SDP_K_FN and SDP_T_FN"
#endif

namespace sdp {

template <int K>
static inline bool dispatch_range(int k, bool pad, bool rev, const ScoreParams& p, cudaStream_t st) {
    if (k == K) { launch_score_K<K>(pad, rev, p, st); return true; }
    if constexpr (K < SDP_K_HI) return dispatch_range<K + 1>(k, pad, rev, p, st);
    else return false;
}

bool SDP_K_FN(int K, bool pad, bool rev, const ScoreParams& p, cudaStream_t st) {
    if (K < SDP_K_LO || K > SDP_K_HI) return false;
    return dispatch_range<SDP_K_LO>(K, pad, rev, p, st);
}

template <int K>
static inline bool dispatch_trace(int k, bool pad, const ScoreParams& p, const TraceDP& t, cudaStream_t st) {
    if (k == K) { launch_trace_K<K>(pad, p, t, st); return true; }
    if constexpr (K < SDP_K_HI) return dispatch_trace<K + 1>(k, pad, p, t, st);
    else return false;
}

bool SDP_T_FN(int K, bool pad, const ScoreParams& p, const TraceDP& t, cudaStream_t st) {
    if (K < SDP_K_LO || K > SDP_K_HI) return false;
    return dispatch_trace<SDP_K_LO>(K, pad, p, t, st);
}

}  // namespace sdp
