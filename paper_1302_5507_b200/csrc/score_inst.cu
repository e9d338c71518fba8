// score_inst.cu -- instantiations of the traceback DP kernel for K in [SDP_K_LO, SDP_K_HI]. The build compiles
// this file once per K range (-DSDP_K_LO=.. -DSDP_K_HI=.. -DSDP_T_FN=..) so the 64 kernels (32 column counts x
// {exact, padded read length}) compile in parallel. (The score kernels live in score_cubin.cu.)
#include "trace_kernel.cuh"

#if !defined(SDP_K_LO) || !defined(SDP_K_HI) || !defined(SDP_T_FN)
#error "define SDP_K_LO, SDP_K_HI and SDP_T_FN"
#endif

namespace sdp {

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
