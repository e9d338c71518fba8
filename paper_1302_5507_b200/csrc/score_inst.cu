// score_inst.cu -- instantiations of the score kernel for K in [SDP_K_LO, SDP_K_HI]. The build
// compiles this file once per K range (-DSDP_K_LO=.. -DSDP_K_HI=.. -DSDP_K_FN=..) so the 128
// kernels (32 column counts x forward/reverse x exact/padded read length) compile in parallel.
#include "score_kernel.cuh"

#ifndef SDP_K_LO
#error "define SDP_K_LO, SDP_K_HI and SDP_K_FN"
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

}  // namespace sdp
