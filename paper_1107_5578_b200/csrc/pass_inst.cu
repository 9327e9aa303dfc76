// pass_inst.cu -- instantiates the pass kernels for ONE transform length; compiled once per
// CWO_LOGN in [5, 14] (see build.py) so the ten lengths build in parallel.
#include "fold_kernel.cuh"
#include "cluster_kernel.cuh"
#include "prefetch_kernel.cuh"
#include "lineconv_kernel.cuh"
#include "linefft_kernel.cuh"
#include "rowpair_kernel.cuh"
#include "colpad_kernel.cuh"
#include "colfold_kernel.cuh"

#ifndef CWO_LOGN
#error "compile with -DCWO_LOGN=<5..14>"
#endif

namespace cwo {
#define CWO_CAT2(a, b) a##b
#define CWO_CAT(a, b) CWO_CAT2(a, b)
cudaError_t CWO_CAT(launch_pass_, CWO_LOGN)(int kind, int pad, int mid, int n_tiles, cudaStream_t s,
                                            const PassParams& p) {
    return launch_pass_impl<CWO_LOGN>(kind, pad, mid, n_tiles, s, p);
}
#if CWO_LOGN >= 8 && CWO_LOGN <= 13
cudaError_t CWO_CAT(launch_conv_, CWO_LOGN)(int variant, cudaStream_t s, const ConvParams& p) {
    return launch_lineconv_impl<CWO_LOGN>(variant, s, p);
}
cudaError_t CWO_CAT(launch_linefft_, CWO_LOGN)(cudaStream_t s, const LineFftParams& p) {
    return launch_linefft_impl<CWO_LOGN>(s, p);
}
#endif
}  // namespace cwo
