// inst.cu -- every kernel of ONE transform length (compile with -DTBS_N=32 ... 4096; build.py builds the eight
// lengths in parallel and links them with tbs.cu).
#include "dispatch_impl.cuh"

#ifndef TBS_N
#error "compile with -DTBS_N=<transform length>"
#endif

namespace tbs {
template cudaError_t launch_row_n<TBS_N>(bool, const RowArgs &, cudaStream_t, bool, LaunchOpt);
template cudaError_t launch_conv_n<TBS_N>(const ColArgs &, const CUtensorMap *, int, cudaStream_t, bool, LaunchOpt);
#if TBS_N <= 512
template cudaError_t launch_col_n<TBS_N>(int, const ColArgs &, int, cudaStream_t, bool, LaunchOpt);
#endif
}  // namespace tbs
