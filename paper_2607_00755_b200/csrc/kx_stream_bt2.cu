// kx_stream_bt2.cu -- the streaming kernels (kx_stream.cuh) for member groups of 2
#include "kx_stream.cuh"

cudaError_t kx_launch_stream_bt2(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st,
                                 unsigned* bar_total, cudaStream_t s, const KxRun* run)
{
    return launch_stream_m<2>(d, sm_count, f, yd, B, st, bar_total, s, run);
}
