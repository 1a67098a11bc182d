// ms_launch.h -- launchers exported by the per-n translation units (ms_inst.cu, -DMS_N=2..9 -DMS_PART=0..2).
#pragma once
#include "ms_params.h"

namespace ms {
#define MS_DECL(n)                                                                                   \
    cudaError_t launch_gen_fast_##n(const GenParams& P, int massmode, bool pdf, bool toy, cudaStream_t stream);   \
    cudaError_t launch_gen_exact_##n(const GenParams& P, int massmode, bool pdf, bool toy, cudaStream_t stream);  \
    cudaError_t launch_inverse_##n(const InvParams& P, bool massive, cudaStream_t stream);                        \
    cudaError_t launch_chili_##n(const ChiliParams& P, cudaStream_t stream);                       \
    cudaError_t launch_rescale_##n(const RescaleParams& P, cudaStream_t stream);
MS_DECL(2) MS_DECL(3) MS_DECL(4) MS_DECL(5) MS_DECL(6) MS_DECL(7) MS_DECL(8) MS_DECL(9)
#undef MS_DECL
}  // namespace ms
