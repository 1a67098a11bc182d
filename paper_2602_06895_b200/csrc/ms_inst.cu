// ms_inst.cu -- compiled once per multiplicity (-DMS_N=2..9): instantiates the per-n kernels and exports one
// launcher each, so that the eight translation units build in parallel.
#include "ms_kernels.cuh"
#include "ms_launch.h"

#ifndef MS_N
#error "compile with -DMS_N=<n>"
#endif

namespace ms {

template <class K>
static int grid_for(K kernel, int64_t N, size_t smem)
{
    int dev = 0, sms = 0, per_sm = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, kBlock, smem);
    if (per_sm < 1) per_sm = 1;
    const int64_t tiles = (N + kBlock - 1) / kBlock;
    const int64_t resident = (int64_t)sms * per_sm;   // one persistent wave: a multiple of the SM count
    return (int)(tiles < resident ? tiles : resident);
}

template <bool EXACT, bool MASSIVE>
static cudaError_t launch_gen_t(const GenParams& P, cudaStream_t stream)
{
    auto kernel = gen_kernel<MS_N, EXACT, MASSIVE>;
    const size_t smem = P.grid_dims > 0 ? (size_t)P.grid_dims * P.grid_bins * sizeof(double2) : 0;
    if (smem > 48 * 1024) {
        cudaError_t err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (err != cudaSuccess) return err;
    }
    kernel<<<grid_for(kernel, P.N, smem), kBlock, smem, stream>>>(P);
    return cudaGetLastError();
}

#define MS_CAT2(a, b) a##b
#define MS_CAT(a, b) MS_CAT2(a, b)

cudaError_t MS_CAT(launch_gen_, MS_N)(const GenParams& P, bool exact, bool massive, cudaStream_t stream)
{
    if (exact) return massive ? launch_gen_t<true, true>(P, stream) : launch_gen_t<true, false>(P, stream);
    return massive ? launch_gen_t<false, true>(P, stream) : launch_gen_t<false, false>(P, stream);
}

cudaError_t MS_CAT(launch_inverse_, MS_N)(const InvParams& P, cudaStream_t stream)
{
    auto kernel = inverse_kernel<MS_N>;
    kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    return cudaGetLastError();
}

cudaError_t MS_CAT(launch_rescale_, MS_N)(const RescaleParams& P, cudaStream_t stream)
{
    auto kernel = rescale_kernel<MS_N>;
    kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    return cudaGetLastError();
}

}  // namespace ms
