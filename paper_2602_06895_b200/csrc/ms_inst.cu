// ms_inst.cu -- compiled per multiplicity and part (-DMS_N=2..9 -DMS_PART=0|1|2): instantiates the per-n kernels and
// exports one launcher each, so that the translation units build in parallel.
//   part 0: generation kernels with the FastRambo mass chain; part 1: with the exact Rambo mass chain;
//   part 2: FastRambo inverse and stand-alone massive rescale.
#include "ms_kernels.cuh"
#include "ms_launch.h"

#if !defined(MS_N) || !defined(MS_PART)
#error "compile with -DMS_N=<n> -DMS_PART=<0|1|2>"
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

#define MS_CAT2(a, b) a##b
#define MS_CAT(a, b) MS_CAT2(a, b)

#if MS_PART == 0 || MS_PART == 1
constexpr bool kExact = MS_PART == 1;

template <int MASSMODE, bool PDF, bool TOY, bool ROWS, int GRID>
static cudaError_t launch_gen_t(const GenParams& P, cudaStream_t stream)
{
    auto kernel = gen_kernel<MS_N, kExact, MASSMODE, PDF, TOY, ROWS, GRID>;
    const size_t smem = GRID != 0 ? (size_t)P.grid_dims * P.grid_bins * sizeof(double2) : 0;
    if (smem > 48 * 1024) {
        cudaError_t err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (err != cudaSuccess) return err;
    }
    kernel<<<grid_for(kernel, P.N, smem), kBlock, smem, stream>>>(P);
    return cudaGetLastError();
}

#if MS_PART == 0
cudaError_t MS_CAT(launch_gen_fast_, MS_N)
#else
cudaError_t MS_CAT(launch_gen_exact_, MS_N)
#endif
    (const GenParams& P, int massmode, bool pdf, bool toy, cudaStream_t stream)
{
    if (P.x_rows != nullptr)
        return massmode == 2 ? launch_gen_t<2, false, false, true, 0>(P, stream)
                             : launch_gen_t<0, false, false, true, 0>(P, stream);
    // grid kind: 0 none, 1 any bin count, 6 / 7: 64 / 128 bins (the bin and the in-bin offset come straight from the
    // Philox mantissa: ms_kernels.cuh, UniformSource)
    const int gk = P.grid_dims <= 0 ? 0 : (P.grid_bins == 64 ? 2 : P.grid_bins == 128 ? 3 : 1);
    const int sel = gk * 4 + (pdf ? 2 : 0) + (toy ? 1 : 0);
#define MS_GK(v) ((v) / 4 == 0 ? 0 : (v) / 4 == 1 ? 1 : (v) / 4 == 2 ? 6 : 7)
#define MS_CASE(v)                                                                                               \
    case v:                                                                                                      \
        return massmode == 0   ? launch_gen_t<0, ((v) & 2) != 0, ((v) & 1) != 0, false, MS_GK(v)>(P, stream)    \
               : massmode == 1 ? launch_gen_t<1, ((v) & 2) != 0, ((v) & 1) != 0, false, MS_GK(v)>(P, stream)    \
                               : launch_gen_t<2, ((v) & 2) != 0, ((v) & 1) != 0, false, MS_GK(v)>(P, stream);
    switch (sel) {
        MS_CASE(0) MS_CASE(1) MS_CASE(2) MS_CASE(3) MS_CASE(4) MS_CASE(5) MS_CASE(6) MS_CASE(7)
        MS_CASE(8) MS_CASE(9) MS_CASE(10) MS_CASE(11) MS_CASE(12) MS_CASE(13) MS_CASE(14) MS_CASE(15)
        default: return cudaErrorInvalidValue;
    }
#undef MS_CASE
#undef MS_GK
}
#else
cudaError_t MS_CAT(launch_inverse_, MS_N)(const InvParams& P, bool massive, cudaStream_t stream)
{
    if (P.edges != nullptr) {                               // straight through the inverse of a 64- or 128-bin grid
        if (massive || MS_N < 2 || (P.grid_bins != 64 && P.grid_bins != 128)) return cudaErrorInvalidValue;
        const int levels = P.grid_bins == 64 ? 6 : 7;
        const size_t smem = vinv_table_bytes(3 * MS_N - 4, P.grid_bins, levels);
        auto kernel = levels == 6 ? inverse_kernel<MS_N, false, 6> : inverse_kernel<MS_N, false, 7>;
        if (smem > 48 * 1024) {
            const cudaError_t err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
            if (err != cudaSuccess) return err;
        }
        kernel<<<grid_for(kernel, P.N, smem), kBlock, smem, stream>>>(P);
    } else if (massive) {
        auto kernel = inverse_kernel<MS_N, true>;
        kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    } else {
        auto kernel = inverse_kernel<MS_N, false>;
        kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    }
    return cudaGetLastError();
}

cudaError_t MS_CAT(launch_chili_, MS_N)(const ChiliParams& P, cudaStream_t stream)
{
    if (P.x_rows != nullptr) {
        auto kernel = chili_kernel<MS_N, true>;
        kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    } else {
        auto kernel = chili_kernel<MS_N, false>;
        kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    }
    return cudaGetLastError();
}

cudaError_t MS_CAT(launch_rescale_, MS_N)(const RescaleParams& P, cudaStream_t stream)
{
    auto kernel = rescale_kernel<MS_N>;
    kernel<<<grid_for(kernel, P.N, 0), kBlock, 0, stream>>>(P);
    return cudaGetLastError();
}
#endif

}  // namespace ms
