// bench_probes.cu -- measurement helpers of bench.py (NOT part of the product library: built into its own
// libms_bench_probes.so beside this file by bench_probes.py; nothing in paper_2602_06895_b200/ or include/ refers to it).
//
//   probe_dfma / probe_dfma3 : sustained fp64-pipe rate, DFMA with a constant-bank operand / three register operands
//   probe_write              : the generation kernel's store pattern with no arithmetic behind it
//   probe_mix                : the issue model behind DESIGN.md section 5 -- a loop of 4 DFMA plus K instructions of another
//                              kind (logic, IMAD, IMAD.WIDE, FFMA, MUFU, F2I/I2F, LDS): if the other instructions issue in
//                              the second cycle a DFMA holds its pipe, the loop costs max(8, 4 + K) cycles, else 8 + K
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

constexpr int kBlock = 256;

__global__ void __launch_bounds__(kBlock) probe_dfma_kernel(int iters, double* sink)
{
    double a0 = threadIdx.x * 1e-3, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
    const double m = 0.999999, c = 1e-7;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    sink[(int64_t)blockIdx.x * kBlock + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

__global__ void __launch_bounds__(kBlock) probe_dfma3_kernel(int iters, double* sink)
{
    double a[8], b[8], c[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        a[i] = threadIdx.x * 1e-3 + i;
        b[i] = 0.999999 - 1e-9 * (threadIdx.x + i);
        c[i] = 1e-7 * (1 + i + (threadIdx.x & 3));
    }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i) a[i] = fma(a[i], b[i], c[i]);
    }
    sink[(int64_t)blockIdx.x * kBlock + threadIdx.x] = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
}

__global__ void __launch_bounds__(kBlock) probe_write_kernel(int64_t N, int rows, double* out, int64_t ld)
{
    const int64_t n_tiles = (N + kBlock - 1) / kBlock;
    for (int64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const int64_t e = tile * kBlock + threadIdx.x;
        if (e >= N) continue;
        const double v = (double)e;
        for (int r = 0; r < rows; ++r) __stcs(out + (int64_t)r * ld + e, v + (double)r);
    }
}

// Dependent DFMA chain, `chains` independent chains per thread (1, 2, 4 or 8), launched with ONE warp per block: the time per
// DFMA of a single warp = the dependent-issue latency (chains = 1) and how many chains a scheduler needs to hide it.
template <int CH>
__global__ void probe_dfma_latency_kernel(int iters, double* sink)
{
    double a[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) a[i] = threadIdx.x * 1e-3 + i;
    const double m = 0.999999, c = 1e-7;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < CH; ++i) a[i] = fma(a[i], m, c);
    }
    double acc = 0.0;
#pragma unroll
    for (int i = 0; i < CH; ++i) acc += a[i];
    sink[(int64_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// KIND: 0 none, 1 LOP3 (alu pipe), 2 IMAD (32-bit), 3 IMAD.WIDE.U32, 4 FFMA, 5 MUFU.RCP (fp32), 6 F2I + I2F (fp64 <-> s32),
//       7 LDS.64, 8 IADD3, 9 MUFU.RCP64H
template <int KIND, int K, int ND>
__global__ void __launch_bounds__(kBlock) probe_mix_kernel(int iters, double* sink)
{
    __shared__ double s_buf[kBlock + 8];
    s_buf[threadIdx.x] = threadIdx.x;
    __syncthreads();
    double a[4];
    uint32_t x[8];
    float f[8];
    uint64_t wd[8];
    double dd[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) a[i] = threadIdx.x * 1e-3 + i;
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        x[i] = threadIdx.x * 2654435761u + i;
        f[i] = 1.0f + 1e-3f * (threadIdx.x + i);
        wd[i] = x[i];
        dd[i] = 1.0 + 1e-3 * (threadIdx.x + i);
    }
    const double m = 0.999999, c = 1e-7;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(s_buf) + 8u * (threadIdx.x & 31);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < ND; ++i) a[i & 3] = fma(a[i & 3], m, c);
#pragma unroll
        for (int j = 0; j < K; ++j) {
            const int r = j & 7, q = (j + 1) & 7;
            if constexpr (KIND == 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[r]) : "r"(x[q]), "r"((uint32_t)it));
            if constexpr (KIND == 2) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[r]) : "r"(x[q]), "r"((uint32_t)it));
            if constexpr (KIND == 3) asm volatile("mad.wide.u32 %0, %1, %2, %0;" : "+l"(wd[r]) : "r"(x[q]), "r"(0xD2511F53u));
            if constexpr (KIND == 4) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[r]) : "f"(f[q]), "f"(1e-7f));
            if constexpr (KIND == 5) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(f[r]));
            if constexpr (KIND == 6) {
                int t;
                asm volatile("cvt.rzi.s32.f64 %0, %1;" : "=r"(t) : "d"(dd[r]));
                asm volatile("cvt.rn.f64.s32 %0, %1;" : "=d"(dd[r]) : "r"(t + 1));
            }
            if constexpr (KIND == 7) asm volatile("ld.shared.f64 %0, [%1];" : "=d"(dd[r]) : "r"(sbase + 8u * (uint32_t)r));
            if constexpr (KIND == 8) asm volatile("add.u32 %0, %0, %1;" : "+r"(x[r]) : "r"(x[q]));
            if constexpr (KIND == 9) asm volatile("rcp.approx.ftz.f64 %0, %0;" : "+d"(dd[r]));
        }
    }
    double acc = (a[0] + a[1]) + (a[2] + a[3]);
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += (double)x[i] + (double)f[i] + (double)wd[i] + dd[i];
    sink[(int64_t)blockIdx.x * kBlock + threadIdx.x] = acc;
}

template <int KIND, int ND>
cudaError_t launch_mix(int k, int blocks, int iters, double* sink, cudaStream_t s)
{
    switch (k) {
        case 0: probe_mix_kernel<KIND, 0, ND><<<blocks, kBlock, 0, s>>>(iters, sink); break;
        case 2: probe_mix_kernel<KIND, 2, ND><<<blocks, kBlock, 0, s>>>(iters, sink); break;
        case 4: probe_mix_kernel<KIND, 4, ND><<<blocks, kBlock, 0, s>>>(iters, sink); break;
        case 8: probe_mix_kernel<KIND, 8, ND><<<blocks, kBlock, 0, s>>>(iters, sink); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace

extern "C" {

int probe_dfma(int blocks, int iters, double* d_sink, void* stream)
{
    probe_dfma_kernel<<<blocks, kBlock, 0, (cudaStream_t)stream>>>(iters, d_sink);
    return (int)cudaGetLastError();
}

int probe_dfma3(int blocks, int iters, double* d_sink, void* stream)
{
    probe_dfma3_kernel<<<blocks, kBlock, 0, (cudaStream_t)stream>>>(iters, d_sink);
    return (int)cudaGetLastError();
}

int probe_write(int64_t N, int rows, double* d_out, int64_t ld, void* stream)
{
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int64_t blocks = (N + kBlock - 1) / kBlock;
    const int grid = (int)(blocks < (int64_t)sms * 8 ? blocks : (int64_t)sms * 8);
    probe_write_kernel<<<grid, kBlock, 0, (cudaStream_t)stream>>>(N, rows, d_out, ld);
    return (int)cudaGetLastError();
}

// one warp per block, `blocks` blocks; chains = independent DFMA chains per thread
int probe_dfma_latency(int chains, int blocks, int iters, double* d_sink, void* stream)
{
    cudaStream_t s = (cudaStream_t)stream;
    switch (chains) {
        case 1: probe_dfma_latency_kernel<1><<<blocks, 32, 0, s>>>(iters, d_sink); break;
        case 2: probe_dfma_latency_kernel<2><<<blocks, 32, 0, s>>>(iters, d_sink); break;
        case 4: probe_dfma_latency_kernel<4><<<blocks, 32, 0, s>>>(iters, d_sink); break;
        case 8: probe_dfma_latency_kernel<8><<<blocks, 32, 0, s>>>(iters, d_sink); break;
        default: return (int)cudaErrorInvalidValue;
    }
    return (int)cudaGetLastError();
}

// per iteration and thread: nd (0 or 4) DFMA + k (0, 2, 4, 8) instructions of `kind` (see probe_mix_kernel)
int probe_mix(int kind, int k, int nd, int blocks, int iters, double* d_sink, void* stream)
{
    cudaStream_t s = (cudaStream_t)stream;
#define MS_KIND(KD) \
    case KD: return (int)(nd == 4 ? launch_mix<KD, 4>(k, blocks, iters, d_sink, s) : launch_mix<KD, 0>(k, blocks, iters, d_sink, s));
    switch (kind) {
        MS_KIND(0) MS_KIND(1) MS_KIND(2) MS_KIND(3) MS_KIND(4) MS_KIND(5) MS_KIND(6) MS_KIND(7) MS_KIND(8) MS_KIND(9)
        default: return (int)cudaErrorInvalidValue;
    }
#undef MS_KIND
}

}  // extern "C"
