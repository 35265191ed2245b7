// bz_issue_probe.cu -- stand-alone measurement tool (not part of libbz.so): how the instruction mix of collide_kernel
// shares an SM sub-partition's issue port.  profiles/r2_collide_issue_model.md keeps its output and the reading.
//   part 1  8 independent DFMA chains and 8 independent chains of another opcode per thread, NF : NI interleaved,
//           16 warps per SM (4 per sub-partition, as in collide_kernel): cycles per step and instructions per cycle
//   part 2  four Philox4x32-10 blocks per thread (bz_sample.cuh: what one sampling pass of collide_kernel computes),
//           alone and with independent DFMAs interleaved
// Build: python -m paper_1912_04457_b200.build issue_probe ; run: paper_1912_04457_b200/bz_issue_probe
#include <cstdio>
#include <cuda_runtime.h>

#include "bz_sample.cuh"

namespace {

// IOP: 0 xor (LOP3), 1 add (IADD3), 2 mad.lo (IMAD), 3 mul.wide + xor (IMAD.WIDE, the Philox round), 4 FFMA
template <int IOP>
__device__ __forceinline__ void iop(unsigned& y, unsigned z, unsigned ua)
{
    if (IOP == 0) asm volatile("xor.b32 %0, %0, %1;" : "+r"(y) : "r"(z));
    if (IOP == 1) asm volatile("add.u32 %0, %0, %1;" : "+r"(y) : "r"(z));
    if (IOP == 2) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(y) : "r"(ua), "r"(z));
    if (IOP == 3) {
        unsigned long long w;
        asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w) : "r"(y), "r"(ua));
        y = (unsigned)(w >> 32) ^ (unsigned)w;
    }
    if (IOP == 4) {
        float f = __uint_as_float(y);
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f) : "f"(__uint_as_float(ua)), "f"(__uint_as_float(z)));
        y = __float_as_uint(f);
    }
}

template <int IOP, int NF, int NI>
__global__ void __launch_bounds__(512, 1) mix_kernel(double* out, unsigned* iout, int iters, double a, unsigned ua)
{
    double x[8];
    unsigned y[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { x[j] = threadIdx.x + j; y[j] = threadIdx.x + j; }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int r = 0; r < 8; ++r) {
#pragma unroll
            for (int j = 0; j < (NF > NI ? NF : NI); ++j) {
                if (j < NF) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x[j & 7]) : "d"(a), "d"(x[(j + 1) & 7]));
                if (j < NI) iop<IOP>(y[j & 7], y[(j + 1) & 7], ua);
            }
        }
    }
    double sx = 0;
    unsigned sy = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) { sx += x[j]; sy += y[j]; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = sx;
    iout[blockIdx.x * blockDim.x + threadIdx.x] = sy;
}

template <int NF>
__global__ void __launch_bounds__(512, 1) philox_kernel(unsigned* iout, double* dout, int iters, uint32_t seed, double a)
{
    uint32_t acc = 0;
    double x[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = threadIdx.x + j;
    for (int i = 0; i < iters; ++i) {
        uint32_t w[4][4];
#pragma unroll
        for (int b = 0; b < 4; ++b) bz::philox4x32_10(b, threadIdx.x + 32 * i, blockIdx.x, 7u, seed, 3u, w[b]);
#pragma unroll
        for (int j = 0; j < NF; ++j) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(x[j & 7]) : "d"(a), "d"(x[(j + 1) & 7]));
#pragma unroll
        for (int b = 0; b < 4; ++b) acc ^= w[b][0] ^ w[b][1] ^ w[b][2] ^ w[b][3];
    }
    double sx = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) sx += x[j];
    iout[blockIdx.x * blockDim.x + threadIdx.x] = acc;
    dout[blockIdx.x * blockDim.x + threadIdx.x] = sx;
}

double g_mhz = 1965.0;
double* g_out;
unsigned* g_iout;

template <typename F>
double cycles_of(F launch)
{
    launch(10);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    launch(0);
    cudaEventRecord(e1);
    cudaEventSynchronize(e1);
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    return ms * 1e-3 * g_mhz * 1e6;
}

template <int IOP, int NF, int NI>
void run_mix(const char* name, int sms)
{
    const int iters = 10000;
    const double cyc = cycles_of([&](int warm) { mix_kernel<IOP, NF, NI><<<sms, 512>>>(g_out, g_iout, warm ? warm : iters, 1.0000001, 3u); });
    const double steps = iters * 8.0;                       // per warp; 4 warps per sub-partition
    printf("%-12s DFMA:other = %d:%d   %6.2f cycles per step and warp   DFMA/clk %.3f   other/clk %.3f\n", name, NF, NI,
           cyc / steps / 4.0, 4 * NF * steps / cyc, 4 * NI * steps / cyc);
}

template <int NF>
void run_philox(int sms)
{
    const int iters = 2000;
    const double cyc = cycles_of([&](int warm) { philox_kernel<NF><<<sms, 512>>>(g_iout, g_out, warm ? warm : iters, 1u, 1.0000001); });
    printf("4 Philox4x32-10 blocks + %3d DFMA per thread: %6.1f sub-partition cycles per warp pass\n", NF, cyc / iters / 4.0);
}

}  // namespace

int main()
{
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, 0) != cudaSuccess) { fprintf(stderr, "no CUDA device\n"); return 1; }
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    g_mhz = khz / 1000.0;
    const int sms = prop.multiProcessorCount;
    cudaMalloc(&g_out, (size_t)sms * 512 * 8);
    cudaMalloc(&g_iout, (size_t)sms * 512 * 4);
    printf("%s, %d SMs, %.0f MHz (cycles assume the maximum clock), 16 warps per SM\n", prop.name, sms, g_mhz);
    run_mix<0, 8, 0>("dfma", sms);
    run_mix<0, 0, 8>("xor", sms); run_mix<1, 0, 8>("add", sms); run_mix<2, 0, 8>("imad", sms); run_mix<3, 0, 8>("mulwide+xor", sms); run_mix<4, 0, 8>("ffma", sms);
    run_mix<0, 4, 4>("dfma+xor", sms); run_mix<0, 4, 8>("dfma+xor", sms); run_mix<0, 2, 8>("dfma+xor", sms);
    run_mix<1, 4, 4>("dfma+add", sms); run_mix<1, 4, 8>("dfma+add", sms);
    run_mix<2, 4, 4>("dfma+imad", sms); run_mix<2, 4, 8>("dfma+imad", sms); run_mix<2, 2, 8>("dfma+imad", sms);
    run_mix<3, 4, 4>("dfma+mulw", sms); run_mix<3, 4, 8>("dfma+mulw", sms);
    run_mix<4, 4, 4>("dfma+ffma", sms); run_mix<4, 4, 8>("dfma+ffma", sms);
    run_philox<0>(sms); run_philox<80>(sms); run_philox<160>(sms); run_philox<240>(sms);
    return 0;
}
