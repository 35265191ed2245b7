// bz_calibrate.cu -- FP64 FMA peak of the device, measured: the second leg of the roofline north_star defines for the
// collision kernel ("the slower of FP64 FMA peak and gathered/scattered bytes at HBM bandwidth").  MEASURED_PEAKS.json
// carries HBM and bf16 numbers only, so bench.py asks the library.  Register-resident chains of dependent DFMAs, 8
// independent chains per thread, 2048 threads per SM: nothing but the FP64 pipe is exercised.
#include "bz_internal.h"

namespace bz {
namespace {

constexpr int kChains = 8, kUnroll = 8;

__global__ void __launch_bounds__(1024) dfma_kernel(double* __restrict__ out, int iters, double a, double b)
{
    double x[kChains];
#pragma unroll
    for (int i = 0; i < kChains; ++i) x[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < kUnroll; ++r)
#pragma unroll
            for (int i = 0; i < kChains; ++i) x[i] = fma(x[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kChains; ++i) s += x[i];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace
}  // namespace bz

extern "C" int bz_measure_fp64_peak(double* tflops_out)
{
    using namespace bz;
    if (!tflops_out) return -1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -2;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return -2;
    const int blocks = 2 * sms, threads = 1024, iters = 4000;
    double* out = nullptr;
    if (cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)) != cudaSuccess) return -3;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = 0;
    double best = 0.0;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = -2;
    for (int rep = 0; rc == 0 && rep < 4; ++rep) {               // rep 0 warms up
        cudaEventRecord(e0, nullptr);
        dfma_kernel<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
        ++g_launch_count;
        cudaEventRecord(e1, nullptr);
        if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = -2; break; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        const double flop = 2.0 * blocks * (double)threads * iters * kUnroll * kChains;
        if (rep > 0 && ms > 0.f && flop / (ms * 1e-3) / 1e12 > best) best = flop / (ms * 1e-3) / 1e12;
    }
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(out);
    *tflops_out = best;
    return rc;
}
