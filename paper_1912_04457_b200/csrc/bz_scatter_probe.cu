// bz_scatter_probe.cu -- measurement tool, NOT part of libbz.so: the scatter designs NS names ("warp-aggregated
// shared-memory atomics with a global flush, or a sort-by-target-cell segmented reduction, picked by measurement") and
// the ones tried on the way, on the deposit stream of one collision step of one spatial cell:
//   n accepted samples, each with 4 target momentum cells (uniform over the Np cells of the tile, as the kinematic
//   samples are to a good approximation) and S = 7 deposits per cell; the result is dN[cell][8] (or [species][cell]).
// Build:  python -m paper_1912_04457_b200.build scatter_probe     Run:  paper_1912_04457_b200/bz_scatter_probe [np] [samples_per_cell]
// Output: one line per variant, nanoseconds per sample and cell updates per second; profiles/r2_scatter_variants.md keeps it.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <vector>

#include <cub/cub.cuh>

#define CK(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { std::printf("CUDA error %s at %s:%d\n", cudaGetErrorString(e_), __FILE__, __LINE__); std::exit(1); } } while (0)

namespace {

constexpr int kS = 7;

__device__ __forceinline__ uint32_t hash32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352dU; x ^= x >> 15; x *= 0x846ca68bU; x ^= x >> 16;
    return x;
}
// target cell c (0..3) of sample q, and its deposit for species a: cheap, reproducible, no memory traffic
__device__ __forceinline__ unsigned target_of(unsigned q, int c, unsigned Np) { return hash32(4u * q + (unsigned)c + 0x9e3779b9u) % Np; }
__device__ __forceinline__ double deposit_of(unsigned q, int c, int a) { return (c < 2 ? -1.0 : 1.0) * (1.0 + 0.001 * (double)((q + 7u * a) & 1023u)); }

__device__ __forceinline__ void red_add(double* p, double v) { asm volatile("red.global.add.f64 [%0], %1;" ::"l"(p), "d"(v)); }

// A: one 8-byte reduction per lane into the species-major layout dN[a][cell]: 32 lanes, 32 sectors
__global__ void scatter_species_major(double* dN, unsigned n, unsigned Np)
{
    for (unsigned q = blockIdx.x * blockDim.x + threadIdx.x; q < n; q += gridDim.x * blockDim.x)
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const unsigned cell = target_of(q, c, Np);
#pragma unroll
            for (int a = 0; a < kS; ++a) red_add(dN + (size_t)a * Np + cell, deposit_of(q, c, a));
        }
}

// B: cell-major dN[cell][8]; a warp handles 32 samples, one sample per instruction: lane = (cell c, slot a), 8 lanes per
// 64-byte cell (the form collide_kernel uses; its deposits come from shared memory, here from registers)
__global__ void scatter_cell_major(double* dN, unsigned n, unsigned Np)
{
    const int lane = threadIdx.x & 31, c = lane >> 3, a = lane & 7;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned q0 = warp * 32u; q0 < n; q0 += nwarps * 32u)
        for (unsigned q = q0; q < q0 + 32u && q < n; ++q) {
            const unsigned cell = target_of(q, c, Np);
            if (a < kS) red_add(dN + (size_t)cell * 8 + a, deposit_of(q, c, a));
        }
}

// C: shared-memory fp64 atomics into a tile that fits (Np * 8 doubles <= 200 KB), one CTA per SM, then a global flush
__global__ void scatter_smem_atomics(double* dN, unsigned n, unsigned Np)
{
    extern __shared__ double tile[];
    for (unsigned k = threadIdx.x; k < Np * 8u; k += blockDim.x) tile[k] = 0.0;
    __syncthreads();
    const int lane = threadIdx.x & 31, c = lane >> 3, a = lane & 7;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned q0 = warp * 32u; q0 < n; q0 += nwarps * 32u)
        for (unsigned q = q0; q < q0 + 32u && q < n; ++q) {
            const unsigned cell = target_of(q, c, Np);
            if (a < kS) atomicAdd(&tile[(size_t)cell * 8 + a], deposit_of(q, c, a));
        }
    __syncthreads();
    for (unsigned k = threadIdx.x; k < Np * 8u; k += blockDim.x)
        if (tile[k] != 0.0) red_add(dN + k, tile[k]);
}

// D: TMA bulk reduction, 64 bytes per (sample, cell): cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64.  The
// deposits of a warp's sample are staged in shared memory (4 x 64 B), one lane per cell issues the bulk operation.
__global__ void scatter_bulk_reduce(double* dN, unsigned n, unsigned Np)
{
    __shared__ __align__(128) double stage[8][2][32];     // [warp][buffer][4 cells x 8]
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, c = lane >> 3, a = lane & 7;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    int buf = 0;
    for (unsigned q0 = warp * 32u; q0 < n; q0 += nwarps * 32u)
        for (unsigned q = q0; q < q0 + 32u && q < n; ++q) {
            // the buffer used two samples ago must have been read by its bulk operations
            asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
            __syncwarp();
            stage[w][buf][lane] = a < kS ? deposit_of(q, c, a) : 0.0;
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncwarp();
            if (a == 0) {
                const unsigned cell = target_of(q, c, Np);
                const unsigned src = (unsigned)__cvta_generic_to_shared(&stage[w][buf][c * 8]);
                asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.f64 [%0], [%1], 64;" ::"l"(dN + (size_t)cell * 8), "r"(src) : "memory");
            }
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
            buf ^= 1;
        }
    asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// E: sort by target cell + segmented reduction.  Step 1 writes the (cell, index) pairs and the 64-byte deposit records,
// step 2 sorts the pairs (cub radix sort), step 3 walks the sorted pairs: one warp-slot of 8 lanes per target cell run.
__global__ void emit_records(unsigned* keys, unsigned* idx, double* rec, unsigned n, unsigned Np)
{
    const int lane = threadIdx.x & 31, c = lane >> 3, a = lane & 7;
    const unsigned warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (unsigned q0 = warp * 32u; q0 < n; q0 += nwarps * 32u)
        for (unsigned q = q0; q < q0 + 32u && q < n; ++q) {
            rec[(size_t)(4u * q + c) * 8 + a] = a < kS ? deposit_of(q, c, a) : 0.0;
            if (a == 0) { keys[4u * q + c] = target_of(q, c, Np); idx[4u * q + c] = 4u * q + c; }
        }
}
__global__ void segmented_reduce(const unsigned* keys, const unsigned* idx, const double* rec, double* dN, unsigned m)
{
    // 8 lanes per position; a group starts a run where the key changes and sums it sequentially (runs are ~ 4 n / Np long)
    const unsigned g = (blockIdx.x * blockDim.x + threadIdx.x) >> 3, a = threadIdx.x & 7;
    if (g >= m) return;
    const unsigned key = keys[g];
    if (g > 0 && keys[g - 1] == key) return;
    double acc = 0.0;
    for (unsigned k = g; k < m && keys[k] == key; ++k) acc += rec[(size_t)idx[k] * 8 + a];
    dN[(size_t)key * 8 + a] += acc;
}

float time_ms(cudaEvent_t e0, cudaEvent_t e1) { float ms = 0.f; CK(cudaEventElapsedTime(&ms, e0, e1)); return ms; }

}  // namespace

int main(int argc, char** argv)
{
    const int np = argc > 1 ? std::atoi(argv[1]) : 30;            // config 2: 30^3 cells
    const int ns = argc > 2 ? std::atoi(argv[2]) : 256;           // config 2: 256 samples per cell
    const unsigned Np = (unsigned)np * np * np;
    const unsigned n = (unsigned)(0.46 * (double)Np * ns);        // accepted samples of one step (S9: 46 %)
    int sms = 0;
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0));
    std::printf("tile: %d^3 = %u cells x 8 doubles = %.0f KB, %u accepted samples, %u cell updates, %d SMs\n", np, Np, Np * 64.0 / 1024, n, 4 * n, sms);
    double *dN = nullptr, *rec = nullptr;
    unsigned *keys = nullptr, *idx = nullptr, *keys2 = nullptr, *idx2 = nullptr;
    CK(cudaMalloc(&dN, (size_t)Np * 8 * sizeof(double)));
    CK(cudaMalloc(&rec, (size_t)4 * n * 8 * sizeof(double)));
    CK(cudaMalloc(&keys, (size_t)4 * n * 4)); CK(cudaMalloc(&idx, (size_t)4 * n * 4));
    CK(cudaMalloc(&keys2, (size_t)4 * n * 4)); CK(cudaMalloc(&idx2, (size_t)4 * n * 4));
    size_t tmp_bytes = 0;
    CK(cub::DeviceRadixSort::SortPairs(nullptr, tmp_bytes, keys, keys2, idx, idx2, (int)(4 * n)));
    void* tmp = nullptr;
    CK(cudaMalloc(&tmp, tmp_bytes));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0)); CK(cudaEventCreate(&e1));
    std::vector<double> ref((size_t)Np * 8), got((size_t)Np * 8);
    auto report = [&](const char* name, float ms, bool check) {
        CK(cudaMemcpy(got.data(), dN, got.size() * sizeof(double), cudaMemcpyDeviceToHost));
        double err = 0.0, mx = 0.0;
        if (check) for (size_t k = 0; k < got.size(); ++k) { err = std::max(err, std::fabs(got[k] - ref[k])); mx = std::max(mx, std::fabs(ref[k])); }
        std::printf("%-58s %8.3f ms  %7.3f ns/sample  %.3e cell updates/s  %s\n", name, ms, ms * 1e6 / n, 4.0 * n / (ms * 1e-3),
                    check ? (err <= 1e-9 * mx ? "sums agree" : "SUMS DIFFER") : "(reference)");
    };
    const int reps = 5;
    // B first: it is the reference result
    for (int variant = 0; variant < 5; ++variant) {
        if (variant == 2 && (size_t)Np * 64 > 200 * 1024) {
            std::printf("%-58s tile does not fit in shared memory (%.0f KB > 200 KB)\n", "C  shared-memory atomicAdd(double) + flush", Np * 64.0 / 1024);
            continue;
        }
        float best = 1e30f;
        for (int r = 0; r < reps; ++r) {
            CK(cudaMemset(dN, 0, (size_t)Np * 8 * sizeof(double)));
            CK(cudaEventRecord(e0));
            if (variant == 0) scatter_cell_major<<<sms * 8, 256>>>(dN, n, Np);
            else if (variant == 1) scatter_species_major<<<sms * 8, 256>>>(dN, n, Np);
            else if (variant == 2) {
                CK(cudaFuncSetAttribute(scatter_smem_atomics, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(Np * 64)));
                scatter_smem_atomics<<<sms, 512, Np * 64>>>(dN, n, Np);
            } else if (variant == 3) scatter_bulk_reduce<<<sms * 8, 256>>>(dN, n, Np);
            else {
                emit_records<<<sms * 8, 256>>>(keys, idx, rec, n, Np);
                CK(cub::DeviceRadixSort::SortPairs(tmp, tmp_bytes, keys, keys2, idx, idx2, (int)(4 * n)));
                segmented_reduce<<<(4 * n * 8 + 255) / 256, 256>>>(keys2, idx2, rec, dN, 4 * n);
            }
            CK(cudaEventRecord(e1));
            CK(cudaEventSynchronize(e1));
            CK(cudaGetLastError());
            best = std::min(best, time_ms(e0, e1));
        }
        if (variant == 0) { CK(cudaMemcpy(ref.data(), dN, ref.size() * sizeof(double), cudaMemcpyDeviceToHost)); }
        static const char* names[5] = { "B  RED.E.ADD.F64, 8 lanes per 64-byte cell (cell-major)", "A  RED.E.ADD.F64, one 8-byte sector per lane (species-major)",
                                        "C  shared-memory atomicAdd(double) + flush", "D  cp.reduce.async.bulk 64 B per (sample, cell)",
                                        "E  sort by target cell (cub radix) + segmented reduction" };
        if (variant == 1) {                                  // other layout: compare the transposed sums
            std::vector<double> t((size_t)Np * 8, 0.0);
            CK(cudaMemcpy(got.data(), dN, (size_t)kS * Np * sizeof(double), cudaMemcpyDeviceToHost));
            for (int a = 0; a < kS; ++a) for (unsigned c = 0; c < Np; ++c) t[(size_t)c * 8 + a] = got[(size_t)a * Np + c];
            double err = 0.0, mx = 0.0;
            for (size_t k = 0; k < t.size(); ++k) { err = std::max(err, std::fabs(t[k] - ref[k])); mx = std::max(mx, std::fabs(ref[k])); }
            std::printf("%-58s %8.3f ms  %7.3f ns/sample  %.3e cell updates/s  %s\n", names[1], best, best * 1e6 / n, 4.0 * n / (best * 1e-3), err <= 1e-9 * mx ? "sums agree" : "SUMS DIFFER");
        } else {
            report(names[variant], best, variant != 0);
        }
    }
    return 0;
}
