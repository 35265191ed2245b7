// bz_noalloc.cu -- bz_moments_noalloc: the moments of bz_moments (Eq. 10-11; regulator mass of Eq. 8) for a
// caller that holds f on the device itself and must not, or cannot, allocate device memory.
//
// Who that is.  bz_create reserves 2 copies of f plus two cell-major staging copies (about 4.3 x the size of f): a solver of
// the user's own whose f already fills most of the card (the paper's 20^3 x 40^3 grid is 28.7 GB per copy) cannot afford a
// context just to read n, e and m^2 off its state.  The same holds for an in-situ monitor that runs beside a long step on
// another stream (cudaMalloc / cudaFree synchronise the whole device and would stall that step) and for a process whose
// device memory has been handed in full to a framework's pool, where a raw cudaMalloc simply fails.
//
// How.  bz_moments needs one piece of scratch: the row sums [Nx][S][3] that rowsum_kernel leaves for moments_kernel.  Here that
// scratch is the file-scope array g_noalloc_rowsum below: kNoallocMaxRows rows, 1.5 MiB, part of the library's image on EVERY
// GPU that loads libbz.so, held until the process exits.  Nothing is allocated, freed or resized by the entry point, and it
// calls no library routine that allocates; the momentum tables of the context path (|p|, d3p/((2 pi)^3 |p|) per cell) are
// recomputed in registers instead of being read from a table.
//
// In HOST code the name g_noalloc_rowsum is only a handle for the runtime, not a device address: a kernel handed
// `g_noalloc_rowsum` from the host would fault (or, where the GPU can reach host memory, quietly use the wrong bytes).  The
// device address is asked for once per device with cudaGetSymbolAddress, with that device current, and cached.
#include <atomic>
#include <cstdio>

#include "bz_internal.h"

namespace bz {
namespace {

constexpr int kNoallocMaxRows = 65536;       // Nx * S rows of 3 doubles: 1.5 MiB (config 4: 28672 rows; 20^3 cells x 7 species: 56000)
constexpr int kNoallocMaxDevices = 64;

static __device__ __align__(256) double g_noalloc_rowsum[(size_t)kNoallocMaxRows * 3];

std::atomic<double*> g_scratch_addr[kNoallocMaxDevices];     // per device: device address of g_noalloc_rowsum (nullptr = not asked yet)
thread_local char g_noalloc_err[256] = "";

// Row sums of ONE spatial cell per CTA, all S species: sum f, sum |p| f, sum f d3p/((2pi)^3 |p|) over the Np momentum cells,
// the same three sums in the same order of additions as rowsum_kernel (thread t takes cells t, t + 256, ...; xor-shuffle
// tree; the 8 warps in order), so that the two paths agree to the last bit as long as the tables do.  |p| and the weight
// follow bz_create's host loop operation by operation (single roundings, no contraction); the weight is 0 at p = 0 (S10).
// Every row of the cell is WRITTEN, never accumulated into: stale contents of the scratch from an earlier call are harmless.
__global__ void __launch_bounds__(256) rowsum_noalloc_kernel(const double* __restrict__ f, double* __restrict__ rowsum, int S, int Np,
                                                             int n, double pmin, double dp, double d3p, double twopi3)
{
    const double* fx = f + (size_t)blockIdx.x * S * Np;
    double s0[7], s1[7], s2[7];
#pragma unroll
    for (int a = 0; a < 7; ++a) { s0[a] = 0.0; s1[a] = 0.0; s2[a] = 0.0; }
    for (int p = threadIdx.x; p < Np; p += blockDim.x) {
        const int ix = p % n, iy = (p / n) % n, iz = p / (n * n);
        const double px = __dadd_rn(pmin, __dmul_rn((double)ix + 0.5, dp));
        const double py = __dadd_rn(pmin, __dmul_rn((double)iy + 0.5, dp));
        const double pz = __dadd_rn(pmin, __dmul_rn((double)iz + 0.5, dp));
        const double E = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(px, px), __dmul_rn(py, py)), __dmul_rn(pz, pz)));
        const double w = E > 0.0 ? __ddiv_rn(d3p, __dmul_rn(twopi3, E)) : 0.0;
#pragma unroll
        for (int a = 0; a < 7; ++a)
            if (a < S) {
                const double v = fx[(size_t)a * Np + p];
                s0[a] += v; s1[a] += E * v; s2[a] += w * v;
            }
    }
    __shared__ double sh[7][3][8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
#pragma unroll
    for (int a = 0; a < 7; ++a) {
        if (a < S) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                s0[a] += __shfl_xor_sync(0xffffffffu, s0[a], o);
                s1[a] += __shfl_xor_sync(0xffffffffu, s1[a], o);
                s2[a] += __shfl_xor_sync(0xffffffffu, s2[a], o);
            }
            if (lane == 0) { sh[a][0][warp] = s0[a]; sh[a][1][warp] = s1[a]; sh[a][2][warp] = s2[a]; }
        }
    }
    __syncthreads();
    if ((int)threadIdx.x < 3 * S) {
        const int a = threadIdx.x / 3, k = threadIdx.x % 3;
        double t = 0.0;
        for (int w8 = 0; w8 < 8; ++w8) t += sh[a][k][w8];
        rowsum[((size_t)blockIdx.x * S + a) * 3 + k] = t;
    }
}

int noalloc_fail(int rc, const char* text)
{
    std::snprintf(g_noalloc_err, sizeof g_noalloc_err, "%s", text);
    return rc;
}

// Set-up, once per device: the device address of the static scratch on the device that is current now.
int scratch_address(double** out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return noalloc_fail(-2, cudaGetErrorString(e));
    if (dev < 0 || dev >= kNoallocMaxDevices) return noalloc_fail(-2, "bz_moments_noalloc: device ordinal beyond the per-device table");
    double* p = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        void* q = nullptr;
        e = cudaGetSymbolAddress(&q, g_noalloc_rowsum);          // the handle -> this device's copy of the array
        if (e != cudaSuccess || !q) {
            std::snprintf(g_noalloc_err, sizeof g_noalloc_err, "bz_moments_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return -2;
        }
        p = static_cast<double*>(q);
        g_scratch_addr[dev].store(p, std::memory_order_release);   // two threads racing here store the same address
    }
    *out = p;
    return 0;
}

}  // namespace
}  // namespace bz

using namespace bz;

extern "C" {

int bz_moments_noalloc(const bz_grid* g, const int* species, int n_species, double alpha_s, double m_D, const double* f_dev,
                       double* out_dev, void* cuda_stream)
{
    g_noalloc_err[0] = 0;
    if (!g || !species || !f_dev || !out_dev || n_species < 1 || n_species > 7) return noalloc_fail(-1, "bz_moments_noalloc: bad argument");
    if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->np < 2 || g->np > 1024 || !(g->pmax > g->pmin) || !(g->dx > 0.0) || !(alpha_s > 0.0))
        return noalloc_fail(-1, "bz_moments_noalloc: bad grid or coupling");
    for (int a = 0; a < n_species; ++a)
        if (species[a] < 0 || species[a] > 6 || (a > 0 && species[a] <= species[a - 1]))
            return noalloc_fail(-1, "bz_moments_noalloc: species ids must be 0..6, strictly ascending");
    const long long Nx = (long long)g->nx * g->ny * g->nz, rows = Nx * n_species;
    if (rows > kNoallocMaxRows) {
        std::snprintf(g_noalloc_err, sizeof g_noalloc_err,
                      "bz_moments_noalloc: %lld spatial cells x %d species = %lld rows, the static scratch holds %d; use bz_moments on a context",
                      Nx, n_species, rows, kNoallocMaxRows);
        return -5;
    }
    double* scratch = nullptr;
    if (int rc = scratch_address(&scratch)) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int S = n_species, Np = g->np * g->np * g->np;
    const double L = g->pmax - g->pmin, dp = L / g->np, d3p = (dp * dp) * dp;
    const double twopi3 = (2.0 * kPi) * (2.0 * kPi) * (2.0 * kPi);
    rowsum_noalloc_kernel<<<(unsigned)Nx, 256, 0, st>>>(f_dev, scratch, S, Np, g->np, g->pmin, dp, d3p, twopi3);
    ++g_launch_count;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return noalloc_fail(-2, cudaGetErrorString(e));
    double deg[7];
    for (int a = 0; a < 7; ++a) deg[a] = a < S ? (species[a] == 0 ? 16.0 : 6.0) : 1.0;      // N_g = 2 x 8, N_q = 2 x 3
    const double d3x = ((g->dx * g->dx) * g->dx) / ((kHbarc * kHbarc) * kHbarc);
    e = launch_moments(scratch, out_dev, (int)Nx, S, deg, species[0] == 0 ? 1u : 0u, 4.0 * kPi * alpha_s, m_D > 0.0 ? m_D * m_D : 0.0,
                       d3p / twopi3, d3x, 0, (int)Nx, st);
    if (e != cudaSuccess) return noalloc_fail(-2, cudaGetErrorString(e));
    return 0;
}

const char* bz_noalloc_last_error(void) { return g_noalloc_err; }

}  // extern "C"
