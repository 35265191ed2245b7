// bz_transport.cu -- upwind free streaming + forward Euler (S8a.6, S8a.7), row sums, regulator mass and moments
// (S8a.1, S8a.8).  All HBM-bound: one coalesced pass over f, momentum index fastest.
#include "bz_internal.h"

namespace bz {

namespace {

// One thread per (xcell, pcell), looping over the species: f is read and written coalesced in pcell for every
// species, the collision deposits of the cell come from the cell-major scratch (64 contiguous bytes per thread).  Upwind flux form of the drift term of Eq. 13:
// dF = - sum_d [ max(c_d,0) (f(x) - f(x - e_d)) + min(c_d,0) (f(x + e_d) - f(x)) ],  c_d = v_d dt/dx, periodic.
template <int kMode>
__global__ void __launch_bounds__(256, 4) transport_kernel(const TransportParams P)
{
    // blockIdx.x = spatial cell (fastest), blockIdx.y = chunk of 256 momentum cells: the blocks in flight share one
    // momentum chunk of ALL spatial cells (Nx x S x 2 KB, 58 MB for config 4), which fits L2, so the three upwind
    // neighbour reads hit L2 instead of HBM (x-major order: the z neighbour is 256 rows = 198 MB away and misses)
    const int xcell = P.x_begin + blockIdx.x;
    const int ix = xcell % P.nx, iy = (xcell / P.nx) % P.ny, iz = xcell / (P.nx * P.ny);
    const size_t row = (size_t)P.S * P.Np;                    // doubles per spatial cell
    const int xm = (ix + P.nx - 1) % P.nx - ix, xp = (ix + 1) % P.nx - ix;
    const int ym = ((iy + P.ny - 1) % P.ny - iy) * P.nx, yp = ((iy + 1) % P.ny - iy) * P.nx;
    const int zm = ((iz + P.nz - 1) % P.nz - iz) * P.nx * P.ny, zp = ((iz + 1) % P.nz - iz) * P.nx * P.ny;
    for (int pc = blockIdx.y * blockDim.x + threadIdx.x; pc < P.Np; pc += gridDim.y * blockDim.x) {
        const double cx = P.vx[pc] * P.cfl, cy = P.vy[pc] * P.cfl, cz = P.vz[pc] * P.cfl;
        // only the upwind neighbour of each axis is read
        const ptrdiff_t ox = (ptrdiff_t)(cx > 0.0 ? xm : xp) * (ptrdiff_t)row;
        const ptrdiff_t oy = (ptrdiff_t)(cy > 0.0 ? ym : yp) * (ptrdiff_t)row;
        const ptrdiff_t oz = (ptrdiff_t)(cz > 0.0 ? zm : zp) * (ptrdiff_t)row;
        const double ax = fabs(cx), ay = fabs(cy), az = fabs(cz);
        if (kMode == 0) {
            for (int a = 0; a < P.S; ++a) {
                const size_t idx = (size_t)xcell * row + (size_t)a * P.Np + pc;
                const double f0 = P.f[idx];
                // max(c,0)(f0 - f-) + min(c,0)(f+ - f0) = |c| (f0 - f_upwind)
                double acc = ax * (f0 - P.f[idx + ox]);
                acc += ay * (f0 - P.f[idx + oy]);
                acc += az * (f0 - P.f[idx + oz]);
                P.out[idx] = -acc;
            }
        } else {
            // Euler: the cell's collision deposits come from the cell-major scratch (64 contiguous bytes per thread,
            // reset to 0 here) and the new f also goes out cell-major, as the next step's gather source f_aos
            double2* dn = reinterpret_cast<double2*>(P.dN_aos + ((size_t)xcell * P.Np + pc) * P.SP);
            double2* fo = reinterpret_cast<double2*>(P.f_aos_out + ((size_t)xcell * P.Np + pc) * P.SP);
            double d[8], fn[8];
            if (P.SP == 8) {
#pragma unroll
                for (int q = 0; q < 4; ++q) { const double2 v = dn[q]; d[2 * q] = v.x; d[2 * q + 1] = v.y; }
            } else {
                d[0] = P.dN_aos[(size_t)xcell * P.Np + pc];
            }
#pragma unroll
            for (int a = 0; a < 7; ++a) {
                fn[a] = 0.0;
                if (a < P.S) {
                    const size_t idx = (size_t)xcell * row + (size_t)a * P.Np + pc;
                    const double f0 = P.f[idx];
                    if (kMode == 2) {
                        fn[a] = (f0 + P.out[idx]) + d[a] / P.inv_deg[a];      // the increment of Eq. 15 is already in out
                    } else {
                        double acc = ax * (f0 - P.f[idx + ox]);
                        acc += ay * (f0 - P.f[idx + oy]);
                        acc += az * (f0 - P.f[idx + oz]);
                        fn[a] = (f0 - acc) + d[a] / P.inv_deg[a];
                    }
                    P.out[idx] = fn[a];
                }
            }
            fn[7] = 0.0;
            if (P.SP == 8) {
#pragma unroll
                for (int q = 0; q < 4; ++q) { dn[q] = make_double2(0.0, 0.0); fo[q] = make_double2(fn[2 * q], fn[2 * q + 1]); }
            } else {
                P.dN_aos[(size_t)xcell * P.Np + pc] = 0.0;      // SP == 1: f itself is the gather source
            }
        }
    }
    if (kMode != 0) {
        // bz_step_n: the device step counter (the next step's Philox key word) moves on once per launch
        if (P.step_ptr && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) *P.step_ptr += 1u;
    }
}

// One CTA per (xcell, a) row: sum f, sum |p| f, sum f d3p/((2pi)^3 |p|) over the Np momentum cells.
__global__ void __launch_bounds__(256) rowsum_kernel(const double* __restrict__ f, const double* __restrict__ absp,
                                                     const double* __restrict__ w_invE, double* __restrict__ rowsum, int Np)
{
    const double* fr = f + (size_t)blockIdx.x * Np;
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (int p = threadIdx.x; p < Np; p += blockDim.x) {
        const double v = fr[p];
        s0 += v; s1 += absp[p] * v; s2 += w_invE[p] * v;
    }
    __shared__ double sh[3][8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        s0 += __shfl_xor_sync(0xffffffffu, s0, o);
        s1 += __shfl_xor_sync(0xffffffffu, s1, o);
        s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sh[0][warp] = s0; sh[1][warp] = s1; sh[2][warp] = s2; }
    __syncthreads();
    if (threadIdx.x < 3) {
        double t = 0.0;
        for (int w = 0; w < 8; ++w) t += sh[threadIdx.x][w];
        rowsum[(size_t)blockIdx.x * 3 + threadIdx.x] = t;
    }
}

// per-cell (n, e) and m2 copied behind them (all blocks); totals over the own cells x_begin..x_end: block b < 2 S sums
// total b = (species b / 2, n or e) with all its threads (strided partial sums, then a fixed-order tree: the result
// does not depend on the launch)
__global__ void __launch_bounds__(256) moments_kernel(const double* __restrict__ rowsum, double* __restrict__ mom, int Nx, int S,
                               unsigned glue_slot_mask, double g2, double mD2, double d3p_over_2pi3, double d3x, int x_begin, int x_end, const double d0, const double d1,
                               const double d2, const double d3, const double d4, const double d5, const double d6)
{
    const double deg[7] = { d0, d1, d2, d3, d4, d5, d6 };
    const size_t rows = (size_t)Nx * S;
    for (size_t r = blockIdx.x * (size_t)blockDim.x + threadIdx.x; r < rows; r += (size_t)gridDim.x * blockDim.x) {
        const int a = (int)(r % S);
        mom[2 * r + 0] = deg[a] * rowsum[3 * r + 0] * d3p_over_2pi3;
        mom[2 * r + 1] = deg[a] * rowsum[3 * r + 1] * d3p_over_2pi3;
    }
    for (size_t x = blockIdx.x * (size_t)blockDim.x + threadIdx.x; x < (size_t)Nx; x += (size_t)gridDim.x * blockDim.x)
        mom[2 * rows + 2 * S + x] = regulator_m2(rowsum, (int)x, S, glue_slot_mask, g2, mD2);
    if (blockIdx.x < 2 * S) {
        const int a = blockIdx.x >> 1, c = blockIdx.x & 1;
        double t = 0.0;
        for (int x = x_begin + threadIdx.x; x < x_end; x += blockDim.x)
            t += (deg[a] * rowsum[3 * ((size_t)x * S + a) + c] * d3p_over_2pi3) * d3x;
        __shared__ double sh[256];
        sh[threadIdx.x] = t;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
            __syncthreads();
        }
        if (threadIdx.x == 0) mom[2 * rows + blockIdx.x] = sh[0];
    }
}

}  // namespace

cudaError_t launch_transport(const TransportParams& P, int mode, cudaStream_t st)
{
    int chunks = (P.Np + 255) / 256;
    if (chunks > 65535) chunks = 65535;
    dim3 grid(P.x_count, chunks);
    if (mode == 0) transport_kernel<0><<<grid, 256, 0, st>>>(P);
    else if (mode == 1) transport_kernel<1><<<grid, 256, 0, st>>>(P);
    else transport_kernel<2><<<grid, 256, 0, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_rowsums(const double* f, const double* absp, const double* w_invE, double* rowsum, int rows, int Np,
                           cudaStream_t st)
{
    rowsum_kernel<<<rows, 256, 0, st>>>(f, absp, w_invE, rowsum, Np);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_moments(const double* rowsum, double* mom, int Nx, int S, const double* deg, unsigned glue_slot_mask, double g2,
                           double mD2, double d3p_over_2pi3, double d3x, int x_begin, int x_end, cudaStream_t st)
{
    int blocks = (Nx * S + 255) / 256;
    const int sms = device_sms();
    if (blocks > sms) blocks = sms;
    if (blocks < 2 * S) blocks = 2 * S;          // one block per total
    moments_kernel<<<blocks, 256, 0, st>>>(rowsum, mom, Nx, S, glue_slot_mask, g2, mD2, d3p_over_2pi3, d3x, x_begin, x_end, deg[0], deg[1], deg[2], deg[3], deg[4],
                                           deg[5], deg[6]);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
