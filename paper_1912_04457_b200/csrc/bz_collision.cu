// bz_collision.cu -- the fused sample -> |M|^2 -> bracket -> symmetric deposit kernel (S8a.2-8a.5).
//
// Mapping: one warp owns one p1 momentum cell at a time; its 32 lanes take the cell's N_s samples 32 at a time.
// f at the p1 cell is a warp-wide broadcast load, the slot-1 deposits of all samples of the cell are summed in
// registers and leave the warp as ONE atomic per species (shuffle reduction); the other three cells of a sample
// are random in the momentum tile, their deposits go out as fire-and-forget fp64 reductions (RED.E.ADD.F64) into
// the deposit scratch, which stays resident in L2 (a spatial cell's tile is <= 1.5 MB).
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

constexpr int kWarpsPerCta = 8;

__device__ __forceinline__ void red_add(double* addr, double v)
{
    if (v != 0.0) atomicAdd(addr, v);   // result unused: compiles to RED
}

template <int kMask>
__global__ void __launch_bounds__(kWarpsPerCta * 32) collide_kernel(const CollideParams P)
{
    const unsigned mask = kMask >= 0 ? (unsigned)kMask : P.mask;
    constexpr bool kGlue = kMask < 0 || (kMask & 1);
    constexpr bool kQuark = kMask < 0 || (kMask & 0x7E);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int xcell = blockIdx.y;
    const size_t tile = (size_t)xcell * P.S * P.Np;
    const double* __restrict__ ft = P.f + tile;
    double* __restrict__ dNt = P.dN + tile;
    const double m2 = P.m2[xcell];
    const int n = P.g.n;

    for (int i = blockIdx.x * kWarpsPerCta + warp; i < P.Np; i += gridDim.x * kWarpsPerCta) {
        const int ipx = i % n, ipy = (i / n) % n, ipz = i / (n * n);
        const double p1x = cell_centre(P.g, ipx), p1y = cell_centre(P.g, ipy), p1z = cell_centre(P.g, ipz);
        const double E1 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p1x, p1x), __dmul_rn(p1y, p1y)), __dmul_rn(p1z, p1z)));
        double fi[7], accI[7];
#pragma unroll
        for (int a = 0; a < 7; ++a) {
            accI[a] = 0.0;
            fi[a] = ((mask >> a) & 1u) ? ft[(size_t)P.slot[a] * P.Np + i] : 0.0;
        }
        for (int smp = lane; smp < P.Ns; smp += 32) {
            const Sample sm = gen_sample(P.g, P.seed, P.step, (uint32_t)xcell, (uint32_t)i, (uint32_t)smp, p1x, p1y, p1z, E1);
            if (!sm.flag) continue;
            double fj[7], fk[7], fl[7];
#pragma unroll
            for (int a = 0; a < 7; ++a) {
                if ((mask >> a) & 1u) {
                    const double* fa = ft + (size_t)P.slot[a] * P.Np;
                    fj[a] = fa[sm.j]; fk[a] = fa[sm.k]; fl[a] = fa[sm.l];
                } else {
                    fj[a] = fk[a] = fl[a] = 0.0;
                }
            }
            const double w = P.K / sm.E1E2;
            const MsqSet M = msq_set<kGlue, kQuark>(sm.s, sm.t, sm.u, m2, P.g4 * w);
            double dI[7], dJ[7], dK[7], dL[7];
            deposit<kMask>(mask, fi, fj, fk, fl, M, dI, dJ, dK, dL);
#pragma unroll
            for (int a = 0; a < 7; ++a) {
                if ((mask >> a) & 1u) {
                    double* da = dNt + (size_t)P.slot[a] * P.Np;
                    red_add(da + sm.j, dJ[a]);
                    red_add(da + sm.k, dK[a]);
                    red_add(da + sm.l, dL[a]);
                    accI[a] += dI[a];
                }
            }
        }
        // slot-1 deposits of the whole cell: one atomic per species
#pragma unroll
        for (int a = 0; a < 7; ++a) {
            if ((mask >> a) & 1u) {
                double v = accI[a];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) red_add(dNt + (size_t)P.slot[a] * P.Np + i, v);
            }
        }
    }
}

__global__ void debug_samples_kernel(const CollideParams P, int xcell, int p_begin, int p_end, int* cells, double* stu)
{
    const long long total = (long long)(p_end - p_begin) * P.Ns;
    const int n = P.g.n;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int i = p_begin + (int)(q / P.Ns), smp = (int)(q % P.Ns);
        const int ipx = i % n, ipy = (i / n) % n, ipz = i / (n * n);
        const double p1x = cell_centre(P.g, ipx), p1y = cell_centre(P.g, ipy), p1z = cell_centre(P.g, ipz);
        const double E1 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p1x, p1x), __dmul_rn(p1y, p1y)), __dmul_rn(p1z, p1z)));
        const Sample sm = gen_sample(P.g, P.seed, P.step, (uint32_t)xcell, (uint32_t)i, (uint32_t)smp, p1x, p1y, p1z, E1);
        cells[4 * q + 0] = sm.j; cells[4 * q + 1] = sm.k; cells[4 * q + 2] = sm.l; cells[4 * q + 3] = sm.flag;
        if (stu) { stu[3 * q + 0] = sm.s; stu[3 * q + 1] = sm.t; stu[3 * q + 2] = sm.u; }
    }
}

__global__ void finalize_kernel(double* __restrict__ dN, double* __restrict__ dF, int S, int Np, size_t total,
                                const double d0, const double d1, const double d2, const double d3, const double d4,
                                const double d5, const double d6)
{
    const double deg[7] = { d0, d1, d2, d3, d4, d5, d6 };
    for (size_t q = blockIdx.x * (size_t)blockDim.x + threadIdx.x; q < total; q += (size_t)gridDim.x * blockDim.x) {
        const int a = (int)((q / Np) % S);
        dF[q] = dN[q] / deg[a];
        dN[q] = 0.0;
    }
}

}  // namespace

cudaError_t launch_collide(const CollideParams& P, cudaStream_t st)
{
    const int cells_per_cta = kWarpsPerCta * 2;
    dim3 grid((P.Np + cells_per_cta - 1) / cells_per_cta, P.Nx), block(kWarpsPerCta * 32);
    switch (P.mask) {
    case 0x01u: collide_kernel<0x01><<<grid, block, 0, st>>>(P); break;
    case 0x7Eu: collide_kernel<0x7E><<<grid, block, 0, st>>>(P); break;
    case 0x7Fu: collide_kernel<0x7F><<<grid, block, 0, st>>>(P); break;
    default:    collide_kernel<-1><<<grid, block, 0, st>>>(P); break;
    }
    return cudaGetLastError();
}

cudaError_t launch_debug_samples(const CollideParams& P, int xcell, int p_begin, int p_end, int* cells, double* stu,
                                 cudaStream_t st)
{
    const long long total = (long long)(p_end - p_begin) * P.Ns;
    if (total <= 0) return cudaSuccess;
    const int blocks = (int)((total + 127) / 128 < 148 * 16 ? (total + 127) / 128 : 148 * 16);
    debug_samples_kernel<<<blocks, 128, 0, st>>>(P, xcell, p_begin, p_end, cells, stu);
    return cudaGetLastError();
}

cudaError_t launch_finalize(double* dN, double* dF, int Nx, int S, int Np, const double* deg, cudaStream_t st)
{
    const size_t total = (size_t)Nx * S * Np;
    const int blocks = (int)((total + 255) / 256 < 148 * 8 ? (total + 255) / 256 : 148 * 8);
    finalize_kernel<<<blocks, 256, 0, st>>>(dN, dF, S, Np, total, deg[0], deg[1], deg[2], deg[3], deg[4], deg[5], deg[6]);
    return cudaGetLastError();
}

}  // namespace bz
