// bz_is.cu -- test exports of the weighted samplers of NEXT rank 3: importance-sampled t
// (gen_sample_is_pair) and in-box CM direction (gen_sample_box_pair), both in bz_sample.cuh.  The collision term itself
// runs in collide_kernel (bz_collision.cu) with the sampler as a template parameter; the kernel here only writes out
// what a sampler draws, so that cells, (s, t, u) and weights can be compared bit for bit with the oracle.
#include "bz_internal.h"

namespace bz {

namespace {

// kSampler 1: importance-sampled t (regulator m2), 2: in-box direction.  Writes (j, k, l, flag), (s, t, u) and the weight
// of every sample of cells [p_begin, p_begin + p_count) of spatial cell x_begin.
template <int kSampler>
__global__ void __launch_bounds__(128) weighted_debug_kernel(const PaperParams P, double m2, int* dbg_cells, double* dbg_stu, double* dbg_w)
{
    const long long total = (long long)P.p_count * P.Ns;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int i = P.p_begin + (int)(q / P.Ns), smp = (int)(q % P.Ns);
        double p1x, p1y, p1z, E1;
        cell_kinematics(P.g, i, p1x, p1y, p1z, E1);
        const uint32_t xr = (uint32_t)P.x_begin + P.x_rng_offset;
        Sample sm;
        unsigned kstart = 0u;
        do {                                                 // the generator of the collision kernel, attempts two at a time
            if (kSampler == 1) sm = gen_sample_is_pair(P.g, P.seed, P.step, xr, (uint32_t)i, (uint32_t)smp, kstart, p1x, p1y, p1z, E1, m2);
            else sm = gen_sample_box_pair(P.g, P.seed, P.step, xr, (uint32_t)i, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
            kstart += 2u;
        } while (sm.retry);
        dbg_cells[4 * q + 0] = sm.j; dbg_cells[4 * q + 1] = sm.k; dbg_cells[4 * q + 2] = sm.l; dbg_cells[4 * q + 3] = sm.flag;
        dbg_stu[3 * q + 0] = sm.s; dbg_stu[3 * q + 1] = sm.t; dbg_stu[3 * q + 2] = sm.u;
        dbg_w[q] = sm.w;
    }
}

}  // namespace

cudaError_t launch_weighted_debug(const PaperParams& P, int sampler, double m2, int* cells, double* stu, double* w, int sms, cudaStream_t st)
{
    const long long total = (long long)P.p_count * P.Ns;
    if (total <= 0) return cudaSuccess;
    long long blocks = (total + 127) / 128;
    if (blocks > (long long)sms * 16) blocks = (long long)sms * 16;
    if (sampler == 1) weighted_debug_kernel<1><<<(int)blocks, 128, 0, st>>>(P, m2, cells, stu, w);
    else weighted_debug_kernel<2><<<(int)blocks, 128, 0, st>>>(P, m2, cells, stu, w);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
