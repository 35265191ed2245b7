// bz_diag.cu -- reporting kernel for reading S8 of SURVEY.md 8c: the regulated Table I is evaluated literally
// and can be negative (e.g. q qbar <-> g g when s is not large against m^2); the harness reports how often.  Outside the hot
// path: the kernel regenerates the kinematic samples of the collision kernel (same generator, same Philox counters),
// evaluates the ten distinct |M|^2 of a sample with the regulator of its spatial cell and counts the negative ones.
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

__global__ void __launch_bounds__(128) msq_sign_kernel(const CollideParams P, int x_begin, int x_end, unsigned long long* __restrict__ counts)
{
    const long long per_x = (long long)P.Np * P.Ns, total = per_x * (x_end - x_begin);
    unsigned acc[15];
#pragma unroll
    for (int k = 0; k < 15; ++k) acc[k] = 0u;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long rounds = (total + stride - 1) / stride;                  // whole warps stay in the loop for the shuffles below
    for (long long r = 0; r < rounds; ++r) {
        const long long q = r * stride + blockIdx.x * (long long)blockDim.x + threadIdx.x;
        if (q < total) {
            const int x = x_begin + (int)(q / per_x);
            const long long rem = q % per_x;
            const int i = (int)(rem / P.Ns), smp = (int)(rem % P.Ns);
            double p1x, p1y, p1z, E1;
            cell_kinematics(P.g, i, p1x, p1y, p1z, E1);
            Sample sm;
            unsigned kstart = 0u;
            do {
                sm = gen_sample_pair(P.g, P.seed, P.step, (uint32_t)x + P.x_rng_offset, (uint32_t)i, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
                kstart += 2u;
            } while (sm.retry);
            if (sm.flag) {
                const double m2 = regulator_m2(P.rowsum, x, P.S, P.glue_slot_mask, P.g2, P.mD2);
                MsqSet M = msq_set<true, true>(sm.s, sm.t, sm.u, m2, 1.0);
                if (P.has_ovr) msq_apply_override(M, P.msq_ovr, 1.0);
                // slot 1 + 2 kind + crossed, kinds in the order of bz_set_msq_override (A, 11, 1B, ANN, QQGG, QG, GG)
                const double v[14] = { M.a_t, M.a_u, M.m11, M.m11, M.m1b_t, M.m1b_u, M.ann, M.ann, M.qqgg, M.qqgg, M.qg_t, M.qg_u, M.gg, M.gg };
                acc[0] += 1u;
#pragma unroll
                for (int k = 0; k < 14; ++k) acc[1 + k] += v[k] < 0.0 ? 1u : 0u;
            }
        }
    }
#pragma unroll
    for (int k = 0; k < 15; ++k) {
        const unsigned t = __reduce_add_sync(0xffffffffu, acc[k]);
        if ((threadIdx.x & 31) == 0 && t) atomicAdd(&counts[k], (unsigned long long)t);
    }
}

}  // namespace

cudaError_t launch_msq_signs(const CollideParams& P, int x_begin, int x_end, unsigned long long* counts, int sms, cudaStream_t st)
{
    const long long total = (long long)P.Np * P.Ns * (x_end - x_begin);
    if (total <= 0) return cudaSuccess;
    long long blocks = (total + 127) / 128;
    if (blocks > (long long)sms * 16) blocks = (long long)sms * 16;
    msq_sign_kernel<<<(int)blocks, 128, 0, st>>>(P, x_begin, x_end, counts);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
