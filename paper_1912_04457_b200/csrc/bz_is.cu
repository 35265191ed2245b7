// bz_is.cu -- NEXT rank 3 of SURVEY.md 8f: importance sampling of the t/u-channel peaks of Table I.
// The hot path draws the CM direction isotropically (t uniform on [-s, 0]); here t comes from
//   p(t) = (1/2) [g(t) + g(-s - t)],  g(t) = 1 / ((m^2 - t)^2 (1/m^2 - 1/(s + m^2))),
// the azimuth about the CM direction of p1 is uniform, and every deposit carries the weight (1/s)/p(t): the same
// expectation as bz_collision with a smaller variance when m^2 << s (oracle pin I4: spread x 0.6 at m_D = 0.25 GeV).
// Philox blocks 0, 1 (p2, as the hot path), 96 (t, branch) and 97.. (azimuth).  Everything that decides a cell index
// is a single correctly rounded operation in the oracle's association order (bit-exact cells).
// One lane per sample, a warp per 32 samples of ONE grid point: the slot-1 deposits of the warp are summed by shuffles
// and leave as one reduction per species; the other three cells get one RED per species and lane.  The channel algebra
// is the factorised one of the hot path (bz_channels.cuh).
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

#define MUL __dmul_rn
#define ADD __dadd_rn
#define SUB __dsub_rn
#define DIV __ddiv_rn

struct IsSample {
    int flag, j, k, l;
    double s, t, u, E1E2, w;
};

__device__ __forceinline__ IsSample gen_sample_is(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xc, uint32_t pcell,
                                                  uint32_t smp, double m2)
{
    IsSample o;
    o.flag = 0; o.j = 0; o.k = -1; o.l = -1; o.s = 0.0; o.t = 0.0; o.u = 0.0; o.E1E2 = 0.0; o.w = 0.0;
    double p1x, p1y, p1z, E1;
    cell_kinematics(g, (int)pcell, p1x, p1y, p1z, E1);
    uint32_t w0[4], w1[4], w2[4];
    philox4x32_10(0u, smp, pcell, xc, seed, step, w0);
    philox4x32_10(1u, smp, pcell, xc, seed, step, w1);
    philox4x32_10(96u, smp, pcell, xc, seed, step, w2);
    const double p2x = ADD(g.pmin, MUL(uniform52(w0[0], w0[1]), g.L));
    const double p2y = ADD(g.pmin, MUL(uniform52(w0[2], w0[3]), g.L));
    const double p2z = ADD(g.pmin, MUL(uniform52(w1[0], w1[1]), g.L));
    const double E2 = __dsqrt_rn(ADD(ADD(MUL(p2x, p2x), MUL(p2y, p2y)), MUL(p2z, p2z)));
    const double d12 = ADD(ADD(MUL(p1x, p2x), MUL(p1y, p2y)), MUL(p1z, p2z));
    const double s = MUL(2.0, SUB(MUL(E1, E2), d12));
    o.E1E2 = E1 * E2;
    {
        bool in;
        int a = bin_axis_exact(p2x, g, in), b = bin_axis_exact(p2y, g, in), c = bin_axis_exact(p2z, g, in);
        a = min(max(a, 0), g.n - 1); b = min(max(b, 0), g.n - 1); c = min(max(c, 0), g.n - 1);
        o.j = a + g.n * (b + g.n * c);
    }
    if (!(s > 0.0)) return o;
    // t and its weight
    const double ut = uniform52(w2[0], w2[1]), ub = uniform52(w2[2], w2[3]);
    double t, w;
    if (m2 > 0.0) {
        const double lo = DIV(1.0, ADD(s, m2)), hi = DIV(1.0, m2);
        const double r = ADD(lo, MUL(ut, SUB(hi, lo)));
        const double tt = SUB(m2, DIV(1.0, r));
        t = ub < 0.5 ? tt : SUB(-s, tt);
        const double dt_ = SUB(m2, t), du_ = SUB(m2, SUB(-s, t));
        const double norm = SUB(hi, lo);
        const double pt = MUL(0.5, ADD(DIV(1.0, MUL(MUL(dt_, dt_), norm)), DIV(1.0, MUL(MUL(du_, du_), norm))));
        w = DIV(DIV(1.0, s), pt);
    } else {
        t = MUL(-s, ut);
        w = 1.0;
    }
    double cs = ADD(1.0, DIV(MUL(2.0, t), s));
    if (cs > 1.0) cs = 1.0;
    if (cs < -1.0) cs = -1.0;
    const double sn = __dsqrt_rn(SUB(1.0, MUL(cs, cs)));
    // azimuth: first point of the sequence inside the unit disc (von Neumann); (1, 0) after 62 failures
    double ca = 1.0, sa = 0.0;
    for (uint32_t k = 0; k < 62u; ++k) {
        uint32_t wa[4];
        philox4x32_10(97u + k, smp, pcell, xc, seed, step, wa);
        const double v1 = ADD(MUL(2.0, uniform52(wa[0], wa[1])), -1.0), v2 = ADD(MUL(2.0, uniform52(wa[2], wa[3])), -1.0);
        const double q = ADD(MUL(v1, v1), MUL(v2, v2));
        if (q < 1.0 && q > 0.0) {
            ca = DIV(SUB(MUL(v1, v1), MUL(v2, v2)), q);
            sa = DIV(MUL(MUL(2.0, v1), v2), q);
            break;
        }
    }
    // CM direction of p1 and an orthonormal basis around it
    const double Px = ADD(p1x, p2x), Py = ADD(p1y, p2y), Pz = ADD(p1z, p2z);
    const double E = ADD(E1, E2), M = __dsqrt_rn(s);
    const double Pp1 = ADD(ADD(MUL(Px, p1x), MUL(Py, p1y)), MUL(Pz, p1z));
    const double fac = DIV(SUB(DIV(Pp1, ADD(E, M)), E1), M);
    const double qx = ADD(p1x, MUL(Px, fac)), qy = ADD(p1y, MUL(Py, fac)), qz = ADD(p1z, MUL(Pz, fac));
    const double qn = __dsqrt_rn(ADD(ADD(MUL(qx, qx), MUL(qy, qy)), MUL(qz, qz)));
    if (!(qn > 0.0)) return o;
    const double ex = DIV(qx, qn), ey = DIV(qy, qn), ez = DIV(qz, qn);
    const double ax_ = fabs(ex), ay_ = fabs(ey), az_ = fabs(ez);
    double hx = 0.0, hy = 0.0, hz = 0.0, he;
    if (ax_ <= ay_ && ax_ <= az_) { hx = 1.0; he = ex; } else if (ay_ <= az_) { hy = 1.0; he = ey; } else { hz = 1.0; he = ez; }
    double axx = SUB(hx, MUL(he, ex)), axy = SUB(hy, MUL(he, ey)), axz = SUB(hz, MUL(he, ez));
    const double an = __dsqrt_rn(ADD(ADD(MUL(axx, axx), MUL(axy, axy)), MUL(axz, axz)));
    axx = DIV(axx, an); axy = DIV(axy, an); axz = DIV(axz, an);
    const double bx = SUB(MUL(ey, axz), MUL(ez, axy)), by = SUB(MUL(ez, axx), MUL(ex, axz)), bz_ = SUB(MUL(ex, axy), MUL(ey, axx));
    const double nx = ADD(MUL(cs, ex), MUL(sn, ADD(MUL(ca, axx), MUL(sa, bx))));
    const double ny = ADD(MUL(cs, ey), MUL(sn, ADD(MUL(ca, axy), MUL(sa, by))));
    const double nz = ADD(MUL(cs, ez), MUL(sn, ADD(MUL(ca, axz), MUL(sa, bz_))));
    // boost back (S8c step 2)
    const double cc = ADD(ADD(MUL(Px, nx), MUL(Py, ny)), MUL(Pz, nz));
    const double h = ADD(1.0, DIV(cc, ADD(E, M)));
    const double p3x = MUL(0.5, ADD(MUL(M, nx), MUL(Px, h))), p3y = MUL(0.5, ADD(MUL(M, ny), MUL(Py, h)));
    const double p3z = MUL(0.5, ADD(MUL(M, nz), MUL(Pz, h)));
    const double p4x = SUB(Px, p3x), p4y = SUB(Py, p3y), p4z = SUB(Pz, p3z);
    const double E3 = MUL(0.5, ADD(E, cc));
    const double d13 = ADD(ADD(MUL(p1x, p3x), MUL(p1y, p3y)), MUL(p1z, p3z));
    o.s = s;
    o.t = MUL(-2.0, SUB(MUL(E1, E3), d13));              // t of the constructed momenta: the one Table I sees
    o.u = SUB(-s, o.t);
    o.k = bin_cell_exact(p3x, p3y, p3z, g);
    o.l = bin_cell_exact(p4x, p4y, p4z, g);
    o.flag = (o.k >= 0) && (o.l >= 0);
    o.w = w;
    return o;
}

#undef MUL
#undef ADD
#undef SUB
#undef DIV

__device__ __forceinline__ void red_add_nz(double* dst, double v)
{
    if (v != 0.0) asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst), "d"(v) : "memory");
}

// kDebug: write (j, k, l, flag), (s, t, u) and the weight of every sample of cells [p_begin, p_begin + p_count) of x_begin
template <int kDebug>
__global__ void __launch_bounds__(128) is_kernel(const PaperParams P, const double* __restrict__ m2_cell, double dbg_m2, int* dbg_cells,
                                                 double* dbg_stu, double* dbg_w)
{
    const int lane = threadIdx.x & 31;
    const long long chunks = (P.Ns + 31) / 32;                       // warps per grid point
    const long long n_items = (long long)P.x_count * P.p_count * chunks;
    const long long warp0 = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5, n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long item = warp0; item < n_items; item += n_warps) {
        const int chunk = (int)(item % chunks);
        const long long r1 = item / chunks;
        const int i = P.p_begin + (int)(r1 % P.p_count), xcell = P.x_begin + (int)(r1 / P.p_count);
        const int smp = chunk * 32 + lane;
        const bool valid = smp < P.Ns;
        const double m2 = kDebug ? dbg_m2 : m2_cell[xcell];
        IsSample sm;
        sm.flag = 0; sm.j = 0; sm.k = -1; sm.l = -1; sm.s = sm.t = sm.u = sm.E1E2 = sm.w = 0.0;
        if (valid) sm = gen_sample_is(P.g, P.seed, P.step, (uint32_t)xcell + P.x_rng_offset, (uint32_t)i, (uint32_t)smp, m2);
        if (kDebug) {
            if (valid) {
                const long long q = ((long long)(i - P.p_begin)) * P.Ns + smp;
                dbg_cells[4 * q + 0] = sm.j; dbg_cells[4 * q + 1] = sm.k; dbg_cells[4 * q + 2] = sm.l; dbg_cells[4 * q + 3] = sm.flag;
                dbg_stu[3 * q + 0] = sm.s; dbg_stu[3 * q + 1] = sm.t; dbg_stu[3 * q + 2] = sm.u;
                dbg_w[q] = sm.w;
            }
            continue;
        }
        const double* fx = P.f + (size_t)xcell * P.S * P.Np;
        double* dx = P.dN + (size_t)xcell * P.S * P.Np;
        double d[4][7];
#pragma unroll
        for (int sl = 0; sl < 4; ++sl)
#pragma unroll
            for (int a = 0; a < 7; ++a) d[sl][a] = 0.0;
        if (sm.flag) {
            double fi[7], fj[7], fk[7], fl[7];
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                const int a = P.slot[id];
                const bool on = a >= 0;
                fi[id] = on ? fx[(size_t)a * P.Np + i] : 0.0;     fj[id] = on ? fx[(size_t)a * P.Np + sm.j] : 0.0;
                fk[id] = on ? fx[(size_t)a * P.Np + sm.k] : 0.0;  fl[id] = on ? fx[(size_t)a * P.Np + sm.l] : 0.0;
            }
            const double g4w = P.g4 * (P.Kp / sm.E1E2) * sm.w;      // g^4 K / (E1 E2) x importance weight
            MsqSet M = msq_set<true, true>(sm.s, sm.t, sm.u, m2, g4w);
            if (P.has_ovr) msq_apply_override(M, P.msq_ovr, g4w);
            deposit<-1>(P.mask, fi, fj, fk, fl, M, d[0], d[1], d[2], d[3]);
        }
#pragma unroll
        for (int id = 0; id < 7; ++id) {
            const int a = P.slot[id];
            if (a < 0) continue;                                     // warp-uniform
            double v = d[0][id];                                     // slot 1: the grid point, common to the warp
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red_add_nz(dx + (size_t)a * P.Np + i, v);
            if (sm.flag) {
                red_add_nz(dx + (size_t)a * P.Np + sm.j, d[1][id]);
                red_add_nz(dx + (size_t)a * P.Np + sm.k, d[2][id]);
                red_add_nz(dx + (size_t)a * P.Np + sm.l, d[3][id]);
            }
        }
    }
}

}  // namespace

cudaError_t launch_is_collide(const PaperParams& P, const double* m2_cell, int sms, cudaStream_t st)
{
    const long long warps = (long long)P.x_count * P.p_count * ((P.Ns + 31) / 32);
    if (warps <= 0) return cudaSuccess;
    // grid-stride over warp items in order: launch only the CTAs that are resident at once, so that the warps in flight
    // stay within one or two spatial cells (ncu on a 16-CTAs-per-SM grid: 20 x the compulsory DRAM traffic)
    int per_sm = 1;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, is_kernel<0>, 128, 0);
    if (per_sm < 1) per_sm = 1;
    long long blocks = (warps + 3) / 4;
    if (blocks > (long long)sms * per_sm) blocks = (long long)sms * per_sm;
    is_kernel<0><<<(int)blocks, 128, 0, st>>>(P, m2_cell, 0.0, nullptr, nullptr, nullptr);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_is_debug(const PaperParams& P, double m2, int* cells, double* stu, double* w, int sms, cudaStream_t st)
{
    const long long warps = (long long)P.x_count * P.p_count * ((P.Ns + 31) / 32);
    if (warps <= 0) return cudaSuccess;
    long long blocks = (warps + 3) / 4;
    if (blocks > (long long)sms * 16) blocks = (long long)sms * 16;
    is_kernel<1><<<(int)blocks, 128, 0, st>>>(P, nullptr, m2, cells, stu, w);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
