// bz_sample.cuh -- Philox4x32-10 and the kinematic sample (S8c steps 1-3), device side.
//
// Bit-exactness contract (NS, S8c step 2): every floating-point operation that can influence a sampled cell
// index is a single correctly rounded IEEE operation, in the association order S8c writes, with no FMA
// contraction.  The __d*_rn intrinsics are never contracted by nvcc, whatever -fmad says.
#pragma once
#include <cstdint>

namespace bz {

struct GridConst {          // S8c step 0, computed once on the host in fp64
    int n;                  // momentum cells per axis
    double pmin, L, dp;     // box edge, box length pmax - pmin, cell width L/n
    double inv_dp;          // n / L, only for the guarded fast path of the binning
};

// ---- S8c step 1: Philox4x32-10 (Salmon et al. 2011), key = (seed, step), counter = (blk, sample, pcell, xcell)
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0, n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// U(a,b) = (m + 1/2) 2^-52 with the 52-bit integer m = (a>>6)<<26 | (b>>6).  2^52 + m is assembled in the mantissa,
// then 2^52 - 1/2 is subtracted: both steps are exact, the product with 2^-52 is exact.
__device__ __forceinline__ double uniform52(uint32_t a, uint32_t b)
{
    const double d = __hiloint2double((int)(0x43300000u | (a >> 12)), (int)(((a >> 6) << 26) | (b >> 6)));
    return __dmul_rn(__dadd_rn(d, -4503599627370495.5), 2.220446049250313e-16);
}

// ---- S8c step 3: cell index along one axis.  q = (p - pmin)/dp, inside iff 0 <= q < n, idx = floor(q).
// The division is replaced by a multiplication whenever the product is safely away from an integer (its error
// is < 1e-13 for |q| < 1e3, the guard is 1e-9), so the result equals the division's bit for bit.
__device__ __forceinline__ int bin_axis(double p, const GridConst& g, bool& inside)
{
    const double x = __dsub_rn(p, g.pmin);
    double q = __dmul_rn(x, g.inv_dp);
    double fl = floor(q);
    const double fr = q - fl;
    if (!(fr > 1e-9 && fr < 1.0 - 1e-9) || !(fabs(q) < 1e3)) {
        q = __ddiv_rn(x, g.dp);
        fl = floor(q);
    }
    inside = (q >= 0.0) && (q < (double)g.n);
    return (int)fl;
}

__device__ __forceinline__ int bin_cell(double px, double py, double pz, const GridConst& g)
{
    bool ix, iy, iz;
    const int a = bin_axis(px, g, ix), b = bin_axis(py, g, iy), c = bin_axis(pz, g, iz);
    return (ix && iy && iz) ? a + g.n * (b + g.n * c) : -1;
}

struct Sample {
    int flag, j, k, l;
    double s, t, u, E1E2;
};

// One kinematic sample (S8c step 2).  p1 = centre of pcell; E1 passed in (same for all samples of the cell).
__device__ __forceinline__ Sample gen_sample(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xcell,
                                             uint32_t pcell, uint32_t smp, double p1x, double p1y, double p1z,
                                             double E1)
{
    Sample o;
    o.flag = 0; o.k = -1; o.l = -1; o.s = 0.0; o.t = 0.0; o.u = 0.0;
    uint32_t w[4];
    philox4x32_10(0u, smp, pcell, xcell, seed, step, w);
    const double u0 = uniform52(w[0], w[1]), u1 = uniform52(w[2], w[3]);
    philox4x32_10(1u, smp, pcell, xcell, seed, step, w);
    const double u2 = uniform52(w[0], w[1]);
    const double p2x = __dadd_rn(g.pmin, __dmul_rn(u0, g.L));
    const double p2y = __dadd_rn(g.pmin, __dmul_rn(u1, g.L));
    const double p2z = __dadd_rn(g.pmin, __dmul_rn(u2, g.L));
    const double E2 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p2x, p2x), __dmul_rn(p2y, p2y)), __dmul_rn(p2z, p2z)));
    const double d12 = __dadd_rn(__dadd_rn(__dmul_rn(p1x, p2x), __dmul_rn(p1y, p2y)), __dmul_rn(p1z, p2z));
    const double s = __dmul_rn(2.0, __dsub_rn(__dmul_rn(E1, E2), d12));
    {   // p2 is inside by construction; clamp defensively
        bool in;
        int a = bin_axis(p2x, g, in), b = bin_axis(p2y, g, in), c = bin_axis(p2z, g, in);
        a = min(max(a, 0), g.n - 1); b = min(max(b, 0), g.n - 1); c = min(max(c, 0), g.n - 1);
        o.j = a + g.n * (b + g.n * c);
    }
    o.E1E2 = E1 * E2;
    if (!(s > 0.0)) return o;

    // Marsaglia: first attempt k with q = v1^2 + v2^2 < 1
    double nx = 0.0, ny = 0.0, nz = 1.0;
    for (uint32_t k = 0; k < 62u; ++k) {
        philox4x32_10(2u + k, smp, pcell, xcell, seed, step, w);
        const double v1 = __dadd_rn(__dmul_rn(2.0, uniform52(w[0], w[1])), -1.0);
        const double v2 = __dadd_rn(__dmul_rn(2.0, uniform52(w[2], w[3])), -1.0);
        const double q = __dadd_rn(__dmul_rn(v1, v1), __dmul_rn(v2, v2));
        if (q < 1.0) {
            const double r = __dsqrt_rn(__dsub_rn(1.0, q));
            nx = __dmul_rn(__dmul_rn(2.0, v1), r);
            ny = __dmul_rn(__dmul_rn(2.0, v2), r);
            nz = __dsub_rn(1.0, __dmul_rn(2.0, q));
            break;
        }
    }
    const double Px = __dadd_rn(p1x, p2x), Py = __dadd_rn(p1y, p2y), Pz = __dadd_rn(p1z, p2z);
    const double E = __dadd_rn(E1, E2), M = __dsqrt_rn(s);
    const double cc = __dadd_rn(__dadd_rn(__dmul_rn(Px, nx), __dmul_rn(Py, ny)), __dmul_rn(Pz, nz));
    const double h = __dadd_rn(1.0, __ddiv_rn(cc, __dadd_rn(E, M)));
    const double p3x = __dmul_rn(0.5, __dadd_rn(__dmul_rn(M, nx), __dmul_rn(Px, h)));
    const double p3y = __dmul_rn(0.5, __dadd_rn(__dmul_rn(M, ny), __dmul_rn(Py, h)));
    const double p3z = __dmul_rn(0.5, __dadd_rn(__dmul_rn(M, nz), __dmul_rn(Pz, h)));
    const double p4x = __dsub_rn(Px, p3x), p4y = __dsub_rn(Py, p3y), p4z = __dsub_rn(Pz, p3z);
    const double E3 = __dmul_rn(0.5, __dadd_rn(E, cc));
    const double d13 = __dadd_rn(__dadd_rn(__dmul_rn(p1x, p3x), __dmul_rn(p1y, p3y)), __dmul_rn(p1z, p3z));
    const double t = __dmul_rn(-2.0, __dsub_rn(__dmul_rn(E1, E3), d13));
    const double u = __dsub_rn(-s, t);
    o.s = s; o.t = t; o.u = u;
    o.k = bin_cell(p3x, p3y, p3z, g);
    o.l = bin_cell(p4x, p4y, p4z, g);
    o.flag = (o.k >= 0) && (o.l >= 0);
    return o;
}

// centre of cell i along one axis: pmin + (i + 0.5) * dp, as S8c step 0 writes it
__device__ __forceinline__ double cell_centre(const GridConst& g, int i)
{
    return __dadd_rn(g.pmin, __dmul_rn(__dadd_rn((double)i, 0.5), g.dp));
}

}  // namespace bz
