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
    // guarded fast path of the binning: floor(p * bin_a + bin_b) ~ floor(2^bin_shift * (p - pmin) / dp)
    double bin_a, bin_b;
    int bin_shift;
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
// The same uniform times 2^52, i.e. m + 1/2 (exact): a product u * c equals fl((m + 1/2) * (c 2^-52)) bit for bit, because
// scaling by 2^-52 is exact on either side of the single rounding.
__device__ __forceinline__ double uniform52_scaled(uint32_t a, uint32_t b)
{
    const double d = __hiloint2double((int)(0x43300000u | (a >> 12)), (int)(((a >> 6) << 26) | (b >> 6)));
    return __dadd_rn(d, -4503599627370495.5);
}
// v = 2 U - 1 = (m + 1/2) 2^-51 - 1 = (2 m + 1 - 2^52) 2^-52: an odd multiple of 2^-52 below 1 in magnitude, exactly
// representable, so S8c's two rounded steps "2 * u" and "- 1" are both exact and this single fused one gives the same bits
__device__ __forceinline__ double symmetric52(uint32_t a, uint32_t b)
{
    const double d = __hiloint2double((int)(0x43300000u | (a >> 12)), (int)(((a >> 6) << 26) | (b >> 6)));
    return fma(__dadd_rn(d, -4503599627370495.5), 4.440892098500626e-16, -1.0);
}

// ---- S8c step 3: cell index along one axis.  q = (p - pmin)/dp, inside iff 0 <= q < n, idx = floor(q).
// Exact form (the definition): one correctly rounded subtraction and division.
__device__ __forceinline__ int bin_axis_exact(double p, const GridConst& g, bool& inside)
{
    const double q = __ddiv_rn(__dsub_rn(p, g.pmin), g.dp);
    inside = (q >= 0.0) && (q < (double)g.n);
    return (int)floor(q);
}
__device__ __forceinline__ int bin_cell_exact(double px, double py, double pz, const GridConst& g)
{
    bool ix, iy, iz;
    const int a = bin_axis_exact(px, g, ix), b = bin_axis_exact(py, g, iy), c = bin_axis_exact(pz, g, iz);
    return (ix && iy && iz) ? a + g.n * (b + g.n * c) : -1;
}
// Fast form: t = floor(2^k q') with q' = fma(p, 2^k/dp, -pmin 2^k/dp), |q' - q| 2^k < 1e-6 (the host picks k <= 20 so that
// 2^k |q| < 2^31 for every reachable momentum; a saturated conversion lands outside [0, n) like the true q).
// idx = t >> k and the inside test are those of the exact q unless t is within 2 units of a multiple of 2^k; then
// `risky` is set and the caller repeats the binning with the exact form.  Cost: 1 DFMA + 1 F2I + 5 integer ops.
__device__ __forceinline__ int bin_axis_fast(double p, const GridConst& g, bool& inside, bool& risky)
{
    const int t = __double2int_rd(fma(p, g.bin_a, g.bin_b));
    const unsigned mask = (1u << g.bin_shift) - 1u;
    const int idx = t >> g.bin_shift;
    risky = risky || (((unsigned)(t - 2) & mask) > mask - 4u);
    inside = (unsigned)idx < (unsigned)g.n;
    return idx;
}
__device__ __forceinline__ int bin_cell_fast(double px, double py, double pz, const GridConst& g, bool& risky)
{
    bool ix, iy, iz;
    const int a = bin_axis_fast(px, g, ix, risky), b = bin_axis_fast(py, g, iy, risky), c = bin_axis_fast(pz, g, iz, risky);
    return (ix && iy && iz) ? a + g.n * (b + g.n * c) : -1;
}

struct Sample {
    int flag;        // 1: both outgoing legs in the box and s > 0 -> the sample deposits
    int retry;       // 1: s > 0 but neither Marsaglia attempt of this call was accepted: call again with kstart + 2
    int j, k, l;     // cells of p2, p3, p4 (k = l = -1 when !(s > 0); k or l = -1 when that leg leaves the box)
    double s, t, u, E1E2;
};

// momentum and energy of the centre of cell i (S8c step 0 / step 2)
__device__ __forceinline__ double cell_centre(const GridConst& g, int i)
{
    return __dadd_rn(g.pmin, __dmul_rn(__dadd_rn((double)i, 0.5), g.dp));
}
__device__ __forceinline__ void cell_kinematics(const GridConst& g, int pcell, double& p1x, double& p1y, double& p1z, double& E1)
{
    const int n = g.n, ipx = pcell % n, ipy = (pcell / n) % n, ipz = pcell / (n * n);
    p1x = cell_centre(g, ipx); p1y = cell_centre(g, ipy); p1z = cell_centre(g, ipz);
    E1 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p1x, p1x), __dmul_rn(p1y, p1y)), __dmul_rn(p1z, p1z)));
}

// One kinematic sample (S8c steps 1-3) with Marsaglia attempts kstart and kstart + 1 (kstart even).  All four Philox
// blocks (0, 1, 2 + kstart, 3 + kstart) are independent and issued together, there is no data-dependent loop: a lane
// whose two attempts both fail (probability 0.046) reports retry = 1 and is finished by a later call.  The sequence
// of attempts, and therefore the accepted direction, is exactly that of the one-attempt-at-a-time loop of S8c.
__device__ __forceinline__ Sample gen_sample_pair(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xcell,
                                                  uint32_t pcell, uint32_t smp, uint32_t kstart, double p1x, double p1y,
                                                  double p1z, double E1)
{
    Sample o;
    o.flag = 0; o.retry = 0; o.k = -1; o.l = -1; o.s = 0.0; o.t = 0.0; o.u = 0.0;
    uint32_t w0[4], w1[4], wa[4], wb[4];
    philox4x32_10(0u, smp, pcell, xcell, seed, step, w0);
    philox4x32_10(1u, smp, pcell, xcell, seed, step, w1);
    philox4x32_10(2u + kstart, smp, pcell, xcell, seed, step, wa);
    philox4x32_10(3u + kstart, smp, pcell, xcell, seed, step, wb);
    const double L52 = g.L * 2.220446049250313e-16;       // L 2^-52, exact
    const double p2x = __dadd_rn(g.pmin, __dmul_rn(uniform52_scaled(w0[0], w0[1]), L52));
    const double p2y = __dadd_rn(g.pmin, __dmul_rn(uniform52_scaled(w0[2], w0[3]), L52));
    const double p2z = __dadd_rn(g.pmin, __dmul_rn(uniform52_scaled(w1[0], w1[1]), L52));
    const double E2 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p2x, p2x), __dmul_rn(p2y, p2y)), __dmul_rn(p2z, p2z)));
    const double d12 = __dadd_rn(__dadd_rn(__dmul_rn(p1x, p2x), __dmul_rn(p1y, p2y)), __dmul_rn(p1z, p2z));
    const double e12 = __dmul_rn(E1, E2);
    const double s = __dmul_rn(2.0, __dsub_rn(e12, d12));
    o.E1E2 = e12;

    // Marsaglia: attempt k is accepted iff q_k = v1^2 + v2^2 < 1; after 62 failures the direction is (0, 0, 1)
    double v1 = symmetric52(wa[0], wa[1]);
    double v2 = symmetric52(wa[2], wa[3]);
    double q = __dadd_rn(__dmul_rn(v1, v1), __dmul_rn(v2, v2));
    const double v1b = symmetric52(wb[0], wb[1]);
    const double v2b = symmetric52(wb[2], wb[3]);
    const double qb = __dadd_rn(__dmul_rn(v1b, v1b), __dmul_rn(v2b, v2b));
    bool found = q < 1.0;
    if (!found) { v1 = v1b; v2 = v2b; q = qb; found = qb < 1.0; }
    double nx, ny, nz;
    {
        const double r = __dsqrt_rn(__dsub_rn(1.0, found ? q : 0.0));
        nx = __dmul_rn(__dmul_rn(2.0, v1), r);
        ny = __dmul_rn(__dmul_rn(2.0, v2), r);
        nz = __dsub_rn(1.0, __dmul_rn(2.0, q));
    }
    if (kstart >= 62u) { nx = 0.0; ny = 0.0; nz = 1.0; found = true; }

    const double Px = __dadd_rn(p1x, p2x), Py = __dadd_rn(p1y, p2y), Pz = __dadd_rn(p1z, p2z);
    const double E = __dadd_rn(E1, E2), M = __dsqrt_rn(s > 0.0 ? s : 0.0);
    const double cc = __dadd_rn(__dadd_rn(__dmul_rn(Px, nx), __dmul_rn(Py, ny)), __dmul_rn(Pz, nz));
    const double h = __dadd_rn(1.0, __ddiv_rn(cc, __dadd_rn(E, M)));
    const double p3x = __dmul_rn(0.5, __dadd_rn(__dmul_rn(M, nx), __dmul_rn(Px, h)));
    const double p3y = __dmul_rn(0.5, __dadd_rn(__dmul_rn(M, ny), __dmul_rn(Py, h)));
    const double p3z = __dmul_rn(0.5, __dadd_rn(__dmul_rn(M, nz), __dmul_rn(Pz, h)));
    const double p4x = __dsub_rn(Px, p3x), p4y = __dsub_rn(Py, p3y), p4z = __dsub_rn(Pz, p3z);
    const double E3 = __dmul_rn(0.5, __dadd_rn(E, cc));
    const double d13 = __dadd_rn(__dadd_rn(__dmul_rn(p1x, p3x), __dmul_rn(p1y, p3y)), __dmul_rn(p1z, p3z));
    const double t = __dmul_rn(-2.0, __dsub_rn(__dmul_rn(E1, E3), d13));

    bool risky = false;
    int j = bin_cell_fast(p2x, p2y, p2z, g, risky);
    int k = bin_cell_fast(p3x, p3y, p3z, g, risky);
    int l = bin_cell_fast(p4x, p4y, p4z, g, risky);
    if (risky) {                                         // ~4e-5 of the samples: repeat with the definition
        j = bin_cell_exact(p2x, p2y, p2z, g);
        k = bin_cell_exact(p3x, p3y, p3z, g);
        l = bin_cell_exact(p4x, p4y, p4z, g);
    }
    if (j < 0) {                                         // p2 is inside by construction; clamp defensively (S8c step 3)
        bool in;
        int a = bin_axis_exact(p2x, g, in), b = bin_axis_exact(p2y, g, in), c = bin_axis_exact(p2z, g, in);
        a = min(max(a, 0), g.n - 1); b = min(max(b, 0), g.n - 1); c = min(max(c, 0), g.n - 1);
        j = a + g.n * (b + g.n * c);
    }
    o.j = j;
    if (!(s > 0.0)) return o;                            // p1 = 0 cell, exact collinearity, rounding: no deposit, no retry
    if (!found) { o.retry = 1; return o; }
    o.s = s; o.t = t; o.u = __dsub_rn(-s, t);
    o.k = k; o.l = l;
    o.flag = (k >= 0) && (l >= 0);
    return o;
}

}  // namespace bz
