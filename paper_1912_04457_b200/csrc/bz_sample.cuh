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
    double w;        // weight of the sample (1 for the uniform sampler; importance-sampled t, in-box direction: see below)
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
// gen_sample_words: the same with the four Philox blocks supplied by the caller (w0, w1: blocks 0, 1; wa, wb: blocks
// 2 + kstart, 3 + kstart).  The collision kernel computes them itself on a fresh pass, where the block number, the p1 cell
// and the spatial cell are warp-uniform: of the 20 multiplications of a block only 16 then depend on the lane (round 1 is
// uniform, rounds 2 and 3 have one uniform product each) and the compiler moves the other 4 to the uniform datapath.
__device__ __forceinline__ Sample gen_sample_words(const GridConst& g, const uint32_t (&w0)[4], const uint32_t (&w1)[4],
                                                   const uint32_t (&wa)[4], const uint32_t (&wb)[4], uint32_t kstart, double p1x,
                                                   double p1y, double p1z, double E1)
{
    Sample o;
    o.flag = 0; o.retry = 0; o.k = -1; o.l = -1; o.s = 0.0; o.t = 0.0; o.u = 0.0; o.w = 1.0;
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
__device__ __forceinline__ Sample gen_sample_pair(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xcell,
                                                  uint32_t pcell, uint32_t smp, uint32_t kstart, double p1x, double p1y,
                                                  double p1z, double E1)
{
    uint32_t w0[4], w1[4], wa[4], wb[4];
    philox4x32_10(0u, smp, pcell, xcell, seed, step, w0);
    philox4x32_10(1u, smp, pcell, xcell, seed, step, w1);
    philox4x32_10(2u + kstart, smp, pcell, xcell, seed, step, wa);
    philox4x32_10(3u + kstart, smp, pcell, xcell, seed, step, wb);
    return gen_sample_words(g, w0, w1, wa, wb, kstart, p1x, p1y, p1z, E1);
}

#define BZ_MUL __dmul_rn
#define BZ_ADD __dadd_rn
#define BZ_SUB __dsub_rn
#define BZ_DIV __ddiv_rn

// p2 (Philox blocks 0, 1), E2, s and the cell of p2: the part of S8c step 2-3 all samplers share
__device__ __forceinline__ void sample_p2(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xcell, uint32_t pcell, uint32_t smp,
                                          double p1x, double p1y, double p1z, double E1, double& p2x, double& p2y, double& p2z,
                                          double& E2, double& s, int& j)
{
    uint32_t w0[4], w1[4];
    philox4x32_10(0u, smp, pcell, xcell, seed, step, w0);
    philox4x32_10(1u, smp, pcell, xcell, seed, step, w1);
    const double L52 = g.L * 2.220446049250313e-16;
    p2x = BZ_ADD(g.pmin, BZ_MUL(uniform52_scaled(w0[0], w0[1]), L52));
    p2y = BZ_ADD(g.pmin, BZ_MUL(uniform52_scaled(w0[2], w0[3]), L52));
    p2z = BZ_ADD(g.pmin, BZ_MUL(uniform52_scaled(w1[0], w1[1]), L52));
    E2 = __dsqrt_rn(BZ_ADD(BZ_ADD(BZ_MUL(p2x, p2x), BZ_MUL(p2y, p2y)), BZ_MUL(p2z, p2z)));
    const double d12 = BZ_ADD(BZ_ADD(BZ_MUL(p1x, p2x), BZ_MUL(p1y, p2y)), BZ_MUL(p1z, p2z));
    s = BZ_MUL(2.0, BZ_SUB(BZ_MUL(E1, E2), d12));
    // guarded fast binning (bin_axis_fast), the definition only inside the guard band; p2 is inside by construction, the clamp
    // is the defensive one of S8c step 3
    bool risky = false;
    j = bin_cell_fast(p2x, p2y, p2z, g, risky);
    if (risky || j < 0) {
        bool in;
        int a = bin_axis_exact(p2x, g, in), b = bin_axis_exact(p2y, g, in), c = bin_axis_exact(p2z, g, in);
        a = min(max(a, 0), g.n - 1); b = min(max(b, 0), g.n - 1); c = min(max(c, 0), g.n - 1);
        j = a + g.n * (b + g.n * c);
    }
}

// boost of the CM pair (M/2)(1, n) back, t, and the cells of p3, p4 (S8c steps 2-3)
__device__ __forceinline__ void sample_boost(const GridConst& g, double p1x, double p1y, double p1z, double E1, double Px, double Py,
                                             double Pz, double E, double M, double nx, double ny, double nz, Sample& o)
{
    const double cc = BZ_ADD(BZ_ADD(BZ_MUL(Px, nx), BZ_MUL(Py, ny)), BZ_MUL(Pz, nz));
    const double h = BZ_ADD(1.0, BZ_DIV(cc, BZ_ADD(E, M)));
    const double p3x = BZ_MUL(0.5, BZ_ADD(BZ_MUL(M, nx), BZ_MUL(Px, h))), p3y = BZ_MUL(0.5, BZ_ADD(BZ_MUL(M, ny), BZ_MUL(Py, h)));
    const double p3z = BZ_MUL(0.5, BZ_ADD(BZ_MUL(M, nz), BZ_MUL(Pz, h)));
    const double p4x = BZ_SUB(Px, p3x), p4y = BZ_SUB(Py, p3y), p4z = BZ_SUB(Pz, p3z);
    const double E3 = BZ_MUL(0.5, BZ_ADD(E, cc));
    const double d13 = BZ_ADD(BZ_ADD(BZ_MUL(p1x, p3x), BZ_MUL(p1y, p3y)), BZ_MUL(p1z, p3z));
    o.t = BZ_MUL(-2.0, BZ_SUB(BZ_MUL(E1, E3), d13));                  // t of the constructed momenta: the one Table I sees
    o.u = BZ_SUB(-o.s, o.t);
    bool risky = false;
    o.k = bin_cell_fast(p3x, p3y, p3z, g, risky);
    o.l = bin_cell_fast(p4x, p4y, p4z, g, risky);
    if (risky) {                                         // ~4e-5 of the samples: repeat with the definition
        o.k = bin_cell_exact(p3x, p3y, p3z, g);
        o.l = bin_cell_exact(p4x, p4y, p4z, g);
    }
    o.flag = (o.k >= 0) && (o.l >= 0);
}

// orthonormal pair (e1, e2) around the unit vector a: h = the coordinate axis with the smallest |a_c| (first on ties),
// e1 = (h - (h.a) a)/|..|, e2 = a x e1
__device__ __forceinline__ void sample_frame(double ax, double ay, double az, double& e1x, double& e1y, double& e1z, double& e2x,
                                             double& e2y, double& e2z)
{
    const double fx = fabs(ax), fy = fabs(ay), fz = fabs(az);
    double hx = 0.0, hy = 0.0, hz = 0.0, ha;
    if (fx <= fy && fx <= fz) { hx = 1.0; ha = ax; } else if (fy <= fz) { hy = 1.0; ha = ay; } else { hz = 1.0; ha = az; }
    e1x = BZ_SUB(hx, BZ_MUL(ha, ax)); e1y = BZ_SUB(hy, BZ_MUL(ha, ay)); e1z = BZ_SUB(hz, BZ_MUL(ha, az));
    const double en = __dsqrt_rn(BZ_ADD(BZ_ADD(BZ_MUL(e1x, e1x), BZ_MUL(e1y, e1y)), BZ_MUL(e1z, e1z)));
    e1x = BZ_DIV(e1x, en); e1y = BZ_DIV(e1y, en); e1z = BZ_DIV(e1z, en);
    e2x = BZ_SUB(BZ_MUL(ay, e1z), BZ_MUL(az, e1y)); e2y = BZ_SUB(BZ_MUL(az, e1x), BZ_MUL(ax, e1z)); e2z = BZ_SUB(BZ_MUL(ax, e1y), BZ_MUL(ay, e1x));
}

// ---- NEXT rank 3 (S8f): importance sampling of the t/u-channel peaks of Table I (oracle: gen_sample_is).
//   p(t) = (1/2) [g(t) + g(-s - t)],  g(t) = 1 / ((m^2 - t)^2 (1/m^2 - 1/(s + m^2))),  weight (1/s)/p(t);
//   Philox blocks 0, 1 (p2), 96 (t, branch) and 97 + k (azimuth attempt k: first point of the sequence inside the unit
//   disc, (cos, sin) = (v1^2 - v2^2, 2 v1 v2)/q; (1, 0) after 62 failures).  Attempts kstart and kstart + 1 per call,
//   retry = 1 if both fail, like gen_sample_pair.  m2 <= 0: t uniform, weight 1.
__device__ __forceinline__ Sample gen_sample_is_pair(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xcell, uint32_t pcell,
                                                     uint32_t smp, uint32_t kstart, double p1x, double p1y, double p1z, double E1, double m2)
{
    Sample o;
    o.flag = 0; o.retry = 0; o.k = -1; o.l = -1; o.s = 0.0; o.t = 0.0; o.u = 0.0; o.w = 0.0;
    double p2x, p2y, p2z, E2, s;
    sample_p2(g, seed, step, xcell, pcell, smp, p1x, p1y, p1z, E1, p2x, p2y, p2z, E2, s, o.j);
    o.E1E2 = E1 * E2;
    if (!(s > 0.0)) return o;
    uint32_t w2[4], wa[4], wb[4];
    philox4x32_10(96u, smp, pcell, xcell, seed, step, w2);
    philox4x32_10(97u + kstart, smp, pcell, xcell, seed, step, wa);
    philox4x32_10(98u + kstart, smp, pcell, xcell, seed, step, wb);
    const double ut = uniform52(w2[0], w2[1]), ub = uniform52(w2[2], w2[3]);
    double t, w;
    if (m2 > 0.0) {
        const double lo = BZ_DIV(1.0, BZ_ADD(s, m2)), hi = BZ_DIV(1.0, m2);
        const double r = BZ_ADD(lo, BZ_MUL(ut, BZ_SUB(hi, lo)));
        const double tt = BZ_SUB(m2, BZ_DIV(1.0, r));
        t = ub < 0.5 ? tt : BZ_SUB(-s, tt);
        const double dt_ = BZ_SUB(m2, t), du_ = BZ_SUB(m2, BZ_SUB(-s, t));
        const double norm = BZ_SUB(hi, lo);
        const double pt = BZ_MUL(0.5, BZ_ADD(BZ_DIV(1.0, BZ_MUL(BZ_MUL(dt_, dt_), norm)), BZ_DIV(1.0, BZ_MUL(BZ_MUL(du_, du_), norm))));
        w = BZ_DIV(BZ_DIV(1.0, s), pt);
    } else {
        t = BZ_MUL(-s, ut);
        w = 1.0;
    }
    double cs = BZ_ADD(1.0, BZ_DIV(BZ_MUL(2.0, t), s));
    if (cs > 1.0) cs = 1.0;
    if (cs < -1.0) cs = -1.0;
    const double sn = __dsqrt_rn(BZ_SUB(1.0, BZ_MUL(cs, cs)));
    // azimuth
    double ca = 1.0, sa = 0.0;
    bool found = kstart >= 62u;
    if (!found) {
        double v1 = symmetric52(wa[0], wa[1]), v2 = symmetric52(wa[2], wa[3]);
        double q = BZ_ADD(BZ_MUL(v1, v1), BZ_MUL(v2, v2));
        found = q < 1.0 && q > 0.0;
        if (!found && kstart + 1u < 62u) {
            v1 = symmetric52(wb[0], wb[1]); v2 = symmetric52(wb[2], wb[3]);
            q = BZ_ADD(BZ_MUL(v1, v1), BZ_MUL(v2, v2));
            found = q < 1.0 && q > 0.0;
        }
        if (found) {
            ca = BZ_DIV(BZ_SUB(BZ_MUL(v1, v1), BZ_MUL(v2, v2)), q);
            sa = BZ_DIV(BZ_MUL(BZ_MUL(2.0, v1), v2), q);
        }
    }
    if (!found) { o.retry = 1; return o; }
    // CM direction of p1 and an orthonormal basis around it
    const double Px = BZ_ADD(p1x, p2x), Py = BZ_ADD(p1y, p2y), Pz = BZ_ADD(p1z, p2z);
    const double E = BZ_ADD(E1, E2), M = __dsqrt_rn(s);
    const double Pp1 = BZ_ADD(BZ_ADD(BZ_MUL(Px, p1x), BZ_MUL(Py, p1y)), BZ_MUL(Pz, p1z));
    const double fac = BZ_DIV(BZ_SUB(BZ_DIV(Pp1, BZ_ADD(E, M)), E1), M);
    const double qx = BZ_ADD(p1x, BZ_MUL(Px, fac)), qy = BZ_ADD(p1y, BZ_MUL(Py, fac)), qz = BZ_ADD(p1z, BZ_MUL(Pz, fac));
    const double qn = __dsqrt_rn(BZ_ADD(BZ_ADD(BZ_MUL(qx, qx), BZ_MUL(qy, qy)), BZ_MUL(qz, qz)));
    if (!(qn > 0.0)) return o;
    const double ex = BZ_DIV(qx, qn), ey = BZ_DIV(qy, qn), ez = BZ_DIV(qz, qn);
    double ax, ay, az, bx, by, bz_;
    sample_frame(ex, ey, ez, ax, ay, az, bx, by, bz_);
    const double nx = BZ_ADD(BZ_MUL(cs, ex), BZ_MUL(sn, BZ_ADD(BZ_MUL(ca, ax), BZ_MUL(sa, bx))));
    const double ny = BZ_ADD(BZ_MUL(cs, ey), BZ_MUL(sn, BZ_ADD(BZ_MUL(ca, ay), BZ_MUL(sa, by))));
    const double nz = BZ_ADD(BZ_MUL(cs, ez), BZ_MUL(sn, BZ_ADD(BZ_MUL(ca, az), BZ_MUL(sa, bz_))));
    o.s = s;
    sample_boost(g, p1x, p1y, p1z, E1, Px, Py, Pz, E, M, nx, ny, nz, o);
    o.w = w;
    return o;
}

// ---- NEXT rank 3 (S8f), other half: the CM direction from the tightest of the three zones |a_c . n| <= beta_c outside
// which p3 or p4 leaves the momentum box (oracle: gen_sample_box).  p3 = P/2 + A n with rows A_c = (M e_c + P_c P/(E + M))/2,
// |A_c| = sqrt(s + P_c^2)/2; both legs stay in on axis c iff |A_c . n| <= b_c = L/2 - |P_c/2 - (pmin + L/2)|.  The zone with
// the smallest beta_c = min(1, b_c/|A_c|) is sampled exactly (Archimedes: z = a . n uniform on [-beta, beta], area fraction
// beta = the sample's weight), the other two by rejection.  Same Philox blocks (0, 1, 2 + k) and the same Marsaglia
// acceptance q < 1 as gen_sample_pair: z = beta (1 - 2 q), (cos, sin) = (v1, v2)/sqrt(q).
__device__ __forceinline__ Sample gen_sample_box_pair(const GridConst& g, uint32_t seed, uint32_t step, uint32_t xcell, uint32_t pcell,
                                                      uint32_t smp, uint32_t kstart, double p1x, double p1y, double p1z, double E1)
{
    Sample o;
    o.flag = 0; o.retry = 0; o.k = -1; o.l = -1; o.s = 0.0; o.t = 0.0; o.u = 0.0; o.w = 0.0;
    double p2x, p2y, p2z, E2, s;
    sample_p2(g, seed, step, xcell, pcell, smp, p1x, p1y, p1z, E1, p2x, p2y, p2z, E2, s, o.j);
    o.E1E2 = E1 * E2;
    if (!(s > 0.0)) return o;
    const double P[3] = { BZ_ADD(p1x, p2x), BZ_ADD(p1y, p2y), BZ_ADD(p1z, p2z) };
    const double E = BZ_ADD(E1, E2), M = __dsqrt_rn(s), EM = BZ_ADD(E, M);
    const double B = BZ_MUL(0.5, g.L), pc0 = BZ_ADD(g.pmin, B);
    double beta = 2.0, An = 0.0;
    int cs = 0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double b = BZ_SUB(B, fabs(BZ_SUB(BZ_MUL(0.5, P[d]), pc0)));
        const double an = BZ_MUL(0.5, __dsqrt_rn(BZ_ADD(s, BZ_MUL(P[d], P[d]))));
        double bt = BZ_DIV(b, an);
        if (bt > 1.0) bt = 1.0;
        if (bt < beta) { beta = bt; cs = d; An = an; }
    }
    if (!(beta > 0.0)) return o;
    const double Pc = cs == 0 ? P[0] : (cs == 1 ? P[1] : P[2]);
    const double gq = BZ_DIV(Pc, EM);
    double a[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        const double v = d == cs ? BZ_MUL(0.5, BZ_ADD(M, BZ_MUL(P[d], gq))) : BZ_MUL(0.5, BZ_MUL(P[d], gq));
        a[d] = BZ_DIV(v, An);
    }
    double e1x, e1y, e1z, e2x, e2y, e2z;
    sample_frame(a[0], a[1], a[2], e1x, e1y, e1z, e2x, e2y, e2z);
    // direction
    double zz = 0.0, rho = 1.0, cphi = 1.0, sphi = 0.0;          // after 62 failures: n = e1
    bool found = kstart >= 62u;
    if (!found) {
        uint32_t wa[4], wb[4];
        philox4x32_10(2u + kstart, smp, pcell, xcell, seed, step, wa);
        philox4x32_10(3u + kstart, smp, pcell, xcell, seed, step, wb);
        double v1 = symmetric52(wa[0], wa[1]), v2 = symmetric52(wa[2], wa[3]);
        double q = BZ_ADD(BZ_MUL(v1, v1), BZ_MUL(v2, v2));
        found = q < 1.0;
        if (!found && kstart + 1u < 62u) {
            v1 = symmetric52(wb[0], wb[1]); v2 = symmetric52(wb[2], wb[3]);
            q = BZ_ADD(BZ_MUL(v1, v1), BZ_MUL(v2, v2));
            found = q < 1.0;
        }
        if (found) {
            zz = BZ_MUL(beta, BZ_SUB(1.0, BZ_MUL(2.0, q)));
            rho = __dsqrt_rn(BZ_SUB(1.0, BZ_MUL(zz, zz)));
            const double rq = __dsqrt_rn(q);
            cphi = BZ_DIV(v1, rq); sphi = BZ_DIV(v2, rq);
        }
    }
    if (!found) { o.retry = 1; return o; }
    const double nx = BZ_ADD(BZ_MUL(zz, a[0]), BZ_MUL(rho, BZ_ADD(BZ_MUL(cphi, e1x), BZ_MUL(sphi, e2x))));
    const double ny = BZ_ADD(BZ_MUL(zz, a[1]), BZ_MUL(rho, BZ_ADD(BZ_MUL(cphi, e1y), BZ_MUL(sphi, e2y))));
    const double nz = BZ_ADD(BZ_MUL(zz, a[2]), BZ_MUL(rho, BZ_ADD(BZ_MUL(cphi, e1z), BZ_MUL(sphi, e2z))));
    o.s = s;
    sample_boost(g, p1x, p1y, p1z, E1, P[0], P[1], P[2], E, M, nx, ny, nz, o);
    o.w = beta;
    return o;
}

#undef BZ_MUL
#undef BZ_ADD
#undef BZ_SUB
#undef BZ_DIV

}  // namespace bz
