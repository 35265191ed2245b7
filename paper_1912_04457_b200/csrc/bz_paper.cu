// bz_paper.cu -- NEXT rank 1 of SURVEY.md 8f: the paper's own collision path.
//   Grid point p (cell centre) = the OUTGOING particle d of Eq. 5; integration variables (k1x, k1y, k3x, k3y,
//   k3z) uniform in the momentum box (Eq. 20); k1z from the two roots of E1 + E2 = E3 + Ep with weight 1/|J|
//   (Eq. 17-19); k2 = k3 + p - k1; massive dispersion E^a = sqrt(p^2 + m_a^2(x)) from the thermal masses of
//   Eq. 8-9; symmetrical sampling (Eq. 22): the same weight goes to the cells of k1, k2 (-) and k3, p (+).
// With masses the kinematics depend on the species of the four legs, so a sample is NOT shared by all channels as in
// the hot path: the ordered channels (S8c step 5) are grouped by their tuple of mass classes (g, u, d, s) and every
// group solves its own roots.  One lane per (spatial cell, grid point, sample) for the first stage of the root solving; its
// candidates, the kept roots and the (root, channel) pairs go through per-warp rings to later phases that run on full
// warps (paper_queue_kernel); deposits are fp64 reductions (RED.E.ADD.F64) into dF, which a second kernel divides by N_a.  Everything that decides a cell index
// uses single correctly rounded operations in the association order of the oracle (bit-exact sampled cells).
#include <vector>

#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

// ---------------------------------------------------------------------------------------------- host: channel table
// Ordered channels a(k1) b(k2) -> c(k3) d(p) of the active species (Eq. 3-4; S8c step 5), sorted by the mass
// classes of the four legs.  kind: 0 A, 1 11, 2 1B, 3 ANN, 4 QQGG, 5 QG, 6 GG (Table I); crossed: M(s,u,t).
namespace {

int cls_of_id(int id) { return id == 0 ? 0 : 1 + (id - 1) / 2; }
int anti_of_id(int id) { return (id & 1) ? id + 1 : id - 1; }

}  // namespace

void build_paper_channels(const int* species, int S, std::vector<PaperChannel>& table, std::vector<PaperGroup>& groups)
{
    int slot[7];
    for (int id = 0; id < 7; ++id) slot[id] = -1;
    for (int a = 0; a < S; ++a) slot[species[a]] = a;
    std::vector<PaperChannel> all;
    auto emit = [&](int ia, int ib, int ic, int id, int kind, int crossed) {
        PaperChannel ch;
        ch.a = (unsigned char)slot[ia]; ch.b = (unsigned char)slot[ib]; ch.c = (unsigned char)slot[ic]; ch.d = (unsigned char)slot[id];
        ch.kind = (unsigned char)kind; ch.crossed = (unsigned char)crossed;
        ch.glue = (unsigned char)((ia == 0) | (ib == 0) << 1 | (ic == 0) << 2 | (id == 0) << 3);
        ch.key = (unsigned char)(cls_of_id(ia) | cls_of_id(ib) << 2 | cls_of_id(ic) << 4 | cls_of_id(id) << 6);
        all.push_back(ch);
    };
    auto pair_active = [&](int fl) { return slot[1 + 2 * fl] >= 0 && slot[2 + 2 * fl] >= 0; };
    for (int x = 0; x < S; ++x) for (int y = 0; y < S; ++y) {
        const int ia = species[x], ib = species[y];
        const bool ga = ia == 0, gb = ib == 0;
        if (ga && gb) {                                           // g g -> g g; g g -> q qbar in both orders
            emit(0, 0, 0, 0, 6, 0);
            for (int fl = 0; fl < 3; ++fl) if (pair_active(fl)) { emit(0, 0, 1 + 2 * fl, 2 + 2 * fl, 4, 0); emit(0, 0, 2 + 2 * fl, 1 + 2 * fl, 4, 0); }
        } else if (ga != gb) {                                    // q g -> q g, straight and crossed
            emit(ia, ib, ia, ib, 5, 0); emit(ia, ib, ib, ia, 5, 1);
        } else if (ia == ib) {                                    // q1 q1 -> q1 q1 (listed once: t <-> u symmetric)
            emit(ia, ia, ia, ia, 1, 0);
        } else if (ib == anti_of_id(ia)) {                        // q1 q1bar -> q1 q1bar, -> q2 q2bar, -> g g
            emit(ia, ib, ia, ib, 2, 0); emit(ia, ib, ib, ia, 2, 1);
            for (int fl = 0; fl < 3; ++fl) {
                if (fl == (ia - 1) / 2 || !pair_active(fl)) continue;
                emit(ia, ib, 1 + 2 * fl, 2 + 2 * fl, 3, 0); emit(ia, ib, 2 + 2 * fl, 1 + 2 * fl, 3, 0);
            }
            if (slot[0] >= 0) emit(ia, ib, 0, 0, 4, 0);
        } else {                                                  // different flavours (or q1 q2bar): straight and crossed
            emit(ia, ib, ia, ib, 0, 0); emit(ia, ib, ib, ia, 0, 1);
        }
    }
    table.clear(); groups.clear();
    std::vector<char> used(all.size(), 0);
    for (size_t q0 = 0; q0 < all.size(); ++q0) {                  // groups in the order of first appearance
        if (used[q0]) continue;
        PaperGroup g;
        g.key = all[q0].key; g.begin = (int)table.size();
        for (size_t q = q0; q < all.size(); ++q) if (!used[q] && all[q].key == g.key) { table.push_back(all[q]); used[q] = 1; }
        g.end = (int)table.size();
        groups.push_back(g);
    }
}

// ------------------------------------------------------------------------------------------------------ device
namespace {

struct Root {
    int i1, i2;
    double w_inv;          // |J| E1 E2 E3 Ep
    double s, t, u;
};

// Eq. 17-19 for one mass tuple: see oracle/bzo.c paper_roots for the algebra (two squarings of E1 + E2 = Et give
// a z^2 - C Pz z + (Et^2 A1 - C^2/4) = 0).  Single rounded operations, the oracle's association order.
// energies of the two outgoing legs for the four mass classes: E3[c] = sqrt(k3^2 + m_c^2), Ep[c] = sqrt(p^2 + m_c^2), with
// the association of paper_roots; the roots of a tuple take E3 of its third and Ep of its fourth class
struct PaperLegs {
    double E3[4], Ep[4];
    __device__ __forceinline__ PaperLegs(const double (&p)[3], const double (&k3)[3], const double* m)
    {
        const double k2 = __dadd_rn(__dadd_rn(__dmul_rn(k3[0], k3[0]), __dmul_rn(k3[1], k3[1])), __dmul_rn(k3[2], k3[2]));
        const double p2 = __dadd_rn(__dadd_rn(__dmul_rn(p[0], p[0]), __dmul_rn(p[1], p[1])), __dmul_rn(p[2], p[2]));
#pragma unroll
        for (int c = 0; c < 4; ++c) { E3[c] = __dsqrt_rn(__dadd_rn(k2, m[c])); Ep[c] = __dsqrt_rn(__dadd_rn(p2, m[c])); }
    }
    __device__ __forceinline__ double e3(int c) const { return c == 0 ? E3[0] : (c == 1 ? E3[1] : (c == 2 ? E3[2] : E3[3])); }
    __device__ __forceinline__ double ep(int c) const { return c == 0 ? Ep[0] : (c == 1 ? Ep[1] : (c == 2 ? Ep[2] : Ep[3])); }
};

// The root solving in two stages, so that the kernel can compact the few candidates that pass the cheap first stage
// before it runs the expensive second one (paper_queue_kernel).  Both use single rounded operations in the oracle's
// association order; stage 2 recomputes the tuple's constants from the same inputs with the same operations, so the two
// stages together give the bits of the one-piece form.
#define MUL __dmul_rn
#define ADD __dadd_rn
#define SUB __dsub_rn
// Stage 1: the quadratic for z = k1z, the sign test of the squarings and the box test of the z components of k1 and k2
// (S9).  Returns a bit mask: bit 0 = the + root is a candidate, bit 1 = the - root; z and the z cell indices b1, b2 per sign.
__device__ __forceinline__ int paper_roots_stage1(const GridConst& g, const double (&p)[3], const double (&k3)[3], double k1x, double k1y,
                                                  double m1, double m2, double E3, double Ep, double (&zr)[2], int (&b1r)[2], int (&b2r)[2])
{
    const double Et = ADD(E3, Ep);
    const double Px = ADD(k3[0], p[0]), Py = ADD(k3[1], p[1]), Pz = ADD(k3[2], p[2]);
    const double A1 = ADD(ADD(MUL(k1x, k1x), MUL(k1y, k1y)), m1);
    const double qx = SUB(Px, k1x), qy = SUB(Py, k1y);
    const double A2 = ADD(ADD(MUL(qx, qx), MUL(qy, qy)), m2);
    const double Et2 = MUL(Et, Et), Pz2 = MUL(Pz, Pz);
    const double C = SUB(SUB(ADD(Et2, A1), A2), Pz2);
    const double a = SUB(Et2, Pz2);
    if (!(a > 0.0)) return 0;
    const double D = SUB(MUL(C, C), MUL(MUL(4.0, a), A1));
    if (!(D > 0.0)) return 0;
    const double sq = MUL(Et, __dsqrt_rn(D)), CP = MUL(C, Pz), a2 = MUL(2.0, a);
    int cand = 0;
#pragma unroll
    for (int sign = 0; sign < 2; ++sign) {
        const double z = __ddiv_rn(sign == 0 ? ADD(CP, sq) : SUB(CP, sq), a2);
        if (!(ADD(C, MUL(MUL(2.0, Pz), z)) >= 0.0)) continue;
        // the box test of the two z components (S9): most roots end here.  Guarded fast binning (bin_axis_fast: 1 DFMA +
        // conversion), the definition's subtraction and division only inside the guard band around a cell edge
        const double k2z = SUB(Pz, z);
        bool in1, in2, risky = false;
        int b1 = bin_axis_fast(z, g, in1, risky), b2 = bin_axis_fast(k2z, g, in2, risky);
        if (risky) { b1 = bin_axis_exact(z, g, in1); b2 = bin_axis_exact(k2z, g, in2); }
        if (!(in1 && in2)) continue;
        cand |= 1 << sign;
        zr[sign] = z; b1r[sign] = b1; b2r[sign] = b2;
    }
    return cand;
}

// Stage 2 for one candidate z: the energies of the incoming legs, the spurious-root test E1 <= Et, the Jacobian of Eq. 19
// and (s, t, u) of the constructed momenta.  False: the root is dropped.
__device__ __forceinline__ bool paper_roots_stage2(const double (&p)[3], const double (&k3)[3], double k1x, double k1y, double m1, double m2,
                                                   double m3, double m4, double E3, double Ep, double z, Root& r)
{
    const double Et = ADD(E3, Ep);
    const double Px = ADD(k3[0], p[0]), Py = ADD(k3[1], p[1]), Pz = ADD(k3[2], p[2]);
    const double A1 = ADD(ADD(MUL(k1x, k1x), MUL(k1y, k1y)), m1);
    const double qx = SUB(Px, k1x), qy = SUB(Py, k1y);
    const double A2 = ADD(ADD(MUL(qx, qx), MUL(qy, qy)), m2);
    const double Et2 = MUL(Et, Et), Pz2 = MUL(Pz, Pz);
    const double k2z = SUB(Pz, z);
    const double E1 = __dsqrt_rn(ADD(A1, MUL(z, z)));
    if (!(E1 <= Et)) return false;
    const double E2 = __dsqrt_rn(ADD(A2, MUL(k2z, k2z)));
    if (!(E1 > 0.0 && E2 > 0.0)) return false;
    const double J = SUB(__ddiv_rn(z, E1), __ddiv_rn(k2z, E2));          // Eq. 19
    if (J == 0.0) return false;
    r.w_inv = fabs(J) * (((E1 * E2) * E3) * Ep);
    r.s = SUB(Et2, ADD(ADD(MUL(Px, Px), MUL(Py, Py)), Pz2));
    r.t = SUB(ADD(m1, m3), MUL(2.0, SUB(MUL(E1, E3), ADD(ADD(MUL(k1x, k3[0]), MUL(k1y, k3[1])), MUL(z, k3[2])))));
    r.u = SUB(ADD(m1, m4), MUL(2.0, SUB(MUL(E1, Ep), ADD(ADD(MUL(k1x, p[0]), MUL(k1y, p[1])), MUL(z, p[2])))));
    return true;
}
#undef MUL
#undef ADD
#undef SUB

// Both stages for one mass tuple (the debug export).  Bit mask: bit 0 = the + root is kept (out[0]), bit 1 = the - root (out[1]).
__device__ __forceinline__ int paper_roots_core(const GridConst& g, const double (&p)[3], const double (&k3)[3], double k1x, double k1y,
                                                double m1, double m2, double m3, double m4, double E3, double Ep, int ixy1, int ixy2,
                                                Root (&out)[2])
{
    double z[2];
    int b1[2], b2[2];
    const int cand = paper_roots_stage1(g, p, k3, k1x, k1y, m1, m2, E3, Ep, z, b1, b2);
    int nr = 0;
#pragma unroll
    for (int sign = 0; sign < 2; ++sign) {
        if (!((cand >> sign) & 1)) continue;
        if (!paper_roots_stage2(p, k3, k1x, k1y, m1, m2, m3, m4, E3, Ep, z[sign], out[sign])) continue;
        out[sign].i1 = ixy1 + g.n * g.n * b1[sign]; out[sign].i2 = ixy2 + g.n * g.n * b2[sign];
        nr |= 1 << sign;
    }
    return nr;
}

__device__ __forceinline__ int paper_roots(const GridConst& g, const double (&p)[3], const double (&k3)[3], double k1x, double k1y,
                                           double m1, double m2, double m3, double m4, int ixy1, int ixy2, Root (&out)[2])
{
    const double E3 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(k3[0], k3[0]), __dmul_rn(k3[1], k3[1])), __dmul_rn(k3[2], k3[2])), m3));
    const double Ep = __dsqrt_rn(__dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(p[0], p[0]), __dmul_rn(p[1], p[1])), __dmul_rn(p[2], p[2])), m4));
    const int kept = paper_roots_core(g, p, k3, k1x, k1y, m1, m2, m3, m4, E3, Ep, ixy1, ixy2, out);
    if (kept == 2) out[0] = out[1];                       // the oracle's order: +, then -
    return kept == 3 ? 2 : (kept ? 1 : 0);
}

__device__ __forceinline__ void red_add(double* dst, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst), "d"(v) : "memory");
}

// test export: the roots of ONE mass tuple (P.dbg_msq) for every sample of cells [p_begin, p_begin + p_count) of x_begin,
// thread per sample, the same draw and root solving as paper_queue_kernel
constexpr int kPaperThreads = 64;

__global__ void __launch_bounds__(kPaperThreads) paper_debug_kernel(const PaperParams P, int* dbg_cells, double* dbg_stu)
{
    const long long total = (long long)P.x_count * P.p_count * P.Ns;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int smp = (int)(q % P.Ns);
        const long long r1 = q / P.Ns;
        const int i = P.p_begin + (int)(r1 % P.p_count), xcell = P.x_begin + (int)(r1 / P.p_count);
        double p[3], Emassless;
        cell_kinematics(P.g, i, p[0], p[1], p[2], Emassless);
        // the five integration variables of Eq. 20: Philox blocks 64, 65, 66 (the CM sampler owns 0..63)
        uint32_t w0[4], w1[4], w2[4];
        const uint32_t xc = (uint32_t)xcell + P.x_rng_offset;
        philox4x32_10(64u, (uint32_t)smp, (uint32_t)i, xc, P.seed, P.step, w0);
        philox4x32_10(65u, (uint32_t)smp, (uint32_t)i, xc, P.seed, P.step, w1);
        philox4x32_10(66u, (uint32_t)smp, (uint32_t)i, xc, P.seed, P.step, w2);
        double k3[3];
        k3[0] = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w0[0], w0[1]), P.g.L));
        k3[1] = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w0[2], w0[3]), P.g.L));
        k3[2] = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w1[0], w1[1]), P.g.L));
        const double k1x = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w1[2], w1[3]), P.g.L));
        const double k1y = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w2[0], w2[1]), P.g.L));
        const int i3 = bin_cell_exact(k3[0], k3[1], k3[2], P.g);
        // transverse cells of k1 (inside by construction) and of k2 = k3 + p - k1: the same for every mass tuple and root;
        // a sample whose k2x or k2y leaves the box deposits nothing whatever the masses are (S9)
        int ixy1, ixy2;
        bool k2_in;
        {
            bool ia, ib, ic, id;
            const int a1 = bin_axis_exact(k1x, P.g, ia), b1 = bin_axis_exact(k1y, P.g, ib);
            const double qx = __dsub_rn(__dadd_rn(k3[0], p[0]), k1x), qy = __dsub_rn(__dadd_rn(k3[1], p[1]), k1y);
            const int a2 = bin_axis_exact(qx, P.g, ic), b2 = bin_axis_exact(qy, P.g, id);
            ixy1 = a1 + P.g.n * b1; ixy2 = a2 + P.g.n * b2;
            k2_in = ia && ib && ic && id;
        }
        {
            Root rt[2];
            const int nr = !k2_in ? 0 : paper_roots(P.g, p, k3, k1x, k1y, P.dbg_msq[0], P.dbg_msq[1], P.dbg_msq[2], P.dbg_msq[3], ixy1, ixy2, rt);
            int* oc = dbg_cells + 6 * q;
            double* os = dbg_stu + 6 * q;
            oc[0] = i3; oc[1] = nr;
            for (int r = 0; r < 2; ++r) {
                oc[2 + 2 * r] = r < nr ? rt[r].i1 : -1; oc[3 + 2 * r] = r < nr ? rt[r].i2 : -1;
                os[3 * r] = r < nr ? rt[r].s : 0.0; os[3 * r + 1] = r < nr ? rt[r].t : 0.0; os[3 * r + 2] = r < nr ? rt[r].u : 0.0;
            }
        }
    }
}

// ---- the kernel bz_collision_paper launches ------------------------------------------------------------------------
// Only 0.14-0.16 roots per mass tuple survive the box test.  History: a thread-per-sample kernel walked the channel loop of
// every tuple with 6 of 32 lanes active; a warp-cooperative version (the owner of a surviving root publishes it, the
// whole warp works its channels off) fixed that for the massless case (one tuple, 127 channels) but with four distinct
// masses a tuple has few channels, so 29 lanes idled and every root cost a shared-memory column reduction: 0.010 of the
// FP64 peak on config 4 (ncu: 16 of 32 lanes active, 23 % occupancy).  Here every phase whose survivors are sparse hands
// them to the next one through a ring in shared memory, so that each phase runs on full warps:
//   samples  32 samples per pass (Philox, k3, k1x, k1y, the cells that depend on neither masses nor roots); the ~45 % whose k3,
//            k2x, k2y are inside the box go to the sample ring.
//   stage 1  whenever 32 live samples wait: lanes = samples, warp-uniform loop over the distinct (canonical) mass tuples of the spatial cell, listed once
//            per spatial cell; E3 and Ep once per mass class (4 + 4 square roots per sample instead of 2 per tuple); the
//            quadratic for k1z and the box test of the z components (guarded fast binning).  Candidates (z, source lane,
//            tuple, z cells) go to the candidate ring.
//   stage 2  whenever 32 candidates wait (and at the end of the pass: they refer to the pass's samples): lanes =
//            candidates, the sample comes from the source lane by shuffles; E1, E2, the Jacobian, (s, t, u).  Kept roots go
//            to the ring of root records: cells of k1, k2, k3, p, (s, t, u), |J| E1 E2 E3 Ep, tuple.
//   deposit  whenever 32 roots wait: lanes = roots for Table I at the root's massive (s, t, u), stored per root in shared
//            memory; then lanes = (root, channel) pairs of the whole batch (prefix sum of the roots' channel counts, the
//            tuples' channel lists built once per spatial cell): 4 loads, the bracket of Eq. 5, 4 reductions per pair.
// ncu on the first queue version showed stall_no_instruction as large as the memory stalls: the kernel was 63-88 KB of
// code.  Stage 2 is therefore expanded at one place only and the deposit is a non-inlined function with scalar arguments
// (kernel parameters are __grid_constant__: no local copy); that alone was worth 15 %.
constexpr int kQWarps = 8, kQRing = 64, kQCand = 128;
struct QWarp {                         // per warp, in dynamic shared memory (13.7 KB)
    unsigned cell[4][kQRing];          // root records: cells of k1, k2, k3, p
    double s[kQRing], t[kQRing], u[kQRing], w_inv[kQRing];
    unsigned char rti[kQRing];         // the record's canonical mass tuple (index into tup / choff)
    // per spatial cell (classes with bit-identical masses are merged: "canonical" tuples)
    unsigned short ckey[64];           // canonical tuple key of every channel group
    unsigned tup[64];                  // the distinct canonical tuples: key | first group << 16
    unsigned short choff[66];          // channels of tuple ti: chlist[choff[ti] .. choff[ti + 1])
    unsigned char chlist[128];         // indices into the channel table
    int ntup;
    double msm[4];                     // the spatial cell's four masses^2
    // candidates of stage 1 waiting for stage 2 (they refer to the samples the warp's lanes hold at the moment):
    double cz[kQCand];                 // z component of k1 (a tuple adds at most 64 candidates to fewer than 32 waiting ones)
    unsigned long long cmeta[kQCand];  // source lane | canonical tuple key << 5 | tuple index << 13 | z cell of k1 << 19 | z cell of k2 << 30
    // samples that can deposit at all (k3 and the transverse components of k1, k2 inside the box: about half), compacted over
    // the sampling passes so that stage 1 runs on full warps: p, k3, k1x, k1y and the cells
    double sv[8][kQRing];
    int si[4][kQRing];                 // transverse cell parts of k1 and k2, cell of k3, cell of p
    // deposit scratch: Table I of the 32 roots of a batch, [2 kind + crossed][root], and the running channel counts
    double mvs[10][32];                // a_t, a_u, m11, m1b_t, m1b_u, ann, qqgg, qg_t, qg_u, gg
    int pre[33];
};

// Every mass is zero (no bz_thermal_masses / bz_set_masses call yet): one tuple, the root serves ALL channels, and their sum is
// the hot path's factorised algebra (bz_channels.cuh) on the four cells -- 4 x S loads and reductions per root instead of 4
// per channel.  (A separate kernel instantiation: inlined into the general kernel it cost that one 40 %.)
__device__ __noinline__ void paper_deposit_massless(const PaperParams& P, QWarp& q, int lane, int head, int nb, int xcell, double mreg)
{
    if (lane >= nb) return;
    const int r = (head + lane) & (kQRing - 1);
    const double* fx = P.f + (size_t)xcell * P.Np * P.SP;                 // cell-major: the S values of a cell are adjacent
    double* dx = P.dN + (size_t)xcell * P.Np * P.SP;
    const double w = P.Kp / q.w_inv[r];
    MsqSet M = msq_set<true, true>(q.s[r], q.t[r], q.u[r], mreg, P.g4 * w);
    if (P.has_ovr) msq_apply_override(M, P.msq_ovr, P.g4 * w);
    const unsigned c1 = q.cell[0][r], c2 = q.cell[1][r], c3 = q.cell[2][r], c4 = q.cell[3][r];
    double fv[4][7], d[4][7];
#pragma unroll
    for (int id = 0; id < 7; ++id) {
        const int a = P.slot[id];
        fv[0][id] = a >= 0 ? fx[(size_t)c1 * P.SP + a] : 0.0; fv[1][id] = a >= 0 ? fx[(size_t)c2 * P.SP + a] : 0.0;
        fv[2][id] = a >= 0 ? fx[(size_t)c3 * P.SP + a] : 0.0; fv[3][id] = a >= 0 ? fx[(size_t)c4 * P.SP + a] : 0.0;
    }
    deposit<-1>(P.mask, fv[0], fv[1], fv[2], fv[3], M, d[0], d[1], d[2], d[3]);
#pragma unroll
    for (int id = 0; id < 7; ++id) {
        const int a = P.slot[id];
        if (a < 0) continue;
        if (d[0][id] != 0.0) red_add(dx + (size_t)c1 * P.SP + a, d[0][id]);
        if (d[1][id] != 0.0) red_add(dx + (size_t)c2 * P.SP + a, d[1][id]);
        if (d[2][id] != 0.0) red_add(dx + (size_t)c3 * P.SP + a, d[2][id]);
        if (d[3][id] != 0.0) red_add(dx + (size_t)c4 * P.SP + a, d[3][id]);
    }
}

// With masses a root serves only the channels of its own mass tuple (7 on average on config 4, up to 90 when classes
// coincide).  Lanes = roots for Table I (stored per root in shared memory), then lanes = (root, channel) pairs of the whole
// batch, flattened through a prefix sum of the roots' channel counts: every pair costs 4 loads, the bracket of Eq. 5 and 4
// reductions, with no lane waiting for another root's longer channel list.
// Not inlined (three call sites; the kernel's code has to fit the instruction cache, ncu: stall_no_instruction) and with
// scalar arguments: a reference to the kernel's parameter struct would make the callee read it back from local memory.
__device__ __noinline__ void paper_deposit_pairs(QWarp& q, int lane, int head, int nb, const double* __restrict__ fx, double* __restrict__ dx,
                                                 const unsigned long long* __restrict__ table, unsigned SP, double Kp, double g4, double mreg,
                                                 const double* ovr /* 7 user-defined |M|^2 / g^4, or NULL */)
{
    const unsigned full = 0xffffffffu;
    const bool on = lane < nb;
    const int r = (head + lane) & (kQRing - 1);
    int cnt = 0;
    if (on) {
        const double w = Kp / q.w_inv[r];
        MsqSet M = msq_set<true, true>(q.s[r], q.t[r], q.u[r], mreg, g4 * w);
        if (ovr) {
            double o7[7];
#pragma unroll
            for (int k = 0; k < 7; ++k) o7[k] = ovr[k];
            msq_apply_override(M, o7, g4 * w);
        }
        const int ti = q.rti[r];
        cnt = (int)q.choff[ti + 1] - (int)q.choff[ti];
        q.mvs[0][lane] = M.a_t; q.mvs[1][lane] = M.a_u; q.mvs[2][lane] = M.m11; q.mvs[3][lane] = M.m1b_t; q.mvs[4][lane] = M.m1b_u;
        q.mvs[5][lane] = M.ann; q.mvs[6][lane] = M.qqgg; q.mvs[7][lane] = M.qg_t; q.mvs[8][lane] = M.qg_u; q.mvs[9][lane] = M.gg;
    }
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(full, incl, o); if (lane >= o) incl += v; }
    q.pre[lane + 1] = incl;
    if (lane == 0) q.pre[0] = 0;
    const int total = __shfl_sync(full, incl, 31);
    __syncwarp();
    for (int base = 0; base < total; base += 32) {
        const int fl = base + lane;
        if (fl < total) {
            int lo = 0;                                   // the root that owns pair fl: the largest lo with pre[lo] <= fl
#pragma unroll
            for (int stp = 16; stp > 0; stp >>= 1) { if (q.pre[lo + stp] <= fl) lo += stp; }
            const int rr = (head + lo) & (kQRing - 1);
            // one 8-byte load of the channel: a | b << 8 | c << 16 | d << 24 | kind << 32 | crossed << 40 | glue << 48 (PaperChannel)
            const unsigned long long ch = __ldg(table + q.chlist[(int)q.choff[q.rti[rr]] + (fl - q.pre[lo])]);
            const unsigned lo32 = (unsigned)ch, hi32 = (unsigned)(ch >> 32);
            // cell-major gather source and deposit scratch (f_aos, dN_aos): the pairs of one root sit in neighbouring lanes and
            // touch the same four 64-byte cells, so their loads and reductions share sectors
            const size_t oa = (size_t)q.cell[0][rr] * SP + (lo32 & 255u), ob = (size_t)q.cell[1][rr] * SP + ((lo32 >> 8) & 255u);
            const size_t oc = (size_t)q.cell[2][rr] * SP + ((lo32 >> 16) & 255u), od = (size_t)q.cell[3][rr] * SP + (lo32 >> 24);
            const double fa = fx[oa], fb = fx[ob], fc = fx[oc], fd = fx[od];
            const unsigned glue = hi32 >> 16;
            // F = 1 + f (gluon), 1 - f (quark): 1 + sign * f with sign = +-1 is the same rounded sum
            const double Fa = fma((glue & 1u) ? 1.0 : -1.0, fa, 1.0), Fb = fma((glue & 2u) ? 1.0 : -1.0, fb, 1.0);
            const double Fc = fma((glue & 4u) ? 1.0 : -1.0, fc, 1.0), Fd = fma((glue & 8u) ? 1.0 : -1.0, fd, 1.0);
            const double fwd = fa * fb * Fc * Fd - Fa * Fb * fc * fd;             // Eq. 5 bracket
            // row of Table I: first row of the kind (A 0, 11 2, 1B 3, ANN 5, QQGG 6, QG 7, GG 9) + 1 if crossed (kinds A, 1B, QG only)
            const double A = q.mvs[((0x9765320u >> (4u * (hi32 & 255u))) & 15u) + ((hi32 >> 8) & 255u)][lo] * fwd;
            if (A != 0.0) {
                red_add(dx + oa, -A); red_add(dx + ob, -A);                        // Eq. 22
                red_add(dx + oc, A);  red_add(dx + od, A);
            }
        }
    }
    __syncwarp();                                        // the scratch is rewritten by the next batch
}

template <bool kAllMassless>
__device__ __forceinline__ void paper_deposit_batch(const PaperParams& P, QWarp& q, int lane, int head, int nb, int xcell, double mreg)
{
    if constexpr (kAllMassless) {
        paper_deposit_massless(P, q, lane, head, nb, xcell, mreg);
    } else {
        static_assert(sizeof(PaperChannel) == 8, "PaperChannel is read as one 8-byte word");
        const size_t tile = (size_t)xcell * P.Np * P.SP;
        paper_deposit_pairs(q, lane, head, nb, P.f + tile, P.dN + tile, reinterpret_cast<const unsigned long long*>(P.table), (unsigned)P.SP,
                            P.Kp, P.g4, mreg, P.has_ovr ? P.msq_ovr : nullptr);
    }
}

template <bool kAllMassless>
__global__ void __launch_bounds__(32 * kQWarps, kAllMassless ? 1 : 2) paper_queue_kernel(const __grid_constant__ PaperParams P)
{
    extern __shared__ __align__(16) unsigned char paper_smem[];
    QWarp& q = reinterpret_cast<QWarp*>(paper_smem)[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const unsigned full = 0xffffffffu, lt = (1u << lane) - 1u;
    const long long per_x = (long long)P.p_count * P.Ns;
    const long long chunks_per_x = (per_x + 31) / 32;
    // Spatial cells go round-robin to up to 8 groups of CTAs, the chunks of a cell are strided over the warps of its group: a
    // warp stays in one spatial cell for a long run of passes (its rings are drained only when it leaves), and the cells in
    // flight (8 x 1.7 MB of f_aos + dN_aos tiles on config 4) stay in L2; 16 and 32 groups measured 4-6 % slower.
    const int G = P.cta_groups;
    const int grp = (int)blockIdx.x % G;
    const long long wg = (long long)(blockIdx.x / G) * kQWarps + (threadIdx.x >> 5);
    const long long Wg = (long long)((gridDim.x - grp + G - 1) / G) * kQWarps;
    int head = 0, count = 0;            // ring of root records
    int chead = 0, ccount = 0;          // ring of stage-1 candidates (empty between solving passes)
    int shead = 0, scount = 0;          // ring of samples that can deposit
    int cur_x = -1;
    double mreg = 0.0;
    int xi = grp;                       // the warp's next chunk: chunk cnk of the xi-th spatial cell of the launch
    long long cnk = wg;
    // Three things a trip of this loop can do, each written once (the kernel's code has to fit the instruction cache):
    // generate 32 samples of the current spatial cell and keep the live ones; solve a warp of live samples; move on to the
    // next spatial cell (the rings never mix spatial cells: they are drained first).
    for (;;) {
        const bool have = xi < P.x_count && wg < chunks_per_x;
        const int xnext = have ? P.x_begin + xi : -2;
        if (have && xnext == cur_x && scount < 32) {
            // ---- generate: the five integration variables of Eq. 20 (Philox blocks 64, 65, 66; the CM sampler owns 0..63) and
            // the cells that depend on neither masses nor roots; a sample whose k3, k2x or k2y leaves the box deposits nothing (S9)
            const long long local = cnk * 32 + lane;
            const bool valid = local < per_x;
            const long long lc = valid ? local : per_x - 1;
            const int smp = (int)(lc % P.Ns), i = P.p_begin + (int)(lc / P.Ns);
            double p[3], Emassless;
            cell_kinematics(P.g, i, p[0], p[1], p[2], Emassless);
            uint32_t w0[4], w1[4], w2[4];
            const uint32_t xc = (uint32_t)cur_x + P.x_rng_offset;
            philox4x32_10(64u, (uint32_t)smp, (uint32_t)i, xc, P.seed, P.step, w0);
            philox4x32_10(65u, (uint32_t)smp, (uint32_t)i, xc, P.seed, P.step, w1);
            philox4x32_10(66u, (uint32_t)smp, (uint32_t)i, xc, P.seed, P.step, w2);
            double k3[3];
            k3[0] = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w0[0], w0[1]), P.g.L));
            k3[1] = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w0[2], w0[3]), P.g.L));
            k3[2] = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w1[0], w1[1]), P.g.L));
            const double k1x = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w1[2], w1[3]), P.g.L));
            const double k1y = __dadd_rn(P.g.pmin, __dmul_rn(uniform52(w2[0], w2[1]), P.g.L));
            const int i3 = bin_cell_exact(k3[0], k3[1], k3[2], P.g);
            bool ia, ib, ic, id;
            const int a1 = bin_axis_exact(k1x, P.g, ia), b1 = bin_axis_exact(k1y, P.g, ib);
            const double qx = __dsub_rn(__dadd_rn(k3[0], p[0]), k1x), qy = __dsub_rn(__dadd_rn(k3[1], p[1]), k1y);
            const int a2 = bin_axis_exact(qx, P.g, ic), b2 = bin_axis_exact(qy, P.g, id);
            const bool live = valid && i3 >= 0 && ia && ib && ic && id;
            const unsigned lm = __ballot_sync(full, live);
            if (live) {
                const int w = (shead + scount + __popc(lm & lt)) & (kQRing - 1);
                q.sv[0][w] = p[0]; q.sv[1][w] = p[1]; q.sv[2][w] = p[2]; q.sv[3][w] = k3[0]; q.sv[4][w] = k3[1]; q.sv[5][w] = k3[2];
                q.sv[6][w] = k1x; q.sv[7][w] = k1y;
                q.si[0][w] = a1 + P.g.n * b1; q.si[1][w] = a2 + P.g.n * b2; q.si[2][w] = i3; q.si[3][w] = i;
            }
            scount += __popc(lm);
            cnk += Wg;
            if (cnk >= chunks_per_x) { cnk = wg; xi += G; }
            __syncwarp();
            continue;
        }
        if (scount > 0) {
            // ---- solve: lanes = live samples (a full warp unless the spatial cell or the launch ends)
            const int ns = min(scount, 32);
            const bool live = lane < ns;
            const int sr = (shead + (live ? lane : 0)) & (kQRing - 1);
            double p[3], k3[3];
            p[0] = q.sv[0][sr]; p[1] = q.sv[1][sr]; p[2] = q.sv[2][sr]; k3[0] = q.sv[3][sr]; k3[1] = q.sv[4][sr]; k3[2] = q.sv[5][sr];
            const double k1x = q.sv[6][sr], k1y = q.sv[7][sr];
            const int ixy1 = q.si[0][sr], ixy2 = q.si[1][sr], i3 = q.si[2][sr], i = q.si[3][sr];
            shead = (shead + ns) & (kQRing - 1);
            scount -= ns;
            // energies of the outgoing legs, once per mass class (the roots of a tuple take E3 of its third, Ep of its fourth class)
            const PaperLegs L(p, k3, q.msm);
            // stage 2 for candidates [chead, chead + nb): lanes = candidates; the sample a candidate belongs to lives in the registers
            // of its source lane and comes over by shuffles; E3 and Ep are recomputed with PaperLegs' operations (the same bits)
            auto stage2_batch = [&](int nb) {
                const bool on = lane < nb;
                const int cr = (chead + lane) & (kQCand - 1);
                const unsigned long long meta = on ? q.cmeta[cr] : (unsigned long long)lane;
                const double z = on ? q.cz[cr] : 0.0;
                const int src = (int)(meta & 31ull), ck = (int)((meta >> 5) & 255ull), cti = (int)((meta >> 13) & 63ull);
                const int b1 = (int)((meta >> 19) & 2047ull), b2 = (int)((meta >> 30) & 2047ull);
                double sp[3], sk3[3];
#pragma unroll
                for (int d = 0; d < 3; ++d) { sp[d] = __shfl_sync(full, p[d], src); sk3[d] = __shfl_sync(full, k3[d], src); }
                const double sk1x = __shfl_sync(full, k1x, src), sk1y = __shfl_sync(full, k1y, src);
                const int sxy1 = __shfl_sync(full, ixy1, src), sxy2 = __shfl_sync(full, ixy2, src);
                const int si3 = __shfl_sync(full, i3, src), si = __shfl_sync(full, i, src);
                bool kept = false;
                Root rt;
                if (on) {
                    const double m1 = q.msm[ck & 3], m2 = q.msm[(ck >> 2) & 3], m3 = q.msm[(ck >> 4) & 3], m4 = q.msm[(ck >> 6) & 3];
                    const double kk = __dadd_rn(__dadd_rn(__dmul_rn(sk3[0], sk3[0]), __dmul_rn(sk3[1], sk3[1])), __dmul_rn(sk3[2], sk3[2]));
                    const double pp = __dadd_rn(__dadd_rn(__dmul_rn(sp[0], sp[0]), __dmul_rn(sp[1], sp[1])), __dmul_rn(sp[2], sp[2]));
                    const double E3 = __dsqrt_rn(__dadd_rn(kk, m3)), Ep = __dsqrt_rn(__dadd_rn(pp, m4));
                    kept = paper_roots_stage2(sp, sk3, sk1x, sk1y, m1, m2, m3, m4, E3, Ep, z, rt);
                }
                const unsigned has = __ballot_sync(full, kept);
                if (kept) {
                    const int w = (head + count + __popc(has & lt)) & (kQRing - 1);
                    const int n2 = P.g.n * P.g.n;
                    q.cell[0][w] = (unsigned)(sxy1 + n2 * b1); q.cell[1][w] = (unsigned)(sxy2 + n2 * b2); q.cell[2][w] = (unsigned)si3; q.cell[3][w] = (unsigned)si;
                    q.s[w] = rt.s; q.t[w] = rt.t; q.u[w] = rt.u; q.w_inv[w] = rt.w_inv;
                    q.rti[w] = (unsigned char)cti;
                }
                count += __popc(has);
                chead = (chead + nb) & (kQCand - 1);
                ccount -= nb;
                __syncwarp();
                if (count >= 32) {
                    paper_deposit_batch<kAllMassless>(P, q, lane, head, 32, cur_x, mreg);
                    head = (head + 32) & (kQRing - 1);
                    count -= 32;
                    __syncwarp();
                }
            };
            // one more trip than there are tuples: the last one only drains the candidates (they refer to this pass's samples,
            // none is carried over).  stage2_batch is expanded at this one place.
            const int ntup = q.ntup;
            for (int ti = 0; ti <= ntup; ++ti) {                               // warp-uniform: one spatial cell per warp
                const bool last = ti == ntup;
                if (!last) {
                    // stage 1 for every lane: 0.14-0.16 candidates per lane and tuple pass the box test
                    const int ck = (int)(q.tup[ti] & 0xffffu);
                    double zr[2];
                    int b1r[2], b2r[2];
                    const int cand = live ? paper_roots_stage1(P.g, p, k3, k1x, k1y, q.msm[ck & 3], q.msm[(ck >> 2) & 3], L.e3((ck >> 4) & 3), L.ep((ck >> 6) & 3), zr, b1r, b2r) : 0;
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        const bool mine = (cand >> r) & 1;
                        const unsigned has = __ballot_sync(full, mine);
                        if (mine) {
                            const int w = (chead + ccount + __popc(has & lt)) & (kQCand - 1);
                            q.cz[w] = zr[r];
                            q.cmeta[w] = (unsigned long long)lane | (unsigned long long)ck << 5 | (unsigned long long)ti << 13 |
                                         (unsigned long long)b1r[r] << 19 | (unsigned long long)b2r[r] << 30;
                        }
                        ccount += __popc(has);
                    }
                    __syncwarp();
                }
                while (ccount >= 32 || (last && ccount > 0)) stage2_batch(min(ccount, 32));   // full warps of candidates
            }
            continue;
        }
        // ---- the sample ring is empty: the end, or the next spatial cell
        if (!have || xnext != cur_x) {
            while (count > 0) { const int nb = min(count, 32); paper_deposit_batch<kAllMassless>(P, q, lane, head, nb, cur_x, mreg); head = (head + nb) & (kQRing - 1); count -= nb; }
            __syncwarp();
        }
        if (!have) break;
        {
            cur_x = xnext;
            const double* m = P.mass2 + 4 * (size_t)cur_x;
            mreg = P.mD2 > 0.0 ? P.mD2 : m[0];
            // classes with bit-identical masses share their roots: every class is mapped to the first class with its mass
            unsigned rep = 0u;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                int rc = c;
                for (int c2 = c - 1; c2 >= 0; --c2) if (m[c2] == m[c]) rc = c2;
                rep |= (unsigned)rc << (2 * c);
            }
            auto rp0 = [&](int cls) { return (int)((rep >> (2 * cls)) & 3u); };
            auto canon0 = [&](int key) { return rp0(key & 3) | rp0((key >> 2) & 3) << 2 | rp0((key >> 4) & 3) << 4 | rp0((key >> 6) & 3) << 6; };
            // canonical key of every channel group; the distinct ones in the order of their first group; their channel lists
            for (int g0 = lane; g0 < P.n_groups; g0 += 32) q.ckey[g0] = (unsigned short)canon0(P.groups[g0].key);
            __syncwarp();
            int nt = 0;
            for (int g0 = lane; g0 < ((P.n_groups + 31) & ~31); g0 += 32) {
                bool first = g0 < P.n_groups;
                for (int g1 = 0; g1 < g0 && first; ++g1) first = q.ckey[g1] != q.ckey[g0];
                const unsigned fm = __ballot_sync(full, first);
                if (first) q.tup[nt + __popc(fm & lt)] = (unsigned)q.ckey[g0] | (unsigned)g0 << 16;
                nt += __popc(fm);
            }
            __syncwarp();
            int run = 0;                                     // channels of the tuples before this trip's
            for (int t0 = lane; t0 < ((nt + 31) & ~31); t0 += 32) {
                int cnt = 0;
                const unsigned key = t0 < nt ? (q.tup[t0] & 0xffffu) : 0xffffffffu;
                for (int g1 = 0; g1 < P.n_groups; ++g1) if (q.ckey[g1] == key) cnt += P.groups[g1].end - P.groups[g1].begin;
                int incl = cnt;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(full, incl, o); if (lane >= o) incl += v; }
                int w = run + incl - cnt;
                if (t0 < nt) {
                    q.choff[t0] = (unsigned short)w;
                    for (int g1 = 0; g1 < P.n_groups; ++g1)
                        if (q.ckey[g1] == key) for (int c = P.groups[g1].begin; c < P.groups[g1].end; ++c) q.chlist[w++] = (unsigned char)c;
                }
                run += __shfl_sync(full, incl, 31);
            }
            if (lane == 0) { q.choff[nt] = (unsigned short)run; q.ntup = nt; }
            if (lane < 4) q.msm[lane] = m[lane];
            __syncwarp();
        }
    }
}

__global__ void __launch_bounds__(256) combine_kernel(const double* __restrict__ f, double* __restrict__ out,
                                                      const double* __restrict__ dFc, size_t n_values)
{
    for (size_t q = blockIdx.x * (size_t)blockDim.x + threadIdx.x; q < n_values; q += (size_t)gridDim.x * blockDim.x)
        out[q] = (f[q] + out[q]) + dFc[q];
}

}  // namespace

cudaError_t launch_combine(const double* f, double* out, const double* dFc, size_t n_values, cudaStream_t st)
{
    combine_kernel<<<device_sms() * 8, 256, 0, st>>>(f, out, dFc, n_values);
    ++g_launch_count;
    return cudaGetLastError();
}

constexpr int kPaperGroupsMax = 8;       // groups of CTAs at most (16 and 32 measured slower)
cudaError_t launch_paper_collide(const PaperParams& P, int sms, cudaStream_t st)
{
    const long long total = (long long)P.x_count * P.p_count * P.Ns;
    if (total <= 0) return cudaSuccess;
    if (P.n_groups > 64) return cudaErrorInvalidValue;       // the records carry a 64-bit mask of channel groups (7 species: 40)
    if (P.n_channels > 128) return cudaErrorInvalidValue;    // the per-tuple channel lists hold byte indices into the table
    const size_t smem = sizeof(QWarp) * kQWarps;
    // the attribute belongs to the (function, device) pair: one flag per device, not per process
    static bool configured[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !configured[dev]) {
        e = cudaFuncSetAttribute(paper_queue_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(paper_queue_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) configured[dev] = true;
    }
    int per_sm = 1;                      // only the CTAs resident at once: the warps in flight stay within a few spatial cells
    if (P.all_massless) cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, paper_queue_kernel<true>, 32 * kQWarps, smem);
    else cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, paper_queue_kernel<false>, 32 * kQWarps, smem);
    if (per_sm < 1) per_sm = 1;
    long long blocks = (total / 32 + kQWarps) / kQWarps;
    if (blocks > (long long)sms * per_sm) blocks = (long long)sms * per_sm;
    // groups of CTAs: as many as kPaperGroupsMax, but no idle groups in the last round of cells beyond 1/8 of the work
    PaperParams Q = P;
    int best = 1;
    for (int g = 1; g <= kPaperGroupsMax && g <= P.x_count && g <= (int)blocks; ++g) {
        const int rounds = (P.x_count + g - 1) / g;
        if ((long long)rounds * g * 7 <= (long long)P.x_count * 8) best = g;
    }
    Q.cta_groups = best;
    if (P.all_massless) paper_queue_kernel<true><<<(int)blocks, 32 * kQWarps, smem, st>>>(Q);
    else paper_queue_kernel<false><<<(int)blocks, 32 * kQWarps, smem, st>>>(Q);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_paper_debug(const PaperParams& P, int* cells, double* stu, int sms, cudaStream_t st)
{
    const long long total = (long long)P.x_count * P.p_count * P.Ns;
    if (total <= 0) return cudaSuccess;
    long long blocks = (total + kPaperThreads - 1) / kPaperThreads;
    if (blocks > (long long)sms * 32) blocks = (long long)sms * 32;
    paper_debug_kernel<<<(int)blocks, kPaperThreads, 0, st>>>(P, cells, stu);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
