// bz_paper.cu -- NEXT rank 1 of SURVEY.md 8f: the paper's own collision path.
//   Grid point p (cell centre) = the OUTGOING particle d of Eq. 5; integration variables (k1x, k1y, k3x, k3y,
//   k3z) uniform in the momentum box (Eq. 20); k1z from the two roots of E1 + E2 = E3 + Ep with weight 1/|J|
//   (Eq. 17-19); k2 = k3 + p - k1; massive dispersion E^a = sqrt(p^2 + m_a^2(x)) from the thermal masses of
//   Eq. 8-9; symmetrical sampling (Eq. 22): the same weight goes to the cells of k1, k2 (-) and k3, p (+).
// With masses the kinematics depend on the species of the four legs, so a sample is NOT shared by all channels as in
// the hot path: the ordered channels (S8c step 5) are grouped by their tuple of mass classes (g, u, d, s) and every
// group solves its own roots.  One lane per (spatial cell, grid point, sample) for the root solving; the surviving roots
// are worked off by the whole warp (paper_coop_kernel), their deposits summed per (slot, species) in shared memory and
// issued as fp64 reductions (RED.E.ADD.F64) into dF, which a second kernel divides by N_a.  The thread-per-sample
// kernel (paper_kernel) is kept for the debug export of the roots.  Everything that decides a cell index uses single correctly rounded operations in the
// association order of the oracle (bit-exact sampled cells).
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
__device__ __forceinline__ int paper_roots(const GridConst& g, const double (&p)[3], const double (&k3)[3], double k1x, double k1y,
                                           double m1, double m2, double m3, double m4, int ixy1, int ixy2, Root (&out)[2])
{
#define MUL __dmul_rn
#define ADD __dadd_rn
#define SUB __dsub_rn
    const double E3 = __dsqrt_rn(ADD(ADD(ADD(MUL(k3[0], k3[0]), MUL(k3[1], k3[1])), MUL(k3[2], k3[2])), m3));
    const double Ep = __dsqrt_rn(ADD(ADD(ADD(MUL(p[0], p[0]), MUL(p[1], p[1])), MUL(p[2], p[2])), m4));
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
    int nr = 0;
#pragma unroll
    for (int sign = 0; sign < 2; ++sign) {
        const double z = __ddiv_rn(sign == 0 ? ADD(CP, sq) : SUB(CP, sq), a2);
        if (!(ADD(C, MUL(MUL(2.0, Pz), z)) >= 0.0)) continue;
        // the box test of the two z components first (S9): most roots end here, before two square roots and two
        // divisions; the transverse components of k1 and k2 do not depend on the root and were binned by the caller
        const double k2z = SUB(Pz, z);
        bool in1, in2;
        const int b1 = bin_axis_exact(z, g, in1), b2 = bin_axis_exact(k2z, g, in2);
        if (!(in1 && in2)) continue;
        const int i1 = ixy1 + g.n * g.n * b1, i2 = ixy2 + g.n * g.n * b2;
        const double E1 = __dsqrt_rn(ADD(A1, MUL(z, z)));
        if (!(E1 <= Et)) continue;
        const double E2 = __dsqrt_rn(ADD(A2, MUL(k2z, k2z)));
        if (!(E1 > 0.0 && E2 > 0.0)) continue;
        const double J = SUB(__ddiv_rn(z, E1), __ddiv_rn(k2z, E2));          // Eq. 19
        if (J == 0.0) continue;
        Root& r = out[nr++];
        r.i1 = i1; r.i2 = i2;
        r.w_inv = fabs(J) * (((E1 * E2) * E3) * Ep);
        r.s = SUB(Et2, ADD(ADD(MUL(Px, Px), MUL(Py, Py)), Pz2));
        r.t = SUB(ADD(m1, m3), MUL(2.0, SUB(MUL(E1, E3), ADD(ADD(MUL(k1x, k3[0]), MUL(k1y, k3[1])), MUL(z, k3[2])))));
        r.u = SUB(ADD(m1, m4), MUL(2.0, SUB(MUL(E1, Ep), ADD(ADD(MUL(k1x, p[0]), MUL(k1y, p[1])), MUL(z, p[2])))));
    }
#undef MUL
#undef ADD
#undef SUB
    return nr;
}

__device__ __forceinline__ void red_add(double* dst, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst), "d"(v) : "memory");
}

// mode 0: collision; mode 1: debug (writes the roots of one mass tuple instead of depositing)
constexpr int kPaperThreads = 64;

template <int kDebug>
__global__ void __launch_bounds__(kPaperThreads) paper_kernel(const PaperParams P, int* dbg_cells, double* dbg_stu)
{
    __shared__ double sh_fv[28 * kPaperThreads], sh_acc[28 * kPaperThreads];
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
        const double* m = P.mass2 + 4 * (size_t)xcell;
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
        if (kDebug) {
            Root rt[2];
            const int nr = !k2_in ? 0 : paper_roots(P.g, p, k3, k1x, k1y, P.dbg_msq[0], P.dbg_msq[1], P.dbg_msq[2], P.dbg_msq[3], ixy1, ixy2, rt);
            int* oc = dbg_cells + 6 * q;
            double* os = dbg_stu + 6 * q;
            oc[0] = i3; oc[1] = nr;
            for (int r = 0; r < 2; ++r) {
                oc[2 + 2 * r] = r < nr ? rt[r].i1 : -1; oc[3 + 2 * r] = r < nr ? rt[r].i2 : -1;
                os[3 * r] = r < nr ? rt[r].s : 0.0; os[3 * r + 1] = r < nr ? rt[r].t : 0.0; os[3 * r + 2] = r < nr ? rt[r].u : 0.0;
            }
            continue;
        }
        if (i3 < 0 || !k2_in) continue;
        const double mreg = P.mD2 > 0.0 ? P.mD2 : m[0];
        const double* fx = P.f + (size_t)xcell * P.S * P.Np;
        double* dx = P.dN + (size_t)xcell * P.S * P.Np;
        // Mass classes with bit-identical masses (e.g. m_u = m_d = m_s for flavour-symmetric f, or all 0) have the same
        // roots: every class is mapped to the first class with its mass, and all groups with the same mapped tuple share
        // one root solve, one gather of the 4 x S occupation numbers and one flush of the deposits.
        int rep[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            rep[c] = c;
            for (int c2 = c - 1; c2 >= 0; --c2) if (m[c2] == m[c]) rep[c] = c2;
        }
        auto canon = [&](int key) { return rep[key & 3] | rep[(key >> 2) & 3] << 2 | rep[(key >> 4) & 3] << 4 | rep[(key >> 6) & 3] << 6; };
        // The 4 x S occupation numbers and the 4 x S deposit sums of the root being worked on live in shared memory,
        // [entry][thread]: they are indexed by the channel table (run-time indices), which in registers would mean local
        // memory; lanes of a warp read the same entry of consecutive threads, i.e. conflict-free.
        double* fv = sh_fv + threadIdx.x;
        double* acc = sh_acc + threadIdx.x;
        unsigned done[8] = { 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u };
        for (int gi = 0; gi < P.n_groups; ++gi) {
            const int ck = canon(P.groups[gi].key);
            if ((done[ck >> 5] >> (ck & 31)) & 1u) continue;
            done[ck >> 5] |= 1u << (ck & 31);
            Root rt[2];
            const int nr = paper_roots(P.g, p, k3, k1x, k1y, m[ck & 3], m[(ck >> 2) & 3], m[(ck >> 4) & 3], m[(ck >> 6) & 3], ixy1, ixy2, rt);
            for (int r = 0; r < nr; ++r) {
                const Root& R = rt[r];
                const double w = P.Kp / R.w_inv;
                MsqSet M = msq_set<true, true>(R.s, R.t, R.u, mreg, P.g4 * w);
                if (P.has_ovr) msq_apply_override(M, P.msq_ovr, P.g4 * w);
                const double mv[10] = { M.a_t, M.a_u, M.m11, M.m11, M.m1b_t, M.m1b_u, M.ann, M.ann, M.qqgg, M.qqgg };
                const int cell[4] = { R.i1, R.i2, i3, i };
#pragma unroll
                for (int sl = 0; sl < 4; ++sl)
                    for (int a = 0; a < P.S; ++a) {
                        fv[(sl * 7 + a) * kPaperThreads] = fx[(size_t)a * P.Np + cell[sl]];
                        acc[(sl * 7 + a) * kPaperThreads] = 0.0;
                    }
                for (int gj = gi; gj < P.n_groups; ++gj) {
                    const PaperGroup G = P.groups[gj];
                    if (canon(G.key) != ck) continue;
                    for (int c = G.begin; c < G.end; ++c) {
                        const PaperChannel ch = P.table[c];
                        const double fa = fv[ch.a * kPaperThreads], fb = fv[(7 + ch.b) * kPaperThreads];
                        const double fc = fv[(14 + ch.c) * kPaperThreads], fd = fv[(21 + ch.d) * kPaperThreads];
                        const double Fa = (ch.glue & 1) ? 1.0 + fa : 1.0 - fa, Fb = (ch.glue & 2) ? 1.0 + fb : 1.0 - fb;
                        const double Fc = (ch.glue & 4) ? 1.0 + fc : 1.0 - fc, Fd = (ch.glue & 8) ? 1.0 + fd : 1.0 - fd;
                        const double fwd = fa * fb * Fc * Fd - Fa * Fb * fc * fd;             // Eq. 5 bracket
                        const double Mv = ch.kind == 5 ? (ch.crossed ? M.qg_u : M.qg_t) : ch.kind == 6 ? M.gg : mv[2 * ch.kind + ch.crossed];
                        const double A = Mv * fwd;
                        acc[ch.a * kPaperThreads] -= A; acc[(7 + ch.b) * kPaperThreads] -= A;            // Eq. 22
                        acc[(14 + ch.c) * kPaperThreads] += A; acc[(21 + ch.d) * kPaperThreads] += A;
                    }
                }
#pragma unroll
                for (int sl = 0; sl < 4; ++sl)
                    for (int a = 0; a < P.S; ++a) {
                        const double v = acc[(sl * 7 + a) * kPaperThreads];
                        if (v != 0.0) red_add(dx + (size_t)a * P.Np + cell[sl], v);
                    }
            }
        }
    }
}

// ---- warp-cooperative version (the one bz_collision_paper launches) ------------------------------------------------
// Only 0.14-0.16 roots per mass tuple survive the box test, so in the thread-per-sample kernel above a warp walks the
// channel loop of every tuple with 6 of 32 lanes active (ncu).  Here the lanes of a warp still own one sample each for
// the root solving, but every surviving root is then worked off by the WHOLE warp: the owner publishes the root's
// |M|^2 values and cells in shared memory, lanes 0..27 gather the 4 x S occupation numbers, the 32 lanes take the
// channels of the tuple 32 at a time, each adding its deposits to a private column of a [28][33] shared array, and
// lanes 0..27 sum the rows and issue one RED per non-zero (slot, species).  A warp never spans two spatial cells, so
// the loop over mass tuples is warp-uniform.
constexpr int kCoopWarps = 4;
struct CoopShared {
    double M[14];              // |M|^2 x weight by 2 * kind + crossed
    int cells[4];
    double fv[28];             // f_a at the four cells, [slot * 7 + a]
    double acc[28][33];        // deposits, one column per lane
};

__global__ void __launch_bounds__(32 * kCoopWarps) paper_coop_kernel(const PaperParams P)
{
    __shared__ CoopShared sh_all[kCoopWarps];
    CoopShared& sh = sh_all[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const unsigned full = 0xffffffffu;
    const long long per_x = (long long)P.p_count * P.Ns;
    const long long chunks_per_x = (per_x + 31) / 32;
    const long long n_items = chunks_per_x * P.x_count;
    const long long warp0 = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5, n_warps = ((long long)gridDim.x * blockDim.x) >> 5;
#pragma unroll
    for (int k = 0; k < 28; ++k) sh.acc[k][lane] = 0.0;       // kept all-zero between roots: a reducer re-zeroes its row
    __syncwarp();
    for (long long item = warp0; item < n_items; item += n_warps) {
        const int xcell = P.x_begin + (int)(item / chunks_per_x);
        const long long local = (item % chunks_per_x) * 32 + lane;
        const bool valid = local < per_x;
        const long long lc = valid ? local : per_x - 1;
        const int smp = (int)(lc % P.Ns), i = P.p_begin + (int)(lc / P.Ns);
        double p[3], Emassless;
        cell_kinematics(P.g, i, p[0], p[1], p[2], Emassless);
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
        int ixy1, ixy2;
        bool live;
        {
            bool ia, ib, ic, id;
            const int a1 = bin_axis_exact(k1x, P.g, ia), b1 = bin_axis_exact(k1y, P.g, ib);
            const double qx = __dsub_rn(__dadd_rn(k3[0], p[0]), k1x), qy = __dsub_rn(__dadd_rn(k3[1], p[1]), k1y);
            const int a2 = bin_axis_exact(qx, P.g, ic), b2 = bin_axis_exact(qy, P.g, id);
            ixy1 = a1 + P.g.n * b1; ixy2 = a2 + P.g.n * b2;
            live = valid && i3 >= 0 && ia && ib && ic && id;
        }
        const double* m = P.mass2 + 4 * (size_t)xcell;
        const double mreg = P.mD2 > 0.0 ? P.mD2 : m[0];
        const double* fx = P.f + (size_t)xcell * P.S * P.Np;
        double* dx = P.dN + (size_t)xcell * P.S * P.Np;
        unsigned rep = 0u;                                 // 2 bits per class: the first class with the same mass
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            int rc = c;
            for (int c2 = c - 1; c2 >= 0; --c2) if (m[c2] == m[c]) rc = c2;
            rep |= (unsigned)rc << (2 * c);
        }
        auto rp = [&](int cls) { return (int)((rep >> (2 * cls)) & 3u); };
        auto canon = [&](int key) { return rp(key & 3) | rp((key >> 2) & 3) << 2 | rp((key >> 4) & 3) << 4 | rp((key >> 6) & 3) << 6; };
        unsigned done[8] = { 0u, 0u, 0u, 0u, 0u, 0u, 0u, 0u };
        for (int gi = 0; gi < P.n_groups; ++gi) {                          // warp-uniform: one spatial cell per warp
            const int ck = canon(P.groups[gi].key);
            if ((done[ck >> 5] >> (ck & 31)) & 1u) continue;
            done[ck >> 5] |= 1u << (ck & 31);
            // this lane's channels of the tuple (c = lane + 32 k), found once per tuple, not once per root
            unsigned mine = 0u;
            for (int k = 0; lane + 32 * k < P.n_channels && k < 8; ++k)
                if (canon(P.table[lane + 32 * k].key) == ck) mine |= 1u << k;
            Root rt[2];
            const int nr = live ? paper_roots(P.g, p, k3, k1x, k1y, m[ck & 3], m[(ck >> 2) & 3], m[(ck >> 4) & 3], m[(ck >> 6) & 3], ixy1, ixy2, rt) : 0;
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                unsigned owners = __ballot_sync(full, r < nr);
                if (!owners) continue;
                MsqSet M = {};
                if (r < nr) {                                              // the owners, in parallel
                    const double w = P.Kp / rt[r].w_inv;
                    M = msq_set<true, true>(rt[r].s, rt[r].t, rt[r].u, mreg, P.g4 * w);
                    if (P.has_ovr) msq_apply_override(M, P.msq_ovr, P.g4 * w);
                }
                while (owners) {
                    const int L = __ffs(owners) - 1;
                    owners &= owners - 1;
                    if (lane == L) {
                        sh.M[0] = M.a_t; sh.M[1] = M.a_u; sh.M[2] = M.m11; sh.M[3] = M.m11; sh.M[4] = M.m1b_t; sh.M[5] = M.m1b_u;
                        sh.M[6] = M.ann; sh.M[7] = M.ann; sh.M[8] = M.qqgg; sh.M[9] = M.qqgg; sh.M[10] = M.qg_t; sh.M[11] = M.qg_u;
                        sh.M[12] = M.gg; sh.M[13] = M.gg;
                        sh.cells[0] = rt[r].i1; sh.cells[1] = rt[r].i2; sh.cells[2] = i3; sh.cells[3] = i;
                    }
                    __syncwarp();
                    if (lane < 28) {
                        const int a = lane % 7;
                        sh.fv[lane] = a < P.S ? fx[(size_t)a * P.Np + sh.cells[lane / 7]] : 0.0;
                    }
                    __syncwarp();
                    unsigned rows = 0u;                        // rows of sh.acc this lane touches
                    for (unsigned left = mine; left; left &= left - 1u) {
                        const PaperChannel ch = P.table[lane + 32 * (__ffs(left) - 1)];
                        rows |= 1u << ch.a | 1u << (7 + ch.b) | 1u << (14 + ch.c) | 1u << (21 + ch.d);
                        const double fa = sh.fv[ch.a], fb = sh.fv[7 + ch.b], fc = sh.fv[14 + ch.c], fd = sh.fv[21 + ch.d];
                        const double Fa = (ch.glue & 1) ? 1.0 + fa : 1.0 - fa, Fb = (ch.glue & 2) ? 1.0 + fb : 1.0 - fb;
                        const double Fc = (ch.glue & 4) ? 1.0 + fc : 1.0 - fc, Fd = (ch.glue & 8) ? 1.0 + fd : 1.0 - fd;
                        const double fwd = fa * fb * Fc * Fd - Fa * Fb * fc * fd;             // Eq. 5 bracket
                        const double A = sh.M[2 * ch.kind + ch.crossed] * fwd;
                        sh.acc[ch.a][lane] -= A; sh.acc[7 + ch.b][lane] -= A;                 // Eq. 22
                        sh.acc[14 + ch.c][lane] += A; sh.acc[21 + ch.d][lane] += A;
                    }
                    rows = __reduce_or_sync(full, rows);
                    __syncwarp();
                    if ((rows >> lane) & 1u) {                 // lane < 28: sum the row, re-zero it, one reduction
                        double v = 0.0;
#pragma unroll
                        for (int j = 0; j < 32; ++j) { v += sh.acc[lane][j]; sh.acc[lane][j] = 0.0; }
                        if (v != 0.0) red_add(dx + (size_t)(lane % 7) * P.Np + sh.cells[lane / 7], v);
                    }
                    __syncwarp();
                }
            }
        }
    }
}

__global__ void __launch_bounds__(256) paper_finalize_kernel(double* __restrict__ dF, size_t n_values, int S, int Np, const double d0,
                                                              const double d1, const double d2, const double d3, const double d4,
                                                              const double d5, const double d6)
{
    const double deg[7] = { d0, d1, d2, d3, d4, d5, d6 };
    for (size_t q = blockIdx.x * (size_t)blockDim.x + threadIdx.x; q < n_values; q += (size_t)gridDim.x * blockDim.x)
        dF[q] = dF[q] / deg[(q / Np) % S];
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
    combine_kernel<<<148 * 8, 256, 0, st>>>(f, out, dFc, n_values);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_paper_collide(const PaperParams& P, int sms, cudaStream_t st)
{
    const long long total = (long long)P.x_count * P.p_count * P.Ns;
    if (total <= 0) return cudaSuccess;
    int per_sm = 1;                      // only the CTAs resident at once: the warps in flight stay within a few spatial cells
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, paper_coop_kernel, 32 * kCoopWarps, 0);
    if (per_sm < 1) per_sm = 1;
    long long blocks = (total / 32 + kCoopWarps) / kCoopWarps;
    if (blocks > (long long)sms * per_sm) blocks = (long long)sms * per_sm;
    paper_coop_kernel<<<(int)blocks, 32 * kCoopWarps, 0, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_paper_debug(const PaperParams& P, int* cells, double* stu, int sms, cudaStream_t st)
{
    const long long total = (long long)P.x_count * P.p_count * P.Ns;
    if (total <= 0) return cudaSuccess;
    long long blocks = (total + kPaperThreads - 1) / kPaperThreads;
    if (blocks > (long long)sms * 32) blocks = (long long)sms * 32;
    paper_kernel<1><<<(int)blocks, kPaperThreads, 0, st>>>(P, cells, stu);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_paper_finalize(double* dF, size_t n_values, int S, int Np, const double* deg, cudaStream_t st)
{
    paper_finalize_kernel<<<148 * 8, 256, 0, st>>>(dF, n_values, S, Np, deg[0], deg[1], deg[2], deg[3], deg[4], deg[5], deg[6]);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
