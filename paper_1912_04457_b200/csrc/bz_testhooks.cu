// bz_testhooks.cu -- TEST-ONLY object, built into libbz_testhooks.so, never linked into libbz.so and never loaded by the
// product (paper_1912_04457_b200/bz.py).  It compiles the per-sample channel algebra of the kernels (bz_channels.cuh,
// S8c steps 4-6) for the HOST so that tests/test_host_logic.py can check its factorised form against the oracle's
// channel-by-channel definition on a box without a GPU.
#include "bz_channels.cuh"
#include "bz_testhooks.h"

extern "C" int bz_debug_deposit_host(const int* species, int n_species, double alpha_s, const double* fv, double s, double t, double u,
                                     double m2, double w, int variant, double* out)
{
    using namespace bz;
    if (!species || !fv || !out || n_species < 1 || n_species > 7) return -1;
    unsigned mask = 0;
    for (int a = 0; a < n_species; ++a) {
        if (species[a] < 0 || species[a] > 6) return -1;
        mask |= 1u << species[a];
    }
    double f[4][7], d[4][7];
    for (int sl = 0; sl < 4; ++sl)
        for (int id = 0; id < 7; ++id) f[sl][id] = ((mask >> id) & 1u) ? fv[sl * 7 + id] : 0.0;
    const double g2 = 4.0 * 3.14159265358979323846 * alpha_s;
    const MsqSet M = msq_set<true, true>(s, t, u, m2, g2 * g2 * w);
    if (variant == 0) {                                          // the whole bracket in one piece
        deposit<-1>(mask, f[0], f[1], f[2], f[3], M, d[0], d[1], d[2], d[3]);
        for (int sl = 0; sl < 4; ++sl)
            for (int id = 0; id < 7; ++id) out[sl * 7 + id] = d[sl][id];
        return 0;
    }
    // the collision kernel's form: the gain half on the cells (i, j | k, l) and, for the loss half, the gain half of the
    // time-reversed channels on (k, l | i, j), evaluated separately and added (P = f at the incoming cells, Q = 1 +- f at
    // the outgoing ones; inactive species 0 on both sides)
    double h[2][4][7];
    for (int half = 0; half < 2; ++half) {
        double P[2][7], Q[2][7], dd[4][7];
        const int in0 = half == 0 ? 0 : 2, out0 = half == 0 ? 2 : 0;
        for (int id = 0; id < 7; ++id) {
            const bool on = (mask >> id) & 1u;
            for (int c = 0; c < 2; ++c) {
                P[c][id] = on ? f[in0 + c][id] : 0.0;
                Q[c][id] = !on ? 0.0 : (id == 0 ? 1.0 + f[out0 + c][id] : 1.0 - f[out0 + c][id]);     // F = 1 + f (gluon), 1 - f (quark)
            }
        }
        deposit_half<-1>(mask, P[0], P[1], Q[0], Q[1], M, dd[0], dd[1], dd[2], dd[3]);
        for (int c = 0; c < 2; ++c)
            for (int id = 0; id < 7; ++id) { h[half][in0 + c][id] = dd[c][id]; h[half][out0 + c][id] = dd[2 + c][id]; }
    }
    for (int sl = 0; sl < 4; ++sl)
        for (int id = 0; id < 7; ++id) out[sl * 7 + id] = h[0][sl][id] + h[1][sl][id];
    return 0;
}
