// bz_channels.cuh -- |M|^2 of Table I and the per-sample channel algebra (S8c steps 4-6).
//
// The 127 ordered channels of the 7-species mixture (S8c step 5) are not looped over.  Every channel's bracket
// (Eq. 5) factorises into an "incoming" and an "outgoing" pair product, and the channels fall into three
// families that share the cell routing of their species:
//   t-family  a: i->k, b: j->l   (straight elastic, incl. gg->gg and q q->q q)      |M|^2(s,t,u)
//   u-family  a: i->l, b: j->k   (crossed elastic)                                   |M|^2(s,u,t)
//   s-family  (a,abar) or (g,g) at (i,j)  ->  (c,cbar) or (g,g) at (k,l)             annihilation / pair creation
// Within a family the sum over the partner species is a short dot product with at most four distinct |M|^2
// values, so one sample costs O(S) fused multiply-adds instead of 127 x 12.  The result differs from the
// channel-by-channel sum only by fp64 rounding order (bounded by the gross sum of S16).
//
// Arrays are indexed by species id 0..6; entries of inactive species must hold f = 0 and are masked out where
// a vanishing f alone does not switch a channel off (pair creation into an absent flavour).
#pragma once

#if defined(__CUDACC__)
#define BZ_HD __host__ __device__ __forceinline__
#else
#define BZ_HD inline
#endif

namespace bz {

constexpr int kMaxSpecies = 7;

// the <= 10 distinct values one kinematic sample needs, each already multiplied by g^4 * w
struct MsqSet {
    double gg;            // gg -> gg
    double qqgg;          // q qbar <-> g g            (t <-> u symmetric)
    double qg_t, qg_u;    // q g -> q g, straight / crossed
    double m11;           // q1 q1 -> q1 q1             (t <-> u symmetric)
    double m1b_t, m1b_u;  // q1 q1bar -> q1 q1bar, straight / crossed
    double ann;           // q1 q1bar -> q2 q2bar       (t <-> u symmetric)
    double a_t, a_u;      // q1 q2 -> q1 q2 (different flavours), straight / crossed
    // differences to the different-flavour value, formed without cancellation from the terms of Table I:
    double d11;           // m11 - a_t   = M_A(s,u,t) - (32/3) s^2/(tt ut)
    double d1b_t, d1b_u;  // m1b_t - a_t = M_ann - (32/3) u^2/(tt s);  m1b_u - a_u = M_ann - (32/3) t^2/(ut s)
};

// 1/x to ~1 ulp without the IEEE division sequence: the 20-bit hardware seed (MUFU.RCP64H) and two Newton steps.
// Nothing here feeds a sampled index, so correct rounding is not required (S8c step 4: "FMA allowed from here on").
BZ_HD double rcp_fast(double x)
{
#if defined(__CUDA_ARCH__)
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
#else
    return 1.0 / x;
#endif
}

// Table I with the regulated propagators tt = t - m^2, ut = u - m^2; SU(3): 8 dF^2 CF^2/dA = 16,
// 16 dF CF (CF - CA/2) = -32/3, 8 dF CF^2 = 128/3, 8 dF CF CA = 96, 16 dA CA^2 = 1152.
template <bool kGlue, bool kQuark>
BZ_HD MsqSet msq_set(double s, double t, double u, double m2, double g4w)
{
    MsqSet M = {};
    const double it = rcp_fast(t - m2), iu = rcp_fast(u - m2), is = rcp_fast(s);
    const double s2 = s * s, t2 = t * t, u2 = u * u;
    const double it2 = it * it, iu2 = iu * iu, is2 = is * is;
    const double c16 = 16.0 * g4w, c323 = (32.0 / 3.0) * g4w, c1283 = (128.0 / 3.0) * g4w;
    const double at = c16 * (s2 + u2) * it2;       // M_A(s,t,u)
    const double au = c16 * (s2 + t2) * iu2;       // M_A(s,u,t)
    const double ann = c16 * (t2 + u2) * is2;      // M_ann
    if (kQuark) {
        M.a_t = at;
        M.a_u = au;
        M.ann = ann;
        M.d11 = au - c323 * s2 * (it * iu);
        M.d1b_t = ann - c323 * u2 * (it * is);
        M.d1b_u = ann - c323 * t2 * (iu * is);
        M.m11 = at + M.d11;
        M.m1b_t = at + M.d1b_t;
        M.m1b_u = au + M.d1b_u;
    }
    if (kGlue && kQuark) {
        M.qqgg = c1283 * (u * it + t * iu) - 6.0 * ann;
        M.qg_t = 6.0 * at - c1283 * (u * is + s * iu);
        M.qg_u = 6.0 * au - c1283 * (t * is + s * it);
    }
    if (kGlue) M.gg = 1152.0 * g4w * (3.0 - s * u * it2 - s * t * iu2 - t * u * is2);
    return M;
}

// User-defined matrix elements ("an API for users to define their own matrix elements"): a constant per kind
// of Table I, in the order A, 11, 1B, ANN, QQGG, QG, GG.  ovr[kind] >= 0 replaces that kind (straight and crossed)
// by ovr[kind] * g4w (the caller passes value / g^4); the differences the channel algebra uses are re-formed.
BZ_HD void msq_apply_override(MsqSet& M, const double (&ovr)[7], double g4w)
{
    if (ovr[0] >= 0.0) M.a_t = M.a_u = ovr[0] * g4w;
    if (ovr[1] >= 0.0) M.m11 = ovr[1] * g4w;
    if (ovr[2] >= 0.0) M.m1b_t = M.m1b_u = ovr[2] * g4w;
    if (ovr[3] >= 0.0) M.ann = ovr[3] * g4w;
    if (ovr[4] >= 0.0) M.qqgg = ovr[4] * g4w;
    if (ovr[5] >= 0.0) M.qg_t = M.qg_u = ovr[5] * g4w;
    if (ovr[6] >= 0.0) M.gg = ovr[6] * g4w;
    M.d11 = M.m11 - M.a_t;
    M.d1b_t = M.m1b_t - M.a_t;
    M.d1b_u = M.m1b_u - M.a_u;
}

// Deposits of one sample in number units: dI, dJ, dK, dL for the cells of p1, p2, p3, p4 (Eq. 22, P:201:
// every channel adds -A, -A, +A, +A).  kMask >= 0: compile-time species mask; kMask < 0: use rt_mask.
template <int kMask>
BZ_HD void deposit(unsigned rt_mask, const double (&fi)[7], const double (&fj)[7], const double (&fk)[7],
                   const double (&fl)[7], const MsqSet& M, double (&dI)[7], double (&dJ)[7], double (&dK)[7],
                   double (&dL)[7])
{
    const unsigned mask = kMask >= 0 ? (unsigned)kMask : rt_mask;
#define BZ_ON(a) (((mask) >> (a)) & 1u)
    const bool glue = BZ_ON(0);
    // F = 1 + f (gluon), 1 - f (quark, antiquark)
    double Fi[7], Fj[7], Fk[7], Fl[7];
    Fi[0] = 1.0 + fi[0]; Fj[0] = 1.0 + fj[0]; Fk[0] = 1.0 + fk[0]; Fl[0] = 1.0 + fl[0];
#pragma unroll
    for (int a = 1; a < 7; ++a) { Fi[a] = 1.0 - fi[a]; Fj[a] = 1.0 - fj[a]; Fk[a] = 1.0 - fk[a]; Fl[a] = 1.0 - fl[a]; }
#pragma unroll
    for (int a = 0; a < 7; ++a) dI[a] = dJ[a] = dK[a] = dL[a] = 0.0;

    // ------------------------------------------------------------------ t-family: a i->k, b j->l
    {
        double X[7], Y[7], Z[7], W[7], Xf[3], Yf[3], Zf[3], Wf[3];
#pragma unroll
        for (int a = 0; a < 7; ++a) {
            X[a] = fi[a] * Fk[a]; Y[a] = Fi[a] * fk[a];
            Z[a] = fj[a] * Fl[a]; W[a] = Fj[a] * fl[a];
        }
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            Xf[p] = X[1 + 2 * p] + X[2 + 2 * p]; Yf[p] = Y[1 + 2 * p] + Y[2 + 2 * p];
            Zf[p] = Z[1 + 2 * p] + Z[2 + 2 * p]; Wf[p] = W[1 + 2 * p] + W[2 + 2 * p];
        }
        const double Xq = (Xf[0] + Xf[1]) + Xf[2], Yq = (Yf[0] + Yf[1]) + Yf[2];
        const double Zq = (Zf[0] + Zf[1]) + Zf[2], Wq = (Wf[0] + Wf[1]) + Wf[2];
        if (glue) {
            const double T = X[0] * (M.gg * Z[0] + M.qg_t * Zq) - Y[0] * (M.gg * W[0] + M.qg_t * Wq);
            const double U = Z[0] * (M.gg * X[0] + M.qg_t * Xq) - W[0] * (M.gg * Y[0] + M.qg_t * Yq);
            dI[0] -= T; dK[0] += T; dJ[0] -= U; dL[0] += U;
        }
        // partner sum of quark a: qg_t [g] + m11 [a] + m1b_t [abar] + a_t [the other four] = the base over ALL partners
        // at the different-flavour value plus the two differences (see the bound in DESIGN.md 6)
        const double bZ = M.qg_t * Z[0] + M.a_t * Zq, bW = M.qg_t * W[0] + M.a_t * Wq;
        const double bX = M.qg_t * X[0] + M.a_t * Xq, bY = M.qg_t * Y[0] + M.a_t * Yq;
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            if (!BZ_ON(a)) continue;
            const int ab = (a & 1) ? a + 1 : a - 1;
            const double ZM = fma(M.d11, Z[a], fma(M.d1b_t, Z[ab], bZ));
            const double WM = fma(M.d11, W[a], fma(M.d1b_t, W[ab], bW));
            const double XM = fma(M.d11, X[a], fma(M.d1b_t, X[ab], bX));
            const double YM = fma(M.d11, Y[a], fma(M.d1b_t, Y[ab], bY));
            const double T = X[a] * ZM - Y[a] * WM;
            const double U = Z[a] * XM - W[a] * YM;
            dI[a] -= T; dK[a] += T; dJ[a] -= U; dL[a] += U;
        }
    }
    // ------------------------------------------------------------------ u-family: a i->l, b j->k
    {
        double X[7], Y[7], Z[7], W[7], Xf[3], Yf[3], Zf[3], Wf[3];
#pragma unroll
        for (int a = 0; a < 7; ++a) {
            X[a] = fi[a] * Fl[a]; Y[a] = Fi[a] * fl[a];
            Z[a] = fj[a] * Fk[a]; W[a] = Fj[a] * fk[a];
        }
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            Xf[p] = X[1 + 2 * p] + X[2 + 2 * p]; Yf[p] = Y[1 + 2 * p] + Y[2 + 2 * p];
            Zf[p] = Z[1 + 2 * p] + Z[2 + 2 * p]; Wf[p] = W[1 + 2 * p] + W[2 + 2 * p];
        }
        const double Xq = (Xf[0] + Xf[1]) + Xf[2], Yq = (Yf[0] + Yf[1]) + Yf[2];
        const double Zq = (Zf[0] + Zf[1]) + Zf[2], Wq = (Wf[0] + Wf[1]) + Wf[2];
        if (glue) {
            const double T = M.qg_u * (X[0] * Zq - Y[0] * Wq);
            const double U = M.qg_u * (Z[0] * Xq - W[0] * Yq);
            dI[0] -= T; dL[0] += T; dJ[0] -= U; dK[0] += U;
        }
        // partner sum of quark a: qg_u [g] + m1b_u [abar] + a_u [the other four]; the same-species partner belongs to
        // the t-family only (M_11 is t <-> u symmetric and listed once), so it is taken out of the base again
        const double bZ = M.qg_u * Z[0] + M.a_u * Zq, bW = M.qg_u * W[0] + M.a_u * Wq;
        const double bX = M.qg_u * X[0] + M.a_u * Xq, bY = M.qg_u * Y[0] + M.a_u * Yq;
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            if (!BZ_ON(a)) continue;
            const int ab = (a & 1) ? a + 1 : a - 1;
            const double ZM = fma(-M.a_u, Z[a], fma(M.d1b_u, Z[ab], bZ));
            const double WM = fma(-M.a_u, W[a], fma(M.d1b_u, W[ab], bW));
            const double XM = fma(-M.a_u, X[a], fma(M.d1b_u, X[ab], bX));
            const double YM = fma(-M.a_u, Y[a], fma(M.d1b_u, Y[ab], bY));
            const double T = X[a] * ZM - Y[a] * WM;
            const double U = Z[a] * XM - W[a] * YM;
            dI[a] -= T; dL[a] += T; dJ[a] -= U; dK[a] += U;
        }
    }
    // ------------------------------------------------------------------ s-family: pairs at (i,j) -> pairs at (k,l)
    {
        // quark "state a": a at the first cell of the pair, abar at the second; valid only if both are active
        double In[7], Ib[7], Out[7], Ob[7], Inf[3], Ibf[3], Outf[3], Obf[3];
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            const int ab = (a & 1) ? a + 1 : a - 1;
            const bool ok = BZ_ON(a) && BZ_ON(ab);
            In[a] = ok ? fi[a] * fj[ab] : 0.0;  Ib[a] = ok ? Fi[a] * Fj[ab] : 0.0;
            Out[a] = ok ? Fk[a] * Fl[ab] : 0.0; Ob[a] = ok ? fk[a] * fl[ab] : 0.0;
        }
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            Inf[p] = In[1 + 2 * p] + In[2 + 2 * p];    Ibf[p] = Ib[1 + 2 * p] + Ib[2 + 2 * p];
            Outf[p] = Out[1 + 2 * p] + Out[2 + 2 * p]; Obf[p] = Ob[1 + 2 * p] + Ob[2 + 2 * p];
        }
        const double Ing = glue ? fi[0] * fj[0] : 0.0, Ibg = glue ? Fi[0] * Fj[0] : 0.0;
        const double Outg = glue ? Fk[0] * Fl[0] : 0.0, Obg = glue ? fk[0] * fl[0] : 0.0;
        if (glue) {
            const double Sg = M.qqgg * (Ing * ((Outf[0] + Outf[1]) + Outf[2]) - Ibg * ((Obf[0] + Obf[1]) + Obf[2]));
            const double Rg = M.qqgg * (Outg * ((Inf[0] + Inf[1]) + Inf[2]) - Obg * ((Ibf[0] + Ibf[1]) + Ibf[2]));
            dI[0] -= Sg; dJ[0] -= Sg; dK[0] += Rg; dL[0] += Rg;
        }
        // partner sum of the quark pair of flavour p: q qbar <-> g g plus annihilation into the OTHER flavours = the
        // base over all flavours minus its own
        const double Outq = (Outf[0] + Outf[1]) + Outf[2], Obq = (Obf[0] + Obf[1]) + Obf[2];
        const double Inq = (Inf[0] + Inf[1]) + Inf[2], Ibq = (Ibf[0] + Ibf[1]) + Ibf[2];
        const double bOut = M.qqgg * Outg + M.ann * Outq, bOb = M.qqgg * Obg + M.ann * Obq;
        const double bIn = M.qqgg * Ing + M.ann * Inq, bIb = M.qqgg * Ibg + M.ann * Ibq;
        double pOut[3], pOb[3], pIn[3], pIb[3];
#pragma unroll
        for (int p = 0; p < 3; ++p) {
            pOut[p] = fma(-M.ann, Outf[p], bOut); pOb[p] = fma(-M.ann, Obf[p], bOb);
            pIn[p] = fma(-M.ann, Inf[p], bIn);    pIb[p] = fma(-M.ann, Ibf[p], bIb);
        }
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            const int ab = (a & 1) ? a + 1 : a - 1;
            if (!(BZ_ON(a) && BZ_ON(ab))) continue;
            const int p = (a - 1) >> 1;
            const double S = In[a] * pOut[p] - Ib[a] * pOb[p];
            const double R = Out[a] * pIn[p] - Ob[a] * pIb[p];
            dI[a] -= S; dJ[ab] -= S; dK[a] += R; dL[ab] += R;
        }
    }
#undef BZ_ON
}

// ---- the same algebra, one half of the bracket at a time ---------------------------------------------------------------
// Every channel's bracket is  f_a(i) f_b(j) F_c(k) F_d(l)  -  F_a(i) F_b(j) f_c(k) f_d(l)  (Eq. 5).  deposit_half
// evaluates the GAIN product of all channels: P holds the incoming-side factors f at the cells (i, j), Q the outgoing-side
// factors F = 1 +- f at (k, l); its deposits are -H, -H at (i, j) and +H, +H at (k, l) (Eq. 22).  The LOSS product of a
// channel a b -> c d is the gain product of the time-reversed channel c d -> a b on the cells (k, l | i, j) -- same s, t,
// u, same |M|^2, and the channel table is closed under time reversal (S8c step 5) -- so the loss half of all channels is
// deposit_half called with the two pairs of cells exchanged.  The collision kernel gives the two halves of a sample to two
// lanes (half the registers per lane, the same instruction stream for both) and adds the two sets of deposits when it
// flushes them; each half's deposits cancel exactly by themselves, so particle number is conserved as before.  Entries
// of inactive species must be 0 in P and in Q.
template <int kMask>
BZ_HD void deposit_half(unsigned rt_mask, const double (&Pi)[7], const double (&Pj)[7], const double (&Qk)[7],
                        const double (&Ql)[7], const MsqSet& M, double (&dI)[7], double (&dJ)[7], double (&dK)[7],
                        double (&dL)[7])
{
    const unsigned mask = kMask >= 0 ? (unsigned)kMask : rt_mask;
#define BZ_ON(a) (((mask) >> (a)) & 1u)
    const bool glue = BZ_ON(0);
#pragma unroll
    for (int a = 0; a < 7; ++a) dI[a] = dJ[a] = dK[a] = dL[a] = 0.0;
    // ------------------------------------------------------------------ t-family: a i->k, b j->l
    {
        double X[7], Z[7];
#pragma unroll
        for (int a = 0; a < 7; ++a) { X[a] = Pi[a] * Qk[a]; Z[a] = Pj[a] * Ql[a]; }
        const double Xq = ((X[1] + X[2]) + (X[3] + X[4])) + (X[5] + X[6]);
        const double Zq = ((Z[1] + Z[2]) + (Z[3] + Z[4])) + (Z[5] + Z[6]);
        if (glue) {
            const double T = X[0] * (M.gg * Z[0] + M.qg_t * Zq);
            const double U = Z[0] * (M.gg * X[0] + M.qg_t * Xq);
            dI[0] -= T; dK[0] += T; dJ[0] -= U; dL[0] += U;
        }
        const double bZ = M.qg_t * Z[0] + M.a_t * Zq, bX = M.qg_t * X[0] + M.a_t * Xq;
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            if (!BZ_ON(a)) continue;
            const int ab = (a & 1) ? a + 1 : a - 1;
            const double T = X[a] * fma(M.d11, Z[a], fma(M.d1b_t, Z[ab], bZ));
            const double U = Z[a] * fma(M.d11, X[a], fma(M.d1b_t, X[ab], bX));
            dI[a] -= T; dK[a] += T; dJ[a] -= U; dL[a] += U;
        }
    }
    // ------------------------------------------------------------------ u-family: a i->l, b j->k
    {
        double X[7], Z[7];
#pragma unroll
        for (int a = 0; a < 7; ++a) { X[a] = Pi[a] * Ql[a]; Z[a] = Pj[a] * Qk[a]; }
        const double Xq = ((X[1] + X[2]) + (X[3] + X[4])) + (X[5] + X[6]);
        const double Zq = ((Z[1] + Z[2]) + (Z[3] + Z[4])) + (Z[5] + Z[6]);
        if (glue) {
            const double T = M.qg_u * (X[0] * Zq);
            const double U = M.qg_u * (Z[0] * Xq);
            dI[0] -= T; dL[0] += T; dJ[0] -= U; dK[0] += U;
        }
        const double bZ = M.qg_u * Z[0] + M.a_u * Zq, bX = M.qg_u * X[0] + M.a_u * Xq;
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            if (!BZ_ON(a)) continue;
            const int ab = (a & 1) ? a + 1 : a - 1;
            const double T = X[a] * fma(-M.a_u, Z[a], fma(M.d1b_u, Z[ab], bZ));
            const double U = Z[a] * fma(-M.a_u, X[a], fma(M.d1b_u, X[ab], bX));
            dI[a] -= T; dL[a] += T; dJ[a] -= U; dK[a] += U;
        }
    }
    // ------------------------------------------------------------------ s-family: pairs at (i,j) -> pairs at (k,l)
    {
        double In[7], Out[7], Inf[3], Outf[3];
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            const int ab = (a & 1) ? a + 1 : a - 1;
            const bool ok = BZ_ON(a) && BZ_ON(ab);
            In[a] = ok ? Pi[a] * Pj[ab] : 0.0;
            Out[a] = ok ? Qk[a] * Ql[ab] : 0.0;
        }
#pragma unroll
        for (int p = 0; p < 3; ++p) { Inf[p] = In[1 + 2 * p] + In[2 + 2 * p]; Outf[p] = Out[1 + 2 * p] + Out[2 + 2 * p]; }
        const double Inq = (Inf[0] + Inf[1]) + Inf[2], Outq = (Outf[0] + Outf[1]) + Outf[2];
        const double Ing = glue ? Pi[0] * Pj[0] : 0.0, Outg = glue ? Qk[0] * Ql[0] : 0.0;
        if (glue) {
            const double Sg = M.qqgg * (Ing * Outq), Rg = M.qqgg * (Outg * Inq);
            dI[0] -= Sg; dJ[0] -= Sg; dK[0] += Rg; dL[0] += Rg;
        }
        const double bOut = M.qqgg * Outg + M.ann * Outq, bIn = M.qqgg * Ing + M.ann * Inq;
#pragma unroll
        for (int a = 1; a < 7; ++a) {
            const int ab = (a & 1) ? a + 1 : a - 1;
            if (!(BZ_ON(a) && BZ_ON(ab))) continue;
            const int p = (a - 1) >> 1;
            const double S = In[a] * fma(-M.ann, Outf[p], bOut);
            const double R = Out[a] * fma(-M.ann, Inf[p], bIn);
            dI[a] -= S; dJ[ab] -= S; dK[a] += R; dL[ab] += R;
        }
    }
#undef BZ_ON
}

}  // namespace bz
