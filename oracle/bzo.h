/*
 * bzo.h -- CPU ORACLE for the Monte Carlo 2->2 collision term (arXiv:1912.04457).
 *
 * TEST INFRASTRUCTURE ONLY.  This is a plain, slow, sequential fp64 restatement of the
 * method; it is imported only by tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs.  It shares no code with the CUDA library
 * (paper_1912_04457_b200/csrc) and neither includes the other.
 *
 * Citations: "P:nnn" = /root/reference/PAPER.md line nnn; "S8c step k" = SURVEY.md
 * section 8c, step k (the reading of the points the paper leaves open); "NS" =
 * BASELINE.json north_star.
 *
 * All pointers are HOST pointers.  Every function returns 0 on success, a negative
 * value on a bad argument (-1) or allocation failure (-3).
 *
 * Layout (S8a):  f[(xcell*S + a)*Np + pcell],  pcell = ipx + n*(ipy + n*ipz),
 *                xcell = ix + nx*(iy + ny*iz),  a = index into the active species list.
 * Species ids: 0 = g, 1 = u, 2 = ubar, 3 = d, 4 = dbar, 5 = s, 6 = sbar.
 */
#ifndef BZO_H
#define BZO_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct bzo_ctx bzo_ctx;

typedef struct {
    int nx, ny, nz;      /* spatial cells (1,1,1 = homogeneous)          */
    double dx;           /* spatial cell edge, fm                         */
    int np;              /* momentum cells per axis                       */
    double pmin, pmax;   /* momentum box edges, GeV (same on every axis)  */
} bzo_grid;

/* matrix-element kinds of Table I, in the order of S8c step 4 */
enum { BZO_M_A = 0, BZO_M_11 = 1, BZO_M_1B = 2, BZO_M_ANN = 3, BZO_M_QQGG = 4, BZO_M_QG = 5, BZO_M_GG = 6,
       BZO_N_KINDS = 7 };

/* one ordered channel a(slot1,cell i) b(slot2,cell j) -> c(slot3,cell k) d(slot4,cell l); S8c step 5 */
typedef struct { int a, b, c, d; int kind; int crossed; } bzo_channel;

/* everything one kinematic sample produces (S8c steps 1-3); used by the pins P1, P2 */
typedef struct {
    int flag;            /* 1 = deposits, 0 = contributes nothing                              */
    int j, k, l;         /* cells of p2, p3, p4; k = l = -1 if !(s > 0); k or l = -1 if outside */
    int attempts;        /* Marsaglia attempts used (1..62), 63 = exhausted                    */
    double s, t, u, E1, E2, E3;
    double p1[3], p2[3], p3[3], p4[3], nhat[3];
} bzo_sample;

int  bzo_create (const bzo_grid* grid, const int* species, int n_species,
                 double alpha_s, double m_D, bzo_ctx** out);   /* m_D <= 0: m^2 from f (Eq. 8) */
int  bzo_destroy(bzo_ctx*);
int  bzo_set_seed   (bzo_ctx*, unsigned long long seed);       /* low 32 bits are used (S8c step 1)   */
int  bzo_set_samples(bzo_ctx*, int samples_per_cell);
int  bzo_set_threads(bzo_ctx*, int n);                         /* OpenMP threads, default 1           */
int  bzo_get_threads(const bzo_ctx*);
int  bzo_set_f  (bzo_ctx*, const double* f);
int  bzo_get_f  (const bzo_ctx*, double* f);
int  bzo_set_step(bzo_ctx*, unsigned step);                    /* internal step counter of bzo_step   */
/* Slab of a larger periodic domain (S8e: the collision term is local in x, Eq. 5; only the drift stencil of
 * Eq. 13 couples neighbouring cells).  The context's z layers [z_begin, z_end) are this slab's own cells, the layers
 * outside are halo copies the caller refreshes before every step.  Only own cells collide and enter the totals of
 * bzo_moments; the Philox spatial counter of local cell x is x + xcell_offset, so that a cell draws the same
 * samples as in the undecomposed domain.  Default: offset 0, all layers. */
int  bzo_set_slab(bzo_ctx*, unsigned xcell_offset, int z_begin, int z_end);

/* dF = dt * C_a[f] (S8c steps 1-6).  Also fills the per-value gross |A| sum (S16), see bzo_get_gross. */
int  bzo_collision(bzo_ctx*, double dt_fm, unsigned step, double* dF);
int  bzo_get_gross(const bzo_ctx*, double* gross);             /* sum|A| / N_a per value, same layout  */
/* dF = upwind free-streaming increment (S8a.6; flux form of Eq. 13) */
int  bzo_stream   (bzo_ctx*, double dt_fm, double* dF);
/* ---- NEXT rank 2 (S8f): the paper's own left-hand side -------------------------------------------------------
 * Thermal masses^2 per spatial cell, mass2[x][4] = (m_g^2, m_u^2, m_d^2, m_s^2), m_qbar = m_q (Eq. 8-9).
 * bzo_thermal_masses evaluates Eq. 8-9 on the current f with E_p^a = sqrt(p^2 + m_a^2) from the masses stored so far
 * (0 at start = the first-step prescription E_p = |p|) and stores the result; out may be NULL. */
int  bzo_set_masses(bzo_ctx*, const double* mass2);
int  bzo_get_masses(const bzo_ctx*, double* mass2);
int  bzo_thermal_masses(bzo_ctx*, double* out);
/* energy balance (Eq. 11-12, 26): out[x][5] = T^00_kin(x), then Q_c(x) = sum_{a in class c} N_a int d3p f_a/((2pi)^3 E^a)
 * for c = g, u, d, s, with E^a = sqrt(p^2 + m_a^2(x)) from the stored masses; S_ex^nu = (1/2) sum_c (d^nu m_c^2) Q_c */
int  bzo_energy_diag(const bzo_ctx*, double* out);
/* dF = -dt { drift + force } of Eq. 15: central differences in x and p, periodic in both,
 * E_p^a(x) = sqrt(p^2 + m_a^2(x)) from the stored masses */
int  bzo_vlasov   (bzo_ctx*, double dt_fm, double* dF);
/* transport used by bzo_step: 0 = upwind massless (default), 1 = Eq. 15 with the masses re-evaluated from the old f
 * every step, 2 = Eq. 15 with the masses as stored */
int  bzo_set_transport(bzo_ctx*, int scheme);
/* collision term used by bzo_step: 0 = bzo_collision (default), 1 = bzo_collision_paper, 2 = bzo_collision_is, 3 = bzo_collision_box */
int  bzo_set_collision(bzo_ctx*, int mode);
/* ---- NEXT rank 3 (S8f): importance sampling of the t/u-channel peaks of Table I --------------------------------
 * bzo_collision_is: the estimator of bzo_collision with t drawn from (1/2)[g(t) + g(u)], g ~ 1/(m^2 - t)^2, the azimuth
 * about the CM direction of p1 uniformly, and every deposit multiplied by the weight (1/s)/p(t): same expectation.
 * bzo_sample_one_is: one such sample (fields as bzo_sample_one; attempts = azimuth attempts) and its weight. */
int  bzo_collision_is(bzo_ctx*, double dt_fm, unsigned step, double* dF);
int  bzo_sample_one_is(const bzo_ctx*, unsigned step, int xcell, int pcell, int sample, double m2, bzo_sample* out, double* weight);
/* ---- NEXT rank 3 (S8f), the other half: the CM direction is drawn uniformly from the tightest of the three zones
 * |a_c . n| <= beta_c of the sphere outside which p3 or p4 leaves the momentum box (Archimedes: area fraction beta_c, z
 * uniform), weight beta: same expectation as bzo_collision (Eq. 20), 78 % instead of 46 % of the samples deposit.
 * Same Philox blocks and Marsaglia acceptance as bzo_collision.  bzo_sample_one_box: one such sample and its weight. */
int  bzo_collision_box(bzo_ctx*, double dt_fm, unsigned step, double* dF);
int  bzo_sample_one_box(const bzo_ctx*, unsigned step, int xcell, int pcell, int sample, bzo_sample* out, double* weight);

/* ---- NEXT rank 1 (S8f): the paper's own collision path (Eq. 17-21, massive dispersion) ----------------------------
 * one root of E1 + E2 = E3 + Ep (Eq. 18-19): momenta k1, k2, their cells, the four energies, the Jacobian of Eq. 19 and
 * the massive Mandelstam variables */
typedef struct { double k1[3], k2[3]; int i1, i2; double E1, E2, E3, Ep, J, s, t, u; } bzo_proot;
/* the sample (step, xcell, pcell, sample) of the paper's sampler for one mass tuple msq = (m_a^2, m_b^2, m_c^2, m_d^2):
 * k3 (drawn), its cell, and the 0..2 roots kept; returns their number */
int  bzo_paper_sample(const bzo_ctx*, unsigned step, int xcell, int pcell, int sample, const double msq[4],
                      double k3_out[3], int* i3_out, bzo_proot out[2]);
/* dF = dt C[f] with the paper's sampler and E^a = sqrt(p^2 + m_a^2(x)) from the stored thermal masses; also fills
 * the gross sums (bzo_get_gross) */
int  bzo_collision_paper(bzo_ctx*, double dt_fm, unsigned step, double* dF);
/* the same, channel by channel: every ordered channel solves its own roots, nothing is shared between channels
 * (Eq. 3-4 as printed); the check of bzo_collision_paper's grouping by mass tuple.  Sequential. */
int  bzo_collision_paper_plain(bzo_ctx*, double dt_fm, unsigned step, double* dF);
/* f <- (f + dF_stream) + dF_coll, both from the old f (Eq. 15 unsplit); step counter ++ */
int  bzo_step     (bzo_ctx*, double dt_fm);
/* out = [N_x][S][2] (n, e) then [S][2] totals (N, E) then m^2[N_x]  (Eq. 10-11; Eq. 8) */
int  bzo_moments  (bzo_ctx*, double* out);

/* sampled cells of p1 cells [pcell_begin, pcell_end) of one spatial cell:
 * cells[n][Ns][4] = (j, k, l, flag), stu[n][Ns][3] = (s, t, u) or NULL */
int  bzo_debug_samples(bzo_ctx*, unsigned step, int xcell, int pcell_begin, int pcell_end,
                       int* cells, double* stu);

/* ---- hooks that exist only so the pins can reach the oracle's own arithmetic ---- */
/* full kinematic record of one sample */
int  bzo_sample_one(const bzo_ctx*, unsigned step, int xcell, int pcell, int sample, bzo_sample* out);
/* Philox4x32-10 block (S8c step 1) and the two uniforms made from it */
void bzo_philox4x32_10(const unsigned ctr[4], const unsigned key[2], unsigned out[4]);
double bzo_uniform(unsigned a, unsigned b);
/* Table I value for one kind (straight); crossed = same with t and u exchanged */
double bzo_msq(int kind, double s, double t, double u, double m2, double g4);
/* channel table */
int  bzo_n_channels(const bzo_ctx*);
int  bzo_get_channels(const bzo_ctx*, bzo_channel* out);
/* |M|^2 override per kind: value >= 0 replaces Table I for that kind (P:89 user-defined matrix
 * elements); value < 0 restores Table I.  Used by pin P10. */
int  bzo_set_msq_override(bzo_ctx*, int kind, double value);
/* The per-sample channel loop (S8c step 6) on caller-supplied occupation numbers:
 * fv[slot][a] = f_a at the cell of slot (0..3 = i, j, k, l).  Writes dN[slot][a] (number units,
 * signed deposits -A,-A,+A,+A summed over channels), fwd[ch] per channel, and returns sum|A|. */
double bzo_sample_channels(const bzo_ctx*, const double* fv, double s, double t, double u,
                           double E1, double E2, double m2, double dt_fm,
                           double* dN, double* fwd);
/* One spatial cell's collision on a caller-supplied tile f_tile[S][Np], p1 cells [p_begin, p_end).
 * mode 0 = symmetric (the method, Eq. 22), mode 1 = labelled (no reuse: only the slot-1 deposit,
 * weight 1/2 instead of 1/8; pin P5).  dN[S][Np] and gross[S][Np] (may be NULL) are ACCUMULATED
 * into, in number units (not divided by N_a).  m2_out receives the regulator used. */
int  bzo_collision_tile(const bzo_ctx*, double dt_fm, unsigned step, int xcell, const double* f_tile,
                        int p_begin, int p_end, int mode, double* dN, double* gross, double* m2_out);
/* regulator mass^2 of one tile (Eq. 8 with E_p = |p|) */
double bzo_regulator_m2(const bzo_ctx*, const double* f_tile);

#ifdef __cplusplus
}
#endif
#endif
