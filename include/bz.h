/*
 * bz.h -- C ABI of the B200 (sm_100a) library for the Monte Carlo 2->2 collision term of the relativistic
 * Boltzmann equation for gluons and 3-flavour quarks/antiquarks (arXiv:1912.04457), with upwind free
 * streaming, a forward-Euler step and number/energy moments.
 *
 * Citations: "P:nnn" = line nnn of the paper text; "S8x" = SURVEY.md section 8x; "NS" = BASELINE.json
 * north_star (which names these entry points: bz_create(grid, species, alpha_s, m_D), bz_set_f, bz_collision -> dF,
 * bz_stream, bz_step, bz_moments).
 *
 * Conventions (S8b)
 *   - every function returns int: 0 = OK, -1 bad argument, -2 CUDA error (text via bz_last_error), -3 out of
 *     memory, -4 wrong state (a half-built context, or a call that the context's current settings do not allow).  No
 *     exceptions, no aborts, nothing is printed.
 *   - bz_ctx is opaque and OWNS its device buffers (f, f_new, the deposit scratch dN, m^2 per spatial cell,
 *     moment partials).  The caller owns every pointer it passes in.
 *   - pointers named *_dev are DEVICE pointers (e.g. torch tensor .data_ptr()); *_host are HOST pointers;
 *     where a flag `on_device` is given the pointer is interpreted accordingly.
 *   - work is enqueued on the CUDA stream given to bz_set_stream (default: the legacy default stream) and is
 *     asynchronous unless the call says "synchronises".  A context is not thread safe.
 *   - there is no CPU fallback: without a CUDA device bz_create fails with -2.
 *
 * Data layout (S8a), all fp64:
 *   f[(xcell*S + a)*Np + pcell],  pcell = ipx + np*(ipy + np*ipz),  xcell = ix + nx*(iy + ny*iz),
 *   a = index into the ascending list of active species ids (0 = g, 1 = u, 2 = ubar, 3 = d, 4 = dbar, 5 = s,
 *   6 = sbar), Np = np^3, momentum cells contiguous per (spatial cell, species).
 *   dF arrays have the same layout and size S*Nx*Np doubles.
 */
#ifndef BZ_H
#define BZ_H
#ifdef __cplusplus
extern "C" {
#endif

typedef struct bz_ctx bz_ctx;

typedef struct {
    int nx, ny, nz;      /* spatial cells (1,1,1 = homogeneous), periodic                      */
    double dx;           /* spatial cell edge, fm                                               */
    int np;              /* momentum cells per axis (2..1024)                                   */
    double pmin, pmax;   /* momentum box edges, GeV, same on every axis; uniform cells  */
} bz_grid;

/* Create a context on the CUDA device that is current in the calling thread; every later call on the context switches
 * to that device for its duration, so contexts on several devices can be driven from one thread.
 * species: n_species ids in 0..6, strictly ascending.  alpha_s > 0.  Limits: 2 <= np <= 1024; nx*ny*nz*np^3 < 2^32
 * (the Philox counter words and the work items are 32 bits wide).
 * On failure *out is NULL if no context object was created (bad argument), otherwise a half-built context: it holds
 * the error text for bz_last_error and whatever device buffers were allocated before the failure, answers every other
 * call with -4, and the caller MUST bz_destroy it.
 * m_D > 0: fixed regulator mass (GeV) in the t/u propagators of Table I;
 * m_D <= 0: regulator mass^2 = the gluon thermal mass of Eq. 8 evaluated from the current f with
 * E_p = |p|, one value per spatial cell, recomputed at every bz_collision / bz_step (S8a.1, S7).
 * f starts as 0, seed 0, 64 samples per cell, step counter 0. */
int bz_create(const bz_grid* grid, const int* species, int n_species, double alpha_s, double m_D, bz_ctx** out);
int bz_destroy(bz_ctx* ctx);

int bz_set_stream(bz_ctx* ctx, void* cuda_stream);              /* cudaStream_t; NULL = default stream        */
int bz_set_seed(bz_ctx* ctx, unsigned long long seed);          /* Philox key word 0 = low 32 bits (S8c step 1) */
int bz_set_samples(bz_ctx* ctx, int samples_per_cell);          /* kinematic samples per (xcell, pcell) (S3), 1..2^24 */
int bz_set_step(bz_ctx* ctx, unsigned step);                    /* step counter used by bz_step               */

/* User-defined matrix elements ("We also provide an application programming interface (API) for users to
 * define their own matrix elements"): replace one kind of Table I by a constant |M|^2 = value (summed
 * over colours and helicities like Table I, dimensionless), for the straight and the crossed ordering alike.
 * kind: 0 = q1 q2 -> q1 q2 (different flavours, all four rows), 1 = q1 q1 -> q1 q1, 2 = q1 q1bar -> q1 q1bar,
 * 3 = q1 q1bar -> q2 q2bar, 4 = q1 q1bar <-> g g, 5 = q g -> q g, 6 = g g -> g g.  value >= 0 overrides, value < 0
 * restores Table I.  Takes effect at the next bz_collision / bz_step.  -1 on a bad kind or NaN. */
int bz_set_msq_override(bz_ctx* ctx, int kind, double value);

/* Slab of a larger periodic domain (S8e).  The collision term is local in x (Eq. 5); only the drift stencil of
 * Eq. 13 couples neighbouring spatial cells, through the upwind neighbour one cell away.  A domain split
 * along z therefore needs ONE exchange step per Euler step: each slab keeps a copy of its two neighbours' boundary
 * layers ("halo" layers).  After bz_set_slab the context's z layers [z_begin, z_end) are the slab's own cells and the
 * layers outside are halo copies that the caller refreshes (bz_copy_layers) before every bz_step / bz_stream:
 *   - bz_collision / bz_step collide only the own cells (dF_coll = 0 elsewhere) and draw the samples of local cell x
 *     from the Philox spatial counter x + xcell_offset (mod 2^32), i.e. the cell's index in the undecomposed domain;
 *   - the totals of bz_moments run over the own cells only (per-cell values are written for every layer);
 *   - bz_stream / the transport part of bz_step treat the context's grid as periodic as always: the values they
 *     leave in the halo layers are meaningless and are overwritten by the next refresh.
 * Default: offset 0, all layers own.  Returns -1 unless 0 <= z_begin <= z_end <= nz. */
int bz_set_slab(bz_ctx* ctx, unsigned xcell_offset, int z_begin, int z_end);

/* Copy n_layers whole z layers (nx*ny*S*Np doubles each, contiguous in the layout above) starting at layer z0
 * between the context's f and a DEVICE buffer: to_ctx != 0 writes f, to_ctx == 0 reads it.  Asynchronous on the
 * context's stream.  This is the pack/unpack of the halo exchange (the transfer itself is the caller's: NCCL
 * send/recv of the buffer through torch.distributed, paper_1912_04457_b200/slab.py). */
int bz_copy_layers(bz_ctx* ctx, int z0, int n_layers, double* buf_dev, int to_ctx);

/* Copy S*Nx*Np doubles into / out of the context.  on_device != 0: f is a device pointer (async copy on the
 * context's stream); on_device == 0: f is a host pointer and the call synchronises the stream. */
int bz_set_f(bz_ctx* ctx, const double* f, int on_device);
int bz_get_f(bz_ctx* ctx, double* f, int on_device);

/* dF = dt * C_a[f]: Monte Carlo estimate (Eq. 20) of the 2->2 collision term (Eq. 3-5) with
 * symmetrical sampling (Eq. 22): for every (xcell, p1 cell, sample) a Philox4x32-10 keyed (seed, step),
 * counter (block, sample, pcell, xcell) draws p2 uniform in the box and an isotropic centre-of-mass direction
 * (Marsaglia), p3 and p4 follow by the boost, all ordered LO QCD channels of Table I are evaluated with the
 * Bose/Fermi gain-loss bracket of Eq. 5, and the same weight goes with - to the p1, p2 cells and with + to the
 * p3, p4 cells (S8c steps 0-6).  dF_dev: device pointer, S*Nx*Np doubles, overwritten.  dt_fm in fm/c.
 * Asynchronous. */
int bz_collision(bz_ctx* ctx, double dt_fm, unsigned step, double* dF_dev);

/* dF = first-order upwind finite-volume free-streaming increment, periodic, velocity p/|p| at the momentum cell
 * centre (flux form of the drift term of Eq. 13; S8a.6).  Asynchronous. */
int bz_stream(bz_ctx* ctx, double dt_fm, double* dF_dev);

/* ---- NEXT rank 2 of SURVEY.md 8f: the paper's own left-hand side (massive dispersion, drift AND force) ----------
 * Thermal masses^2 per spatial cell, mass2[x][4] = (m_g^2, m_u^2, m_d^2, m_s^2) in GeV^2, m_qbar = m_q, 0 at start.
 * bz_thermal_masses evaluates Eq. 8 and Eq. 9 on the current f,
 *     m_g^2 = g^2 [6 I_g + sum_q I_q],  m_qi^2 = (4/3) g^2 [2 I_g + I_qi + I_qbar_i],  I_a = sum_cells d3p f_a / ((2pi)^3 E_p^a),
 * with E_p^a = sqrt(p^2 + m_a^2(x)) from the masses stored so far (all 0 before the first call: the first-step
 * prescription E_p = |p| of P:107; a cell with E = 0 is skipped), stores the result in the context and, if
 * out_host != NULL, copies the Nx*4 doubles to the host (then it synchronises).  bz_set_masses sets them directly
 * from HOST memory (e.g. the constant m_g^2 = 0.5 GeV^2 of Fig. 5); synchronises. */
int bz_thermal_masses(bz_ctx* ctx, double* out_host);
int bz_set_masses(bz_ctx* ctx, const double* mass2_host);

/* Energy balance with dynamical masses (Eq. 11-12; Eq. 26), written to HOST memory, 5 doubles per
 * spatial cell: out[x][0] = T^00_kin(x) = sum_a N_a sum_cells d3p E_p^a f_a / (2pi)^3 (GeV^4), out[x][1 + c] = Q_c(x) =
 * sum_{a in mass class c} N_a sum_cells d3p f_a / ((2pi)^3 E_p^a) (GeV^2) for c = g, u, d, s, with E_p^a from the
 * stored masses.  The source term of Eq. 12 is S_ex^nu = (1/2) sum_c (d^nu m_c^2) Q_c; Eq. 26 compares d_0 T^00_kin with
 * S_ex^0 (the caller differences T^00 and the masses over steps, as the paper does for Fig. 6).  Synchronises. */
int bz_energy_diag(bz_ctx* ctx, double* out_host);

/* dF = -dt { drift + force } of Eq. 15, the central-difference form of the left-hand side of Eq. 13
 * (P:133), with E_p^a(x) = sqrt(p^2 + m_a^2(x)) from the stored masses; periodic in x and in p.  Per axis i:
 *   drift_i = [ p_i f_p(x+)/E_p(x+) - p_i f_p(x-)/E_p(x-) ] / (2 dx)
 *   force_i = -[ f_{p+}(x) (E_{p+}(x+) - E_{p+}(x-))/(2 dx) - f_{p-}(x) (E_{p-}(x+) - E_{p-}(x-))/(2 dx) ] / (2 dp)
 * dF_dev: device pointer, S*Nx*Np doubles, overwritten.  Asynchronous. */
int bz_vlasov(bz_ctx* ctx, double dt_fm, double* dF_dev);

/* ---- NEXT rank 1 of SURVEY.md 8f: the paper's own collision path ---------------------------------------------
 * dF = dt * C_a[f] estimated as the paper does (Eq. 17-21): the grid point p (cell centre) is the OUTGOING
 * particle d of Eq. 5; (k1x, k1y, k3x, k3y, k3z) are uniform in the momentum box (Eq. 20, V_domain = L^5,
 * Philox blocks 64-66 of the (seed, step) / (block, sample, pcell, xcell) stream); k1z runs over the roots of
 * E1 + E2 = E3 + Ep with weight 1/|J| (Eq. 18-19); k2 = k3 + p - k1; dispersion E^a = sqrt(p^2 + m_a^2(x)) with the
 * stored thermal masses (bz_thermal_masses / bz_set_masses; all 0 = massless), so every tuple of mass classes solves its
 * own roots; Table I is evaluated at the root's massive s, t, u with the regulator m_g^2(x) (m_D^2 if m_D > 0);
 * symmetrical sampling (Eq. 22): A = Kp |M|^2 [f f F F - F F f f] / (|J| E1 E2 E3 Ep) goes with - to the cells of k1, k2
 * and with + to those of k3, p; Kp = (dt/hbarc) L^5 / (Ns (2 pi)^5 16) / 8.  A root with k1 or k2 outside the box is
 * dropped (S9).  dF_dev: device pointer, S*Nx*Np doubles, overwritten.  Asynchronous.  Honours bz_set_slab and
 * bz_set_msq_override. */
int bz_collision_paper(bz_ctx* ctx, double dt_fm, unsigned step, double* dF_dev);

/* ---- NEXT rank 3 of SURVEY.md 8f: importance sampling of the t/u-channel peaks ------------------------------------
 * dF = dt * C_a[f] with the estimator of bz_collision, except that the momentum transfer is not uniform on [-s, 0]
 * (isotropic CM direction) but drawn from p(t) = (1/2)[g(t) + g(-s - t)], g(t) = 1/((m^2 - t)^2 (1/m^2 - 1/(s + m^2))),
 * where Table I peaks, with the azimuth about the CM direction of p1 uniform, and every deposit is
 * multiplied by the weight (1/s)/p(t): same expectation, smaller variance for m^2 << s.  p1, p2 and s are those of
 * bz_collision for the same (seed, step) (Philox blocks 0, 1); t uses block 96, the azimuth blocks 97...  m^2 is the
 * regulator of the spatial cell (an empty cell, m^2 = 0: uniform t, weight 1).  dF_dev: device pointer, S*Nx*Np
 * doubles, overwritten.  Asynchronous.  Honours bz_set_slab and bz_set_msq_override. */
int bz_collision_is(bz_ctx* ctx, double dt_fm, unsigned step, double* dF_dev);

/* ---- NEXT rank 3 of SURVEY.md 8f, the other half: in-box sampling of the CM direction ----------------------------------
 * dF = dt * C_a[f] with the estimator of bz_collision, except that the CM direction n is not uniform on the sphere.  With
 * p3 = P/2 + A n, rows A_c = (M e_c + P_c P/(E + M))/2 of the boost of S8c step 2, |A_c| = sqrt(s + P_c^2)/2, both outgoing
 * legs stay inside the momentum box on axis c iff |a_c . n| <= beta_c = min(1, (L/2 - |P_c/2 - box centre|)/|A_c|), a_c =
 * A_c/|A_c|: the accepted set (reading S9) is the intersection of three zones of the sphere.  The zone with the smallest
 * beta_c is sampled exactly -- z = a . n uniform on [-beta, beta], azimuth uniform: Archimedes' hat-box theorem, area
 * fraction beta -- and every deposit is multiplied by beta; the other two zones still reject.  Eq. 20's expectation
 * is unchanged because the integrand vanishes outside the zone; 78 % of the samples deposit instead of 46 %.
 * Same Philox blocks (0, 1, 2 + k) and the same Marsaglia acceptance as bz_collision: z = beta (1 - 2 q), (cos, sin) =
 * (v1, v2)/sqrt(q).  dF_dev: device pointer, S*Nx*Np doubles, overwritten.  Asynchronous.  Honours bz_set_slab and
 * bz_set_msq_override. */
int bz_collision_box(bz_ctx* ctx, double dt_fm, unsigned step, double* dF_dev);

/* Test-only: the samples of bz_collision_box: cells_dev[n][Ns][4] = (j, k, l, flag), stu_dev[n][Ns][3] = (s, t, u),
 * w_dev[n][Ns] = the weight beta (0 where !(s > 0)). */
int bz_debug_samples_box(bz_ctx* ctx, unsigned step, int xcell, int pcell_begin, int pcell_end, int* cells_dev,
                         double* stu_dev, double* w_dev);

/* Test-only: the samples of bz_collision_is for regulator m2 (GeV^2): cells_dev[n][Ns][4] = (j, k, l, flag),
 * stu_dev[n][Ns][3] = (s, t, u) of the constructed momenta, w_dev[n][Ns] = the weight (0 where !(s > 0)). */
int bz_debug_samples_is(bz_ctx* ctx, unsigned step, int xcell, int pcell_begin, int pcell_end, double m2, int* cells_dev,
                        double* stu_dev, double* w_dev);

/* Collision term used by bz_step: 0 (default, NS) = the massless centre-of-mass sampler of bz_collision; 1 = the
 * paper's own sampler of bz_collision_paper.  With mode 1 and transport scheme 1, bz_step is the paper's program as a
 * whole: thermal masses from the old f (Eq. 8-9), collision term by Eq. 17-21 with those masses, Eq. 15 for the
 * drift and force terms, forward Euler.  2 = the importance-sampled estimator of bz_collision_is, 3 = the in-box estimator
 * of bz_collision_box.  -1 on a bad mode. */
int bz_set_collision(bz_ctx* ctx, int mode);

/* Test-only: the roots of the paper sampler for ONE mass tuple msq_host = (m_a^2, m_b^2, m_c^2, m_d^2), p1 cells
 * [pcell_begin, pcell_end) of spatial cell xcell: cells_dev[n][Ns][6] = (cell of k3, number of roots kept, cell of k1
 * and of k2 for root 0, the same for root 1; -1 where there is none), stu_dev[n][Ns][6] = (s, t, u) of root 0 and 1. */
int bz_debug_paper_samples(bz_ctx* ctx, unsigned step, int xcell, int pcell_begin, int pcell_end, const double* msq_host,
                           int* cells_dev, double* stu_dev);

/* Test-only, host only (needs no device): the ordered channel table of the paper sampler for a species list (Eq. 3-4,
 * S8c step 5), 7 ints per channel (a, b, c, d as layout indices, kind, crossed, mass-class key) into out_host (at most
 * `capacity` channels are written); returns the number of channels. */
int bz_debug_paper_channels(const int* species, int n_species, int* out_host, int capacity);

/* Transport scheme used by bz_step: 0 (default, NS) = first-order upwind drift with massless velocities (bz_stream);
 * 1 = Eq. 15 (bz_vlasov) with the thermal masses re-evaluated from the old f at the start of every step;
 * 2 = Eq. 15 with the masses as stored (bz_set_masses / the last bz_thermal_masses).  The collision term is chosen
 * independently with bz_set_collision. */
int bz_set_transport(bz_ctx* ctx, int scheme);

/* One forward-Euler step (Eq. 15 unsplit; S8a.7): f <- (f + dF_stream) + dF_coll with both increments
 * from the old f and the context's step counter as the Philox step; the counter is then incremented.
 * Asynchronous. */
int bz_step(bz_ctx* ctx, double dt_fm);

/* n forward-Euler steps, equivalent to n calls of bz_step.  The paper's runs are 10^4 - 10^6 steps of a 30^3 grid (P:330,
 * P:348), i.e. steps of a few hundred microseconds, where the time between kernels counts: with transport scheme 0 and
 * collision mode 0, 2 or 3 two consecutive steps (f -> f_new -> f: row sums, collision kernel, stream + Euler kernel,
 * twice) are captured once as a CUDA graph on a stream of the library's own and replayed; the Philox step word lives on
 * the device, is read by the collision kernel and advanced by the Euler kernel, so nothing returns to the host between
 * steps.  Other settings run the plain loop.  Same results as n x bz_step up to the summation order of the deposits.
 * Asynchronous with respect to the host like bz_step (the context's stream waits for the replays); the step copied to
 * the device word is read from host memory at the call.  n = 0 is a no-op; n < 0: -1. */
int bz_step_n(bz_ctx* ctx, double dt_fm, int n);

/* The same step end to end from HOST memory: f_in_host (S*Nx*Np doubles, ideally pinned) replaces the context's f,
 * one bz_step is taken, and the new f is written to f_out_host; the context keeps the new f and the incremented step
 * counter exactly as after bz_set_f + bz_step + bz_get_f.  With at least 3 z layers and transport scheme 0 the work
 * is pipelined in chunks of z layers over three streams -- host-to-device copies of the chunks to come, collision of
 * chunk k (the collision term needs only the chunk's own cells, Eq. 5), stream + Euler of chunk k-1 (its upwind
 * stencil needs the old f of both z neighbours: it is issued as soon as chunk k has arrived) and the device-to-host
 * copy of its result run concurrently; the first and the last chunk are handled in quarters on large grids --
 * otherwise it is that plain sequence.  Same results as the plain sequence up to the summation order of the deposits.  Synchronises.
 * Slab contexts (bz_set_slab): both host buffers still have the size of the whole context, but only the OWN layers are
 * read from f_in_host and written to f_out_host; the halo layers must have been refreshed on the device (bz_copy_layers)
 * before the call, from the neighbours' boundary layers of the same new f (paper_1912_04457_b200/slab.py, step_host);
 * needs transport scheme 0 and collision mode 0 (-4 otherwise). */
int bz_step_host(bz_ctx* ctx, double dt_fm, const double* f_in_host, double* f_out_host);

/* Moments of the current f (Eq. 10; T^00 of Eq. 11, massless; S8a.8) written to HOST memory:
 *   out_host[(xcell*S + a)*2 + {0,1}] = n_a(x) in GeV^3, e_a(x) in GeV^4;
 *   then S pairs (N_a, E_a) = sum_x (n, e) dx^3/hbarc^3  (dimensionless, GeV);
 *   then Nx values m^2(x) in GeV^2 (the regulator of S8a.1 for the current f, or m_D^2).
 * Size 2*S*Nx + 2*S + Nx doubles.  Synchronises. */
int bz_moments(bz_ctx* ctx, double* out_host);

/* The same moments for a caller that keeps f in device memory of its own and cannot allocate any: no context, no
 * cudaMalloc / cudaFree, no allocating library call, in this call or behind it.  Meant for
 *   - a solver whose own f already fills most of the card: a context costs about 4.3 x the size of f (f, f_new and two
 *     cell-major staging copies), which such a caller does not have, just to read n, e and m^2 off its state;
 *   - a monitor that runs beside a long step on another stream: cudaMalloc and cudaFree synchronise the whole device
 *     and would stall that step;
 *   - a process whose device memory belongs in full to a framework's pool, where a raw cudaMalloc fails.
 * Arguments: grid, species, n_species, alpha_s, m_D as for bz_create (same checks); f_dev: DEVICE pointer, S*Nx*Np
 * doubles in the layout above, read only; out_dev: DEVICE pointer, 2*S*Nx + 2*S + Nx doubles, overwritten, with the
 * content bz_moments writes to the host (totals over all cells); cuda_stream: cudaStream_t, NULL = default stream.  The
 * caller owns both buffers; they must live on the device that is current in the calling thread.  Asynchronous.
 * Scratch: the row sums between the two kernels (3 doubles per (spatial cell, species)) live in a fixed array inside
 * the library image, 65536 rows = 1.5 MiB, which every GPU that loads the library holds until the process exits.
 * Limit: nx*ny*nz * n_species <= 65536 (config 4 has 28672, the paper's 20^3 cells x 7 species 56000); a larger
 * grid is refused with -5 before anything is launched.
 * First call on a device: it also looks up the array's device address (cudaGetSymbolAddress, once per device, cached;
 * the runtime may load the library's kernels onto the device at that moment).  Make that first call before any stream
 * capture begins.
 * Sharing: all calls on a device, from every thread and stream, use the one array.  Each call overwrites the rows it
 * reads before reading them, so what an earlier call left behind never shows; but two calls that overlap on the GPU
 * (different streams, no ordering between them) race on the array and both results are then undefined.  Order such
 * calls yourself (same stream, or an event).
 * Returns 0, -1 bad argument, -2 CUDA error, -5 grid beyond the scratch; bz_noalloc_last_error gives the text of
 * the calling thread's last failure ("" after a success). */
int bz_moments_noalloc(const bz_grid* grid, const int* species, int n_species, double alpha_s, double m_D,
                       const double* f_dev, double* out_dev, void* cuda_stream);
const char* bz_noalloc_last_error(void);

/* Text of the last CUDA error seen by this context ("" if none). */
const char* bz_last_error(const bz_ctx* ctx);

/* Kernel timing for the roofline report: while profiling is on (on != 0), bz_step / bz_collision bracket two groups
 * of launches with CUDA events on the context's stream: group 0 = the collision kernel (with the cell-major staging
 * copy when one is needed), group 1 = the stream + Euler kernel of bz_step.  bz_get_profile synchronises the stream,
 * writes the summed duration (milliseconds) and the number of bracketed regions of that group since the last call,
 * and clears the group's record. */
int bz_set_profile(bz_ctx* ctx, int on);
int bz_get_profile(bz_ctx* ctx, int group, double* ms_total, int* launches);

/* FP64 FMA peak of the current device in TFLOP/s, measured with a register-resident DFMA chain kernel on the default
 * stream (a few milliseconds; synchronises).  This is the FP64 leg of the roofline NS defines for the collision
 * kernel ("the slower of FP64 FMA peak and gathered/scattered bytes at HBM bandwidth").  Needs no context. */
int bz_measure_fp64_peak(double* tflops_out_host);

/* Number of CUDA kernels this library has launched in this process so far (all contexts); bench.py reports the
 * difference over its timed region as "gpu_launches". */
unsigned long long bz_launch_count(void);

/* Kinematic samples drawn by the hot path's collision kernel (bz_collision, bz_step, bz_step_host) since the last
 * reset: generated = spatial cells x momentum cells x samples per cell of every launch; accepted = those with s > 0 and
 * both outgoing legs inside the momentum box (reading S9: the others deposit nothing), counted on the device by the
 * kernel itself.  bench.py weights the roofline with accepted / generated.  reset != 0 clears both.  Synchronises. */
int bz_get_sample_counts(bz_ctx* ctx, unsigned long long* generated_out, unsigned long long* accepted_out, int reset);

/* Reading S8 of SURVEY.md 8c: Table I with the regulator in the t and u propagators is evaluated literally
 * and can turn negative (e.g. q qbar <-> g g, where -96 (t^2 + u^2)/s^2 stays while the regulated part shrinks); nothing
 * is clamped.  This call reports how often: it regenerates the kinematic samples that bz_collision draws for `step` in
 * spatial cells [xcell_begin, xcell_end), evaluates the |M|^2 of every kind and ordering with each cell's regulator for
 * the current f (honouring bz_set_msq_override) and writes 15 counters to HOST memory: out_host[0] = samples that
 * deposit; out_host[1 + 2*kind + crossed] = those of them with |M|^2(kind, ordering) < 0, kind as in
 * bz_set_msq_override, crossed = 1 for the t <-> u exchanged ordering (the same number for the symmetric kinds).
 * Weighted with the number of ordered channels of each (kind, ordering) this is the fraction of negative
 * (sample, channel) pairs.  Not part of the timed path.  Synchronises. */
int bz_msq_sign_counts(bz_ctx* ctx, unsigned step, int xcell_begin, int xcell_end, unsigned long long* out_host);

/* ---- test-only exports ---------------------------------------------------------------------------------- */
/* Sampled cells of p1 cells [pcell_begin, pcell_end) of spatial cell xcell, needed for the "bit-exact sampled
 * indices" target of NS: cells_dev[n][Ns][4] = (j, k, l, flag) int32, stu_dev[n][Ns][3] = (s, t, u) or NULL.
 * k = l = -1 when !(s > 0); k or l = -1 when that leg leaves the box; flag = 1 iff the sample deposits. */
int bz_debug_samples(bz_ctx* ctx, unsigned step, int xcell, int pcell_begin, int pcell_end,
                     int* cells_dev, double* stu_dev);

#ifdef __cplusplus
}
#endif
#endif
