// bz_internal.h -- context and kernel-launcher declarations shared by the translation units of libbz.so.
#pragma once
#include <cuda_runtime.h>

#include <atomic>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/bz.h"
#include "bz_sample.cuh"

namespace bz {

constexpr double kHbarc = 0.1973269804;   // GeV fm (S8c step 0)
constexpr double kPi = 3.14159265358979323846;

struct CollideParams {
    GridConst g;
    const double* f_aos;  // [Nx][Np][SP] cell-major staging copy of f (pad slots 0)
    double* dN_aos;       // [Nx][Np][SP] deposit scratch in number units, zero on entry
    const double* rowsum; // [Nx][S][3] row sums of the current f (rowsum_kernel): [2] = sum f d3p/((2pi)^3 |p|)
    double g2, mD2;       // 4 pi alpha_s; m_D^2 if m_D > 0 (fixed regulator), else 0: m^2(x) from the row sums (Eq. 8, S8a.1)
    unsigned glue_slot_mask;   // bit a: layout index a is the gluon
    const double* cell_tab;   // [Np][4] (p1x, p1y, p1z, E1) of the momentum cell centres
    int S, Np, Nx, Ns;
    unsigned long long* counters;   // device [1]: kinematic samples accepted (both outgoing legs in the box), accumulated over launches
    unsigned* work_counter;   // device [2]: next work item of the persistent kernel, CTAs that have finished; both 0 on entry,
                              // reset by the last CTA to finish
    unsigned n_items;         // Nx * regions_per_x work items, item = xcell * regions_per_x + region
    int x_begin;              // first colliding spatial cell (items address xcell = x_begin + item / regions_per_x)
    uint32_t x_rng_offset;    // Philox spatial counter = xcell + x_rng_offset (slab of a larger domain, bz_set_slab)
    int units_per_item, ppc;  // passes of 32 samples per work item; passes per p1 cell = ceil(Ns / 32)
    int regions_per_x;        // work items per spatial cell = ceil(Np * ppc / units_per_item)
    uint32_t seed, step;
    const uint32_t* step_ptr; // device: if not NULL the Philox step is read from here (captured graphs, bz_step_n), else `step`
    double g4K;           // (4 pi alpha_s)^2 * K,  K = dtG Vp / (2048 pi^4 Ns)    (S8c step 0)
    unsigned mask;        // bit id set <=> species id active
    int slot[7];          // species id -> index a in the layout (or -1)
    int has_ovr;          // bz_set_msq_override: some kind of Table I is replaced by a constant
    double msq_ovr[7];    // per kind: value / g^4, or -1 (Table I)
    int sampler;          // 0 isotropic CM direction (hot path), 1 importance-sampled t, 2 in-box direction (NEXT rank 3)
};

// NEXT rank 1 (bz_paper.cu): ordered channel a(k1) b(k2) -> c(k3) d(p), layout indices; groups share a mass-class tuple
struct PaperChannel { unsigned char a, b, c, d, kind, crossed, glue /* bit s: leg s is a gluon */, key /* classes, 2 bits per leg */; };
struct PaperGroup { int key, begin, end; };
struct PaperParams {
    GridConst g;
    const double* f;          // cell-major copy of f, [Nx][Np][SP] (the collision kernel's gather source f_aos; f itself if SP == 1)
    double* dN;               // cell-major deposit scratch dN_aos [Nx][Np][SP], number units, zero before the launch
    int SP;                   // doubles per cell in the two: 1 (one species) or 8
    int cta_groups;           // spatial cells are dealt round-robin to this many groups of CTAs (launch_paper_collide)
    const double* mass2;      // [Nx][4] thermal masses^2 (Eq. 8-9)
    const PaperChannel* table;
    const PaperGroup* groups;
    int n_groups, n_channels;
    int S, Np, Ns;
    int x_begin, x_count, p_begin, p_count;
    uint32_t seed, step, x_rng_offset;
    double Kp, g4, mD2;       // Kp = (dt/hbarc) L^5 / (Ns (2 pi)^5 16) / 8;  mD2 > 0: fixed regulator, else m_g^2(x)
    int has_ovr;
    int all_massless;         // the host knows every stored thermal mass is 0 (never set): one tuple, factorised channel algebra
    double msq_ovr[7];
    double dbg_msq[4];        // debug launch: the mass tuple whose roots are written out
    unsigned mask;            // bz_is.cu: active species ids
    int slot[7];              // bz_is.cu: species id -> layout index (or -1)
};

struct TransportParams {
    const double* f;      // old f
    double* dN_aos;       // collision deposits [Nx][Np][SP] (number units), reset to 0 when consumed
    double* out;          // f_new or dF
    double* f_aos_out;    // mode 1: the new f once more, cell-major [Nx][Np][SP] (the next step's gather source); unused if SP == 1
    uint32_t* step_ptr;   // modes 1, 2: if not NULL the device step counter is incremented (captured graphs, bz_step_n)
    int SP;
    const double* vx; const double* vy; const double* vz;   // [Np] p/|p| at the cell centre (0 at p = 0)
    int nx, ny, nz, S, Np;
    int x_begin, x_count; // spatial cells [x_begin, x_begin + x_count) are updated (all by default)
    double cfl;           // dt / dx
    double inv_deg[7];    // per layout index a: 1/N_a is NOT used (division kept exact); holds N_a
};

struct bz_ctx_impl {
    bz_grid grid;
    int device;                      // the CUDA device the context was created on; every entry point switches to it
    int S, Nx, Np, Ns;
    int species[7], slot[7];
    unsigned mask;
    double alpha_s, m_D;
    uint32_t seed, step;
    uint32_t xoff;                   // bz_set_slab: Philox spatial counter offset
    int zb, ze;                      // bz_set_slab: own z layers [zb, ze); the others are halo copies
    double msq_ovr[7];               // bz_set_msq_override: constant |M|^2 per kind of Table I, < 0 = Table I
    double* mass2;                   // device [Nx][4]: thermal masses^2 m_g^2, m_u^2, m_d^2, m_s^2 (Eq. 8-9); 0 at start
    bool masses_zero;                // no bz_thermal_masses / bz_set_masses call yet: mass2 is all 0
    double* E_tab;                   // device [Nx][4][Np] energies sqrt(p^2 + m^2), allocated at the first bz_vlasov / scheme >= 1 step
    int* x_nb;                       // device [Nx][6] periodic spatial neighbour offsets (built with E_tab)
    unsigned char* p_wrap;           // device [Np] momentum wrap flags (built with E_tab)
    PaperChannel* paper_table;       // device: channel table of the paper sampler (built at the first bz_collision_paper)
    PaperGroup* paper_groups;        // device
    int paper_n_groups, paper_n_channels;
    int coll_mode;                   // bz_set_collision: 0 CM sampler (hot path), 1 the paper's sampler, 2 importance-sampled t, 3 in-box direction
    double* dF_scratch;              // device n_values, allocated at the first bz_step with coll_mode 1
    double* diag;                    // device [Nx][5], allocated at the first bz_energy_diag
    unsigned long long* sign_counts; // device [15], allocated at the first bz_msq_sign_counts
    int scheme;                      // bz_set_transport: 0 upwind massless (NS), 1 Eq. 15 + masses per step, 2 Eq. 15, masses as set
    cudaStream_t stream;
    size_t n_values;
    double *f, *f_new;               // device, n_values each (API layout [Nx][S][Np])
    double *f_aos, *dN_aos;          // device, Nx*Np*SP each (cell-major staging for the collision kernel)
    int SP;                          // doubles per cell in the staging layout
    unsigned long long* counters;    // device [1]: samples accepted by the collision kernels since the last reset
    unsigned long long generated;    // host: samples generated by the collision kernels since the last reset
    unsigned* work_counter;          // device [2]: work-item counter and finished-CTA counter of the collision kernel (self-resetting)
    bool aos_valid;                  // f_aos holds the current f (written by the Euler kernel; bz_set_f invalidates)
    bool rowsum_valid;               // rowsum / m2 belong to the current f
    int sms;                         // SMs of the device (persistent grid size)
    double *rowsum;                  // device [Nx][S][3]: sum f, sum |p| f, sum f d3p/((2pi)^3 |p|) of the current f
    double *mom;                     // device [2*S*Nx + 2*S + Nx]
    double *absp, *w_invE, *vx, *vy, *vz;   // device [Np] tables
    double *cell_tab;                // device [Np][4]: p1x, p1y, p1z, E1 (built on the device, bit-exact arithmetic)
    // bz_step_n: two consecutive steps (f -> f_new -> f) captured as one CUDA graph on a stream of the library's own
    cudaStream_t gstream;
    // one instantiated graph per buffer parity (slot 0: the pair starts with f in the lower of the two buffers, slot 1: in the
    // upper one), so that calls with an odd n, which alternate the parity, replay instead of re-capturing
    cudaGraphExec_t gexec[2];
    uint32_t* step_dev;              // device: the Philox step word the captured kernels read and advance
    struct GraphKey { double dt; int Ns, coll_mode, zb, ze; uint32_t seed, xoff; double ovr[7]; const double* f; } gkey[2];
    std::string err;
    bool profile;
    std::vector<cudaEvent_t> prof_events[2];
    cudaStream_t copy_in, copy_out;  // bz_step_host: H2D / D2H streams (created at first use)
    std::vector<cudaEvent_t> pipe_events;   // bz_step_host: per chunk h2d-done and transport-done events (created at first use)   // start/stop pairs: [0] collision (pack + collide), [1] stream + Euler
};

#ifdef __CUDACC__
// regulator mass^2 of spatial cell x (S8a.1): m_D^2 if fixed, else Eq. 8 with E_p = |p| from the row sums,
// g^2 sum_a c_a rowsum[x][a][2], c = 6 for the gluon row, 1 for quark rows.  One definition for the collision kernel and
// for bz_moments, so that the m^2 reported is bit for bit the one used.
__device__ __forceinline__ double regulator_m2(const double* __restrict__ rowsum, int x, int S, unsigned glue_slot_mask, double g2, double mD2)
{
    if (mD2 > 0.0) return mD2;
    double acc = 0.0;
    for (int a = 0; a < S; ++a) acc += (((glue_slot_mask >> a) & 1u) ? 6.0 : 1.0) * rowsum[((size_t)x * S + a) * 3 + 2];
    return g2 * acc;
}
#endif

// kernels launched by this library in this process (bz_launch_count); bumped by every launcher below
extern std::atomic<unsigned long long> g_launch_count;

// SMs of the device that is current in the calling thread (cached per device; 148 if the query fails): the grid cap of the
// grid-stride launchers that do not get the context's SM count
int device_sms();

// launchers (each returns the cudaError_t of the launch)
int collide_slots_per_cell(unsigned mask);
void collide_item_geometry(int Np, int Nx, int Ns, int sms, int* units_per_item, int* ppc, int* regions_per_x);
cudaError_t launch_collide(const CollideParams& P, int sms, cudaStream_t st);
cudaError_t launch_cell_table(const GridConst& g, int Np, double* tab, cudaStream_t st);
cudaError_t launch_pack(const double* f, double* f_aos, int Nx, int S, int SP, int Np, cudaStream_t st);
cudaError_t launch_debug_samples(const CollideParams& P, int xcell, int p_begin, int p_end, int* cells, double* stu,
                                 cudaStream_t st);
// dF = dN_aos / N_a (transposed to the API layout), dN_aos = 0
cudaError_t launch_finalize(double* dN_aos, double* dF, int Nx, int S, int SP, int Np, const double* deg, cudaStream_t st);
// mode 0: out = dF_stream;  mode 1: out = (f + dF_stream) + dN/N_a and dN = 0;
// mode 2: out = (f + out) + dN/N_a and dN = 0 (out holds a transport increment computed elsewhere: bz_vlasov.cu)
cudaError_t launch_transport(const TransportParams& P, int mode, cudaStream_t st);
// rowsum[x][a][0..2]
cudaError_t launch_rowsums(const double* f, const double* absp, const double* w_invE, double* rowsum, int rows, int Np,
                           cudaStream_t st);
// mom = per-cell (n, e), totals, m2(x) = regulator_m2
cudaError_t launch_moments(const double* rowsum, double* mom, int Nx, int S, const double* deg, unsigned glue_slot_mask, double g2,
                           double mD2, double d3p_over_2pi3, double d3x, int x_begin, int x_end, cudaStream_t st);

// NEXT rank 2 (bz_vlasov.cu): thermal masses of Eq. 8-9 and the central-difference drift + force of Eq. 15
cudaError_t launch_thermal_masses(const double* f, const double* cell_tab, double* mass2, int Nx, int S, int Np,
                                  unsigned cls_bits, unsigned id_bits, double g2, double w, cudaStream_t st);
cudaError_t launch_energy_diag(const double* f, const double* cell_tab, const double* mass2, double* diag, int Nx, int S, int Np,
                               unsigned cls_bits, unsigned id_bits, double w, cudaStream_t st);
cudaError_t launch_vlasov(const double* f, double* out, int nx, int ny, int nz, int S, int Np, const double* cell_tab,
                          const double* mass2, double* E_tab, const int* x_nb, const unsigned char* p_wrap, int n, double dt,
                          double dx, double dp, unsigned cls_bits, cudaStream_t st);

// reading S8 (bz_diag.cu): counts[0] += accepted samples of spatial cells [x_begin, x_end), counts[1 + 2 kind + crossed] += those
// whose |M|^2 of that kind and ordering is negative
cudaError_t launch_msq_signs(const CollideParams& P, int x_begin, int x_end, unsigned long long* counts, int sms, cudaStream_t st);
// NEXT rank 3 (bz_is.cu): what the weighted samplers draw (sampler 1: importance-sampled t with regulator m2, 2: in-box)
cudaError_t launch_weighted_debug(const PaperParams& P, int sampler, double m2, int* cells, double* stu, double* w, int sms, cudaStream_t st);
// NEXT rank 1 (bz_paper.cu)
void build_paper_channels(const int* species, int S, std::vector<PaperChannel>& table, std::vector<PaperGroup>& groups);
cudaError_t launch_paper_collide(const PaperParams& P, int sms, cudaStream_t st);
cudaError_t launch_paper_debug(const PaperParams& P, int* cells, double* stu, int sms, cudaStream_t st);
// out = (f + out) + dFc (forward Euler with both increments given, the oracle's association)
cudaError_t launch_combine(const double* f, double* out, const double* dFc, size_t n_values, cudaStream_t st);

}  // namespace bz
