// bz_api.cu -- the C ABI of include/bz.h: context, argument checks, kernel sequencing.  No compute on the host
// except the O(Np) cell-centre tables built once in bz_create.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <vector>

#include "bz_channels.cuh"
#include "bz_internal.h"

using namespace bz;

struct bz_ctx : public bz_ctx_impl {};

namespace bz {
std::atomic<unsigned long long> g_launch_count{0};

int device_sms()
{
    static std::atomic<int> cache[64];
    int dev = 0, n = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return 148;
    n = cache[dev].load(std::memory_order_relaxed);
    if (n > 0) return n;
    if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n < 1) return 148;
    cache[dev].store(n, std::memory_order_relaxed);
    return n;
}
}

namespace {

int fail_cuda(bz_ctx* c, cudaError_t e, const char* where)
{
    c->err = std::string(where) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? -3 : -2;
}
#define BZ_CUDA(call, where)                                  \
    do {                                                      \
        cudaError_t e_ = (call);                              \
        if (e_ != cudaSuccess) return fail_cuda(c, e_, where); \
    } while (0)

// Every entry point runs on the device the context was created on, whatever device is current in the calling thread
// (the previous one is restored on return).  A failing cudaSetDevice leaves a sticky error the next CUDA call reports.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev)
    {
        int cur = -1;
        if (dev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != dev && cudaSetDevice(dev) == cudaSuccess) prev = cur;
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
#define BZ_ON_DEVICE(c) DeviceGuard device_guard_((c)->device)

double degeneracy(int id) { return id == 0 ? 16.0 : 6.0; }   // N_g = 2 x 8, N_q = 2 x 3

void fill_deg(const bz_ctx* c, double (&deg)[7])
{
    for (int a = 0; a < 7; ++a) deg[a] = a < c->S ? degeneracy(c->species[a]) : 1.0;
}

GridConst grid_const(const bz_ctx* c)
{
    GridConst g;
    g.n = c->grid.np;
    g.pmin = c->grid.pmin;
    g.L = c->grid.pmax - c->grid.pmin;
    g.dp = g.L / g.n;
    // fast path of the binning (bz_sample.cuh): 2^k q with k <= 20 chosen so that 2^k |q| < 2^31 for every reachable
    // momentum component, |p| <= E1 + E2 <= 2 sqrt(3) max(|pmin|, |pmax|)
    const double pm = std::fmax(std::fabs(c->grid.pmin), std::fabs(c->grid.pmax));
    const double qmax = (2.0 * std::sqrt(3.0) * pm + std::fabs(g.pmin)) / g.dp + 2.0;
    int k = 20;
    while (k > 0 && std::ldexp(qmax, k) >= 1073741824.0) --k;
    if (k >= 6) {
        g.bin_shift = k;
        g.bin_a = std::ldexp(1.0 / g.dp, k);
        g.bin_b = -g.pmin * g.bin_a;
    } else {                        // degenerate box far from the origin: every sample takes the exact binning
        g.bin_shift = 4; g.bin_a = 0.0; g.bin_b = 0.0;
    }
    return g;
}

CollideParams collide_params(const bz_ctx* c, double dt_fm, unsigned step)
{
    CollideParams P;
    P.g = grid_const(c);
    P.f_aos = c->SP == 1 ? c->f : c->f_aos;    // one species: the API layout is already cell-major
    P.dN_aos = c->dN_aos; P.rowsum = c->rowsum; P.cell_tab = c->cell_tab; P.counters = c->counters;
    P.g2 = 4.0 * kPi * c->alpha_s; P.mD2 = c->m_D > 0.0 ? c->m_D * c->m_D : 0.0; P.glue_slot_mask = (c->mask & 1u) ? 1u : 0u;   // the gluon, if active, is layout index 0
    collide_item_geometry(c->Np, c->Nx, c->Ns, c->sms, &P.units_per_item, &P.ppc, &P.regions_per_x);
    P.work_counter = c->work_counter; P.step_ptr = nullptr;
    const int layer = c->grid.nx * c->grid.ny;              // only the slab's own z layers collide (bz_set_slab)
    P.n_items = (unsigned)((c->ze - c->zb) * layer) * (unsigned)P.regions_per_x; P.x_begin = c->zb * layer;
    P.x_rng_offset = c->xoff;
    P.S = c->S; P.Np = c->Np; P.Nx = c->Nx; P.Ns = c->Ns;
    P.seed = c->seed; P.step = step;
    const double Vp = (P.g.L * P.g.L) * P.g.L, dtG = dt_fm / kHbarc;
    const double K = dtG * Vp / (2048.0 * (kPi * kPi * kPi * kPi) * c->Ns);
    const double g2 = 4.0 * kPi * c->alpha_s;
    P.g4K = (g2 * g2) * K;
    P.mask = c->mask;
    for (int a = 0; a < 7; ++a) P.slot[a] = c->slot[a];
    P.sampler = 0;
    P.has_ovr = 0;
    for (int k = 0; k < 7; ++k) {
        P.msq_ovr[k] = c->msq_ovr[k] >= 0.0 ? c->msq_ovr[k] / (g2 * g2) : -1.0;
        if (c->msq_ovr[k] >= 0.0) P.has_ovr = 1;
    }
    return P;
}

// CUDA events around a group of launches while profiling is on
int prof_mark(bz_ctx* c, int group)
{
    if (!c->profile) return 0;
    cudaEvent_t e = nullptr;
    BZ_CUDA(cudaEventCreate(&e), "event");
    BZ_CUDA(cudaEventRecord(e, c->stream), "event record");
    c->prof_events[group].push_back(e);
    return 0;
}

// sampler: 0 the hot path's isotropic CM direction, 1 importance-sampled t, 2 in-box direction (collide_kernel's template)
int run_collide(bz_ctx* c, double dt_fm, unsigned step, int sampler = 0)
{
    if (int rc = prof_mark(c, 0)) return rc;
    if (c->SP != 1 && !c->aos_valid) {
        BZ_CUDA(launch_pack(c->f, c->f_aos, c->Nx, c->S, c->SP, c->Np, c->stream), "pack");
        c->aos_valid = true;
    }
    if ((long long)c->Np * ((c->Ns + 31) / 32) >= (1LL << 31)) { c->err = "collision: momentum cells x ceil(samples / 32) must stay below 2^31"; return -1; }
    CollideParams P = collide_params(c, dt_fm, step);
    P.sampler = sampler;
    BZ_CUDA(launch_collide(P, c->sms, c->stream), "collide");
    c->generated += (unsigned long long)(P.n_items / (unsigned)P.regions_per_x) * (unsigned long long)c->Np * (unsigned long long)c->Ns;
    return prof_mark(c, 0);
}

// row sums of the current f: the regulator mass^2 of S8a.1 and the moments of S8a.8 are functions of them (regulator_m2)
int update_m2(bz_ctx* c)
{
    if (c->rowsum_valid) return 0;
    BZ_CUDA(launch_rowsums(c->f, c->absp, c->w_invE, c->rowsum, c->Nx * c->S, c->Np, c->stream), "rowsums");
    c->rowsum_valid = true;
    return 0;
}

// species layout index -> mass class (0 = g, 1 + flavour) and species id, 3 bits each
void class_bits(const bz_ctx* c, unsigned& cls, unsigned& ids)
{
    cls = 0; ids = 0;
    for (int a = 0; a < c->S; ++a) {
        const int id = c->species[a];
        cls |= (unsigned)(id == 0 ? 0 : 1 + (id - 1) / 2) << (3 * a);
        ids |= (unsigned)id << (3 * a);
    }
}

int run_thermal_masses(bz_ctx* c)
{
    unsigned cls, ids;
    class_bits(c, cls, ids);
    const double L = c->grid.pmax - c->grid.pmin, dp = L / c->grid.np, d3p = (dp * dp) * dp;
    const double twopi3 = (2.0 * kPi) * (2.0 * kPi) * (2.0 * kPi);
    c->masses_zero = false;
    BZ_CUDA(launch_thermal_masses(c->f, c->cell_tab, c->mass2, c->Nx, c->S, c->Np, cls, ids, 4.0 * kPi * c->alpha_s,
                                  d3p / twopi3, c->stream), "thermal masses");
    return 0;
}

}  // namespace

extern "C" {

static int create_impl(const bz_grid* g, const int* species, int n_species, double alpha_s, double m_D, bz_ctx** out)
{
    if (out) *out = nullptr;
    if (!g || !species || !out || n_species < 1 || n_species > 7) return -1;
    if (g->nx < 1 || g->ny < 1 || g->nz < 1 || g->np < 2 || g->np > 1024 || !(g->pmax > g->pmin) || !(g->dx > 0.0) ||
        !(alpha_s > 0.0))
        return -1;
    for (int a = 0; a < n_species; ++a) {
        if (species[a] < 0 || species[a] > 6) return -1;
        if (a > 0 && species[a] <= species[a - 1]) return -1;
    }
    int ndev = 0;
    bz_ctx* c = new (std::nothrow) bz_ctx();
    if (!c) return -3;
    *out = c;                                   // returned even on failure so that bz_last_error can be read
    c->grid = *g; c->S = n_species; c->Nx = g->nx * g->ny * g->nz; c->Np = g->np * g->np * g->np; c->Ns = 64;
    c->mask = 0;
    for (int a = 0; a < 7; ++a) c->slot[a] = -1;
    for (int a = 0; a < n_species; ++a) { c->species[a] = species[a]; c->slot[species[a]] = a; c->mask |= 1u << species[a]; }
    c->device = -1;
    c->alpha_s = alpha_s; c->m_D = m_D; c->seed = 0; c->step = 0; c->stream = nullptr; c->profile = false; c->copy_in = nullptr; c->copy_out = nullptr;
    c->xoff = 0u; c->zb = 0; c->ze = g->nz;
    for (int k = 0; k < 7; ++k) c->msq_ovr[k] = -1.0;
    c->mass2 = nullptr; c->masses_zero = true; c->coll_mode = 0; c->dF_scratch = nullptr; c->paper_table = nullptr; c->paper_groups = nullptr; c->paper_n_groups = 0; c->paper_n_channels = 0;
    c->E_tab = nullptr; c->x_nb = nullptr; c->p_wrap = nullptr; c->scheme = 0; c->diag = nullptr; c->sign_counts = nullptr;
    c->aos_valid = false; c->rowsum_valid = false;
    c->gstream = nullptr; c->gexec[0] = c->gexec[1] = nullptr; c->step_dev = nullptr; std::memset(c->gkey, 0, sizeof c->gkey);
    c->work_counter = nullptr; c->counters = nullptr; c->generated = 0ull; c->sms = 1;
    c->n_values = (size_t)c->Nx * c->S * c->Np;
    c->f = c->f_new = c->f_aos = c->dN_aos = c->rowsum = c->mom = c->absp = c->w_invE = c->vx = c->vy = c->vz = c->cell_tab = nullptr;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        c->err = "bz_create: no CUDA device (this library has no CPU path)";
        return -2;
    }
    {
        int dev = 0;
        BZ_CUDA(cudaGetDevice(&dev), "cudaGetDevice");
        c->device = dev;                            // the context lives on the device that is current now
        BZ_CUDA(cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev), "SM count");
        if ((long long)c->Nx * c->Np >= (1LL << 32)) { c->err = "bz_create: more than 2^32 (xcell, pcell) pairs"; return -1; }
    }
    const size_t bytes = c->n_values * sizeof(double);
    BZ_CUDA(cudaMalloc(&c->counters, sizeof(unsigned long long)), "cudaMalloc sample counter");
    BZ_CUDA(cudaMemset(c->counters, 0, sizeof(unsigned long long)), "memset sample counter");
    BZ_CUDA(cudaMalloc(&c->work_counter, 2 * sizeof(unsigned)), "cudaMalloc work counter");
    BZ_CUDA(cudaMemset(c->work_counter, 0, 2 * sizeof(unsigned)), "memset work counter");
    BZ_CUDA(cudaMalloc(&c->f, bytes), "cudaMalloc f");
    BZ_CUDA(cudaMalloc(&c->f_new, bytes), "cudaMalloc f_new");
    c->SP = collide_slots_per_cell(c->mask);
    const size_t aos_bytes = (size_t)c->Nx * c->Np * c->SP * sizeof(double);
    BZ_CUDA(cudaMalloc(&c->f_aos, aos_bytes), "cudaMalloc f_aos");
    BZ_CUDA(cudaMalloc(&c->dN_aos, aos_bytes), "cudaMalloc dN_aos");
    BZ_CUDA(cudaMalloc(&c->mass2, (size_t)c->Nx * 4 * sizeof(double)), "cudaMalloc mass2");
    BZ_CUDA(cudaMemset(c->mass2, 0, (size_t)c->Nx * 4 * sizeof(double)), "memset mass2");
    BZ_CUDA(cudaMalloc(&c->rowsum, (size_t)c->Nx * c->S * 3 * sizeof(double)), "cudaMalloc rowsum");
    BZ_CUDA(cudaMalloc(&c->mom, ((size_t)2 * c->S * c->Nx + 2 * c->S + c->Nx) * sizeof(double)), "cudaMalloc mom");
    BZ_CUDA(cudaMalloc(&c->absp, 5 * (size_t)c->Np * sizeof(double)), "cudaMalloc tables");
    c->w_invE = c->absp + c->Np; c->vx = c->w_invE + c->Np; c->vy = c->vx + c->Np; c->vz = c->vy + c->Np;
    BZ_CUDA(cudaMalloc(&c->cell_tab, 4 * (size_t)c->Np * sizeof(double)), "cudaMalloc cell table");
    BZ_CUDA(launch_cell_table(grid_const(c), c->Np, c->cell_tab, nullptr), "cell table");
    BZ_CUDA(cudaMemset(c->f, 0, bytes), "memset f");
    BZ_CUDA(cudaMemset(c->f_new, 0, bytes), "memset f_new");
    BZ_CUDA(cudaMemset(c->dN_aos, 0, aos_bytes), "memset dN_aos");
    // cell-centre tables: |p|, d3p/((2pi)^3 |p|) (0 at p = 0, S10), p/|p| (0 at p = 0)
    {
        const int n = g->np;
        const double L = g->pmax - g->pmin, dp = L / n, d3p = (dp * dp) * dp;
        const double twopi3 = (2.0 * kPi) * (2.0 * kPi) * (2.0 * kPi);
        std::vector<double> tab(5 * (size_t)c->Np);
        for (int pc = 0; pc < c->Np; ++pc) {
            const double px = g->pmin + ((pc % n) + 0.5) * dp, py = g->pmin + (((pc / n) % n) + 0.5) * dp,
                         pz = g->pmin + ((pc / (n * n)) + 0.5) * dp;
            const double E = std::sqrt((px * px + py * py) + pz * pz);
            tab[pc] = E;
            tab[(size_t)c->Np + pc] = E > 0.0 ? d3p / (twopi3 * E) : 0.0;
            tab[2 * (size_t)c->Np + pc] = E > 0.0 ? px / E : 0.0;
            tab[3 * (size_t)c->Np + pc] = E > 0.0 ? py / E : 0.0;
            tab[4 * (size_t)c->Np + pc] = E > 0.0 ? pz / E : 0.0;
        }
        BZ_CUDA(cudaMemcpy(c->absp, tab.data(), tab.size() * sizeof(double), cudaMemcpyHostToDevice), "upload tables");
    }
    return 0;
}

int bz_create(const bz_grid* g, const int* species, int n_species, double alpha_s, double m_D, bz_ctx** out)
{
    const int rc = create_impl(g, species, n_species, alpha_s, m_D, out);
    if (rc != 0 && out && *out && (*out)->f) {       // half-built: every entry point but bz_last_error / bz_destroy answers -4
        cudaFree((*out)->f);
        (*out)->f = nullptr;
    }
    return rc;
}

int bz_destroy(bz_ctx* c)
{
    if (!c) return -1;
    BZ_ON_DEVICE(c);
    cudaFree(c->f); cudaFree(c->f_new); cudaFree(c->f_aos); cudaFree(c->dN_aos); cudaFree(c->work_counter); cudaFree(c->counters); cudaFree(c->rowsum); cudaFree(c->mom);
    cudaFree(c->absp); cudaFree(c->cell_tab); cudaFree(c->mass2); cudaFree(c->E_tab); cudaFree(c->x_nb); cudaFree(c->p_wrap); cudaFree(c->dF_scratch); cudaFree(c->paper_table); cudaFree(c->paper_groups); cudaFree(c->diag); cudaFree(c->sign_counts);
    for (cudaGraphExec_t ge : c->gexec) if (ge) cudaGraphExecDestroy(ge);
    if (c->gstream) cudaStreamDestroy(c->gstream);
    cudaFree(c->step_dev);
    for (auto& v : c->prof_events) for (cudaEvent_t e : v) cudaEventDestroy(e);
    for (cudaEvent_t e : c->pipe_events) cudaEventDestroy(e);
    if (c->copy_in) cudaStreamDestroy(c->copy_in);
    if (c->copy_out) cudaStreamDestroy(c->copy_out);
    delete c;
    return 0;
}

int bz_set_stream(bz_ctx* c, void* s) { if (!c) return -1; c->stream = (cudaStream_t)s; return 0; }
int bz_set_seed(bz_ctx* c, unsigned long long seed) { if (!c) return -1; c->seed = (uint32_t)seed; return 0; }
int bz_set_samples(bz_ctx* c, int n) { if (!c || n < 1 || n > (1 << 24)) return -1; c->Ns = n; return 0; }
int bz_set_step(bz_ctx* c, unsigned step) { if (!c) return -1; c->step = step; return 0; }

int bz_set_msq_override(bz_ctx* c, int kind, double value)
{
    if (!c || kind < 0 || kind > 6 || value != value) return -1;
    c->msq_ovr[kind] = value;
    return 0;
}

int bz_set_slab(bz_ctx* c, unsigned xcell_offset, int z_begin, int z_end)
{
    if (!c || z_begin < 0 || z_end > c->grid.nz || z_begin > z_end) return -1;
    // the cell-major copy of f is only kept up to date for the own layers (bz_copy_layers): a new range starts afresh
    if (z_begin != c->zb || z_end != c->ze) c->aos_valid = false;
    c->xoff = xcell_offset; c->zb = z_begin; c->ze = z_end;
    return 0;
}

int bz_copy_layers(bz_ctx* c, int z0, int n_layers, double* buf_dev, int to_ctx)
{
    if (!c || !buf_dev || z0 < 0 || n_layers < 0 || z0 + n_layers > c->grid.nz) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    const size_t layer = (size_t)c->grid.nx * c->grid.ny * c->S * c->Np;      // doubles per z layer, contiguous in f
    double* p = c->f + (size_t)z0 * layer;
    if (n_layers == 0) return 0;
    BZ_CUDA(cudaMemcpyAsync(to_ctx ? p : buf_dev, to_ctx ? buf_dev : p, (size_t)n_layers * layer * sizeof(double),
                            cudaMemcpyDeviceToDevice, c->stream), "bz_copy_layers");
    if (to_ctx) {
        // halo layers never collide: the collision kernel's cell-major copy only has to follow the slab's own layers
        if (z0 < c->ze && z0 + n_layers > c->zb) c->aos_valid = false;
        c->rowsum_valid = false;
    }
    return 0;
}
const char* bz_last_error(const bz_ctx* c) { return c ? c->err.c_str() : "null context"; }

int bz_set_f(bz_ctx* c, const double* f, int on_device)
{
    if (!c || !f) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    BZ_CUDA(cudaMemcpyAsync(c->f, f, c->n_values * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                            c->stream), "bz_set_f copy");
    c->aos_valid = false; c->rowsum_valid = false;
    if (!on_device) BZ_CUDA(cudaStreamSynchronize(c->stream), "bz_set_f sync");
    return 0;
}

int bz_get_f(bz_ctx* c, double* f, int on_device)
{
    if (!c || !f) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    BZ_CUDA(cudaMemcpyAsync(f, c->f, c->n_values * sizeof(double), on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                            c->stream), "bz_get_f copy");
    if (!on_device) BZ_CUDA(cudaStreamSynchronize(c->stream), "bz_get_f sync");
    return 0;
}

int bz_collision(bz_ctx* c, double dt_fm, unsigned step, double* dF_dev)
{
    if (!c || !dF_dev) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    if (int rc = update_m2(c)) return rc;
    if (int rc = run_collide(c, dt_fm, step)) return rc;
    double deg[7];
    fill_deg(c, deg);
    BZ_CUDA(launch_finalize(c->dN_aos, dF_dev, c->Nx, c->S, c->SP, c->Np, deg, c->stream), "finalize");
    return 0;
}

static TransportParams transport_params(const bz_ctx* c, double dt_fm, double* out)
{
    TransportParams T;
    T.f = c->f; T.dN_aos = c->dN_aos; T.SP = c->SP; T.out = out; T.f_aos_out = c->f_aos; T.vx = c->vx; T.vy = c->vy; T.vz = c->vz;
    T.nx = c->grid.nx; T.ny = c->grid.ny; T.nz = c->grid.nz; T.S = c->S; T.Np = c->Np;
    T.x_begin = 0; T.x_count = c->Nx;
    T.cfl = dt_fm / c->grid.dx;
    T.step_ptr = nullptr;
    fill_deg(c, T.inv_deg);
    return T;
}

int bz_stream(bz_ctx* c, double dt_fm, double* dF_dev)
{
    if (!c || !dF_dev) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    BZ_CUDA(launch_transport(transport_params(c, dt_fm, dF_dev), 0, c->stream), "stream");
    return 0;
}

static int run_vlasov(bz_ctx* c, double dt_fm, double* out)
{
    unsigned cls, ids;
    class_bits(c, cls, ids);
    const double dp = (c->grid.pmax - c->grid.pmin) / c->grid.np;
    if (!c->E_tab) {
        // first use: the energy table and the two periodic-wrap tables of the stencil (index bookkeeping only)
        BZ_CUDA(cudaMalloc(&c->E_tab, (size_t)c->Nx * 4 * c->Np * sizeof(double)), "cudaMalloc E_tab");
        BZ_CUDA(cudaMalloc(&c->x_nb, (size_t)c->Nx * 6 * sizeof(int)), "cudaMalloc x_nb");
        BZ_CUDA(cudaMalloc(&c->p_wrap, (size_t)c->Np), "cudaMalloc p_wrap");
        const int nx = c->grid.nx, ny = c->grid.ny, nz = c->grid.nz, n = c->grid.np;
        std::vector<int> nb((size_t)c->Nx * 6);
        for (int x = 0; x < c->Nx; ++x) {
            const int ix = x % nx, iy = (x / nx) % ny, iz = x / (nx * ny);
            nb[6 * (size_t)x + 0] = (ix + nx - 1) % nx - ix;               nb[6 * (size_t)x + 1] = (ix + 1) % nx - ix;
            nb[6 * (size_t)x + 2] = ((iy + ny - 1) % ny - iy) * nx;        nb[6 * (size_t)x + 3] = ((iy + 1) % ny - iy) * nx;
            nb[6 * (size_t)x + 4] = ((iz + nz - 1) % nz - iz) * nx * ny;   nb[6 * (size_t)x + 5] = ((iz + 1) % nz - iz) * nx * ny;
        }
        std::vector<unsigned char> pw((size_t)c->Np);
        for (int pc = 0; pc < c->Np; ++pc) {
            const int q[3] = { pc % n, (pc / n) % n, pc / (n * n) };
            unsigned w = 0;
            for (int d = 0; d < 3; ++d) w |= (q[d] == 0 ? 1u : 0u) << (2 * d) | (q[d] == n - 1 ? 1u : 0u) << (2 * d + 1);
            pw[pc] = (unsigned char)w;
        }
        BZ_CUDA(cudaMemcpyAsync(c->x_nb, nb.data(), nb.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream), "upload x_nb");
        BZ_CUDA(cudaMemcpyAsync(c->p_wrap, pw.data(), pw.size(), cudaMemcpyHostToDevice, c->stream), "upload p_wrap");
        BZ_CUDA(cudaStreamSynchronize(c->stream), "table sync");
    }
    BZ_CUDA(launch_vlasov(c->f, out, c->grid.nx, c->grid.ny, c->grid.nz, c->S, c->Np, c->cell_tab, c->mass2, c->E_tab,
                          c->x_nb, c->p_wrap, c->grid.np, dt_fm, c->grid.dx, dp, cls, c->stream), "vlasov");
    return 0;
}

int bz_set_transport(bz_ctx* c, int scheme) { if (!c || scheme < 0 || scheme > 2) return -1; c->scheme = scheme; return 0; }

int bz_set_masses(bz_ctx* c, const double* mass2_host)
{
    if (!c || !mass2_host) return -1;
    if (!c->f || !c->mass2) return -4;
    BZ_ON_DEVICE(c);
    c->masses_zero = false;
    BZ_CUDA(cudaMemcpyAsync(c->mass2, mass2_host, (size_t)c->Nx * 4 * sizeof(double), cudaMemcpyHostToDevice, c->stream), "set masses");
    BZ_CUDA(cudaStreamSynchronize(c->stream), "set masses sync");
    return 0;
}

int bz_thermal_masses(bz_ctx* c, double* out_host)
{
    if (!c) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    if (int rc = run_thermal_masses(c)) return rc;
    if (out_host) {
        BZ_CUDA(cudaMemcpyAsync(out_host, c->mass2, (size_t)c->Nx * 4 * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "masses copy");
        BZ_CUDA(cudaStreamSynchronize(c->stream), "masses sync");
    }
    return 0;
}

int bz_energy_diag(bz_ctx* c, double* out_host)
{
    if (!c || !out_host) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    unsigned cls, ids;
    class_bits(c, cls, ids);
    const double L = c->grid.pmax - c->grid.pmin, dp = L / c->grid.np, d3p = (dp * dp) * dp;
    const double twopi3 = (2.0 * kPi) * (2.0 * kPi) * (2.0 * kPi);
    if (!c->diag) BZ_CUDA(cudaMalloc(&c->diag, (size_t)c->Nx * 5 * sizeof(double)), "cudaMalloc diag");   // kept with the context
    BZ_CUDA(launch_energy_diag(c->f, c->cell_tab, c->mass2, c->diag, c->Nx, c->S, c->Np, cls, ids, d3p / twopi3, c->stream), "energy diag");
    BZ_CUDA(cudaMemcpyAsync(out_host, c->diag, (size_t)c->Nx * 5 * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "diag copy");
    BZ_CUDA(cudaStreamSynchronize(c->stream), "diag sync");
    return 0;
}

int bz_vlasov(bz_ctx* c, double dt_fm, double* dF_dev)
{
    if (!c || !dF_dev) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    return run_vlasov(c, dt_fm, dF_dev);
}

int bz_set_collision(bz_ctx* c, int mode) { if (!c || mode < 0 || mode > 3) return -1; c->coll_mode = mode; return 0; }

// bz_step with the paper's own collision term (rank 1): masses (scheme 1), bz_collision_paper into a scratch, the
// transport increment of the chosen scheme into f_new, then f_new = (f + dF_transport) + dF_coll
static int step_paper(bz_ctx* c, double dt_fm)
{
    if (c->scheme == 1) { if (int rc = run_thermal_masses(c)) return rc; }     // masses from the old f, used by both terms
    if (!c->dF_scratch) BZ_CUDA(cudaMalloc(&c->dF_scratch, c->n_values * sizeof(double)), "cudaMalloc dF scratch");
    if (int rc = bz_collision_paper(c, dt_fm, c->step, c->dF_scratch)) return rc;
    if (c->scheme == 0) BZ_CUDA(launch_transport(transport_params(c, dt_fm, c->f_new), 0, c->stream), "stream");
    else if (int rc = run_vlasov(c, dt_fm, c->f_new)) return rc;
    BZ_CUDA(launch_combine(c->f, c->f_new, c->dF_scratch, c->n_values, c->stream), "combine");
    double* t = c->f; c->f = c->f_new; c->f_new = t;
    c->rowsum_valid = false; c->aos_valid = false;
    c->step += 1;
    return 0;
}

int bz_step(bz_ctx* c, double dt_fm)
{
    if (!c) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    if (c->coll_mode == 1) return step_paper(c, dt_fm);
    if (int rc = update_m2(c)) return rc;
    if (int rc = run_collide(c, dt_fm, c->step, c->coll_mode == 0 ? 0 : c->coll_mode - 1)) return rc;   // modes 2, 3: the weighted samplers
    if (c->scheme == 1) { if (int rc = run_thermal_masses(c)) return rc; }     // masses from the old f
    if (int rc = prof_mark(c, 1)) return rc;
    if (c->scheme == 0) BZ_CUDA(launch_transport(transport_params(c, dt_fm, c->f_new), 1, c->stream), "stream+euler");
    else {
        if (int rc = run_vlasov(c, dt_fm, c->f_new)) return rc;
        BZ_CUDA(launch_transport(transport_params(c, dt_fm, c->f_new), 2, c->stream), "euler");
    }
    if (int rc = prof_mark(c, 1)) return rc;
    double* t = c->f; c->f = c->f_new; c->f_new = t;
    c->rowsum_valid = false;          // f changed; f_aos was rewritten with the new f by the Euler kernel
    c->step += 1;
    return 0;
}


// field by field: the struct has padding, which an assignment need not copy
static bool same_graph_key(const bz_ctx::GraphKey& a, const bz_ctx::GraphKey& b)
{
    if (!(a.dt == b.dt) || a.Ns != b.Ns || a.coll_mode != b.coll_mode || a.zb != b.zb || a.ze != b.ze || a.seed != b.seed ||
        a.xoff != b.xoff || a.f != b.f)
        return false;
    for (int k = 0; k < 7; ++k) if (!(a.ovr[k] == b.ovr[k])) return false;
    return true;
}

/* n steps without returning to the host in between: see include/bz.h */
int bz_step_n(bz_ctx* c, double dt_fm, int n)
{
    if (!c || n < 0) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    // Eq. 15 transport and the paper's sampler keep per-step host logic (mass updates, scratch buffers): plain loop
    const bool graphable = c->scheme == 0 && c->coll_mode != 1 && !c->profile;
    int done = 0;
    // the first step (and one more if an odd number is left) goes the ordinary way: it also configures the kernels and
    // brings the cell-major copy and the row-sum bookkeeping into the state the captured steps start from
    while (done < n && (!graphable || done == 0 || ((n - done) & 1))) {
        if (int rc = bz_step(c, dt_fm)) return rc;
        ++done;
    }
    if (done == n) return 0;
    const int pairs = (n - done) / 2;
    if (!c->gstream) BZ_CUDA(cudaStreamCreateWithFlags(&c->gstream, cudaStreamNonBlocking), "graph stream");
    if (!c->step_dev) BZ_CUDA(cudaMalloc(&c->step_dev, sizeof(uint32_t)), "cudaMalloc step word");
    bz_ctx::GraphKey key;
    key.dt = dt_fm; key.Ns = c->Ns; key.coll_mode = c->coll_mode; key.zb = c->zb; key.ze = c->ze; key.seed = c->seed; key.xoff = c->xoff;
    for (int k = 0; k < 7; ++k) key.ovr[k] = c->msq_ovr[k];
    key.f = c->f;
    const int slot = c->f < c->f_new ? 0 : 1;             // buffer parity of the pair's first step
    cudaGraphExec_t& gexec = c->gexec[slot];
    if (!gexec || !same_graph_key(key, c->gkey[slot])) {
        if (gexec) { cudaGraphExecDestroy(gexec); gexec = nullptr; }
        cudaGraph_t graph = nullptr;
        unsigned long long captured = 0ull;               // the launchers count what they enqueue; nothing runs during capture
        BZ_CUDA(cudaStreamBeginCapture(c->gstream, cudaStreamCaptureModeThreadLocal), "begin capture");
        cudaError_t e = cudaSuccess;
        double* fa = c->f;
        double* fb = c->f_new;
        for (int half = 0; half < 2 && e == cudaSuccess; ++half) {
            e = launch_rowsums(fa, c->absp, c->w_invE, c->rowsum, c->Nx * c->S, c->Np, c->gstream);
            ++captured;
            if (e != cudaSuccess) break;
            CollideParams P = collide_params(c, dt_fm, 0u);
            P.step_ptr = c->step_dev;
            P.sampler = c->coll_mode == 0 ? 0 : c->coll_mode - 1;
            if (c->SP == 1) P.f_aos = fa;                      // one species: f itself is the gather source
            e = launch_collide(P, c->sms, c->gstream);
            ++captured;
            if (e != cudaSuccess) break;
            TransportParams T = transport_params(c, dt_fm, fb);
            T.f = fa; T.step_ptr = c->step_dev;
            e = launch_transport(T, 1, c->gstream);
            ++captured;
            std::swap(fa, fb);
        }
        cudaError_t e2 = cudaStreamEndCapture(c->gstream, &graph);
        g_launch_count -= captured;
        if (e == cudaSuccess) e = e2;
        if (e == cudaSuccess) e = cudaGraphInstantiate(&gexec, graph, 0);
        if (graph) cudaGraphDestroy(graph);
        if (e != cudaSuccess) { gexec = nullptr; return fail_cuda(c, e, "bz_step_n: graph capture"); }
        c->gkey[slot] = key;
    }
    // order: whatever the context's stream has queued -> the graph launches -> the context's stream again
    cudaEvent_t ev = nullptr;
    BZ_CUDA(cudaEventCreateWithFlags(&ev, cudaEventDisableTiming), "event");
    cudaError_t e = cudaEventRecord(ev, c->stream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->gstream, ev, 0);
    const uint32_t step0 = c->step;
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->step_dev, &step0, sizeof step0, cudaMemcpyHostToDevice, c->gstream);
    for (int q = 0; q < pairs && e == cudaSuccess; ++q) e = cudaGraphLaunch(gexec, c->gstream);
    if (e == cudaSuccess) e = cudaEventRecord(ev, c->gstream);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(c->stream, ev, 0);
    cudaEventDestroy(ev);
    if (e != cudaSuccess) return fail_cuda(c, e, "bz_step_n: graph launch");
    c->step += 2u * (unsigned)pairs;
    g_launch_count += 6ull * (unsigned long long)pairs;
    c->generated += 2ull * (unsigned long long)pairs * (unsigned long long)((c->ze - c->zb) * c->grid.nx * c->grid.ny) * (unsigned long long)c->Np * (unsigned long long)c->Ns;
    c->rowsum_valid = false;          // the row sums on the device belong to the f before the last step
    c->aos_valid = true;
    return 0;
}

/* Pipelined end-to-end step: see include/bz.h.  Chunks of z layers flow H2D -> (row sums, m^2, cell-major copy,
 * collision) -> stream + Euler -> D2H on three streams; the collision term of a chunk needs only that chunk's f
 * (Eq. 5 is local in x), the upwind stencil of chunk k needs the old f of chunks k - 1 and k + 1 as well. */
int bz_step_host(bz_ctx* c, double dt_fm, const double* f_in_host, double* f_out_host)
{
    if (!c || !f_in_host || !f_out_host) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    const int nzl = c->grid.nz, layer_cells = c->grid.nx * c->grid.ny;
    const int lpc = (nzl + 15) / 16;                             // z layers per chunk: at most 16 chunks
    const int K = (nzl + lpc - 1) / lpc;
    const bool slab = c->zb != 0 || c->ze != nzl;
    if (slab && (c->scheme != 0 || c->coll_mode != 0)) { c->err = "bz_step_host: a slab context needs transport scheme 0 and collision mode 0"; return -4; }
    if (!slab && (c->scheme != 0 || c->coll_mode != 0 || K < 3)) {                    // nothing to overlap (or Eq. 15 transport): the plain sequence
        if (int rc = bz_set_f(c, f_in_host, 0)) return rc;
        if (int rc = bz_step(c, dt_fm)) return rc;
        return bz_get_f(c, f_out_host, 0);
    }
    if (!c->copy_in) {
        BZ_CUDA(cudaStreamCreateWithFlags(&c->copy_in, cudaStreamNonBlocking), "copy stream");
        BZ_CUDA(cudaStreamCreateWithFlags(&c->copy_out, cudaStreamNonBlocking), "copy stream");
    }
    // Pieces: a chunk is lpc whole z layers; the first and the last chunk are cut into four pieces of cells, so that the first
    // collision waits for a quarter of a chunk's upload and only a quarter of a chunk's download is left after the last one.
    struct Piece { int chunk, x0, nx; };
    std::vector<Piece> pieces;
    auto x0_of = [&](int k) { return k * lpc * layer_cells; };
    auto nx_of = [&](int k) { return (std::min(nzl, (k + 1) * lpc) - k * lpc) * layer_cells; };
    for (int k = 0; k < K; ++k) {
        // (only where a quarter is still a few milliseconds of collisions: every launch of the persistent kernel has a ramp and a tail)
        const int n = nx_of(k);
        const bool big = (double)n * (double)c->Np * (double)c->Ns >= 1e8;
        const int nsub = ((k == 0 || k == K - 1) && n % 4 == 0 && big) ? 4 : 1;
        for (int q = 0; q < nsub; ++q) pieces.push_back({ k, x0_of(k) + q * (n / nsub), n / nsub });
    }
    const int NP = (int)pieces.size();
    while ((int)c->pipe_events.size() < 2 * NP + 1) {
        cudaEvent_t e = nullptr;
        BZ_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming), "pipe event");
        c->pipe_events.push_back(e);
    }
    cudaEvent_t* h2d_done = c->pipe_events.data();               // [NP]
    cudaEvent_t* tr_done = c->pipe_events.data() + NP;           // [NP]
    cudaEvent_t start = c->pipe_events[2 * NP];
    const size_t cell_vals = (size_t)c->S * c->Np;               // doubles per spatial cell
    // the copy streams start after whatever the context's stream has queued so far
    BZ_CUDA(cudaEventRecord(start, c->stream), "record");
    BZ_CUDA(cudaStreamWaitEvent(c->copy_in, start, 0), "wait");
    BZ_CUDA(cudaStreamWaitEvent(c->copy_out, start, 0), "wait");
    // own cells of a piece (bz_set_slab: halo layers are refreshed on the device by the caller, they are neither read from
    // nor written to the host buffers, and they do not collide)
    const int own_b = c->zb * layer_cells, own_e = c->ze * layer_cells;
    auto own_x0 = [&](const Piece& p) { return std::max(own_b, p.x0); };
    auto own_nx = [&](const Piece& p) { return std::max(0, std::min(own_e, p.x0 + p.nx) - std::max(own_b, p.x0)); };
    // uploads: chunk 0, then chunk K - 1 (the domain is periodic in z: chunk 0's drift stencil needs it), then 1 ... K - 2
    for (int pass = 0; pass < 3; ++pass)
        for (int q = 0; q < NP; ++q) {
            const Piece& p = pieces[q];
            const int cls = p.chunk == 0 ? 0 : (p.chunk == K - 1 ? 1 : 2);
            if (cls != pass) continue;
            const size_t off = (size_t)own_x0(p) * cell_vals, cnt = (size_t)own_nx(p) * cell_vals;
            if (cnt) BZ_CUDA(cudaMemcpyAsync(c->f + off, f_in_host + off, cnt * sizeof(double), cudaMemcpyHostToDevice, c->copy_in), "h2d");
            BZ_CUDA(cudaEventRecord(h2d_done[q], c->copy_in), "record");
        }
    auto transport_piece = [&](int q) -> int {
        const Piece& p = pieces[q];
        if (int rc = prof_mark(c, 1)) return rc;
        TransportParams T = transport_params(c, dt_fm, c->f_new);
        T.x_begin = p.x0; T.x_count = p.nx;
        BZ_CUDA(launch_transport(T, 1, c->stream), "stream+euler");
        if (int rc = prof_mark(c, 1)) return rc;
        BZ_CUDA(cudaEventRecord(tr_done[q], c->stream), "record");
        BZ_CUDA(cudaStreamWaitEvent(c->copy_out, tr_done[q], 0), "wait");
        const size_t off = (size_t)own_x0(p) * cell_vals, cnt = (size_t)own_nx(p) * cell_vals;
        if (cnt) BZ_CUDA(cudaMemcpyAsync(f_out_host + off, c->f_new + off, cnt * sizeof(double), cudaMemcpyDeviceToHost, c->copy_out), "d2h");
        return 0;
    };
    for (int q = 0; q < NP; ++q) {
        const Piece& p = pieces[q];
        BZ_CUDA(cudaStreamWaitEvent(c->stream, h2d_done[q], 0), "wait");
        // With the first piece of chunk k here (k >= 1; the uploads are in order and chunk K - 1 came second), every piece of
        // chunk k - 1 is collided and has both z neighbours' old f on the device: they go out now, under the collisions to come.
        // (Measured on config 4: the three chunk downloads that used to follow the last collision were 11 of the 17 ms an
        // end-to-end step lost.)
        if (p.chunk >= 1 && pieces[q - 1].chunk != p.chunk) {
            BZ_CUDA(cudaStreamWaitEvent(c->stream, h2d_done[NP - 1], 0), "wait");     // the last piece of chunk K - 1 (k = 1: chunk 0 wraps around)
            for (int r = 0; r < q; ++r) if (pieces[r].chunk == p.chunk - 1) { if (int rc = transport_piece(r)) return rc; }
        }
        BZ_CUDA(launch_rowsums(c->f + (size_t)p.x0 * cell_vals, c->absp, c->w_invE, c->rowsum + (size_t)p.x0 * c->S * 3, p.nx * c->S, c->Np,
                               c->stream), "rowsums");
        if (c->SP != 1)
            BZ_CUDA(launch_pack(c->f + (size_t)p.x0 * cell_vals, c->f_aos + (size_t)p.x0 * c->Np * c->SP, p.nx, c->S, c->SP, c->Np,
                                c->stream), "pack");
        if (own_nx(p) > 0) {                                     // collision of the piece's own cells
            CollideParams P = collide_params(c, dt_fm, c->step);
            P.x_begin = own_x0(p);
            P.n_items = (unsigned)own_nx(p) * (unsigned)P.regions_per_x;
            if (int rc = prof_mark(c, 0)) return rc;
            BZ_CUDA(launch_collide(P, c->sms, c->stream), "collide");
            if (int rc = prof_mark(c, 0)) return rc;
            c->generated += (unsigned long long)own_nx(p) * (unsigned long long)c->Np * (unsigned long long)c->Ns;
        }
        // the pieces of the last chunk have had their neighbours (chunks K - 2 and 0) for a long time: out at once
        if (p.chunk == K - 1) { if (int rc = transport_piece(q)) return rc; }
    }
    double* t = c->f; c->f = c->f_new; c->f_new = t;
    c->aos_valid = true; c->rowsum_valid = false;
    c->step += 1;
    BZ_CUDA(cudaStreamSynchronize(c->copy_out), "d2h sync");
    BZ_CUDA(cudaStreamSynchronize(c->stream), "sync");
    return 0;
}

/* ---- NEXT rank 1: the paper's own sampler (bz_paper.cu) ---- */
static int paper_params(bz_ctx* c, double dt_fm, unsigned step, PaperParams& P)
{
    if (!c->paper_table) {
        std::vector<PaperChannel> table;
        std::vector<PaperGroup> groups;
        build_paper_channels(c->species, c->S, table, groups);
        BZ_CUDA(cudaMalloc(&c->paper_table, table.size() * sizeof(PaperChannel)), "cudaMalloc channel table");
        BZ_CUDA(cudaMalloc(&c->paper_groups, groups.size() * sizeof(PaperGroup)), "cudaMalloc channel groups");
        BZ_CUDA(cudaMemcpy(c->paper_table, table.data(), table.size() * sizeof(PaperChannel), cudaMemcpyHostToDevice), "upload table");
        BZ_CUDA(cudaMemcpy(c->paper_groups, groups.data(), groups.size() * sizeof(PaperGroup), cudaMemcpyHostToDevice), "upload groups");
        c->paper_n_groups = (int)groups.size(); c->paper_n_channels = (int)table.size();
    }
    P.g = grid_const(c);
    P.f = c->SP == 1 ? c->f : c->f_aos; P.dN = c->dN_aos; P.SP = c->SP; P.mass2 = c->mass2; P.table = c->paper_table; P.groups = c->paper_groups;
    P.n_groups = c->paper_n_groups; P.n_channels = c->paper_n_channels; P.S = c->S; P.Np = c->Np; P.Ns = c->Ns;
    const int layer = c->grid.nx * c->grid.ny;
    P.x_begin = c->zb * layer; P.x_count = (c->ze - c->zb) * layer; P.p_begin = 0; P.p_count = c->Np;
    P.seed = c->seed; P.step = step; P.x_rng_offset = c->xoff;
    const double L = P.g.L, twopi = 2.0 * kPi, twopi5 = ((twopi * twopi) * (twopi * twopi)) * twopi;
    P.Kp = (dt_fm / kHbarc) * ((L * L) * (L * L) * L) / ((double)c->Ns * twopi5 * 16.0) * 0.125;
    const double g2 = 4.0 * kPi * c->alpha_s;
    P.g4 = g2 * g2;
    P.mD2 = c->m_D > 0.0 ? c->m_D * c->m_D : 0.0;
    P.all_massless = c->masses_zero ? 1 : 0;
    P.has_ovr = 0;
    for (int k = 0; k < 7; ++k) {
        P.msq_ovr[k] = c->msq_ovr[k] >= 0.0 ? c->msq_ovr[k] / P.g4 : -1.0;
        if (c->msq_ovr[k] >= 0.0) P.has_ovr = 1;
    }
    for (int k = 0; k < 4; ++k) P.dbg_msq[k] = 0.0;
    P.mask = c->mask;
    for (int a = 0; a < 7; ++a) P.slot[a] = c->slot[a];
    return 0;
}

int bz_collision_paper(bz_ctx* c, double dt_fm, unsigned step, double* dF_dev)
{
    if (!c || !dF_dev) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    // gathers from the cell-major copy of f and deposits into the cell-major scratch, like the hot path (run_collide)
    if (c->SP != 1 && !c->aos_valid) {
        BZ_CUDA(launch_pack(c->f, c->f_aos, c->Nx, c->S, c->SP, c->Np, c->stream), "pack");
        c->aos_valid = true;
    }
    PaperParams P;
    if (int rc = paper_params(c, dt_fm, step, P)) return rc;
    BZ_CUDA(launch_paper_collide(P, c->sms, c->stream), "paper collide");
    double deg[7];
    fill_deg(c, deg);
    BZ_CUDA(launch_finalize(c->dN_aos, dF_dev, c->Nx, c->S, c->SP, c->Np, deg, c->stream), "finalize");   // dF = dN / N_a, scratch back to 0
    return 0;
}

int bz_debug_paper_samples(bz_ctx* c, unsigned step, int xcell, int pcell_begin, int pcell_end, const double* msq_host,
                           int* cells_dev, double* stu_dev)
{
    if (!c || !msq_host || !cells_dev || !stu_dev || xcell < 0 || xcell >= c->Nx || pcell_begin < 0 || pcell_end > c->Np ||
        pcell_begin > pcell_end)
        return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    PaperParams P;
    if (int rc = paper_params(c, 1.0, step, P)) return rc;
    P.x_begin = xcell; P.x_count = 1; P.p_begin = pcell_begin; P.p_count = pcell_end - pcell_begin;
    for (int k = 0; k < 4; ++k) P.dbg_msq[k] = msq_host[k];
    BZ_CUDA(launch_paper_debug(P, cells_dev, stu_dev, c->sms, c->stream), "paper debug");
    return 0;
}

int bz_debug_paper_channels(const int* species, int n_species, int* out_host, int capacity)
{
    if (!species || n_species < 1 || n_species > 7 || (capacity > 0 && !out_host)) return -1;
    for (int a = 0; a < n_species; ++a)
        if (species[a] < 0 || species[a] > 6 || (a > 0 && species[a] <= species[a - 1])) return -1;
    std::vector<PaperChannel> table;
    std::vector<PaperGroup> groups;
    build_paper_channels(species, n_species, table, groups);
    for (size_t q = 0; q < table.size() && (int)q < capacity; ++q) {
        int* o = out_host + 7 * q;
        o[0] = table[q].a; o[1] = table[q].b; o[2] = table[q].c; o[3] = table[q].d; o[4] = table[q].kind; o[5] = table[q].crossed;
        o[6] = table[q].key;
    }
    return (int)table.size();
}

/* ---- NEXT rank 3: the weighted samplers (importance-sampled t, in-box direction) run in collide_kernel ---- */
static int collision_weighted(bz_ctx* c, double dt_fm, unsigned step, double* dF_dev, int sampler)
{
    if (!c || !dF_dev) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    if (int rc = update_m2(c)) return rc;
    if (int rc = run_collide(c, dt_fm, step, sampler)) return rc;
    double deg[7];
    fill_deg(c, deg);
    BZ_CUDA(launch_finalize(c->dN_aos, dF_dev, c->Nx, c->S, c->SP, c->Np, deg, c->stream), "finalize");
    return 0;
}

int bz_collision_is(bz_ctx* c, double dt_fm, unsigned step, double* dF_dev) { return collision_weighted(c, dt_fm, step, dF_dev, 1); }
int bz_collision_box(bz_ctx* c, double dt_fm, unsigned step, double* dF_dev) { return collision_weighted(c, dt_fm, step, dF_dev, 2); }

static int debug_weighted(bz_ctx* c, unsigned step, int xcell, int pcell_begin, int pcell_end, int sampler, double m2, int* cells_dev,
                          double* stu_dev, double* w_dev)
{
    if (!c || !cells_dev || !stu_dev || !w_dev || xcell < 0 || xcell >= c->Nx || pcell_begin < 0 || pcell_end > c->Np ||
        pcell_begin > pcell_end)
        return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    PaperParams P;
    if (int rc = paper_params(c, 1.0, step, P)) return rc;
    P.x_begin = xcell; P.x_count = 1; P.p_begin = pcell_begin; P.p_count = pcell_end - pcell_begin;
    BZ_CUDA(launch_weighted_debug(P, sampler, m2, cells_dev, stu_dev, w_dev, c->sms, c->stream), "weighted sampler debug");
    return 0;
}

int bz_debug_samples_is(bz_ctx* c, unsigned step, int xcell, int pcell_begin, int pcell_end, double m2, int* cells_dev,
                        double* stu_dev, double* w_dev)
{
    return debug_weighted(c, step, xcell, pcell_begin, pcell_end, 1, m2, cells_dev, stu_dev, w_dev);
}

int bz_debug_samples_box(bz_ctx* c, unsigned step, int xcell, int pcell_begin, int pcell_end, int* cells_dev, double* stu_dev,
                         double* w_dev)
{
    return debug_weighted(c, step, xcell, pcell_begin, pcell_end, 2, 0.0, cells_dev, stu_dev, w_dev);
}

int bz_moments(bz_ctx* c, double* out_host)
{
    if (!c || !out_host) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    if (int rc = update_m2(c)) return rc;
    double deg[7];
    fill_deg(c, deg);
    const double L = c->grid.pmax - c->grid.pmin, dp = L / c->grid.np, d3p = (dp * dp) * dp;
    const double twopi3 = (2.0 * kPi) * (2.0 * kPi) * (2.0 * kPi);
    const double d3x = ((c->grid.dx * c->grid.dx) * c->grid.dx) / ((kHbarc * kHbarc) * kHbarc);
    BZ_CUDA(launch_moments(c->rowsum, c->mom, c->Nx, c->S, deg, (c->mask & 1u) ? 1u : 0u, 4.0 * kPi * c->alpha_s,
                           c->m_D > 0.0 ? c->m_D * c->m_D : 0.0, d3p / twopi3, d3x,
                           c->zb * c->grid.nx * c->grid.ny, c->ze * c->grid.nx * c->grid.ny, c->stream), "moments");
    const size_t cnt = (size_t)2 * c->S * c->Nx + 2 * c->S + c->Nx;
    BZ_CUDA(cudaMemcpyAsync(out_host, c->mom, cnt * sizeof(double), cudaMemcpyDeviceToHost, c->stream), "moments copy");
    BZ_CUDA(cudaStreamSynchronize(c->stream), "moments sync");
    return 0;
}

int bz_set_profile(bz_ctx* c, int on) { if (!c) return -1; c->profile = on != 0; return 0; }

int bz_get_profile(bz_ctx* c, int group, double* ms_total, int* launches)
{
    if (!c || !ms_total || !launches || group < 0 || group > 1) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    BZ_CUDA(cudaStreamSynchronize(c->stream), "profile sync");
    std::vector<cudaEvent_t>& ev = c->prof_events[group];
    double tot = 0.0;
    for (size_t q = 0; q + 1 < ev.size(); q += 2) {
        float ms = 0.f;
        BZ_CUDA(cudaEventElapsedTime(&ms, ev[q], ev[q + 1]), "event elapsed");
        tot += ms;
    }
    *ms_total = tot;
    *launches = (int)(ev.size() / 2);
    for (cudaEvent_t e : ev) cudaEventDestroy(e);
    ev.clear();
    return 0;
}

unsigned long long bz_launch_count(void) { return g_launch_count.load(); }

int bz_get_sample_counts(bz_ctx* c, unsigned long long* generated_out, unsigned long long* accepted_out, int reset)
{
    if (!c || !generated_out || !accepted_out) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    unsigned long long acc = 0ull;
    BZ_CUDA(cudaMemcpyAsync(&acc, c->counters, sizeof acc, cudaMemcpyDeviceToHost, c->stream), "sample counter copy");
    BZ_CUDA(cudaStreamSynchronize(c->stream), "sample counter sync");
    *generated_out = c->generated; *accepted_out = acc;
    if (reset) {
        BZ_CUDA(cudaMemsetAsync(c->counters, 0, sizeof acc, c->stream), "sample counter reset");
        c->generated = 0ull;
    }
    return 0;
}

int bz_msq_sign_counts(bz_ctx* c, unsigned step, int xcell_begin, int xcell_end, unsigned long long* out_host)
{
    if (!c || !out_host || xcell_begin < 0 || xcell_end > c->Nx || xcell_begin > xcell_end) return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    if (int rc = update_m2(c)) return rc;                // the regulator of every spatial cell for the current f
    if (!c->sign_counts) BZ_CUDA(cudaMalloc(&c->sign_counts, 15 * sizeof(unsigned long long)), "cudaMalloc sign counters");   // kept with the context
    BZ_CUDA(cudaMemsetAsync(c->sign_counts, 0, 15 * sizeof(unsigned long long), c->stream), "sign counters reset");
    BZ_CUDA(launch_msq_signs(collide_params(c, 1.0, step), xcell_begin, xcell_end, c->sign_counts, c->sms, c->stream), "msq signs");
    BZ_CUDA(cudaMemcpyAsync(out_host, c->sign_counts, 15 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, c->stream), "sign counters copy");
    BZ_CUDA(cudaStreamSynchronize(c->stream), "sign counters sync");
    return 0;
}

int bz_debug_samples(bz_ctx* c, unsigned step, int xcell, int pcell_begin, int pcell_end, int* cells_dev, double* stu_dev)
{
    if (!c || !cells_dev || xcell < 0 || xcell >= c->Nx || pcell_begin < 0 || pcell_end > c->Np || pcell_begin > pcell_end)
        return -1;
    if (!c->f) return -4;
    BZ_ON_DEVICE(c);
    BZ_CUDA(launch_debug_samples(collide_params(c, 1.0, step), xcell, pcell_begin, pcell_end, cells_dev, stu_dev, c->stream),
            "debug_samples");
    return 0;
}

}  // extern "C"
