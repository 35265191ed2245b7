// bz_vlasov.cu -- NEXT rank 2 of SURVEY.md 8f: the paper's own left-hand side.
//   mass_kernel    thermal masses^2 per spatial cell, Eq. 8-9, with E_p^a = sqrt(p^2 + m_a^2) from the
//                  masses of the previous evaluation (0 at start = the first-step prescription E_p = |p|)
//   vlasov_class_kernel  dF = -dt { drift + force } of Eq. 15: central differences in x and in p, periodic in both
//                  (P:139).  In bz_step the increment lands in f_new and transport_kernel<2> adds f and the collision
//                  deposits (forward Euler, Eq. 15 solved for f(t + dt)).
//   energy_kernel  E_p^a(x) table for the mass classes present (one square root per entry instead of 18 per value).
#include "bz_internal.h"

namespace bz {

namespace {

// species layout index a -> mass class (0 = g, 1 + flavour for q and qbar) is passed as 3 bits per slot in cls_bits
__device__ __forceinline__ int class_of(unsigned cls_bits, int a) { return (int)((cls_bits >> (3 * a)) & 7u); }

// 1/x to ~1 ulp: the hardware seed and two Newton steps instead of the IEEE division sequence (nothing here decides an index)
__device__ __forceinline__ double rcp_newton(double x)
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    y = fma(y, e, y);
    e = fma(-x, y, 1.0);
    return fma(y, e, y);
}

__global__ void __launch_bounds__(256) mass_kernel(const double* __restrict__ f, const double* __restrict__ cell_tab,
                                                   double* __restrict__ mass2, int S, int Np, unsigned cls_bits,
                                                   unsigned id_bits, double g2, double w /* d3p / (2 pi)^3 */)
{
    const int x = blockIdx.x;
    __shared__ double m_old[4];
    __shared__ double part[7][8];
    if (threadIdx.x < 4) m_old[threadIdx.x] = mass2[4 * (size_t)x + threadIdx.x];
    __syncthreads();
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int a = 0; a < S; ++a) {
        const double m2 = m_old[class_of(cls_bits, a)];
        const double* fa = f + ((size_t)x * S + a) * Np;
        double sum = 0.0;
        for (int pc = threadIdx.x; pc < Np; pc += blockDim.x) {
            const double2 u = __ldg(reinterpret_cast<const double2*>(cell_tab) + 2 * (size_t)pc);
            const double pz = __ldg(cell_tab + 4 * (size_t)pc + 2);
            const double E = sqrt(((u.x * u.x + u.y * u.y) + pz * pz) + m2);
            if (E > 0.0) sum += w * rcp_newton(E) * fa[pc];
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) part[a][warp] = sum;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double I[7] = { 0, 0, 0, 0, 0, 0, 0 };                 // by species id
        for (int a = 0; a < S; ++a) {
            double t = 0.0;
            for (int q = 0; q < 8; ++q) t += part[a][q];
            I[(id_bits >> (3 * a)) & 7u] = t;
        }
        double quarks = 0.0;
        for (int id = 1; id < 7; ++id) quarks += I[id];
        mass2[4 * (size_t)x + 0] = g2 * (6.0 * I[0] + quarks);                                   // Eq. 8
        for (int fl = 0; fl < 3; ++fl)
            mass2[4 * (size_t)x + 1 + fl] = (4.0 / 3.0) * g2 * ((2.0 * I[0] + I[1 + 2 * fl]) + I[2 + 2 * fl]);   // Eq. 9
    }
}

// Energy balance (Eq. 11-12, 26): diag[x][0] = T^00_kin(x), diag[x][1 + c] = Q_c(x) for the mass classes c = g, u, d, s
__global__ void __launch_bounds__(256) diag_kernel(const double* __restrict__ f, const double* __restrict__ cell_tab,
                                                   const double* __restrict__ mass2, double* __restrict__ diag, int S, int Np,
                                                   unsigned cls_bits, unsigned id_bits, double w /* d3p / (2 pi)^3 */)
{
    const int x = blockIdx.x;
    __shared__ double part[2][7][8];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int a = 0; a < S; ++a) {
        const double m2 = mass2[4 * (size_t)x + class_of(cls_bits, a)];
        const double* fa = f + ((size_t)x * S + a) * Np;
        double se = 0.0, sq = 0.0;
        for (int pc = threadIdx.x; pc < Np; pc += blockDim.x) {
            const double2 u = __ldg(reinterpret_cast<const double2*>(cell_tab) + 2 * (size_t)pc);
            const double pz = __ldg(cell_tab + 4 * (size_t)pc + 2);
            const double E = sqrt(((u.x * u.x + u.y * u.y) + pz * pz) + m2), v = fa[pc];
            se += E * v;
            if (E > 0.0) sq += v * rcp_newton(E);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { se += __shfl_xor_sync(0xffffffffu, se, o); sq += __shfl_xor_sync(0xffffffffu, sq, o); }
        if (lane == 0) { part[0][a][warp] = se; part[1][a][warp] = sq; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double out[5] = { 0, 0, 0, 0, 0 };
        for (int a = 0; a < S; ++a) {
            double te = 0.0, tq = 0.0;
            for (int q = 0; q < 8; ++q) { te += part[0][a][q]; tq += part[1][a][q]; }
            const double Na = ((id_bits >> (3 * a)) & 7u) == 0u ? 16.0 : 6.0;      // N_g, N_q
            out[0] += Na * te * w;
            out[1 + class_of(cls_bits, a)] += Na * tq * w;
        }
        for (int k = 0; k < 5; ++k) diag[5 * (size_t)x + k] = out[k];
    }
}

// E_tab[(x*4 + cls)*Np + pc] = sqrt(p^2 + m_cls^2(x)) for the mass classes present: one square root per entry, so
// that the stencil kernel below reads its 18 energies per (cell, class) instead of recomputing them
__global__ void __launch_bounds__(256) energy_kernel(const double* __restrict__ cell_tab, const double* __restrict__ mass2,
                                                     double* __restrict__ E_tab, int Np, unsigned cls_present)
{
    const int x = blockIdx.x;
    for (int pc = blockIdx.y * blockDim.x + threadIdx.x; pc < Np; pc += gridDim.y * blockDim.x) {
        const double a = __ldg(cell_tab + 4 * (size_t)pc), b = __ldg(cell_tab + 4 * (size_t)pc + 1), c = __ldg(cell_tab + 4 * (size_t)pc + 2);
        const double p2 = (a * a + b * b) + c * c;
#pragma unroll
        for (int cls = 0; cls < 4; ++cls)
            if ((cls_present >> cls) & 1u) E_tab[((size_t)x * 4 + cls) * Np + pc] = sqrt(p2 + __ldg(mass2 + 4 * (size_t)x + cls));
    }
}

struct VlasovParams {
    const double* f;              // [Nx][S][Np]
    double* out;                  // dF, same layout
    const double* cell_tab;       // [Np][4] px, py, pz, |p|
    const double* E_tab;          // [Nx][4][Np] energies of the mass classes present (energy_kernel)
    const int* x_nb;              // [Nx][6] cell index offsets of the spatial neighbours (-x, +x, -y, +y, -z, +z), periodic
    const unsigned char* p_wrap;  // [Np] bit 2d: the -e_d momentum neighbour wraps, bit 2d + 1: the +e_d one
    int nx, ny, nz, S, Np, n;     // n = momentum cells per axis
    int chunks_per_block;
    double dt, inv_2dx, inv_2dp;
    unsigned cls_bits;
};

// ---- the stencil kernel bz_vlasov launches -----------------------------------------------------------------------------
// One thread per (spatial cell, mass class, momentum cell); blockIdx.x = spatial cell (fastest): the blocks in flight share
// one (class, 256-cell momentum chunk) slice of all spatial cells, so the six spatial neighbours are L2 hits; a block walks
// chunks_per_block consecutive chunks (about 8 p_z planes) so that the +-n^2 momentum neighbours are still in L2 when they
// are touched again.  The periodic wraps come from two small tables built once per context (x_nb: neighbour cell offsets
// per spatial cell, p_wrap: one flag byte per momentum cell), p_i / E from a Newton reciprocal.
// History (config 4): the round-1 kernel, one thread per value and SPECIES, issued 30 global loads per value (12 of f, 18 of
// the energy table) and sat at 90 % of the L1 data pipe (5.7 ms with the energy table).  Two restructurings were measured
// slower:
// staging every energy and f plane in shared memory, one block per (spatial cell, mass class) sweeping the p_z planes
// (12.1 ms: an 8-byte LDS of a warp costs the same two wavefronts of that pipe as an 8-byte LDG, and the block-wide syncs
// per plane expose the load latency), and one thread per (p_x, p_y) column walking p_z with register windows (15.7 ms: 156
// registers, 8 warps per SM).  What is kept is what needs neither: one thread per value, but the thread serves
// ALL species of its mass class (q and qbar share the 18 energies) and takes the p_x neighbours -- of f and of the energy
// difference E(x + e_x) - E(x - e_x) -- from the neighbouring lanes by warp shuffles (lanes at the ends of a p_x row or of
// the warp load theirs): 14 energy loads per class and 11 f loads per species, 19 per value for the mixture instead of 30
// -- which bought 2 % (5.59 ms): with the L1 pipe relieved the kernel is bound by the L2 -> L1 traffic of its scattered
// 8-byte neighbour loads; the next step would be the plane sweep again, software-pipelined instead of block-synchronous.
__global__ void __launch_bounds__(256) vlasov_class_kernel(const VlasovParams V)
{
    const int xcell = blockIdx.x;
    int cls = -1;                                            // the blockIdx.z-th mass class present
    {
        unsigned present = 0;
        for (int a = 0; a < V.S; ++a) present |= 1u << class_of(V.cls_bits, a);
        int k = blockIdx.z;
        for (int c = 0; c < 4; ++c) if ((present >> c) & 1u) { if (k == 0) { cls = c; break; } --k; }
    }
    if (cls < 0) return;
    int sp[2] = { 0, 0 }, nsp = 0;                           // the species (layout indices) of the class: q and qbar, or g
    for (int a = 0; a < V.S; ++a) if (class_of(V.cls_bits, a) == cls && nsp < 2) sp[nsp++] = a;
    const int lane = threadIdx.x & 31, n = V.n;
    const size_t row = (size_t)V.S * V.Np;
    const int* xnb = V.x_nb + 6 * (size_t)xcell;             // cell index offsets of x -+ dx e_d (periodic)
    const double* Ex = V.E_tab + ((size_t)xcell * 4 + cls) * V.Np;
    for (int ch = 0; ch < V.chunks_per_block; ++ch) {
        const int pc_raw = (blockIdx.y * V.chunks_per_block + ch) * blockDim.x + threadIdx.x;
        if (pc_raw - lane >= V.Np) return;                   // the whole warp is past the end
        const bool on = pc_raw < V.Np;
        const int pc = on ? pc_raw : V.Np - 1;
        const unsigned wrap = V.p_wrap[pc];                  // bit 2d: p - dp e_d wraps, bit 2d + 1: p + dp e_d wraps
        // p_x neighbours from the lanes next door, except at the ends of a p_x row and of the warp
        const bool ld_m = lane == 0 || (wrap & 1u) || !on, ld_p = lane == 31 || (wrap & 2u) || pc_raw + 1 >= V.Np;
        double acc[2] = { 0.0, 0.0 };
        int pstr = 1;
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            const int pom = ((wrap >> (2 * d)) & 1u) ? (n - 1) * pstr : -pstr;       // periodic in p
            const int pop = ((wrap >> (2 * d + 1)) & 1u) ? -(n - 1) * pstr : pstr;
            pstr *= n;
            const double pd = __ldg(V.cell_tab + 4 * (size_t)pc + d);
            const ptrdiff_t om = __ldg(xnb + 2 * d), op = __ldg(xnb + 2 * d + 1);
            const double* Em = Ex + pc + om * 4 * V.Np;      // energies at x - dx e_d
            const double* Ep = Ex + pc + op * 4 * V.Np;      // energies at x + dx e_d
            const double Exp = __ldg(Ep), Exm = __ldg(Em);
            const double cp = Exp > 0.0 ? pd * rcp_newton(Exp) : 0.0, cm = Exm > 0.0 ? pd * rcp_newton(Exm) : 0.0;   // S10
            double Gp, Gm;
            if (d == 0) {
                const double dE = Exp - Exm;
                Gp = __shfl_sync(0xffffffffu, dE, (lane + 1) & 31); Gm = __shfl_sync(0xffffffffu, dE, (lane + 31) & 31);
                if (ld_p) Gp = __ldg(Ep + pop) - __ldg(Em + pop);
                if (ld_m) Gm = __ldg(Ep + pom) - __ldg(Em + pom);
                Gp *= V.inv_2dx; Gm *= V.inv_2dx;
            } else {
                Gp = (__ldg(Ep + pop) - __ldg(Em + pop)) * V.inv_2dx;       // dE/dx at p + dp e_d
                Gm = (__ldg(Ep + pom) - __ldg(Em + pom)) * V.inv_2dx;       // dE/dx at p - dp e_d
            }
#pragma unroll
            for (int s = 0; s < 2; ++s) {
                if (s < nsp) {
                    const double* fx = V.f + (size_t)xcell * row + (size_t)sp[s] * V.Np + pc;
                    const double fxm = __ldg(fx + om * (ptrdiff_t)row), fxp = __ldg(fx + op * (ptrdiff_t)row);
                    double fpm, fpp;
                    if (d == 0) {
                        const double f0 = __ldg(fx);
                        fpp = __shfl_sync(0xffffffffu, f0, (lane + 1) & 31); fpm = __shfl_sync(0xffffffffu, f0, (lane + 31) & 31);
                        if (ld_p) fpp = __ldg(fx + pop);
                        if (ld_m) fpm = __ldg(fx + pom);
                    } else {
                        fpm = __ldg(fx + pom); fpp = __ldg(fx + pop);
                    }
                    const double drift = (cp * fxp - cm * fxm) * V.inv_2dx;
                    const double force = -(fpp * Gp - fpm * Gm) * V.inv_2dp;
                    acc[s] += drift + force;
                }
            }
        }
#pragma unroll
        for (int s = 0; s < 2; ++s)
            if (s < nsp && on) V.out[(size_t)xcell * row + (size_t)sp[s] * V.Np + pc] = -V.dt * acc[s];
    }
}

}  // namespace

cudaError_t launch_thermal_masses(const double* f, const double* cell_tab, double* mass2, int Nx, int S, int Np,
                                  unsigned cls_bits, unsigned id_bits, double g2, double w, cudaStream_t st)
{
    mass_kernel<<<Nx, 256, 0, st>>>(f, cell_tab, mass2, S, Np, cls_bits, id_bits, g2, w);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_energy_diag(const double* f, const double* cell_tab, const double* mass2, double* diag, int Nx, int S, int Np,
                               unsigned cls_bits, unsigned id_bits, double w, cudaStream_t st)
{
    diag_kernel<<<Nx, 256, 0, st>>>(f, cell_tab, mass2, diag, S, Np, cls_bits, id_bits, w);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_vlasov(const double* f, double* out, int nx, int ny, int nz, int S, int Np, const double* cell_tab,
                          const double* mass2, double* E_tab, const int* x_nb, const unsigned char* p_wrap, int n, double dt,
                          double dx, double dp, unsigned cls_bits, cudaStream_t st)
{
    unsigned present = 0;
    for (int a = 0; a < S; ++a) present |= 1u << ((cls_bits >> (3 * a)) & 7u);
    int chunks = (Np + 255) / 256;
    if (chunks > 65535) return cudaErrorInvalidValue;
    energy_kernel<<<dim3(nx * ny * nz, chunks), 256, 0, st>>>(cell_tab, mass2, E_tab, Np, present);
    ++g_launch_count;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    VlasovParams V;
    V.f = f; V.out = out; V.cell_tab = cell_tab; V.E_tab = E_tab; V.x_nb = x_nb; V.p_wrap = p_wrap; V.nx = nx; V.ny = ny; V.nz = nz; V.S = S; V.Np = Np; V.n = n;
    V.dt = dt; V.inv_2dx = 1.0 / (2.0 * dx); V.inv_2dp = 1.0 / (2.0 * dp); V.cls_bits = cls_bits;
    V.chunks_per_block = (8 * n * n + 255) / 256;
    if (V.chunks_per_block > chunks) V.chunks_per_block = chunks;
    const int groups = (chunks + V.chunks_per_block - 1) / V.chunks_per_block;
    int n_cls = 0;
    for (int c = 0; c < 4; ++c) n_cls += (present >> c) & 1u;
    vlasov_class_kernel<<<dim3(nx * ny * nz, groups, n_cls), 256, 0, st>>>(V);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
