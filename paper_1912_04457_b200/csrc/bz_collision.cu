// bz_collision.cu -- sample -> |M|^2 -> bracket -> symmetric deposit (S8a.2-8a.5), as two kernels per chunk of
// spatial cells, coupled through a record buffer in HBM:
//
//   sample_kernel   one warp per "region" (C consecutive p1 cells of one spatial cell), lanes = samples.  Pure ALU:
//                   Philox4x32-10, the boost, the binning.  Light on registers, so 4-6x more warps are resident
//                   than the deposit kernel could afford and the long dependent chains (10 Philox rounds, sqrt,
//                   div) overlap across warps.  About 46 % of the samples keep both outgoing legs in the box; they
//                   are compacted (ballot + prefix) into the region's slice of the record buffer:
//                   (i, j, k, l) cells, s, t and the weight K/(E1 E2) -- 40 bytes per accepted sample.
//   deposit_kernel  one warp per region, always full batches of 32 accepted samples.
//       gather   cp.async (LDGSTS) from the cell-major staging copy f_aos[xcell][pcell][SP] (SP = 8 doubles = 64 B per
//                cell) into shared memory: for one sample the 32 lanes fetch its 4 cells x 8 slots, i.e. 8 sectors per
//                instruction instead of 32 scattered ones, and the next batch's gather is in flight while the current
//                batch is computed (double buffer).
//       compute  each lane takes its own sample: <= 10 |M|^2 values, factorised channel algebra (bz_channels.cuh),
//                4 x S deposits written back to shared memory.
//       scatter  the same 8-lanes-per-cell mapping issues fp64 reductions (RED.E.ADD.F64, no return value) into the
//                cell-major deposit scratch dN_aos, which stays in L2 while its spatial cell is being worked on.
// Measured on B200 (profiles/): a RED (LDG) whose 32 lanes hit 32 different sectors costs 48 (32) cycles of the SM's
// L1TEX path, the 8-lanes-per-cell form 15.7 (8.5) cycles for the same number of lanes.
// The record buffer costs 2 x 40 B x 0.46 = 37 B of HBM traffic per sample, ~10 % of a step at the measured rates.
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

constexpr int kSampleWarps = 8;                  // warps per CTA, sample_kernel
constexpr int kDepositWarps = 8;                 // warps per CTA, deposit_kernel

// doubles per cell in the staging layout: 1 for the pure-glue mask, 8 (half a 128-byte line) otherwise
template <int kMask>
struct MaskTraits {
    static constexpr int SP = kMask == 0x01 ? 1 : 8;
};
// layout index of species id = number of active ids below it
__device__ __forceinline__ int slot_of(unsigned mask, int id) { return __popc(mask & ((1u << id) - 1u)); }

// ------------------------------------------------------------------------------------------------ sampling
__global__ void __launch_bounds__(kSampleWarps * 32) sample_kernel(const CollideParams P, int x_begin)
{
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int region_in_x = blockIdx.x * kSampleWarps + warp;            // region index inside the spatial cell
    if (region_in_x >= P.regions_per_x) return;
    const int xcell = x_begin + blockIdx.y;
    const size_t region = (size_t)blockIdx.y * P.regions_per_x + region_in_x;
    int4* __restrict__ rc = P.rec_cells + region * P.region_cap;
    double* __restrict__ rs = P.rec_s + region * P.region_cap;
    double* __restrict__ rt = P.rec_t + region * P.region_cap;
    double* __restrict__ rw = P.rec_w + region * P.region_cap;
    const int n = P.g.n;
    const int i_begin = region_in_x * P.cells_per_region, i_end = min(i_begin + P.cells_per_region, P.Np);
    int count = 0;
    for (int i = i_begin; i < i_end; ++i) {
        const int ipx = i % n, ipy = (i / n) % n, ipz = i / (n * n);
        const double p1x = cell_centre(P.g, ipx), p1y = cell_centre(P.g, ipy), p1z = cell_centre(P.g, ipz);
        const double E1 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p1x, p1x), __dmul_rn(p1y, p1y)), __dmul_rn(p1z, p1z)));
        for (int base = 0; base < P.Ns; base += 32) {
            const int smp = base + lane;
            Sample sa;
            sa.flag = 0;
            if (smp < P.Ns)
                sa = gen_sample(P.g, P.seed, P.step, (uint32_t)xcell, (uint32_t)i, (uint32_t)smp, p1x, p1y, p1z, E1);
            const unsigned acc = __ballot_sync(0xffffffffu, sa.flag);
            if (sa.flag) {
                const int pos = count + __popc(acc & ((1u << lane) - 1u));
                rc[pos] = make_int4(i, sa.j, sa.k, sa.l);
                rs[pos] = sa.s; rt[pos] = sa.t; rw[pos] = P.K / sa.E1E2;
            }
            count += __popc(acc);
        }
    }
    if (lane == 0) P.rec_count[region] = count;
}

// ------------------------------------------------------------------------------------------------ deposits
template <int kSP>
struct WarpSmem {
    int cell[2][32][4];                          // i, j, k, l of the batch's samples
    double stage[2][32 * (4 * kSP + 1)];         // f in, deposits out; odd stride: conflict-free per-lane access
};

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int kMask>
__global__ void __launch_bounds__(kDepositWarps * 32) deposit_kernel(const CollideParams P, int x_begin)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    constexpr int kStride = 4 * kSP + 1;
    constexpr bool kGlue = kMask < 0 || (kMask & 1);
    constexpr bool kQuark = kMask < 0 || (kMask & 0x7E);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    WarpSmem<kSP>& sm = reinterpret_cast<WarpSmem<kSP>*>(smem_raw)[warp];
    const unsigned mask = kMask >= 0 ? (unsigned)kMask : P.mask;

    const int region_in_x = blockIdx.x * kDepositWarps + warp;
    if (region_in_x >= P.regions_per_x) return;
    const int xcell = x_begin + blockIdx.y;
    const size_t region = (size_t)blockIdx.y * P.regions_per_x + region_in_x;
    const int4* __restrict__ rc = P.rec_cells + region * P.region_cap;
    const double* __restrict__ rs = P.rec_s + region * P.region_cap;
    const double* __restrict__ rt = P.rec_t + region * P.region_cap;
    const double* __restrict__ rw = P.rec_w + region * P.region_cap;
    const double* __restrict__ f_cell = P.f_aos + (size_t)xcell * P.Np * kSP;
    double* __restrict__ dN_cell = P.dN_aos + (size_t)xcell * P.Np * kSP;
    const double m2 = P.m2[xcell];
    const int count = P.rec_count[region];
    const int nb = (count + 31) >> 5;
    if (nb == 0) return;

    // issue the gather of batch b into buffer b & 1; returns this lane's (s, t, w)
    auto prefetch = [&](int b, double& s, double& t, double& w) {
        const int e = b * 32 + lane, nvalid = min(32, count - b * 32), buf = b & 1;
        int4 c = make_int4(0, 0, 0, 0);
        s = 1.0; t = -0.5; w = 0.0;
        if (lane < nvalid) { c = rc[e]; s = rs[e]; t = rt[e]; w = rw[e]; }
        *reinterpret_cast<int4*>(&sm.cell[buf][lane][0]) = c;
        __syncwarp();
#pragma unroll 8
        for (int m = 0; m < 4 * kSP; ++m) {
            const int q = m * 32 + lane;
            const int ee = q / (4 * kSP), rem = q % (4 * kSP), cc = rem / kSP, sl = rem % kSP;
            if (ee < nvalid) cp_async8(&sm.stage[buf][ee * kStride + rem], f_cell + (size_t)sm.cell[buf][ee][cc] * kSP + sl);
        }
        cp_async_commit();
    };

    double s, t, w, s_next = 1.0, t_next = -0.5, w_next = 0.0;
    prefetch(0, s, t, w);
    for (int b = 0; b < nb; ++b) {
        const int buf = b & 1, nvalid = min(32, count - b * 32);
        if (b + 1 < nb) {
            prefetch(b + 1, s_next, t_next, w_next);
            cp_async_wait<1>();
        } else {
            cp_async_wait<0>();
        }
        __syncwarp();

        // ---- compute: lane e owns sample e of the batch
        if (lane < nvalid) {
            double* st = sm.stage[buf] + lane * kStride;
            double fi[7], fj[7], fk[7], fl[7];
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                if ((mask >> id) & 1u) {
                    const int sl = slot_of(mask, id);
                    fi[id] = st[sl]; fj[id] = st[kSP + sl]; fk[id] = st[2 * kSP + sl]; fl[id] = st[3 * kSP + sl];
                } else {
                    fi[id] = fj[id] = fk[id] = fl[id] = 0.0;
                }
            }
            const double u = __dsub_rn(-s, t);
            const MsqSet M = msq_set<kGlue, kQuark>(s, t, u, m2, P.g4 * w);
            double dI[7], dJ[7], dK[7], dL[7];
            deposit<kMask>(mask, fi, fj, fk, fl, M, dI, dJ, dK, dL);
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                if ((mask >> id) & 1u) {
                    const int sl = slot_of(mask, id);
                    st[sl] = dI[id]; st[kSP + sl] = dJ[id]; st[2 * kSP + sl] = dK[id]; st[3 * kSP + sl] = dL[id];
                }
            }
        }
        __syncwarp();

        // ---- scatter: 32/kSP cells per instruction, kSP consecutive lanes on the slots of one cell
#pragma unroll 8
        for (int m = 0; m < 4 * kSP; ++m) {
            const int q = m * 32 + lane;
            const int ee = q / (4 * kSP), rem = q % (4 * kSP), cc = rem / kSP, sl = rem % kSP;
            if (ee < nvalid && sl < P.S) {
                const double v = sm.stage[buf][ee * kStride + rem];
                if (v != 0.0) atomicAdd(dN_cell + (size_t)sm.cell[buf][ee][cc] * kSP + sl, v);   // result unused: RED
            }
        }
        __syncwarp();
        s = s_next; t = t_next; w = w_next;
    }
}

__global__ void debug_samples_kernel(const CollideParams P, int xcell, int p_begin, int p_end, int* cells, double* stu)
{
    const long long total = (long long)(p_end - p_begin) * P.Ns;
    const int n = P.g.n;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int i = p_begin + (int)(q / P.Ns), smp = (int)(q % P.Ns);
        const int ipx = i % n, ipy = (i / n) % n, ipz = i / (n * n);
        const double p1x = cell_centre(P.g, ipx), p1y = cell_centre(P.g, ipy), p1z = cell_centre(P.g, ipz);
        const double E1 = __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(p1x, p1x), __dmul_rn(p1y, p1y)), __dmul_rn(p1z, p1z)));
        const Sample sm = gen_sample(P.g, P.seed, P.step, (uint32_t)xcell, (uint32_t)i, (uint32_t)smp, p1x, p1y, p1z, E1);
        cells[4 * q + 0] = sm.j; cells[4 * q + 1] = sm.k; cells[4 * q + 2] = sm.l; cells[4 * q + 3] = sm.flag;
        if (stu) { stu[3 * q + 0] = sm.s; stu[3 * q + 1] = sm.t; stu[3 * q + 2] = sm.u; }
    }
}

// f (species-major, the API layout) -> cell-major staging copy f_aos[x][p][SP]; pad slots are written as 0
__global__ void __launch_bounds__(256) pack_kernel(const double* __restrict__ f, double* __restrict__ f_aos, int S, int SP, int Np)
{
    const int xcell = blockIdx.y;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= Np) return;
    const double* fx = f + (size_t)xcell * S * Np;
    double* o = f_aos + ((size_t)xcell * Np + p) * SP;
    for (int a = 0; a < SP; ++a) o[a] = a < S ? fx[(size_t)a * Np + p] : 0.0;
}

// dF[x][a][p] = dN_aos[x][p][a] / N_a, and the scratch is reset to 0
__global__ void __launch_bounds__(256) finalize_kernel(double* __restrict__ dN_aos, double* __restrict__ dF, int S, int SP, int Np,
                                                        const double d0, const double d1, const double d2, const double d3,
                                                        const double d4, const double d5, const double d6)
{
    const double deg[7] = { d0, d1, d2, d3, d4, d5, d6 };
    const int xcell = blockIdx.y;
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= Np) return;
    double* src = dN_aos + ((size_t)xcell * Np + p) * SP;
    double* dx = dF + (size_t)xcell * S * Np;
    for (int a = 0; a < S; ++a) {
        dx[(size_t)a * Np + p] = src[a] / deg[a];
        src[a] = 0.0;
    }
}

template <int kMask>
cudaError_t launch_deposit(const CollideParams& P, int x_begin, int nxc, cudaStream_t st)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    const size_t smem = sizeof(WarpSmem<kSP>) * kDepositWarps;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(deposit_kernel<kMask>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    dim3 grid((P.regions_per_x + kDepositWarps - 1) / kDepositWarps, nxc), block(kDepositWarps * 32);
    deposit_kernel<kMask><<<grid, block, smem, st>>>(P, x_begin);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace

int collide_slots_per_cell(unsigned mask) { return mask == 0x01u ? 1 : 8; }

// p1 cells per region: long regions amortise the final partial batch, short ones fill the GPU on small grids
int collide_cells_per_region(int Np, int Nx)
{
    const long long total_cells = (long long)Np * Nx;
    const long long c = total_cells / (148LL * 8 * 8);
    return (int)(c < 1 ? 1 : (c > 16 ? 16 : c));
}

cudaError_t launch_collide(const CollideParams& P, cudaStream_t st)
{
    for (int x0 = 0; x0 < P.Nx; x0 += P.x_per_chunk) {
        const int nxc = P.Nx - x0 < P.x_per_chunk ? P.Nx - x0 : P.x_per_chunk;
        dim3 grid((P.regions_per_x + kSampleWarps - 1) / kSampleWarps, nxc), block(kSampleWarps * 32);
        sample_kernel<<<grid, block, 0, st>>>(P, x0);
        ++g_launch_count;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        switch (P.mask) {
        case 0x01u: e = launch_deposit<0x01>(P, x0, nxc, st); break;
        case 0x7Eu: e = launch_deposit<0x7E>(P, x0, nxc, st); break;
        case 0x7Fu: e = launch_deposit<0x7F>(P, x0, nxc, st); break;
        default:    e = launch_deposit<-1>(P, x0, nxc, st); break;
        }
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

cudaError_t launch_debug_samples(const CollideParams& P, int xcell, int p_begin, int p_end, int* cells, double* stu,
                                 cudaStream_t st)
{
    const long long total = (long long)(p_end - p_begin) * P.Ns;
    if (total <= 0) return cudaSuccess;
    const int blocks = (int)((total + 127) / 128 < 148 * 16 ? (total + 127) / 128 : 148 * 16);
    debug_samples_kernel<<<blocks, 128, 0, st>>>(P, xcell, p_begin, p_end, cells, stu);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_pack(const double* f, double* f_aos, int Nx, int S, int SP, int Np, cudaStream_t st)
{
    dim3 grid((Np + 255) / 256, Nx);
    pack_kernel<<<grid, 256, 0, st>>>(f, f_aos, S, SP, Np);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_finalize(double* dN_aos, double* dF, int Nx, int S, int SP, int Np, const double* deg, cudaStream_t st)
{
    dim3 grid((Np + 255) / 256, Nx);
    finalize_kernel<<<grid, 256, 0, st>>>(dN_aos, dF, S, SP, Np, deg[0], deg[1], deg[2], deg[3], deg[4], deg[5], deg[6]);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
