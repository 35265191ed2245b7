// bz_collision.cu -- sample -> |M|^2 -> bracket -> symmetric deposit (S8a.2-8a.5) as ONE persistent kernel of 16
// identical warps per SM (one CTA of 512 threads per SM, 128 registers per thread: the whole register file).
//
// Every warp runs the same loop over work items (a run of p1 cells of one spatial cell, pulled from a global counter):
//   sample   lanes = samples: Philox4x32-10, the boost, the binning (bz_sample.cuh).  About 46 % of the samples keep both
//            outgoing legs in the box; they are compacted (ballot + prefix) into the warp's ring of 64 records in shared
//            memory: the four cells as indices into the whole grid (xcell * Np + pcell), s, t, E1 E2, the regulator.
//   gather   as soon as the ring holds 16 records: cp.async (LDGSTS, 16 bytes per lane, L1 bypassed) of the 4 cells x 64
//            bytes of each from the cell-major staging copy f_aos[xcell][pcell][8] into the warp's stage buffer: 4 lanes
//            fetch one cell, one instruction fetches 8 cells.  The warp then runs its next sampling pass; the gather
//            lands underneath it.
//   algebra  TWO lanes per sample: the loss half of every channel's bracket is the gain half of the time-reversed channel
//            (deposit_half, bz_channels.cuh), so lane m evaluates all gain terms of sample m on the cells (i, j | k, l) and
//            lane m + 16 the same code on (k, l | i, j), each with half the registers the whole bracket needs -- which is
//            what lets all 16 warps be identical instead of a few fat "consumer" warps that everything else waits for.
//            Each lane writes its 4 x S deposits back to the stage buffer.
//   scatter  one sample per instruction: lane = (cell, slot), 8 lanes per 64-byte cell add the two halves and issue one
//            fp64 reduction (RED.E.ADD.F64, no return value) into the cell-major scratch dN_aos, which stays in L2 while
//            its spatial cell is being worked on.
// History (config 4, ncu): the first version of this file specialised 16 producer + 4 consumer warps (mbarrier
// hand-off, setmaxnreg 64/224).  Its FP64 pipe was busy 41 % of the cycles and 73 % of the producers' batches had to wait
// for their consumer (160 try_wait iterations each, 18 % of all executed instructions): a consumer warp alone on its SM
// sub-partition ran at 0.16 instructions per cycle.  See profiles/r2_collide_kernel_ncu_baseline.md.
// Pure glue (one species): one double per cell, the API layout is already cell-major; lane = sample, the four gathers
// are plain loads and the four reductions leave straight from the registers.
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

constexpr int kWarps = 16;
constexpr int kCollideThreads = 32 * kWarps;
constexpr int kRing = 64;                        // records per warp (a sampling pass adds at most 32)
constexpr int kRetryCap = 64;                    // per warp: samples whose two Marsaglia attempts both failed
constexpr int kMaxDevices = 64;

// doubles per cell in the global staging layout: 1 for the pure-glue mask, 8 (half a 128-byte line) otherwise
template <int kMask>
struct MaskTraits {
    static constexpr int SP = kMask == 0x01 ? 1 : 8;
};
// layout index of species id = number of active ids below it
__host__ __device__ constexpr int slot_of(unsigned mask, int id)
{
    int n = 0;
    for (int b = 0; b < id; ++b) n += (mask >> b) & 1u;
    return n;
}

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
// No "memory" clobber on cp.async and red: volatile asm statements keep their order among themselves (the gathers stay
// between the previous batch's reductions and the wait_group that precedes every read of the stage buffer), and without
// the clobber the compiler may hoist the shared-memory loads of the NEXT cell index / deposit above them instead of
// serialising load -> use -> load (ncu: the dependent LDS -> IMAD.WIDE pairs were the stall points of gather and scatter).
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
// fp64 reduction without return value (RED.E.ADD.F64)
__device__ __forceinline__ void red_add(double* gdst, double v)
{
    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(gdst), "d"(v));
}

// ------------------------------------------------------------------------------------------------ shared memory
// Per warp.  kSP == 8: the stage buffer holds, per sample of the batch in flight, the occupation numbers of its 4 cells
// on the way in ([0, 32): 4 cells x 8 doubles, overwritten by the forward half's deposits) and the reversed half's
// deposits ([32, 64)); 66 doubles per sample.  Every cell is 16-byte aligned (cp.async 16).  The two halves of a sample
// sit in different half warps (lane and lane + 16), so a quarter warp's eight 16-byte accesses go to eight consecutive
// samples, 33 x 16 bytes apart: eight different bank groups, no conflicts.
template <int kSP>
struct alignas(16) WarpMem {
    static constexpr int kBatch = kSP == 1 ? 32 : 16;    // samples per algebra pass
    static constexpr int kStride = 66, kLoss = 32;
    double stage[kSP == 1 ? 2 : 16 * kStride];
    double p1tab[32][4];                                 // (p1x, p1y, p1z, E1) of the p1 cells of the current work item
    unsigned cell[4][kRing + 4];                         // [slot i, j, k, l][record]: indices into the whole grid, xcell * Np + pcell
                                                         // (rows 272 bytes apart: the four slots' 16-byte reads hit different banks)
    double s[kRing], t[kRing], e12[kRing];               // Mandelstam s, t and E1 E2 of the sample
    double w[kRing];                                     // weight of the sample (weighted samplers only)
    double m2x;                                          // regulator mass^2 of the current spatial cell
    int2 retry[kRetryCap];
};

// momentum and energy of the centre of a p1 cell from the table built by cell_table_kernel (same arithmetic as
// cell_kinematics, done once per context instead of once per warp pass)
__device__ __forceinline__ void cell_lookup(const double* __restrict__ tab, int pcell, double& p1x, double& p1y, double& p1z,
                                            double& E1)
{
    const double2 a = __ldg(reinterpret_cast<const double2*>(tab) + 2 * (size_t)pcell);
    const double2 b = __ldg(reinterpret_cast<const double2*>(tab) + 2 * (size_t)pcell + 1);
    p1x = a.x; p1y = a.y; p1z = b.x; E1 = b.y;
}

// ---- gather: the 4 x 64 bytes of records [head, head + nb) into the stage buffer (kSP == 8).  head is a multiple of 16
// (a batch never wraps around the ring), so the cell indices of a lane's eight samples are two 16-byte loads.
template <int kSP>
__device__ __forceinline__ void issue_gather(WarpMem<kSP>& wm, const double* __restrict__ f_aos, int lane, int head, int nb)
{
    using W = WarpMem<kSP>;
    const int sub = lane >> 4, cc = (lane >> 2) & 3, q = lane & 3;     // lanes 0-15: samples 0-7, lanes 16-31: samples 8-15; 4 lanes per cell
    const double* __restrict__ src = f_aos + q * 2;
    double* dst = wm.stage + sub * 8 * W::kStride + cc * 8 + q * 2;
    const unsigned* cp = &wm.cell[cc][head + sub * 8];
    if (nb == W::kBatch) {
        const uint4 c0 = *reinterpret_cast<const uint4*>(cp), c1 = *reinterpret_cast<const uint4*>(cp + 4);
        const unsigned ci[8] = { c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w };
#pragma unroll
        for (int k = 0; k < 8; ++k) cp_async16(dst + k * W::kStride, src + (size_t)ci[k] * 8);
    } else {
        for (int k = 0; k < 8 && sub * 8 + k < nb; ++k) cp_async16(dst + k * W::kStride, src + (size_t)cp[k] * 8);
    }
    cp_async_commit();
}

// ---- algebra + scatter of records [head, head + nb), kSP == 8: two lanes per sample
template <int kMask, int kSP, int kSampler>
__device__ __forceinline__ void consume_batch(WarpMem<kSP>& wm, const CollideParams& P, int lane, unsigned mask, int head, int nb,
                                              double m2)
{
    using W = WarpMem<kSP>;
    constexpr bool kGlue = kMask < 0 || (kMask & 1);
    constexpr bool kQuark = kMask < 0 || (kMask & 0x7E);
    cp_async_wait_all();
    __syncwarp();                                        // every lane's gathers have landed
    // The loss half of a channel a b -> c d at the cells (i, j | k, l) is the GAIN half of the time-reversed channel
    // c d -> a b at the cells (k, l | i, j): same s, t, u, same |M|^2 (the table is closed under time reversal, S8c step 5),
    // and its deposits -H at (k, l), +H at (i, j) are exactly the loss term's.  So both lanes of a sample run the same gain
    // algebra; the second one just takes the four cells in the order k, l, i, j, on the way in and on the way out.
    const int m = lane & 15;                             // lanes 0-15: the forward halves of samples 0-15, lanes 16-31: the reversed ones
    const int rev = (lane >> 4) * 16;                    // doubles: offset of the lane's "incoming" pair of cells
    double* st = wm.stage + m * W::kStride;
    const double* sin_ = st + rev;                       // incoming legs: cells (i, j) or, reversed, (k, l)
    const double* sout = st + (16 - rev);                // outgoing legs
    double d[4][7];
    const bool work = m < nb;
    if (work) {
        const int r = head + m;
        const double s = wm.s[r], t = wm.t[r];
        double g4w = P.g4K * rcp_fast(wm.e12[r]);                         // g^4 K / (E1 E2), S8c step 6
        if constexpr (kSampler != 0) g4w *= wm.w[r];                      // x the sampler's weight
        // gain factors: P = f at the incoming cells, Q = F = 1 + f (gluon), 1 - f (quark) at the outgoing ones
        double Pi[7], Pj[7], Qk[7], Ql[7];
        if constexpr (kMask >= 0) {
            constexpr unsigned km = (unsigned)kMask;
            constexpr int kPairs = (slot_of(km, 7) + 1) / 2;
            double2 v[4][4];
#pragma unroll
            for (int q = 0; q < kPairs; ++q) {
                v[0][q] = *reinterpret_cast<const double2*>(sin_ + 2 * q); v[1][q] = *reinterpret_cast<const double2*>(sin_ + 8 + 2 * q);
                v[2][q] = *reinterpret_cast<const double2*>(sout + 2 * q); v[3][q] = *reinterpret_cast<const double2*>(sout + 8 + 2 * q);
            }
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                if ((kMask >> id) & 1) {
                    const int a = slot_of(km, id);
                    Pi[id] = (a & 1) ? v[0][a >> 1].y : v[0][a >> 1].x; Pj[id] = (a & 1) ? v[1][a >> 1].y : v[1][a >> 1].x;
                    const double fk = (a & 1) ? v[2][a >> 1].y : v[2][a >> 1].x, fl = (a & 1) ? v[3][a >> 1].y : v[3][a >> 1].x;
                    Qk[id] = id == 0 ? 1.0 + fk : 1.0 - fk; Ql[id] = id == 0 ? 1.0 + fl : 1.0 - fl;
                } else {
                    Pi[id] = Pj[id] = Qk[id] = Ql[id] = 0.0;
                }
            }
        } else {
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                if ((mask >> id) & 1u) {
                    const int a = slot_of(mask, id);
                    Pi[id] = sin_[a]; Pj[id] = sin_[8 + a];
                    const double fk = sout[a], fl = sout[8 + a];
                    Qk[id] = id == 0 ? 1.0 + fk : 1.0 - fk; Ql[id] = id == 0 ? 1.0 + fl : 1.0 - fl;
                } else {
                    Pi[id] = Pj[id] = Qk[id] = Ql[id] = 0.0;
                }
            }
        }
        const double u = __dsub_rn(-s, t);
        MsqSet M = msq_set<kGlue, kQuark>(s, t, u, m2, g4w);
        // user-defined matrix elements (bz_set_msq_override) run on the runtime-mask instantiation, so that the
        // specialised mixture kernels carry no extra registers for them
        if constexpr (kMask < 0) { if (P.has_ovr) msq_apply_override(M, P.msq_ovr, g4w); }
        deposit_half<kMask>(mask, Pi, Pj, Qk, Ql, M, d[0], d[1], d[2], d[3]);
    }
    __syncwarp();                                        // both lanes of every pair have read the gathered f
    if (work) {
        // d[0], d[1] belong to the lane's incoming cells, d[2], d[3] to its outgoing ones: back in the order i, j, k, l
        double* oin = st + (lane >> 4) * W::kLoss + rev;
        double* oout = st + (lane >> 4) * W::kLoss + (16 - rev);
        if constexpr (kMask >= 0) {
            constexpr unsigned km = (unsigned)kMask;
            constexpr int kS = slot_of(km, 7), kPairs = (kS + 1) / 2;
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                double o[8];
#pragma unroll
                for (int a = 0; a < 8; ++a) o[a] = 0.0;
#pragma unroll
                for (int id = 0; id < 7; ++id)
                    if ((kMask >> id) & 1) o[slot_of(km, id)] = d[c][id];
                double* dst = (c < 2 ? oin : oout) + (c & 1) * 8;
#pragma unroll
                for (int q = 0; q < kPairs; ++q)
                    *reinterpret_cast<double2*>(dst + 2 * q) = make_double2(o[2 * q], o[2 * q + 1]);
            }
        } else {
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                double* dst = (c < 2 ? oin : oout) + (c & 1) * 8;
#pragma unroll
                for (int a = 0; a < 8; ++a) dst[a] = 0.0;
#pragma unroll
                for (int id = 0; id < 7; ++id)
                    if ((mask >> id) & 1u) dst[slot_of(mask, id)] = d[c][id];
            }
        }
    }
    __syncwarp();
    // scatter: one sample per instruction, lane = (cell cc, slot sl) of the sample, 8 lanes per 64-byte cell; the cell
    // indices (four 16-byte loads: a batch never wraps around the ring) and the sums of the two halves are collected
    // first, then the reductions go out
    {
        const int cc = lane >> 3, sl = lane & 7;
        if (sl < P.S) {
            double* __restrict__ gdst = P.dN_aos + sl;
            const double* src = wm.stage + lane;
            const unsigned* cp = &wm.cell[cc][head];
            if (nb == W::kBatch) {
#pragma unroll
                for (int q0 = 0; q0 < W::kBatch; q0 += 8) {
                    const uint4 c0 = *reinterpret_cast<const uint4*>(cp + q0), c1 = *reinterpret_cast<const uint4*>(cp + q0 + 4);
                    const unsigned ci[8] = { c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w };
                    double v[8];
#pragma unroll
                    for (int q = 0; q < 8; ++q) v[q] = src[(q0 + q) * W::kStride] + src[(q0 + q) * W::kStride + W::kLoss];
#pragma unroll
                    for (int q = 0; q < 8; ++q) red_add(gdst + (size_t)ci[q] * 8, v[q]);
                }
            } else {
                for (int q = 0; q < nb; ++q) red_add(gdst + (size_t)cp[q] * 8, src[q * W::kStride] + src[q * W::kStride + W::kLoss]);
            }
        }
    }
    __syncwarp();                                        // the stage buffer may be overwritten by the next gather
}

// ---- pure glue: lane = sample, plain loads, the whole bracket in one lane, four reductions from the registers
template <int kSampler>
__device__ __forceinline__ void consume_batch_glue(WarpMem<1>& wm, const CollideParams& P, int lane, int head, int nb, double m2)
{
    if (lane < nb) {
        const int r = head + lane;
        const uint4 cl = make_uint4(wm.cell[0][r], wm.cell[1][r], wm.cell[2][r], wm.cell[3][r]);
        const double s = wm.s[r], t = wm.t[r];
        double g4w = P.g4K * rcp_fast(wm.e12[r]);
        if constexpr (kSampler != 0) g4w *= wm.w[r];
        const double fi = __ldg(P.f_aos + cl.x), fj = __ldg(P.f_aos + cl.y), fk = __ldg(P.f_aos + cl.z), fl = __ldg(P.f_aos + cl.w);
        const double u = __dsub_rn(-s, t);
        MsqSet M = msq_set<true, false>(s, t, u, m2, g4w);
        if (P.has_ovr) msq_apply_override(M, P.msq_ovr, g4w);
        // g g -> g g at (i,j) -> (k,l): the only channel (S8c step 5); the t-family's gluon term counted with X = Z roles
        const double Fi = 1.0 + fi, Fj = 1.0 + fj, Fk = 1.0 + fk, Fl = 1.0 + fl;
        const double T = M.gg * ((fi * Fk) * (fj * Fl) - (Fi * fk) * (Fj * fl));
        red_add(P.dN_aos + cl.x, -T); red_add(P.dN_aos + cl.y, -T);
        red_add(P.dN_aos + cl.z, T); red_add(P.dN_aos + cl.w, T);
    }
}

// ------------------------------------------------------------------------------------------------ the kernel
// kSampler: 0 = isotropic CM direction (the hot path, NS), 1 = importance-sampled t, 2 = in-box direction (bz_sample.cuh)
template <int kMask, int kSampler>
__global__ void __launch_bounds__(kCollideThreads, 1) collide_kernel(const CollideParams P)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    using W = WarpMem<kSP>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // lane and warp through volatile asm: ptxas otherwise re-derives them from S2R SR_TID.X a dozen times per loop iteration
    // (the special-register read is slow and sat on the critical path of gather and scatter)
    int lane, warp;
    asm volatile("mov.u32 %0, %%laneid;" : "=r"(lane));
    asm volatile("{\n .reg .u32 t;\n mov.u32 t, %%tid.x;\n shr.u32 %0, t, 5;\n}" : "=r"(warp));
    W& wm = reinterpret_cast<W*>(smem_raw)[warp];
    const unsigned mask = kMask >= 0 ? (unsigned)kMask : P.mask;
    const uint32_t step = P.step_ptr ? *P.step_ptr : P.step;

    // Loop state, all warp-uniform and deliberately few: whatever lives across the three inlined phases competes with
    // them for the 128 registers (the first version kept the p1 momentum, m^2 and half a dozen flags here; they were
    // spilled to local memory and their reloads were 10 % of the kernel's stall samples).
    int head = 0, count = 0;             // ring: records [head, head + count)
    int nb = 0;                          // > 0: the gather of records [head, head + nb) is in flight
    int rcount = 0;                      // entries in the retry list
    int xcell = -1, i = 0, i0 = 0, base = 0, units_left = 0;   // current item: units_left passes of 32 samples left, the next one
                                                                // starts at sample `base` of p1 cell i of xcell (i0 = the item's first cell)
    unsigned next_item = 0xffffffffu;    // decoded later; 0xffffffff: none fetched yet
    bool exhausted = false;
    unsigned n_acc = 0u;                 // samples accepted by this warp (bz_get_sample_counts)
    unsigned pref_item = 0u;             // lane 0: the item after next_item, fetched while the current one is worked on
    if (lane == 0) pref_item = atomicAdd(P.work_counter, 1u);

    for (;;) {
        // ---- A: fresh work?  An item of ANOTHER spatial cell is only adopted once ring and retry list are empty
        bool fresh = units_left > 0;
        if (!fresh && !exhausted) {
            if (next_item == 0xffffffffu) {
                next_item = __reduce_max_sync(0xffffffffu, lane == 0 ? pref_item : 0u);   // REDUX: the result is provably warp-uniform
                if (next_item >= P.n_items) { exhausted = true; next_item = 0xffffffffu; }
            }
            if (next_item != 0xffffffffu) {
                const int nxt_x = P.x_begin + (int)(next_item / (unsigned)P.regions_per_x);
                if (nxt_x == xcell || (count == 0 && rcount == 0)) {
                    const int region = (int)(next_item % (unsigned)P.regions_per_x);
                    if (nxt_x != xcell) { xcell = nxt_x; if (lane == 0) wm.m2x = regulator_m2(P.rowsum, xcell, P.S, P.glue_slot_mask, P.g2, P.mD2); }
                    // an item is a run of units_per_item passes (32 samples each) through the p1 cells, ppc passes per cell
                    const int u0 = region * P.units_per_item, u1 = min(u0 + P.units_per_item, P.Np * P.ppc);
                    i = i0 = u0 / P.ppc; base = (u0 - i0 * P.ppc) * 32; units_left = u1 - u0;
                    next_item = 0xffffffffu;
                    fresh = units_left > 0;
                    if (lane == 0) pref_item = atomicAdd(P.work_counter, 1u);
                    // the item's p1 cells (at most 32): one coalesced read of the cell table into shared memory
                    if (i0 + lane <= (u1 - 1) / P.ppc) {
                        const double2* src = reinterpret_cast<const double2*>(P.cell_tab) + 2 * (size_t)(i0 + lane);
                        double2* dst = reinterpret_cast<double2*>(&wm.p1tab[lane][0]);
                        dst[0] = __ldg(src); dst[1] = __ldg(src + 1);
                    }
                    __syncwarp();
                }
            }
        }
        // ---- B: a batch is ready and nothing is in flight: start its gather
        if (nb == 0 && (count >= W::kBatch || (!fresh && rcount == 0 && count > 0))) {
            nb = min(count, W::kBatch);
            if constexpr (kSP != 1) issue_gather<kSP>(wm, P.f_aos, lane, head, nb);
        }
        // ---- C: one sampling pass (a full warp of retries if there is one, else fresh samples), covering the gather
        const bool can_sample = (fresh || rcount > 0) && count + 32 <= kRing;
        if (can_sample) {
            int ci, smp;
            unsigned kstart;
            bool active;
            double p1x, p1y, p1z, E1;
            const uint32_t xr = (uint32_t)xcell + P.x_rng_offset;
            [[maybe_unused]] uint32_t w0[4], w1[4], wa[4], wb[4];      // Philox blocks 0, 1, 2 + kstart, 3 + kstart (uniform sampler)
            if (rcount >= 32 || !fresh) {
                const int nr = min(rcount, 32);
                rcount -= nr;
                active = lane < nr;
                const int2 e = active ? wm.retry[rcount + lane] : make_int2(0, 0);
                ci = e.x; smp = e.y & 0x1ffffff; kstart = (unsigned)e.y >> 25;
                cell_lookup(P.cell_tab, ci, p1x, p1y, p1z, E1);           // per lane
                __syncwarp();                                    // the entries are read before new ones are appended
                if constexpr (kSampler == 0) {
                    philox4x32_10(0u, (uint32_t)smp, (uint32_t)ci, xr, P.seed, step, w0);
                    philox4x32_10(1u, (uint32_t)smp, (uint32_t)ci, xr, P.seed, step, w1);
                    philox4x32_10(2u + kstart, (uint32_t)smp, (uint32_t)ci, xr, P.seed, step, wa);
                    philox4x32_10(3u + kstart, (uint32_t)smp, (uint32_t)ci, xr, P.seed, step, wb);
                }
            } else {
                const double2 a = *reinterpret_cast<const double2*>(&wm.p1tab[i - i0][0]), b = *reinterpret_cast<const double2*>(&wm.p1tab[i - i0][2]);
                p1x = a.x; p1y = a.y; p1z = b.x; E1 = b.y;
                ci = i; smp = base + lane; kstart = 0u;
                active = smp < P.Ns;
                // fresh pass: block number, p1 cell and spatial cell are warp-uniform, only the sample index depends on the
                // lane -- 16 of the 20 multiplications of a block are per-lane work, the rest goes to the uniform datapath
                if constexpr (kSampler == 0) {
                    philox4x32_10(0u, (uint32_t)smp, (uint32_t)i, xr, P.seed, step, w0);
                    philox4x32_10(1u, (uint32_t)smp, (uint32_t)i, xr, P.seed, step, w1);
                    philox4x32_10(2u, (uint32_t)smp, (uint32_t)i, xr, P.seed, step, wa);
                    philox4x32_10(3u, (uint32_t)smp, (uint32_t)i, xr, P.seed, step, wb);
                }
                base += 32; --units_left;
                if (base >= P.Ns) { base = 0; ++i; }
            }
            Sample sa;
            sa.flag = 0; sa.retry = 0;
            if (active) {
                if constexpr (kSampler == 0) sa = gen_sample_words(P.g, w0, w1, wa, wb, kstart, p1x, p1y, p1z, E1);
                else if constexpr (kSampler == 1) sa = gen_sample_is_pair(P.g, P.seed, step, xr, (uint32_t)ci, (uint32_t)smp, kstart, p1x, p1y, p1z, E1, wm.m2x);
                else sa = gen_sample_box_pair(P.g, P.seed, step, xr, (uint32_t)ci, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
            }
            const unsigned lt = (1u << lane) - 1u;
            const unsigned rb = __ballot_sync(0xffffffffu, sa.retry);
            if (rb) {
                if (sa.retry) wm.retry[rcount + __popc(rb & lt)] = make_int2(ci, smp | (int)((kstart + 2u) << 25));
                rcount += __popc(rb);
            }
            // compact the accepted samples into the ring
            const unsigned acc = __ballot_sync(0xffffffffu, sa.flag);
            if (sa.flag) {
                const int r = (head + count + __popc(acc & lt)) & (kRing - 1);
                const unsigned xb = (unsigned)xcell * (unsigned)P.Np;
                wm.cell[0][r] = xb + (unsigned)ci; wm.cell[1][r] = xb + (unsigned)sa.j; wm.cell[2][r] = xb + (unsigned)sa.k; wm.cell[3][r] = xb + (unsigned)sa.l;
                wm.s[r] = sa.s; wm.t[r] = sa.t; wm.e12[r] = sa.E1E2;
                if constexpr (kSampler != 0) wm.w[r] = sa.w;
            }
            const int na = __popc(acc);
            count += na;
            n_acc += (unsigned)na;
            __syncwarp();                                    // records and retry entries are visible to all lanes
        }
        // ---- D: the batch in flight: algebra and scatter
        if (nb > 0) {
            if constexpr (kSP == 1) consume_batch_glue<kSampler>(wm, P, lane, head, nb, wm.m2x);
            else consume_batch<kMask, kSP, kSampler>(wm, P, lane, mask, head, nb, wm.m2x);
            count -= nb;
            head = count == 0 ? 0 : (head + nb) & (kRing - 1);   // only the last batch before a drain is partial: head stays a multiple of kBatch
            nb = 0;
        } else if (!can_sample && exhausted && count == 0) {
            break;
        }
    }
    if (lane == 0 && P.counters) atomicAdd(P.counters, (unsigned long long)n_acc);
    // the last CTA to finish resets the work counter for the next launch (also the next replay of a captured graph)
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        const unsigned prev = atomicAdd(P.work_counter + 1, 1u);
        if (prev == gridDim.x - 1) { P.work_counter[0] = 0u; P.work_counter[1] = 0u; }
    }
}

// p1-cell table: (p1x, p1y, p1z, E1) of every momentum cell centre, with the arithmetic of S8c steps 0 and 2
__global__ void cell_table_kernel(const GridConst g, int Np, double* __restrict__ tab)
{
    const int pc = blockIdx.x * blockDim.x + threadIdx.x;
    if (pc >= Np) return;
    double p1x, p1y, p1z, E1;
    cell_kinematics(g, pc, p1x, p1y, p1z, E1);
    tab[4 * (size_t)pc + 0] = p1x; tab[4 * (size_t)pc + 1] = p1y; tab[4 * (size_t)pc + 2] = p1z; tab[4 * (size_t)pc + 3] = E1;
}

__global__ void debug_samples_kernel(const CollideParams P, int xcell, int p_begin, int p_end, int* cells, double* stu)
{
    const long long total = (long long)(p_end - p_begin) * P.Ns;
    for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < total; q += (long long)gridDim.x * blockDim.x) {
        const int i = p_begin + (int)(q / P.Ns), smp = (int)(q % P.Ns);
        double p1x, p1y, p1z, E1;
        cell_kinematics(P.g, i, p1x, p1y, p1z, E1);
        Sample sm;
        unsigned kstart = 0u;
        do {                                                 // the generator of the collision kernel, attempts two at a time
            sm = gen_sample_pair(P.g, P.seed, P.step, (uint32_t)xcell + P.x_rng_offset, (uint32_t)i, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
            kstart += 2u;
        } while (sm.retry);
        cells[4 * q + 0] = sm.j; cells[4 * q + 1] = sm.k; cells[4 * q + 2] = sm.l; cells[4 * q + 3] = sm.flag;
        if (stu) { stu[3 * q + 0] = sm.s; stu[3 * q + 1] = sm.t; stu[3 * q + 2] = sm.u; }
    }
}

// f (species-major, the API layout) -> cell-major staging copy f_aos[x][p][SP]; pad slots are written as 0
__global__ void __launch_bounds__(256) pack_kernel(const double* __restrict__ f, double* __restrict__ f_aos, int S, int SP, int Np)
{
    const int xcell = blockIdx.x;
    const double* fx = f + (size_t)xcell * S * Np;
    for (int p = blockIdx.y * blockDim.x + threadIdx.x; p < Np; p += gridDim.y * blockDim.x) {
        double* o = f_aos + ((size_t)xcell * Np + p) * SP;
        for (int a = 0; a < SP; ++a) o[a] = a < S ? fx[(size_t)a * Np + p] : 0.0;
    }
}

// dF[x][a][p] = dN_aos[x][p][a] / N_a, and the scratch is reset to 0
__global__ void __launch_bounds__(256) finalize_kernel(double* __restrict__ dN_aos, double* __restrict__ dF, int S, int SP, int Np,
                                                        const double d0, const double d1, const double d2, const double d3,
                                                        const double d4, const double d5, const double d6)
{
    const double deg[7] = { d0, d1, d2, d3, d4, d5, d6 };
    const int xcell = blockIdx.x;
    double* dx = dF + (size_t)xcell * S * Np;
    for (int p = blockIdx.y * blockDim.x + threadIdx.x; p < Np; p += gridDim.y * blockDim.x) {
        double* src = dN_aos + ((size_t)xcell * Np + p) * SP;
        for (int a = 0; a < S; ++a) {
            dx[(size_t)a * Np + p] = src[a] / deg[a];
            src[a] = 0.0;
        }
    }
}

template <int kMask, int kSampler>
cudaError_t launch_collide_mask(const CollideParams& P, int ctas, cudaStream_t st)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    const size_t smem = sizeof(WarpMem<kSP>) * kWarps;
    // the attribute belongs to the (function, device) pair: one flag per device, not per process
    static bool configured[kMaxDevices] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices || !configured[dev]) {
        e = cudaFuncSetAttribute(collide_kernel<kMask, kSampler>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < kMaxDevices) configured[dev] = true;
    }
    collide_kernel<kMask, kSampler><<<ctas, kCollideThreads, smem, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

// the weighted samplers (NEXT rank 3) are instantiated for the pure-glue mask, the full mixture and the run-time mask
template <int kSampler>
cudaError_t launch_collide_weighted(const CollideParams& P, int ctas, cudaStream_t st)
{
    if (P.mask == 0x01u) return launch_collide_mask<0x01, kSampler>(P, ctas, st);
    if (P.mask == 0x7Fu && !P.has_ovr) return launch_collide_mask<0x7F, kSampler>(P, ctas, st);
    return launch_collide_mask<-1, kSampler>(P, ctas, st);
}

}  // namespace

int collide_slots_per_cell(unsigned mask) { return mask == 0x01u ? 1 : 8; }

// Work items: a run of `units` passes of 32 samples (ppc = ceil(Ns / 32) passes per p1 cell).  About 8 items per warp:
// long items amortise the hand-over between items, short ones balance the load on small grids (config 0 has 2.9 passes
// per warp in all).  Items of a cell or more are whole cells, at most 32 (the warp's p1 table).
void collide_item_geometry(int Np, int Nx, int Ns, int sms, int* units_per_item, int* ppc_out, int* regions_per_x)
{
    const int ppc = (Ns + 31) / 32;
    const long long total = (long long)Np * Nx * ppc;
    const long long slots = (long long)sms * kWarps * 8;
    long long u = (total + slots - 1) / slots;
    if (u < 1) u = 1;
    if (u >= ppc) { u = (u / ppc) * ppc; if (u > 32LL * ppc) u = 32LL * ppc; }
    *units_per_item = (int)u; *ppc_out = ppc;
    *regions_per_x = (int)(((long long)Np * ppc + u - 1) / u);
}

// one persistent CTA per SM (fewer when there is less work than warps)
cudaError_t launch_collide(const CollideParams& P, int sms, cudaStream_t st)
{
    int ctas = (int)((P.n_items + kWarps - 1) / kWarps);
    if (ctas > sms) ctas = sms;
    if (ctas < 1) ctas = 1;
    if (P.sampler == 1) return launch_collide_weighted<1>(P, ctas, st);
    if (P.sampler == 2) return launch_collide_weighted<2>(P, ctas, st);
    if (P.has_ovr && P.mask != 0x01u) return launch_collide_mask<-1, 0>(P, ctas, st);
    switch (P.mask) {
    case 0x01u: return launch_collide_mask<0x01, 0>(P, ctas, st);
    case 0x7Eu: return launch_collide_mask<0x7E, 0>(P, ctas, st);
    case 0x7Fu: return launch_collide_mask<0x7F, 0>(P, ctas, st);
    default:    return launch_collide_mask<-1, 0>(P, ctas, st);
    }
}

cudaError_t launch_debug_samples(const CollideParams& P, int xcell, int p_begin, int p_end, int* cells, double* stu,
                                 cudaStream_t st)
{
    const long long total = (long long)(p_end - p_begin) * P.Ns;
    if (total <= 0) return cudaSuccess;
    const long long cap = (long long)device_sms() * 16;
    const int blocks = (int)((total + 127) / 128 < cap ? (total + 127) / 128 : cap);
    debug_samples_kernel<<<blocks, 128, 0, st>>>(P, xcell, p_begin, p_end, cells, stu);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_cell_table(const GridConst& g, int Np, double* tab, cudaStream_t st)
{
    cell_table_kernel<<<(Np + 255) / 256, 256, 0, st>>>(g, Np, tab);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_pack(const double* f, double* f_aos, int Nx, int S, int SP, int Np, cudaStream_t st)
{
    dim3 grid(Nx, min((Np + 255) / 256, 65535));
    pack_kernel<<<grid, 256, 0, st>>>(f, f_aos, S, SP, Np);
    ++g_launch_count;
    return cudaGetLastError();
}

cudaError_t launch_finalize(double* dN_aos, double* dF, int Nx, int S, int SP, int Np, const double* deg, cudaStream_t st)
{
    dim3 grid(Nx, min((Np + 255) / 256, 65535));
    finalize_kernel<<<grid, 256, 0, st>>>(dN_aos, dF, S, SP, Np, deg[0], deg[1], deg[2], deg[3], deg[4], deg[5], deg[6]);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace bz
