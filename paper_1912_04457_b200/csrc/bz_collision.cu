// bz_collision.cu -- sample -> |M|^2 -> bracket -> symmetric deposit (S8a.2-8a.5) as ONE persistent, warp-specialised
// kernel (one CTA of 16 warps per SM):
//
//   producer warps (12, warpgroups 1-3, 88 registers after setmaxnreg.dec)
//       sample   pull work items (a run of p1 cells of one spatial cell) from a global counter; lanes = samples:
//                Philox4x32-10, the boost, the binning (bz_sample.cuh).  About 46 % of the samples keep both outgoing
//                legs in the box; they are compacted (ballot + prefix) straight into the record arrays of one of the
//                warp's two shared-memory batch slots: (i, j, k, l), s, t and the weight K/(E1 E2).
//       gather   when a slot holds 32 records: cp.async (LDGSTS) of the 4 x S occupation numbers of every sample from
//                the cell-major staging copy f_aos[xcell][pcell][SP] (SP = 8 doubles = 64 B per cell) into the slot;
//                for one sample the 32 lanes fetch its 4 cells x 8 slots, i.e. 8 sectors per instruction instead of 32
//                scattered ones.  Completion is signalled to the consumer by cp.async.mbarrier.arrive on the slot's
//                "full" mbarrier: the producer never waits for its own gathers and goes on sampling.
//       scatter  when the warp needs the slot again and the consumer has signalled "done": the same 8-lanes-per-cell
//                mapping issues fp64 reductions (RED.E.ADD.F64, no return value) of the slot's 4 x S deposits into
//                the cell-major scratch dN_aos, which stays in L2 while its spatial cell is being worked on.
//   consumer warps (4, warpgroup 0, one per SM sub-partition, 240 registers after setmaxnreg.inc)
//       compute  serve three producers each in rotation: wait "full", every lane takes one sample of the batch:
//                <= 10 |M|^2 values, factorised channel algebra (bz_channels.cuh), the 4 x S deposits overwrite the
//                gathered f in the slot, arrive on "done".
// The ALU-bound sampling and the latency-bound gather/scatter overlap on the same SM, the register file is split
// 240 / 88 between the two roles, and no sample record ever leaves the SM.
// Measured on B200 (profiles/): a RED (LDG) whose 32 lanes hit 32 different sectors costs 48 (32) cycles of the SM's
// L1TEX path, the 8-lanes-per-cell form 15.7 (8.5) cycles for the same number of lanes.
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

constexpr int kConsumerWarps = 4;                // warpgroup 0
constexpr int kProducerWarps = 12;               // warpgroups 1..3
constexpr int kProducersPerConsumer = kProducerWarps / kConsumerWarps;
constexpr int kCollideThreads = 32 * (kConsumerWarps + kProducerWarps);
constexpr int kSlots = 2;                        // batch slots per producer warp
constexpr int kConsumerRegs = 240, kProducerRegs = 88;   // 128 x 240 + 384 x 88 = 64512 <= 65536

// doubles per cell in the global staging layout: 1 for the pure-glue mask, 8 (half a 128-byte line) otherwise
template <int kMask>
struct MaskTraits {
    static constexpr int SP = kMask == 0x01 ? 1 : 8;
};
// layout index of species id = number of active ids below it
__device__ __forceinline__ int slot_of(unsigned mask, int id) { return __popc(mask & ((1u << id) - 1u)); }

// ------------------------------------------------------------------------------------------------ PTX helpers
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* b, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* b)
{
    asm volatile("{\n .reg .b64 st;\n mbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(smem_u32(b)) : "memory");
}
// arrive on b when all cp.async issued so far by this thread have landed (does not add to the expected count)
__device__ __forceinline__ void mbar_arrive_on_cp_async(uint64_t* b)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}
// one try_wait: the hardware suspends the warp until the phase completes or ~ns nanoseconds have passed
__device__ __forceinline__ bool mbar_try_wait(uint64_t* b, unsigned parity, unsigned ns)
{
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity), "r"(ns) : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* b, unsigned parity)
{
    while (!mbar_try_wait(b, parity, 2000u)) {}
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
// fp64 reduction without return value (RED.E.ADD.F64), skipped for an exact zero
__device__ __forceinline__ void red_add_nonzero(double* gdst, double v)
{
    asm volatile("{\n .reg .pred p;\n setp.neu.f64 p, %1, 0d0000000000000000;\n @p red.global.add.f64 [%0], %1;\n}"
                 ::"l"(gdst), "d"(v) : "memory");
}
template <int N>
__device__ __forceinline__ void setmaxnreg_inc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N)); }
template <int N>
__device__ __forceinline__ void setmaxnreg_dec() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N)); }

// ------------------------------------------------------------------------------------------------ batch slot
// One batch of <= 32 accepted samples in shared memory.  stage holds, per sample, the occupation numbers of its 4 cells
// (kCS doubles per cell) on the way in and the 4 x S deposits on the way out; the odd stride makes both the per-sample
// access of the consumer (lane = sample) and the per-cell access of the producer (lanes = slots of a cell) conflict free.
template <int kSP>
struct Slot {
    static constexpr int kCS = kSP == 1 ? 1 : 7;         // doubles per cell
    static constexpr int kStride = 4 * kCS + 1;          // doubles per sample
    double stage[32 * kStride];
    double s[32], t[32], e12[32];                        // Mandelstam s, t and E1 E2 of the sample
    int cell[32][4];                                     // i, j, k, l
    double m2;                                           // regulator mass^2 of the batch's spatial cell
    int nvalid;                                          // samples in the batch; < 0: the producer has finished
    int xcell;
    uint64_t full;                                       // producer -> consumer: records + gathered f are in place
    uint64_t done;                                       // consumer -> producer: deposits are in place
};

constexpr int kRetryCap = 64;                    // per producer warp: samples whose two Marsaglia attempts both failed

// lane -> element of a sample: kSP slots of each of the 4 cells; 32 / (4 kSP) samples per instruction
template <int kSP>
struct LaneMap {
    static constexpr int kEPS = 4 * kSP;                 // lanes per sample
    static constexpr int kSPI = 32 / kEPS;               // samples per instruction
    int sub, cc, sl;
    __device__ __forceinline__ explicit LaneMap(int lane) : sub(lane / kEPS), cc((lane % kEPS) / kSP), sl(lane % kSP) {}
};

// ---- producer: issue the gather of the slot's batch and hand the slot to the consumer
template <int kSP>
__device__ __forceinline__ void submit_slot(Slot<kSP>& sl, const CollideParams& P, int lane, int nvalid, int xcell, double m2)
{
    using S = Slot<kSP>;
    if (lane == 0) { sl.nvalid = nvalid; sl.xcell = xcell; sl.m2 = m2; }
    __syncwarp();                                        // the records written by all lanes are visible to all lanes
    if (nvalid > 0) {
        const LaneMap<kSP> lm(lane);
        if (lm.sl < P.S) {                               // pad lanes (slot 7 of a cell) sit the gather out
            const double* __restrict__ src = P.f_aos + (size_t)xcell * P.Np * kSP + lm.sl;
            double* dst = sl.stage + lm.sub * S::kStride + lm.cc * S::kCS + lm.sl;
            const int* cp = &sl.cell[lm.sub][lm.cc];
            if (nvalid == 32) {
#pragma unroll
                for (int m0 = 0; m0 < 32; m0 += LaneMap<kSP>::kSPI)
                    cp_async8(dst + m0 * S::kStride, src + (size_t)cp[4 * m0] * kSP);
            } else {
                for (int m0 = 0; m0 + lm.sub < nvalid; m0 += LaneMap<kSP>::kSPI)
                    cp_async8(dst + m0 * S::kStride, src + (size_t)cp[4 * m0] * kSP);
            }
        }
    }
    mbar_arrive_on_cp_async(&sl.full);                   // 32 deferred arrivals: this lane's gathers have landed
    if (lane == 0) mbar_arrive(&sl.full);                // + 1: header and records (release)
}

// ---- producer: flush the deposits the consumer left in the slot
template <int kSP>
__device__ __forceinline__ void scatter_slot(Slot<kSP>& sl, const CollideParams& P, int lane)
{
    using S = Slot<kSP>;
    const int nvalid = sl.nvalid;
    const LaneMap<kSP> lm(lane);
    if (lm.sl < P.S) {
        double* __restrict__ dst = P.dN_aos + (size_t)sl.xcell * P.Np * kSP + lm.sl;
        const double* src = sl.stage + lm.sub * S::kStride + lm.cc * S::kCS + lm.sl;
        const int* cp = &sl.cell[lm.sub][lm.cc];
        if (nvalid == 32) {
#pragma unroll
            for (int m0 = 0; m0 < 32; m0 += LaneMap<kSP>::kSPI)
                red_add_nonzero(dst + (size_t)cp[4 * m0] * kSP, src[m0 * S::kStride]);
        } else {
            for (int m0 = 0; m0 + lm.sub < nvalid; m0 += LaneMap<kSP>::kSPI)
                red_add_nonzero(dst + (size_t)cp[4 * m0] * kSP, src[m0 * S::kStride]);
        }
    }
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int kMask>
__global__ void __launch_bounds__(kCollideThreads, 1) collide_kernel(const CollideParams P)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    using S = Slot<kSP>;
    constexpr bool kGlue = kMask < 0 || (kMask & 1);
    constexpr bool kQuark = kMask < 0 || (kMask & 0x7E);
    extern __shared__ __align__(16) unsigned char smem_raw[];
    S* slots = reinterpret_cast<S*>(smem_raw);           // [kProducerWarps][kSlots]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x < kProducerWarps * kSlots) {
        mbar_init(&slots[threadIdx.x].full, 33);
        mbar_init(&slots[threadIdx.x].done, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    if (warp < kConsumerWarps) {
        // ======================================================================================== consumer
        setmaxnreg_inc<kConsumerRegs>();
        const unsigned mask = kMask >= 0 ? (unsigned)kMask : P.mask;
        unsigned alive = (1u << kProducersPerConsumer) - 1u;   // producers of this consumer still running
        unsigned cur = 0;                                      // bit q: next slot of producer q
        unsigned par = 0;                                      // bit 2q+slot: parity of the next "full" phase
        int q = 0;
        while (alive) {
            // poll the alive producers in rotation; each try suspends the warp for at most ~0.3 us
            if (!((alive >> q) & 1u)) { q = (q + 1) % kProducersPerConsumer; continue; }
            const int si = (cur >> q) & 1u;
            S& sl = slots[(warp + kConsumerWarps * q) * kSlots + si];
            if (!mbar_try_wait(&sl.full, (par >> (2 * q + si)) & 1u, 300u)) { q = (q + 1) % kProducersPerConsumer; continue; }
            par ^= 1u << (2 * q + si);
            cur ^= 1u << q;
            const int nvalid = sl.nvalid;
            if (nvalid < 0) { alive &= ~(1u << q); q = (q + 1) % kProducersPerConsumer; continue; }
            if (lane < nvalid) {
                double* st = sl.stage + lane * S::kStride;
                const double s = sl.s[lane], t = sl.t[lane], m2 = sl.m2;
                const double g4w = P.g4K * rcp_fast(sl.e12[lane]);            // g^4 K / (E1 E2), S8c step 6
                double fi[7], fj[7], fk[7], fl[7];
#pragma unroll
                for (int id = 0; id < 7; ++id) {
                    if ((mask >> id) & 1u) {
                        const int a = slot_of(mask, id);
                        fi[id] = st[a]; fj[id] = st[S::kCS + a]; fk[id] = st[2 * S::kCS + a]; fl[id] = st[3 * S::kCS + a];
                    } else {
                        fi[id] = fj[id] = fk[id] = fl[id] = 0.0;
                    }
                }
                const double u = __dsub_rn(-s, t);
                const MsqSet M = msq_set<kGlue, kQuark>(s, t, u, m2, g4w);
                double dI[7], dJ[7], dK[7], dL[7];
                deposit<kMask>(mask, fi, fj, fk, fl, M, dI, dJ, dK, dL);
#pragma unroll
                for (int id = 0; id < 7; ++id) {
                    if ((mask >> id) & 1u) {
                        const int a = slot_of(mask, id);
                        st[a] = dI[id]; st[S::kCS + a] = dJ[id]; st[2 * S::kCS + a] = dK[id]; st[3 * S::kCS + a] = dL[id];
                    }
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&sl.done);
            q = (q + 1) % kProducersPerConsumer;
        }
        return;
    }

    // ============================================================================================ producer
    setmaxnreg_dec<kProducerRegs>();
    const int pw = warp - kConsumerWarps;
    S* my = slots + pw * kSlots;
    int2* retry = reinterpret_cast<int2*>(slots + kProducerWarps * kSlots) + pw * kRetryCap;
    int cur = 0;                         // slot being filled
    int count = 0;                       // records in it
    int rcount = 0;                      // entries in the retry list
    unsigned busy = 0;                   // bit s: slot s is with the consumer (submitted, deposits not yet flushed)
    unsigned dpar = 0;                   // bit s: parity of the next "done" phase of slot s
    for (;;) {
        unsigned item = 0;
        if (lane == 0) item = atomicAdd(P.work_counter, 1u);
        item = __shfl_sync(0xffffffffu, item, 0);
        if (item >= P.n_items) break;
        const int xi = (int)(item / (unsigned)P.regions_per_x), region = (int)(item % (unsigned)P.regions_per_x);
        const int xcell = P.x_begin + xi;
        const double m2 = P.m2[xcell];
        const int i_end = min((region + 1) * P.cells_per_region, P.Np);
        int i = region * P.cells_per_region, base = 0;
        double p1x = 0.0, p1y = 0.0, p1z = 0.0, E1 = 0.0;
        bool cell_valid = false;
        for (;;) {
            // ---- next 32 (cell, sample, first attempt) triples: a full warp of retries if there is one, else fresh samples
            int ci, smp;
            unsigned kstart;
            bool active;
            if (rcount >= 32 || (i >= i_end && rcount > 0)) {
                const int nr = min(rcount, 32);
                rcount -= nr;
                active = lane < nr;
                const int2 e = active ? retry[rcount + lane] : make_int2(0, 0);
                ci = e.x; smp = e.y & 0x1ffffff; kstart = (unsigned)e.y >> 25;
                cell_kinematics(P.g, ci, p1x, p1y, p1z, E1);              // per lane
                cell_valid = false;
            } else if (i < i_end) {
                if (!cell_valid) { cell_kinematics(P.g, i, p1x, p1y, p1z, E1); cell_valid = true; }
                ci = i; smp = base + lane; kstart = 0u;
                active = smp < P.Ns;
                base += 32;
                if (base >= P.Ns) { base = 0; ++i; cell_valid = false; }
            } else {
                break;
            }
            Sample sa;
            sa.flag = 0; sa.retry = 0;
            if (active)
                sa = gen_sample_pair(P.g, P.seed, P.step, (uint32_t)xcell, (uint32_t)ci, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
            const unsigned lt = (1u << lane) - 1u;
            const unsigned rb = __ballot_sync(0xffffffffu, sa.retry);
            if (rb) {
                if (sa.retry) retry[rcount + __popc(rb & lt)] = make_int2(ci, smp | (int)((kstart + 2u) << 25));
                rcount += __popc(rb);
                __syncwarp();
            }
            // ---- compact the accepted samples into the current slot; a full slot goes to the consumer
            const unsigned acc = __ballot_sync(0xffffffffu, sa.flag);
            if (acc == 0u) continue;
            int pos = count + __popc(acc & lt);
            if (sa.flag && pos < 32) {
                S& sl = my[cur];
                *reinterpret_cast<int4*>(&sl.cell[pos][0]) = make_int4(ci, sa.j, sa.k, sa.l);
                sl.s[pos] = sa.s; sl.t[pos] = sa.t; sl.e12[pos] = sa.E1E2;
            }
            count += __popc(acc);
            if (count >= 32) {
                submit_slot<kSP>(my[cur], P, lane, 32, xcell, m2);
                busy |= 1u << cur;
                cur ^= 1;
                if ((busy >> cur) & 1u) {                    // make the other slot writable: wait for the consumer, flush
                    mbar_wait(&my[cur].done, (dpar >> cur) & 1u);
                    dpar ^= 1u << cur;
                    busy &= ~(1u << cur);
                    scatter_slot<kSP>(my[cur], P, lane);
                    __syncwarp();
                }
                count -= 32;
                pos -= 32;
                if (sa.flag && pos >= 0) {
                    S& sl = my[cur];
                    *reinterpret_cast<int4*>(&sl.cell[pos][0]) = make_int4(ci, sa.j, sa.k, sa.l);
                    sl.s[pos] = sa.s; sl.t[pos] = sa.t; sl.e12[pos] = sa.E1E2;
                }
            }
        }
        if (count > 0) {                                     // batches never mix spatial cells: flush the partial one
            submit_slot<kSP>(my[cur], P, lane, count, xcell, m2);
            busy |= 1u << cur;
            cur ^= 1;
            if ((busy >> cur) & 1u) {
                mbar_wait(&my[cur].done, (dpar >> cur) & 1u);
                dpar ^= 1u << cur;
                busy &= ~(1u << cur);
                scatter_slot<kSP>(my[cur], P, lane);
                __syncwarp();
            }
            count = 0;
        }
    }
    submit_slot<kSP>(my[cur], P, lane, -1, 0, 0.0);          // terminator (the current slot is always writable)
    cur ^= 1;
    if ((busy >> cur) & 1u) {
        mbar_wait(&my[cur].done, (dpar >> cur) & 1u);
        scatter_slot<kSP>(my[cur], P, lane);
    }
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
            sm = gen_sample_pair(P.g, P.seed, P.step, (uint32_t)xcell, (uint32_t)i, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
            kstart += 2u;
        } while (sm.retry);
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
cudaError_t launch_collide_mask(const CollideParams& P, int ctas, cudaStream_t st)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    const size_t smem = sizeof(Slot<kSP>) * kProducerWarps * kSlots + sizeof(int2) * kRetryCap * kProducerWarps;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(collide_kernel<kMask>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    collide_kernel<kMask><<<ctas, kCollideThreads, smem, st>>>(P);
    ++g_launch_count;
    return cudaGetLastError();
}

}  // namespace

int collide_slots_per_cell(unsigned mask) { return mask == 0x01u ? 1 : 8; }

// p1 cells per work item: long items amortise the final partial batch, short ones balance the load on small grids
int collide_cells_per_region(int Np, int Nx, int sms)
{
    const long long total_cells = (long long)Np * Nx;
    const long long c = total_cells / ((long long)sms * kProducerWarps * 8);
    return (int)(c < 1 ? 1 : (c > 32 ? 32 : c));
}

// one persistent CTA per SM (fewer when there is less work than producer warps)
cudaError_t launch_collide(const CollideParams& P, int sms, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(P.work_counter, 0, sizeof(unsigned), st);
    if (e != cudaSuccess) return e;
    int ctas = (int)((P.n_items + kProducerWarps - 1) / kProducerWarps);
    if (ctas > sms) ctas = sms;
    if (ctas < 1) ctas = 1;
    switch (P.mask) {
    case 0x01u: return launch_collide_mask<0x01>(P, ctas, st);
    case 0x7Eu: return launch_collide_mask<0x7E>(P, ctas, st);
    case 0x7Fu: return launch_collide_mask<0x7F>(P, ctas, st);
    default:    return launch_collide_mask<-1>(P, ctas, st);
    }
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
