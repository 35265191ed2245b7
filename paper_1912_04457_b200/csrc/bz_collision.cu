// bz_collision.cu -- sample -> |M|^2 -> bracket -> symmetric deposit (S8a.2-8a.5) as ONE persistent, warp-specialised
// kernel (one CTA of 20 warps per SM):
//
//   producer warps (16, warpgroups 1-4, 64 registers after setmaxnreg.dec)
//       sample   pull work items (a run of p1 cells of one spatial cell) from a global counter; lanes = samples:
//                Philox4x32-10, the boost, the binning (bz_sample.cuh).  About 46 % of the samples keep both outgoing
//                legs in the box; they are compacted (ballot + prefix) straight into one of the warp's two record
//                buffers in shared memory: (i, j, k, l), s, t and E1 E2.
//       gather   when a record buffer holds 32 samples: cp.async (LDGSTS, 16 bytes per lane, L1 bypassed) of the
//                4 cells x 64 bytes of every sample from the cell-major staging copy f_aos[xcell][pcell][8] into the
//                warp's stage buffer: 4 lanes fetch one cell, one instruction fetches 8 cells = 16 sectors instead of
//                32 scattered ones.  Completion is signalled to the consumer by cp.async.mbarrier.arrive on the
//                "full" mbarrier: the producer never waits for its own gathers and goes on sampling into the other
//                record buffer.
//   consumer warps (4, warpgroup 0, one per SM sub-partition, 224 registers after setmaxnreg.inc)
//       compute  serve four producers each (non-blocking probes in rotation): every lane takes one sample of the batch:
//                <= 10 |M|^2 values, factorised channel algebra (bz_channels.cuh); the 4 x S deposits overwrite the
//                gathered f in the stage buffer; arrive on "done".
//       (pure glue, one double per cell: the consumer issues its four reductions straight from the registers.)
//   producer, scatter: when the warp's next batch is complete and "done" has been signalled, it flushes the stage
//                buffer with fp64 reductions (RED.E.ADD.F64, no return value), one sample per instruction with 8 lanes
//                per 64-byte cell, into the cell-major scratch dN_aos, which stays in L2 while its spatial cell is
//                being worked on; then it gathers the new batch into the same buffer.
// The ALU-bound sampling and the latency-bound gather/scatter overlap on the same SM, the register file is split
// 224 / 64 between the two roles (640 threads launch with 96 registers each; setmaxnreg only moves registers inside
// that pool of 61440), and no sample record ever leaves the SM.  Measured on B200, config 4 (ablations, ms per
// launch of 211): sampling + compaction alone 102, consumer algebra +75, RED flush +43, cp.async gather +27 -- the
// parts add up, i.e. the kernel is bound by issue slots (FP64 instructions occupy the 16-lane pipe for 2 cycles),
// not by latency: 12 -> 16 producer warps gave +4 %.
// Measured on B200 (microbenchmark over all 148 SMs): a RED whose 32 lanes hit 32 different sectors
// costs 48 cycles of the SM's L1TEX path, the 8-lanes-per-cell form 15.7; chip-wide that form saturates at ~6e10 cell
// updates/s (the L2 reduction rate).  The 64-byte TMA bulk reduction (cp.reduce.async.bulk.add.f64) reaches the same
// chip-wide rate but is a uniform-datapath instruction: per-lane addresses cost an 8-instruction elect loop per cell
// against 1.5 instructions per cell here, so it is not used.
#include "bz_channels.cuh"
#include "bz_internal.h"

namespace bz {

namespace {

#ifndef BZ_PRODUCER_WARPS
#define BZ_PRODUCER_WARPS 16
#endif
#ifndef BZ_CONSUMER_REGS
#define BZ_CONSUMER_REGS 224
#endif
#ifndef BZ_PRODUCER_REGS
#define BZ_PRODUCER_REGS 64
#endif
constexpr int kConsumerWarps = 4;                // warpgroup 0
constexpr int kProducerWarps = BZ_PRODUCER_WARPS;   // warpgroups 1..
constexpr int kProducersPerConsumer = kProducerWarps / kConsumerWarps;
constexpr int kCollideThreads = 32 * (kConsumerWarps + kProducerWarps);
constexpr int kConsumerRegs = BZ_CONSUMER_REGS, kProducerRegs = BZ_PRODUCER_REGS;
// setmaxnreg moves registers inside the pool the CTA was launched with (threads x launch registers, the launch count
// being 64 K / threads rounded down to a multiple of 8): a split that needs more never gets its .inc granted and hangs
constexpr int kLaunchRegs = (65536 / kCollideThreads) / 8 * 8;
static_assert(128 * kConsumerRegs + 32 * kProducerWarps * kProducerRegs <= kCollideThreads * kLaunchRegs, "register pool");

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
// non-blocking probe of a phase
__device__ __forceinline__ bool mbar_test_wait(uint64_t* b, unsigned parity)
{
    unsigned ok;
    asm volatile("{\n .reg .pred p;\n mbarrier.test_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_u32(b)), "r"(parity) : "memory");
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
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
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

// ------------------------------------------------------------------------------------------------ shared memory
// Records of one batch of <= 32 accepted samples.
struct Rec {
    int cell[32][4];                                     // i, j, k, l
    double s[32], t[32], e12[32];                        // Mandelstam s, t and E1 E2 of the sample
};

// Per producer warp: two record buffers (one being filled, one with the consumer) and one stage buffer that holds,
// per sample, the occupation numbers of its 4 cells on the way in and the deposits on the way out.
//   kSP == 8: 8 doubles (64 B, one staging-layout cell) per cell, 34 doubles per sample: every cell is 16-byte aligned
//             (cp.async 16) and the consumer's 16-byte accesses (lane = sample, 272 B apart = 17 x 16)
//             are bank-conflict free.
//   kSP == 1: 1 double per cell, 5 doubles per sample (odd stride: conflict free for 8-byte accesses).
template <int kSP>
struct alignas(16) Chan {
    static constexpr int kCS = kSP == 1 ? 1 : 8;         // doubles per cell
    static constexpr int kStride = kSP == 1 ? 5 : 34;    // doubles per sample
    double stage[32 * kStride];
    Rec rec[2];
    double m2;                                           // regulator mass^2 of the batch's spatial cell
    int nvalid;                                          // samples in the batch; < 0: the producer has finished
    int xcell;
    int ridx;                                            // record buffer of the batch
    int pad_;
    uint64_t full;                                       // producer -> consumer: records + gathered f are in place
    uint64_t done;                                       // consumer -> producer: the stage buffer may be overwritten
};

constexpr int kMaxDevices = 64;
constexpr int kRetryCap = 64;                    // per producer warp: samples whose two Marsaglia attempts both failed

// ---- producer: wait until the stage buffer is free, issue the gather of the batch in rec[ridx], hand it to the consumer
template <int kSP>
__device__ __noinline__ unsigned submit_batch(Chan<kSP>& ch, const double* __restrict__ f_aos, double* __restrict__ dN_aos,
                                              int Np, int S, int lane, int ridx, int nvalid, int xcell, double m2,
                                              unsigned in_flight, unsigned dpar)
{
    using C = Chan<kSP>;
    if (in_flight) {                                     // the previous batch: flush the deposits the consumer left
        mbar_wait(&ch.done, dpar);
        dpar ^= 1u;
        if constexpr (kSP != 1) {
            // one sample per instruction: lane = (cell cc, slot sl) of the sample, 8 lanes per 64-byte cell
            const int pn = ch.nvalid, cc = lane >> 3, sl = lane & 7;
            if (sl < S) {
                double* __restrict__ gdst = dN_aos + (size_t)ch.xcell * Np * 8 + sl;
                const double* src = ch.stage + lane;
                const int* cp = &ch.rec[ridx ^ 1].cell[0][cc];
                if (pn == 32) {
#pragma unroll
                    for (int m = 0; m < 32; ++m) red_add_nonzero(gdst + (size_t)cp[4 * m] * 8, src[m * C::kStride]);
                } else {
                    for (int m = 0; m < pn; ++m) red_add_nonzero(gdst + (size_t)cp[4 * m] * 8, src[m * C::kStride]);
                }
            }
            __syncwarp();
        }
    }
    if (lane == 0) { ch.nvalid = nvalid; ch.xcell = xcell; ch.m2 = m2; ch.ridx = ridx; }
    __syncwarp();                                        // the records written by all lanes are visible to all lanes
    if (nvalid > 0) {
        const int* cells = &ch.rec[ridx].cell[0][0];
        if constexpr (kSP == 1) {
            const int sub = lane >> 2, cc = lane & 3;    // 8 samples per instruction, 4 lanes (cells) each
            const double* __restrict__ src = f_aos + (size_t)xcell * Np;
            double* dst = ch.stage + sub * C::kStride + cc;
            const int* cp = cells + sub * 4 + cc;
#pragma unroll
            for (int m0 = 0; m0 < 32; m0 += 8)
                if (m0 + sub < nvalid) cp_async8(dst + m0 * C::kStride, src + cp[4 * m0]);
        } else {
            const int sub = lane >> 4, cc = (lane >> 2) & 3, q = lane & 3;   // 2 samples per instruction, 4 lanes per cell
            const double* __restrict__ src = f_aos + (size_t)xcell * Np * 8 + q * 2;
            double* dst = ch.stage + sub * C::kStride + cc * 8 + q * 2;
            const int* cp = cells + sub * 4 + cc;
            if (nvalid == 32) {
#pragma unroll
                for (int m0 = 0; m0 < 32; m0 += 2)
                    cp_async16(dst + m0 * C::kStride, src + (size_t)cp[4 * m0] * 8);
            } else {
                for (int m0 = 0; m0 + sub < nvalid; m0 += 2)
                    cp_async16(dst + m0 * C::kStride, src + (size_t)cp[4 * m0] * 8);
            }
        }
    }
    mbar_arrive_on_cp_async(&ch.full);                   // 32 deferred arrivals: this lane's gathers have landed
    if (lane == 0) mbar_arrive(&ch.full);                // + 1: header and records (release)
    return dpar;                                         // parity of the "done" phase this batch will complete
}

// ---- consumer: one sample per lane: |M|^2, channel algebra, deposits; then the scatter of the lane's four cells
template <int kMask, int kSP>
__device__ __forceinline__ void consume_batch(Chan<kSP>& ch, const CollideParams& P, int lane, unsigned mask)
{
    using C = Chan<kSP>;
    constexpr bool kGlue = kMask < 0 || (kMask & 1);
    constexpr bool kQuark = kMask < 0 || (kMask & 0x7E);
    const int nvalid = ch.nvalid;
    const Rec& R = ch.rec[ch.ridx];
    if (lane < nvalid) {
        double* st = ch.stage + lane * C::kStride;
        const double s = R.s[lane], t = R.t[lane], m2 = ch.m2;
        const double g4w = P.g4K * rcp_fast(R.e12[lane]);                 // g^4 K / (E1 E2), S8c step 6
        const int4 cl = *reinterpret_cast<const int4*>(&R.cell[lane][0]);
        double fi[7], fj[7], fk[7], fl[7];
        if constexpr (kSP == 8 && kMask >= 0) {
            // compile-time layout: 16-byte loads, the registers are picked statically
            constexpr int kPairs = (slot_of((unsigned)kMask, 7) + 1) / 2;
            double2 v[4][4];
#pragma unroll
            for (int c = 0; c < 4; ++c)
#pragma unroll
                for (int q = 0; q < kPairs; ++q) v[c][q] = *reinterpret_cast<const double2*>(st + c * 8 + 2 * q);
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                if ((kMask >> id) & 1) {
                    constexpr unsigned km = (unsigned)kMask;
                    const int a = slot_of(km, id);
                    fi[id] = (a & 1) ? v[0][a >> 1].y : v[0][a >> 1].x;
                    fj[id] = (a & 1) ? v[1][a >> 1].y : v[1][a >> 1].x;
                    fk[id] = (a & 1) ? v[2][a >> 1].y : v[2][a >> 1].x;
                    fl[id] = (a & 1) ? v[3][a >> 1].y : v[3][a >> 1].x;
                } else {
                    fi[id] = fj[id] = fk[id] = fl[id] = 0.0;
                }
            }
        } else {
#pragma unroll
            for (int id = 0; id < 7; ++id) {
                if ((mask >> id) & 1u) {
                    const int a = slot_of(mask, id);
                    fi[id] = st[a]; fj[id] = st[C::kCS + a]; fk[id] = st[2 * C::kCS + a]; fl[id] = st[3 * C::kCS + a];
                } else {
                    fi[id] = fj[id] = fk[id] = fl[id] = 0.0;
                }
            }
        }
        const double u = __dsub_rn(-s, t);
        MsqSet M = msq_set<kGlue, kQuark>(s, t, u, m2, g4w);
        // user-defined matrix elements (bz_set_msq_override) run on the runtime-mask instantiation (and the light
        // pure-glue one), so that the specialised mixture kernels carry no extra registers for them
        if constexpr (kMask < 0 || kMask == 0x01) { if (P.has_ovr) msq_apply_override(M, P.msq_ovr, g4w); }
        double d[4][7];
        deposit<kMask>(mask, fi, fj, fk, fl, M, d[0], d[1], d[2], d[3]);
        if constexpr (kSP == 1) {
            // pure glue: four scalar reductions straight from the registers
            double* __restrict__ dst = P.dN_aos + (size_t)ch.xcell * P.Np;
            red_add_nonzero(dst + cl.x, d[0][0]); red_add_nonzero(dst + cl.y, d[1][0]);
            red_add_nonzero(dst + cl.z, d[2][0]); red_add_nonzero(dst + cl.w, d[3][0]);
        } else {
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
#pragma unroll
                    for (int q = 0; q < kPairs; ++q)
                        *reinterpret_cast<double2*>(st + c * 8 + 2 * q) = make_double2(o[2 * q], o[2 * q + 1]);
                }
            } else {
#pragma unroll
                for (int id = 0; id < 7; ++id) {
                    if ((mask >> id) & 1u) {
                        const int a = slot_of(mask, id);
                        st[a] = d[0][id]; st[8 + a] = d[1][id]; st[16 + a] = d[2][id]; st[24 + a] = d[3][id];
                    }
                }
            }
            // slots that hold no species keep the zeros they were gathered with (pack_kernel writes the pads as 0)
        }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&ch.done);
}

// momentum and energy of the centre of a p1 cell from the table built by cell_table_kernel (same arithmetic as
// cell_kinematics, done once per context instead of once per warp pass)
__device__ __forceinline__ void cell_lookup(const double* __restrict__ tab, int pcell, double& p1x, double& p1y, double& p1z,
                                            double& E1)
{
    const double2 a = __ldg(reinterpret_cast<const double2*>(tab) + 2 * (size_t)pcell);
    const double2 b = __ldg(reinterpret_cast<const double2*>(tab) + 2 * (size_t)pcell + 1);
    p1x = a.x; p1y = a.y; p1z = b.x; E1 = b.y;
}

// ------------------------------------------------------------------------------------------------ the kernel
template <int kMask>
__global__ void __launch_bounds__(kCollideThreads, 1) collide_kernel(const CollideParams P)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    using C = Chan<kSP>;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    C* chans = reinterpret_cast<C*>(smem_raw);           // [kProducerWarps]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x < kProducerWarps) {
        mbar_init(&chans[threadIdx.x].full, 33);
        mbar_init(&chans[threadIdx.x].done, 1);
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.next_counter = 0u;   // the other launch parity: idle during this launch
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    __syncthreads();

    if (warp < kConsumerWarps) {
        // ======================================================================================== consumer
        setmaxnreg_inc<kConsumerRegs>();
        const unsigned mask = kMask >= 0 ? (unsigned)kMask : P.mask;
        unsigned alive = (1u << kProducersPerConsumer) - 1u;   // producers of this consumer still running
        unsigned par = 0;                                      // bit q: parity of the next "full" phase of producer q
        int q = 0, misses = 0;
        while (alive) {
            // probe the alive producers in rotation without blocking; only after a whole round of misses suspend
            // (for at most ~0.2 us) on the next one
            if ((alive >> q) & 1u) {
                C& ch = chans[warp + kConsumerWarps * q];
                const unsigned pq = (par >> q) & 1u;
                const bool ready = misses < kProducersPerConsumer ? mbar_test_wait(&ch.full, pq) : mbar_try_wait(&ch.full, pq, 200u);
                if (ready) {
                    par ^= 1u << q;
                    misses = 0;
                    if (ch.nvalid < 0) alive &= ~(1u << q);
                    else consume_batch<kMask, kSP>(ch, P, lane, mask);
                } else {
                    misses = misses < kProducersPerConsumer ? misses + 1 : 0;
                }
            }
            q = (q + 1 == kProducersPerConsumer) ? 0 : q + 1;
        }
        return;
    }

    // ============================================================================================ producer
    setmaxnreg_dec<kProducerRegs>();
    const int pw = warp - kConsumerWarps;
    C& ch = chans[pw];
    int2* retry = reinterpret_cast<int2*>(chans + kProducerWarps) + pw * kRetryCap;
    int cur = 0;                         // record buffer being filled
    int count = 0;                       // records in it
    int rcount = 0;                      // entries in the retry list
    unsigned in_flight = 0;              // a batch has been submitted and its "done" phase not yet consumed
    unsigned long long n_acc = 0ull;     // samples accepted by this warp (bz_get_sample_counts)
    unsigned dpar = 0;                   // parity of the next "done" phase
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
                cell_lookup(P.cell_tab, ci, p1x, p1y, p1z, E1);           // per lane
                cell_valid = false;
            } else if (i < i_end) {
                if (!cell_valid) { cell_lookup(P.cell_tab, i, p1x, p1y, p1z, E1); cell_valid = true; }
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
                sa = gen_sample_pair(P.g, P.seed, P.step, (uint32_t)xcell + P.x_rng_offset, (uint32_t)ci, (uint32_t)smp, kstart, p1x, p1y, p1z, E1);
            const unsigned lt = (1u << lane) - 1u;
            const unsigned rb = __ballot_sync(0xffffffffu, sa.retry);
            if (rb) {
                if (sa.retry) retry[rcount + __popc(rb & lt)] = make_int2(ci, smp | (int)((kstart + 2u) << 25));
                rcount += __popc(rb);
                __syncwarp();
            }
            // ---- compact the accepted samples into the current record buffer; a full buffer goes to the consumer
            const unsigned acc = __ballot_sync(0xffffffffu, sa.flag);
            n_acc += (unsigned)__popc(acc);
            if (acc == 0u) continue;
            int pos = count + __popc(acc & lt);
            if (sa.flag && pos < 32) {
                Rec& r = ch.rec[cur];
                *reinterpret_cast<int4*>(&r.cell[pos][0]) = make_int4(ci, sa.j, sa.k, sa.l);
                r.s[pos] = sa.s; r.t[pos] = sa.t; r.e12[pos] = sa.E1E2;
            }
            count += __popc(acc);
            if (count >= 32) {
                dpar = submit_batch<kSP>(ch, P.f_aos, P.dN_aos, P.Np, P.S, lane, cur, 32, xcell, m2, in_flight, dpar); in_flight = 1u;
                cur ^= 1;                                    // its previous batch is done: submit_batch has waited for it
                count -= 32;
                pos -= 32;
                if (sa.flag && pos >= 0) {
                    Rec& r = ch.rec[cur];
                    *reinterpret_cast<int4*>(&r.cell[pos][0]) = make_int4(ci, sa.j, sa.k, sa.l);
                    r.s[pos] = sa.s; r.t[pos] = sa.t; r.e12[pos] = sa.E1E2;
                }
            }
        }
        if (count > 0) {                                     // batches never mix spatial cells: flush the partial one
            dpar = submit_batch<kSP>(ch, P.f_aos, P.dN_aos, P.Np, P.S, lane, cur, count, xcell, m2, in_flight, dpar); in_flight = 1u;
            cur ^= 1;
            count = 0;
        }
    }
    submit_batch<kSP>(ch, P.f_aos, P.dN_aos, P.Np, P.S, lane, cur, -1, 0, 0.0, in_flight, dpar);   // flush the last batch, then the terminator
    if (lane == 0 && P.counters) atomicAdd(P.counters, n_acc);
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

template <int kMask>
cudaError_t launch_collide_mask(const CollideParams& P, int ctas, cudaStream_t st)
{
    constexpr int kSP = MaskTraits<kMask>::SP;
    const size_t smem = sizeof(Chan<kSP>) * kProducerWarps + sizeof(int2) * kRetryCap * kProducerWarps;
    // the attribute belongs to the (function, device) pair: one flag per device, not per process
    static bool configured[kMaxDevices] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices || !configured[dev]) {
        e = cudaFuncSetAttribute(collide_kernel<kMask>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < kMaxDevices) configured[dev] = true;
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
    int ctas = (int)((P.n_items + kProducerWarps - 1) / kProducerWarps);
    if (ctas > sms) ctas = sms;
    if (ctas < 1) ctas = 1;
    if (P.has_ovr && P.mask != 0x01u) return launch_collide_mask<-1>(P, ctas, st);
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
