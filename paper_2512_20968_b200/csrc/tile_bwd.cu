// tile_bwd.cu -- mesh_attn_tile_bwd: per-pair attention backward of a simulated GPU's tile
// (Alg.3 l.3-5, L250-253; kernel inputs (Q_i, KV_j, O_i, dO_i), L236).
//
// One persistent CTA per SM walks the work list.  A work item is a 128-key block of one
// (simulated GPU g, KV partition v, KV head); the CTA keeps K and V of the block resident in
// shared memory and dK, dV in TMEM, and streams 128-row Q / dO blocks of every Q partition
// of the tile (and every query head of the GQA group).  Per Q block, five tcgen05 MMAs:
//
//   S^T  = K Q^T            (TMEM columns   0..127)      P^T = scale * exp2(S^T*c - lse*log2e)  (bf16, over S^T)
//   dP^T = V dO^T           (TMEM columns 128..255)      dS^T = P^T o (dP^T - delta)    (bf16, smem)
//   dV  += P^T  dO          (TMEM columns 384..511)      A operand P^T straight from TMEM
//   dK  += dS^T Q           (TMEM columns 256..383)      A operand dS^T from smem (K-major)
//   dQ^T = K^T dS^T         (TMEM columns 128..255, reusing dP^T once consumed)
//                                                        A = K tile read M-major, B = dS^T read N-major
//
// dQ is produced TRANSPOSED (TMEM lane = head-dim index d, column = query): a drain thread then writes 32
// consecutive floats of a dQ row per warp instruction into a row-major shared-memory staging tile, and the TMA
// engine adds the tile into global dQ (cp.reduce.async.bulk.tensor, add.f32): full lines per request at the L2
// atomic rate (6.1 TB/s measured; plain red.global with lane = query row: 2.9 TB/s), and none of it in the SM's
// load/store queue (512 red.global per step delayed every tcgen05.ld / ld.shared of the compute warps by hundreds
// of clocks; profiles/r01_v5_README.md).
//
//   warp 0      TMA producer: K,V per item; Q (+ exponent offsets, delta) per step through a 2-stage ring; dO through
//               a single buffer (dO(i+1) is only needed a full step after dV(i) released it)
//   warp 1      MMA issuer (one thread)
//   warp 2      TMEM allocator
//   warps 4-7   compute group 0: key row = TMEM lane, query columns  0..63  of the block
//   warps 8-11  compute group 1: key row = TMEM lane, query columns 64..127
//               each: S^T -> P^T (regs + TMEM), dP^T -> dS^T (smem); epilogue: group 0 drains dK, group 1 drains dV
//   warps 12-15 dQ drain group: dQ^T row d = TMEM lane -> registers (TMEM released) -> staging ring -> TMA reduce,
//               overlapping the next step's MMAs
//
// The softmax scale is folded into P^T (its log2 is part of the exponent offset the preprocess kernel wrote), so
// dS^T, dQ^T and dK come out already scaled and only dV is divided by it, once per item in the epilogue.
//
// dQ, dK, dV are accumulated into global fp32 with atomics: the sums over the Q group, the KV
// group (Alg.3 l.6-7, L254-255) and the GQA head group all land in the same buffers.
//
// kSplit (plan precision = 1): P and dS are fed to the tensor core as hi + lo bf16 pairs (two
// MMAs each for dV, dK, dQ^T), which brings the operand rounding from 2^-9 to 2^-17 relative;
// needed when |dS| is large (outlier scores, BASELINE.json configs[2]).
#include <cuda_bf16.h>

#include <atomic>

#include "plan.hpp"
#include "sm100.cuh"
#include "tile_kernels.hpp"

namespace mesh_attn {
using namespace sm100;

namespace {

constexpr int kBwdThreads = 512;
#ifndef MESH_ATTN_BWD_POLY_OF_4
#define MESH_ATTN_BWD_POLY_OF_4 0        // exponentials per 4 evaluated on the FMA pipe instead of the MUFU
#endif
constexpr int kBwdPolyOf4 = MESH_ATTN_BWD_POLY_OF_4;
// Ablation builds (tuning only, results are WRONG): bit 0 = the compute groups skip P^T / dS^T (they only pass the barriers on),
// bit 1 = the dQ drain group skips the TMEM load, the exchange, the staging and the reduces.  What is left of the step time
// tells which role bounds the kernel (profiles/r02_v4_README.md).
#ifndef MESH_ATTN_BWD_ABLATE
#define MESH_ATTN_BWD_ABLATE 0
#endif
constexpr int kAblate = MESH_ATTN_BWD_ABLATE;
// register budget per thread (setmaxnreg): 128 x kCtrlRegs + 256 x kComputeRegs + 128 x kDrainRegs <= 65536
constexpr int kCtrlRegs = 80, kComputeRegs = 136, kDrainRegs = 160;
template <int kRegs> __device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegs)); }
template <int kRegs> __device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegs)); }

template <int D, bool kSplit, bool kExch> struct BwdCfg {
    static_assert(!(kSplit && kExch), "the dQ exchange is built for the single-operand mode only");
    static_assert(D == 128, "backward kernel: dQ^T needs head_dim = UMMA M = 128");
    static constexpr int kBoxes = D / 64;
    static constexpr int kTileBytes = kBlock * D * 2;          // [128 x D] bf16
    static constexpr int kDsBytes = kBlock * kBlock * 2;        // dS^T [128 kv x 128 q] bf16
    static constexpr int kNumDs = kSplit ? 2 : 1;               // hi (+ lo)
    static constexpr int kStages = kSplit ? 1 : 2;              // Q ring; split mode trades the second Q stage for the dS lo tile
    static constexpr int kStgRows = kExch ? kBwdStgRowsExch : kBwdStgRows;   // dQ staging: a ring of kStgBufs buffers of [kStgRows queries][D] fp32
    static constexpr int kStgBytes = kBwdStgBytes;
    static constexpr int kStgBufs = kStgBytes / (kStgRows * D * 4);
    static_assert(kStgBufs >= 1 && kStgBufs * kStgRows * D * 4 == kStgBytes, "staging rows must divide the staging memory");
    static constexpr int kDrainRows = kExch ? kBlock / 2 : kBlock;   // query rows of a step this CTA reduces into global dQ
    // kExch: the peer's dQ^T half for this CTA's queries arrives as bf16 ([8 octets of queries][D][8]) in the FIRST HALF of the
    // staging memory, is added to the registers, and then the whole 64-row fp32 sum is staged over it
    static constexpr int kRecvBytes = (kBlock / 2) * D * 2;
    static_assert(!kExch || (kDrainRows * D * 4 == kStgBytes && 2 * kRecvBytes == kStgBytes), "the exchange stages a whole step at once");
    static constexpr int kOffK = 0;
    static constexpr int kOffV = kTileBytes;
    static constexpr int kOffQ = 2 * kTileBytes;                // kStages Q tiles
    static constexpr int kOffdO = kOffQ + kStages * kTileBytes; // ONE dO tile: dO(i+1) is only needed a full step after dV(i) freed it
    static constexpr int kOffDs = kOffdO + kTileBytes;
    static constexpr int kOffStg = kOffDs + kNumDs * kDsBytes;  // dQ staging for the TMA reduce
    static constexpr int kOffRecv = kOffStg;                    // aliases the first half of the staging memory (kExch)
    static constexpr int kOffVec = kOffStg + kStgBytes;         // per Q stage: log2(scale)-lse*log2e [128], delta[128] fp32
    static constexpr int kOffBars = kOffVec + kStages * 1024;
    static constexpr int kSchedSlots = 2;                       // ring of work-item indices handed out by the scheduler warp
    static constexpr int kNumBars = 2 + 2 * kStages + 12 + 3 * kSchedSlots;
    static constexpr int kSmemBytes = kOffBars + kNumBars * 8 + 16 + 16 + kWatchdogBytes;   // + TMEM slot + item ring + watchdog state (last 16 bytes)
    static constexpr uint32_t kColS = 0, kColDP = 128, kColDK = 256, kColDV = 384;
};

// The 128-row Q blocks of a backward work item in plan order, as RUNS: for every segment (Q partition u, local rows
// [begin, end)) and every query head of the GQA group, the consecutive blocks with at least one visible (query, key)
// pair.  Every role iterates the same runs; inside a run a step is just s0 += 128, so the per-step state is two
// registers and the segment bookkeeping (which may live in local memory) is touched once per run.
struct QWalk {
    const Geom& gm;
    const Seg* segs;
    int nseg, g, v, t0, head_kv;
    int si = -1, hh = 0, s_lo = 0, s_hi = 0, u = 0, urow = 0, off = 0;
    __device__ __forceinline__ QWalk(const Geom& gm_, const Seg* segs_, int nseg_, int g_, int v_, int t0_, int head_kv_)
        : gm(gm_), segs(segs_), nseg(nseg_), g(g_), v(v_), t0(t0_), head_kv(head_kv_) {}
    // next run: row-addressing index of Q partition u (plan.hpp q_row_part), query head h, first local query row s0, number of blocks n >= 1, causal offset off
    __device__ bool next_run(int& u_out, int& h_out, int& s0_out, int& n_out, int& off_out)
    {
        while (true) {
            if (si >= 0 && s_lo < s_hi && hh < gm.group) {
                u_out = urow; h_out = head_kv * gm.group + hh; s0_out = s_lo; n_out = (s_hi - s_lo) / kBlock; off_out = off;
                ++hh;
                return true;
            }
            if (++si >= nseg) return false;
            const Seg sg = segs[si];
            u = (g / gm.a) * gm.a + sg.part_local;
            urow = q_row_part(gm, u, sg.part_local);
            hh = 0;
            s_lo = sg.begin;
            s_hi = sg.end;
            off = 0x20000000;
            if (gm.causal) {
                off = causal_off(gm, u, v);
                const int x = t0 - off - (kBlock - 1);          // first query row that sees key t0 is t0 - off
                if (x > s_lo) s_lo = min(s_hi, ((x + kBlock - 1) / kBlock) * kBlock);
            }
        }
    }
    // total number of steps of the item (consumes the walk)
    __device__ int count_steps()
    {
        int total = 0, a, b, c, n, d;
        while (next_run(a, b, c, n, d)) total += n;
        return total;
    }
};
// One step forward over the runs: (u, h, off) change once per run, s0 advances by 128 inside it.
struct QStep {
    int u = 0, h = 0, s0 = 0, off = 0, left = 0;
    __device__ __forceinline__ bool next(QWalk& w)
    {
        if (left > 0) { s0 += kBlock; --left; return true; }
        int n;
        if (!w.next_run(u, h, s0, n, off)) return false;
        left = n - 1;
        return true;
    }
};

struct BwdItemCtx {
    BwdItem it;
    int g_local, g, v, vrow, nseg;
    const Seg* segs;
};

__device__ __forceinline__ BwdItemCtx load_bwd_item(const BwdParams& p, int idx)
{
    BwdItemCtx c;
    c.g_local = idx / p.items_per_gpu;
    c.it = p.items[idx - c.g_local * p.items_per_gpu];
    c.g = p.g_first + c.g_local;
    c.v = kv_partition(p.gm, c.g, c.it.kv_local);
    c.vrow = kv_row_part(p.gm, c.v, c.it.kv_local);
    const SegList sl = p.seglists[c.it.seglist];
    c.segs = p.segs + sl.offset;
    c.nseg = sl.count;
    return c;
}

__device__ __forceinline__ void bulk_load(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void red_add_v4(float* addr, float a, float b, float c, float d)
{
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(a), "f"(b), "f"(c), "f"(d) : "memory");
}
// TMA tensor reduction: global[tile at (c0..c3)] += smem tile (fp32), tracked by the thread's bulk async-group.  The dQ lines are hit again by
// every key block that sweeps the same query rows: evict_last keeps them in L2 (+0.3 % on C2 / C4, +0.15 % on C5, back to back)
__device__ __forceinline__ void tma_reduce_add_4d(const CUtensorMap* m, const void* smem_src, int c0, int c1, int c2, int c3)
{
    asm volatile("cp.reduce.async.bulk.tensor.4d.global.shared::cta.add.tile.bulk_group.L2::cache_hint [%0, {%2, %3, %4, %5}], [%1], %6;"
                 ::"l"(reinterpret_cast<uint64_t>(m)), "r"(smem_u32(smem_src)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(kEvictLast) : "memory");
}
// TMEM accumulator [128 lanes x D columns] -> x scale -> atomic add into a global row of D floats
// (item epilogue only: once per 128-key block)
template <int D> __device__ __forceinline__ void drain_rows(uint32_t taddr, float* grow, float scale, int dv)
{
#pragma unroll 1
    for (int ch = 0; ch < dv / 32; ++ch) {                  // dv = the tensors' head_dim (64: the upper accumulator columns are zero)
        uint32_t r[32];
        tmem_ld_x32(taddr + ch * 32, r);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 32; i += 4)
            red_add_v4(grow + ch * 32 + i, __uint_as_float(r[i]) * scale, __uint_as_float(r[i + 1]) * scale,
                       __uint_as_float(r[i + 2]) * scale, __uint_as_float(r[i + 3]) * scale);
    }
}

// kPair: the kernel runs as thread-block clusters of two CTAs that take work items 2k and 2k+1, which the planner has
// checked to walk the SAME sequence of Q blocks (BwdParams::pair).  Each CTA then loads only half of every Q / dO tile
// (64 rows) and the TMA multicasts it into both CTAs' shared memory, which halves the L2 -> SM tile traffic; a tile slot
// is released to both loaders (multicast tcgen05.commit) because either one writes into both CTAs.  tmQ / tmdO are then
// tensor maps with 64-row boxes.
//
// kPairMode 2 (kExch) -- the pair's dQ exchange.  Both CTAs hold a dQ^T contribution [128 d x 128 queries] for the SAME 128
// query rows (their key blocks differ).  Instead of adding both to global memory, each CTA keeps the half of its tile that
// belongs to "its" 64 queries (CTA rank r: queries 64r .. 64r+63 of the step) and sends the other half to its peer through
// distributed shared memory as bf16 (16 KB per step and direction; fp32 would be 32 KB, measured at ~10 B/clk: too slow,
// profiles/r01_v6_README.md); the receiver adds the peer's half to its own fp32 half and reduces 64 instead of 128 query
// rows into global dQ: HALF the L2 atomics per step, which is what bounds the kernel.  The exchanged half
// is rounded to bf16 (2^-9 relative, the precision the dS^T operand already has); precision = 1 plans do not use it.
// Drain thread d of CTA r holds dQ^T row d; element (d, query) travels from thread d to thread d of the peer, so the
// exchange buffer is addressed [octet of queries][d] x 16 bytes: conflict-free 512-byte warp stores (st.async, which also
// completes the receiver's transaction barrier) and loads.  `send_ok` is the receiver handing the buffer back.
template <int D, bool kSplit, int kPairMode>
__global__ void __launch_bounds__(kBwdThreads, 1)
tile_bwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmdO,
                const __grid_constant__ CUtensorMap tmdQ, const BwdParams p)
{
    constexpr bool kPair = kPairMode >= 1, kExch = kPairMode == 2;
    using Cfg = BwdCfg<D, kSplit, kExch>;
    extern __shared__ __align__(1024) uint8_t smem[];
    uint8_t* sK = smem + Cfg::kOffK;
    uint8_t* sV = smem + Cfg::kOffV;
    uint8_t* sDs = smem + Cfg::kOffDs;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cfg::kOffBars);
    uint64_t* kv_full = bars + 0;
    uint64_t* kv_empty = bars + 1;
    uint64_t* qd_full = bars + 2;                       // [kStages]
    uint64_t* qd_empty = qd_full + Cfg::kStages;        // [kStages]
    uint64_t* s_full = qd_empty + Cfg::kStages;
    uint64_t* p_full = s_full + 1;
    uint64_t* dp_full = s_full + 2;
    uint64_t* ds_full = s_full + 3;
    uint64_t* dq_full = s_full + 4;
    uint64_t* dq_empty = s_full + 5;
    uint64_t* dkv_full = s_full + 6;
    uint64_t* dkv_empty = s_full + 7;
    uint64_t* do_full = s_full + 8;
    uint64_t* do_empty = s_full + 9;
    uint64_t* send_ok = s_full + 10;                    // kExch: the peer's receive buffer is free for this step's half (remote arrive)
    uint64_t* recv_full = s_full + 11;                  // kExch: the peer's dQ^T half for this CTA's queries has landed in sRecv (transaction count)
    uint64_t* sched_full = s_full + 12;                 // [kSchedSlots] the scheduler warp has put the next work-item index into slot k
    uint64_t* sched_empty = sched_full + Cfg::kSchedSlots;   // [kSchedSlots] every role has read slot k
    uint64_t* peer_free = sched_empty + Cfg::kSchedSlots;    // [kSchedSlots] kPair, rank 0: the peer's slot k is armed for the next index
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(peer_free + Cfg::kSchedSlots);
    volatile int* sched_idx = reinterpret_cast<volatile int*>(tmem_slot + 4);
    uint8_t* sdO = smem + Cfg::kOffdO;
    float* sStg = reinterpret_cast<float*>(smem + Cfg::kOffStg);
    auto sQ = [&](int st) { return smem + Cfg::kOffQ + st * Cfg::kTileBytes; };
    auto sLse = [&](int st) { return reinterpret_cast<float*>(smem + Cfg::kOffVec + st * 1024); };
    auto sDelta = [&](int st) { return reinterpret_cast<float*>(smem + Cfg::kOffVec + st * 1024 + 512); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const Geom& gm = p.gm;
    const int total_items = p.items_per_gpu * p.g_count;
    const long long N = gm.rows_q;
    constexpr int kCompute = 2 * kBlock;                // threads of the two compute groups
    constexpr int kSchedReaders = 2 + kCompute + kBlock;   // threads that read every work-item index: producer, MMA issuer, compute groups, drain group

    if (smem_u32(smem) & 1023u) {                       // the 128-byte swizzle needs a 1024-byte aligned base: report, do not trap
        if (threadIdx.x == 0 && p.status != nullptr && atomicCAS_system(p.status, 0, 2) == 0) { p.status[1] = (int)blockIdx.x; __threadfence_system(); }
        return;
    }
    if (threadIdx.x == 0) {
        watchdog_init(p.status);
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmdO); prefetch_tmap(&tmdQ);
        mbar_init(kv_full, 1);
        mbar_init(kv_empty, 1);
        for (int s = 0; s < Cfg::kStages; ++s) { mbar_init(&qd_full[s], 1); mbar_init(&qd_empty[s], kPair ? 2 : 1); }
        mbar_init(s_full, 1);
        mbar_init(p_full, kCompute);
        mbar_init(dp_full, 1);
        mbar_init(ds_full, kCompute);
        mbar_init(dq_full, 1);
        mbar_init(dq_empty, kBlock);
        mbar_init(dkv_full, 1);
        mbar_init(dkv_empty, kCompute);
        mbar_init(do_full, 1);
        mbar_init(do_empty, kPair ? 2 : 1);
        mbar_init(recv_full, 1);
        mbar_init(send_ok, 1);
        for (int k = 0; k < Cfg::kSchedSlots; ++k) {
            mbar_init(&sched_full[k], 1);
            mbar_init(&sched_empty[k], kSchedReaders + ((kPair && cluster_ctarank() == 1) ? 1 : 0));   // rank 1's scheduler reads the ring too
            mbar_init(&peer_free[k], 1);
        }
        fence_mbar_init();
    }
    if (warp == 2) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    if constexpr (kPair) cluster_sync();                // the peer's barriers are initialised before anything is sent to them
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t pair_rank = kPair ? cluster_ctarank() : 0;

    // Work items are handed out DYNAMICALLY: the scheduler warp takes the next index (the next pair of indices, for a cluster)
    // from a global counter and publishes it through a ring in shared memory, which every role reads in order.  With the static
    // round-robin (item = blockIdx.x + k gridDim.x) the persistent CTAs, whose items differ in length under the causal mask, drift
    // apart by hundreds of items, and the Q / dO / dQ rows they stream stop being shared in L2 (profiles/r02_v1_README.md:
    // 55 % of the dQ reductions and 58 % of the tile loads of a BASELINE.json configs[4] launch miss L2); taking items in list
    // order keeps every running CTA inside the same ~148 consecutive items.
    uint32_t sc_slot = 0, sc_phase = 0;
    auto next_item = [&]() -> int {
        if constexpr (kPair) mbar_wait_cluster(&sched_full[sc_slot], sc_phase);   // rank 1's index arrives from the peer (st.async)
        else mbar_wait(&sched_full[sc_slot], sc_phase);
        const int v = sched_idx[sc_slot];
        mbar_arrive(&sched_empty[sc_slot]);
        if (++sc_slot == Cfg::kSchedSlots) { sc_slot = 0; sc_phase ^= 1; }
        return v;
    };

    if (warp < 4) reg_dealloc<kCtrlRegs>();
    if (warp == 3) {
        // =============================== work-item scheduler ===============================
        if (elect_one()) {
            if (!kPair || pair_rank == 0) {
                const uint32_t peer_idx = kPair ? mapa(smem_u32(const_cast<int*>(sched_idx)), 1u) : 0u;
                const uint32_t peer_full = kPair ? mapa(smem_u32(sched_full), 1u) : 0u;
                uint32_t slot = 0, phase = 0;
                while (true) {
                    mbar_wait(&sched_empty[slot], phase ^ 1);                    // the slot's previous index has been read by every role
                    if constexpr (kPair) mbar_wait(&peer_free[slot], phase);     // ... and the peer's slot is armed
                    const int v = atomicAdd(p.counter, kPair ? 2 : 1);
                    sched_idx[slot] = v;
                    mbar_arrive(&sched_full[slot]);
                    if constexpr (kPair)                                         // the peer takes the odd item of the pair
                        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.b32 [%0], %1, [%2];"
                                     ::"r"(peer_idx + slot * 4), "r"(v + 1), "r"(peer_full + slot * 8) : "memory");
                    if (v >= total_items) break;
                    if (++slot == Cfg::kSchedSlots) { slot = 0; phase ^= 1; }
                }
            } else {
                // rank 1: arm a slot (expect the 4 bytes of the index), tell rank 0, and follow the ring like every other role to
                // learn when it ends
                const uint32_t r0_free = mapa(smem_u32(peer_free), 0u);
                for (int k = 0; k < Cfg::kSchedSlots; ++k) { mbar_expect_tx(&sched_full[k], 4); mbar_arrive_remote(r0_free + k * 8); }
                uint32_t slot = 0, phase = 0;
                while (true) {
                    const int v = next_item();
                    if (v >= total_items) break;
                    mbar_wait(&sched_empty[slot], phase);                        // every role has read it: arm the slot again
                    mbar_expect_tx(&sched_full[slot], 4);
                    mbar_arrive_remote(r0_free + slot * 8);
                    if (++slot == Cfg::kSchedSlots) { slot = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 0) {
        // =============================== TMA producer ===============================
        if (elect_one()) {
            uint32_t stage = 0, ring_phase = 0, kv_phase = 0, do_ph = 0;
            const float* nlse = p.ws + p.ws_plane;                            // ws[1] = log2(scale) - lse*log2e
            for (int idx = next_item(); idx < total_items; idx = next_item()) {
                const BwdItemCtx c = load_bwd_item(p, idx);
                QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
                QStep q;
                bool first = true;
                while (q.next(walk)) {
                    const int u = q.u, h = q.h, s0 = q.s0;
                    if (first) {
                        first = false;
                        mbar_wait(kv_empty, kv_phase ^ 1);
                        kv_phase ^= 1;
                        mbar_expect_tx(kv_full, 2 * Cfg::kTileBytes);
                        for (int bx = 0; bx < Cfg::kBoxes; ++bx) {
                            tma_load_4d(sK + bx * (kBlock * 128), &tmK, kv_full, bx * 64, c.it.head_kv, c.vrow * gm.L + c.it.t0, c.it.batch, kEvictFirst);
                            tma_load_4d(sV + bx * (kBlock * 128), &tmV, kv_full, bx * 64, c.it.head_kv, c.vrow * gm.L + c.it.t0, c.it.batch, kEvictFirst);
                        }
                    }
                    mbar_wait(&qd_empty[stage], ring_phase ^ 1);
                    mbar_expect_tx(&qd_full[stage], Cfg::kTileBytes + 1024);
                    const int row = u * gm.L + s0;
                    for (int bx = 0; bx < Cfg::kBoxes; ++bx) {
                        if constexpr (kPair)
                            tma_load_4d_mc(sQ(stage) + bx * (kBlock * 128) + pair_rank * (64 * 128), &tmQ, &qd_full[stage], bx * 64, h,
                                           row + pair_rank * 64, c.it.batch, 3, kEvictLast);
                        else
                            tma_load_4d(sQ(stage) + bx * (kBlock * 128), &tmQ, &qd_full[stage], bx * 64, h, row, c.it.batch, kEvictLast);
                    }
                    const size_t vec = (size_t)c.it.batch * p.vec_stride_b + (size_t)h * N + row;
                    bulk_load(sLse(stage), nlse + vec, 512, &qd_full[stage]);
                    bulk_load(sDelta(stage), p.ws + vec, 512, &qd_full[stage]);
                    if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                    mbar_wait(do_empty, do_ph ^ 1);      // dV of the previous step has consumed the dO tile
                    do_ph ^= 1;
                    mbar_expect_tx(do_full, Cfg::kTileBytes);
                    for (int bx = 0; bx < Cfg::kBoxes; ++bx) {
                        if constexpr (kPair)
                            tma_load_4d_mc(sdO + bx * (kBlock * 128) + pair_rank * (64 * 128), &tmdO, do_full, bx * 64, h, row + pair_rank * 64,
                                           c.it.batch, 3, kEvictLast);
                        else
                            tma_load_4d(sdO + bx * (kBlock * 128), &tmdO, do_full, bx * 64, h, row, c.it.batch, kEvictLast);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =============================== MMA issuer ===============================
        if (elect_one()) {
            constexpr uint32_t idesc_kk = umma_idesc(kBlock, kBlock, false, false);   // S^T, dP^T: both operands K-major over head_dim
            constexpr uint32_t idesc_tn = umma_idesc(kBlock, D, false, true);         // dV (A in TMEM), dK (A smem K-major); B row-major [q x d]
            constexpr uint32_t idesc_nn = umma_idesc(D, kBlock, true, true);          // dQ^T: A = K tile M-major, B = dS^T N-major
            uint32_t stage = 0, ring_phase = 0, kv_phase = 0, p_ph = 0, ds_ph = 0, dqe_ph = 0, dkve_ph = 0, do_ph = 0;
            PT_DECL;
            const uint32_t aK = smem_u32(sK), aV = smem_u32(sV), aDs = smem_u32(sDs), adO = smem_u32(sdO);
            auto issue_dP = [&]() {                                                  // dP^T = V dO^T once the step's dO tile landed
                mbar_wait(do_full, do_ph);
                do_ph ^= 1;
                tc_fence_after();
                // the k-loops of the five MMAs are unrolled by 2, not 8: the issuer's warp sat at instruction fetch in 21 % of its ncu samples
                // (four roles share an SM sub-partition's instruction cache); measured 8 / 4 / 2 / 1: tile_bwd C2 1031 / 1026 / 1039 / 1015 TFLOP/s
#pragma unroll 2
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t o = (kk / 4) * (kBlock * 128) + (kk % 4) * 32;
                    umma_ss(tmem + Cfg::kColDP, umma_desc(aV + o, 16, 1024), umma_desc(adO + o, 16, 1024), idesc_kk, kk > 0);
                }
                umma_commit(dp_full);
            };
            auto mma_kmajor = [&](uint32_t dcol, uint32_t a, uint32_t b) {          // D = A B^T, both K-major over head_dim
#pragma unroll 2
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t o = (kk / 4) * (kBlock * 128) + (kk % 4) * 32;
                    umma_ss(tmem + dcol, umma_desc(a + o, 16, 1024), umma_desc(b + o, 16, 1024), idesc_kk, kk > 0);
                }
            };
            auto next_stage = [&]() {                                                // wait for the next Q/dO stage, return its slot
                mbar_wait(&qd_full[stage], ring_phase);
                tc_fence_after();
                const uint32_t st = stage;
                if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                return st;
            };
            for (int idx = next_item(); idx < total_items; idx = next_item()) {
                const BwdItemCtx c = load_bwd_item(p, idx);
                QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
                const int nsteps = walk.count_steps();
                if (nsteps == 0) continue;
                int i = 0;
                bool have = true;
                mbar_wait(kv_full, kv_phase);
                kv_phase ^= 1;
                mbar_wait(dkv_empty, dkve_ph ^ 1);      // previous item's dK/dV drained from TMEM
                dkve_ph ^= 1;
                uint32_t st_cur = next_stage();         // prologue: S^T(0), dP^T(0)
                mma_kmajor(Cfg::kColS, aK, smem_u32(sQ(st_cur)));
                umma_commit(s_full);
                issue_dP();
                while (have) {
                    const bool more = i + 1 < nsteps;
                    const uint32_t aQ = smem_u32(sQ(st_cur));
                    PT_MARK(0);
                    // dV += P^T dO   (P^T bf16 in TMEM: group w's 64 queries at columns 64w.. (hi) and 64w+32.. (lo))
                    mbar_wait(p_full, p_ph);
                    p_ph ^= 1;
                    tc_fence_after();
                    PT_MARK(1);
#pragma unroll
                    for (int x = 0; x < Cfg::kNumDs; ++x)
#pragma unroll 2
                        for (int kk = 0; kk < kBlock / 16; ++kk)
                            umma_ts(tmem + Cfg::kColDV, tmem + Cfg::kColS + (kk >> 2) * 64 + x * 32 + (kk & 3) * 8,
                                    umma_desc(adO + kk * 2048, kBlock * 128, 1024), idesc_tn, (i > 0 || kk > 0 || x > 0) ? 1u : 0u);
                    if constexpr (kPair) umma_commit_mc(do_empty, 3);      // the dO tile may be refilled for the next step
                    else umma_commit(do_empty);
                    uint32_t st_next = 0;
                    if (Cfg::kStages > 1 && more) {      // S^T(i+1) as early as possible: P^T(i+1) is computed under this step's MMAs
                        st_next = next_stage();
                        mma_kmajor(Cfg::kColS, aK, smem_u32(sQ(st_next)));
                        umma_commit(s_full);
                    }
                    // dQ^T = K^T dS^T first: the drain group empties it while dK += dS^T Q runs, so dP^T(i+1), which reuses its
                    // TMEM columns, is not held up (the Q ring has its own two stages, so releasing Q a little later costs nothing)
                    PT_MARK(2);
                    mbar_wait(ds_full, ds_ph);
                    ds_ph ^= 1;
                    tc_fence_after();
                    PT_MARK(3);
                    auto issue_dq = [&]() {
#pragma unroll
                        for (int x = 0; x < Cfg::kNumDs; ++x)
#pragma unroll 2
                            for (int kk = 0; kk < kBlock / 16; ++kk)
                                umma_ss(tmem + Cfg::kColDP, umma_desc(aK + kk * 2048, kBlock * 128, 1024),
                                        umma_desc(aDs + x * Cfg::kDsBytes + kk * 2048, kBlock * 128, 1024), idesc_nn, (kk > 0 || x > 0) ? 1u : 0u);
                        umma_commit(dq_full);
                    };
                    auto issue_dk = [&]() {
#pragma unroll
                        for (int x = 0; x < Cfg::kNumDs; ++x)
#pragma unroll 2
                            for (int kk = 0; kk < kBlock / 16; ++kk)
                                umma_ss(tmem + Cfg::kColDK, umma_desc(aDs + x * Cfg::kDsBytes + (kk / 4) * (kBlock * 128) + (kk % 4) * 32, 16, 1024),
                                        umma_desc(aQ + kk * 2048, kBlock * 128, 1024), idesc_tn, (i > 0 || kk > 0 || x > 0) ? 1u : 0u);
                        if constexpr (kPair) umma_commit_mc(&qd_empty[st_cur], 3);
                        else umma_commit(&qd_empty[st_cur]);
                    };
                    if constexpr (Cfg::kStages == 1) {   // single Q stage (hi+lo operands): dK first, it is what releases the stage, so that
                        issue_dk();                      // Q(i+1) is loaded under the two dQ^T MMAs instead of after them
                        issue_dq();
                    } else {
                        issue_dq();
                        issue_dk();
                    }
                    if (Cfg::kStages == 1 && more) {     // single stage: Q(i+1) can only land once dK(i) released the stage
                        st_next = next_stage();
                        mma_kmajor(Cfg::kColS, aK, smem_u32(sQ(st_next)));
                        umma_commit(s_full);
                    }
                    PT_MARK(4);
                    if (more) {                          // dP^T(i+1) once dQ^T(i) has left TMEM
                        mbar_wait(dq_empty, dqe_ph);
                        dqe_ph ^= 1;
                        tc_fence_after();
                        PT_MARK(5);
                        issue_dP();
                    } else {
                        umma_commit(dkv_full);
                        umma_commit(kv_empty);
                        mbar_wait(dq_empty, dqe_ph);     // keep the phase bookkeeping aligned
                        dqe_ph ^= 1;
                    }
                    st_cur = st_next;
                    have = more;
                    ++i;
                }
            }
            PT_REPORT("bwd MMA thread clocks per step: wait_p, issue dV+S(next), wait_ds, issue dK+dQ, wait_dq_empty (loop-back = issue dP)");
        }
    } else if (warp >= 4 && warp < 12) {
        // =============================== compute groups ===============================
        // thread = (key row `row` = TMEM lane, query-column half `wg`): 64 elements of S^T / dP^T per step
        reg_alloc<kComputeRegs>();
        const int wg = (warp - 4) >> 2;
        const int row = ((warp & 3) << 5) | lane;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + lane_base + Cfg::kColS + wg * 64;      // S^T columns of this half; P^T (bf16) is written over them
        const uint32_t tDP = tmem + lane_base + Cfg::kColDP + wg * 64;    // dP^T columns of this half; later dQ^T (lane = d, column = query)
        uint8_t* sDsHalf = sDs + wg * (kBlock * 128);                     // [128 key rows][64 queries] bf16, 128-byte swizzled rows
        uint32_t stage = 0, ring_phase = 0, s_ph = 0, dp_ph = 0, dq_ph = 0, dkv_ph = 0;
        float pr[64];                                                     // P^T of the current step (fp32), reused for dS^T
        const f32x2 c22 = pack2(gm.scale_log2, gm.scale_log2);
        PT_DECL;

        auto next_stage = [&]() {
            mbar_wait(&qd_full[stage], ring_phase);                       // Q/dO tiles and the -lse*log2e / delta vectors landed
            const uint32_t st = stage;
            if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
            return st;
        };
        // P^T = scale * exp2(S^T * scale*log2e - lse*log2e) (the offset in smem is log2(scale) - lse*log2e), causal mask on
        // blocks that straddle the diagonal only
        auto compute_P = [&](uint32_t st, int t0, int s0, int off) {
            const float4* nl4 = reinterpret_cast<const float4*>(sLse(st) + wg * 64);
            const bool masked = gm.causal && (t0 + kBlock - 1 - off - s0 > 0);     // block-uniform
            mbar_wait(s_full, s_ph);
            s_ph ^= 1;
            tc_fence_after();
            PT_MARK(3);
            if (kAblate & 1) { tc_fence_before(); mbar_arrive(p_full); return; }
            uint32_t(&pu)[64] = reinterpret_cast<uint32_t(&)[64]>(pr);      // S^T lands in the registers P^T is computed in
            tmem_ld_x32(tS, *reinterpret_cast<uint32_t(*)[32]>(&pu[0]));
            tmem_ld_x32(tS + 32, *reinterpret_cast<uint32_t(*)[32]>(&pu[32]));
            tmem_ld_wait();
#pragma unroll
            for (int q4 = 0; q4 < 64; q4 += 4) {
                const float4 l4 = nl4[q4 / 4];
                float x0, x1, x2, x3;
                unpack2(fma2(pack2(pr[q4 + 0], pr[q4 + 1]), c22, pack2(l4.x, l4.y)), x0, x1);
                unpack2(fma2(pack2(pr[q4 + 2], pr[q4 + 3]), c22, pack2(l4.z, l4.w)), x2, x3);
                // kBwdPolyOf4 of every 4 exponentials on the FMA pipe, the rest on the MUFU (x <= 0 here: P <= scale)
                pr[q4 + 0] = (0 < kBwdPolyOf4) ? ex2_poly(x0) : ex2(x0);
                pr[q4 + 1] = (1 < kBwdPolyOf4) ? ex2_poly(x1) : ex2(x1);
                pr[q4 + 2] = (2 < kBwdPolyOf4) ? ex2_poly(x2) : ex2(x2);
                pr[q4 + 3] = (3 < kBwdPolyOf4) ? ex2_poly(x3) : ex2(x3);
            }
            if (masked) {
                const int cmin = t0 + row - off - s0 - wg * 64;            // local query column c visible to this key iff c >= cmin
#pragma unroll
                for (int c = 0; c < 64; ++c) if (c < cmin) pr[c] = 0.f;
            }
            // all 64 S^T columns of this half are in registers: P^T may now overwrite them
            if constexpr (!kSplit) {
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    uint32_t pk[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) pk[j] = pack_bf16x2(pr[hf * 32 + 2 * j], pr[hf * 32 + 2 * j + 1]);
                    tmem_st_x16(tS + hf * 16, pk);
                }
            } else {
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    uint32_t hi[16], lo[16];
#pragma unroll
                    for (int j = 0; j < 16; ++j) split_bf16x2(pr[hf * 32 + 2 * j], pr[hf * 32 + 2 * j + 1], hi[j], lo[j]);
                    tmem_st_x16(tS + hf * 16, hi);
                    tmem_st_x16(tS + 32 + hf * 16, lo);
                }
            }
            tmem_st_wait();
            tc_fence_before();
            mbar_arrive(p_full);
        };
        // dS^T = P^T o (dP^T - delta) -> bf16 -> smem (K-major rows for dK, read N-major for dQ^T)
        auto compute_dS = [&](uint32_t st) {
            const float4* dl4 = reinterpret_cast<const float4*>(sDelta(st) + wg * 64);
            mbar_wait(dp_full, dp_ph);           // also: dQ^T / dK of the previous step have finished reading the dS tile
            dp_ph ^= 1;
            tc_fence_after();
            PT_MARK(1);
            if (kAblate & 1) { tc_fence_before(); mbar_arrive(ds_full); return; }
            uint32_t ra[16], rb[16];             // 16-column chunks: chunk c+1 is in flight while chunk c is processed
            // delta of the NEXT 8 columns is loaded while the current 8 are computed: the shared memory is busy with the MMAs' operand
            // reads and a broadcast ld.shared takes ~80 clocks here (ncu: 12 % of a compute warp's samples sat at the first use of it)
            float4 da_next = dl4[0], db_next = dl4[1];
            auto ds_chunk = [&](int c16, const uint32_t (&r)[16]) {
#pragma unroll
                for (int k = 0; k < 2; ++k) {                              // 8 columns = one 16-byte chunk of the row
                    const float4 da = da_next, db = db_next;
                    if (c16 * 2 + k < 7) { da_next = dl4[c16 * 4 + k * 2 + 2]; db_next = dl4[c16 * 4 + k * 2 + 3]; }
                    const int c = c16 * 16 + k * 8;
                    float d0, d1, d2, d3, d4, d5, d6, d7;        // dS = P o (dP - delta), two elements per instruction
                    unpack2(mul2(pack2(pr[c + 0], pr[c + 1]), add2(pack2(__uint_as_float(r[k * 8 + 0]), __uint_as_float(r[k * 8 + 1])), pack2(-da.x, -da.y))), d0, d1);
                    unpack2(mul2(pack2(pr[c + 2], pr[c + 3]), add2(pack2(__uint_as_float(r[k * 8 + 2]), __uint_as_float(r[k * 8 + 3])), pack2(-da.z, -da.w))), d2, d3);
                    unpack2(mul2(pack2(pr[c + 4], pr[c + 5]), add2(pack2(__uint_as_float(r[k * 8 + 4]), __uint_as_float(r[k * 8 + 5])), pack2(-db.x, -db.y))), d4, d5);
                    unpack2(mul2(pack2(pr[c + 6], pr[c + 7]), add2(pack2(__uint_as_float(r[k * 8 + 6]), __uint_as_float(r[k * 8 + 7])), pack2(-db.z, -db.w))), d6, d7);
                    const uint32_t o = sw128_offset(row, c16 * 2 + k);
                    if constexpr (!kSplit) {
                        *reinterpret_cast<uint4*>(sDsHalf + o) =
                            make_uint4(pack_bf16x2(d0, d1), pack_bf16x2(d2, d3), pack_bf16x2(d4, d5), pack_bf16x2(d6, d7));
                    } else {
                        uint32_t h0, h1, h2, h3, l0, l1, l2, l3;
                        split_bf16x2(d0, d1, h0, l0); split_bf16x2(d2, d3, h1, l1);
                        split_bf16x2(d4, d5, h2, l2); split_bf16x2(d6, d7, h3, l3);
                        *reinterpret_cast<uint4*>(sDsHalf + o) = make_uint4(h0, h1, h2, h3);
                        *reinterpret_cast<uint4*>(sDsHalf + Cfg::kDsBytes + o) = make_uint4(l0, l1, l2, l3);
                    }
                }
            };
            tmem_ld_x16(tDP, ra);
            tmem_ld_wait();
            PT_MARK(5);
            tmem_ld_x16(tDP + 16, rb);
            ds_chunk(0, ra);
            tmem_ld_wait();
            tmem_ld_x16(tDP + 32, ra);
            ds_chunk(1, rb);
            tmem_ld_wait();
            tmem_ld_x16(tDP + 48, rb);
            ds_chunk(2, ra);
            tmem_ld_wait();
            ds_chunk(3, rb);
            PT_MARK(6);
            fence_proxy_async_smem();
            tc_fence_before();
            mbar_arrive(ds_full);
        };
        for (int idx = next_item(); idx < total_items; idx = next_item()) {
            const BwdItemCtx c = load_bwd_item(p, idx);
            QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
            QStep q;
            bool have = q.next(walk);
            if (!have) continue;
            uint32_t st_cur = next_stage();
            compute_P(st_cur, c.it.t0, q.s0, q.off);
            while (have) {
                const bool more = q.next(walk);              // q now describes step i+1 (dS^T(i) needs nothing of step i)
                PT_MARK(0);
                compute_dS(st_cur);
                PT_MARK(2);
                if (more) {
                    st_cur = next_stage();
                    compute_P(st_cur, c.it.t0, q.s0, q.off);
                }
                PT_MARK(4);
                have = more;
            }
            // epilogue: group 0 drains dK (x softmax scale), group 1 drains dV
            mbar_wait(dkv_full, dkv_ph);
            dkv_ph ^= 1;
            tc_fence_after();
            float* grow = (wg == 0 ? p.dK : p.dV) + (size_t)c.it.batch * p.k_stride_b + ((size_t)c.vrow * gm.L + c.it.t0 + row) * p.k_stride_row +
                          (size_t)c.it.head_kv * p.k_stride_h;
            drain_rows<D>(tmem + lane_base + (wg == 0 ? Cfg::kColDK : Cfg::kColDV), grow, wg == 0 ? 1.0f : 1.0f / gm.scale, gm.head_dim);
            tc_fence_before();
            mbar_arrive(dkv_empty);
        }
        PT_REPORT("bwd compute clocks per step: wait dP, fence+arrive(ds), wait S, P, first dP ld, dS chunks, 0");
    }
    else if (warp >= 12) {
        // =============================== dQ drain group ===============================
        // thread = head-dim index d (TMEM lane): dQ^T row d, all 128 queries of the step -> registers (the TMEM columns are
        // released at once) -> shared-memory staging (a ring of four [16 queries][128 d] fp32 buffers) -> one
        // cp.reduce.async.bulk.tensor (add.f32) per 16-query slice, up to three in flight while the next slice is written.  The TMA engine does the L2 atomics at the same rate as
        // red.global (6.1 vs 6.4 TB/s measured) but no instruction of it goes through the SM's load/store queue, where
        // 512 reds per step used to delay every tcgen05.ld / ld.shared / st.shared of the compute warps by hundreds of clocks.
        reg_alloc<kDrainRegs>();
        const int d = ((warp & 3) << 5) | lane;
        const uint32_t tDQ = tmem + ((uint32_t)((warp & 3) * 32) << 16) + Cfg::kColDP;
        const bool issuer = threadIdx.x == 12 * 32;
        const int dv = gm.head_dim;                      // 64: dQ^T rows 64..127 are zero and stay in the CTA
        uint32_t dq_ph = 0;
        // kExch: this CTA reduces queries own0 .. own0+63 of every step and sends the others to the peer
        const uint32_t own0 = kExch ? pair_rank * (kBlock / 2) : 0, peer0 = kBlock / 2 - own0;
        const uint8_t* sRecv = smem + Cfg::kOffRecv;
        const uint32_t my_slot = (uint32_t)d * 16u;                                       // + octet * (D * 16)
        const uint32_t peer_recv = kExch ? mapa(smem_u32(sRecv), pair_rank ^ 1u) + my_slot : 0u;
        const uint32_t peer_recv_full = kExch ? mapa(smem_u32(recv_full), pair_rank ^ 1u) : 0u;
        constexpr int kSlices = Cfg::kDrainRows / Cfg::kStgRows;
        const uint32_t peer_send_ok = kExch ? mapa(smem_u32(send_ok), pair_rank ^ 1u) : 0u;
        uint32_t rf_ph = 0, sok_ph = 0;
        PT_DECL;
        for (int idx = next_item(); idx < total_items; idx = next_item()) {
            const BwdItemCtx c = load_bwd_item(p, idx);
            QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
            QStep q;
            while (q.next(walk)) {
                PT_MARK(0);
                if (kAblate & 2) {
                    mbar_wait(dq_full, dq_ph);
                    dq_ph ^= 1;
                    tc_fence_after();
                    tc_fence_before();
                    mbar_arrive(dq_empty);
                    continue;
                }
                if constexpr (kExch) {
                    // One step of the exchange (see the kernel's header comment).  The staging memory is used twice per step: its
                    // first half receives the peer's bf16 half, then all of it holds this CTA's 64 fp32 rows, reduced as kSlices
                    // boxes in bulk groups of their own, the first-half boxes first.  The TMA works on them during the next step's
                    // load / send / wait, so this group never waits for a reduce it has just issued.
                    if (issuer) mbar_expect_tx(recv_full, Cfg::kRecvBytes);      // what the peer will send for this step
                    mbar_wait(dq_full, dq_ph);
                    dq_ph ^= 1;
                    tc_fence_after();
                    uint32_t r[kBlock / 2], rp[kBlock / 2];      // this CTA's / the peer's query columns of dQ^T row d
                    tmem_ld_x32(tDQ + peer0, *reinterpret_cast<uint32_t(*)[32]>(&rp[0]));
                    tmem_ld_x32(tDQ + peer0 + 32, *reinterpret_cast<uint32_t(*)[32]>(&rp[32]));
                    tmem_ld_x32(tDQ + own0, *reinterpret_cast<uint32_t(*)[32]>(&r[0]));
                    tmem_ld_x32(tDQ + own0 + 32, *reinterpret_cast<uint32_t(*)[32]>(&r[32]));
                    tmem_ld_wait();
                    tc_fence_before();
                    mbar_arrive(dq_empty);           // TMEM columns free again: dP^T of the next step may start
                    PT_MARK(1);
                    if (issuer) {                    // the previous step's first-half boxes have been read: the peer may send into that half
                        // (head_dim 64: the staged rows are half as long, all of them lie in the receive area: wait for every box)
                        if (dv == D) asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(kSlices / 2) : "memory");
                        else asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
                        mbar_arrive_remote(peer_send_ok);
                    }
                    mbar_wait(send_ok, sok_ph);      // ... and the peer's first half is free for this CTA's data
                    sok_ph ^= 1;
#pragma unroll
                    for (int o = 0; o < kBlock / 16; ++o)        // 8 queries = 16 bytes of bf16 per store
                        st_async_v4(peer_recv + o * (D * 16),
                                    pack_bf16x2(__uint_as_float(rp[8 * o + 0]), __uint_as_float(rp[8 * o + 1])),
                                    pack_bf16x2(__uint_as_float(rp[8 * o + 2]), __uint_as_float(rp[8 * o + 3])),
                                    pack_bf16x2(__uint_as_float(rp[8 * o + 4]), __uint_as_float(rp[8 * o + 5])),
                                    pack_bf16x2(__uint_as_float(rp[8 * o + 6]), __uint_as_float(rp[8 * o + 7])), peer_recv_full);
                    PT_MARK(2);
                    mbar_wait_cluster(recv_full, rf_ph);         // the peer's half for this CTA's queries has landed: add it
                    rf_ph ^= 1;
                    PT_MARK(3);
#pragma unroll
                    for (int o = 0; o < kBlock / 16; ++o) {
                        const uint4 w = *reinterpret_cast<const uint4*>(sRecv + o * (D * 16) + my_slot);
                        r[8 * o + 0] = __float_as_uint(__uint_as_float(r[8 * o + 0]) + __uint_as_float(w.x << 16));
                        r[8 * o + 1] = __float_as_uint(__uint_as_float(r[8 * o + 1]) + __uint_as_float(w.x & 0xffff0000u));
                        r[8 * o + 2] = __float_as_uint(__uint_as_float(r[8 * o + 2]) + __uint_as_float(w.y << 16));
                        r[8 * o + 3] = __float_as_uint(__uint_as_float(r[8 * o + 3]) + __uint_as_float(w.y & 0xffff0000u));
                        r[8 * o + 4] = __float_as_uint(__uint_as_float(r[8 * o + 4]) + __uint_as_float(w.z << 16));
                        r[8 * o + 5] = __float_as_uint(__uint_as_float(r[8 * o + 5]) + __uint_as_float(w.z & 0xffff0000u));
                        r[8 * o + 6] = __float_as_uint(__uint_as_float(r[8 * o + 6]) + __uint_as_float(w.w << 16));
                        r[8 * o + 7] = __float_as_uint(__uint_as_float(r[8 * o + 7]) + __uint_as_float(w.w & 0xffff0000u));
                    }
                    PT_MARK(4);
                    if (issuer) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the previous step's second-half boxes too
                    named_bar_sync(1, kBlock);       // every thread has consumed the received half: the sums may be staged over it
#pragma unroll
                    for (int j = 0; j < kBlock / 2; ++j)
                        if (d < dv) sStg[j * dv + d] = __uint_as_float(r[j]);
                    fence_proxy_async_smem();
                    named_bar_sync(1, kBlock);
                    if (issuer) {
#pragma unroll
                        for (int k = 0; k < kSlices; ++k) {
                            tma_reduce_add_4d(&tmdQ, sStg + k * (Cfg::kStgRows * dv), 0, q.h, q.u * gm.L + q.s0 + (int)own0 + k * Cfg::kStgRows, c.it.batch);
                            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                        }
                    }
                } else {
                    mbar_wait(dq_full, dq_ph);
                    dq_ph ^= 1;
                    tc_fence_after();
                    uint32_t r[kBlock];
#pragma unroll
                    for (int ch = 0; ch < kBlock / 32; ++ch) tmem_ld_x32(tDQ + ch * 32, *reinterpret_cast<uint32_t(*)[32]>(&r[ch * 32]));
                    tmem_ld_wait();
                    tc_fence_before();
                    mbar_arrive(dq_empty);               // TMEM columns free again: dP^T of the next step may start
                    PT_MARK(1);
#pragma unroll
                    for (int k = 0; k < kSlices; ++k) {   // 16-query slice k through staging buffer k % kStgBufs
                        float* stg = sStg + (k % Cfg::kStgBufs) * (Cfg::kStgRows * D);      // rows of dv floats (the reduce's box)
                        if (issuer) asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(Cfg::kStgBufs - 1) : "memory");   // slice k - kStgBufs has been read
                        named_bar_sync(1, kBlock);
#pragma unroll
                        for (int j = 0; j < Cfg::kStgRows; ++j)
                            if (d < dv) stg[j * dv + d] = __uint_as_float(r[k * Cfg::kStgRows + j]);
                        fence_proxy_async_smem();
                        named_bar_sync(1, kBlock);
                        if (issuer) {
                            tma_reduce_add_4d(&tmdQ, stg, 0, q.h, q.u * gm.L + q.s0 + k * Cfg::kStgRows, c.it.batch);
                            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                        }
                    }
                }
                PT_MARK(5);
            }
        }
        if (issuer) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");       // every reduce has landed before the CTA exits
        PT_REPORT("bwd drain clocks per step: wait dQ + ld, wait send_ok + send, wait recv, add, staging + TMA reduce (no exchange: wait dQ + ld, 0, 0, 0, staging)");
    }

    tc_fence_before();
    __syncthreads();
    if constexpr (kPair) cluster_sync();                // no CTA leaves while its peer may still write into it or arrive on its barriers
    if (warp == 2) tmem_dealloc<512>(tmem);
}

template <int D, bool kSplit, int kPairMode>
int launch_one(const BwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV, const CUtensorMap& tmdO,
               const CUtensorMap& tmdQ, int grid, cudaStream_t stream)
{
    using Cfg = BwdCfg<D, kSplit, kPairMode == 2>;
    static_assert(Cfg::kSmemBytes <= 227 * 1024, "tile_bwd shared memory over the 227 KB CTA limit");
    auto kernel = tile_bwd_kernel<D, kSplit, kPairMode>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes);
    if (e != cudaSuccess) return (int)e;
    cudaLaunchConfig_t cfg{};
    cfg.blockDim = dim3(kBwdThreads);
    cfg.dynamicSmemBytes = Cfg::kSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    if (kPairMode) {
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        // co-resident 2-CTA clusters of this kernel (GPCs with an odd SM count leave one SM out), cached per device
        constexpr int kMaxDevices = 64;
        static std::atomic<int> max_clusters[kMaxDevices];      // 0 = not queried yet, else count + 1
        int dev = 0;
        e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return (int)e;
        int n = (dev >= 0 && dev < kMaxDevices) ? max_clusters[dev].load(std::memory_order_relaxed) - 1 : -1;
        if (n < 0) {
            cfg.gridDim = dim3(2);
            e = cudaOccupancyMaxActiveClusters(&n, kernel, &cfg);
            if (e != cudaSuccess) return (int)e;
            if (dev >= 0 && dev < kMaxDevices) max_clusters[dev].store(n + 1, std::memory_order_relaxed);
        }
        if (n <= 0) return (int)cudaErrorLaunchOutOfResources;
        grid = (grid / 2 < n ? grid / 2 : n) * 2;
    }
    cfg.gridDim = dim3(grid);
    e = cudaLaunchKernelEx(&cfg, kernel, tmQ, tmK, tmV, tmdO, tmdQ, p);
    return e != cudaSuccess ? (int)e : (int)cudaGetLastError();
}

}  // namespace

int launch_tile_bwd(const BwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV, const CUtensorMap& tmdO,
                    const CUtensorMap& tmdQ, int num_sms, cudaStream_t stream)
{
    // head_dim 64 runs the head_dim-128 kernel: the TMA zero-fills the out-of-bounds upper 64 columns of every tile
    if (p.gm.head_dim != 128 && p.gm.head_dim != 64) return (int)cudaErrorNotSupported;
    const int total = p.items_per_gpu * p.g_count;
    if (total <= 0) return 0;
    const int grid = total < num_sms ? total : num_sms;
    if (p.pair == 2 && !p.split) return launch_one<128, false, 2>(p, tmQ, tmK, tmV, tmdO, tmdQ, grid, stream);
    if (p.pair)
        return p.split ? launch_one<128, true, 1>(p, tmQ, tmK, tmV, tmdO, tmdQ, grid, stream)
                       : launch_one<128, false, 1>(p, tmQ, tmK, tmV, tmdO, tmdQ, grid, stream);
    return p.split ? launch_one<128, true, 0>(p, tmQ, tmK, tmV, tmdO, tmdQ, grid, stream)
                   : launch_one<128, false, 0>(p, tmQ, tmK, tmV, tmdO, tmdQ, grid, stream);
}

}  // namespace mesh_attn
