// tile_fwd.cu -- mesh_attn_tile_fwd: blockwise softmax attention of a simulated GPU's tile
// (Alg.2 l.3-5, L171-173; per-pair form O_ij, lse_ij = Attention(Q_i, K_j, V_j), L81-84).
//
// One persistent CTA per SM walks the work list.  A work item is up to two 128-row Q
// sub-tiles of one (simulated GPU g, Q partition u, head); the CTA streams the KV blocks
// (128 keys) of the item's segment list in plan order and keeps the online softmax
// (running max m, running sum l) in registers, one query row per thread:
//
//   warp 0      TMA producer: Q sub-tiles once per item, K/V blocks through a smem ring
//   warp 1      MMA issuer (one thread): S_t = Q_t K^T and O_t += P_t V with tcgen05.mma,
//               accumulators in TMEM (S_0,S_1: columns 0..255; O_0,O_1: columns 256..511)
//   warp 2      TMEM allocator
//   warps 4-7   softmax of sub-tile 0: tcgen05.ld S row -> mask (diagonal blocks only) ->
//   warps 8-11  softmax of sub-tile 1:   exp2 -> P (bf16) back into TMEM over S -> rescale O
//
// The two sub-tiles ping-pong: while the tensor core runs PV/QK for one sub-tile the other
// sub-tile's softmax runs on the CUDA cores.  P is consumed by the PV MMA straight from
// TMEM (A operand), V is the MN-major B operand, so neither is re-staged through smem.
//
// Softmax details, each from a measurement (profiles/): the whole 128-column score row of a thread
// is held in registers (one TMEM read per block); the reference max only follows the running max
// when it moved by more than 2^8, so the accumulator rescale is rare; the arithmetic is packed
// fp32x2; a compile-time fraction of the exponentials can run on the FMA pipe (degree-3 polynomial;
// MESH_ATTN_POLY_OF_8, default 0: under the power cap the MUFU is the cheaper place); P is handed over in two 64-key
// halves so the PV MMA starts while the second half is still being exponentiated; single-thread
// roles are entered through elect.sync so TMA / MMA issue runs on the uniform datapath.
// kSplit (plan precision = 1): P as hi + lo bf16, two PV MMAs.
#include <cuda_bf16.h>

#include <atomic>

#include "plan.hpp"
#include "sm100.cuh"
#include "tile_kernels.hpp"

namespace mesh_attn {
using namespace sm100;

namespace {

constexpr int kThreads = 384;
constexpr int kLoaderWarp = 0, kMmaWarp = 1, kAllocWarp = 2, kSchedWarp = 3, kSoftmaxWarp0 = 4;
constexpr int kSchedSlots = 2;           // ring of work-item indices handed out by the scheduler warp
// register budget per thread (setmaxnreg): 128 x kCtrlRegs + 256 x kSoftmaxRegs <= 65536
constexpr int kCtrlRegs = 88, kSoftmaxRegs = 208;
constexpr float kRescaleStep = 8.f;      // log2 domain: the accumulator is rescaled only when the row max moved by > 2^8
#ifndef MESH_ATTN_POLY_OF_8
#define MESH_ATTN_POLY_OF_8 0            // exponentials per 8 evaluated on the FMA pipe (packed fp32x2 polynomial) instead of the MUFU.
                                         // Round 1 (static item order, C2 at burst clocks): 0 / 2 / 4 of 8 -> 6.08 / 5.89 / 6.19 ms per launch.
                                         // Round 2 (dynamic item order; C5 and C4 run under the power cap, where the polynomial's extra
                                         // instructions cost clock): C5 tile_fwd 1057 / 1037 / 1040 / 999 / 997 TFLOP/s for 0 / 1 / 2 / 3 / 4 of 8,
                                         // C4 1056 / 1036 (0 / 1), C2 1124 / 1126: all on the MUFU (profiles/r02_v1_README.md)
#endif

// Ablation build (tuning only, results are WRONG): 1 = the softmax groups skip the TMEM load, the max, the exponentials and the P
// store (they only pass the barriers on): what is left is the time of the MMAs and the TMA loads (profiles/r02_v4_README.md).
#ifndef MESH_ATTN_FWD_ABLATE
#define MESH_ATTN_FWD_ABLATE 0
#endif
constexpr int kFwdAblate = MESH_ATTN_FWD_ABLATE;

template <int N> struct IntTag { static constexpr int value = N; };
template <int kRegs> __device__ __forceinline__ void reg_alloc() { asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(kRegs)); }
template <int kRegs> __device__ __forceinline__ void reg_dealloc() { asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(kRegs)); }

// kPair: the kernel runs as clusters of two CTAs that take work items 2k and 2k+1, which the planner has checked to stream the
// SAME K / V blocks (FwdParams::pair), and every MMA is a tcgen05 cta_group::2 MMA of M = 256 issued by rank 0: 128 query rows
// of each CTA against one K / V block of which each CTA's shared memory holds HALF -- K rows 64r..64r+63 (B of S = Q K^T is
// K-major, split along N = keys), V columns 64r..64r+63 (B of O += P V is MN-major, split along N = head_dim).  Per block a
// CTA's tensor core then reads 128 KB of operands instead of 192 KB and the TMA writes 32 KB instead of 64 KB: shared-memory
// bandwidth (128 B/clk), which bounds the single-CTA kernel (profiles/r02_v4_README.md), is no longer the limit.
template <int D, bool kPair> struct FwdCfg {
    static_assert(!kPair || D == 128, "the CTA-pair kernel is built for head_dim 128");
    static constexpr int kBoxes = D / 64;                  // 64-element (128-byte) TMA boxes per row
    static constexpr int kTileBytes = kBlock * D * 2;      // one [128 x D] bf16 tile
    static constexpr int kSlotBytes = kPair ? kTileBytes / 2 : kTileBytes;   // a ring slot: a K or V tile, or this CTA's half of one
    static constexpr int kStages = (D == 128 ? 5 : 8) * (kPair ? 2 : 1);     // K/V ring slots
    static constexpr int kSmemQ = 2 * kTileBytes;
    static constexpr int kSmemRing = kStages * kSlotBytes;
    static constexpr int kNumBars = 2 + 2 * kStages + 8 + 3 * kSchedSlots;
    static constexpr int kSmemBytes = kSmemQ + kSmemRing + kNumBars * 8 + 16 + 16 + 1024 + kWatchdogBytes;   // + TMEM slot, item ring, alignment slack, watchdog state (last 16 bytes)
    static constexpr uint32_t kColS = 0, kColO = 256;      // TMEM columns
};

// The 128-key KV blocks of a work item in plan order: segment by segment (KV partition v, local key rows
// [begin, end) clipped to the rows visible to the item's last query row), block by block.  Every role runs the same
// nest; f(vrow, t0, off): row-addressing index of the KV partition, first local key row, causal offset (key t visible to row s iff t <= s + off).
struct KvRange { int v, vrow, off, t_lo, t_hi; };   // vrow: partition index that addresses v's rows (plan.hpp kv_row_part)
__device__ __forceinline__ KvRange kv_range(const Geom& gm, const Seg sg, int g, int u, int q_last)
{
    KvRange r;
    r.v = kv_partition(gm, g, sg.part_local);
    r.vrow = kv_row_part(gm, r.v, sg.part_local);
    r.t_lo = sg.begin;
    r.t_hi = sg.end;
    r.off = 0x20000000;
    if (gm.causal) {
        r.off = causal_off(gm, u, r.v);
        const int lim = q_last + r.off;                 // last visible key row for the item's last query row
        r.t_hi = lim < sg.begin ? sg.begin : min(sg.end, (lim / kBlock + 1) * kBlock);
    }
    return r;
}
template <class F>
__device__ __forceinline__ void for_each_kv_block(const Geom& gm, const Seg* segs, int nseg, int g, int u, int q_last, F&& f)
{
    for (int si = 0; si < nseg; ++si) {
        const KvRange r = kv_range(gm, segs[si], g, u, q_last);
        for (int t0 = r.t_lo; t0 < r.t_hi; t0 += kBlock) f(r.vrow, t0, r.off);
    }
}
__device__ __forceinline__ int count_kv_blocks(const Geom& gm, const Seg* segs, int nseg, int g, int u, int q_last)
{
    int n = 0;
    for (int si = 0; si < nseg; ++si) {
        const KvRange r = kv_range(gm, segs[si], g, u, q_last);
        n += (r.t_hi - r.t_lo) / kBlock;
    }
    return n;
}

struct ItemCtx {
    FwdItem it;
    int g_local, g, u, nt, nseg;
    const Seg* segs;
};

__device__ __forceinline__ ItemCtx load_item(const FwdParams& p, int idx)
{
    ItemCtx c;
    c.g_local = idx / p.items_per_gpu;
    c.it = p.items[idx - c.g_local * p.items_per_gpu];
    c.g = p.g_first + c.g_local;
    c.u = (c.g / p.gm.a) * p.gm.a + c.it.u_local;
    c.nt = c.it.nrows / kBlock;
    const SegList sl = p.seglists[c.it.seglist];
    c.segs = p.segs + sl.offset;
    c.nseg = sl.count;
    return c;
}

template <int D, bool kSplit, bool kPair>
__global__ void __launch_bounds__(kThreads, 1)
tile_fwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const FwdParams p)      // kPair: tmK has 64-row boxes
{
    static_assert(!(kPair && kSplit), "the CTA-pair kernel is built for the single-operand mode");
    using Cfg = FwdCfg<D, kPair>;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sQ = smem;
    uint8_t* sRing = smem + Cfg::kSmemQ;
    uint64_t* bars = reinterpret_cast<uint64_t*>(sRing + Cfg::kSmemRing);
    uint64_t* q_full = bars + 0;
    uint64_t* q_empty = bars + 1;
    uint64_t* kv_full = bars + 2;
    uint64_t* kv_empty = kv_full + Cfg::kStages;
    uint64_t* s_full = kv_empty + Cfg::kStages;   // [2]
    uint64_t* p_half = s_full + 2;                // [2 sub-tiles][2 column halves]: P is handed to the PV MMA in two halves
    uint64_t* o_full = p_half + 4;                // [2]
    uint64_t* sched_full = o_full + 2;            // [kSchedSlots] the scheduler warp has put the next work-item index into slot k
    uint64_t* sched_empty = sched_full + kSchedSlots;   // [kSchedSlots] every role has read slot k
    uint64_t* peer_free = sched_empty + kSchedSlots;    // [kSchedSlots] kPair, rank 0: the peer's slot k is armed for the next index
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(peer_free + kSchedSlots);
    volatile int* sched_idx = reinterpret_cast<volatile int*>(tmem_slot + 4);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const Geom& gm = p.gm;
    const int total_items = p.items_per_gpu * p.g_count;
    const uint32_t pair_rank = kPair ? cluster_ctarank() : 0;
    const bool leader = pair_rank == 0;                 // issues the pair's MMAs, owns the barriers the operands land on

    if (warp == kLoaderWarp && lane == 0) {
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV);
        watchdog_init(p.status);
        mbar_init(q_full, 1);
        mbar_init(q_empty, 1);
        for (int s = 0; s < Cfg::kStages; ++s) { mbar_init(&kv_full[s], 1); mbar_init(&kv_empty[s], 1); }
        for (int t = 0; t < 2; ++t) { mbar_init(&s_full[t], 1); mbar_init(&o_full[t], 1); }
        for (int t = 0; t < 4; ++t) mbar_init(&p_half[t], kPair ? kBlock + kBlock / 32 : kBlock);   // + one arrival per softmax warp of the peer
        for (int k = 0; k < kSchedSlots; ++k) {
            mbar_init(&sched_full[k], 1);
            // readers: loader, MMA issuer (rank 0), softmax groups; the peer's scheduler thread follows its ring too
            mbar_init(&sched_empty[k], 1 + (leader ? 1 : 0) + 2 * kBlock + ((kPair && !leader) ? 1 : 0));
            mbar_init(&peer_free[k], 1);
        }
        fence_mbar_init();
    }
    if (warp == kAllocWarp) {
        if constexpr (kPair) tmem_alloc_2cta<512>(tmem_slot);
        else tmem_alloc<512>(tmem_slot);
    }
    tc_fence_before();
    __syncthreads();
    if constexpr (kPair) cluster_sync();                // the peer's barriers are initialised before anything is sent to them
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    // Work items are handed out DYNAMICALLY (a global counter, published through a ring in shared memory that every role reads
    // in order): with the static round-robin the persistent CTAs, whose items differ in length under the causal mask, drift
    // apart by hundreds of items and the K / V blocks they stream stop being shared in L2 (see tile_bwd.cu).
    uint32_t sc_slot = 0, sc_phase = 0;
    auto next_item = [&]() -> int {
        if constexpr (kPair) mbar_wait_cluster(&sched_full[sc_slot], sc_phase);   // rank 1's index arrives from the peer (st.async)
        else mbar_wait(&sched_full[sc_slot], sc_phase);
        const int v = sched_idx[sc_slot];
        mbar_arrive(&sched_empty[sc_slot]);
        if (++sc_slot == kSchedSlots) { sc_slot = 0; sc_phase ^= 1; }
        return v;
    };

    if (warp < kSoftmaxWarp0) reg_dealloc<kCtrlRegs>();
    if (warp == kSchedWarp) {
        // =============================== work-item scheduler ===============================
        if (elect_one()) {
            if (leader) {
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
                    if (++slot == kSchedSlots) { slot = 0; phase ^= 1; }
                }
            } else {
                // rank 1: arm a slot (expect the 4 bytes of the index), tell rank 0, and follow the ring like every other role
                const uint32_t r0_free = mapa(smem_u32(peer_free), 0u);
                for (int k = 0; k < kSchedSlots; ++k) { mbar_expect_tx(&sched_full[k], 4); mbar_arrive_remote(r0_free + k * 8); }
                uint32_t slot = 0, phase = 0;
                while (true) {
                    const int v = next_item();
                    if (v >= total_items) break;
                    mbar_wait(&sched_empty[slot], phase);                        // every role has read it: arm the slot again
                    mbar_expect_tx(&sched_full[slot], 4);
                    mbar_arrive_remote(r0_free + slot * 8);
                    if (++slot == kSchedSlots) { slot = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == kLoaderWarp) {
        // =============================== TMA producer ===============================
        if (elect_one()) {
            uint32_t stage = 0, ring_phase = 0, q_phase = 0;
            // kPair: every load lands in this CTA's shared memory and completes its bytes on RANK 0's barrier (the MMA issuer waits
            // there for both CTAs' operands); rank 0 alone arms the barrier, with the bytes of both CTAs
            const uint32_t q_full_r0 = kPair ? mapa(smem_u32(q_full), 0u) : 0u, kv_full_r0 = kPair ? mapa(smem_u32(kv_full), 0u) : 0u;
            for (int idx = next_item(); idx < total_items; idx = next_item()) {
                const ItemCtx c = load_item(p, idx);
                bool first = true;
                for_each_kv_block(gm, c.segs, c.nseg, c.g, c.u, c.it.q0 + c.it.nrows - 1, [&](int v, int t0, int) {
                    if (first) {
                        first = false;
                        mbar_wait(q_empty, q_phase ^ 1);
                        q_phase ^= 1;
                        if (leader) mbar_expect_tx(q_full, (kPair ? 2 : 1) * c.nt * Cfg::kTileBytes);
                        for (int t = 0; t < c.nt; ++t)
                            for (int bx = 0; bx < Cfg::kBoxes; ++bx) {
                                const int row = q_row_part(gm, c.u, c.it.u_local) * gm.L + c.it.q0 + t * kBlock;
                                if constexpr (kPair)
                                    tma_load_4d_2cta(sQ + t * Cfg::kTileBytes + bx * (kBlock * 128), &tmQ, q_full_r0, bx * 64, c.it.head, row, c.it.batch, kEvictFirst);
                                else
                                    tma_load_4d(sQ + t * Cfg::kTileBytes + bx * (kBlock * 128), &tmQ, q_full, bx * 64, c.it.head, row, c.it.batch, kEvictFirst);
                            }
                    }
                    const int hk = c.it.head / gm.group;
                    for (int kv = 0; kv < 2; ++kv) {       // K block then V block through the ring
                        mbar_wait(&kv_empty[stage], ring_phase ^ 1);
                        if constexpr (kPair) {
                            if (leader) mbar_expect_tx(&kv_full[stage], Cfg::kTileBytes);      // both CTAs' halves
                            uint8_t* dst = sRing + stage * Cfg::kSlotBytes;
                            if (kv == 0)                                                       // K rows 64r .. 64r+63: two [64 x 64] boxes
                                for (int bx = 0; bx < Cfg::kBoxes; ++bx)
                                    tma_load_4d_2cta(dst + bx * (kBlock / 2 * 128), &tmK, kv_full_r0 + stage * 8, bx * 64, hk,
                                                     v * gm.L + t0 + (int)pair_rank * (kBlock / 2), c.it.batch, kEvictLast);
                            else                                                               // V columns 64r .. 64r+63: one [128 x 64] box
                                tma_load_4d_2cta(dst, &tmV, kv_full_r0 + stage * 8, (int)pair_rank * 64, hk, v * gm.L + t0, c.it.batch, kEvictLast);
                        } else {
                            mbar_expect_tx(&kv_full[stage], Cfg::kTileBytes);
                            for (int bx = 0; bx < Cfg::kBoxes; ++bx)
                                tma_load_4d(sRing + stage * Cfg::kTileBytes + bx * (kBlock * 128), kv == 0 ? &tmK : &tmV, &kv_full[stage],
                                            bx * 64, hk, v * gm.L + t0, c.it.batch, kEvictLast);
                        }
                        if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                    }
                });
            }
        }
    } else if (warp == kMmaWarp) {
        // =============================== MMA issuer (kPair: rank 0 issues for both CTAs) ===============================
        if (leader && elect_one()) {
            constexpr int kM = kPair ? 2 * kBlock : kBlock;
            constexpr uint32_t idesc_qk = umma_idesc(kM, kBlock, false, false);
            constexpr uint32_t idesc_pv = umma_idesc(kM, D, false, true);
            auto commit = [&](uint64_t* bar) {               // kPair: the same barrier of both CTAs
                if constexpr (kPair) umma_commit_2cta(bar);
                else umma_commit(bar);
            };
            uint32_t stage = 0, ring_phase = 0, q_phase = 0, p_phase[2] = {0, 0};
            PT_DECL;
            auto ring_wait = [&](uint32_t& slot) {
                mbar_wait(&kv_full[stage], ring_phase);
                slot = stage;
                if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
            };
            auto issue_qk = [&](int t, uint32_t kslot) {
                const uint32_t qa = smem_u32(sQ + t * Cfg::kTileBytes), ka = smem_u32(sRing + kslot * Cfg::kSlotBytes);
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t o = (kk / 4) * (kBlock * 128) + (kk % 4) * 32;
                    if constexpr (kPair) {                   // this CTA's K half: 64 rows per 64-column box
                        const uint32_t ob = (kk / 4) * (kBlock / 2 * 128) + (kk % 4) * 32;
                        umma_ss_2cta(tmem + Cfg::kColS + t * kBlock, umma_desc(qa + o, 16, 1024), umma_desc(ka + ob, 16, 1024), idesc_qk, kk > 0);
                    } else {
                        umma_ss(tmem + Cfg::kColS + t * kBlock, umma_desc(qa + o, 16, 1024), umma_desc(ka + o, 16, 1024), idesc_qk, kk > 0);
                    }
                }
            };
            // P (bf16) in TMEM over S: hi at columns 0..63, lo at 64..127; `half` = keys 0..63 or 64..127 of the block
            auto issue_pv = [&](int t, uint32_t vslot, int half, bool acc) {
                const uint32_t va = smem_u32(sRing + vslot * Cfg::kSlotBytes);
#pragma unroll
                for (int x = 0; x < (kSplit ? 2 : 1); ++x)
#pragma unroll
                    for (int k4 = 0; k4 < kBlock / 32; ++k4) {
                        const int kk = half * (kBlock / 32) + k4;
                        if constexpr (kPair)                 // this CTA's V half: the 64 head_dim columns of one box, all 128 keys
                            umma_ts_2cta(tmem + Cfg::kColO + t * D, tmem + Cfg::kColS + t * kBlock + kk * 8,
                                         umma_desc(va + kk * 2048, kBlock * 128, 1024), idesc_pv, (acc || k4 > 0) ? 1u : 0u);
                        else
                            umma_ts(tmem + Cfg::kColO + t * D, tmem + Cfg::kColS + t * kBlock + x * 64 + kk * 8,
                                    umma_desc(va + kk * 2048, kBlock * 128, 1024), idesc_pv, (acc || k4 > 0 || x > 0) ? 1u : 0u);
                    }
            };
            for (int idx = next_item(); idx < total_items; idx = next_item()) {
                const ItemCtx c = load_item(p, idx);
                const int nb = count_kv_blocks(gm, c.segs, c.nseg, c.g, c.u, c.it.q0 + c.it.nrows - 1);
                if (nb == 0) continue;
                mbar_wait(q_full, q_phase);
                q_phase ^= 1;
                uint32_t kslot, vslot;
                ring_wait(kslot);
                tc_fence_after();
                for (int t = 0; t < c.nt; ++t) { issue_qk(t, kslot); commit(&s_full[t]); }
                commit(&kv_empty[kslot]);
                for (int j = 0; j < nb; ++j) {
                    const bool more = j + 1 < nb;
                    PT_MARK(0);
                    ring_wait(vslot);
                    if (more) ring_wait(kslot);
                    PT_MARK(1);
                    for (int t = 0; t < c.nt; ++t) {
                        // (kPair: P lives in tensor memory, ordered by the tcgen05 fences on both sides of the barrier: the wait needs no
                        // cluster-scope acquire, which would cost a cache invalidation per wait)
                        mbar_wait(&p_half[2 * t], p_phase[t]);       // the PV MMA starts on the first 64 keys while the softmax
                        tc_fence_after();                             // group is still exponentiating the other 64
                        PT_MARK(2 + 2 * t);
                        issue_pv(t, vslot, 0, j > 0);
                        mbar_wait(&p_half[2 * t + 1], p_phase[t]);
                        p_phase[t] ^= 1;
                        tc_fence_after();
                        issue_pv(t, vslot, 1, true);
                        if (more) { issue_qk(t, kslot); commit(&s_full[t]); }
                        else commit(&o_full[t]);
                        PT_MARK(3 + 2 * t);
                    }
                    commit(&kv_empty[vslot]);
                    if (more) commit(&kv_empty[kslot]);
                }
                commit(q_empty);
            }
            PT_REPORT("fwd MMA thread clocks per block: ring_wait, wait_p0, issue0, wait_p1, issue1");
        }
    } else if (warp >= kSoftmaxWarp0) {
        // =============================== softmax / epilogue ===============================
        reg_alloc<kSoftmaxRegs>();
        const int t = (warp - kSoftmaxWarp0) >> 2;              // sub-tile of this warpgroup
        const int row = threadIdx.x - kSoftmaxWarp0 * 32 - t * kBlock;   // 0..127 = TMEM lane
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + lane_base + Cfg::kColS + t * kBlock;
        const uint32_t tO = tmem + lane_base + Cfg::kColO + t * D;
        const float c2 = gm.scale_log2;
        const uint32_t p_half_r0 = kPair ? mapa(smem_u32(p_half), 0u) : 0u;
        uint32_t s_phase = 0, o_phase = 0;
        PT_DECL;
        for (int idx = next_item(); idx < total_items; idx = next_item()) {
            const ItemCtx c = load_item(p, idx);
            if (t >= c.nt) continue;
            const int srow = c.it.q0 + t * kBlock + row;            // local query row
            const size_t slot = ((size_t)c.g_local * gm.slots_per_gpu + c.it.slot) * gm.batch + c.it.batch;
            float* out = p.partial_O + ((slot * gm.L + srow) * gm.heads_q + c.it.head) * (size_t)D;
            float* out_lse = p.partial_lse + (slot * gm.heads_q + c.it.head) * (size_t)gm.L + srow;
            // m: the reference max the exponentials are taken against (log2 domain, scaled).  It only follows the true
            // running max when that has moved by more than kRescaleStep: P then stays <= 2^kRescaleStep, and the
            // accumulator rescale (a TMEM round trip) is rare.  O / l is exact for any reference.
            float m = -INFINITY, l = 0.f;
            int j = 0;
            for_each_kv_block(gm, c.segs, c.nseg, c.g, c.u, c.it.q0 + c.it.nrows - 1, [&](int, int t0, int off) {
                PT_MARK(0);
                mbar_wait(&s_full[t], s_phase);
                s_phase ^= 1;
                tc_fence_after();
                if (kFwdAblate & 1) {
                    tc_fence_before();
                    if (kPair && !leader) {
                        __syncwarp();
                        if (lane == 0) { mbar_arrive_remote(p_half_r0 + (2 * t) * 8); mbar_arrive_remote(p_half_r0 + (2 * t + 1) * 8); }
                    } else {
                        mbar_arrive(&p_half[2 * t]);
                        mbar_arrive(&p_half[2 * t + 1]);
                    }
                    ++j;
                    return;
                }
                uint32_t s[kBlock];                                 // the whole score row of this thread
#pragma unroll
                for (int ch = 0; ch < kBlock / 32; ++ch) tmem_ld_x32(tS + ch * 32, *reinterpret_cast<uint32_t(*)[32]>(&s[ch * 32]));
                PT_MARK(1);
                tmem_ld_wait();
                PT_MARK(2);
                // key column c of this block is visible iff c <= row + dlt; only blocks that straddle the diagonal mask
                const int dlt = c.it.q0 + t * kBlock + off - t0;
                const bool masked = gm.causal && dlt < kBlock - 1;
                if (masked) {
                    const int lim = row + dlt;
#pragma unroll
                    for (int i = 0; i < kBlock; ++i) if (i > lim) s[i] = 0xff800000u;   // -inf
                }
                float mx0 = -INFINITY, mx1 = -INFINITY, mx2 = -INFINITY, mx3 = -INFINITY;
                // eight independent chains: the pass is latency-bound (four chains: C2 tile_fwd 1133 -> 1143 TFLOP/s)
                float mx4 = -INFINITY, mx5 = -INFINITY, mx6 = -INFINITY, mx7 = -INFINITY;
#pragma unroll
                for (int i = 0; i < kBlock; i += 16) {
                    mx0 = fmaxf(mx0, fmaxf(__uint_as_float(s[i + 0]), __uint_as_float(s[i + 1])));
                    mx1 = fmaxf(mx1, fmaxf(__uint_as_float(s[i + 2]), __uint_as_float(s[i + 3])));
                    mx2 = fmaxf(mx2, fmaxf(__uint_as_float(s[i + 4]), __uint_as_float(s[i + 5])));
                    mx3 = fmaxf(mx3, fmaxf(__uint_as_float(s[i + 6]), __uint_as_float(s[i + 7])));
                    mx4 = fmaxf(mx4, fmaxf(__uint_as_float(s[i + 8]), __uint_as_float(s[i + 9])));
                    mx5 = fmaxf(mx5, fmaxf(__uint_as_float(s[i + 10]), __uint_as_float(s[i + 11])));
                    mx6 = fmaxf(mx6, fmaxf(__uint_as_float(s[i + 12]), __uint_as_float(s[i + 13])));
                    mx7 = fmaxf(mx7, fmaxf(__uint_as_float(s[i + 14]), __uint_as_float(s[i + 15])));
                }
                mx0 = fmaxf(mx0, fmaxf(mx4, mx5));
                mx1 = fmaxf(mx1, fmaxf(mx6, mx7));
                const float m_blk = fmaxf(fmaxf(mx0, mx1), fmaxf(mx2, mx3)) * c2;
                if (j == 0) {
                    m = m_blk;
                } else if (__any_sync(0xffffffffu, m_blk > m + kRescaleStep)) {   // warp-uniform: TMEM ops are warp-collective
                    const float m_new = fmaxf(m, m_blk);
                    const float alpha = (m_new == -INFINITY) ? 1.f : ex2(m - m_new);   // m = -inf -> 0
                    l *= alpha;
                    m = m_new;
#pragma unroll 1
                    for (int ch = 0; ch < D / 32; ++ch) {
                        uint32_t r[32];
                        tmem_ld_x32(tO + ch * 32, r);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 32; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) * alpha);
                        tmem_st_x32(tO + ch * 32, r);
                    }
                }
                PT_MARK(3);
                const float neg_m = (m == -INFINITY) ? 0.f : -m;
                // p = exp2(s*c2 - m).  Unmasked blocks: kPolyOf8 of every 8 on the FMA pipe (degree-3 polynomial), the
                // rest on the MUFU; diagonal blocks: all on the MUFU (exp2(-inf) must be exactly 0 there).
                f32x2 lacc0 = 0ull, lacc1 = 0ull;                    // two (even, odd) partial row sums
                const f32x2 c22 = pack2(c2, c2), nm2 = pack2(neg_m, neg_m);
                auto exp_row = [&](auto poly_tag) {
                    constexpr int kPoly = decltype(poly_tag)::value;
#pragma unroll
                    for (int ch = 0; ch < kBlock / 32; ++ch) {
                        uint32_t hi[16], lo[16];
#pragma unroll
                        for (int i = 0; i < 32; i += 2) {
                            float x0, x1;
                            unpack2(fma2(pack2(__uint_as_float(s[ch * 32 + i]), __uint_as_float(s[ch * 32 + i + 1])), c22, nm2), x0, x1);
                            float p0, p1;
                            if ((i & 7) < kPoly) ex2_poly2(x0, x1, p0, p1);       // pairs: kPoly of every 8 elements
                            else { p0 = ex2(x0); p1 = ex2(x1); }
                            if ((i & 2) == 0) lacc0 = add2(lacc0, pack2(p0, p1));
                            else lacc1 = add2(lacc1, pack2(p0, p1));
                            if constexpr (kSplit) split_bf16x2(p0, p1, hi[i / 2], lo[i / 2]);
                            else hi[i / 2] = pack_bf16x2(p0, p1);
                        }
                        // the whole S row is in registers: P (bf16) may overwrite any of its columns
                        tmem_st_x16(tS + ch * 16, hi);
                        if constexpr (kSplit) tmem_st_x16(tS + 64 + ch * 16, lo);
                        if (ch & 1) {                                 // half of the keys done: hand it to the PV MMA
                            tmem_st_wait();
                            tc_fence_before();
                            if (kPair && !leader) {                   // the issuer is in the peer CTA: one arrival per warp on ITS barrier
                                __syncwarp();
                                if (lane == 0) mbar_arrive_remote(p_half_r0 + (2 * t + (ch >> 1)) * 8);
                            } else {
                                mbar_arrive(&p_half[2 * t + (ch >> 1)]);
                            }
                        }
                    }
                };
                if (masked) exp_row(IntTag<0>{});
                else exp_row(IntTag<MESH_ATTN_POLY_OF_8>{});
                float l0, l1;
                unpack2(add2(lacc0, lacc1), l0, l1);
                l += l0 + l1;
                PT_MARK(4);
                PT_MARK(5);
                ++j;
            });
            if (j == 0) {                      // no visible key for the whole item (reading R5)
#pragma unroll 4
                for (int d = 0; d < D; d += 4) *reinterpret_cast<float4*>(out + d) = make_float4(0.f, 0.f, 0.f, 0.f);
                *out_lse = -INFINITY;
                continue;
            }
            mbar_wait(&o_full[t], o_phase);
            o_phase ^= 1;
            tc_fence_after();
            const float inv_l = l > 0.f ? 1.f / l : 0.f;
#pragma unroll 1
            for (int ch = 0; ch < D / 32; ++ch) {
                uint32_t r[32];
                tmem_ld_x32(tO + ch * 32, r);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 32; i += 4)
                    *reinterpret_cast<float4*>(out + ch * 32 + i) =
                        make_float4(__uint_as_float(r[i]) * inv_l, __uint_as_float(r[i + 1]) * inv_l, __uint_as_float(r[i + 2]) * inv_l,
                                    __uint_as_float(r[i + 3]) * inv_l);
            }
            *out_lse = l > 0.f ? (m + lg2(l)) * 0.6931471805599453f : -INFINITY;
        }
        PT_REPORT("fwd softmax clocks per block: wait_s+issue_ld, wait_ld, mask+max+rescale, exp+st, st_wait+arrive");
    }

    tc_fence_before();
    __syncthreads();
    if constexpr (kPair) cluster_sync();                // no CTA leaves while its peer may still read its operands or arrive on its barriers
    if (warp == kAllocWarp) {
        if constexpr (kPair) tmem_dealloc_2cta<512>(tmem);
        else tmem_dealloc<512>(tmem);
    }
}

template <int D, bool kSplit, bool kPair>
int launch_fwd_one(const FwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV, int grid, cudaStream_t stream)
{
    using Cfg = FwdCfg<D, kPair>;
    static_assert(Cfg::kSmemBytes <= 227 * 1024, "tile_fwd shared memory over the 227 KB CTA limit");
    auto kernel = tile_fwd_kernel<D, kSplit, kPair>;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::kSmemBytes);
    if (e != cudaSuccess) return (int)e;
    cudaLaunchConfig_t cfg{};
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = Cfg::kSmemBytes;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    if (kPair) {
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
    e = cudaLaunchKernelEx(&cfg, kernel, tmQ, tmK, tmV, p);
    return e != cudaSuccess ? (int)e : (int)cudaGetLastError();
}

}  // namespace

int launch_tile_fwd(const FwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV, int num_sms,
                    cudaStream_t stream)
{
    const int total = p.items_per_gpu * p.g_count;
    if (total <= 0) return 0;
    const int grid = total < num_sms ? total : num_sms;
    if (p.pair) {                                       // checked by the caller: head_dim 128, single-operand mode, an even item count
        if (p.gm.head_dim != 128 || p.split || (total & 1)) return (int)cudaErrorInvalidValue;
        return launch_fwd_one<128, false, true>(p, tmQ, tmK, tmV, grid, stream);
    }
    if (p.gm.head_dim == 128)
        return p.split ? launch_fwd_one<128, true, false>(p, tmQ, tmK, tmV, grid, stream) : launch_fwd_one<128, false, false>(p, tmQ, tmK, tmV, grid, stream);
    return p.split ? launch_fwd_one<64, true, false>(p, tmQ, tmK, tmV, grid, stream) : launch_fwd_one<64, false, false>(p, tmQ, tmK, tmV, grid, stream);
}

}  // namespace mesh_attn
