// tile_bwd.cu -- mesh_attn_tile_bwd: per-pair attention backward of a simulated GPU's tile
// (Alg.3 l.3-5, L250-253; kernel inputs (Q_i, KV_j, O_i, dO_i), L236).
//
// One persistent CTA per SM walks the work list.  A work item is a 128-key block of one
// (simulated GPU g, KV partition v, KV head); the CTA keeps K and V of the block resident in
// shared memory and dK, dV in TMEM, and streams 128-row Q / dO blocks of every Q partition
// of the tile (and every query head of the GQA group).  Per Q block, five tcgen05 MMAs:
//
//   S^T  = K Q^T            (TMEM columns   0..127)      P^T = exp2(S^T*c - lse)  (bf16, over S^T)
//   dP^T = V dO^T           (TMEM columns 128..255)      dS^T = P^T o (dP^T - delta) (bf16, smem)
//   dV  += P^T  dO          (TMEM columns 384..511)      A operand P^T straight from TMEM
//   dK  += dS^T Q           (TMEM columns 256..383)      A operand dS^T from smem (K-major)
//   dQ   = dS K             (TMEM columns 128..255, reusing dP^T once consumed)
//                                                        A operand the same smem buffer read M-major
//
//   warp 0      TMA producer: K,V per item; Q, dO, lse, delta per step through a 2-stage ring
//   warp 1      MMA issuer (one thread)
//   warp 2      TMEM allocator
//   warps 4-7   one key row per thread: S^T -> P^T, dP^T -> dS^T; dK epilogue
//   warps 8-11  one query row per thread: dQ drain (x scale, red.global.add); dV epilogue
//
// dQ, dK, dV are accumulated into global fp32 with vector atomics: the sums over the Q group,
// the KV group (Alg.3 l.6-7, L254-255) and the GQA head group all land in the same buffers.
#include <cuda_bf16.h>

#include "plan.hpp"
#include "sm100.cuh"
#include "tile_kernels.hpp"

namespace mesh_attn {
using namespace sm100;

namespace {

constexpr int kBwdThreads = 384;
constexpr float kLog2e = 1.4426950408889634f;

template <int D> struct BwdCfg {
    static constexpr int kBoxes = D / 64;
    static constexpr int kTileBytes = kBlock * D * 2;          // [128 x D] bf16
    static constexpr int kDsBytes = kBlock * kBlock * 2;        // dS^T [128 kv x 128 q] bf16
    static constexpr int kStages = 2;
    static constexpr int kOffK = 0;
    static constexpr int kOffV = kTileBytes;
    static constexpr int kOffStage = 2 * kTileBytes;            // per stage: Q tile, dO tile
    static constexpr int kOffDs = kOffStage + kStages * 2 * kTileBytes;
    static constexpr int kOffVec = kOffDs + kDsBytes;           // per stage: lse[128], delta[128] fp32
    static constexpr int kOffBars = kOffVec + kStages * 1024;
    static constexpr int kNumBars = 2 + 2 * kStages + 8;
    static constexpr int kSmemBytes = kOffBars + kNumBars * 8 + 16;
    static constexpr uint32_t kColS = 0, kColDP = 128, kColDK = 256, kColDV = 384;
};

// Walks the 128-row Q blocks of a backward work item in plan order: for every segment
// (Q partition u, local rows [begin, end)), every query head of the GQA group, every block with
// at least one visible (query, key) pair.  Every role runs the same walk.
struct QWalk {
    const Geom& gm;
    const Seg* segs;
    int nseg, g, v, t0, head_kv;
    int si = -1, hh = 0, s = 0, s_lo = 0, s_hi = 0, u = 0, off = 0;
    __device__ QWalk(const Geom& gm_, const Seg* segs_, int nseg_, int g_, int v_, int t0_, int head_kv_)
        : gm(gm_), segs(segs_), nseg(nseg_), g(g_), v(v_), t0(t0_), head_kv(head_kv_) {}
    // next block: Q partition u, query head h, first local query row s0, causal offset off
    __device__ bool next(int& u_out, int& h_out, int& s0_out, int& off_out)
    {
        while (true) {
            if (si >= 0 && s < s_hi) { u_out = u; h_out = head_kv * gm.group + hh; s0_out = s; off_out = off; s += kBlock; return true; }
            if (si >= 0 && s_lo < s_hi && ++hh < gm.group) { s = s_lo; continue; }
            if (++si >= nseg) return false;
            const Seg sg = segs[si];
            u = (g / gm.a) * gm.a + sg.part_local;
            hh = 0;
            s_lo = sg.begin;
            s_hi = sg.end;
            off = 0x20000000;
            if (gm.causal) {
                off = causal_off(gm, u, v);
                const int x = t0 - off - (kBlock - 1);          // first query row that sees key t0 is t0 - off
                if (x > s_lo) s_lo = min(s_hi, ((x + kBlock - 1) / kBlock) * kBlock);
            }
            s = s_lo;
        }
    }
};

struct BwdItemCtx {
    BwdItem it;
    int g_local, g, v, nseg;
    const Seg* segs;
};

__device__ __forceinline__ BwdItemCtx load_bwd_item(const BwdParams& p, int idx)
{
    BwdItemCtx c;
    c.g_local = idx / p.items_per_gpu;
    c.it = p.items[idx - c.g_local * p.items_per_gpu];
    c.g = p.g_first + c.g_local;
    c.v = kv_partition(p.gm, c.g, c.it.kv_local);
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
__device__ __forceinline__ float bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }

// TMEM accumulator [128 lanes x D columns] -> x scale -> atomic add into a global row of D floats
template <int D> __device__ __forceinline__ void drain_rows(uint32_t taddr, float* grow, float scale)
{
#pragma unroll 1
    for (int ch = 0; ch < D / 32; ++ch) {
        uint32_t r[32];
        tmem_ld_x32(taddr + ch * 32, r);
        tmem_ld_wait();
#pragma unroll
        for (int i = 0; i < 32; i += 4)
            red_add_v4(grow + ch * 32 + i, __uint_as_float(r[i]) * scale, __uint_as_float(r[i + 1]) * scale,
                       __uint_as_float(r[i + 2]) * scale, __uint_as_float(r[i + 3]) * scale);
    }
}

template <int D>
__global__ void __launch_bounds__(kBwdThreads, 1)
tile_bwd_kernel(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmdO, const BwdParams p)
{
    using Cfg = BwdCfg<D>;
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
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(s_full + 8);
    auto sQ = [&](int st) { return smem + Cfg::kOffStage + st * 2 * Cfg::kTileBytes; };
    auto sdO = [&](int st) { return smem + Cfg::kOffStage + st * 2 * Cfg::kTileBytes + Cfg::kTileBytes; };
    auto sLse = [&](int st) { return reinterpret_cast<float*>(smem + Cfg::kOffVec + st * 1024); };
    auto sDelta = [&](int st) { return reinterpret_cast<float*>(smem + Cfg::kOffVec + st * 1024 + 512); };

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const Geom& gm = p.gm;
    const int total_items = p.items_per_gpu * p.g_count;
    const long long N = (long long)gm.n * gm.L;

    if (threadIdx.x == 0) {
        if (smem_u32(smem) & 1023u) { printf("mesh_attn tile_bwd: dynamic smem base not 1024-byte aligned\n"); __trap(); }
        prefetch_tmap(&tmQ); prefetch_tmap(&tmK); prefetch_tmap(&tmV); prefetch_tmap(&tmdO);
        mbar_init(kv_full, 1);
        mbar_init(kv_empty, 1);
        for (int s = 0; s < Cfg::kStages; ++s) { mbar_init(&qd_full[s], 1); mbar_init(&qd_empty[s], 1); }
        mbar_init(s_full, 1);
        mbar_init(p_full, kBlock);
        mbar_init(dp_full, 1);
        mbar_init(ds_full, kBlock);
        mbar_init(dq_full, 1);
        mbar_init(dq_empty, kBlock);
        mbar_init(dkv_full, 1);
        mbar_init(dkv_empty, 2 * kBlock);
        fence_mbar_init();
    }
    if (warp == 2) tmem_alloc<512>(tmem_slot);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        // =============================== TMA producer ===============================
        if (lane == 0) {
            uint32_t stage = 0, ring_phase = 0, kv_phase = 0;
            for (int idx = blockIdx.x; idx < total_items; idx += gridDim.x) {
                const BwdItemCtx c = load_bwd_item(p, idx);
                QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
                int u, h, s0, off;
                bool first = true;
                while (walk.next(u, h, s0, off)) {
                    if (first) {
                        first = false;
                        mbar_wait(kv_empty, kv_phase ^ 1);
                        kv_phase ^= 1;
                        mbar_expect_tx(kv_full, 2 * Cfg::kTileBytes);
                        for (int bx = 0; bx < Cfg::kBoxes; ++bx) {
                            tma_load_4d(sK + bx * (kBlock * 128), &tmK, kv_full, bx * 64, c.it.head_kv, c.v * gm.L + c.it.t0, c.it.batch, kEvictFirst);
                            tma_load_4d(sV + bx * (kBlock * 128), &tmV, kv_full, bx * 64, c.it.head_kv, c.v * gm.L + c.it.t0, c.it.batch, kEvictFirst);
                        }
                    }
                    mbar_wait(&qd_empty[stage], ring_phase ^ 1);
                    mbar_expect_tx(&qd_full[stage], 2 * Cfg::kTileBytes + 1024);
                    const int row = u * gm.L + s0;
                    for (int bx = 0; bx < Cfg::kBoxes; ++bx) {
                        tma_load_4d(sQ(stage) + bx * (kBlock * 128), &tmQ, &qd_full[stage], bx * 64, h, row, c.it.batch, kEvictLast);
                        tma_load_4d(sdO(stage) + bx * (kBlock * 128), &tmdO, &qd_full[stage], bx * 64, h, row, c.it.batch, kEvictLast);
                    }
                    const size_t vec = ((size_t)c.it.batch * gm.heads_q + h) * N + row;
                    bulk_load(sLse(stage), p.lse + vec, 512, &qd_full[stage]);
                    bulk_load(sDelta(stage), p.delta + vec, 512, &qd_full[stage]);
                    if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // =============================== MMA issuer ===============================
        if (lane == 0) {
            constexpr uint32_t idesc_kk = umma_idesc(kBlock, kBlock, false, false);   // S^T, dP^T
            constexpr uint32_t idesc_tn = umma_idesc(kBlock, D, false, true);         // dV (A in TMEM), dK (A smem K-major)
            constexpr uint32_t idesc_nn = umma_idesc(kBlock, D, true, true);          // dQ (A smem M-major)
            uint32_t stage = 0, ring_phase = 0, kv_phase = 0, p_ph = 0, ds_ph = 0, dqe_ph = 0, dkve_ph = 0;
            const uint32_t aK = smem_u32(sK), aV = smem_u32(sV), aDs = smem_u32(sDs);
            auto mma_kmajor = [&](uint32_t dcol, uint32_t a, uint32_t b) {          // D = A B^T, both K-major over head_dim
#pragma unroll
                for (int kk = 0; kk < D / 16; ++kk) {
                    const uint32_t o = (kk / 4) * (kBlock * 128) + (kk % 4) * 32;
                    umma_ss(tmem + dcol, umma_desc(a + o, 16, 1024), umma_desc(b + o, 16, 1024), idesc_kk, kk > 0);
                }
            };
            for (int idx = blockIdx.x; idx < total_items; idx += gridDim.x) {
                const BwdItemCtx c = load_bwd_item(p, idx);
                QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
                int u, h, s0, off, i = 0;
                uint32_t st_cur = 0;
                bool have = walk.next(u, h, s0, off);
                if (!have) continue;
                mbar_wait(kv_full, kv_phase);
                kv_phase ^= 1;
                mbar_wait(dkv_empty, dkve_ph ^ 1);      // previous item's dK/dV drained from TMEM
                dkve_ph ^= 1;
                // prologue: S^T(0), dP^T(0)
                mbar_wait(&qd_full[stage], ring_phase);
                tc_fence_after();
                st_cur = stage;
                mma_kmajor(Cfg::kColS, aK, smem_u32(sQ(st_cur)));
                umma_commit(s_full);
                mma_kmajor(Cfg::kColDP, aV, smem_u32(sdO(st_cur)));
                umma_commit(dp_full);
                if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                while (have) {
                    const bool more = walk.next(u, h, s0, off);
                    const uint32_t aQ = smem_u32(sQ(st_cur)), adO = smem_u32(sdO(st_cur));
                    // dV += P^T dO
                    mbar_wait(p_full, p_ph);
                    p_ph ^= 1;
                    tc_fence_after();
#pragma unroll
                    for (int kk = 0; kk < kBlock / 16; ++kk)
                        umma_ts(tmem + Cfg::kColDV, tmem + Cfg::kColS + kk * 8, umma_desc(adO + kk * 2048, kBlock * 128, 1024), idesc_tn,
                                (i > 0 || kk > 0) ? 1u : 0u);
                    uint32_t st_next = 0;
                    if (more) {                          // S^T(i+1) as early as possible
                        mbar_wait(&qd_full[stage], ring_phase);
                        tc_fence_after();
                        st_next = stage;
                        if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                        mma_kmajor(Cfg::kColS, aK, smem_u32(sQ(st_next)));
                        umma_commit(s_full);
                    }
                    // dK += dS^T Q ; dQ = dS K
                    mbar_wait(ds_full, ds_ph);
                    ds_ph ^= 1;
                    tc_fence_after();
#pragma unroll
                    for (int kk = 0; kk < kBlock / 16; ++kk)
                        umma_ss(tmem + Cfg::kColDK, umma_desc(aDs + (kk / 4) * (kBlock * 128) + (kk % 4) * 32, 16, 1024),
                                umma_desc(aQ + kk * 2048, kBlock * 128, 1024), idesc_tn, (i > 0 || kk > 0) ? 1u : 0u);
#pragma unroll
                    for (int kk = 0; kk < kBlock / 16; ++kk)
                        umma_ss(tmem + Cfg::kColDP, umma_desc(aDs + kk * 2048, kBlock * 128, 1024), umma_desc(aK + kk * 2048, kBlock * 128, 1024),
                                idesc_nn, kk > 0);
                    umma_commit(dq_full);
                    umma_commit(&qd_empty[st_cur]);
                    if (more) {                          // dP^T(i+1) once dQ(i) has left TMEM
                        mbar_wait(dq_empty, dqe_ph);
                        dqe_ph ^= 1;
                        tc_fence_after();
                        mma_kmajor(Cfg::kColDP, aV, smem_u32(sdO(st_next)));
                        umma_commit(dp_full);
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
        }
    } else if (warp >= 4 && warp < 8) {
        // =============================== S^T -> P^T, dP^T -> dS^T (one key row per thread) ===============================
        const int row = threadIdx.x - 128;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tS = tmem + lane_base + Cfg::kColS, tDP = tmem + lane_base + Cfg::kColDP, tDK = tmem + lane_base + Cfg::kColDK;
        uint32_t stage = 0, ring_phase = 0, s_ph = 0, dp_ph = 0, dq_ph = 0, dkv_ph = 0;
        for (int idx = blockIdx.x; idx < total_items; idx += gridDim.x) {
            const BwdItemCtx c = load_bwd_item(p, idx);
            QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
            int u, h, s0, off, i = 0;
            while (walk.next(u, h, s0, off)) {
                mbar_wait(&qd_full[stage], ring_phase);   // lse / delta of this step landed (bulk copies on the same barrier)
                const float* lse = sLse(stage);
                const float* delta = sDelta(stage);
                // query column cq of this block is visible to key row `row` iff cq >= cmin
                const int cmin = c.it.t0 + row - off - s0;
                const bool masked = gm.causal && (c.it.t0 + kBlock - 1 - off - s0 > 0);
                uint32_t pk[kBlock / 2];
                mbar_wait(s_full, s_ph);
                s_ph ^= 1;
                tc_fence_after();
#pragma unroll
                for (int ch = 0; ch < kBlock / 32; ++ch) {
                    uint32_t r[32];
                    tmem_ld_x32(tS + ch * 32, r);
                    tmem_ld_wait();
#pragma unroll
                    for (int q4 = 0; q4 < 32; q4 += 4) {
                        const float4 l4 = *reinterpret_cast<const float4*>(lse + ch * 32 + q4);
                        float p0 = ex2(fmaf(__uint_as_float(r[q4 + 0]), gm.scale_log2, -l4.x * kLog2e));
                        float p1 = ex2(fmaf(__uint_as_float(r[q4 + 1]), gm.scale_log2, -l4.y * kLog2e));
                        float p2 = ex2(fmaf(__uint_as_float(r[q4 + 2]), gm.scale_log2, -l4.z * kLog2e));
                        float p3 = ex2(fmaf(__uint_as_float(r[q4 + 3]), gm.scale_log2, -l4.w * kLog2e));
                        if (masked) {
                            const int cq = ch * 32 + q4;
                            if (cq + 0 < cmin) p0 = 0.f;
                            if (cq + 1 < cmin) p1 = 0.f;
                            if (cq + 2 < cmin) p2 = 0.f;
                            if (cq + 3 < cmin) p3 = 0.f;
                        }
                        pk[ch * 16 + q4 / 2] = pack_bf16x2(p0, p1);
                        pk[ch * 16 + q4 / 2 + 1] = pack_bf16x2(p2, p3);
                    }
                    tmem_st_x16(tS + ch * 16, *reinterpret_cast<uint32_t(*)[16]>(&pk[ch * 16]));
                }
                tmem_st_wait();
                tc_fence_before();
                mbar_arrive(p_full);

                mbar_wait(dp_full, dp_ph);
                dp_ph ^= 1;
                if (i > 0) { mbar_wait(dq_full, dq_ph); dq_ph ^= 1; }     // dS buffer free: dK/dQ MMAs of the previous step done
                tc_fence_after();
#pragma unroll
                for (int ch = 0; ch < kBlock / 32; ++ch) {
                    uint32_t r[32];
                    tmem_ld_x32(tDP + ch * 32, r);
                    tmem_ld_wait();
                    uint8_t* half = sDs + (ch / 2) * (kBlock * 128);
#pragma unroll
                    for (int k = 0; k < 4; ++k) {                          // 8 columns = one 16-byte chunk
                        uint32_t w[4];
#pragma unroll
                        for (int j = 0; j < 4; ++j) {
                            const int cq = ch * 32 + k * 8 + j * 2;
                            const uint32_t pw = pk[cq / 2];
                            const float d0 = bf16lo(pw) * (__uint_as_float(r[k * 8 + j * 2]) - delta[cq]);
                            const float d1 = bf16hi(pw) * (__uint_as_float(r[k * 8 + j * 2 + 1]) - delta[cq + 1]);
                            w[j] = pack_bf16x2(d0, d1);
                        }
                        *reinterpret_cast<uint4*>(half + sw128_offset(row, (ch & 1) * 4 + k)) = make_uint4(w[0], w[1], w[2], w[3]);
                    }
                }
                fence_proxy_async_smem();
                tc_fence_before();
                mbar_arrive(ds_full);
                if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1; }
                ++i;
            }
            if (i == 0) continue;
            mbar_wait(dq_full, dq_ph);           // last step's dq_full (not consumed above)
            dq_ph ^= 1;
            // epilogue: dK rows (x softmax scale)
            mbar_wait(dkv_full, dkv_ph);
            dkv_ph ^= 1;
            tc_fence_after();
            float* grow = p.dK + (size_t)c.it.batch * p.k_stride_b + ((size_t)c.v * gm.L + c.it.t0 + row) * p.k_stride_row +
                          (size_t)c.it.head_kv * p.k_stride_h;
            drain_rows<D>(tDK, grow, gm.scale);
            tc_fence_before();
            mbar_arrive(dkv_empty);
        }
    } else if (warp >= 8) {
        // =============================== dQ drain (one query row per thread); dV epilogue ===============================
        const int row = threadIdx.x - 256;
        const uint32_t lane_base = (uint32_t)((warp & 3) * 32) << 16;
        const uint32_t tDQ = tmem + lane_base + Cfg::kColDP, tDV = tmem + lane_base + Cfg::kColDV;
        uint32_t dq_ph = 0, dkv_ph = 0;
        for (int idx = blockIdx.x; idx < total_items; idx += gridDim.x) {
            const BwdItemCtx c = load_bwd_item(p, idx);
            QWalk walk(gm, c.segs, c.nseg, c.g, c.v, c.it.t0, c.it.head_kv);
            int u, h, s0, off, i = 0;
            while (walk.next(u, h, s0, off)) {
                float* grow = p.dQ + (size_t)c.it.batch * p.q_stride_b + ((size_t)u * gm.L + s0 + row) * p.q_stride_row + (size_t)h * p.q_stride_h;
                mbar_wait(dq_full, dq_ph);
                dq_ph ^= 1;
                tc_fence_after();
                uint32_t r[D / 32][32];
#pragma unroll
                for (int ch = 0; ch < D / 32; ++ch) tmem_ld_x32(tDQ + ch * 32, r[ch]);
                tmem_ld_wait();
                tc_fence_before();
                mbar_arrive(dq_empty);           // TMEM columns free again: dP^T of the next step may start
#pragma unroll
                for (int ch = 0; ch < D / 32; ++ch)
#pragma unroll
                    for (int k = 0; k < 32; k += 4)
                        red_add_v4(grow + ch * 32 + k, __uint_as_float(r[ch][k]) * gm.scale, __uint_as_float(r[ch][k + 1]) * gm.scale,
                                   __uint_as_float(r[ch][k + 2]) * gm.scale, __uint_as_float(r[ch][k + 3]) * gm.scale);
                ++i;
            }
            if (i == 0) continue;
            mbar_wait(dkv_full, dkv_ph);
            dkv_ph ^= 1;
            tc_fence_after();
            float* grow = p.dV + (size_t)c.it.batch * p.k_stride_b + ((size_t)c.v * gm.L + c.it.t0 + row) * p.k_stride_row +
                          (size_t)c.it.head_kv * p.k_stride_h;
            drain_rows<D>(tDV, grow, 1.0f);
            tc_fence_before();
            mbar_arrive(dkv_empty);
        }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 2) tmem_dealloc<512>(tmem);
}

}  // namespace

int launch_tile_bwd(const BwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV, const CUtensorMap& tmdO,
                    int num_sms, cudaStream_t stream)
{
    if (p.split) return (int)cudaErrorNotSupported;
    const int total = p.items_per_gpu * p.g_count;
    if (total <= 0) return 0;
    const int grid = total < num_sms ? total : num_sms;
    cudaError_t e;
    if (p.gm.head_dim == 128) {
        e = cudaFuncSetAttribute(tile_bwd_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, BwdCfg<128>::kSmemBytes);
        if (e != cudaSuccess) return (int)e;
        tile_bwd_kernel<128><<<grid, kBwdThreads, BwdCfg<128>::kSmemBytes, stream>>>(tmQ, tmK, tmV, tmdO, p);
    } else {
        e = cudaFuncSetAttribute(tile_bwd_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, BwdCfg<64>::kSmemBytes);
        if (e != cudaSuccess) return (int)e;
        tile_bwd_kernel<64><<<grid, kBwdThreads, BwdCfg<64>::kSmemBytes, stream>>>(tmQ, tmK, tmV, tmdO, p);
    }
    return (int)cudaGetLastError();
}

}  // namespace mesh_attn
