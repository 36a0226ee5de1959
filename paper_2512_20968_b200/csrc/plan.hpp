// plan.hpp -- host-side plan object and the device-resident work-list records shared by the
// planner (planner.cpp) and the kernels (*.cu).  Notation follows the paper: n = a*b
// partitions, tile height a (Q group size), tile width b (KV group size), GPU g has tile
// row r = g / a and tile column c = g mod a.
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "mesh_attn.h"

#if defined(__CUDACC__)
#define MA_HD __host__ __device__
#else
#define MA_HD
#endif

namespace mesh_attn {

constexpr int kBlock = 128;      // rows of a Q sub-tile and keys of a KV block (one UMMA M / N)

// ---- device-visible records (plain structs, no pointers) ------------------------------------

// One tile-forward work item: up to two 128-row Q sub-tiles of (batch, Q partition u, head),
// traversing the KV segments of seg list `seglist` in plan order.
struct FwdItem {
    int16_t batch;
    int16_t u_local;   // Q partition u = r*a + u_local
    int16_t head;      // query head
    int16_t seglist;   // index into SegList table
    int32_t q0;        // first local row (multiple of 128)
    int16_t nrows;     // 128 or 256
    int16_t slot;      // output slot inside the simulated GPU's partial buffers
};

// One tile-backward work item: a 128-key block of (batch, KV partition kv_local, KV head),
// traversing the Q segments of seg list `seglist` (all query heads of the GQA group).
struct BwdItem {
    int16_t batch;
    int16_t kv_local;  // KV partition v = I_g^KV[kv_local]
    int16_t head_kv;
    int16_t seglist;
    int32_t t0;        // first local key row (multiple of 128)
    int32_t pad;
};

// A contiguous run of local rows [begin, end) of partition index `part_local`
// (kv_local for forward seg lists, u_local for backward seg lists); multiples of 128.
struct Seg {
    int32_t part_local;
    int32_t begin;
    int32_t end;
};

struct SegList {
    int32_t offset;
    int32_t count;
};

// Geometry every kernel needs (passed by value inside the kernel parameter block).
struct Geom {
    int32_t n, a, b, L;
    int32_t batch, heads_q, heads_kv, head_dim, group;  // group = heads_q / heads_kv
    int32_t causal, kvr, striped;
    int32_t slots_per_gpu;
    // rows of the query-shaped (Q, O, dO, dQ, lse, delta) and key-shaped (K, V, dK, dV) tensors a call receives:
    // n*L for the simulated-GPU calls; a*L and b*L for the per-rank calls (mesh_attn_rank_*), whose tensors hold only
    // the gathered partitions of ONE GPU, slot k = k-th entry of I_g^Q / I_g^KV
    int32_t rows_q, rows_kv;
    int32_t local;      // 1: per-rank tensors (row of partition = slot*L + s), 0: all n partitions (row = p*L + s)
    float scale;        // softmax scale
    float scale_log2;   // scale * log2(e)
};

// KV partition id of simulated GPU g's kv_local-th footprint entry.
inline MA_HD int kv_partition(const Geom& gm, int g, int kv_local)
{
    const int c = g % gm.a;
    return gm.kvr ? c + kv_local * gm.a : c * gm.b + kv_local;
}

// Partition index that addresses the rows of Q partition u / KV partition v in the tensors of the call
inline MA_HD int q_row_part(const Geom& gm, int u, int u_local) { return gm.local ? u_local : u; }
inline MA_HD int kv_row_part(const Geom& gm, int v, int kv_local) { return gm.local ? kv_local : v; }

// Causal offset of pair (Q_u, KV_v): key local row t is visible to query local row s iff
// t <= s + off.  Contiguous: pos = p*L+s  ->  off = (u-v)*L.  Striped: pos = s*n+p  ->
// off = 0 if v <= u else -1 (reading R6).
inline MA_HD int causal_off(const Geom& gm, int u, int v)
{
    if (gm.striped) return v <= u ? 0 : -1;
    return (u - v) * gm.L;
}

}  // namespace mesh_attn

// ---- host plan -------------------------------------------------------------------------------
struct mesh_attn_plan {
    mesh_attn_plan_desc desc{};
    mesh_attn::Geom geom{};
    int k_q = 1, k_kv = 1;
    float gamma = 1.05f, t_ag_q = 0, t_ag_kv = 0, t_rs_q = 0, t_rs_kv = 0, t_c = 0;

    std::vector<int32_t> am;                      // n*n
    // GOO step lists: rows (step, kind, i, j)
    std::vector<int32_t> steps_fwd, steps_bwd;
    std::vector<std::pair<int, int>> order_fwd, order_bwd;   // compute tasks (i, j) in execution order

    // work-list templates (identical for every simulated GPU up to the partition ids)
    std::vector<mesh_attn::FwdItem> fwd_items;
    std::vector<mesh_attn::BwdItem> bwd_items;
    std::vector<mesh_attn::Seg> fwd_segs, bwd_segs;
    std::vector<mesh_attn::SegList> fwd_seglists, bwd_seglists;
    // chunk-granular forward lists for the GOO executor (mesh_attn_forward_goo): the items of compute task C-i-j
    // (Q chunk i of every Q partition x KV chunk j of every KV partition) are
    // goo_items[goo_task[i*k_kv+j].offset .. +count), partial slot = u_local*k_kv + j
    std::vector<mesh_attn::FwdItem> goo_items;
    std::vector<mesh_attn::SegList> goo_task;
    // the same for the backward executor (mesh_attn_backward_goo): items of C-i-j = the 128-key blocks of KV chunk j of every
    // KV partition, each walking Q chunk i of every Q partition (their seg lists are appended to bwd_segs / bwd_seglists)
    std::vector<mesh_attn::BwdItem> goo_bwd_items;
    std::vector<mesh_attn::SegList> goo_bwd_task;
    // forward items 2k, 2k+1 stream the same K / V blocks on every simulated GPU (planner.cpp): tile_fwd then runs as CTA pairs
    // with tcgen05 cta_group::2 MMAs (head_dim 128, single-operand mode); desc.fwd_pairing = 1 forces the single-CTA kernel
    bool fwd_pairable = false;
    bool fwd_pair() const { return fwd_pairable && desc.fwd_pairing != 1 && desc.precision == 0 && geom.head_dim == 128; }
    // backward items 2k and 2k+1 visit the same Q blocks on every simulated GPU (tile_bwd then runs 2-CTA clusters that
    // share the Q / dO tile loads); desc.bwd_pairing selects never / shared loads only / shared loads + dQ exchange
    bool bwd_pairable = false;
    int bwd_pair_mode() const    // 0 single-CTA kernel, 1 paired (multicast Q / dO tiles), 2 paired + dQ exchange
    {
        if (!bwd_pairable || desc.bwd_pairing == 1) return 0;
        return (desc.bwd_pairing == 2 || desc.precision == 1) ? 1 : 2;
    }

    // device copies (null when no CUDA device was present at creation)
    int device = -1;
    int num_sms = 0;
    void* d_blob = nullptr;
    // status words of the kernels' watchdog (sm100.cuh): pinned host memory mapped into the device; [0] != 0 = a kernel of this
    // plan reported a fault (1: mbarrier wait timed out, 2: misaligned shared memory), [1..4] = block, thread, barrier, parity
    int* h_status = nullptr;
    int* d_status = nullptr;
    int* d_counter = nullptr;    // tile_bwd's work-item counter (inside d_blob), zeroed on the launch stream before every launch
    const mesh_attn::FwdItem* d_fwd_items = nullptr;
    const mesh_attn::FwdItem* d_goo_items = nullptr;
    const mesh_attn::BwdItem* d_goo_bwd_items = nullptr;
    const mesh_attn::BwdItem* d_bwd_items = nullptr;
    const mesh_attn::Seg* d_fwd_segs = nullptr;
    const mesh_attn::Seg* d_bwd_segs = nullptr;
    const mesh_attn::SegList* d_fwd_seglists = nullptr;
    const mesh_attn::SegList* d_bwd_seglists = nullptr;
    // copy streams and events of mesh_attn_step_host (cudaStream_t / cudaEvent_t), created with the device copies
    void* s_h2d = nullptr;
    void* s_d2h = nullptr;
    std::vector<void*> copy_events;               // 2*b + 6
};

namespace mesh_attn {
void set_error(const std::string& msg);
int upload_plan(mesh_attn_plan* plan);   // capi.cu
void free_plan_device(mesh_attn_plan* plan);
}  // namespace mesh_attn
