// planner.cpp -- host-side planner of the Mesh-Attention compute core (mesh_attn_plan).
//
// Builds, from a mesh_attn_plan_desc:
//   - the n x n assignment matrix A, basic tiling (L133) or KV partition
//     rotation (L159);
//   - the GOO step list: k_Q + k_KV all-gather tasks, k_Q reduce-scatter tasks and
//     k_Q*k_KV compute tasks scheduled by the step-based greedy heuristic (L194-230);
//   - per-simulated-GPU ordered tile lists and the device work-list templates the tile
//     kernels consume (the order of compute tasks C-i-j fixes, for every Q chunk i, the
//     order in which its KV chunks j are traversed, and the order in which Q chunks are
//     issued; ordering of heads / row blocks inside a task is the kernel's own concern).
// No CUDA calls here except through mesh_attn::upload_plan (capi.cu).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <new>
#include <set>

#include "plan.hpp"

using namespace mesh_attn;

namespace {

struct Task { int kind, idx; };

// Step-based greedy scheduler.  One collective per step plus the
// compute tasks that were ready at the step boundary, filled until gamma*T_comm.
// `with_rs_kv` adds the backward's RS-dKV-j tasks (ready once every C-*-j is done).
void goo_schedule(int k_q, int k_kv, double t_ag_kv, double t_ag_q, double t_rs_q, double t_rs_kv, double t_c,
                  double gamma, bool with_rs_kv, std::vector<int32_t>& rows, std::vector<std::pair<int, int>>& order)
{
    std::vector<char> q_have(k_q, 0), kv_have(k_kv, 0), rsq(k_q, 0), rskv(k_kv, 0);
    std::vector<char> c_done(k_q * k_kv, 0);
    int next_q = 0, next_kv = 0, n_c = 0, n_rsq = 0, n_rskv = 0, step = 0;
    auto done = [&](int i, int j) -> char& { return c_done[i * k_kv + j]; };
    const int need_rskv = with_rs_kv ? k_kv : 0;

    while (n_c < k_q * k_kv || n_rsq < k_q || n_rskv < need_rskv) {
        // compute tasks ready at this step boundary, in (i, j) priority order (L224: favour
        // tasks completing an earlier Q chunk)
        std::vector<std::pair<int, int>> ready;
        for (int i = 0; i < k_q; ++i)
            for (int j = 0; j < k_kv; ++j)
                if (!done(i, j) && q_have[i] && kv_have[j]) ready.push_back({i, j});

        // candidate collectives: lowest-index unscheduled chunk of each type (L226)
        int best_kind = -1, best_idx = -1;
        double best_profit = -1.0, best_t = 0.0;
        auto consider = [&](int kind, int idx, double unlock, double t_comm) {
            const double profit = unlock / t_comm;              // L216
            if (profit > best_profit) { best_profit = profit; best_kind = kind; best_idx = idx; best_t = t_comm; }
        };
        // order of consideration == tie-break order: AG-KV, AG-Q, RS-Q, RS-KV
        if (next_kv < k_kv) {
            int cnt = 0;
            for (int i = 0; i < k_q; ++i) cnt += q_have[i] ? 1 : 0;
            consider(MESH_ATTN_TASK_AG_KV, next_kv, cnt * t_c, t_ag_kv);
        }
        if (next_q < k_q) {
            int cnt = 0;
            for (int j = 0; j < k_kv; ++j) cnt += kv_have[j] ? 1 : 0;
            consider(MESH_ATTN_TASK_AG_Q, next_q, cnt * t_c, t_ag_q);
        }
        for (int i = 0; i < k_q; ++i) {
            if (rsq[i]) continue;
            bool all = true;
            for (int j = 0; j < k_kv; ++j) all = all && done(i, j);
            if (all) { consider(MESH_ATTN_TASK_RS_Q, i, 0.0, t_rs_q); break; }
        }
        if (with_rs_kv)
            for (int j = 0; j < k_kv; ++j) {
                if (rskv[j]) continue;
                bool all = true;
                for (int i = 0; i < k_q; ++i) all = all && done(i, j);
                if (all) { consider(MESH_ATTN_TASK_RS_KV, j, 0.0, t_rs_kv); break; }
            }

        ++step;
        std::vector<std::pair<int, int>> fill;
        if (best_kind < 0) {
            fill.push_back(ready.front());                      // compute-only step (L230)
        } else {
            rows.insert(rows.end(), {step, best_kind, best_kind == MESH_ATTN_TASK_AG_KV || best_kind == MESH_ATTN_TASK_RS_KV ? -1 : best_idx,
                                     best_kind == MESH_ATTN_TASK_AG_KV || best_kind == MESH_ATTN_TASK_RS_KV ? best_idx : -1});
            double total = 0.0;
            for (auto& t : ready) {                              // L220: until the total reaches T_target
                if (total >= gamma * best_t) break;
                fill.push_back(t);
                total += t_c;
            }
        }
        for (auto& t : fill) {
            rows.insert(rows.end(), {step, MESH_ATTN_TASK_C, t.first, t.second});
            order.push_back(t);
            done(t.first, t.second) = 1;
            ++n_c;
        }
        switch (best_kind) {                                     // the collective completes with the step (L210)
            case MESH_ATTN_TASK_AG_KV: kv_have[best_idx] = 1; ++next_kv; break;
            case MESH_ATTN_TASK_AG_Q: q_have[best_idx] = 1; ++next_q; break;
            case MESH_ATTN_TASK_RS_Q: rsq[best_idx] = 1; ++n_rsq; break;
            case MESH_ATTN_TASK_RS_KV: rskv[best_idx] = 1; ++n_rskv; break;
            default: break;
        }
    }
}

// order == 0: one step holding every collective and every compute task, row-major.
void trivial_schedule(int k_q, int k_kv, bool with_rs_kv, std::vector<int32_t>& rows, std::vector<std::pair<int, int>>& order)
{
    for (int j = 0; j < k_kv; ++j) rows.insert(rows.end(), {1, MESH_ATTN_TASK_AG_KV, -1, j});
    for (int i = 0; i < k_q; ++i) rows.insert(rows.end(), {1, MESH_ATTN_TASK_AG_Q, i, -1});
    for (int i = 0; i < k_q; ++i)
        for (int j = 0; j < k_kv; ++j) { rows.insert(rows.end(), {1, MESH_ATTN_TASK_C, i, j}); order.push_back({i, j}); }
    for (int i = 0; i < k_q; ++i) rows.insert(rows.end(), {1, MESH_ATTN_TASK_RS_Q, i, -1});
    if (with_rs_kv) for (int j = 0; j < k_kv; ++j) rows.insert(rows.end(), {1, MESH_ATTN_TASK_RS_KV, -1, j});
}

int fail(int code, const std::string& msg) { set_error(msg); return code; }

template <class T> std::vector<T> first_appearance(const std::vector<std::pair<int, int>>& order, bool first)
{
    std::vector<T> out;
    for (auto& t : order) {
        T x = first ? t.first : t.second;
        if (std::find(out.begin(), out.end(), x) == out.end()) out.push_back(x);
    }
    return out;
}

void build_worklists(mesh_attn_plan* p)
{
    const Geom& gm = p->geom;
    const int Lq = gm.L / p->k_q, Lkv = gm.L / p->k_kv;
    const bool per_pair = p->desc.partial_mode == 1;

    // ---------- forward: item = (batch, u_local, head, <=256-row block) ----------
    // Q chunks in order of first appearance in the compute order; for Q chunk i the KV chunks
    // in the order C-i-j tasks execute.
    const std::vector<int> q_chunks = first_appearance<int>(p->order_fwd, true);
    // seg lists: fused mode -> one list per Q chunk (all b partitions per KV chunk, partition-major inside a
    // chunk as in tile_list); per-pair mode -> one list per (Q chunk, kv_local).  They do not depend on the batch
    // index: built once (FwdItem::seglist is 16 bits; plan_create rejects plans with more than 32767 lists).
    const int n_lists = per_pair ? gm.b : 1;
    std::vector<std::vector<int>> fwd_list_ids(p->k_q);
    for (int i : q_chunks) {
        std::vector<int> kv_chunks;
        for (auto& t : p->order_fwd) if (t.first == i) kv_chunks.push_back(t.second);
        fwd_list_ids[i].resize(n_lists);
        for (int l = 0; l < n_lists; ++l) {
            SegList sl{(int32_t)p->fwd_segs.size(), 0};
            for (int j : kv_chunks)
                for (int jj = 0; jj < gm.b; ++jj) {
                    if (per_pair && jj != l) continue;
                    p->fwd_segs.push_back(Seg{jj, j * Lkv, (j + 1) * Lkv});
                    ++sl.count;
                }
            fwd_list_ids[i][l] = (int)p->fwd_seglists.size();
            p->fwd_seglists.push_back(sl);
        }
    }
    for (int bt = 0; bt < gm.batch; ++bt)
        for (int i : q_chunks) {
            const std::vector<int>& list_ids = fwd_list_ids[i];
            for (int hk = 0; hk < gm.heads_kv; ++hk) {
                std::vector<FwdItem> grp;
                for (int l = 0; l < n_lists; ++l)
                    for (int h = hk * gm.group; h < (hk + 1) * gm.group; ++h)
                        for (int ul = 0; ul < gm.a; ++ul)
                            for (int q0 = i * Lq; q0 < (i + 1) * Lq; q0 += 2 * kBlock) {
                                FwdItem it{};
                                it.batch = (int16_t)bt;
                                it.u_local = (int16_t)ul;
                                it.head = (int16_t)h;
                                it.seglist = (int16_t)list_ids[l];
                                it.q0 = q0;
                                it.nrows = (int16_t)std::min(2 * kBlock, (i + 1) * Lq - q0);
                                it.slot = (int16_t)(per_pair ? ul * gm.b + l : ul);
                                grp.push_back(it);
                            }
                // causal: rows further down see more keys -> issue the longest items first
                if (gm.causal)
                    std::stable_sort(grp.begin(), grp.end(), [](const FwdItem& x, const FwdItem& y) { return x.q0 > y.q0; });
                p->fwd_items.insert(p->fwd_items.end(), grp.begin(), grp.end());
            }
        }

    // ---------- forward, one list per compute task C-i-j (GOO executor) ----------
    p->goo_task.assign((size_t)p->k_q * p->k_kv, SegList{0, 0});
    for (auto& task : p->order_fwd) {
        const int i = task.first, j = task.second;
        SegList sl{(int32_t)p->fwd_segs.size(), 0};
        for (int jj = 0; jj < gm.b; ++jj) { p->fwd_segs.push_back(Seg{jj, j * Lkv, (j + 1) * Lkv}); ++sl.count; }
        const int list_id = (int)p->fwd_seglists.size();
        p->fwd_seglists.push_back(sl);
        SegList range{(int32_t)p->goo_items.size(), 0};
        for (int bt = 0; bt < gm.batch; ++bt)
            for (int hk = 0; hk < gm.heads_kv; ++hk) {
                std::vector<FwdItem> grp;
                for (int h = hk * gm.group; h < (hk + 1) * gm.group; ++h)
                    for (int ul = 0; ul < gm.a; ++ul)
                        for (int q0 = i * Lq; q0 < (i + 1) * Lq; q0 += 2 * kBlock) {
                            FwdItem it{};
                            it.batch = (int16_t)bt;
                            it.u_local = (int16_t)ul;
                            it.head = (int16_t)h;
                            it.seglist = (int16_t)list_id;
                            it.q0 = q0;
                            it.nrows = (int16_t)std::min(2 * kBlock, (i + 1) * Lq - q0);
                            it.slot = (int16_t)(ul * p->k_kv + j);
                            grp.push_back(it);
                        }
                if (gm.causal)
                    std::stable_sort(grp.begin(), grp.end(), [](const FwdItem& x, const FwdItem& y) { return x.q0 > y.q0; });
                p->goo_items.insert(p->goo_items.end(), grp.begin(), grp.end());
            }
        range.count = (int32_t)p->goo_items.size() - range.offset;
        p->goo_task[(size_t)i * p->k_kv + j] = range;
    }

    // ---------- backward: item = (batch, kv_local, kv head, 128-key block) ----------
    // The Q sweep of a key block (every Q chunk of every Q partition of the tile, in the order the C-i-j tasks of KV chunk j
    // execute) is cut into PIECES of at most piece_blocks 128-row blocks, a piece being a run of consecutive segments; a work
    // item is (key block, piece), and all key blocks of a (KV chunk, head, piece) are adjacent in the list, so that the CTAs
    // running at the same time (the kernels take items in list order) sweep the same Q / dO / dQ rows and find them in L2.
    // dK / dV of a key block are accumulated per piece and added atomically like every other partial sum (Alg.3 l.7, PAPER.md
    // L255).  Default: pieces whose working set -- rows x (query heads of a GQA group) x head_dim x (2 + 2 + 4) bytes of Q, dO,
    // dQ -- is 32 MiB, but not shorter than 64 blocks (every item pays a K / V load and a dK / dV epilogue).  Measured
    // (profiles/r02_v1_README.md): BASELINE.json configs[3] (GQA 4:1, 128 MiB per sweep) 908 (one piece) / 957 (64 MiB) /
    // 990 (32 MiB) / 979 (16 MiB) TFLOP/s; configs[4] (64 MiB per sweep) 990 / 990 (32 MiB) / 980 (8 MiB).
    const long long auto_blocks = (32ll << 20) / ((long long)kBlock * gm.group * gm.head_dim * 8);
    const int piece_blocks = p->desc.bwd_piece_blocks > 0 ? p->desc.bwd_piece_blocks : (int)std::max<long long>(64, auto_blocks);
    const std::vector<int> kv_chunks_b = first_appearance<int>(p->order_bwd, false);
    struct Piece { int list_id, max_end; };
    std::vector<std::vector<Piece>> bwd_pieces(p->k_kv);   // seg lists per KV chunk, shared by every batch index
    for (int j : kv_chunks_b) {
        std::vector<int> qc;
        for (auto& t : p->order_bwd) if (t.second == j) qc.push_back(t.first);
        std::vector<Seg> segs;
        for (int i : qc)
            for (int ul = 0; ul < gm.a; ++ul) segs.push_back(Seg{ul, i * Lq, (i + 1) * Lq});
        for (size_t s0 = 0; s0 < segs.size();) {
            SegList sl{(int32_t)p->bwd_segs.size(), 0};
            int blocks = 0, max_end = 0;
            while (s0 < segs.size() && (sl.count == 0 || blocks + Lq / kBlock <= piece_blocks)) {
                p->bwd_segs.push_back(segs[s0]);
                max_end = std::max(max_end, (int)segs[s0].end);
                blocks += Lq / kBlock;
                ++sl.count;
                ++s0;
            }
            bwd_pieces[j].push_back(Piece{(int)p->bwd_seglists.size(), max_end});
            p->bwd_seglists.push_back(sl);
        }
    }
    for (int bt = 0; bt < gm.batch; ++bt)
        for (int j : kv_chunks_b)
            for (int hk = 0; hk < gm.heads_kv; ++hk)
                for (const Piece& pc : bwd_pieces[j]) {
                    std::vector<BwdItem> grp;
                    for (int jj = 0; jj < gm.b; ++jj)
                        for (int t0 = j * Lkv; t0 < (j + 1) * Lkv; t0 += kBlock) {
                            // striped causal layout: key row t is seen by the local query rows >= t (offset 0 or -1, plan.hpp
                            // causal_off), whatever the partitions: a piece that ends at or before t0 has no step for this block
                            if (gm.causal && gm.striped && t0 >= pc.max_end) continue;
                            grp.push_back(BwdItem{(int16_t)bt, (int16_t)jj, (int16_t)hk, (int16_t)pc.list_id, t0, 0});
                        }
                    // causal: early keys are seen by more queries -> longest first
                    if (gm.causal)
                        std::stable_sort(grp.begin(), grp.end(), [](const BwdItem& x, const BwdItem& y) { return x.t0 < y.t0; });
                    p->bwd_items.insert(p->bwd_items.end(), grp.begin(), grp.end());
                }

    // ---------- backward, chunk-granular (GOO executor): one item list per compute task C-i-j ----------
    p->goo_bwd_task.assign((size_t)p->k_q * p->k_kv, SegList{0, 0});
    std::vector<int> goo_list_id(p->k_q);                  // the Q rows of chunk i of every Q partition: one list per Q chunk
    for (int i = 0; i < p->k_q; ++i) {
        SegList sl{(int32_t)p->bwd_segs.size(), 0};
        for (int ul = 0; ul < gm.a; ++ul) { p->bwd_segs.push_back(Seg{ul, i * Lq, (i + 1) * Lq}); ++sl.count; }
        goo_list_id[i] = (int)p->bwd_seglists.size();
        p->bwd_seglists.push_back(sl);
    }
    for (int i = 0; i < p->k_q; ++i)
        for (int j = 0; j < p->k_kv; ++j) {
            SegList range{(int32_t)p->goo_bwd_items.size(), 0};
            for (int bt = 0; bt < gm.batch; ++bt) {
                const int list_id = goo_list_id[i];
                for (int hk = 0; hk < gm.heads_kv; ++hk) {
                    std::vector<BwdItem> grp;
                    for (int jj = 0; jj < gm.b; ++jj)
                        for (int t0 = j * Lkv; t0 < (j + 1) * Lkv; t0 += kBlock)
                            grp.push_back(BwdItem{(int16_t)bt, (int16_t)jj, (int16_t)hk, (int16_t)list_id, t0, 0});
                    if (gm.causal)
                        std::stable_sort(grp.begin(), grp.end(), [](const BwdItem& x, const BwdItem& y) { return x.t0 < y.t0; });
                    p->goo_bwd_items.insert(p->goo_bwd_items.end(), grp.begin(), grp.end());
                }
            }
            range.count = (int32_t)p->goo_bwd_items.size() - range.offset;
            p->goo_bwd_task[(size_t)i * p->k_kv + j] = range;
        }
}

// First Q block of segment sg that item (kv_local, t0) of simulated GPU g visits (the rule of tile_bwd.cu's QWalk).
int bwd_first_row(const Geom& gm, int g, const Seg& sg, int kv_local, int t0)
{
    if (!gm.causal) return sg.begin;
    const int u = (g / gm.a) * gm.a + sg.part_local, v = kv_partition(gm, g, kv_local);
    const int x = t0 - causal_off(gm, u, v) - (kBlock - 1);
    return x > sg.begin ? std::min(sg.end, ((x + kBlock - 1) / kBlock) * kBlock) : sg.begin;
}

// Do backward items 2k and 2k+1 walk the same (Q partition, head, block) sequence on every simulated GPU?
bool bwd_items_pairable(const mesh_attn_plan* p)
{
    const Geom& gm = p->geom;
    const size_t cnt = p->bwd_items.size();
    if (cnt < 2 || cnt % 2) return false;
    // the walk depends on g only through the causal offsets of the contiguous layout
    const int g_span = (gm.causal && !gm.striped) ? gm.n : 1;
    for (int g = 0; g < g_span; ++g)
        for (size_t k = 0; k < cnt; k += 2) {
            const BwdItem &x = p->bwd_items[k], &y = p->bwd_items[k + 1];
            if (x.batch != y.batch || x.head_kv != y.head_kv || x.seglist != y.seglist) return false;
            if (!gm.causal) continue;
            const SegList sl = p->bwd_seglists[x.seglist];
            for (int i = 0; i < sl.count; ++i) {
                const Seg& sg = p->bwd_segs[sl.offset + i];
                if (bwd_first_row(gm, g, sg, x.kv_local, x.t0) != bwd_first_row(gm, g, sg, y.kv_local, y.t0)) return false;
            }
        }
    return true;
}

// Do forward items 2k and 2k+1 stream the same K / V blocks (same batch, KV head, partitions and key rows) on every simulated GPU?
// (tile_fwd.cu kv_range, restated: the visible key rows of a segment are clipped at the item's last query row.)
bool fwd_items_pairable(const mesh_attn_plan* p)
{
    const Geom& gm = p->geom;
    const size_t cnt = p->fwd_items.size();
    if (cnt < 2 || cnt % 2) return false;
    for (size_t k = 0; k < cnt; k += 2) {
        const FwdItem &x = p->fwd_items[k], &y = p->fwd_items[k + 1];
        if (x.batch != y.batch || x.head / gm.group != y.head / gm.group || x.seglist != y.seglist || x.nrows != y.nrows) return false;
        if (!gm.causal) continue;
        const SegList sl = p->fwd_seglists[x.seglist];
        for (int g = 0; g < gm.n; ++g) {
            const int ux = (g / gm.a) * gm.a + x.u_local, uy = (g / gm.a) * gm.a + y.u_local;
            for (int i = 0; i < sl.count; ++i) {
                const Seg& sg = p->fwd_segs[sl.offset + i];
                const int v = kv_partition(gm, g, sg.part_local);
                auto t_hi = [&](const FwdItem& it, int u) {
                    const int lim = it.q0 + it.nrows - 1 + causal_off(gm, u, v);
                    return lim < sg.begin ? sg.begin : std::min<int>(sg.end, (lim / kBlock + 1) * kBlock);
                };
                if (t_hi(x, ux) != t_hi(y, uy)) return false;
            }
        }
    }
    return true;
}

// number of 128x128 score blocks the forward computes for one simulated GPU g and one head
int64_t fwd_blocks_of_gpu(const mesh_attn_plan* p, int g)
{
    const Geom& gm = p->geom;
    const int r = g / gm.a;
    int64_t blocks = 0;
    for (int ul = 0; ul < gm.a; ++ul)
        for (int jj = 0; jj < gm.b; ++jj) {
            const int u = r * gm.a + ul, v = kv_partition(gm, g, jj);
            for (int q0 = 0; q0 < gm.L; q0 += kBlock)
                for (int t0 = 0; t0 < gm.L; t0 += kBlock) {
                    if (gm.causal && t0 > q0 + kBlock - 1 + causal_off(gm, u, v)) continue;
                    ++blocks;
                }
        }
    return blocks;
}

}  // namespace

extern "C" int mesh_attn_plan_create(const mesh_attn_plan_desc* d, mesh_attn_plan** out)
{
    if (out) *out = nullptr;
    if (!d || !out) return fail(MESH_ATTN_EINVAL, "plan_create: null argument");
    if (d->n <= 0 || d->a <= 0 || d->b <= 0 || d->n != d->a * d->b)
        return fail(MESH_ATTN_EINVAL, "plan_create: need n == a*b with positive a, b (PAPER.md L116)");
    if (d->n > 4096) return fail(MESH_ATTN_EINVAL, "plan_create: n too large");
    if (d->batch <= 0 || d->batch > 32767 || d->seq_total <= 0 || d->heads_q <= 0 || d->heads_kv <= 0)
        return fail(MESH_ATTN_EINVAL, "plan_create: batch, seq_total, heads must be positive");
    if (d->seq_total % d->n) return fail(MESH_ATTN_EINVAL, "plan_create: seq_total must be divisible by n");
    const int L = d->seq_total / d->n;
    if (L % kBlock) return fail(MESH_ATTN_EINVAL, "plan_create: partition length L = seq_total/n must be a multiple of 128");
    if (d->heads_q % d->heads_kv) return fail(MESH_ATTN_EINVAL, "plan_create: heads_q must be a multiple of heads_kv (PAPER.md L427)");
    if (d->heads_q > 32767) return fail(MESH_ATTN_EINVAL, "plan_create: too many heads");
    const int U = d->usp_lanes <= 0 ? 1 : d->usp_lanes;
    if (d->heads_kv % U) return fail(MESH_ATTN_EINVAL, "plan_create: heads_kv must be a multiple of usp_lanes (PAPER.md L372-389: each lane holds 1/U of the heads)");
    if ((int64_t)d->n * U > 32767) return fail(MESH_ATTN_EINVAL, "plan_create: n * usp_lanes too large");
    if (d->head_dim != 64 && d->head_dim != 128) return fail(MESH_ATTN_EUNSUPPORTED, "plan_create: head_dim must be 64 or 128");
    for (int v : {d->causal, d->kvr, d->order, d->seq_layout, d->tensor_layout, d->partial_mode, d->precision})
        if (v != 0 && v != 1) return fail(MESH_ATTN_EINVAL, "plan_create: flag fields must be 0 or 1");
    if (d->bwd_piece_blocks < 0) return fail(MESH_ATTN_EINVAL, "plan_create: bwd_piece_blocks must be >= 0 (0 = default)");
    if (d->bwd_pairing < 0 || d->bwd_pairing > 2) return fail(MESH_ATTN_EINVAL, "plan_create: bwd_pairing must be 0 (auto), 1 (never) or 2 (shared tile loads only)");
    if (d->out_dtype < 0 || d->out_dtype > 1) return fail(MESH_ATTN_EINVAL, "plan_create: out_dtype must be 0 (fp32) or 1 (bf16)");
    if (d->fwd_pairing < 0 || d->fwd_pairing > 1) return fail(MESH_ATTN_EINVAL, "plan_create: fwd_pairing must be 0 (auto) or 1 (never)");
    const int k_q = d->k_q <= 0 ? 1 : d->k_q, k_kv = d->k_kv <= 0 ? 1 : d->k_kv;
    if (k_q * k_kv > 16) return fail(MESH_ATTN_EINVAL, "plan_create: k_q*k_kv must be <= 16 (PAPER.md L206)");
    if (L % k_q || (L / k_q) % kBlock || L % k_kv || (L / k_kv) % kBlock)
        return fail(MESH_ATTN_EINVAL, "plan_create: L/k_q and L/k_kv must be multiples of 128");
    if ((int64_t)d->a * d->b > 32767 && d->partial_mode == 1) return fail(MESH_ATTN_EINVAL, "plan_create: too many slots");
    if ((int64_t)d->batch * d->seq_total >= (1ll << 31)) return fail(MESH_ATTN_EINVAL, "plan_create: batch*seq_total must be < 2^31");

    mesh_attn_plan* p = new (std::nothrow) mesh_attn_plan();
    if (!p) return fail(MESH_ATTN_ENOMEM, "plan_create: out of host memory");
    p->desc = *d;
    Geom& gm = p->geom;
    gm.n = d->n; gm.a = d->a; gm.b = d->b; gm.L = L;
    gm.batch = d->batch; gm.heads_q = d->heads_q / U; gm.heads_kv = d->heads_kv / U; gm.head_dim = d->head_dim;   // one lane's heads
    gm.group = d->heads_q / d->heads_kv;
    gm.causal = d->causal; gm.kvr = d->kvr; gm.striped = d->seq_layout;
    gm.slots_per_gpu = d->partial_mode == 1 ? d->a * d->b : d->a;
    gm.rows_q = gm.rows_kv = d->seq_total;   // the simulated-GPU calls see all n partitions; mesh_attn_rank_* override
    gm.local = 0;
    gm.scale = d->softmax_scale > 0.f ? d->softmax_scale : 1.0f / std::sqrt((float)d->head_dim);
    gm.scale_log2 = (float)((double)gm.scale * 1.4426950408889634);
    p->k_q = k_q; p->k_kv = k_kv;
    p->gamma = d->gamma > 0.f ? d->gamma : 1.05f;

    // cost model: the caller's profiled costs (L218) or a bytes/flops default (R11)
    if (d->t_ag_q > 0.f && d->t_ag_kv > 0.f && d->t_rs_q > 0.f && d->t_c > 0.f) {
        p->t_ag_q = d->t_ag_q; p->t_ag_kv = d->t_ag_kv; p->t_rs_q = d->t_rs_q; p->t_c = d->t_c;
        p->t_rs_kv = 2.0f * d->t_rs_q;
    } else {
        const double bw = 4.0e11, lat = 2.0e-5, rate = 8.0e14;
        const double unit_q = (double)L * gm.heads_q * d->head_dim * 2.0, unit_kv = (double)L * gm.heads_kv * d->head_dim * 2.0;
        p->t_ag_q = (float)((d->a - 1) * unit_q / k_q / bw + lat);
        p->t_ag_kv = (float)((d->b - 1) * 2.0 * unit_kv / k_kv / bw + lat);
        p->t_rs_q = (float)((d->a - 1) * unit_q / k_q / bw + lat);
        p->t_rs_kv = (float)((d->b - 1) * 2.0 * unit_kv / k_kv / bw + lat);
        p->t_c = (float)(4.0 * d->head_dim * gm.heads_q * ((double)d->a * L / k_q) * ((double)d->b * L / k_kv) * (d->causal ? 0.5 : 1.0) / rate);
    }

    // assignment matrix
    p->am.assign((size_t)d->n * d->n, -1);
    for (int i = 0; i < d->n; ++i)
        for (int j = 0; j < d->n; ++j) {
            const int r = i / d->a, c = d->kvr ? j % d->a : j / d->b;
            p->am[(size_t)i * d->n + j] = r * d->a + c;
        }

    if (d->order == 1) {
        goo_schedule(k_q, k_kv, p->t_ag_kv, p->t_ag_q, p->t_rs_q, 0.0, p->t_c, p->gamma, false, p->steps_fwd, p->order_fwd);
        // backward (PAPER.md L238 omits the schedule; reading R12, parity unpinned):
        // AG of Q,O,dO costs 3 units of Q, RS-dKV moves K and V gradients, compute is 2.5x forward.
        goo_schedule(k_q, k_kv, p->t_ag_kv, 3.0 * p->t_ag_q, p->t_rs_q, p->t_rs_kv, 2.5 * p->t_c, p->gamma, true, p->steps_bwd, p->order_bwd);
    } else {
        trivial_schedule(k_q, k_kv, false, p->steps_fwd, p->order_fwd);
        trivial_schedule(k_q, k_kv, true, p->steps_bwd, p->order_bwd);
    }
    build_worklists(p);
    p->bwd_pairable = bwd_items_pairable(p);
    p->fwd_pairable = fwd_items_pairable(p);
    if (p->fwd_seglists.size() > 32767 || p->bwd_seglists.size() > 32767) {     // FwdItem / BwdItem::seglist are 16 bits
        delete p;
        return fail(MESH_ATTN_EINVAL, "plan_create: too many segment lists (k_q, k_kv, b too large for partial_mode 1)");
    }

    const int rc = upload_plan(p);
    if (rc != MESH_ATTN_OK) { delete p; return rc; }
    *out = p;
    return MESH_ATTN_OK;
}

extern "C" void mesh_attn_plan_destroy(mesh_attn_plan* p)
{
    if (!p) return;
    free_plan_device(p);
    delete p;
}

extern "C" int mesh_attn_plan_am(const mesh_attn_plan* p, int32_t* am)
{
    if (!p || !am) return fail(MESH_ATTN_EINVAL, "plan_am: null argument");
    std::memcpy(am, p->am.data(), p->am.size() * sizeof(int32_t));
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_plan_footprint(const mesh_attn_plan* p, int32_t g, int32_t* iq, int32_t* ikv)
{
    if (!p || !iq || !ikv) return fail(MESH_ATTN_EINVAL, "plan_footprint: null argument");
    if (g < 0 || g >= p->geom.n) return fail(MESH_ATTN_EINVAL, "plan_footprint: g out of range");
    for (int x = 0; x < p->geom.a; ++x) iq[x] = (g / p->geom.a) * p->geom.a + x;
    for (int t = 0; t < p->geom.b; ++t) ikv[t] = kv_partition(p->geom, g, t);
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_plan_tiles(const mesh_attn_plan* p, int32_t g, int32_t* tiles, int32_t capacity, int32_t* count)
{
    if (!p || !count) return fail(MESH_ATTN_EINVAL, "plan_tiles: null argument");
    if (g < 0 || g >= p->geom.n) return fail(MESH_ATTN_EINVAL, "plan_tiles: g out of range");
    const Geom& gm = p->geom;
    const int total = gm.a * gm.b * p->k_q * p->k_kv;
    *count = total;
    if (!tiles || capacity < total) return fail(MESH_ATTN_EWORKSPACE, "plan_tiles: capacity too small");
    int k = 0;
    for (auto& t : p->order_fwd)
        for (int ul = 0; ul < gm.a; ++ul)
            for (int jj = 0; jj < gm.b; ++jj) {
                tiles[4 * k + 0] = (g / gm.a) * gm.a + ul;
                tiles[4 * k + 1] = kv_partition(gm, g, jj);
                tiles[4 * k + 2] = t.first;
                tiles[4 * k + 3] = t.second;
                ++k;
            }
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_plan_steps(const mesh_attn_plan* p, int32_t pass, int32_t* steps, int32_t capacity, int32_t* count)
{
    if (!p || !count) return fail(MESH_ATTN_EINVAL, "plan_steps: null argument");
    if (pass != 0 && pass != 1) return fail(MESH_ATTN_EINVAL, "plan_steps: pass must be 0 or 1");
    const std::vector<int32_t>& rows = pass == 0 ? p->steps_fwd : p->steps_bwd;
    *count = (int32_t)(rows.size() / 4);
    if (!steps || capacity < *count) return fail(MESH_ATTN_EWORKSPACE, "plan_steps: capacity too small");
    std::memcpy(steps, rows.data(), rows.size() * sizeof(int32_t));
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_plan_timeline(const mesh_attn_plan* p, int32_t pass, double* makespan, double* serial, double* exposed_comm)
{
    if (!p || !makespan || !serial || !exposed_comm) return fail(MESH_ATTN_EINVAL, "plan_timeline: null pointer");
    if (pass != 0 && pass != 1) return fail(MESH_ATTN_EINVAL, "plan_timeline: pass must be 0 or 1");
    const std::vector<int32_t>& rows = pass == 0 ? p->steps_fwd : p->steps_bwd;
    // the same task costs goo_schedule was given for this pass
    const double t_c = pass == 0 ? p->t_c : 2.5 * p->t_c;
    auto cost = [&](int kind) -> double {
        switch (kind) {
            case MESH_ATTN_TASK_AG_KV: return p->t_ag_kv;
            case MESH_ATTN_TASK_AG_Q: return pass == 0 ? p->t_ag_q : 3.0 * p->t_ag_q;
            case MESH_ATTN_TASK_RS_Q: return p->t_rs_q;
            case MESH_ATTN_TASK_RS_KV: return p->t_rs_kv;
            default: return t_c;
        }
    };
    double total = 0.0, ser = 0.0, compute = 0.0;
    for (size_t r = 0; r < rows.size();) {                 // rows (step, kind, i, j), grouped by step
        const int step = rows[r];
        double comm = 0.0, comp = 0.0;
        for (; r < rows.size() && rows[r] == step; r += 4) {
            const int kind = rows[r + 1];
            if (kind == MESH_ATTN_TASK_C) comp += cost(kind);
            else comm += cost(kind);
        }
        total += comm > comp ? comm : comp;
        ser += comm + comp;
        compute += comp;
    }
    if (p->desc.order == 0) total = ser;                   // row-major order schedules no overlap: gather, compute, reduce
    *makespan = total;
    *serial = ser;
    *exposed_comm = total - compute;
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_plan_tam_units(const mesh_attn_plan* p, int32_t gpus_per_node, int32_t alpha, int32_t node, int64_t* q_units,
                             int64_t* kv_units)
{
    if (!p || !q_units || !kv_units) return fail(MESH_ATTN_EINVAL, "plan_tam_units: null pointer");
    const Geom& gm = p->geom;
    if (gpus_per_node <= 0 || alpha <= 0 || gm.a % alpha || gpus_per_node % alpha || gm.b % (gpus_per_node / alpha))
        return fail(MESH_ATTN_EINVAL, "plan_tam_units: alpha must divide a and gpus_per_node, gpus_per_node/alpha must divide b");
    const int rows_per_node = gpus_per_node / alpha, tiles_per_row = gm.a / alpha;
    const int nodes = gm.n / gpus_per_node;
    if (node < 0 || node >= nodes) return fail(MESH_ATTN_EINVAL, "plan_tam_units: node out of range");
    // logical GPU g sits at mesh row r = g / a (its Q group) and column c = g mod a (its KV group)
    auto node_of = [&](int g) { return ((g / gm.a) / rows_per_node) * tiles_per_row + (g % gm.a) / alpha; };
    std::set<int> rows, cols;
    for (int g = 0; g < gm.n; ++g)
        if (node_of(g) == node) { rows.insert(g / gm.a); cols.insert(g % gm.a); }
    int64_t q = 0, kv = 0;
    for (int r : rows)                                     // Q group r = {r a .. r a + a - 1}
        for (int x = r * gm.a; x < (r + 1) * gm.a; ++x)
            if (node_of(x) != node) q += 2;
    for (int c : cols)                                     // KV group c = {c, c + a, c + 2a, ...}
        for (int x = c; x < gm.n; x += gm.a)
            if (node_of(x) != node) kv += 2;
    *q_units = q;
    *kv_units = kv;
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_plan_query(const mesh_attn_plan* p, int32_t what, int64_t* value)
{
    if (!p || !value) return fail(MESH_ATTN_EINVAL, "plan_query: null argument");
    const Geom& gm = p->geom;
    const int64_t N = (int64_t)gm.n * gm.L;
    const long double pairs = gm.causal ? (long double)N * (N + 1) / 2 : (long double)N * N;
    const int64_t unit = (int64_t)gm.batch * gm.L * gm.heads_q;     // (row, head) pairs of one partition of one lane
    const int64_t U = p->desc.usp_lanes > 1 ? p->desc.usp_lanes : 1, Hq = p->desc.heads_q, Hkv = p->desc.heads_kv;
    switch (what) {
        case MESH_ATTN_Q_PARTIAL_O_BYTES: *value = (int64_t)gm.slots_per_gpu * unit * gm.head_dim * 4; break;
        case MESH_ATTN_Q_PARTIAL_LSE_BYTES: *value = (int64_t)gm.slots_per_gpu * unit * 4; break;
        case MESH_ATTN_Q_SLOTS_PER_GPU: *value = gm.slots_per_gpu; break;
        case MESH_ATTN_Q_FLOPS_FWD: *value = (int64_t)(4.0L * gm.head_dim * Hq * gm.batch * pairs); break;
        case MESH_ATTN_Q_FLOPS_BWD: *value = (int64_t)(10.0L * gm.head_dim * Hq * gm.batch * pairs); break;
        case MESH_ATTN_Q_WAVES: *value = gm.b * U; break;
        case MESH_ATTN_Q_MERGE_BYTES: {
            // per output (row, head): m partial rows + m lse read, one row + one lse written (fp32)
            const int64_t m = p->desc.partial_mode == 1 ? (int64_t)gm.a * gm.b : gm.a;
            *value = (int64_t)gm.a * unit * (m + 1) * (gm.head_dim * 4 + 4);
            break;
        }
        case MESH_ATTN_Q_FWD_ITEMS_PER_GPU: *value = (int64_t)p->fwd_items.size(); break;
        case MESH_ATTN_Q_BWD_ITEMS_PER_GPU: *value = (int64_t)p->bwd_items.size(); break;
        case MESH_ATTN_Q_BLOCKS_FWD: {
            int64_t blocks = 0;
            for (int g = 0; g < gm.n; ++g) blocks += fwd_blocks_of_gpu(p, g);
            *value = blocks * Hq * gm.batch;
            break;
        }
        case MESH_ATTN_Q_COMM_UNITS: {
            // every remote Q (+ its returned partial O) counts 1 + 1, every remote KV counts 2
            int64_t units = 0;
            for (int g = 0; g < gm.n; ++g) {
                std::set<int> iq, ikv;
                for (int i = 0; i < gm.n; ++i)
                    for (int j = 0; j < gm.n; ++j)
                        if (p->am[(size_t)i * gm.n + j] == g) { iq.insert(i); ikv.insert(j); }
                iq.erase(g); ikv.erase(g);
                units += 2 * (int64_t)iq.size() + 2 * (int64_t)ikv.size();
            }
            *value = units;
            break;
        }
        case MESH_ATTN_Q_HAS_DEVICE: *value = p->d_blob ? 1 : 0; break;
        case MESH_ATTN_Q_MESH_COMM_BYTES_FWD:
        case MESH_ATTN_Q_MESH_COMM_BYTES_BWD: {
            // each GPU gathers (a-1) remote Q and returns as many partial O, and gathers (b-1) remote
            // K and V: 2(a-1) + 2(b-1) units of N d / n elements; the backward moves twice that (Table 5)
            const long double unit = (long double)gm.batch * gm.n * gm.L * gm.heads_q * gm.head_dim / gm.n * 2.0L;
            const long double fwd = 2.0L * (gm.a + gm.b - 2) * unit;
            *value = (int64_t)(what == MESH_ATTN_Q_MESH_COMM_BYTES_FWD ? fwd : 2.0L * fwd);
            break;
        }
        case MESH_ATTN_Q_RING_COMM_BYTES_FWD: {
            const long double Nd = (long double)gm.batch * gm.n * gm.L * gm.heads_q * gm.head_dim * 2.0L;
            *value = (int64_t)((2.0L - 2.0L / gm.n) * Nd);
            break;
        }
        case MESH_ATTN_Q_BWD_WS_BYTES:
            *value = 2ll * gm.batch * Hq * (int64_t)gm.n * gm.L * 4;
            if (p->desc.out_dtype == 1)         // + the fp32 accumulators of dQ, dK, dV
                *value += (int64_t)gm.batch * gm.n * gm.L * ((int64_t)p->desc.heads_q + 2ll * p->desc.heads_kv) * gm.head_dim * 4;
            break;
        case MESH_ATTN_Q_USP_LANES: *value = U; break;
        case MESH_ATTN_Q_GOO_PARTIAL_O_BYTES: *value = (int64_t)gm.a * p->k_kv * unit * gm.head_dim * 4; break;
        case MESH_ATTN_Q_GOO_PARTIAL_LSE_BYTES: *value = (int64_t)gm.a * p->k_kv * unit * 4; break;
        case MESH_ATTN_Q_GOO_COMM_BYTES: {
            // what the forward step list moves for ONE Q group (its a simulated GPUs): k_q AG-Q + k_q RS-Q + k_kv AG-KV tasks
            const int64_t unit_q = (int64_t)gm.batch * (gm.L / p->k_q) * gm.heads_q * gm.head_dim * 2;
            const int64_t unit_kv = (int64_t)gm.batch * (gm.L / p->k_kv) * gm.heads_kv * gm.head_dim * 2;
            *value = (int64_t)gm.a * (2ll * p->k_q * (gm.a - 1) * unit_q + 2ll * p->k_kv * (gm.b - 1) * unit_kv);
            break;
        }
        case MESH_ATTN_Q_BWD_PAIRED: *value = p->bwd_pair_mode(); break;
        case MESH_ATTN_Q_FWD_PAIRED: *value = p->fwd_pair() ? 1 : 0; break;
        case MESH_ATTN_Q_USP_A2A_BYTES_FWD: {
            // the GPU holds N/(n U) tokens of all heads before the all-to-all and keeps 1/U of them
            const long double tokens = (long double)gm.batch * gm.n * gm.L / ((long double)gm.n * U);
            *value = (int64_t)(tokens * (U - 1) / U * (2.0L * Hq + 2.0L * Hkv) * gm.head_dim * 2.0L);
            break;
        }
        default: return fail(MESH_ATTN_EINVAL, "plan_query: unknown query");
    }
    return MESH_ATTN_OK;
}
