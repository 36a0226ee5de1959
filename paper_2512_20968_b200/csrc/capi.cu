// capi.cu -- C-ABI entry points of libmesh_attn.so (include/mesh_attn.h): argument checking,
// TMA tensor-map construction, kernel launches.  No allocation and no host synchronisation in
// the hot calls; every launch goes to the caller's stream.
#include <algorithm>
#include <atomic>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

#include "plan.hpp"
#include "tile_kernels.hpp"
#include "tmap.hpp"

using namespace mesh_attn;

namespace {
thread_local std::string g_last_error;
std::atomic<long long> g_launches{0};

int fail(int code, const std::string& msg)
{
    g_last_error = msg;
    return code;
}
int cuda_fail(const char* what, int err)
{
    g_last_error = std::string(what) + ": " + cudaGetErrorString((cudaError_t)err);
    return MESH_ATTN_ECUDA;
}

struct Strides { long long b, row, h; };   // element strides of a [B,N,H,D] / [B,H,N,D] tensor with H heads in all
Strides strides_of(const mesh_attn_plan* p, int H, long long rows = 0)
{
    const long long N = rows ? rows : (long long)p->geom.n * p->geom.L, D = p->geom.head_dim;
    if (p->desc.tensor_layout == 0) return {N * H * D, (long long)H * D, D};
    return {N * H * D, D, N * D};
}

// Mesh-USP lane of a range of simulated GPUs / of a Q group: head slice [hq0, hq0 + geom.heads_q)
// of the query-shaped tensors and [hk0, hk0 + geom.heads_kv) of the key-shaped ones; geom holds the LANE's head counts.
struct Lane { int lane; long long hq0, hk0; };
int lanes_of(const mesh_attn_plan* p) { return p->desc.usp_lanes > 1 ? p->desc.usp_lanes : 1; }
Lane lane_at(const mesh_attn_plan* p, int lane) { return {lane, (long long)lane * p->geom.heads_q, (long long)lane * p->geom.heads_kv}; }
bool lane_of_range(const mesh_attn_plan* p, int g_first, int g_count, Lane* out)
{
    const int n = p->geom.n;
    if (g_first < 0 || g_count <= 0 || (long long)g_first + g_count > (long long)n * lanes_of(p)) return false;
    if ((g_first + g_count - 1) / n != g_first / n) return false;
    *out = lane_at(p, g_first / n);
    return true;
}
template <class T> T* head_slice(T* base, long long h0, const Strides& s, int elem_bytes)
{
    return (T*)((char*)base + h0 * s.h * elem_bytes);
}

// plan out_dtype: bytes per element of O (and of dQ, dK, dV in the composite calls)
int out_bytes(const mesh_attn_plan* p) { return p->desc.out_dtype == 1 ? 2 : 4; }
// fp32 accumulators of dQ, dK, dV behind the two planes of bwd_ws (out_dtype = 1 only)
struct GradAcc { float *dQ, *dK, *dV; size_t nq, nk; };
GradAcc grad_acc(const mesh_attn_plan* p, float* bwd_ws)
{
    const size_t N = (size_t)p->geom.n * p->geom.L, B = p->geom.batch, D = p->geom.head_dim;
    GradAcc a;
    a.nq = B * N * p->desc.heads_q * D;
    a.nk = B * N * p->desc.heads_kv * D;
    a.dQ = bwd_ws + 2 * B * p->desc.heads_q * N;
    a.dK = a.dQ + a.nq;
    a.dV = a.dK + a.nk;
    return a;
}

// bf16 tensor map of the lane's head slice: H_lane heads starting at h0 of a tensor with H_all heads
bool make_map(const mesh_attn_plan* p, CUtensorMap* m, const void* base, int H_lane, int H_all, long long h0, int box_rows = kBlock,
              long long rows = 0)
{
    const Strides s = strides_of(p, H_all, rows);
    const uint64_t N = rows ? (uint64_t)rows : (uint64_t)p->geom.n * p->geom.L;
    return make_tmap_bf16_4d(m, head_slice(base, h0, s, 2), p->geom.head_dim, H_lane, N, p->geom.batch, s.h * 2, s.row * 2, s.b * 2, box_rows);
}

// ---- per-kernel device timing (mesh_attn_profile_*): event pairs around each launch ----
struct Profiler {
    bool on = false;
    std::vector<cudaEvent_t> ev;     // 2 per recorded launch
    std::vector<int> kind;
    size_t used = 0, capacity = 0;
} g_prof;

struct ProfScope {                   // records begin at construction, end at destruction, on the launch stream
    cudaStream_t st;
    long long slot = -1;
    ProfScope(int kind, cudaStream_t s) : st(s)
    {
        if (!g_prof.on || g_prof.used >= g_prof.capacity) return;
        slot = (long long)g_prof.used++;
        g_prof.kind[slot] = kind;
        cudaEventRecord(g_prof.ev[2 * slot], st);
    }
    ~ProfScope()
    {
        if (slot >= 0) cudaEventRecord(g_prof.ev[2 * slot + 1], st);
    }
};

// a kernel of this plan reported a fault through its status words (sm100.cuh watchdog): every later call fails loudly
int check_health(const mesh_attn_plan* p, const char* who)
{
    if (!p->h_status) return MESH_ATTN_OK;
    const volatile int* st = p->h_status;
    if (st[0] == 0) return MESH_ATTN_OK;
    char buf[256];
    if (st[0] == 1)
        std::snprintf(buf, sizeof buf, ": an earlier kernel of this plan timed out in an mbarrier wait (block %d, thread %d, barrier 0x%x, parity %d); "
                      "its results are invalid; destroy the plan", st[1], st[2], (unsigned)st[3], st[4]);
    else
        std::snprintf(buf, sizeof buf, ": an earlier kernel of this plan found its dynamic shared memory misaligned (block %d) and did not run", st[1]);
    return fail(MESH_ATTN_ECUDA, std::string(who) + buf);
}

int check_device(const mesh_attn_plan* p, const char* who)
{
    if (!p) return fail(MESH_ATTN_EINVAL, std::string(who) + ": null plan");
    if (!p->d_blob) return fail(MESH_ATTN_ECUDA, std::string(who) + ": plan has no device work lists (no sm_100 CUDA device at plan_create); there is no CPU fallback");
    return check_health(p, who);
}
}  // namespace

namespace mesh_attn {
void set_error(const std::string& msg) { g_last_error = msg; }

int upload_plan(mesh_attn_plan* p)
{
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        (void)cudaGetLastError();
        return MESH_ATTN_OK;   // host-only plan: planner queries work, compute calls return ECUDA
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return cuda_fail("cudaGetDevice", (int)cudaGetLastError());
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return cuda_fail("cudaGetDeviceProperties", (int)cudaGetLastError());
    if (prop.major != 10) return MESH_ATTN_OK;   // not a B200: like no device at all -- a host-only plan whose compute calls return ECUDA
    p->device = dev;
    p->num_sms = prop.multiProcessorCount;
    auto al = [](size_t x) { return (x + 255) & ~size_t(255); };
    const size_t b0 = al(p->fwd_items.size() * sizeof(FwdItem)), b1 = al(p->bwd_items.size() * sizeof(BwdItem)),
                 b2 = al(p->fwd_segs.size() * sizeof(Seg)), b3 = al(p->bwd_segs.size() * sizeof(Seg)),
                 b4 = al(p->fwd_seglists.size() * sizeof(SegList)), b5 = al(p->bwd_seglists.size() * sizeof(SegList)),
                 b6 = al(p->goo_items.size() * sizeof(FwdItem)), b7 = al(p->goo_bwd_items.size() * sizeof(BwdItem));
    char* d = nullptr;
    cudaError_t e = cudaMalloc(&d, b0 + b1 + b2 + b3 + b4 + b5 + b6 + b7 + 256);
    if (e != cudaSuccess) return cuda_fail("cudaMalloc(work lists)", (int)e);
    p->d_blob = d;
    auto put = [&](const void* src, size_t bytes, size_t cap) {
        char* at = d;
        if (bytes && e == cudaSuccess) e = cudaMemcpy(at, src, bytes, cudaMemcpyHostToDevice);   // the first error is the one reported
        d += cap;
        return at;
    };
    p->d_fwd_items = (const FwdItem*)put(p->fwd_items.data(), p->fwd_items.size() * sizeof(FwdItem), b0);
    p->d_bwd_items = (const BwdItem*)put(p->bwd_items.data(), p->bwd_items.size() * sizeof(BwdItem), b1);
    p->d_fwd_segs = (const Seg*)put(p->fwd_segs.data(), p->fwd_segs.size() * sizeof(Seg), b2);
    p->d_bwd_segs = (const Seg*)put(p->bwd_segs.data(), p->bwd_segs.size() * sizeof(Seg), b3);
    p->d_fwd_seglists = (const SegList*)put(p->fwd_seglists.data(), p->fwd_seglists.size() * sizeof(SegList), b4);
    p->d_bwd_seglists = (const SegList*)put(p->bwd_seglists.data(), p->bwd_seglists.size() * sizeof(SegList), b5);
    p->d_goo_items = (const FwdItem*)put(p->goo_items.data(), p->goo_items.size() * sizeof(FwdItem), b6);
    p->d_goo_bwd_items = (const BwdItem*)put(p->goo_bwd_items.data(), p->goo_bwd_items.size() * sizeof(BwdItem), b7);
    p->d_counter = (int*)d;                                 // the trailing 256 bytes of the blob
    if (e != cudaSuccess) { cudaFree(p->d_blob); p->d_blob = nullptr; return cuda_fail("cudaMemcpy(work lists)", (int)e); }
    // watchdog status words: pinned host memory the kernels write through its device mapping (no host sync needed to read it)
    e = cudaHostAlloc((void**)&p->h_status, 8 * sizeof(int), cudaHostAllocMapped);
    if (e == cudaSuccess) {
        std::memset(p->h_status, 0, 8 * sizeof(int));
        e = cudaHostGetDevicePointer((void**)&p->d_status, p->h_status, 0);
    }
    if (e != cudaSuccess) { free_plan_device(p); return cuda_fail("plan_create: status words", (int)e); }
    // step_host's copy engines: one stream per direction, events for the chunk hand-offs (2b + 8, then a per copy direction for
    // the KV columns: the list in mesh_attn_step_host)
    cudaStream_t s0 = nullptr, s1 = nullptr;
    e = cudaStreamCreateWithFlags(&s0, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&s1, cudaStreamNonBlocking);
    p->s_h2d = s0; p->s_d2h = s1;
    for (int i = 0; e == cudaSuccess && i < 2 * p->geom.b + 8 + 2 * p->geom.a; ++i) {
        cudaEvent_t ev = nullptr;
        e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
        if (e == cudaSuccess) p->copy_events.push_back(ev);
    }
    if (e != cudaSuccess) { free_plan_device(p); return cuda_fail("plan_create: copy streams / events", (int)e); }
    return MESH_ATTN_OK;
}

void free_plan_device(mesh_attn_plan* p)
{
    if (p->d_blob) cudaFree(p->d_blob);
    p->d_blob = nullptr;
    if (p->h_status) cudaFreeHost(p->h_status);
    p->h_status = p->d_status = nullptr;
    for (void* ev : p->copy_events) cudaEventDestroy((cudaEvent_t)ev);
    p->copy_events.clear();
    if (p->s_h2d) cudaStreamDestroy((cudaStream_t)p->s_h2d);
    if (p->s_d2h) cudaStreamDestroy((cudaStream_t)p->s_d2h);
    p->s_h2d = p->s_d2h = nullptr;
}
}  // namespace mesh_attn

extern "C" {

// tile_fwd over an item list (the plan's fused list, or one compute task of the GOO executor)
static int launch_fwd_list(const mesh_attn_plan* p, const FwdItem* items, int items_per_gpu, int slots_per_gpu, int32_t g_first, int32_t g_count,
                           const void* Q, const void* K, const void* V, float* partial_O, float* partial_lse, void* stream, const char* who,
                           bool local = false, bool pair = false)
{
    const long long rq = local ? (long long)p->geom.a * p->geom.L : 0, rk = local ? (long long)p->geom.b * p->geom.L : 0;
    if (int rc = check_device(p, who)) return rc;
    if (!Q || !K || !V || !partial_O || !partial_lse) return fail(MESH_ATTN_EINVAL, std::string(who) + ": null pointer");
    Lane ln;
    if (!lane_of_range(p, g_first, g_count, &ln)) return fail(MESH_ATTN_EINVAL, std::string(who) + ": simulated GPU range out of bounds (or crossing a USP lane)");
    if ((long long)g_count * (long long)items_per_gpu >= (1ll << 31)) return fail(MESH_ATTN_EINVAL, std::string(who) + ": too many work items in one call");
    if (items_per_gpu == 0) return MESH_ATTN_OK;
    CUtensorMap tmQ, tmK, tmV;
    if (!make_map(p, &tmQ, Q, p->geom.heads_q, p->desc.heads_q, ln.hq0, kBlock, rq) ||
        !make_map(p, &tmK, K, p->geom.heads_kv, p->desc.heads_kv, ln.hk0, pair ? kBlock / 2 : kBlock, rk) ||   // pair: each CTA loads 64 key rows
        !make_map(p, &tmV, V, p->geom.heads_kv, p->desc.heads_kv, ln.hk0, kBlock, rk))
        return fail(MESH_ATTN_ECUDA, std::string(who) + ": cuTensorMapEncodeTiled failed (pointers must be 16-byte aligned device memory)");
    FwdParams fp;
    fp.gm = p->geom;
    fp.gm.slots_per_gpu = slots_per_gpu;
    if (local) { fp.gm.local = 1; fp.gm.rows_q = (int32_t)rq; fp.gm.rows_kv = (int32_t)rk; }
    fp.items = items;
    fp.segs = p->d_fwd_segs;
    fp.seglists = p->d_fwd_seglists;
    fp.items_per_gpu = items_per_gpu;
    fp.g_first = g_first % p->geom.n;
    fp.g_count = g_count;
    fp.split = p->desc.precision;
    fp.pair = pair ? 1 : 0;
    fp.partial_O = partial_O;
    fp.partial_lse = partial_lse;
    fp.status = p->d_status;
    fp.counter = p->d_counter + 1;                          // tile_fwd's own counter (a forward and a backward may be in flight on one stream)
    {
        const cudaError_t e0 = cudaMemsetAsync(fp.counter, 0, sizeof(int), (cudaStream_t)stream);
        if (e0 != cudaSuccess) return cuda_fail("tile_fwd: work-item counter", (int)e0);
    }
    ProfScope prof(MESH_ATTN_K_TILE_FWD, (cudaStream_t)stream);
    const int e = launch_tile_fwd(fp, tmQ, tmK, tmV, p->num_sms, (cudaStream_t)stream);
    if (e) return cuda_fail(who, e);
    g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

static int launch_merge_slots(const mesh_attn_plan* p, int32_t q_group, int per, int slots_per_gpu, const float* partial_O, const float* partial_lse,
                              void* O, float* lse, void* stream)
{
    if (int rc = check_device(p, "merge")) return rc;
    if (!partial_O || !partial_lse || !O || !lse) return fail(MESH_ATTN_EINVAL, "merge: null pointer");
    if (q_group < 0 || q_group >= p->geom.b * lanes_of(p))
        return fail(MESH_ATTN_EINVAL, "merge: q_group out of range (there are b Q groups per lane, PAPER.md L178)");
    const Lane ln = lane_at(p, q_group / p->geom.b);
    const long long N = (long long)p->geom.n * p->geom.L;
    MergeParams mp;
    mp.gm = p->geom;
    mp.gm.slots_per_gpu = slots_per_gpu;
    mp.q_group = q_group % p->geom.b;
    mp.per = per;
    mp.peers = 0;
    mp.m = p->geom.a * mp.per;
    // rows per block: 2 measured best on every BASELINE.json geometry (isolated launches, 1 / 2 / 4 / 8 rows: C2 4.7 / 5.1 / 5.1 /
    // 4.6, C4 6.25 / 6.48 / 6.25 / 6.13, C5 6.22 / 6.65 / 6.61 / 6.44 TB/s; profiles/r01_v7_README.md): small blocks keep the
    // weight phase short and many blocks streaming
    int rows = 2;
    while (rows > 1 && ((size_t)rows * p->geom.heads_q * mp.m * 4 > 64 * 1024 || p->geom.L % rows)) rows >>= 1;
    if ((size_t)rows * p->geom.heads_q * mp.m * 4 > 200 * 1024) return fail(MESH_ATTN_EUNSUPPORTED, "merge: heads_q * partial count too large");
    mp.rows_per_block = rows;
    mp.partial_O = partial_O;
    mp.partial_lse = partial_lse;
    const Strides s = strides_of(p, p->desc.heads_q);
    mp.O = head_slice((char*)O, ln.hq0, s, out_bytes(p));
    mp.out_bf16 = p->desc.out_dtype == 1;
    mp.lse = lse + ln.hq0 * N;
    mp.lse_stride_b = (long long)p->desc.heads_q * N;
    mp.o_stride_b = s.b; mp.o_stride_row = s.row; mp.o_stride_h = s.h;
    ProfScope prof(MESH_ATTN_K_MERGE, (cudaStream_t)stream);
    const int e = launch_merge(mp, (cudaStream_t)stream);
    if (e) return cuda_fail("merge launch", e);
    g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

int mesh_attn_tile_fwd(const mesh_attn_plan* p, int32_t g_first, int32_t g_count, const void* Q, const void* K, const void* V,
                       float* partial_O, float* partial_lse, void* stream)
{
    if (int rc = check_device(p, "tile_fwd")) return rc;
    return launch_fwd_list(p, p->d_fwd_items, (int)p->fwd_items.size(), p->geom.slots_per_gpu, g_first, g_count, Q, K, V, partial_O, partial_lse, stream,
                           "tile_fwd", false, p->fwd_pair());
}

int mesh_attn_merge(const mesh_attn_plan* p, int32_t q_group, const float* partial_O, const float* partial_lse, void* O, float* lse,
                    void* stream)
{
    if (int rc = check_device(p, "merge")) return rc;
    return launch_merge_slots(p, q_group, p->desc.partial_mode == 1 ? p->geom.b : 1, p->geom.slots_per_gpu, partial_O, partial_lse, O, lse, stream);
}

int mesh_attn_bwd_preprocess(const mesh_attn_plan* p, const void* O, const void* dO, const float* lse, float* bwd_ws, void* stream)
{
    if (int rc = check_device(p, "bwd_preprocess")) return rc;
    if (!O || !dO || !lse || !bwd_ws) return fail(MESH_ATTN_EINVAL, "bwd_preprocess: null pointer");
    DeltaParams dp;
    dp.gm = p->geom;
    dp.gm.heads_q = p->desc.heads_q;      // all lanes in one launch
    dp.gm.heads_kv = p->desc.heads_kv;
    dp.O = O; dp.dO = dO; dp.lse = lse; dp.ws = bwd_ws;
    dp.o_bf16 = p->desc.out_dtype == 1;
    const Strides s = strides_of(p, p->desc.heads_q);
    dp.stride_b = s.b; dp.stride_row = s.row; dp.stride_h = s.h;
    ProfScope prof(MESH_ATTN_K_BWD_PREPROCESS, (cudaStream_t)stream);
    const int e = launch_delta(dp, (cudaStream_t)stream);
    if (e) return cuda_fail("bwd_preprocess launch", e);
    g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

static int launch_bwd(const mesh_attn_plan* p, int32_t g_first, int32_t g_count, const void* Q, const void* K, const void* V,
                      const void* dO, const float* bwd_ws, float* dQ, float* dK, float* dV, void* stream, bool local,
                      const BwdItem* items = nullptr, int items_per_gpu = -1)
{
    const bool own_list = items != nullptr;                 // a compute task of the GOO executor: single-CTA kernel
    if (!own_list) { items = p->d_bwd_items; items_per_gpu = (int)p->bwd_items.size(); }
    if (items_per_gpu == 0) return MESH_ATTN_OK;
    if (int rc = check_device(p, "tile_bwd")) return rc;
    if (!Q || !K || !V || !dO || !bwd_ws || !dQ || !dK || !dV) return fail(MESH_ATTN_EINVAL, "tile_bwd: null pointer");
    Lane ln;
    if (!lane_of_range(p, g_first, g_count, &ln)) return fail(MESH_ATTN_EINVAL, "tile_bwd: simulated GPU range out of bounds (or crossing a USP lane)");
    if ((long long)g_count * (long long)items_per_gpu >= (1ll << 31)) return fail(MESH_ATTN_EINVAL, "tile_bwd: too many work items in one call");
    CUtensorMap tmQ, tmK, tmV, tmdO, tmdQ;
    const long long N = local ? (long long)p->geom.a * p->geom.L : (long long)p->geom.n * p->geom.L;     // query-shaped rows
    const long long Nk = local ? (long long)p->geom.b * p->geom.L : (long long)p->geom.n * p->geom.L;   // key-shaped rows
    const Strides sdq = strides_of(p, p->desc.heads_q, N), sdk = strides_of(p, p->desc.heads_kv, Nk);
    dQ = head_slice(dQ, ln.hq0, sdq, 4);
    dK = head_slice(dK, ln.hk0, sdk, 4);
    dV = head_slice(dV, ln.hk0, sdk, 4);
    // paired items (2-CTA clusters): each CTA loads 64-row halves of the Q / dO tiles and multicasts them
    const int pair = (!own_list && ((long long)g_count * (long long)items_per_gpu) >= 2) ? p->bwd_pair_mode() : 0;
    const int qbox = pair ? kBlock / 2 : kBlock;
    if (!make_map(p, &tmQ, Q, p->geom.heads_q, p->desc.heads_q, ln.hq0, qbox, N) ||
        !make_map(p, &tmK, K, p->geom.heads_kv, p->desc.heads_kv, ln.hk0, kBlock, Nk) ||
        !make_map(p, &tmV, V, p->geom.heads_kv, p->desc.heads_kv, ln.hk0, kBlock, Nk) ||
        !make_map(p, &tmdO, dO, p->geom.heads_q, p->desc.heads_q, ln.hq0, qbox, N) ||
        !make_tmap_f32_4d(&tmdQ, dQ, p->geom.head_dim, p->geom.heads_q, (uint64_t)N, p->geom.batch, sdq.h * 4, sdq.row * 4, sdq.b * 4, pair == 2 ? kBwdStgRowsExch : kBwdStgRows))
        return fail(MESH_ATTN_ECUDA, "tile_bwd: cuTensorMapEncodeTiled failed (pointers must be 16-byte aligned device memory)");
    BwdParams bp;
    bp.gm = p->geom;
    if (local) { bp.gm.local = 1; bp.gm.rows_q = (int32_t)N; bp.gm.rows_kv = (int32_t)Nk; }
    bp.items = items;
    bp.segs = p->d_bwd_segs;
    bp.seglists = p->d_bwd_seglists;
    bp.items_per_gpu = items_per_gpu;
    bp.g_first = g_first % p->geom.n;
    bp.g_count = g_count;
    bp.split = p->desc.precision;
    bp.pair = pair;
    bp.status = p->d_status;
    bp.counter = p->d_counter;
    {   // the kernel's scheduler warps take work items from this counter
        const cudaError_t e0 = cudaMemsetAsync(p->d_counter, 0, sizeof(int), (cudaStream_t)stream);
        if (e0 != cudaSuccess) return cuda_fail("tile_bwd: work-item counter", (int)e0);
    }
    bp.ws = bwd_ws + ln.hq0 * N;
    bp.ws_plane = (long long)p->geom.batch * p->desc.heads_q * N;
    bp.vec_stride_b = (long long)p->desc.heads_q * N;
    bp.dQ = dQ; bp.dK = dK; bp.dV = dV;
    const Strides sq = sdq, sk = sdk;
    bp.q_stride_b = sq.b; bp.q_stride_row = sq.row; bp.q_stride_h = sq.h;
    bp.k_stride_b = sk.b; bp.k_stride_row = sk.row; bp.k_stride_h = sk.h;
    ProfScope prof(MESH_ATTN_K_TILE_BWD, (cudaStream_t)stream);
    const int e = launch_tile_bwd(bp, tmQ, tmK, tmV, tmdO, tmdQ, p->num_sms, (cudaStream_t)stream);
    if (e) return cuda_fail("tile_bwd launch", e);
    g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

int mesh_attn_tile_bwd(const mesh_attn_plan* p, int32_t g_first, int32_t g_count, const void* Q, const void* K, const void* V,
                       const void* dO, const float* bwd_ws, float* dQ, float* dK, float* dV, void* stream)
{
    return launch_bwd(p, g_first, g_count, Q, K, V, dO, bwd_ws, dQ, dK, dV, stream, false);
}

// ---- per-rank calls: the tensors hold only the partitions ONE GPU has after its all-gathers ----
static int check_rank(const mesh_attn_plan* p, int32_t g, const char* who)
{
    if (int rc = check_device(p, who)) return rc;
    if (lanes_of(p) != 1 || p->desc.partial_mode != 0 || p->desc.out_dtype != 0)
        return fail(MESH_ATTN_EUNSUPPORTED, std::string(who) + ": per-rank calls need usp_lanes == 1, partial_mode == 0 and out_dtype == 0");
    if (g < 0 || g >= p->geom.n) return fail(MESH_ATTN_EINVAL, std::string(who) + ": rank g out of range");
    return MESH_ATTN_OK;
}

int mesh_attn_rank_fwd(const mesh_attn_plan* p, int32_t g, const void* Q_loc, const void* K_loc, const void* V_loc, float* partial_O,
                       float* partial_lse, void* stream)
{
    if (int rc = check_rank(p, g, "rank_fwd")) return rc;
    return launch_fwd_list(p, p->d_fwd_items, (int)p->fwd_items.size(), p->geom.slots_per_gpu, g, 1, Q_loc, K_loc, V_loc, partial_O, partial_lse, stream,
                           "rank_fwd", true);
}

static int launch_rank_merge(const mesh_attn_plan* p, const float* partial_O_recv, const float* partial_lse_recv, const float* const* peer_O,
                             const float* const* peer_lse, float* O_own, float* lse_own, void* stream, const char* who)
{
    if (int rc = check_rank(p, 0, who)) return rc;
    if (!O_own || !lse_own) return fail(MESH_ATTN_EINVAL, std::string(who) + ": null pointer");
    const Geom& g0 = p->geom;
    MergeParams mp;
    mp.gm = g0;
    mp.gm.a = 1;                      // one Q partition (the rank's own) ...
    mp.gm.rows_q = g0.L;              // ... in tensors of L rows
    mp.gm.slots_per_gpu = g0.a;
    mp.q_group = 0;
    mp.per = g0.a;                    // slot(k) = k: the partial received from the k-th member of the Q group
    mp.m = g0.a;
    mp.peers = peer_O ? 1 : 0;
    if (peer_O) {
        if (g0.a > kMaxPeers) return fail(MESH_ATTN_EUNSUPPORTED, std::string(who) + ": Q groups of more than 16 GPUs are not supported");
        for (int k = 0; k < g0.a; ++k) {
            if (!peer_O[k] || !peer_lse[k]) return fail(MESH_ATTN_EINVAL, std::string(who) + ": null peer pointer");
            if (((uintptr_t)peer_O[k] & 15) != 0) return fail(MESH_ATTN_EINVAL, std::string(who) + ": peer partials must be 16-byte aligned");
            mp.peer_O[k] = peer_O[k];
            mp.peer_lse[k] = peer_lse[k];
        }
    }
    int rows = 2;                     // as in launch_merge_slots
    while (rows > 1 && ((size_t)rows * g0.heads_q * mp.m * 4 > 64 * 1024 || g0.L % rows)) rows >>= 1;
    if ((size_t)rows * g0.heads_q * mp.m * 4 > 200 * 1024) return fail(MESH_ATTN_EUNSUPPORTED, std::string(who) + ": heads_q * partial count too large");
    mp.rows_per_block = rows;
    mp.partial_O = partial_O_recv;
    mp.partial_lse = partial_lse_recv;
    const Strides s = strides_of(p, g0.heads_q, g0.L);
    mp.O = O_own;
    mp.out_bf16 = 0;
    mp.lse = lse_own;
    mp.lse_stride_b = (long long)g0.heads_q * g0.L;
    mp.o_stride_b = s.b; mp.o_stride_row = s.row; mp.o_stride_h = s.h;
    ProfScope prof(MESH_ATTN_K_MERGE, (cudaStream_t)stream);
    const int e = launch_merge(mp, (cudaStream_t)stream);
    if (e) return cuda_fail(who, e);
    g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

int mesh_attn_rank_merge(const mesh_attn_plan* p, const float* partial_O_recv, const float* partial_lse_recv, float* O_own, float* lse_own,
                         void* stream)
{
    if (!partial_O_recv || !partial_lse_recv) return fail(MESH_ATTN_EINVAL, "rank_merge: null pointer");
    return launch_rank_merge(p, partial_O_recv, partial_lse_recv, nullptr, nullptr, O_own, lse_own, stream, "rank_merge");
}

int mesh_attn_rank_merge_peers(const mesh_attn_plan* p, const float* const* peer_partial_O, const float* const* peer_partial_lse, float* O_own,
                               float* lse_own, void* stream)
{
    if (!peer_partial_O || !peer_partial_lse) return fail(MESH_ATTN_EINVAL, "rank_merge_peers: null pointer table");
    return launch_rank_merge(p, nullptr, nullptr, peer_partial_O, peer_partial_lse, O_own, lse_own, stream, "rank_merge_peers");
}

int mesh_attn_rank_sum_peers(const mesh_attn_plan* p, const float* const* peers, int32_t m, int64_t count, float* out, void* stream)
{
    if (int rc = check_device(p, "rank_sum_peers")) return rc;
    if (!peers || !out) return fail(MESH_ATTN_EINVAL, "rank_sum_peers: null pointer");
    if (m < 1 || m > kMaxPeers) return fail(MESH_ATTN_EUNSUPPORTED, "rank_sum_peers: 1 <= m <= 16 buffers");
    if (count < 0 || (count & 3) || ((uintptr_t)out & 15)) return fail(MESH_ATTN_EINVAL, "rank_sum_peers: count must be a multiple of 4 floats, buffers 16-byte aligned");
    SumParams sp;
    sp.m = m;
    sp.count4 = count / 4;
    sp.out = out;
    for (int k = 0; k < m; ++k) {
        if (!peers[k] || ((uintptr_t)peers[k] & 15)) return fail(MESH_ATTN_EINVAL, "rank_sum_peers: null or misaligned peer pointer");
        sp.src[k] = peers[k];
    }
    const int e = launch_sum_peers(sp, p->num_sms, (cudaStream_t)stream);
    if (e) return cuda_fail("rank_sum_peers launch", e);
    if (count) g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

int mesh_attn_rank_bwd_preprocess(const mesh_attn_plan* p, const float* O_own, const void* dO_own, const float* lse_own, float* ws_own, void* stream)
{
    if (int rc = check_rank(p, 0, "rank_bwd_preprocess")) return rc;
    if (!O_own || !dO_own || !lse_own || !ws_own) return fail(MESH_ATTN_EINVAL, "rank_bwd_preprocess: null pointer");
    DeltaParams dp;
    dp.gm = p->geom;
    dp.gm.rows_q = p->geom.L;
    dp.O = O_own; dp.dO = dO_own; dp.lse = lse_own; dp.ws = ws_own;
    dp.o_bf16 = 0;
    const Strides s = strides_of(p, p->geom.heads_q, p->geom.L);
    dp.stride_b = s.b; dp.stride_row = s.row; dp.stride_h = s.h;
    ProfScope prof(MESH_ATTN_K_BWD_PREPROCESS, (cudaStream_t)stream);
    const int e = launch_delta(dp, (cudaStream_t)stream);
    if (e) return cuda_fail("rank_bwd_preprocess launch", e);
    g_launches.fetch_add(1);
    return MESH_ATTN_OK;
}

int mesh_attn_rank_bwd(const mesh_attn_plan* p, int32_t g, const void* Q_loc, const void* K_loc, const void* V_loc, const void* dO_loc,
                       const float* ws_loc, float* dQ_loc, float* dK_loc, float* dV_loc, void* stream)
{
    if (int rc = check_rank(p, g, "rank_bwd")) return rc;
    return launch_bwd(p, g, 1, Q_loc, K_loc, V_loc, dO_loc, ws_loc, dQ_loc, dK_loc, dV_loc, stream, true);
}

int mesh_attn_forward(const mesh_attn_plan* p, const void* Q, const void* K, const void* V, void* O, float* lse, float* partial_O,
                      float* partial_lse, void* stream)
{
    if (int rc = check_device(p, "forward")) return rc;
    for (int lane = 0; lane < lanes_of(p); ++lane)
        for (int r = 0; r < p->geom.b; ++r) {   // one wave per Q group of each USP lane (L372-389)
            if (int rc = mesh_attn_tile_fwd(p, lane * p->geom.n + r * p->geom.a, p->geom.a, Q, K, V, partial_O, partial_lse, stream)) return rc;
            if (int rc = mesh_attn_merge(p, lane * p->geom.b + r, partial_O, partial_lse, O, lse, stream)) return rc;
        }
    return MESH_ATTN_OK;
}

// bytes the collective task (kind) delivers to / takes from the `a` simulated GPUs of one Q group
static long long goo_task_bytes(const mesh_attn_plan* p, int kind)
{
    const Geom& gm = p->geom;
    const long long unit_q = (long long)gm.batch * (gm.L / p->k_q) * gm.heads_q * gm.head_dim * 2;      // one Q chunk (bf16; O counted alike, L35)
    const long long unit_kv = (long long)gm.batch * (gm.L / p->k_kv) * gm.heads_kv * gm.head_dim * 2;   // one K (or V) chunk
    switch (kind) {
        case MESH_ATTN_TASK_AG_Q: case MESH_ATTN_TASK_RS_Q: return (long long)gm.a * (gm.a - 1) * unit_q;
        case MESH_ATTN_TASK_AG_KV: return (long long)gm.a * (gm.b - 1) * 2 * unit_kv;
        default: return 0;
    }
}

int mesh_attn_forward_goo(const mesh_attn_plan* p, int32_t q_group, const void* Q, const void* K, const void* V, void* O, float* lse,
                          float* partial_O, float* partial_lse, void* comm_ws, int64_t comm_ws_bytes, int32_t comm_repeat, int32_t overlap,
                          void* stream)
{
    if (int rc = check_device(p, "forward_goo")) return rc;
    if (!Q || !K || !V || !O || !lse || !partial_O || !partial_lse) return fail(MESH_ATTN_EINVAL, "forward_goo: null pointer");
    if (comm_repeat < 0 || (comm_repeat > 0 && (!comm_ws || comm_ws_bytes < 4096))) return fail(MESH_ATTN_EINVAL, "forward_goo: comm_ws too small");
    const Geom& gm = p->geom;
    if (q_group < 0 || q_group >= gm.b * lanes_of(p)) return fail(MESH_ATTN_EINVAL, "forward_goo: q_group out of range");
    const int lane = q_group / gm.b, r = q_group % gm.b, g_first = lane * gm.n + r * gm.a, slots = gm.a * p->k_kv;
    cudaStream_t st = (cudaStream_t)stream, cs = overlap ? (cudaStream_t)p->s_h2d : st;
    cudaEvent_t ev_fork = (cudaEvent_t)p->copy_events[2 * gm.b + 6], ev_join = (cudaEvent_t)p->copy_events[2 * gm.b + 7];
    const long long q_bytes = (long long)gm.batch * gm.n * gm.L * p->desc.heads_q * gm.head_dim * 2;
    const long long kv_bytes = (long long)gm.batch * gm.n * gm.L * p->desc.heads_kv * gm.head_dim * 2;
    const long long part_bytes = (long long)gm.a * slots * gm.batch * gm.L * gm.heads_q * gm.head_dim * 4;
    // stand-in for a collective: device-to-device copies of its byte count out of the tensor it would move
    auto copy_bytes = [&](const void* src, long long src_bytes, long long bytes) -> cudaError_t {
        const long long chunk = std::min<long long>(std::min<long long>(src_bytes, comm_ws_bytes), bytes);
        for (int rep = 0; rep < comm_repeat; ++rep)
            for (long long done = 0; done < bytes; done += chunk) {
                const cudaError_t e = cudaMemcpyAsync(comm_ws, src, (size_t)std::min(chunk, bytes - done), cudaMemcpyDeviceToDevice, cs);
                if (e != cudaSuccess) return e;
            }
        return cudaSuccess;
    };
    const std::vector<int32_t>& rows = p->steps_fwd;
    const size_t nrows = rows.size() / 4;
    for (size_t at = 0; at < nrows;) {
        const int step = rows[4 * at];
        cudaError_t e = cudaSuccess;
        if (overlap) {
            e = cudaEventRecord(ev_fork, st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, ev_fork, 0);
        }
        // the step's communication task first (its own stream when overlapping), then its compute tasks
        for (size_t k = at; k < nrows && rows[4 * k] == step && e == cudaSuccess; ++k) {
            const int kind = rows[4 * k + 1];
            if (comm_repeat == 0 || kind == MESH_ATTN_TASK_C) continue;
            const long long bytes = goo_task_bytes(p, kind);
            if (kind == MESH_ATTN_TASK_AG_Q) e = copy_bytes(Q, q_bytes, bytes);
            else if (kind == MESH_ATTN_TASK_RS_Q) e = copy_bytes(partial_O, part_bytes, bytes);
            else if (kind == MESH_ATTN_TASK_AG_KV) {
                e = copy_bytes(K, kv_bytes, bytes / 2);
                if (e == cudaSuccess) e = copy_bytes(V, kv_bytes, bytes / 2);
            }
        }
        if (e != cudaSuccess) return cuda_fail("forward_goo: communication stand-in", (int)e);
        size_t k = at;
        for (; k < nrows && rows[4 * k] == step; ++k) {
            if (rows[4 * k + 1] != MESH_ATTN_TASK_C) continue;
            const SegList task = p->goo_task[(size_t)rows[4 * k + 2] * p->k_kv + rows[4 * k + 3]];
            if (int rc = launch_fwd_list(p, p->d_goo_items + task.offset, task.count, slots, g_first, gm.a, Q, K, V, partial_O, partial_lse, stream,
                                         "forward_goo"))
                return rc;
        }
        if (overlap) {                                       // a step ends when its communication and its computation are done
            e = cudaEventRecord(ev_join, cs);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_join, 0);
            if (e != cudaSuccess) return cuda_fail("forward_goo: step barrier", (int)e);
        }
        at = k;
    }
    return launch_merge_slots(p, q_group, p->k_kv, slots, partial_O, partial_lse, O, lse, stream);
}

int mesh_attn_backward_goo(const mesh_attn_plan* p, int32_t q_group, const void* Q, const void* K, const void* V, const void* dO,
                           const float* bwd_ws, float* dQ, float* dK, float* dV, void* comm_ws, int64_t comm_ws_bytes, int32_t comm_repeat,
                           int32_t overlap, void* stream)
{
    if (int rc = check_device(p, "backward_goo")) return rc;
    if (p->desc.out_dtype != 0) return fail(MESH_ATTN_EUNSUPPORTED, "backward_goo: accumulates into fp32 dQ, dK, dV (plan out_dtype must be 0)");
    if (!Q || !K || !V || !dO || !bwd_ws || !dQ || !dK || !dV) return fail(MESH_ATTN_EINVAL, "backward_goo: null pointer");
    if (comm_repeat < 0 || (comm_repeat > 0 && (!comm_ws || comm_ws_bytes < 4096))) return fail(MESH_ATTN_EINVAL, "backward_goo: comm_ws too small");
    const Geom& gm = p->geom;
    if (q_group < 0 || q_group >= gm.b * lanes_of(p)) return fail(MESH_ATTN_EINVAL, "backward_goo: q_group out of range");
    const int lane = q_group / gm.b, r = q_group % gm.b, g_first = lane * gm.n + r * gm.a;
    cudaStream_t st = (cudaStream_t)stream, cs = overlap ? (cudaStream_t)p->s_h2d : st;
    cudaEvent_t ev_fork = (cudaEvent_t)p->copy_events[2 * gm.b + 6], ev_join = (cudaEvent_t)p->copy_events[2 * gm.b + 7];
    const long long q_bytes = (long long)gm.batch * gm.n * gm.L * p->desc.heads_q * gm.head_dim * 2;
    const long long kv_bytes = (long long)gm.batch * gm.n * gm.L * p->desc.heads_kv * gm.head_dim * 2;
    auto copy_bytes = [&](const void* src, long long src_bytes, long long bytes) -> cudaError_t {
        const long long chunk = std::min<long long>(std::min<long long>(src_bytes, comm_ws_bytes), bytes);
        for (int rep = 0; rep < comm_repeat; ++rep)
            for (long long done = 0; done < bytes; done += chunk) {
                const cudaError_t e = cudaMemcpyAsync(comm_ws, src, (size_t)std::min(chunk, bytes - done), cudaMemcpyDeviceToDevice, cs);
                if (e != cudaSuccess) return e;
            }
        return cudaSuccess;
    };
    const std::vector<int32_t>& rows = p->steps_bwd;
    const size_t nrows = rows.size() / 4;
    for (size_t at = 0; at < nrows;) {
        const int step = rows[4 * at];
        cudaError_t e = cudaSuccess;
        if (overlap) {
            e = cudaEventRecord(ev_fork, st);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(cs, ev_fork, 0);
        }
        // bytes in units of the bf16 inputs, as the paper counts them: AG of Q, O, dO = 3 Q units per chunk,
        // RS-dQ one, AG-KV and RS-dKV a K and a V unit each
        for (size_t k = at; k < nrows && rows[4 * k] == step && e == cudaSuccess; ++k) {
            const int kind = rows[4 * k + 1];
            if (comm_repeat == 0 || kind == MESH_ATTN_TASK_C) continue;
            if (kind == MESH_ATTN_TASK_AG_Q) {
                const long long bytes = goo_task_bytes(p, MESH_ATTN_TASK_AG_Q);
                e = copy_bytes(Q, q_bytes, bytes);
                if (e == cudaSuccess) e = copy_bytes(dO, q_bytes, 2 * bytes);
            } else if (kind == MESH_ATTN_TASK_RS_Q) {
                e = copy_bytes(dQ, 2 * q_bytes, goo_task_bytes(p, MESH_ATTN_TASK_RS_Q));
            } else {                                          // AG-KV, RS-dKV
                const long long bytes = goo_task_bytes(p, MESH_ATTN_TASK_AG_KV);
                e = copy_bytes(kind == MESH_ATTN_TASK_AG_KV ? K : (const void*)dK, kv_bytes, bytes / 2);
                if (e == cudaSuccess) e = copy_bytes(kind == MESH_ATTN_TASK_AG_KV ? V : (const void*)dV, kv_bytes, bytes / 2);
            }
        }
        if (e != cudaSuccess) return cuda_fail("backward_goo: communication stand-in", (int)e);
        size_t k = at;
        for (; k < nrows && rows[4 * k] == step; ++k) {
            if (rows[4 * k + 1] != MESH_ATTN_TASK_C) continue;
            const SegList task = p->goo_bwd_task[(size_t)rows[4 * k + 2] * p->k_kv + rows[4 * k + 3]];
            if (int rc = launch_bwd(p, g_first, gm.a, Q, K, V, dO, bwd_ws, dQ, dK, dV, stream, false, p->d_goo_bwd_items + task.offset, task.count)) return rc;
        }
        if (overlap) {
            e = cudaEventRecord(ev_join, cs);
            if (e == cudaSuccess) e = cudaStreamWaitEvent(st, ev_join, 0);
            if (e != cudaSuccess) return cuda_fail("backward_goo: step barrier", (int)e);
        }
        at = k;
    }
    return MESH_ATTN_OK;
}

int mesh_attn_backward(const mesh_attn_plan* p, const void* Q, const void* K, const void* V, const void* O, const void* dO,
                       const float* lse, float* bwd_ws, void* dQ, void* dK, void* dV, void* stream)
{
    if (int rc = check_device(p, "backward")) return rc;
    if (!dQ || !dK || !dV || !bwd_ws) return fail(MESH_ATTN_EINVAL, "backward: null pointer");
    const Geom& gm = p->geom;
    cudaStream_t st = (cudaStream_t)stream;
    // out_dtype = 1: the atomics accumulate in fp32 behind the two planes of bwd_ws; dQ, dK, dV receive the rounded sums
    const bool bf16_out = p->desc.out_dtype == 1;
    const GradAcc acc = grad_acc(p, bwd_ws);
    float* aQ = bf16_out ? acc.dQ : (float*)dQ;
    float* aK = bf16_out ? acc.dK : (float*)dK;
    float* aV = bf16_out ? acc.dV : (float*)dV;
    cudaError_t e = cudaMemsetAsync(aQ, 0, acc.nq * 4, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(aK, 0, acc.nk * 4, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(aV, 0, acc.nk * 4, st);
    if (e != cudaSuccess) return cuda_fail("backward memset", (int)e);
    if (int rc = mesh_attn_bwd_preprocess(p, O, dO, lse, bwd_ws, stream)) return rc;
    // keep each launch's work-item count below 2^31: one call per Q group
    for (int lane = 0; lane < lanes_of(p); ++lane)
        for (int r = 0; r < gm.b; ++r)
            if (int rc = mesh_attn_tile_bwd(p, lane * gm.n + r * gm.a, gm.a, Q, K, V, dO, bwd_ws, aQ, aK, aV, stream)) return rc;
    if (bf16_out) {
        int err = launch_cast_bf16(aQ, dQ, (long long)acc.nq, p->num_sms, st);
        if (!err) err = launch_cast_bf16(aK, dK, (long long)acc.nk, p->num_sms, st);
        if (!err) err = launch_cast_bf16(aV, dV, (long long)acc.nk, p->num_sms, st);
        if (err) return cuda_fail("backward cast launch", err);
        g_launches.fetch_add(3);
    }
    return MESH_ATTN_OK;
}

int mesh_attn_step_host(const mesh_attn_plan* p, const mesh_attn_host_io* io, void* stream)
{
    if (int rc = check_device(p, "step_host")) return rc;
    if (!io || !io->Q_host || !io->K_host || !io->V_host || !io->d_Q || !io->d_K || !io->d_V || !io->d_O || !io->d_lse || !io->d_partial_O ||
        !io->d_partial_lse)
        return fail(MESH_ATTN_EINVAL, "step_host: null pointer");
    const bool bwd = io->dO_host != nullptr;
    if (bwd && (!io->d_dO || !io->d_bwd_ws || !io->d_dQ || !io->d_dK || !io->d_dV)) return fail(MESH_ATTN_EINVAL, "step_host: null backward buffer");
    const Geom& gm = p->geom;
    const int U = lanes_of(p), nb = gm.b;
    const size_t N = (size_t)gm.n * gm.L;
    const size_t nq = (size_t)gm.batch * N * p->desc.heads_q * gm.head_dim, nk = (size_t)gm.batch * N * p->desc.heads_kv * gm.head_dim;
    const size_t nl = (size_t)gm.batch * N * p->desc.heads_q;
    // out_dtype = 1: O, dQ, dK, dV (device and host) are bf16; the gradients accumulate in fp32 behind the planes of d_bwd_ws
    const bool bf16_out = p->desc.out_dtype == 1;
    const size_t ob = (size_t)out_bytes(p);
    const GradAcc acc = grad_acc(p, (float*)io->d_bwd_ws);
    float* aQ = bf16_out ? acc.dQ : (float*)io->d_dQ;
    float* aK = bf16_out ? acc.dK : (float*)io->d_dK;
    float* aV = bf16_out ? acc.dV : (float*)io->d_dV;
    cudaStream_t st = (cudaStream_t)stream, up = (cudaStream_t)p->s_h2d, down = (cudaStream_t)p->s_d2h;
    auto ev = [&](int i) { return (cudaEvent_t)p->copy_events[i]; };
    // events: 0 start, 1 K,V on the device, 2 dO on the device, 3 forward done, 4 backward done, 5 copies back done,
    //         6+r Q rows of Q group r on the device, 6+b+r dQ rows of Q group r final, 2b+8+c K,V partitions of KV column c on
    //         the device, 2b+8+a+c dK,dV partitions of KV column c final
    // Rows of one partition are one contiguous byte range when batch == 1 in the [B,N,H,D] layout: then Q goes up and dQ comes
    // down Q group by Q group, behind / ahead of the waves that need them, and K, V go up / dK, dV come down KV column by KV
    // column (the b partitions of I^KV of the simulated GPUs g with g mod a = c) around the FIRST forward wave
    // and the LAST backward group, which run one launch per simulated GPU; otherwise whole tensors move.
    const bool rows_contig = gm.batch == 1 && p->desc.tensor_layout == 0;
    const bool by_group = rows_contig && nb > 1;
    const bool by_col = rows_contig && gm.a > 1;
    const size_t q_chunk = nq / nb;                   // elements of one Q group's rows
    const size_t kv_part = nk / gm.n;                 // elements of one KV partition's rows
    const size_t po_gpu = (size_t)gm.slots_per_gpu * gm.batch * gm.L * gm.heads_q * gm.head_dim;     // partial_O floats of one simulated GPU
    const size_t pl_gpu = (size_t)gm.slots_per_gpu * gm.batch * gm.L * gm.heads_q;
    auto ev_col_up = [&](int c) { return ev(2 * nb + 8 + c); };
    auto ev_col_down = [&](int c) { return ev(2 * nb + 8 + gm.a + c); };
    cudaError_t e = cudaEventRecord(ev(0), st);
    auto ok = [&]() { return e == cudaSuccess; };
    if (ok()) e = cudaStreamWaitEvent(up, ev(0), 0);
    if (ok()) e = cudaStreamWaitEvent(down, ev(0), 0);
    // ---- host -> device, in the order the kernels need the data
    auto upload_q = [&](int r) {
        if (by_group) e = cudaMemcpyAsync((char*)io->d_Q + r * q_chunk * 2, (const char*)io->Q_host + r * q_chunk * 2, q_chunk * 2, cudaMemcpyHostToDevice, up);
        else if (r == 0) e = cudaMemcpyAsync(io->d_Q, io->Q_host, nq * 2, cudaMemcpyHostToDevice, up);
        if (ok()) e = cudaEventRecord(ev(6 + r), up);
    };
    if (by_col) {
        upload_q(0);                                   // the first wave starts behind 1 Q group + 1 KV column
        for (int c = 0; c < gm.a && ok(); ++c) {
            for (int t = 0; t < gm.b && ok(); ++t) {
                const size_t at = (size_t)kv_partition(gm, c, t) * kv_part * 2;
                e = cudaMemcpyAsync((char*)io->d_K + at, (const char*)io->K_host + at, kv_part * 2, cudaMemcpyHostToDevice, up);
                if (ok()) e = cudaMemcpyAsync((char*)io->d_V + at, (const char*)io->V_host + at, kv_part * 2, cudaMemcpyHostToDevice, up);
            }
            if (ok()) e = cudaEventRecord(ev_col_up(c), up);
        }
    } else {
        if (ok()) e = cudaMemcpyAsync(io->d_K, io->K_host, nk * 2, cudaMemcpyHostToDevice, up);
        if (ok()) e = cudaMemcpyAsync(io->d_V, io->V_host, nk * 2, cudaMemcpyHostToDevice, up);
    }
    if (ok()) e = cudaEventRecord(ev(1), up);
    for (int r = by_col ? 1 : 0; r < nb && ok(); ++r) upload_q(r);
    if (bwd) {
        if (ok()) e = cudaMemcpyAsync(io->d_dO, io->dO_host, nq * 2, cudaMemcpyHostToDevice, up);      // lands during the forward
        if (ok()) e = cudaEventRecord(ev(2), up);
    }
    if (!ok()) return cuda_fail("step_host H2D", (int)e);
    // ---- forward: wave r of every lane needs K, V and the Q rows of group r; the first wave takes its simulated GPUs one by one,
    // each behind the upload of its own KV column
    if (!by_col) e = cudaStreamWaitEvent(st, ev(1), 0);
    for (int lane = 0; lane < U; ++lane)
        for (int r = 0; r < nb; ++r) {
            if (lane == 0 && ok()) e = cudaStreamWaitEvent(st, ev(6 + r), 0);
            if (!ok()) return cuda_fail("step_host forward", (int)e);
            if (by_col && lane == 0 && r == 0) {
                for (int c = 0; c < gm.a; ++c) {
                    e = cudaStreamWaitEvent(st, ev_col_up(c), 0);
                    if (!ok()) return cuda_fail("step_host forward", (int)e);
                    if (int rc = mesh_attn_tile_fwd(p, c, 1, io->d_Q, io->d_K, io->d_V, (float*)io->d_partial_O + c * po_gpu, (float*)io->d_partial_lse + c * pl_gpu, stream)) return rc;
                }
            } else if (int rc = mesh_attn_tile_fwd(p, lane * gm.n + r * gm.a, gm.a, io->d_Q, io->d_K, io->d_V, (float*)io->d_partial_O, (float*)io->d_partial_lse, stream))
                return rc;
            if (int rc = mesh_attn_merge(p, lane * nb + r, (const float*)io->d_partial_O, (const float*)io->d_partial_lse, io->d_O, (float*)io->d_lse, stream)) return rc;
        }
    e = cudaEventRecord(ev(3), st);
    if (ok()) e = cudaStreamWaitEvent(down, ev(3), 0);
    if (ok() && io->O_host) e = cudaMemcpyAsync(io->O_host, io->d_O, nq * ob, cudaMemcpyDeviceToHost, down);   // during the backward
    if (ok() && io->lse_host) e = cudaMemcpyAsync(io->lse_host, io->d_lse, nl * 4, cudaMemcpyDeviceToHost, down);
    if (bwd) {
        // ---- backward: the simulated GPUs of Q group r hold exactly the Q partitions of group r, so dQ of those rows is
        // final once the last lane's call for r has run (Alg.3 l.6)
        if (ok()) e = cudaStreamWaitEvent(st, ev(2), 0);
        if (ok()) e = cudaMemsetAsync(aQ, 0, nq * 4, st);
        if (ok()) e = cudaMemsetAsync(aK, 0, nk * 4, st);
        if (ok()) e = cudaMemsetAsync(aV, 0, nk * 4, st);
        if (!ok()) return cuda_fail("step_host backward setup", (int)e);
        if (int rc = mesh_attn_bwd_preprocess(p, io->d_O, io->d_dO, (const float*)io->d_lse, (float*)io->d_bwd_ws, stream)) return rc;
        // the last group runs one launch per simulated GPU: dK, dV of KV column c are final once every simulated GPU of the column
        // has run (Alg.3 l.7), and come down behind that launch instead of behind the whole backward
        const bool cols_down = by_col && (io->dK_host || io->dV_host);
        for (int lane = 0; lane < U; ++lane)
            for (int r = 0; r < nb; ++r) {
                const int g_first = lane * gm.n + r * gm.a;
                if (cols_down && lane == U - 1 && r == nb - 1) {
                    for (int c = 0; c < gm.a; ++c) {
                        if (int rc = mesh_attn_tile_bwd(p, g_first + c, 1, io->d_Q, io->d_K, io->d_V, io->d_dO, (const float*)io->d_bwd_ws, aQ, aK, aV, stream)) return rc;
                        if (bf16_out) {
                            for (int t = 0; t < gm.b; ++t) {
                                const size_t at = (size_t)kv_partition(gm, c, t) * kv_part;
                                int err = launch_cast_bf16(aK + at, (char*)io->d_dK + at * 2, (long long)kv_part, p->num_sms, st);
                                if (!err) err = launch_cast_bf16(aV + at, (char*)io->d_dV + at * 2, (long long)kv_part, p->num_sms, st);
                                if (err) return cuda_fail("step_host cast launch", err);
                                g_launches.fetch_add(2);
                            }
                        }
                        e = cudaEventRecord(ev_col_down(c), st);
                        if (ok()) e = cudaStreamWaitEvent(down, ev_col_down(c), 0);
                        for (int t = 0; t < gm.b && ok(); ++t) {
                            const size_t at = (size_t)kv_partition(gm, c, t) * kv_part * ob;
                            if (io->dK_host) e = cudaMemcpyAsync((char*)io->dK_host + at, (const char*)io->d_dK + at, kv_part * ob, cudaMemcpyDeviceToHost, down);
                            if (ok() && io->dV_host) e = cudaMemcpyAsync((char*)io->dV_host + at, (const char*)io->d_dV + at, kv_part * ob, cudaMemcpyDeviceToHost, down);
                        }
                        if (!ok()) return cuda_fail("step_host dK, dV D2H", (int)e);
                    }
                } else if (int rc = mesh_attn_tile_bwd(p, g_first, gm.a, io->d_Q, io->d_K, io->d_V, io->d_dO, (const float*)io->d_bwd_ws, aQ, aK, aV, stream))
                    return rc;
                if (lane == U - 1 && by_group) {
                    if (bf16_out) {                  // the rows of Q group r are final: round them into the caller's dQ
                        if (int err = launch_cast_bf16(aQ + r * q_chunk, (char*)io->d_dQ + r * q_chunk * 2, (long long)q_chunk, p->num_sms, st))
                            return cuda_fail("step_host cast launch", err);
                        g_launches.fetch_add(1);
                    }
                    if (io->dQ_host) {
                        e = cudaEventRecord(ev(6 + nb + r), st);
                        if (ok()) e = cudaStreamWaitEvent(down, ev(6 + nb + r), 0);
                        if (ok()) e = cudaMemcpyAsync((char*)io->dQ_host + r * q_chunk * ob, (const char*)io->d_dQ + r * q_chunk * ob, q_chunk * ob, cudaMemcpyDeviceToHost, down);
                        if (!ok()) return cuda_fail("step_host dQ D2H", (int)e);
                    }
                }
            }
        if (bf16_out) {
            int err = by_group ? 0 : launch_cast_bf16(aQ, io->d_dQ, (long long)nq, p->num_sms, st);
            if (!err && !cols_down) err = launch_cast_bf16(aK, io->d_dK, (long long)nk, p->num_sms, st);
            if (!err && !cols_down) err = launch_cast_bf16(aV, io->d_dV, (long long)nk, p->num_sms, st);
            if (err) return cuda_fail("step_host cast launch", err);
            g_launches.fetch_add((by_group ? 0 : 1) + (cols_down ? 0 : 2));
        }
        e = cudaEventRecord(ev(4), st);
        if (ok()) e = cudaStreamWaitEvent(down, ev(4), 0);
        if (ok() && io->dQ_host && !by_group) e = cudaMemcpyAsync(io->dQ_host, io->d_dQ, nq * ob, cudaMemcpyDeviceToHost, down);
        if (ok() && io->dK_host && !cols_down) e = cudaMemcpyAsync(io->dK_host, io->d_dK, nk * ob, cudaMemcpyDeviceToHost, down);
        if (ok() && io->dV_host && !cols_down) e = cudaMemcpyAsync(io->dV_host, io->d_dV, nk * ob, cudaMemcpyDeviceToHost, down);
    }
    if (ok()) e = cudaEventRecord(ev(5), down);
    if (ok()) e = cudaStreamWaitEvent(st, ev(5), 0);
    if (ok()) e = cudaStreamSynchronize(st);
    if (!ok()) return cuda_fail("step_host D2H", (int)e);
    return check_health(p, "step_host");
}

int64_t mesh_attn_launch_count(void) { return (int64_t)g_launches.load(); }

int mesh_attn_plan_health(const mesh_attn_plan* p)
{
    if (!p) return fail(MESH_ATTN_EINVAL, "plan_health: null plan");
    return check_health(p, "plan_health");
}

int mesh_attn_profile_enable(int32_t on, int32_t capacity)
{
    g_prof.on = false;
    if (!on) return MESH_ATTN_OK;
    if (capacity <= 0) return fail(MESH_ATTN_EINVAL, "profile_enable: capacity must be positive");
    while (g_prof.ev.size() < 2 * (size_t)capacity) {
        cudaEvent_t e;
        const cudaError_t rc = cudaEventCreate(&e);
        if (rc != cudaSuccess) return cuda_fail("profile_enable: cudaEventCreate", (int)rc);
        g_prof.ev.push_back(e);
    }
    g_prof.kind.assign(g_prof.ev.size() / 2, -1);
    g_prof.capacity = (size_t)capacity;
    g_prof.used = 0;
    g_prof.on = true;
    return MESH_ATTN_OK;
}

int mesh_attn_profile_read(int32_t kind, double* ms_total, int64_t* launches)
{
    if (!ms_total || !launches) return fail(MESH_ATTN_EINVAL, "profile_read: null pointer");
    double total = 0.0;
    int64_t cnt = 0;
    for (size_t i = 0; i < g_prof.used; ++i) {
        if (g_prof.kind[i] != kind) continue;
        float ms = 0.f;
        const cudaError_t rc = cudaEventElapsedTime(&ms, g_prof.ev[2 * i], g_prof.ev[2 * i + 1]);
        if (rc != cudaSuccess) return cuda_fail("profile_read: cudaEventElapsedTime (synchronise the stream first)", (int)rc);
        total += ms;
        ++cnt;
    }
    *ms_total = total;
    *launches = cnt;
    return MESH_ATTN_OK;
}

const char* mesh_attn_strerror(int status)
{
    switch (status) {
        case MESH_ATTN_OK: return "ok";
        case MESH_ATTN_EINVAL: return "invalid argument";
        case MESH_ATTN_EUNSUPPORTED: return "unsupported configuration";
        case MESH_ATTN_EWORKSPACE: return "caller buffer too small";
        case MESH_ATTN_ECUDA: return "CUDA error / no CUDA device";
        case MESH_ATTN_ENOMEM: return "out of memory";
        default: return "unknown status";
    }
}

const char* mesh_attn_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
