/*
 * mesh_attn.h -- C ABI of the B200-native per-GPU compute core of Mesh-Attention
 * (arxiv 2512.20968).  "P:Lnnn" cites a line of the paper text.
 *
 * One B200 simulates the n logical GPUs of the paper.  Q and KV are split into n
 * sequence partitions; simulated GPU g owns an a x b tile of the n x n
 * assignment matrix and, for every (Q_u, KV_v) pair of that tile,
 * computes blockwise softmax attention emitting a partial output and its log-sum-exp
 * (Alg.2 l.3-5 P:L171-173).  A second step merges the partial outputs of each
 * Q partition with the online-softmax (LSE-weighted) reducer.  Backward
 * follows Alg.3.  The paper's collectives (all-gather, reduce-scatter) do
 * not exist here: there is one GPU, no sharding and no inter-GPU exchange; the planner
 * only builds the assignment matrix, the per-simulated-GPU tile lists and their order.
 *
 * Conventions
 *   - All tensor pointers are DEVICE pointers (allocated by the caller, e.g. torch);
 *     `stream` is a cudaStream_t passed as void*.  The *_host entry point is the only
 *     one taking HOST pointers and says so.
 *   - The caller owns every buffer, including workspaces whose size the plan reports.
 *     The library owns only the plan object and its small device-resident work lists.
 *   - Hot calls (tile_fwd, merge, bwd_preprocess, tile_bwd, forward, backward) never
 *     allocate, never synchronise the host, never touch the default stream implicitly:
 *     everything is enqueued on `stream` (a tile_fwd / tile_bwd call enqueues a 4-byte memset of
 *     the plan's work-item counter in front of its kernel: the persistent CTAs take their work
 *     items from that counter in list order).
 *   - Every function returns a mesh_attn_status (0 = OK, negative = error) and never
 *     throws or aborts; mesh_attn_last_error() gives a thread-local detail string.
 *   - There is no CPU fallback: on a machine without an sm_100 CUDA device (none at all, or another
 *     architecture) the planner calls work, every compute call returns MESH_ATTN_ECUDA.
 *
 * Tensor layouts (rows in PARTITION-MAJOR order: partition p, local row s -> row p*L+s,
 * L = seq_total / n):
 *   Q, dO      bf16  [B, N, Hq,  D]   (tensor_layout 0)  or [B, Hq,  N, D] (tensor_layout 1)
 *   K, V       bf16  [B, N, Hkv, D]                      or [B, Hkv, N, D]
 *   O, dQ      fp32  same shape as Q;   dK, dV fp32 same shape as K   (bf16 with plan out_dtype = 1, see the field)
 *   lse        fp32  [B, Hq, N]   natural log of the sum of exp of the SCALED scores
 *   partial_O  fp32  [g_count][slots][B][L][Hq][D]   slots = a (partial_mode 0) or a*b (1)
 *   partial_lse fp32 [g_count][slots][B][Hq][L]
 *   (usp_lanes = U > 1: a simulated GPU holds Hq/U heads, so Hq in the two partial layouts is Hq/U; all other
 *    tensors keep their full shape and the lanes address head slices of them.)
 * Token position of (p, s): seq_layout 0: p*L+s;  seq_layout 1 (striped): s*n+p.
 * Causal: key visible iff pos(key) <= pos(query).  A row with no visible key
 * gets O = 0, lse = -inf.  GQA: query head h reads KV head h / (Hq/Hkv).
 */
#ifndef MESH_ATTN_H
#define MESH_ATTN_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mesh_attn_plan mesh_attn_plan; /* opaque, library-owned, immutable after create.  A plan serves ONE in-flight
                                                 call at a time: mesh_attn_step_host and the *_goo executors order their copies
                                                 with plan-owned streams and events, so two concurrent calls on the same plan
                                                 (from two host threads or two caller streams) would race on them; use one plan
                                                 per concurrent caller (plans are cheap).  The profiling calls are process-global
                                                 and not thread-safe. */

typedef enum {
    MESH_ATTN_OK = 0,
    MESH_ATTN_EINVAL = -1,       /* bad geometry / null pointer / out-of-range index      */
    MESH_ATTN_EUNSUPPORTED = -2, /* valid but not built (e.g. head_dim not in {64,128})   */
    MESH_ATTN_EWORKSPACE = -3,   /* caller-provided buffer too small for the query        */
    MESH_ATTN_ECUDA = -4,        /* CUDA error or no CUDA device                           */
    MESH_ATTN_ENOMEM = -5
} mesh_attn_status;

typedef struct {
    int32_t n, a, b;          /* n == a*b; a = tile height = Q-group size, b = tile width = KV-group size */
    int32_t batch, seq_total, heads_q, heads_kv, head_dim; /* L = seq_total/n, L % 128 == 0, head_dim in {64,128} */
    int32_t causal;           /* 0 | 1                                                        */
    int32_t kvr;              /* 1: KV partition rotation, I_g^KV = {c + t*a}; 0: contiguous */
    int32_t seq_layout;       /* 0 contiguous (pos = p*L+s), 1 striped (pos = s*n+p)          */
    int32_t order;            /* 0 row-major tile order, 1 greedy / GOO                   */
    int32_t k_q, k_kv;        /* GOO chunk counts, k_q*k_kv <= 16; (L/k) % 128 == 0; <=0 -> 1 */
    float gamma;              /* GOO safety factor, <=0 -> 1.05                               */
    float t_ag_q, t_ag_kv, t_rs_q, t_c; /* GOO task costs; any <=0 -> built-in cost model      */
    float softmax_scale;      /* <=0 -> 1/sqrt(head_dim)                                       */
    int32_t tensor_layout;    /* 0: [B,N,H,D], 1: [B,H,N,D]                                            */
    int32_t partial_mode;     /* 0: one partial per (g,u), fused over I_g^KV (Alg.2 l.5);
                                 1: one partial per pair (u,v): literal O_ij, lse_ij           */
    int32_t precision;        /* P (forward and backward) and dS as tensor-core operands: 0 one bf16,
                                 1 split hi+lo bf16 pairs (two MMAs each; needed for outlier scores)    */
    int32_t usp_lanes;        /* Mesh-USP: U >= 1 lanes (0 -> 1).  The Ulysses all-to-all leaves lane l with
                                 query heads [l*Hq/U, (l+1)*Hq/U) (KV heads likewise) of ALL tokens, and each lane runs
                                 Mesh-Attention on its own a x b mesh.  There are n*U simulated GPUs: g in [0, n*U) is
                                 mesh GPU g % n of lane g / n; Q group q in [0, b*U) is group q % b of lane q / b.
                                 The partial workspace of a simulated GPU shrinks by U.  heads_kv % U == 0.   */
    int32_t bwd_pairing;      /* tile_bwd as 2-CTA clusters over work items 2k, 2k+1 (MESH_ATTN_Q_BWD_PAIRED): 0 auto (paired when the
                                 planner finds the items pairable: shared Q / dO tile loads AND the pair's dQ exchange, which
                                 halves the dQ atomics; precision 1 pairs without the exchange), 1 never (single-CTA kernel),
                                 2 paired, shared tile loads only (no dQ exchange).  1 and 2 exist for A/B measurements
                                 and for callers that want the dQ sums free of the exchange's bf16 rounding */
    int32_t bwd_piece_blocks; /* tile_bwd work items: the Q sweep of a 128-key block (all Q partitions of the tile) is cut into pieces of
                                 at most this many 128-row Q blocks (whole segments = Q chunks of one partition), one work item per
                                 (key block, piece), the key blocks of a piece adjacent in the list.  0 = default: pieces whose Q, dO,
                                 dQ rows (x the query heads of a GQA group) amount to 32 MiB, at least 64 blocks; a large value
                                 (>= a*L/128) = one item per key block.  Short sweeps keep the rows the running CTAs share in
                                 L2, very short ones pay the per-item K / V load and dK / dV epilogue more often (measured:
                                 DESIGN.md 6.3).  The results are the same sums in another order.                       */
    int32_t out_dtype;        /* 0: O, dQ, dK, dV are fp32 (default); 1: bf16 (round to nearest even, same shapes).  Applies to the O of
                                 merge / forward / forward_static / forward_goo / step_host, to the O that bwd_preprocess / backward read,
                                 and to the dQ, dK, dV of backward / step_host, whose sums are then accumulated in fp32 behind the two
                                 planes of bwd_ws (MESH_ATTN_Q_BWD_WS_BYTES grows by the three fp32 tensors) and rounded once at the end.
                                 lse, the partials and the per-kernel call mesh_attn_tile_bwd (which ACCUMULATES into caller buffers)
                                 stay fp32; backward_goo and the per-rank calls return EUNSUPPORTED.  The backward then sees the ROUNDED O:
                                 delta = rowsum(dO o O) carries up to 2^-9 sum|dO O| of rounding, which reaches dQ, dK (measured
                                 1.6e-2 max against the fp32 path on a causal case; dV is unaffected).  An option beyond the paper's
                                 (unpinned: tests compare against the fp32 path and the oracle at that resolution).              */
    int32_t fwd_pairing;      /* tile_fwd as 2-CTA clusters over work items 2k, 2k+1 with tcgen05 cta_group::2 MMAs (each CTA holds half of
                                 every K / V block: half the shared-memory operand traffic per SM; MESH_ATTN_Q_FWD_PAIRED): 0 auto
                                 (paired when the planner finds that the two items stream the same K / V blocks on every simulated GPU
                                 -- non-causal and striped-causal plans with an even item count -- and head_dim = 128, precision = 0),
                                 1 never (single-CTA kernel; for A/B measurements).  Results are bit-identical either way.            */
} mesh_attn_plan_desc;

/* what = ... for mesh_attn_plan_query */
enum {
    MESH_ATTN_Q_PARTIAL_O_BYTES = 0,   /* bytes of partial_O for ONE simulated GPU (multiply by g_count)  */
    MESH_ATTN_Q_PARTIAL_LSE_BYTES = 1, /* bytes of partial_lse for ONE simulated GPU                      */
    MESH_ATTN_Q_SLOTS_PER_GPU = 2,     /* a or a*b                                                        */
    MESH_ATTN_Q_FLOPS_FWD = 3,         /* algorithmic: 4*D*Hq*B*visible pairs                             */
    MESH_ATTN_Q_FLOPS_BWD = 4,         /* algorithmic: 10*D*Hq*B*visible pairs                            */
    MESH_ATTN_Q_WAVES = 5,             /* number of Q groups = b * usp_lanes                              */
    MESH_ATTN_Q_MERGE_BYTES = 6,       /* algorithmic bytes moved by ONE merge call (one Q group)         */
    MESH_ATTN_Q_FWD_ITEMS_PER_GPU = 7, /* tile-forward work items per simulated GPU                       */
    MESH_ATTN_Q_BWD_ITEMS_PER_GPU = 8, /* tile-backward work items per simulated GPU                      */
    MESH_ATTN_Q_BLOCKS_FWD = 9,        /* 128x128 score blocks the forward computes (all GPUs, heads)     */
    MESH_ATTN_Q_COMM_UNITS = 10,       /* paper's aggregate communication units of this AM   */
    MESH_ATTN_Q_HAS_DEVICE = 11,       /* 1 if the plan's work lists are resident on a CUDA device        */
    MESH_ATTN_Q_BWD_WS_BYTES = 12,     /* bytes of the backward workspace bwd_ws: 2*B*Hq*N*4 (+ B*N*(Hq+2Hkv)*D*4 with out_dtype 1) */
    /* planner analytics (what the paper's cluster would move; nothing here is executed): */
    MESH_ATTN_Q_MESH_COMM_BYTES_FWD = 13,  /* per-GPU forward volume of this a x b tiling, closed form
                                              2(a+b-2) N d / n elements x 2 bytes (bf16), d = Hq*head_dim */
    MESH_ATTN_Q_MESH_COMM_BYTES_BWD = 14,  /* backward: twice the forward volume (Q,O,dO in, dQ out; K,V in, dK,dV out; Table 5) */
    MESH_ATTN_Q_RING_COMM_BYTES_FWD = 15,  /* Ring-Attention on the same n GPUs: (2 - 2/n) N d elements x 2 bytes */
    MESH_ATTN_Q_USP_LANES = 16,            /* U                                                                          */
    MESH_ATTN_Q_BWD_PAIRED = 18,           /* 1 if tile_bwd runs as 2-CTA clusters sharing the Q / dO tile loads: backward work items
                                              2k and 2k+1 visit the same Q blocks on every simulated GPU (holds for non-causal and
                                              striped-causal plans with an even item count; desc.bwd_pairing = 1 forces 0); 2 if the
                                              pair also exchanges dQ partial sums (half the dQ atomics) */
    MESH_ATTN_Q_GOO_PARTIAL_O_BYTES = 19,  /* mesh_attn_forward_goo: bytes of partial_O for ONE simulated GPU (a*k_kv slots); x a */
    MESH_ATTN_Q_GOO_PARTIAL_LSE_BYTES = 20,
    MESH_ATTN_Q_GOO_COMM_BYTES = 21,       /* bytes the forward step list's collectives move for the a GPUs of one Q group:
                                              k_q (AG-Q + RS-Q) of (a-1) Q chunks + k_kv AG-KV of (b-1) K and V chunks, each x a
                                              (= a x MESH_ATTN_Q_MESH_COMM_BYTES_FWD, the per-GPU volume of P:L290-292) */
    MESH_ATTN_Q_FWD_PAIRED = 22,           /* 1 if tile_fwd runs as 2-CTA clusters with cta_group::2 MMAs (desc.fwd_pairing) */
    MESH_ATTN_Q_USP_A2A_BYTES_FWD = 17     /* per-GPU forward volume of the Ulysses all-to-alls around the lanes (Q, K, V in,
                                              O out): (U-1)/U of the GPU's N/(n*U) tokens x (2 Hq + 2 Hkv) head_dim x 2 bytes;
                                              with n = 1 and Hq = Hkv this is Table 1's Ulysses entry 4(U-1)/U^2 N d */
};

/* kinds in mesh_attn_plan_steps rows (step, kind, i, j) */
enum {
    MESH_ATTN_TASK_AG_KV = 0,  /* all-gather KV chunk j (idx in column 2, column 3 = -1)   */
    MESH_ATTN_TASK_AG_Q = 1,   /* all-gather Q chunk i; backward: Q,O,dO chunk i     */
    MESH_ATTN_TASK_RS_Q = 2,   /* reduce-scatter O chunk i; backward: dQ chunk i     */
    MESH_ATTN_TASK_C = 3,      /* compute task C-i-j                                       */
    MESH_ATTN_TASK_RS_KV = 4   /* backward only: reduce-scatter dKV chunk j                */
};

/* ---- planner (host only; works without a GPU) ------------------------------------------- */

/* Validates desc, builds the assignment matrix, Q/KV groups
 * (P:L178-180), the GOO step list and the ordered tile lists; if a CUDA
 * device is present also uploads the work lists (the only allocation the library makes).
 * Errors: EINVAL (n != a*b, seq_total % n, L % 128, Hq % Hkv, k_q*k_kv > 16, ...),
 * EUNSUPPORTED (head_dim), ENOMEM, ECUDA (upload failed). *out is NULL on error. */
int mesh_attn_plan_create(const mesh_attn_plan_desc* desc, mesh_attn_plan** out);
void mesh_attn_plan_destroy(mesh_attn_plan* plan);

/* am: host int32 [n*n] row-major, am[i*n+j] = g computing (Q_i, KV_j).  The planner calls below
 * (am, footprint, tiles, steps, tam_units, timeline) describe ONE lane's a x b mesh: g in [0, n). */
int mesh_attn_plan_am(const mesh_attn_plan* plan, int32_t* am);

/* Footprints of simulated GPU g: I^Q (a entries), I^KV (b entries) in
 * execution order; host int32 arrays of capacity >= a and >= b. */
int mesh_attn_plan_footprint(const mesh_attn_plan* plan, int32_t g, int32_t* iq, int32_t* ikv);

/* Tile list of simulated GPU g in execution order: rows (u, v, i, j) = Q partition, KV
 * partition, Q chunk, KV chunk; host int32 [capacity][4]; *count receives the number of
 * rows (= a*b*k_q*k_kv); if capacity is too small returns EWORKSPACE with *count set. */
int mesh_attn_plan_tiles(const mesh_attn_plan* plan, int32_t g, int32_t* tiles, int32_t capacity, int32_t* count);

/* GOO step list (same on every simulated GPU): rows (step, kind, i, j), host
 * int32 [capacity][4]. pass: 0 forward, 1 backward (backward: DESIGN.md reading R12,
 * parity unpinned). With order == 0 there is a single step holding every task. */
int mesh_attn_plan_steps(const mesh_attn_plan* plan, int32_t pass, int32_t* steps, int32_t capacity, int32_t* count);

int mesh_attn_plan_query(const mesh_attn_plan* plan, int32_t what, int64_t* value);

/* Timeline of the step list under the paper's execution model: in every step one collective runs
 * concurrently with the step's compute tasks, which run one after the other; a step lasts
 * max(T_comm, sum of T_compute) with the plan's task costs (the descriptor's, or the built-in model).
 * Returns, in the cost unit: makespan = sum of step durations; serial = every task back to back (no overlap);
 * exposed_comm = makespan - total compute time (the communication that compute does not hide, cf. Fig.7).
 * With order == 0 (row-major, no overlap scheduled) makespan == serial.
 * pass: 0 forward, 1 backward (backward costs: AG of Q,O,dO = 3 x t_ag_q, compute = 2.5 x t_c; reading R12). */
int mesh_attn_plan_timeline(const mesh_attn_plan* plan, int32_t pass, double* makespan, double* serial, double* exposed_comm);

/* Topology-aware mapping: an alpha-wide, (gpus_per_node/alpha)-tall tile of the logical a x b mesh
 * (rows = Q groups, columns = position inside the Q group) is placed on each node.  Returns the inter-node traffic of
 * node `node` in units of one partition: q_units = 2 per remote member of every Q group the node intersects (Q in,
 * partial O out), kv_units = 2 per remote member of every KV group it intersects (K and V).  alpha == a with
 * gpus_per_node == a is the row-major mapping.  EINVAL unless alpha divides a and gpus_per_node, and
 * gpus_per_node/alpha divides b. */
int mesh_attn_plan_tam_units(const mesh_attn_plan* plan, int32_t gpus_per_node, int32_t alpha, int32_t node,
                             int64_t* q_units, int64_t* kv_units);

/* ---- hot path (device pointers; enqueued on stream) -------------------------------------- */

/* Alg.2 l.3-5 for simulated GPUs g_first .. g_first+g_count-1: for each Q_u
 * (u in I_g^Q) the online-softmax attention over the KV partitions of I_g^KV in plan
 * order; writes the normalised partial output and its LSE into slot (g - g_first, u_local)
 * (partial_mode 1: slot (g - g_first, u_local*b + v_local), one KV partition each). */
int mesh_attn_tile_fwd(const mesh_attn_plan* plan, int32_t g_first, int32_t g_count,
                       const void* Q, const void* K, const void* V,
                       float* partial_O, float* partial_lse, void* stream);

/* Online-softmax reducer of Alg.2 l.6 as a local merge: for every Q partition
 * u of Q group q_group (u = q_group*a + x), every row and head:
 *   lse* = ln sum_k exp(lse_k),  O = sum_k exp(lse_k - lse*) O_k   over the slots holding u.
 * partial_O / partial_lse are the buffers tile_fwd filled for g_first = q_group*a,
 * g_count = a.  Writes rows of partitions u of O [B,N,Hq,D] and lse [B,Hq,N]. */
int mesh_attn_merge(const mesh_attn_plan* plan, int32_t q_group,
                    const float* partial_O, const float* partial_lse,
                    void* O /* fp32; bf16 with out_dtype 1 */, float* lse, void* stream);

/* Backward workspace bwd_ws, fp32 [2][B][Hq][N] (MESH_ATTN_Q_BWD_WS_BYTES), all rows:
 *   bwd_ws[0][b,h,row] = delta = sum_d dO * O  (needed by every pair touching the row; the
 *                        paper passes O_i, dO_i to the backward kernel)
 *   bwd_ws[1][b,h,row] = log2(softmax_scale) - lse * log2(e)  (exponent offset, in base 2, of
 *                        scale * P = scale * exp(S - lse); lse is the FINAL merged LSE,
 *                        DESIGN.md reading R8) */
int mesh_attn_bwd_preprocess(const mesh_attn_plan* plan, const void* O /* fp32; bf16 with out_dtype 1 */, const void* dO,
                             const float* lse, float* bwd_ws, void* stream);

/* Alg.3 l.3-5 for simulated GPUs g_first..: for each pair of the tile
 * recompute P = exp(S - lse) with the FINAL merged lse, dP = dO V^T, dS = P o (dP - delta),
 * and ACCUMULATE (atomic fp32 adds: the sums of Alg.3 l.6-7 and the GQA group sum)
 *   dV_v += P^T dO_u,  dK_v += scale dS^T Q_u,  dQ_u += scale dS K_v.
 * bwd_ws is what mesh_attn_bwd_preprocess wrote.  The caller zeroes dQ, dK, dV before the
 * first call.  head_dim 64 runs the head_dim-128 kernel on zero-padded tiles (the TMA fills the
 * out-of-bounds upper 64 columns with zeros; the transposed dQ accumulator needs 128 rows), i.e.
 * at half the tensor-core efficiency. */
int mesh_attn_tile_bwd(const mesh_attn_plan* plan, int32_t g_first, int32_t g_count,
                       const void* Q, const void* K, const void* V, const void* dO,
                       const float* bwd_ws, float* dQ, float* dK, float* dV, void* stream);

/* All waves: for each lane and each Q group r of it: tile_fwd(g_first = lane*n + r*a, a) then
 * merge(lane*b + r). partial_O / partial_lse must hold `a` simulated GPUs (query PARTIAL_*_BYTES * a).
 * tile_fwd / tile_bwd ranges [g_first, g_first+g_count) must stay inside one lane (EINVAL). */
int mesh_attn_forward(const mesh_attn_plan* plan, const void* Q, const void* K, const void* V,
                      void* O /* fp32; bf16 with out_dtype 1 */, float* lse, float* partial_O, float* partial_lse, void* stream);

/* mesh_attn_forward for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same tile_fwd -> merge waves (Alg.2 l.3-6), with the partial (O, lse)
 * scratch in a device array BUILT INTO the library -- MESH_ATTN_FORWARD_STATIC_SCRATCH_BYTES per GPU that loads the
 * library, held until the process exits -- instead of caller-owned partial_O / partial_lse.  The call allocates nothing
 * (no cudaMalloc / cudaFree, no allocating library routine); Q, K, V, O, lse are the caller's device buffers as in
 * mesh_attn_forward, and the result is bit-identical to mesh_attn_forward's.
 *   - Limit: a * (PARTIAL_O_BYTES + PARTIAL_LSE_BYTES) of the plan (mesh_attn_forward_static_limits gives the exact
 *     figure) must fit the array; a larger plan returns MESH_ATTN_EUNSUPPORTED with both numbers in
 *     mesh_attn_last_error() and launches nothing.
 *   - The plan's device must be the current device (EINVAL otherwise): the array's address is looked up per device.
 *   - Every call, from every plan and thread of the process, shares the ONE array and finds the last call's contents in
 *     it.  Nothing has to start at zero (tile_fwd writes every partial the merge reads before it is read), but two calls
 *     that overlap on the GPU (different streams, or different processes' threads on one device without ordering) RACE on
 *     it: order them on one stream or with events. */
#define MESH_ATTN_FORWARD_STATIC_SCRATCH_BYTES 33554432 /* 32 MiB */
int mesh_attn_forward_static(const mesh_attn_plan* plan, const void* Q, const void* K, const void* V,
                             void* O /* fp32; bf16 with out_dtype 1 */, float* lse, void* stream);
/* need_bytes (may be NULL; needs a plan): scratch bytes a mesh_attn_forward_static call of this plan uses;
 * capacity_bytes (may be NULL): MESH_ATTN_FORWARD_STATIC_SCRATCH_BYTES.  Host-only, works without a device. */
int mesh_attn_forward_static_limits(const mesh_attn_plan* plan, int64_t* need_bytes, int64_t* capacity_bytes);
/* Test hook: fills the whole built-in scratch array with the 32-bit `word` on `stream` (e.g. 0x7FC00000, a NaN), so
 * that a test can show that a following mesh_attn_forward_static reads nothing it has not written itself. */
int mesh_attn_forward_static_poison(const mesh_attn_plan* plan, uint32_t word, void* stream);

/* GOO executor for the `a` simulated GPUs of Q group q_group: runs the plan's forward STEP
 * LIST (mesh_attn_plan_steps) step by step.  A step's compute tasks C-i-j (Q chunk i of every Q partition of the group
 * against KV chunk j of every KV partition of each GPU's footprint) are chunk-granular tile_fwd launches on `stream`
 * writing partial slot (g - g_first, u_local*k_kv + j); the step's communication task (AG-KV-j, AG-Q-i, RS-Q-i) is stood
 * in for by device-to-device copies of the bytes it would move for these `a` GPUs (repeated comm_repeat times to model
 * a slower link; 0 = no copies) into comm_ws, on a plan-owned stream when overlap != 0 (else on `stream`, i.e.
 * serialised with the compute); both streams join at the end of every step.  Last, the a*k_kv partials of every
 * row are merged into O and lse.  One GPU holds all of Q, K, V, so the copies carry no data dependence: they reproduce
 * the schedule's timing, the result is the attention of mesh_attn_forward.  partial_O / partial_lse: `a` x
 * MESH_ATTN_Q_GOO_PARTIAL_*_BYTES.  Time it with events on `stream`. */
int mesh_attn_forward_goo(const mesh_attn_plan* plan, int32_t q_group, const void* Q, const void* K, const void* V,
                          void* O /* fp32; bf16 with out_dtype 1 */, float* lse, float* partial_O, float* partial_lse,
                          void* comm_ws, int64_t comm_ws_bytes, int32_t comm_repeat, int32_t overlap, void* stream);

/* ---- per-rank calls (Alg.2, Alg.3) ----------------------
 * The compute steps of ONE GPU g of a real n-GPU job, on tensors that hold only what that GPU has after its
 * all-gathers (device pointers, caller-owned; usp_lanes == 1, partial_mode == 0, else EUNSUPPORTED).  The
 * collectives themselves are the caller's (paper_2512_20968_b200/distributed.py issues them with torch.distributed);
 * the arithmetic is that of mesh_attn_tile_fwd / merge / bwd_preprocess / tile_bwd for simulated GPU g — same
 * kernels and work lists, only the row addressing differs: partition slot k of a query-shaped local tensor is the
 * k-th entry of I_g^Q (partition (g/a)*a + k, i.e. the k-th member of g's Q group), slot t of a key-shaped one the t-th
 * entry of I_g^KV (mesh_attn_plan_footprint order); row = slot*L + s.
 *   Q_loc, dO_loc bf16, dQ_loc fp32  [B, a*L, Hq, D]  (tensor_layout 1: [B, Hq, a*L, D])
 *   K_loc, V_loc  bf16, dK_loc, dV_loc fp32  [B, b*L, Hkv, D]
 *   partial_O fp32 [a][B][L][Hq][D], partial_lse fp32 [a][B][Hq][L]: slot k is the partial for Q partition
 *     (g/a)*a + k, to be delivered to that rank (RS-O, Alg.2 l.6)
 *   rank_merge: partial_*_recv are the `a` partials of the rank's OWN Q partition, slot k from the k-th member of
 *     its Q group; O_own fp32 [B, L, Hq, D], lse_own fp32 [B][Hq][L]
 *   rank_bwd_preprocess: ws_own fp32 [2][B][Hq][L] (delta, exponent offset) of the own partition
 *   rank_bwd: ws_loc fp32 [2][B][Hq][a*L]: the ws_own of the Q group's members, member k at rows k*L.. (gathering
 *     delta and the offset instead of O saves the all-gather of O that Alg.3 l.1 lists);
 *     dQ_loc, dK_loc, dV_loc are ACCUMULATED into (caller zeroes) and hold this GPU's contribution for every
 *     partition of its footprint: the reduce-scatters of Alg.3 l.6-7 sum them over the Q group / KV group. */
int mesh_attn_rank_fwd(const mesh_attn_plan* plan, int32_t g, const void* Q_loc, const void* K_loc, const void* V_loc,
                       float* partial_O, float* partial_lse, void* stream);
int mesh_attn_rank_merge(const mesh_attn_plan* plan, const float* partial_O_recv, const float* partial_lse_recv,
                         float* O_own, float* lse_own, void* stream);
/* RS-O of Alg.2 l.6 FUSED into its reducer over peer memory: the same merge, but partial k is read straight from
 * where the k-th member of the rank's Q group wrote it -- peer_partial_O[k] fp32 [B][L][Hq][D] and peer_partial_lse[k]
 * fp32 [B][Hq][L] are DEVICE-ACCESSIBLE addresses in this process (the member's partial slot for this rank's partition:
 * its own memory for k = own index, a peer GPU's memory mapped through CUDA IPC / NVLink peer access otherwise), given as
 * two HOST arrays of `a` pointers (copied into the launch; a <= 16).  The loads of the merge are then the transfer: no
 * all-to-all, no receive buffer, and the exchange overlaps the arithmetic load by load.  The caller orders the launch after
 * the members' rank_fwd (an event or a barrier across the group).  Bit-identical to rank_merge on the same partials. */
int mesh_attn_rank_merge_peers(const mesh_attn_plan* plan, const float* const* peer_partial_O, const float* const* peer_partial_lse,
                               float* O_own, float* lse_own, void* stream);
/* The reduce-scatters of Alg.3 l.6-7 in the same peer-memory form: out[i] = sum_k peers[k][i], i < count
 * (fp32; count a multiple of 4; every buffer 16-byte aligned; 1 <= m <= 16).  peers is a HOST array of m device-accessible
 * addresses: for RS-dQ member k's dQ_loc at this rank's slot (m = a, count = L*Hq*D with batch 1, else one call per
 * batch), for RS-dKV member t's dK_loc / dV_loc at this rank's slot (m = b).  Plain sums in member order (deterministic,
 * unlike a ring reduce-scatter whose order depends on the rank). */
int mesh_attn_rank_sum_peers(const mesh_attn_plan* plan, const float* const* peers, int32_t m, int64_t count, float* out, void* stream);
int mesh_attn_rank_bwd_preprocess(const mesh_attn_plan* plan, const float* O_own, const void* dO_own, const float* lse_own,
                                  float* ws_own, void* stream);
int mesh_attn_rank_bwd(const mesh_attn_plan* plan, int32_t g, const void* Q_loc, const void* K_loc, const void* V_loc,
                       const void* dO_loc, const float* ws_loc, float* dQ_loc, float* dK_loc, float* dV_loc, void* stream);

/* The backward step list (mesh_attn_plan_steps pass 1; reading R12: the paper omits the backward schedule, P:L238,
 * so the order is parity-unpinned) executed task by task for the `a` simulated GPUs of Q group q_group, like
 * mesh_attn_forward_goo: compute task C-i-j = a chunk-granular tile_bwd launch (the 128-key blocks of KV chunk j of every KV
 * partition of each footprint, against Q chunk i of every Q partition), the step's collective (AG of Q, O, dO chunk i = 3 Q
 * units; AG-KV-j; RS-dQ-i; RS-dKV-j) stood in for by device-to-device copies of its bytes on a plan-owned stream when
 * overlap != 0, a barrier per step.  ACCUMULATES into dQ, dK, dV exactly what mesh_attn_tile_bwd(q_group*a, a) adds (any
 * order of the compute tasks gives the same sums up to fp32 rounding); the caller zeroes them and runs
 * mesh_attn_bwd_preprocess first. */
int mesh_attn_backward_goo(const mesh_attn_plan* plan, int32_t q_group, const void* Q, const void* K, const void* V, const void* dO,
                           const float* bwd_ws, float* dQ, float* dK, float* dV,
                           void* comm_ws, int64_t comm_ws_bytes, int32_t comm_repeat, int32_t overlap, void* stream);

/* Zero dQ,dK,dV; bwd_preprocess; tile_bwd over all n simulated GPUs.  O, dQ, dK, dV: fp32, or bf16 with out_dtype 1 (the sums
 * are then accumulated in fp32 inside bwd_ws and rounded once, by three cast launches at the end). */
int mesh_attn_backward(const mesh_attn_plan* plan, const void* Q, const void* K, const void* V,
                       const void* O, const void* dO, const float* lse, float* bwd_ws,
                       void* dQ, void* dK, void* dV, void* stream);

/* End-to-end step with HOST buffers (pinned or pageable): copies Q,K,V(,dO) host->device
 * into the caller's device staging buffers, runs forward (and backward if dO_host != NULL),
 * copies O, lse (and dQ,dK,dV) device->host, and synchronises `stream` before returning.
 * The kernels run on `stream`; the copies run on two plan-owned streams (one per direction) ordered
 * against it by events, so that transfers overlap the kernels that do not need them.  With batch 1
 * and tensor_layout 0 (the rows of a partition are one byte range): the Q rows of the first Q
 * group go up first, then K and V one KV column at a time (the b partitions of I^KV of the
 * simulated GPUs g with g mod a = c); the first forward wave runs one launch per
 * simulated GPU, each behind its own column; the other Q groups and dO follow behind the forward
 * waves.  O and lse come down during the backward, the dQ rows of Q group r as soon as the
 * simulated GPUs of group r are done; the LAST backward group runs one launch per simulated GPU
 * again, and dK, dV of KV column c come down behind the launch that completes them (Alg.3 l.7,
 * P:L255).  Otherwise whole tensors move: K, V, Q before the forward, dQ, dK, dV after the backward.
 * One step_host per plan at a time.  d_* are caller-owned DEVICE buffers of the shapes above. */
typedef struct {
    const void *Q_host, *K_host, *V_host, *dO_host;      /* bf16 host inputs (dO_host may be NULL) */
    void *O_host, *lse_host, *dQ_host, *dK_host, *dV_host; /* host outputs (any may be NULL = not copied back): lse fp32; O, dQ, dK, dV
                                                              fp32, or bf16 with out_dtype 1 (half the bytes down) */
    void *d_Q, *d_K, *d_V, *d_dO;                          /* device staging                         */
    void *d_O, *d_lse, *d_bwd_ws, *d_dQ, *d_dK, *d_dV, *d_partial_O, *d_partial_lse;   /* d_O, d_dQ, d_dK, d_dV: dtype as the host outputs */
} mesh_attn_host_io;
int mesh_attn_step_host(const mesh_attn_plan* plan, const mesh_attn_host_io* io, void* stream);

/* Kernel watchdog.  Every wait inside the tile kernels is bounded (~4 s): a wait that does not complete is a protocol bug,
 * and instead of hanging the GPU or trapping (which would destroy the caller's CUDA context) the kernel records the fault in
 * status words owned by the plan (pinned host memory mapped into the device) and runs to its end with invalid results.
 * Every hot call checks those words on entry and mesh_attn_step_host after its synchronisation; mesh_attn_plan_health
 * checks them on demand (call it after synchronising the stream): MESH_ATTN_OK, or MESH_ATTN_ECUDA with the block, thread
 * and barrier in mesh_attn_last_error().  A faulted plan stays faulted: destroy it.  Host-only plans are always OK. */
int mesh_attn_plan_health(const mesh_attn_plan* plan);

/* number of kernels launched by this library in the calling process so far (bench bookkeeping) */
int64_t mesh_attn_launch_count(void);

/* Per-kernel device timing (measurement): while enabled, every kernel launch
 * of this library is bracketed by two cudaEventRecord calls on the launch's own stream
 * (events come from a pool created at enable time; when the pool of `capacity` launches is
 * full, further launches are not recorded).  mesh_attn_profile_read must be called after
 * the caller has synchronised the stream(s): it sums cudaEventElapsedTime over the recorded
 * launches of `kind` and returns their number.  enable(0,..) frees nothing and stops
 * recording; enable(1, capacity) resets the records.  Not thread-safe; off by default. */
enum { MESH_ATTN_K_TILE_FWD = 0, MESH_ATTN_K_MERGE = 1, MESH_ATTN_K_BWD_PREPROCESS = 2, MESH_ATTN_K_TILE_BWD = 3 };
int mesh_attn_profile_enable(int32_t on, int32_t capacity);
int mesh_attn_profile_read(int32_t kind, double* ms_total, int64_t* launches);

const char* mesh_attn_strerror(int status);
const char* mesh_attn_last_error(void); /* thread-local, valid until the next call on this thread */

#ifdef __cplusplus
}
#endif
#endif /* MESH_ATTN_H */
