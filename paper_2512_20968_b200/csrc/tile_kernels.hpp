// tile_kernels.hpp -- parameter blocks and launchers of the CUDA kernels (internal).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

#include "plan.hpp"

namespace mesh_attn {

// tile_bwd's dQ staging: query rows per cp.reduce.async.bulk.tensor box (= box rows of the dQ tensor map built in capi.cu).
// The TMA reduce costs a fixed ~210 clk per box on top of its bytes (measured: 8 KB boxes 509 clk, 4 KB boxes 360 clk each,
// profiles/r02_v1_README.md), and its read of the staging memory completes ~1000-1500 clk after the issue (L2 atomics under load):
// what bounds the drain is the bytes in flight.  Without the pair's dQ exchange: a ring of four 8 KB buffers (16 rows each);
// with it: the step's 64 rows are staged at once and reduced as two 16 KB boxes while the next step's exchange runs.
#ifndef MESH_ATTN_STG_ROWS
#define MESH_ATTN_STG_ROWS 16
#endif
#ifndef MESH_ATTN_STG_ROWS_EXCH
#define MESH_ATTN_STG_ROWS_EXCH 32
#endif
constexpr int kBwdStgRows = MESH_ATTN_STG_ROWS, kBwdStgRowsExch = MESH_ATTN_STG_ROWS_EXCH;
constexpr int kBwdStgBytes = 32 * 1024;

constexpr int kMaxPeers = 16;   // largest Q group the peer-memory merge takes (a <= 16: BASELINE.json's largest mesh)

struct FwdParams {
    Geom gm;
    const FwdItem* items;      // per-simulated-GPU template, items_per_gpu entries
    const Seg* segs;
    const SegList* seglists;
    int items_per_gpu;
    int g_first, g_count;
    int split;                 // precision: 1 = P fed to the PV MMA as hi + lo bf16
    int pair;                  // 1: items 2k, 2k+1 stream the same K / V blocks -> 2-CTA clusters, cta_group::2 MMAs (tmK: 64-row boxes)
    float* partial_O;          // [g_count][slots][B][L][Hq][D]
    float* partial_lse;        // [g_count][slots][B][Hq][L]
    int* status;               // the plan's host-mapped status words (sm100.cuh watchdog); may be null
    int* counter;              // work-item counter of the launch (device memory; zero when the kernel starts)
};

struct BwdParams {
    Geom gm;
    const BwdItem* items;
    const Seg* segs;
    const SegList* seglists;
    int items_per_gpu;
    int g_first, g_count;
    int split;                 // precision: 1 = hi+lo bf16 operands for P and dS
    int pair;                  // 1: items 2k, 2k+1 walk the same Q blocks -> 2-CTA clusters with multicast Q/dO tiles (tmQ, tmdO: 64-row boxes);
                               // 2: the pair also exchanges dQ^T halves (bf16, distributed shared memory) and each CTA reduces 64 of the
                               //    step's 128 query rows (tmdQ: kBwdStgRowsExch-row boxes)
    int* status;               // the plan's host-mapped status words (sm100.cuh watchdog); may be null
    int* counter;              // work-item counter of the launch (device memory; zero when the kernel starts)
    const float* ws;           // [2][B][Hq][N]: delta, log2(scale) - lse*log2e (written by bwd_preprocess); head 0 = first head of the lane
    long long ws_plane;        // elements between ws[0] and ws[1] (B * all heads * N)
    long long vec_stride_b;    // batch stride of the [B][Hq][N] vectors (all heads * N)
    float *dQ, *dK, *dV;       // fp32 accumulators
    // element strides of dQ (query-shaped) and dK/dV (key-shaped) tensors
    long long q_stride_b, q_stride_row, q_stride_h;
    long long k_stride_b, k_stride_row, k_stride_h;
};

struct MergeParams {
    Geom gm;
    int q_group;
    int m;                     // partials per output row
    int per;                   // 1 (fused partials) or b (per-pair partials): slot(k) = (k/per)*slots + u_local*per + k%per
    int rows_per_block;
    const float* partial_O;
    const float* partial_lse;
    // peers != 0 (mesh_attn_rank_merge_peers): partial k is read from peer_O[k] / peer_lse[k] ([B][L][Hq][D] / [B][Hq][L]
    // each, possibly another GPU's memory mapped into this process) instead of slot k of partial_O / partial_lse
    int peers;
    const float* peer_O[kMaxPeers];
    const float* peer_lse[kMaxPeers];
    void* O;                   // fp32, or bf16 when out_bf16 (plan out_dtype = 1)
    int out_bf16;
    float* lse;
    long long lse_stride_b;    // batch stride of lse [B][Hq][N] (all heads * N)
    long long o_stride_b, o_stride_row, o_stride_h;   // element strides of O
};

struct SumParams {               // out[i] = sum_k src[k][i]: the reduce-scatters of Alg.3 l.6-7 read from where the members wrote
    int m;
    long long count4;            // float4 elements
    const float* src[kMaxPeers];
    float* out;
};

struct DeltaParams {
    Geom gm;
    const void* O;             // fp32, or bf16 when o_bf16 (plan out_dtype = 1)
    int o_bf16;
    const void* dO;            // bf16
    const float* lse;          // [B][Hq][N] final merged LSE (natural log)
    float* ws;                 // [2][B][Hq][N]: delta, log2(scale) - lse*log2e
    long long stride_b, stride_row, stride_h;   // element strides shared by O and dO
};

// each returns a cudaError_t value (0 = success)
int launch_tile_fwd(const FwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV, int num_sms,
                    cudaStream_t stream);
int launch_tile_bwd(const BwdParams& p, const CUtensorMap& tmQ, const CUtensorMap& tmK, const CUtensorMap& tmV,
                    const CUtensorMap& tmdO, const CUtensorMap& tmdQ, int num_sms, cudaStream_t stream);
int launch_merge(const MergeParams& p, cudaStream_t stream);
int launch_delta(const DeltaParams& p, cudaStream_t stream);
int launch_sum_peers(const SumParams& p, int num_sms, cudaStream_t stream);
int launch_cast_bf16(const float* src, void* dst, long long count, int num_sms, cudaStream_t stream);   // dst (bf16)[i] = src[i], count % 4 == 0

}  // namespace mesh_attn
