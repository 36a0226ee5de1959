// aux_kernels.cu -- the two HBM-bound kernels of the hot path:
//   merge_kernel   LSE-weighted merge of the partial outputs of a Q group (online-softmax
//                  reducer of PAPER.md L77, Alg.2 l.6 L174; reading R4)
//   delta_kernel   backward preprocess Delta = rowsum(dO o O), plus -lse*log2e
//   cast_kernel    plan out_dtype = 1: the fp32 gradient accumulators -> the caller's bf16 dQ, dK, dV
// Both are streaming kernels: 16-byte vector loads, many independent loads in flight per
// thread, streaming cache hints, no shared-memory reuse of the bulk data.
#include <algorithm>

#include <cuda_bf16.h>

#include "tile_kernels.hpp"

namespace mesh_attn {
namespace {

__device__ __forceinline__ float4 ld_stream(const float4* p)
{
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void st_stream(float4* p, const float4& v)
{
    asm volatile("st.global.cs.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

__device__ __forceinline__ uint2 pack4_bf16(const float4& v)
{
    const __nv_bfloat162 lo = __floats2bfloat162_rn(v.x, v.y), hi = __floats2bfloat162_rn(v.z, v.w);
    return make_uint2(*reinterpret_cast<const uint32_t*>(&lo), *reinterpret_cast<const uint32_t*>(&hi));
}
__device__ __forceinline__ void st_stream_bf16x4(void* p, const float4& v)
{
    const uint2 w = pack4_bf16(v);
    asm volatile("st.global.cs.v2.b32 [%0], {%1, %2};" ::"l"(p), "r"(w.x), "r"(w.y) : "memory");
}

constexpr int kMergeThreads = 256;
constexpr int kMergeUnroll = 8;

// grid: (L / rows_per_block, a, B).  One block merges rows_per_block rows x all Hq heads of one
// Q partition.  Phase 1: one thread per (row, head) turns the m LSE values into weights
// w_k = exp(lse_k - lse*) (smem) and writes lse*.  Phase 2: every thread streams float4 columns:
// out = sum_k w_k * partial_k.
template <int D, bool kPeers>
__global__ void __launch_bounds__(kMergeThreads) merge_kernel(const MergeParams p)
{
    extern __shared__ float w_smem[];            // [rows][Hq][m]
    const Geom& gm = p.gm;
    const int rows = p.rows_per_block, m = p.m, Hq = gm.heads_q;
    const int s0 = blockIdx.x * rows, ul = blockIdx.y, bt = blockIdx.z;
    const int u = p.q_group * gm.a + ul;
    const size_t unit_lse = (size_t)gm.batch * Hq * gm.L;          // one slot of partial_lse
    const size_t unit_o = unit_lse * D;                             // one slot of partial_O

    for (int idx = threadIdx.x; idx < rows * Hq; idx += kMergeThreads) {
        const int r = idx % rows, h = idx / rows;                  // consecutive threads -> consecutive rows (coalesced lse)
        float mx = -INFINITY;
        for (int k = 0; k < m; ++k) {
            const size_t slot = (size_t)(k / p.per) * gm.slots_per_gpu + (size_t)ul * p.per + (k % p.per);
            const float* src_lse = kPeers ? p.peer_lse[k] : p.partial_lse + slot * unit_lse;
            const float x = src_lse[((size_t)bt * Hq + h) * gm.L + s0 + r];
            w_smem[(r * Hq + h) * m + k] = x;
            mx = fmaxf(mx, x);
        }
        float sum = 0.f;
        for (int k = 0; k < m; ++k) {
            const float x = w_smem[(r * Hq + h) * m + k];
            sum += (x == -INFINITY) ? 0.f : __expf(x - mx);
        }
        const float lse = (mx == -INFINITY) ? -INFINITY : mx + __logf(sum);
        for (int k = 0; k < m; ++k) {
            const float x = w_smem[(r * Hq + h) * m + k];
            w_smem[(r * Hq + h) * m + k] = (x == -INFINITY) ? 0.f : __expf(x - lse);
        }
        p.lse[(size_t)bt * p.lse_stride_b + (size_t)h * (size_t)gm.rows_q + (size_t)u * gm.L + s0 + r] = lse;
    }
    __syncthreads();

    constexpr int V = D / 4;                                        // float4 per (row, head)
    const int total = rows * Hq * V;
    const size_t src_at = ((size_t)bt * gm.L + s0) * Hq * V;    // float4 index of the block's first element inside one partial
    const float4* src = reinterpret_cast<const float4*>(p.partial_O) + src_at;
    for (int i = threadIdx.x; i < total; i += kMergeThreads) {
        const int rh = i / V, d4 = i - rh * V;                     // rh = r*Hq + h : contiguous in the partial buffers
        const float* w = w_smem + rh * m;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int k0 = 0; k0 < m; k0 += kMergeUnroll) {
            float4 x[kMergeUnroll];
#pragma unroll
            for (int kk = 0; kk < kMergeUnroll; ++kk) {
                const int k = k0 + kk;
                if (k < m) {
                    const size_t slot = (size_t)(k / p.per) * gm.slots_per_gpu + (size_t)ul * p.per + (k % p.per);
                    x[kk] = ld_stream(kPeers ? reinterpret_cast<const float4*>(p.peer_O[k]) + src_at + i : src + slot * (unit_o / 4) + i);
                }
            }
#pragma unroll
            for (int kk = 0; kk < kMergeUnroll; ++kk) {
                const int k = k0 + kk;
                if (k < m) {
                    const float wk = w[k];
                    acc.x = fmaf(wk, x[kk].x, acc.x); acc.y = fmaf(wk, x[kk].y, acc.y);
                    acc.z = fmaf(wk, x[kk].z, acc.z); acc.w = fmaf(wk, x[kk].w, acc.w);
                }
            }
        }
        const int r = rh / Hq, h = rh - r * Hq;
        const size_t at = (size_t)bt * p.o_stride_b + ((size_t)u * gm.L + s0 + r) * p.o_stride_row + (size_t)h * p.o_stride_h + d4 * 4;
        if (p.out_bf16) st_stream_bf16x4(reinterpret_cast<__nv_bfloat16*>(p.O) + at, acc);
        else st_stream(reinterpret_cast<float4*>(reinterpret_cast<float*>(p.O) + at), acc);
    }
}

// one warp per (batch, row, head): delta = sum_d dO * O
template <int D>
__global__ void __launch_bounds__(256) delta_kernel(const DeltaParams p)
{
    const Geom& gm = p.gm;
    const long long N = gm.rows_q;
    const long long wid = (long long)blockIdx.x * 8 + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (wid >= (long long)gm.batch * N * gm.heads_q) return;
    const int h = (int)(wid % gm.heads_q);
    const long long row = (wid / gm.heads_q) % N;
    const int bt = (int)(wid / ((long long)gm.heads_q * N));
    const size_t base = (size_t)bt * p.stride_b + (size_t)row * p.stride_row + (size_t)h * p.stride_h;
    const __nv_bfloat16* dO = reinterpret_cast<const __nv_bfloat16*>(p.dO) + base;
    float acc = 0.f;
    if (p.o_bf16) {                              // the forward wrote O as bf16 (plan out_dtype = 1)
        const __nv_bfloat16* O = reinterpret_cast<const __nv_bfloat16*>(p.O) + base;
        constexpr int kPer = D / 32;             // elements per lane
#pragma unroll
        for (int i = 0; i < kPer; i += 2) {
            const __nv_bfloat162 o = *reinterpret_cast<const __nv_bfloat162*>(O + lane * kPer + i);
            const __nv_bfloat162 g = *reinterpret_cast<const __nv_bfloat162*>(dO + lane * kPer + i);
            acc += __low2float(o) * __low2float(g) + __high2float(o) * __high2float(g);
        }
    } else if (D == 128) {
        const float* O = reinterpret_cast<const float*>(p.O) + base;
        const float4 o = *reinterpret_cast<const float4*>(O + lane * 4);
        const uint2 g = *reinterpret_cast<const uint2*>(dO + lane * 4);
        const __nv_bfloat162 g0 = *reinterpret_cast<const __nv_bfloat162*>(&g.x), g1 = *reinterpret_cast<const __nv_bfloat162*>(&g.y);
        acc = o.x * __low2float(g0) + o.y * __high2float(g0) + o.z * __low2float(g1) + o.w * __high2float(g1);
    } else {
        const float* O = reinterpret_cast<const float*>(p.O) + base;
        const float2 o = *reinterpret_cast<const float2*>(O + lane * 2);
        const __nv_bfloat162 g = *reinterpret_cast<const __nv_bfloat162*>(dO + lane * 2);
        acc = o.x * __low2float(g) + o.y * __high2float(g);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) {
        const size_t at = ((size_t)bt * gm.heads_q + h) * N + row;
        const float l = p.lse[at];
        p.ws[at] = acc;
        // exponent offset of the backward's P' = scale * exp(S - lse) = exp2(S*scale*log2e + log2(scale) - lse*log2e); a row
        // without visible keys (lse = -inf) only ever meets masked positions: any finite value does
        p.ws[(size_t)gm.batch * gm.heads_q * N + at] = (l == -INFINITY) ? 0.f : fmaf(-l, 1.4426950408889634f, log2f(gm.scale));
    }
}

// out = sum of m buffers (fp32, float4 granularity), grid-stride, up to 8 independent 16-byte loads in flight per thread
__global__ void __launch_bounds__(256) sum_peers_kernel(const SumParams p)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < p.count4; i += stride) {
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int k0 = 0; k0 < p.m; k0 += kMergeUnroll) {
            float4 x[kMergeUnroll];
#pragma unroll
            for (int kk = 0; kk < kMergeUnroll; ++kk)
                if (k0 + kk < p.m) x[kk] = ld_stream(reinterpret_cast<const float4*>(p.src[k0 + kk]) + i);
#pragma unroll
            for (int kk = 0; kk < kMergeUnroll; ++kk)
                if (k0 + kk < p.m) { acc.x += x[kk].x; acc.y += x[kk].y; acc.z += x[kk].z; acc.w += x[kk].w; }
        }
        st_stream(reinterpret_cast<float4*>(p.out) + i, acc);
    }
}

// dst (bf16) = src (fp32), float4 granularity, grid-stride
__global__ void __launch_bounds__(256) cast_kernel(const float* __restrict__ src, void* dst, long long count4)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count4; i += stride)
        st_stream_bf16x4(reinterpret_cast<uint2*>(dst) + i, ld_stream(reinterpret_cast<const float4*>(src) + i));
}

}  // namespace

int launch_cast_bf16(const float* src, void* dst, long long count, int num_sms, cudaStream_t stream)
{
    const long long count4 = count / 4, blocks = (count4 + 255) / 256;
    const unsigned grid = (unsigned)std::min<long long>(blocks, (long long)num_sms * 16);
    if (grid == 0) return 0;
    cast_kernel<<<grid, 256, 0, stream>>>(src, dst, count4);
    return (int)cudaGetLastError();
}

int launch_sum_peers(const SumParams& p, int num_sms, cudaStream_t stream)
{
    const long long blocks = (p.count4 + 255) / 256;
    const unsigned grid = (unsigned)std::min<long long>(blocks, (long long)num_sms * 8);
    if (grid == 0) return 0;
    sum_peers_kernel<<<grid, 256, 0, stream>>>(p);
    return (int)cudaGetLastError();
}

int launch_merge(const MergeParams& p, cudaStream_t stream)
{
    const Geom& gm = p.gm;
    const size_t smem = (size_t)p.rows_per_block * gm.heads_q * p.m * sizeof(float);
    dim3 grid(gm.L / p.rows_per_block, gm.a, gm.batch);
    cudaError_t e;
    auto go = [&](auto kernel) {
        e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return (int)e;
        kernel<<<grid, kMergeThreads, smem, stream>>>(p);
        return (int)cudaGetLastError();
    };
    if (gm.head_dim == 128) return p.peers ? go(merge_kernel<128, true>) : go(merge_kernel<128, false>);
    return p.peers ? go(merge_kernel<64, true>) : go(merge_kernel<64, false>);
}

int launch_delta(const DeltaParams& p, cudaStream_t stream)
{
    const Geom& gm = p.gm;
    const long long warps = (long long)gm.batch * gm.rows_q * gm.heads_q;
    const unsigned grid = (unsigned)((warps + 7) / 8);
    if (gm.head_dim == 128) delta_kernel<128><<<grid, 256, 0, stream>>>(p);
    else delta_kernel<64><<<grid, 256, 0, stream>>>(p);
    return (int)cudaGetLastError();
}

}  // namespace mesh_attn
