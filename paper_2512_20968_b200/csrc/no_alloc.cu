// no_alloc.cu -- mesh_attn_forward_static (include/mesh_attn.h): the forward pass (tile_fwd -> partial (O, lse) -> merge,
// Alg.2) for callers that cannot allocate device memory -- code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc.  The partial (O, lse) scratch that mesh_attn_forward takes from its caller lives
// here in a file-scope device array of kForwardStaticScratchBytes; every GPU that loads the library holds it until exit.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its address on the current device comes
// from cudaGetSymbolAddress, once per device, and that pointer is what the kernels receive.
#include <atomic>
#include <cstdio>
#include <string>

#include "plan.hpp"

namespace {
constexpr long long kForwardStaticScratchBytes = MESH_ATTN_FORWARD_STATIC_SCRATCH_BYTES;
constexpr int kMaxDevices = 64;

static __device__ __align__(256) unsigned char g_forward_scratch[kForwardStaticScratchBytes];

// device code of this file may name the array directly; the fill below is what tests/test_zz_no_alloc.py uses to poison the scratch
// between calls (mesh_attn_forward_static_poison): a forward that read a stale or unwritten partial would turn NaN
__global__ void poison_scratch_kernel(unsigned int word)
{
    uint4* dst = reinterpret_cast<uint4*>(g_forward_scratch);
    const long long count = kForwardStaticScratchBytes / 16;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (long long)gridDim.x * blockDim.x)
        dst[i] = make_uint4(word, word, word, word);
}

std::atomic<unsigned char*> g_scratch_on_device[kMaxDevices];   // the array's address on each device, looked up once

int fail(int code, const std::string& msg)
{
    mesh_attn::set_error(msg);
    return code;
}

// the array's device address on `dev`, which must be the CURRENT device (cudaGetSymbolAddress answers for the current one)
int scratch_address(int dev, unsigned char** out)
{
    unsigned char* ptr = g_scratch_on_device[dev].load(std::memory_order_acquire);
    if (!ptr) {
        void* sym = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&sym, g_forward_scratch);
        if (e != cudaSuccess || !sym)
            return fail(MESH_ATTN_ECUDA, std::string("forward_static: cudaGetSymbolAddress of the scratch array: ") + cudaGetErrorString(e));
        ptr = static_cast<unsigned char*>(sym);
        g_scratch_on_device[dev].store(ptr, std::memory_order_release);   // two threads racing here store the same value
    }
    *out = ptr;
    return MESH_ATTN_OK;
}

int current_device_of(const mesh_attn_plan* p, const char* who, int* dev)
{
    if (!p) return fail(MESH_ATTN_EINVAL, std::string(who) + ": null plan");
    if (p->device < 0 || !p->d_blob)
        return fail(MESH_ATTN_ECUDA, std::string(who) + ": plan has no device work lists (no sm_100 CUDA device at plan_create); there is no CPU fallback");
    const cudaError_t e = cudaGetDevice(dev);
    if (e != cudaSuccess) return fail(MESH_ATTN_ECUDA, std::string(who) + ": cudaGetDevice: " + cudaGetErrorString(e));
    if (*dev != p->device || *dev >= kMaxDevices) {
        char buf[160];
        std::snprintf(buf, sizeof buf, ": the current device is %d, the plan was created on device %d (make it current; at most %d devices)", *dev,
                      p->device, kMaxDevices);
        return fail(MESH_ATTN_EINVAL, std::string(who) + buf);
    }
    return MESH_ATTN_OK;
}
}  // namespace

// bytes of scratch a forward of this plan needs (partial_O then partial_lse of the `a` simulated GPUs of one Q group)
static int64_t scratch_need(const mesh_attn_plan* p, int64_t* lse_at)
{
    int64_t po = 0, pl = 0;
    mesh_attn_plan_query(p, MESH_ATTN_Q_PARTIAL_O_BYTES, &po);
    mesh_attn_plan_query(p, MESH_ATTN_Q_PARTIAL_LSE_BYTES, &pl);
    const int64_t a = p->geom.a;                                 // one Q group = a simulated GPUs in flight at a time
    *lse_at = (po * a + 255) / 256 * 256;                        // partial_lse follows partial_O on a 256-byte boundary
    return *lse_at + pl * a;
}

extern "C" int mesh_attn_forward_static_limits(const mesh_attn_plan* p, int64_t* need_bytes, int64_t* capacity_bytes)
{
    if (capacity_bytes) *capacity_bytes = kForwardStaticScratchBytes;
    if (need_bytes) {
        if (!p) return fail(MESH_ATTN_EINVAL, "forward_static_limits: need_bytes asked without a plan");
        int64_t lse_at = 0;
        *need_bytes = scratch_need(p, &lse_at);
    }
    return MESH_ATTN_OK;
}

extern "C" int mesh_attn_forward_static(const mesh_attn_plan* p, const void* Q, const void* K, const void* V, void* O, float* lse, void* stream)
{
    int dev = -1;
    if (int rc = current_device_of(p, "forward_static", &dev)) return rc;
    if (!Q || !K || !V || !O || !lse) return fail(MESH_ATTN_EINVAL, "forward_static: null pointer");
    int64_t lse_at = 0;
    const int64_t need = scratch_need(p, &lse_at);
    if (need > kForwardStaticScratchBytes) {
        char buf[256];
        std::snprintf(buf, sizeof buf,
                      "forward_static: this plan needs %lld bytes of partial (O, lse) scratch, the built-in array holds %lld; "
                      "use mesh_attn_forward with caller-owned partial_O / partial_lse",
                      (long long)need, (long long)kForwardStaticScratchBytes);
        return fail(MESH_ATTN_EUNSUPPORTED, buf);
    }
    unsigned char* scratch = nullptr;
    if (int rc = scratch_address(dev, &scratch)) return rc;
    // nothing in the scratch has to start at zero: tile_fwd writes every (slot, row, head) of the partials the merge reads
    // (fully masked pairs included: O = 0, lse = -inf), so the last call's contents are overwritten before they are read
    return mesh_attn_forward(p, Q, K, V, O, lse, reinterpret_cast<float*>(scratch), reinterpret_cast<float*>(scratch + lse_at), stream);
}

extern "C" int mesh_attn_forward_static_poison(const mesh_attn_plan* p, uint32_t word, void* stream)
{
    int dev = -1;
    if (int rc = current_device_of(p, "forward_static_poison", &dev)) return rc;
    poison_scratch_kernel<<<148 * 4, 256, 0, (cudaStream_t)stream>>>(word);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MESH_ATTN_ECUDA, std::string("forward_static_poison launch: ") + cudaGetErrorString(e));
    return MESH_ATTN_OK;
}
