// domain_static.cu -- bh_domain_box_static: S0 (domain box + input validation) for callers that cannot
// give the library any device memory beyond the input and the 32-byte result.
//
// Who that is.  Every other stage of this library keeps its intermediates in a workspace the caller allocates
// (bh_workspace_bytes / bh_create).  Some callers have no way to produce one: a plug-in running inside a host program
// whose own allocator has already taken the whole card, a process held to a fixed device-memory budget (an MPS client
// with a memory limit, a job that shares the GPU) where a cudaMalloc in the middle of a run may simply fail, and a
// time-step loop that cannot afford cudaMalloc / cudaFree because both synchronise the whole device and stall every other
// stream.  Such a caller often still needs the first thing a tree build needs -- the bounding cube of its particles and
// the answer to "is this input valid?" -- for example to choose a key grid or to decide whether particles left its domain.
//
// How.  The reduction is the one k_bbox (keys_sort.cu) does, but its intermediates (one partial box per block and an
// arrival counter) live in a file-scope `static __device__` array below instead of the workspace.  The array is part of the
// library image: every GPU on which the library's kernels get loaded holds its 256 KiB until the process exits, whether or
// not this entry point is ever called there.  That fixed size is where the limit BH_DOMAIN_STATIC_MAX_N comes from.
//
// The array is shared by all calls on a device and keeps whatever the previous call left in it.  Only the arrival counter
// has to start at zero; every call clears it with a cudaMemsetAsync on the caller's stream ahead of the kernel (the
// partial boxes are overwritten before they are read).  Two calls whose work overlaps on the same GPU (different streams,
// or different host threads) use the same counter and the same partials and corrupt each other: callers serialise them.
#include <mutex>

#include "bh_internal.cuh"

namespace bh {

constexpr int kBoxThreads = 256;
constexpr int kBoxPerThread = 16;
constexpr int kBoxTile = kBoxThreads * kBoxPerThread;              // 4096 particles per block, no grid stride
constexpr int kBoxMaxBlocks = BH_DOMAIN_STATIC_MAX_N / kBoxTile;   // 8192
constexpr int kBoxHeaderWords = 64;                                // [0]: blocks that have stored their partial; rest unused
constexpr int kBoxPartialWords = 8;                                // min xyz, max xyz (order-preserving encodings), bad flag, unused
constexpr size_t kBoxScratchWords = (size_t)kBoxHeaderWords + (size_t)kBoxPartialWords * kBoxMaxBlocks;
static_assert(BH_DOMAIN_STATIC_MAX_N % kBoxTile == 0, "the limit is a whole number of tiles");

// The scratch.  In host code this name is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) uint32_t g_domain_scratch[kBoxScratchWords];

__device__ __forceinline__ uint32_t box_f2ord(float f) {
    const uint32_t u = __float_as_uint(f);
    return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}
__device__ __forceinline__ float box_ord2f(uint32_t u) {
    return __uint_as_float((u & 0x80000000u) ? (u & 0x7FFFFFFFu) : ~u);
}

// Block b reduces particles [b * 4096, (b + 1) * 4096) to one partial box in scratch; the block that arrives last folds the
// partials, derives the cube side as k_domain does (2^e with frexpf(extent) = (mu, e)) and writes the result.
__global__ void __launch_bounds__(kBoxThreads) k_bbox_static(const float4* __restrict__ pos, int n, uint32_t* __restrict__ scratch,
                                                             bh_domain_box* __restrict__ out) {
    float mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
    int bad = 0;
    const int base = blockIdx.x * kBoxTile + threadIdx.x;
#pragma unroll
    for (int r0 = 0; r0 < kBoxPerThread; r0 += 4) {
        float4 q[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) q[u] = pos[min(base + (r0 + u) * kBoxThreads, n - 1)];   // a repeated last particle changes nothing
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const float4 p = q[u];
            bad |= !(isfinite(p.x) && isfinite(p.y) && isfinite(p.z) && isfinite(p.w) && p.w > 0.0f);   // A27
            mn[0] = fminf(mn[0], p.x); mx[0] = fmaxf(mx[0], p.x);
            mn[1] = fminf(mn[1], p.y); mx[1] = fmaxf(mx[1], p.y);
            mn[2] = fminf(mn[2], p.z); mx[2] = fmaxf(mx[2], p.z);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            mn[k] = fminf(mn[k], __shfl_xor_sync(0xFFFFFFFFu, mn[k], o));
            mx[k] = fmaxf(mx[k], __shfl_xor_sync(0xFFFFFFFFu, mx[k], o));
        }
        bad |= __shfl_xor_sync(0xFFFFFFFFu, bad, o);
    }
    constexpr int kWarps = kBoxThreads / 32;
    __shared__ uint32_t s_mn[kWarps][3], s_mx[kWarps][3], s_bad[kWarps];
    __shared__ bool s_last;
    const int w = threadIdx.x >> 5;
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { s_mn[w][k] = box_f2ord(mn[k]); s_mx[w][k] = box_f2ord(mx[k]); }
        s_bad[w] = (uint32_t)bad;
    }
    __syncthreads();
    uint32_t* part = scratch + kBoxHeaderWords;
    if (threadIdx.x == 0) {
        uint32_t a[3], b[3], any = 0u;
#pragma unroll
        for (int k = 0; k < 3; ++k) { a[k] = 0xFFFFFFFFu; b[k] = 0u; }
#pragma unroll
        for (int ww = 0; ww < kWarps; ++ww) {
#pragma unroll
            for (int k = 0; k < 3; ++k) { a[k] = min(a[k], s_mn[ww][k]); b[k] = max(b[k], s_mx[ww][k]); }
            any |= s_bad[ww];
        }
        uint32_t* mine = part + (size_t)kBoxPartialWords * blockIdx.x;
#pragma unroll
        for (int k = 0; k < 3; ++k) { mine[k] = a[k]; mine[3 + k] = b[k]; }
        mine[6] = any;
        __threadfence();                                            // the partial is visible before the arrival is
        s_last = atomicAdd(&scratch[0], 1u) == gridDim.x - 1u;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    uint32_t a[3] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu}, b[3] = {0u, 0u, 0u}, any = 0u;
    for (int j = threadIdx.x; j < (int)gridDim.x; j += kBoxThreads) {
        const uint32_t* p = part + (size_t)kBoxPartialWords * j;
#pragma unroll
        for (int k = 0; k < 3; ++k) { a[k] = min(a[k], __ldcg(p + k)); b[k] = max(b[k], __ldcg(p + 3 + k)); }
        any |= __ldcg(p + 6);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            a[k] = min(a[k], __shfl_xor_sync(0xFFFFFFFFu, a[k], o));
            b[k] = max(b[k], __shfl_xor_sync(0xFFFFFFFFu, b[k], o));
        }
        any |= __shfl_xor_sync(0xFFFFFFFFu, any, o);
    }
    __syncthreads();                                                // (s_mn .. s_bad are read no more by thread 0 above)
    if ((threadIdx.x & 31) == 0) {
#pragma unroll
        for (int k = 0; k < 3; ++k) { s_mn[w][k] = a[k]; s_mx[w][k] = b[k]; }
        s_bad[w] = any;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    any = 0u;
    float ext = 0.0f;
    for (int k = 0; k < 3; ++k) {
        uint32_t lo_o = 0xFFFFFFFFu, hi_o = 0u;
        for (int ww = 0; ww < kWarps; ++ww) { lo_o = min(lo_o, s_mn[ww][k]); hi_o = max(hi_o, s_mx[ww][k]); }
        const float lo = box_ord2f(lo_o), hi = box_ord2f(hi_o);
        out->lo[k] = lo;
        out->hi[k] = hi;
        ext = fmaxf(ext, __fsub_rn(hi, lo));
    }
    for (int ww = 0; ww < kWarps; ++ww) any |= s_bad[ww];
    if (!isfinite(ext)) { any = 1u; ext = 1.0f; }
    if (ext == 0.0f) ext = 1.0f;
    int e = 0;
    (void)frexpf(ext, &e);
    out->domain_exp = e;
    out->status = any ? (int32_t)BH_ERR_NONFINITE : (int32_t)BH_OK;
}

// Device address of g_domain_scratch on device `dev`, which must be the current device.  Looked up once per device.
constexpr int kBoxMaxDevices = 64;
static std::mutex g_box_mutex;
static uint32_t* g_box_ptr[kBoxMaxDevices];

static int domain_scratch(int dev, uint32_t** out) {
    if (dev < 0 || dev >= kBoxMaxDevices) return BH_ERR_INVALID_ARG;
    std::lock_guard<std::mutex> hold(g_box_mutex);
    if (!g_box_ptr[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_domain_scratch);
        if (e != cudaSuccess || !p) {
            (void)cudaGetLastError();
            return BH_ERR_CUDA;
        }
        g_box_ptr[dev] = static_cast<uint32_t*>(p);
    }
    *out = g_box_ptr[dev];
    return BH_OK;
}

}  // namespace bh

using namespace bh;

extern "C" int64_t bh_domain_box_static_max_n(void) { return (int64_t)BH_DOMAIN_STATIC_MAX_N; }

extern "C" int bh_domain_box_static(const float* d_pos_mass, int64_t n, bh_domain_box* d_out, void* stream) {
    if (!d_pos_mass || !d_out || n < 1) return BH_ERR_INVALID_ARG;
    if (n > (int64_t)BH_DOMAIN_STATIC_MAX_N) return BH_ERR_TOO_LARGE;      // the static scratch has no room for more partials
    cudaPointerAttributes a0, a1;
    if (cudaPointerGetAttributes(&a0, d_pos_mass) != cudaSuccess || cudaPointerGetAttributes(&a1, d_out) != cudaSuccess ||
        a0.type != cudaMemoryTypeDevice || a1.type != cudaMemoryTypeDevice || a0.device != a1.device) {
        (void)cudaGetLastError();
        return BH_ERR_INVALID_ARG;
    }
    int prev = -1;
    if (cudaGetDevice(&prev) != cudaSuccess) return BH_ERR_CUDA;
    if (prev != a0.device && cudaSetDevice(a0.device) != cudaSuccess) return BH_ERR_CUDA;
    int rc = BH_OK;
    uint32_t* scratch = nullptr;
    rc = domain_scratch(a0.device, &scratch);
    if (rc == BH_OK) {
        const cudaStream_t s = static_cast<cudaStream_t>(stream);
        const unsigned blocks = (unsigned)((n + kBoxTile - 1) / kBoxTile);
        if (cudaMemsetAsync(scratch, 0, kBoxHeaderWords * sizeof(uint32_t), s) != cudaSuccess) rc = BH_ERR_CUDA;
        if (rc == BH_OK) {
            k_bbox_static<<<blocks, kBoxThreads, 0, s>>>(reinterpret_cast<const float4*>(d_pos_mass), (int)n, scratch, d_out);
            if (cudaPeekAtLastError() != cudaSuccess) rc = BH_ERR_CUDA;
        }
    }
    if (prev != a0.device) (void)cudaSetDevice(prev);
    return rc;
}
