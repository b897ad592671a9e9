// direct.cu -- the accuracy reference of PAPER.md:196-200 (Eq.2): softened O(N^2) direct summation in binary64.
// The paper measures the tree code's acceleration error against "a double precision version of Sapporo" (a GPU direct
// N-body code); this is that reference written for sm_100a: one target per thread, sources staged through shared memory
// in tiles, every operation in fp64 from the fp32 inputs (O10, p-p part: phi -= m / rho, a += m dr / rho^3,
// rho^2 = |dr|^2 + eps^2, j != i by index).  It is not on the per-step path.
#include "bh_internal.cuh"

namespace bh {

constexpr int kDirectThreads = 128;

__global__ void __launch_bounds__(kDirectThreads) k_direct(const float4* __restrict__ pos, int64_t n, double eps2, int64_t t0, int64_t t1,
                                                           double* __restrict__ out) {
    __shared__ float4 tile[kDirectThreads];
    const int64_t i = t0 + (int64_t)blockIdx.x * kDirectThreads + threadIdx.x;
    const bool live = i < t1;
    const float4 pi = pos[live ? i : t0];
    const double xi = (double)pi.x, yi = (double)pi.y, zi = (double)pi.z;
    double ax = 0.0, ay = 0.0, az = 0.0, phi = 0.0;
    for (int64_t j0 = 0; j0 < n; j0 += kDirectThreads) {
        const int64_t jl = j0 + threadIdx.x;
        __syncthreads();
        tile[threadIdx.x] = jl < n ? pos[jl] : make_float4(0.f, 0.f, 0.f, 0.f);
        __syncthreads();
        const int cnt = (int)min((int64_t)kDirectThreads, n - j0);
#pragma unroll 4
        for (int k = 0; k < cnt; ++k) {
            const float4 pj = tile[k];
            const double dx = (double)pj.x - xi, dy = (double)pj.y - yi, dz = (double)pj.z - zi;
            const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
            double ri = rsqrt(r2);
            if (j0 + k == i) ri = 0.0;                 // j != i (A19); rsqrt(0) = inf when eps = 0
            const double m = (double)pj.w;
            const double mri = m * ri;
            const double f = mri * ri * ri;
            phi -= mri;
            ax = fma(f, dx, ax);
            ay = fma(f, dy, ay);
            az = fma(f, dz, az);
        }
    }
    if (live) {
        double* o = out + 4 * i;
        o[0] = ax; o[1] = ay; o[2] = az; o[3] = phi;
    }
}

}  // namespace bh

using namespace bh;

extern "C" int bh_direct_forces(const float* d_pos_mass, int64_t n, float eps, int64_t t0, int64_t t1, double* d_acc_pot, void* stream) {
    if (!d_pos_mass || !d_acc_pot || n < 1 || t0 < 0 || t1 > n || t0 >= t1 || !(eps >= 0.0f)) return BH_ERR_INVALID_ARG;
    cudaPointerAttributes a0, a1;
    if (cudaPointerGetAttributes(&a0, d_pos_mass) != cudaSuccess || cudaPointerGetAttributes(&a1, d_acc_pot) != cudaSuccess ||
        a0.type != cudaMemoryTypeDevice || a1.type != cudaMemoryTypeDevice || a0.device != a1.device) {
        (void)cudaGetLastError();
        return BH_ERR_INVALID_ARG;
    }
    if (cudaSetDevice(a0.device) != cudaSuccess) return BH_ERR_CUDA;
    const int64_t blocks = (t1 - t0 + kDirectThreads - 1) / kDirectThreads;
    if (blocks > 0x7FFFFFFF) return BH_ERR_INVALID_ARG;
    k_direct<<<(unsigned)blocks, kDirectThreads, 0, static_cast<cudaStream_t>(stream)>>>(reinterpret_cast<const float4*>(d_pos_mass), n,
                                                                                        (double)eps * (double)eps, t0, t1, d_acc_pot);
    return cudaPeekAtLastError() == cudaSuccess ? BH_OK : BH_ERR_CUDA;
}
