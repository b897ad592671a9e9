// integrate.cu -- S9: shared-step leapfrog (predictor-corrector of Hut et al.; for one shared constant
// step it is kick - drift - kick, O11/A21).  fp32, one fused multiply-add per component, as the oracle states.
#include "bh_internal.cuh"

namespace bh {

// v = fma(a, h, v); x = fma(v, dt, x)
__global__ void __launch_bounds__(256) k_kick_drift(float4* __restrict__ pos, float4* __restrict__ vel, const float4* __restrict__ acc,
                                                    int n, float h, float dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 a = acc[i];
    float4 v = vel[i];
    float4 p = pos[i];
    v.x = __fmaf_rn(a.x, h, v.x); v.y = __fmaf_rn(a.y, h, v.y); v.z = __fmaf_rn(a.z, h, v.z);
    p.x = __fmaf_rn(v.x, dt, p.x); p.y = __fmaf_rn(v.y, dt, p.y); p.z = __fmaf_rn(v.z, dt, p.z);
    vel[i] = v;
    pos[i] = p;
}

__global__ void __launch_bounds__(256) k_kick(float4* __restrict__ vel, const float4* __restrict__ acc, int n, float h) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float4 a = acc[i];
    float4 v = vel[i];
    v.x = __fmaf_rn(a.x, h, v.x); v.y = __fmaf_rn(a.y, h, v.y); v.z = __fmaf_rn(a.z, h, v.z);
    vel[i] = v;
}

int stage_kick_drift(bh_ctx* c, float h, float dt, cudaStream_t s) {
    const int n = (int)c->n;
    BH_LAUNCH(c, k_kick_drift, (unsigned)div_up(n, 256), 256, 0, s, c->ws.pos[c->cur], c->ws.vel[c->cur], c->ws.acc, n, h, dt);
    return BH_OK;
}

int stage_kick(bh_ctx* c, float h, cudaStream_t s) {
    const int n = (int)c->n;
    BH_LAUNCH(c, k_kick, (unsigned)div_up(n, 256), 256, 0, s, c->ws.vel[c->cur], c->ws.acc, n, h);
    return BH_OK;
}

}  // namespace bh
