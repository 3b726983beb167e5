// skv_importance.cu -- per-token importance scores (Alg. 1 step 2; Eq. 13):
//   I[l,j] = A[l,j] * exp(-lambda*(n-1-j)),   A[l,j] = 1/(Hq*w) * sum_{h,i} softmax_j(q_{h,i} . k_j / sqrt(d))
// with the w observation-window queries of every query head (logits as in PAPER.md:109), causal by default.
//
// The attention-mass score runs on the 5th-generation tensor cores: see skv_importance_tc.cu (tcgen05 + TMEM + TMA,
// two passes because the column sums of a row-softmax need every row's normaliser first).  This file holds the
// entry-point dispatch and the KV-norm fallback score of Alg. 1 step 2.
#include <algorithm>

#include <cuda_bf16.h>

#include "skv_common.cuh"

namespace skv {

// ------------------------------------------------------------------------------------------------
// KV-norm fallback: A_j = mean_g ||k_{j,g}||_2, normalised to sum 1 per layer.
// Bandwidth-bound single pass over K plus a per-layer sum.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
kvnorm_kernel(Geom g, const __half *__restrict__ K, float *__restrict__ raw /*[R][L][n]*/)
{
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int lpv = g.D / 8;
    const int hpc = 256 / g.D;                                           // head vectors per 256-element chunk
    const int lane_h = (int)(lane * 8) / g.D, lane_c = (int)(lane * 8) % g.D;   // D is 64, 128 or 256: once per thread
    const int64_t lane_off = (int64_t)lane_h * g.sh + lane_c, chunk_stride = (int64_t)hpc * g.sh;
    // 64 tokens per CTA (8 per warp, interleaved so that the warps of a CTA stream adjacent rows): fat enough that
    // the grid is not CTA-launch-bound
    for (int it = 0; it < 8; ++it) {
    const int64_t j = (int64_t)blockIdx.x * 64 + it * 8 + warp;
    if (j >= g.n) return;
    const __half *row = K + (int64_t)r * g.sr + (int64_t)l * g.sl + j * g.st;
    float acc = 0.f;
    const int row_elems = g.Hkv * g.D;
    for (int e0 = 0; e0 < row_elems; e0 += 1024) {                       // four 16-byte loads in flight per lane
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = e0 + u * 256 + lane * 8;
            v[u] = make_uint4(0, 0, 0, 0);
            if (e < row_elems) {
                const __half *p = row + (int64_t)((e0 >> 8) + u) * chunk_stride + lane_off;
                asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                             : "=r"(v[u].x), "=r"(v[u].y), "=r"(v[u].z), "=r"(v[u].w) : "l"(p));
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = e0 + u * 256 + lane * 8;
            const uint32_t wv[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
            float2 s2 = make_float2(0.f, 0.f);
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const float2 f = g.bf16 ? __bfloat1622float2(*reinterpret_cast<const __nv_bfloat162 *>(&wv[k]))
                                        : __half22float2(*reinterpret_cast<const __half2 *>(&wv[k]));
                s2 = __ffma2_rn(f, f, s2);
            }
            float ss = s2.x + s2.y;
            for (int o = 1; o < lpv; o <<= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
            if ((lane % lpv) == 0 && e < row_elems) acc += sqrtf(ss);
        }
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) raw[((int64_t)r * g.L + l) * g.n + j] = acc / (float)g.Hkv;
    }
}

__global__ void __launch_bounds__(1024)
kvnorm_finish_kernel(Geom g, float lambda, const float *__restrict__ raw, float *__restrict__ importance)
{
    __shared__ double part[32];
    __shared__ double total_s;
    const int64_t off = ((int64_t)blockIdx.y * g.L + blockIdx.x) * g.n;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // fixed-order (deterministic) sum in double: per-thread strided partials, then warp and block trees
    double s = 0.0;
    for (int j = tid; j < g.n; j += blockDim.x) s += (double)raw[off + j];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) part[warp] = s;
    __syncthreads();
    if (warp == 0) {
        double t = part[lane];
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) total_s = t;
    }
    __syncthreads();
    const double total = total_s;
    for (int j = tid; j < g.n; j += blockDim.x) {
        const double a = total > 0.0 ? (double)raw[off + j] / total : 1.0 / (double)g.n;
        importance[off + j] = (float)(a * exp(-(double)lambda * (double)(g.n - 1 - j)));
    }
}

// ------------------------------------------------------------------------------------------------

// ------------------------------------------------------------------------------------------------
// host launchers
// ------------------------------------------------------------------------------------------------
size_t importance_ws_bytes(const Geom &g, int window)
{
    const size_t raw = (size_t)g.R * g.L * g.n * sizeof(float);                // kvnorm raw buffer
    if (window <= 0) return raw;
    const size_t tc = importance_tc_ws_bytes(g, window);
    return tc == 0 ? 0 : std::max(raw, tc);                             // 0: unsupported work decomposition
}

// There is one implementation (tcgen05 / TMEM / TMA); a driver that cannot encode the tensor maps is an error.
cudaError_t launch_importance(const Geom &g, const __half *K, const __half *Q, int window, int causal, float lambda,
                              float *importance, void *ws, size_t, cudaStream_t s)
{
    return launch_importance_tc(g, K, Q, window, causal, lambda, importance, ws, s);
}

cudaError_t launch_importance_kvnorm(const Geom &g, const __half *K, float lambda, float *importance, float *ws,
                                     cudaStream_t s)
{
    dim3 g1((g.n + 63) / 64, g.L, g.R);
    kvnorm_kernel<<<g1, 256, 0, s>>>(g, K, ws);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 g2(g.L, g.R);
    kvnorm_finish_kernel<<<g2, 1024, 0, s>>>(g, lambda, ws, importance);
    return cudaGetLastError();
}

}  // namespace skv
