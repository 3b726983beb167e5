// skv_kvnorm.cu -- the "KV-norm fallback" importance score of Alg. 1 step 2 (reading P15):
//   A[l,j] = mean over KV heads of ||k_{j,g}||_2, normalised to sum 1 per layer;  I[l,j] = A[l,j] exp(-lambda (n-1-j)).
// One bandwidth-bound pass over K (the attention-mass score of Eq. 13 lives in skv_importance_tc.cu).
//
//   kvnorm_fast_kernel  64 tokens per CTA, 8 consecutive tokens per warp, 16-byte streaming loads with the rows of two
//                       tokens in flight per lane; sum of squares per lane in packed fp32 (FFMA2); the lanes of a head
//                       vector are reduced by the transposed group reduction (NCH-1 + log2(LPV/NCH) shuffles for NCH
//                       chunks), the 8 tokens of a warp by a second transposed reduction (9 shuffles for 8 tokens);
//                       writes the raw score of every token and the CTA's partial sum (double, fixed order);
//   kvnorm_kernel       the same result for rows that are not a multiple of 256 elements;
//   kvnorm_finish_kernel  one CTA per 1024 tokens: adds the per-CTA partial sums of its layer in a fixed order
//                       (deterministic), normalises and applies the decay.
#include <algorithm>

#include <cuda_bf16.h>

#include "skv_codec.cuh"

namespace skv {

constexpr int kNormTokens = 64;        // tokens per CTA of the main kernels (= one partial sum)

// sum over the lanes of a head vector of NCH per-lane values, transposed: the first log2(NCH) steps halve the set of
// chunks a lane keeps.  Afterwards the lane holds the head-vector sum of chunk held_chunk<LPV, NCH>(lane).
template <int LPV, int NCH>
__device__ __forceinline__ float group_sum(float (&m)[NCH], uint32_t lane)
{
    float v;
    int o = LPV / 2;
    if (NCH == 4) {
        const bool hi = (lane / (LPV / 2)) & 1;
        const float k0 = (hi ? m[2] : m[0]) + __shfl_xor_sync(0xffffffffu, hi ? m[0] : m[2], LPV / 2);
        const float k1 = (hi ? m[3] : m[1]) + __shfl_xor_sync(0xffffffffu, hi ? m[1] : m[3], LPV / 2);
        const bool hi2 = (lane / (LPV / 4)) & 1;
        v = (hi2 ? k1 : k0) + __shfl_xor_sync(0xffffffffu, hi2 ? k0 : k1, LPV / 4);
        o = LPV / 8;
    } else if (NCH == 2) {
        const bool hi = (lane / (LPV / 2)) & 1;
        v = (hi ? m[1] : m[0]) + __shfl_xor_sync(0xffffffffu, hi ? m[0] : m[1], LPV / 2);
        o = LPV / 4;
    } else {
        v = m[0];
    }
#pragma unroll
    for (; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

template <class E>
__device__ __forceinline__ float sumsq8(const uint4 &v)
{
    using H2 = typename E::H2;
    float2 s = make_float2(0.f, 0.f);
    const float2 a = to_f2(as_pair<H2>(v.x)), b = to_f2(as_pair<H2>(v.y));
    const float2 c = to_f2(as_pair<H2>(v.z)), d = to_f2(as_pair<H2>(v.w));
    s = __ffma2_rn(a, a, s); s = __ffma2_rn(b, b, s); s = __ffma2_rn(c, c, s); s = __ffma2_rn(d, d, s);
    return s.x + s.y;
}

// the CTA's 64 raw scores (in shared memory) -> one double, fixed order
__device__ __forceinline__ void store_partial(const float *sRaw, double *part, uint32_t lane)
{
    double s = (double)sRaw[lane] + (double)sRaw[lane + 32];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) *part = s;
}

template <int D, int NCH, class E>
__global__ void __launch_bounds__(256, 4)
kvnorm_fast_kernel(Geom g, const __half *__restrict__ K, float *__restrict__ raw /*[R][L][n]*/, double *__restrict__ part)
{
    constexpr int LPV = D / 8, HPC = 256 / D;
    constexpr float kRep = (float)NCH / (float)LPV;                    // every (chunk, head) sum sits in LPV/NCH lanes
    __shared__ float sRaw[kNormTokens];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t j0 = (int64_t)blockIdx.x * kNormTokens + warp * 8;
    const int lane_h = (int)(lane * 8) / D, lane_c = (int)(lane * 8) % D;
    const __half *base = K + (int64_t)r * g.sr + (int64_t)l * g.sl + (int64_t)lane_h * g.sh + lane_c;
    const int64_t chunk_stride = (int64_t)HPC * g.sh;
    const float inv_h = 1.0f / (float)g.Hkv;

    float acc[8];
#pragma unroll
    for (int t = 0; t < 8; t += 2) {                                      // two tokens (2 * NCH loads) in flight per lane
        const bool in0 = j0 + t < g.n, in1 = j0 + t + 1 < g.n;            // warp-uniform
        const __half *row0 = base + (j0 + t) * g.st, *row1 = row0 + g.st;
        float a0 = 0.f, a1 = 0.f;
#pragma unroll 1
        for (int cb = 0; cb < g.row_chunks; cb += NCH) {
            uint4 v0[NCH], v1[NCH];
#pragma unroll
            for (int u = 0; u < NCH; ++u) {
                v0[u] = in0 ? ld_stream(row0 + (cb + u) * chunk_stride) : make_uint4(0, 0, 0, 0);
                v1[u] = in1 ? ld_stream(row1 + (cb + u) * chunk_stride) : make_uint4(0, 0, 0, 0);
            }
            float s0[NCH], s1[NCH];
#pragma unroll
            for (int u = 0; u < NCH; ++u) { s0[u] = sumsq8<E>(v0[u]); s1[u] = sumsq8<E>(v1[u]); }
            a0 += sqrtf(group_sum<LPV, NCH>(s0, lane));
            a1 += sqrtf(group_sum<LPV, NCH>(s1, lane));
        }
        acc[t] = a0; acc[t + 1] = a1;
    }
    // sum over the lanes for each of the 8 tokens, transposed: 4 + 2 + 1 + 2 shuffles
    const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
    float q[4], p[2];
#pragma unroll
    for (int i = 0; i < 4; ++i) q[i] = (b4 ? acc[4 + i] : acc[i]) + __shfl_xor_sync(0xffffffffu, b4 ? acc[i] : acc[4 + i], 16);
#pragma unroll
    for (int i = 0; i < 2; ++i) p[i] = (b3 ? q[2 + i] : q[i]) + __shfl_xor_sync(0xffffffffu, b3 ? q[i] : q[2 + i], 8);
    float s = (b2 ? p[1] : p[0]) + __shfl_xor_sync(0xffffffffu, b2 ? p[0] : p[1], 4);
    s += __shfl_xor_sync(0xffffffffu, s, 2);
    s += __shfl_xor_sync(0xffffffffu, s, 1);
    const int tok = (b4 ? 4 : 0) + (b3 ? 2 : 0) + (b2 ? 1 : 0);
    const float score = s * kRep * inv_h;
    if ((lane & 3) == 0) {
        const int64_t j = j0 + tok;
        if (j < g.n) raw[((int64_t)r * g.L + l) * g.n + j] = score;
        sRaw[warp * 8 + tok] = j < g.n ? score : 0.f;
    }
    __syncthreads();
    if (warp == 0) store_partial(sRaw, part + ((int64_t)r * g.L + l) * gridDim.x + blockIdx.x, lane);
}

// generic rows (Hkv*D not a multiple of 256): warp per token, full butterflies
template <class E>
__global__ void __launch_bounds__(256)
kvnorm_kernel(Geom g, const __half *__restrict__ K, float *__restrict__ raw, double *__restrict__ part)
{
    __shared__ float sRaw[kNormTokens];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int lpv = g.D / 8;
    const int row_elems = g.Hkv * g.D;
    for (int it = 0; it < 8; ++it) {
        const int64_t j = (int64_t)blockIdx.x * kNormTokens + warp * 8 + it;
        float acc = 0.f;
        if (j < g.n) {
            const __half *row = K + (int64_t)r * g.sr + (int64_t)l * g.sl + j * g.st;
            for (int e0 = 0; e0 < row_elems; e0 += 256) {
                const int e = e0 + lane * 8;
                uint4 v = make_uint4(0, 0, 0, 0);
                if (e < row_elems) v = ld_stream(row + (int64_t)(e / g.D) * g.sh + e % g.D);
                float ss = sumsq8<E>(v);
                for (int o = 1; o < lpv; o <<= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
                if ((lane % lpv) == 0 && e < row_elems) acc += sqrtf(ss);
            }
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        const float score = acc / (float)g.Hkv;
        if (lane == 0) {
            if (j < g.n) raw[((int64_t)r * g.L + l) * g.n + j] = score;
            sRaw[warp * 8 + it] = j < g.n ? score : 0.f;
        }
    }
    __syncthreads();
    if (warp == 0) store_partial(sRaw, part + ((int64_t)r * g.L + l) * gridDim.x + blockIdx.x, lane);
}

__global__ void __launch_bounds__(1024)
kvnorm_finish_kernel(Geom g, float lambda, int nparts, const float *__restrict__ raw, const double *__restrict__ part,
                     float *__restrict__ importance)
{
    __shared__ double wsum[32];
    __shared__ double total_s;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t rl = (int64_t)r * g.L + l;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    // layer total: the per-CTA partial sums in a fixed order (per-thread strided, then warp and block trees) -- the same
    // value in every CTA of the layer
    double s = 0.0;
    for (int i = tid; i < nparts; i += 1024) s += part[rl * nparts + i];
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) wsum[warp] = s;
    __syncthreads();
    if (warp == 0) {
        double t = wsum[lane];
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
        if (lane == 0) total_s = t;
    }
    __syncthreads();
    const double total = total_s;
    const int j = blockIdx.x * 1024 + (int)tid;
    if (j < g.n) {
        const double a = total > 0.0 ? (double)raw[rl * g.n + j] / total : 1.0 / (double)g.n;
        importance[rl * g.n + j] = (float)(lambda > 0.f ? a * exp(-(double)lambda * (double)(g.n - 1 - j)) : a);
    }
}

// workspace: raw scores f32 [R][L][n] (256-B padded), then the per-CTA partial sums f64 [R][L][ceil(n/64)]
static size_t kvnorm_raw_bytes(const Geom &g) { return ((size_t)g.R * g.L * g.n * sizeof(float) + 255) & ~(size_t)255; }
size_t kvnorm_ws_bytes(const Geom &g)
{
    return kvnorm_raw_bytes(g) + (size_t)g.R * g.L * ((g.n + kNormTokens - 1) / kNormTokens) * sizeof(double);
}

template <int D, class E>
static void launch_kvnorm_d(const Geom &g, const __half *K, float *raw, double *part, dim3 grid, cudaStream_t s)
{
    if ((g.Hkv * D) % 256 == 0) {
        if (g.row_chunks % 4 == 0) kvnorm_fast_kernel<D, 4, E><<<grid, 256, 0, s>>>(g, K, raw, part);
        else if (g.row_chunks % 2 == 0) kvnorm_fast_kernel<D, 2, E><<<grid, 256, 0, s>>>(g, K, raw, part);
        else kvnorm_fast_kernel<D, 1, E><<<grid, 256, 0, s>>>(g, K, raw, part);
    } else {
        kvnorm_kernel<E><<<grid, 256, 0, s>>>(g, K, raw, part);
    }
}

cudaError_t launch_importance_kvnorm(const Geom &g, const __half *K, float lambda, float *importance, void *ws,
                                     cudaStream_t s)
{
    float *raw = reinterpret_cast<float *>(ws);
    double *part = reinterpret_cast<double *>(reinterpret_cast<uint8_t *>(ws) + kvnorm_raw_bytes(g));
    const int nparts = (g.n + kNormTokens - 1) / kNormTokens;
    dim3 g1(nparts, g.L, g.R);
    switch (g.D) {
    case 64:  g.bf16 ? launch_kvnorm_d<64, ElemBF16>(g, K, raw, part, g1, s) : launch_kvnorm_d<64, ElemF16>(g, K, raw, part, g1, s); break;
    case 128: g.bf16 ? launch_kvnorm_d<128, ElemBF16>(g, K, raw, part, g1, s) : launch_kvnorm_d<128, ElemF16>(g, K, raw, part, g1, s); break;
    case 256: g.bf16 ? launch_kvnorm_d<256, ElemBF16>(g, K, raw, part, g1, s) : launch_kvnorm_d<256, ElemF16>(g, K, raw, part, g1, s); break;
    default: return cudaErrorInvalidValue;
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 g2((g.n + 1023) / 1024, g.L, g.R);
    kvnorm_finish_kernel<<<g2, 1024, 0, s>>>(g, lambda, nparts, raw, part, importance);
    return cudaGetLastError();
}

}  // namespace skv
