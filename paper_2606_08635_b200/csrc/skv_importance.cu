// skv_importance.cu -- per-token importance scores (Alg. 1 step 2; Eq. 13):
//   I[l,j] = A[l,j] * exp(-lambda*(n-1-j)),   A[l,j] = 1/(Hq*w) * sum_{h,i} softmax_j(q_{h,i} . k_j / sqrt(d))
// with the w observation-window queries of every query head (logits as in PAPER.md:109), causal by default.
//
// The column sums of a row-softmax need every row's normaliser before any column can be finished, so the
// contraction runs twice (storing the w*Hq x n logits would cost more HBM than recomputing them):
//   pass 1  rowstats : S = Q_g K_g^T on tensor cores (queries = MMA rows), online max / sum-of-exp per query
//                      row over a chunk of keys -> partial (m, z) per (row, chunk)
//   combine          : lse2[row] = log2(sum_j 2^(s_j)) from the partials
//   pass 2  colsum   : S^T = K_g Q_g^T on tensor cores (keys = MMA rows), p = 2^(s - lse2[row]), summed over
//                      the query rows inside each thread and over the KV heads in a fixed order (deterministic;
//                      no atomics), scaled by 1/(Hq*w) and the recency decay.
// fp16 operands, fp32 accumulation (mma.sync.m16n8k16), operands staged in XOR-swizzled shared memory by
// cp.async and fetched with ldmatrix.
#include <stdlib.h>

#include <algorithm>

#include "skv_common.cuh"

namespace skv {

constexpr float kNegBig = -1.0e30f;
constexpr int kP1Keys = 64;          // keys per pass-1 tile
constexpr int kP1Warps = 8;          // 16 query rows per warp -> 128-row block
constexpr int kP2Warps = 8;          // 16 keys per warp -> 128-key tile
constexpr int kP2Keys = 16 * kP2Warps;
constexpr int kP2MaxRows = 256;      // query rows of one KV head held in shared memory at a time

__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, bool valid)
{
    const int sz = valid ? 16 : 0;    // src-size 0 => 16 bytes of zeros
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" :: "r"(dst), "l"(src), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(N) : "memory"); }
__device__ __forceinline__ void ldmatrix_x4(uint32_t addr, uint32_t &r0, uint32_t &r1, uint32_t &r2, uint32_t &r3)
{
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3) : "r"(addr));
}
__device__ __forceinline__ void mma16816(float c[4], const uint32_t a[4], uint32_t b0, uint32_t b1)
{
    asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
                 : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// Shared-memory tile of `rows` x D halves, 16-byte chunks XOR-swizzled with the row index (conflict-free ldmatrix).
template <int D>
__device__ __forceinline__ uint32_t tile_addr(uint32_t base, int row, int chunk)
{
    return base + (uint32_t)row * (D * 2) + (uint32_t)((chunk ^ (row & 7)) << 4);
}

// ------------------------------------------------------------------------------------------------
// pass 1: per query row, (max, sum of 2^(s-max)) over a chunk of keys
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kP1Warps * 32)
imp_rowstats_kernel(Geom g, const __half *__restrict__ K, const __half *__restrict__ Q, int w, int causal,
                    int chunk_keys, int n_chunks, int row_blocks, float2 *__restrict__ partial)
{
    extern __shared__ __align__(128) uint8_t smem_raw[];
    constexpr int KS = D / 16;                           // k-steps
    constexpr int TILE_BYTES = kP1Keys * D * 2;
    const uint32_t sbase = smem_u32(smem_raw);

    const int chunk = blockIdx.x / row_blocks, rb = blockIdx.x % row_blocks;
    const int gh = blockIdx.y;                           // KV head
    const int l = blockIdx.z % g.L, r = blockIdx.z / g.L;
    const int G = g.Hq / g.Hkv, M = G * w;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int n = g.n;
    const float sc = 1.4426950408889634f * rsqrtf((float)D);   // log2(e)/sqrt(d): logits in the log2 domain

    // A fragments: this warp's 16 query rows x D, straight from global (read once)
    const int row0 = rb * (16 * kP1Warps) + warp * 16;
    const __half *Qg = Q + ((((int64_t)r * g.L + l) * g.Hq + (int64_t)gh * G) * w) * D;   // [M][D]
    uint32_t a[KS][4];
    {
        const int ra = row0 + (lane >> 2), rbw = ra + 8;
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
            const int c = ks * 16 + (lane & 3) * 2;
            a[ks][0] = ra < M ? *reinterpret_cast<const uint32_t *>(Qg + (int64_t)ra * D + c) : 0u;
            a[ks][1] = rbw < M ? *reinterpret_cast<const uint32_t *>(Qg + (int64_t)rbw * D + c) : 0u;
            a[ks][2] = ra < M ? *reinterpret_cast<const uint32_t *>(Qg + (int64_t)ra * D + c + 8) : 0u;
            a[ks][3] = rbw < M ? *reinterpret_cast<const uint32_t *>(Qg + (int64_t)rbw * D + c + 8) : 0u;
        }
    }
    // causal limit of the two rows this thread owns: row = hl*w + i  ->  pos = n - w + i
    const int rowA = row0 + (lane >> 2), rowB = rowA + 8;
    const int limA = causal ? (n - w + (rowA % w)) : (n - 1);
    const int limB = causal ? (n - w + (rowB % w)) : (n - 1);

    const int key_beg = chunk * chunk_keys;
    const int key_end = min(n, key_beg + chunk_keys);
    const int n_tiles = (key_end - key_beg + kP1Keys - 1) / kP1Keys;
    const __half *Kg = K + (int64_t)r * g.sr + (int64_t)l * g.sl + (int64_t)gh * g.sh;

    auto load_tile = [&](int t, int stage) {
        const int k0 = key_beg + t * kP1Keys;
        constexpr int CH = D / 8;                        // 16-byte chunks per key row
        for (int idx = tid; idx < kP1Keys * CH; idx += kP1Warps * 32) {
            const int row = idx / CH, cc = idx % CH;
            const int key = k0 + row;
            const bool ok = key < key_end;
            cp_async16(tile_addr<D>(sbase + stage * TILE_BYTES, row, cc), Kg + (int64_t)(ok ? key : 0) * g.st + cc * 8, ok);
        }
    };

    float mA = kNegBig, mB = kNegBig, zA = 0.f, zB = 0.f;
    if (n_tiles > 0) { load_tile(0, 0); }
    cp_async_commit();
    for (int t = 0; t < n_tiles; ++t) {
        if (t + 1 < n_tiles) load_tile(t + 1, (t + 1) & 1);
        cp_async_commit();
        cp_async_wait<1>();
        __syncthreads();
        const uint32_t tb = sbase + (t & 1) * TILE_BYTES;
        float s[kP1Keys / 8][4];
#pragma unroll
        for (int nt = 0; nt < kP1Keys / 8; ++nt) {
            s[nt][0] = s[nt][1] = s[nt][2] = s[nt][3] = 0.f;
#pragma unroll
            for (int ks = 0; ks < KS; ks += 2) {
                uint32_t b0, b1, b2, b3;
                ldmatrix_x4(tile_addr<D>(tb, nt * 8 + (lane & 7), ks * 2 + (lane >> 3)), b0, b1, b2, b3);
                mma16816(s[nt], a[ks], b0, b1);
                mma16816(s[nt], a[ks + 1], b2, b3);
            }
        }
        // online softmax bookkeeping in the log2 domain; this thread: cols nt*8 + 2*(lane&3) + {0,1}
        const int k0 = key_beg + t * kP1Keys + (lane & 3) * 2;
        float tmA = kNegBig, tmB = kNegBig;
#pragma unroll
        for (int nt = 0; nt < kP1Keys / 8; ++nt) {
            const int j = k0 + nt * 8;
            s[nt][0] = (j <= limA && j < key_end) ? s[nt][0] * sc : kNegBig;
            s[nt][1] = (j + 1 <= limA && j + 1 < key_end) ? s[nt][1] * sc : kNegBig;
            s[nt][2] = (j <= limB && j < key_end) ? s[nt][2] * sc : kNegBig;
            s[nt][3] = (j + 1 <= limB && j + 1 < key_end) ? s[nt][3] * sc : kNegBig;
            tmA = fmaxf(tmA, fmaxf(s[nt][0], s[nt][1]));
            tmB = fmaxf(tmB, fmaxf(s[nt][2], s[nt][3]));
        }
        const float nmA = fmaxf(mA, tmA), nmB = fmaxf(mB, tmB);
        zA *= ex2(mA - nmA); zB *= ex2(mB - nmB);
        mA = nmA; mB = nmB;
#pragma unroll
        for (int nt = 0; nt < kP1Keys / 8; ++nt) {
            zA += (s[nt][0] > 0.5f * kNegBig ? ex2(s[nt][0] - mA) : 0.f) + (s[nt][1] > 0.5f * kNegBig ? ex2(s[nt][1] - mA) : 0.f);
            zB += (s[nt][2] > 0.5f * kNegBig ? ex2(s[nt][2] - mB) : 0.f) + (s[nt][3] > 0.5f * kNegBig ? ex2(s[nt][3] - mB) : 0.f);
        }
        __syncthreads();                                  // tile consumed before its buffer is refilled
    }
    cp_async_wait<0>();
    // reduce over the 4 lanes that share a row
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
        const float omA = __shfl_xor_sync(0xffffffffu, mA, o), ozA = __shfl_xor_sync(0xffffffffu, zA, o);
        const float omB = __shfl_xor_sync(0xffffffffu, mB, o), ozB = __shfl_xor_sync(0xffffffffu, zB, o);
        const float nA = fmaxf(mA, omA), nB = fmaxf(mB, omB);
        zA = zA * ex2(mA - nA) + ozA * ex2(omA - nA); mA = nA;
        zB = zB * ex2(mB - nB) + ozB * ex2(omB - nB); mB = nB;
    }
    if ((lane & 3) == 0) {
        // partial[r][l][global row][chunk], global row = gh*M + row
        float2 *p = partial + ((((int64_t)r * g.L + l) * g.Hq * w) + (int64_t)gh * M) * n_chunks;
        if (rowA < M) p[(int64_t)rowA * n_chunks + chunk] = make_float2(mA, zA);
        if (rowB < M) p[(int64_t)rowB * n_chunks + chunk] = make_float2(mB, zB);
    }
}

// ------------------------------------------------------------------------------------------------
// combine: lse2[row] = M + log2(sum_c z_c 2^(m_c - M))
// ------------------------------------------------------------------------------------------------
__global__ void imp_combine_kernel(const float2 *__restrict__ partial, int n_chunks, int64_t rows, float *__restrict__ lse2)
{
    const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= rows) return;
    const float2 *p = partial + row * n_chunks;
    float m = kNegBig;
    for (int c = 0; c < n_chunks; ++c) m = fmaxf(m, p[c].x);
    float z = 0.f;
    for (int c = 0; c < n_chunks; ++c) z += p[c].y * exp2f(p[c].x - m);
    lse2[row] = m + log2f(z);
}

// ------------------------------------------------------------------------------------------------
// pass 2: column sums of the normalised probabilities, all KV heads, one 128-key tile per CTA
// ------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kP2Warps * 32)
imp_colsum_kernel(Geom g, const __half *__restrict__ K, const __half *__restrict__ Q, int w, int causal, float lambda,
                  const float *__restrict__ lse2, float *__restrict__ importance)
{
    extern __shared__ __align__(128) uint8_t smem_raw[];
    constexpr int KS = D / 16;
    constexpr int CH = D / 8;
    constexpr int KTILE_BYTES = kP2Keys * D * 2;
    const uint32_t sK = smem_u32(smem_raw);
    const uint32_t sQ = sK + KTILE_BYTES;
    float *sLse = reinterpret_cast<float *>(smem_raw + KTILE_BYTES + kP2MaxRows * D * 2);

    const int l = blockIdx.y, r = blockIdx.z;
    const int n = g.n, G = g.Hq / g.Hkv, M = G * w;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int key0 = blockIdx.x * kP2Keys;
    const float sc = 1.4426950408889634f * rsqrtf((float)D);

    const int jA = key0 + warp * 16 + (lane >> 2), jB = jA + 8;      // the two keys (MMA rows) of this thread
    float sumA = 0.f, sumB = 0.f;

    for (int gh = 0; gh < g.Hkv; ++gh) {
        const __half *Kg = K + (int64_t)r * g.sr + (int64_t)l * g.sl + (int64_t)gh * g.sh;
        const __half *Qg = Q + ((((int64_t)r * g.L + l) * g.Hq + (int64_t)gh * G) * w) * D;
        const float *lse_g = lse2 + (((int64_t)r * g.L + l) * g.Hq * w) + (int64_t)gh * M;
        for (int m0 = 0; m0 < M; m0 += kP2MaxRows) {
            const int mrows = min(kP2MaxRows, M - m0);
            const int mpad = (mrows + 7) & ~7;
            __syncthreads();                                          // previous contents fully consumed
            if (m0 == 0) {
                for (int idx = tid; idx < kP2Keys * CH; idx += kP2Warps * 32) {
                    const int row = idx / CH, cc = idx % CH;
                    const int key = key0 + row;
                    const bool ok = key < n;
                    cp_async16(tile_addr<D>(sK, row, cc), Kg + (int64_t)(ok ? key : 0) * g.st + cc * 8, ok);
                }
            }
            for (int idx = tid; idx < mpad * CH; idx += kP2Warps * 32) {
                const int row = idx / CH, cc = idx % CH;
                const bool ok = row < mrows;
                cp_async16(tile_addr<D>(sQ, row, cc), Qg + (int64_t)(m0 + (ok ? row : 0)) * D + cc * 8, ok);
            }
            cp_async_commit();
            for (int idx = tid; idx < mpad; idx += kP2Warps * 32) sLse[idx] = idx < mrows ? lse_g[m0 + idx] : 0.f;
            cp_async_wait<0>();
            __syncthreads();

            uint32_t a[KS][4];                                         // this warp's 16 keys x D
#pragma unroll
            for (int ks = 0; ks < KS; ++ks)
                ldmatrix_x4(tile_addr<D>(sK, warp * 16 + (lane & 15), ks * 2 + (lane >> 4)), a[ks][0], a[ks][1], a[ks][2], a[ks][3]);

            for (int nt = 0; nt < mpad / 8; ++nt) {
                float c[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
                for (int ks = 0; ks < KS; ks += 2) {
                    uint32_t b0, b1, b2, b3;
                    ldmatrix_x4(tile_addr<D>(sQ, nt * 8 + (lane & 7), ks * 2 + (lane >> 3)), b0, b1, b2, b3);
                    mma16816(c, a[ks], b0, b1);
                    mma16816(c, a[ks + 1], b2, b3);
                }
                const int q0 = nt * 8 + (lane & 3) * 2, q1 = q0 + 1;  // query rows (MMA columns) of this thread
                const float l0 = sLse[q0], l1 = sLse[q1];
                const int lim0 = causal ? (n - w + ((m0 + q0) % w)) : (n - 1);
                const int lim1 = causal ? (n - w + ((m0 + q1) % w)) : (n - 1);
                const bool v0 = q0 < mrows, v1 = q1 < mrows;
                sumA += (v0 && jA <= lim0 ? ex2(c[0] * sc - l0) : 0.f) + (v1 && jA <= lim1 ? ex2(c[1] * sc - l1) : 0.f);
                sumB += (v0 && jB <= lim0 ? ex2(c[2] * sc - l0) : 0.f) + (v1 && jB <= lim1 ? ex2(c[3] * sc - l1) : 0.f);
            }
        }
    }
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
        sumA += __shfl_xor_sync(0xffffffffu, sumA, o);
        sumB += __shfl_xor_sync(0xffffffffu, sumB, o);
    }
    if ((lane & 3) == 0) {
        const float norm = 1.0f / ((float)g.Hq * (float)w);
        float *out = importance + ((int64_t)r * g.L + l) * n;
        if (jA < n) out[jA] = sumA * norm * expf(-lambda * (float)(n - 1 - jA));
        if (jB < n) out[jB] = sumB * norm * expf(-lambda * (float)(n - 1 - jB));
    }
}

// ------------------------------------------------------------------------------------------------
// KV-norm fallback: A_j = mean_g ||k_{j,g}||_2, normalised to sum 1 per layer.
// Bandwidth-bound single pass over K plus a per-layer sum.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
kvnorm_kernel(Geom g, const __half *__restrict__ K, float *__restrict__ raw /*[R][L][n]*/)
{
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t j = (int64_t)blockIdx.x * 8 + warp;
    if (j >= g.n) return;
    const __half *row = K + (int64_t)r * g.sr + (int64_t)l * g.sl + j * g.st;
    const int lpv = g.D / 8;
    float acc = 0.f;
    for (int e0 = 0; e0 < g.Hkv * g.D; e0 += 256) {
        const int e = e0 + lane * 8;
        float ss = 0.f;
        if (e < g.Hkv * g.D) {
            const uint4 v = *reinterpret_cast<const uint4 *>(row + (int64_t)(e / g.D) * g.sh + (e % g.D));
            const __half2 *h = reinterpret_cast<const __half2 *>(&v);
#pragma unroll
            for (int k = 0; k < 4; ++k) { const float2 f = __half22float2(h[k]); ss += f.x * f.x + f.y * f.y; }
        }
        for (int o = 1; o < lpv; o <<= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
        if ((lane % lpv) == 0 && e < g.Hkv * g.D) acc += sqrtf(ss);
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if (lane == 0) raw[((int64_t)r * g.L + l) * g.n + j] = acc / (float)g.Hkv;
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
// host launchers
// ------------------------------------------------------------------------------------------------
static void p1_chunking(const Geom &g, int &chunk_keys, int &n_chunks)
{
    int ck = (g.n + 15) / 16;
    ck = ((ck + kP1Keys - 1) / kP1Keys) * kP1Keys;
    if (ck < 1024) ck = 1024;
    chunk_keys = ck;
    n_chunks = (g.n + ck - 1) / ck;
}

size_t importance_ws_bytes(const Geom &g, int window)
{
    if (window <= 0) return (size_t)g.R * g.L * g.n * sizeof(float);          // kvnorm raw buffer
    int ck, nc;
    p1_chunking(g, ck, nc);
    const size_t rows = (size_t)g.R * g.L * g.Hq * window;
    const size_t a = rows * nc * sizeof(float2) + rows * sizeof(float) + 256;
    const size_t b = (size_t)g.R * g.L * g.n * sizeof(float);
    const size_t c = importance_tc_ws_bytes(g, window);
    return std::max(a, std::max(b, c));
}

template <int D>
static cudaError_t launch_importance_t(const Geom &g, const __half *K, const __half *Q, int w, int causal, float lambda,
                                       float *importance, void *ws, cudaStream_t s)
{
    int ck, nc;
    p1_chunking(g, ck, nc);
    const int G = g.Hq / g.Hkv, M = G * w;
    const int row_blocks = (M + 16 * kP1Warps - 1) / (16 * kP1Warps);
    const int64_t rows = (int64_t)g.R * g.L * g.Hq * w;
    float2 *partial = reinterpret_cast<float2 *>(ws);
    float *lse2 = reinterpret_cast<float *>(reinterpret_cast<uint8_t *>(ws) + (((size_t)rows * nc * sizeof(float2) + 255) & ~(size_t)255));

    const int smem1 = 2 * kP1Keys * D * 2;
    cudaError_t e = cudaFuncSetAttribute(imp_rowstats_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem1);
    if (e != cudaSuccess) return e;
    dim3 g1(nc * row_blocks, g.Hkv, g.L * g.R);
    imp_rowstats_kernel<D><<<g1, kP1Warps * 32, smem1, s>>>(g, K, Q, w, causal, ck, nc, row_blocks, partial);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;

    imp_combine_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, s>>>(partial, nc, rows, lse2);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;

    const int smem2 = kP2Keys * D * 2 + kP2MaxRows * D * 2 + kP2MaxRows * 4;
    e = cudaFuncSetAttribute(imp_colsum_kernel<D>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem2);
    if (e != cudaSuccess) return e;
    dim3 g2((g.n + kP2Keys - 1) / kP2Keys, g.L, g.R);
    imp_colsum_kernel<D><<<g2, kP2Warps * 32, smem2, s>>>(g, K, Q, w, causal, lambda, lse2, importance);
    return cudaGetLastError();
}

cudaError_t launch_importance(const Geom &g, const __half *K, const __half *Q, int window, int causal, float lambda,
                              float *importance, void *ws, size_t, cudaStream_t s)
{
    // tcgen05 / TMEM / TMA path (skv_importance_tc.cu).  The mma.sync kernels below remain as the fallback for
    // drivers that cannot build the tensor maps, and for A/B comparison (SKV_IMPORTANCE=mma).
    const char *sel = getenv("SKV_IMPORTANCE");
    if (!(sel && sel[0] == 'm')) {
        const cudaError_t e = launch_importance_tc(g, K, Q, window, causal, lambda, importance, ws, s);
        if (e != cudaErrorNotSupported) return e;
    }
    switch (g.D) {
    case 64:  return launch_importance_t<64>(g, K, Q, window, causal, lambda, importance, ws, s);
    case 128: return launch_importance_t<128>(g, K, Q, window, causal, lambda, importance, ws, s);
    case 256: return launch_importance_t<256>(g, K, Q, window, causal, lambda, importance, ws, s);
    default: return cudaErrorInvalidValue;
    }
}

cudaError_t launch_importance_kvnorm(const Geom &g, const __half *K, float lambda, float *importance, float *ws,
                                     cudaStream_t s)
{
    dim3 g1((g.n + 7) / 8, g.L, g.R);
    kvnorm_kernel<<<g1, 256, 0, s>>>(g, K, ws);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 g2(g.L, g.R);
    kvnorm_finish_kernel<<<g2, 1024, 0, s>>>(g, lambda, ws, importance);
    return cudaGetLastError();
}

}  // namespace skv
