// skv_assign.cu -- budgeted tier assignment (Alg. 1 step 3; Prop. 1, PAPER.md:101;
// "Sink positions are pinned before ranking").
//
// One CTA per (layer, request).  The layer's n scores are turned into 32-bit ranking keys held in shared
// memory (global workspace when n*4 exceeds the shared-memory budget): protected positions get the
// sentinel 0xFFFFFFFF (they outrank everything, so the top-n16 set contains them), every other token the
// bits of its non-negative f32 score (NaN / negative / -0 -> 0), which order like the floats.
// Three order statistics (ranks n16, n16+n8, n16+n8+n4) are found together by ONE MSB-first 8-bit radix select of
// four digit passes (thresholds that still share a key prefix share a histogram);
// ties at a threshold are admitted in ascending position (a block scan of the "== threshold" flags),
// which makes the result the unique stable ranking the oracle's sort produces.
#include "skv_common.cuh"

namespace skv {

constexpr int kAssignThreads = 1024;

struct Thresh { uint32_t key; uint32_t n_gt; uint32_t pass_all; uint32_t rank; };

__device__ __forceinline__ uint32_t sanitize_key(float x)
{
    return (x > 0.0f) ? __float_as_uint(x) : 0u;        // NaN compares false -> 0; -0, negatives -> 0
}

// The three order statistics (ranks kth[0] <= kth[1] <= kth[2], 1-based "K-th largest") of keys[0..n) in ONE sweep of
// four MSB-first 8-bit digits.  At a given digit position the candidate sets of the thresholds are defined by their key
// prefixes, which are pairwise equal or disjoint, so every key falls into at most one of (at most three) histograms;
// thresholds that still share a prefix share a histogram.  act[k] = 0 marks a threshold that needs no selection (rank
// 0 or >= n).  Returns, per active threshold, the key of rank kth[k] and the number of strictly greater keys.
__device__ void radix_select3(const uint32_t *keys, int n, const uint32_t (&kth)[3], const bool (&act)[3],
                              uint32_t (*hist)[256] /*[3][256]*/, uint32_t *bcast /*[6]*/, uint32_t (&key_out)[3], uint32_t (&ngt_out)[3])
{
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint32_t prefix[3] = {0, 0, 0}, remaining[3] = {kth[0], kth[1], kth[2]}, mask = 0;
    for (int shift = 24; shift >= 0; shift -= 8) {
        if (tid < 768) (&hist[0][0])[tid] = 0;
        __syncthreads();
        for (int j0 = 0; j0 < n; j0 += blockDim.x) {
            const int j = j0 + tid;
            uint32_t code = 0x400u;                                  // "no histogram"
            if (j < n) {
                const uint32_t key = keys[j], pk = key & mask;
                const int grp = (act[0] && pk == prefix[0]) ? 0 : (act[1] && pk == prefix[1]) ? 1 : (act[2] && pk == prefix[2]) ? 2 : -1;
                if (grp >= 0) code = ((uint32_t)grp << 8) | ((key >> shift) & 0xFFu);
            }
            // warp-aggregated histogram update: one atomic per distinct (histogram, digit) per warp
            const uint32_t peers = __match_any_sync(0xffffffffu, code);
            if (code != 0x400u && lane == (uint32_t)(__ffs(peers) - 1)) atomicAdd(&hist[code >> 8][code & 0xFFu], __popc(peers));
        }
        __syncthreads();
        // (registers, not indexable arrays: select with the warp-uniform k)
        const int k = (int)warp;
        const bool act_k = k == 0 ? act[0] : k == 1 ? act[1] : k == 2 ? act[2] : false;
        if (act_k) {
            const uint32_t prefix_k = k == 0 ? prefix[0] : k == 1 ? prefix[1] : prefix[2];
            const uint32_t rem_k = k == 0 ? remaining[0] : k == 1 ? remaining[1] : remaining[2];
            // the histogram of threshold k is the one of the first active threshold with the same prefix
            const int src = (act[0] && prefix[0] == prefix_k) ? 0 : (act[1] && prefix[1] == prefix_k) ? 1 : k;
            // lane i owns bins [8i, 8i+8); suffix sums from the top digit down
            uint32_t loc[8], sum = 0;
#pragma unroll
            for (int b = 0; b < 8; ++b) { loc[b] = hist[src][lane * 8 + b]; sum += loc[b]; }
            uint32_t incl = sum;                          // inclusive suffix sum over lanes >= this lane
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_down_sync(0xffffffffu, incl, o);
                if (lane + o < 32) incl += y;
            }
            const uint32_t above = incl - sum;            // keys in bins owned by higher lanes
            if (above < rem_k && rem_k <= incl) {
                uint32_t acc = above;
                int b = 7;
#pragma unroll
                for (int bb = 7; bb >= 0; --bb) {         // highest bin whose suffix count reaches the rank
                    if (b == bb) { if (acc + loc[bb] >= rem_k) break; acc += loc[bb]; b = bb - 1; }
                }
                bcast[2 * k] = lane * 8 + b;              // the digit of the K-th largest
                bcast[2 * k + 1] = rem_k - acc;           // its rank inside that bin
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 3; ++k)
            if (act[k]) { prefix[k] |= bcast[2 * k] << shift; remaining[k] = bcast[2 * k + 1]; }
        mask |= 0xFFu << shift;
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) { key_out[k] = prefix[k]; ngt_out[k] = kth[k] - remaining[k]; }
}

__global__ void __launch_bounds__(kAssignThreads)
assign_kernel(Geom g, Intervals prot, const float *__restrict__ importance, uint8_t *__restrict__ tier_map,
              uint32_t *__restrict__ key_ws, int keys_in_smem)
{
    extern __shared__ uint32_t smem[];
    __shared__ uint32_t hist[3][256];
    __shared__ uint32_t bcast[6];
    __shared__ uint32_t warp_tot[3][32];
    __shared__ Thresh th[3];

    const int l = blockIdx.x, r = blockIdx.y, n = g.n;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t off = ((int64_t)r * g.L + l) * n;
    uint32_t *keys = keys_in_smem ? smem : key_ws + off;

    for (int j = tid; j < n; j += blockDim.x) {
        bool p = false;
        for (int q = 0; q < prot.count; ++q) p |= (j >= prot.lo[q] && j < prot.hi[q]);
        keys[j] = p ? 0xFFFFFFFFu : sanitize_key(importance[off + j]);
    }
    __syncthreads();

    const uint32_t K[3] = {(uint32_t)g.n16, (uint32_t)(g.n16 + g.n8), (uint32_t)(g.n16 + g.n8 + g.n4)};
    const bool act[3] = {K[0] > 0 && K[0] < (uint32_t)n, K[1] > 0 && K[1] < (uint32_t)n, K[2] > 0 && K[2] < (uint32_t)n};
    uint32_t skey[3] = {0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu}, sngt[3] = {0, 0, 0};
    if (act[0] || act[1] || act[2]) radix_select3(keys, n, K, act, hist, bcast, skey, sngt);
    if (tid < 3) {
        const int k = (int)tid;
        // K >= n: every token passes this level; K = 0: nobody does (key 0xFFFFFFFF, rank test below fails)
        th[k].key = act[k] ? skey[k] : 0xFFFFFFFFu; th[k].n_gt = act[k] ? sngt[k] : 0u;
        th[k].pass_all = K[k] >= (uint32_t)n ? 1u : 0u; th[k].rank = K[k];
    }
    __syncthreads();

    // position-ordered rank among equals: thread t owns the contiguous chunk [t*c, (t+1)*c)
    // (an ODD chunk length keeps the 32 lanes of a warp on 32 different shared-memory banks)
    const int c = ((n + blockDim.x - 1) / blockDim.x) | 1;
    const int beg = min(n, (int)tid * c), end = min(n, beg + c);
    uint32_t eq[3] = {0, 0, 0};
    for (int j = beg; j < end; ++j) {
        const uint32_t key = keys[j];
#pragma unroll
        for (int k = 0; k < 3; ++k) eq[k] += (key == th[k].key);
    }
    uint32_t excl[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        uint32_t x = eq[k];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= (uint32_t)o) x += y;
        }
        if (lane == 31) warp_tot[k][warp] = x;
        excl[k] = x - eq[k];
    }
    __syncthreads();
    if (warp < 3) {
        const uint32_t w = warp_tot[warp][lane];
        uint32_t s = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
            if (lane >= (uint32_t)o) s += y;
        }
        warp_tot[warp][lane] = s - w;
    }
    __syncthreads();
    uint32_t run[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) run[k] = excl[k] + warp_tot[k][warp];

    uint8_t *out = tier_map + off;
    for (int j = beg; j < end; ++j) {
        const uint32_t key = keys[j];
        uint32_t tier = 0;
        bool done = false;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            bool pass;
            if (th[k].pass_all) pass = true;
            else if (key > th[k].key) pass = true;                       // rank < n_gt < K
            else if (key == th[k].key) pass = (th[k].n_gt + run[k]) < th[k].rank;
            else pass = false;
            if (key == th[k].key) run[k] += 1;
            if (pass && !done) { tier = (k == 0) ? 16u : (k == 1) ? 8u : (uint32_t)g.low_code; done = true; }
        }
        out[j] = (uint8_t)tier;
    }
}

cudaError_t launch_assign(const Geom &g, const Intervals &prot, const float *importance, uint8_t *tier_map,
                          uint32_t *key_ws, cudaStream_t s)
{
    const size_t need = (size_t)g.n * 4;
    const int in_smem = need <= 200 * 1024;
    const size_t dyn = in_smem ? need : 0;
    if (dyn > 48 * 1024) {
        // the attribute is per function and process-wide: always request the SAME maximum, so that concurrent callers
        // with different n cannot lower each other's limit between the attribute call and the launch
        cudaError_t e = cudaFuncSetAttribute(assign_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
        if (e != cudaSuccess) return e;
    }
    dim3 grid(g.L, g.R);
    assign_kernel<<<grid, kAssignThreads, dyn, s>>>(g, prot, importance, tier_map, key_ws, in_smem);
    return cudaGetLastError();
}

}  // namespace skv
