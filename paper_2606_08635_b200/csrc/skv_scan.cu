// skv_scan.cu -- slot prefix sums (SURVEY/DESIGN step a4; not in the paper: the compaction that turns a
// per-token tier map into contiguous per-tier segments).
//
// One CTA per (layer, request).  Counts the FP16 / INT8 / INT4 tokens of every 32-token tile and
// exclusive-scans the counts over the tiles: tile_base[r][l][tile] = (#16, #8, #4 at lower positions).
// Stable compaction: slot of a token = tile_base + number of same-tier tokens before it in its tile.
// The same launch writes the blob metadata (pack: header, tier map, zero pads) or copies the received
// tier map out (unpack).  For sparse blobs (cold-tier upgrades: few shipped tokens, most tiles empty) it also
// emits the compact list of the tiles that carry tokens (tile_base[idx].w, idx < live_count[r][l]), so that the
// pack / patch kernels launch over the live tiles only.
//
// Short sequences (n <= kFuseMaxTokens) do not come here at all: the pack / unpack CTAs count the tiers below
// their own tile themselves (skv_codec.cuh: self_tile_base) and write the metadata, one launch per stage.
#include "skv_common.cuh"

namespace skv {

// counts of 16 / 8 / 4 in a tile, packed 3 x 21 bits into a u64 so one scan serves all three
// (the host rejects n > 2^20, so no field can carry into the next).
__device__ __forceinline__ unsigned long long tile_counts(const uint8_t *tier, int64_t n, int64_t tile, uint32_t low)
{
    const int64_t j0 = tile * kTileTokens;
    uint32_t c16 = 0, c8 = 0, c4 = 0;
    if (j0 + kTileTokens <= n && ((reinterpret_cast<uintptr_t>(tier + j0) & 15) == 0)) {
        const uint4 *p = reinterpret_cast<const uint4 *>(tier + j0);
#pragma unroll
        for (int q = 0; q < kTileTokens / 16; ++q) {
            const uint4 v = p[q];
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k)
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const uint32_t t = (w[k] >> (8 * b)) & 0xFFu;
                    c16 += (t == 16u); c8 += (t == 8u); c4 += (t == low);
                }
        }
    } else {
        for (int i = 0; i < kTileTokens && j0 + i < n; ++i) {
            const uint32_t t = tier[j0 + i];
            c16 += (t == 16u); c8 += (t == 8u); c4 += (t == low);
        }
    }
    return (unsigned long long)c16 | ((unsigned long long)c8 << 21) | ((unsigned long long)c4 << 42);
}

__device__ __forceinline__ unsigned long long warp_incl_scan(unsigned long long x, uint32_t lane)
{
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= (uint32_t)o) x += y;
    }
    return x;
}

template <bool kPack>
__global__ void __launch_bounds__(1024)
tile_scan_kernel(Geom g, Layout lo, const uint8_t *__restrict__ tier_in /* pack: [R][L][n] */,
                 uint8_t *blob /* pack: metadata written; unpack: tier map read */, uint64_t blob_stride,
                 Header256 hdr, uint8_t *__restrict__ tier_out /* unpack: nullable [R][L][n] */,
                 uint4 *__restrict__ tile_base, uint32_t *__restrict__ live_count /* nullable: [R][L], sparse blobs */)
{
    const int l = blockIdx.x, r = blockIdx.y;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    uint8_t *rblob = blob + (uint64_t)r * blob_stride;
    const int64_t n = g.n;
    const uint8_t *tier = kPack ? tier_in + ((int64_t)r * g.L + l) * n
                                : rblob + lo.tier_map_off + (int64_t)l * n;

    __shared__ unsigned long long warp_tot[32];
    __shared__ unsigned long long carry, block_total;
    __shared__ uint32_t warp_live[32];
    __shared__ uint32_t live_carry, live_total;
    if (tid == 0) { carry = 0ull; live_carry = 0u; }
    __syncthreads();

    uint4 *out = tile_base + ((int64_t)r * g.L + l) * g.tiles;
    for (int64_t t0 = 0; t0 < g.tiles; t0 += blockDim.x) {
        const int64_t tile = t0 + tid;
        const unsigned long long c = tile < g.tiles ? tile_counts(tier, n, tile, (uint32_t)g.low_code) : 0ull;
        const unsigned long long x = warp_incl_scan(c, lane);
        const uint32_t live = __ballot_sync(0xffffffffu, c != 0ull);     // tiles of this warp that carry tokens
        if (lane == 31) { warp_tot[warp] = x; warp_live[warp] = (uint32_t)__popc(live); }
        __syncthreads();
        if (warp == 0) {
            const unsigned long long w = warp_tot[lane];
            const unsigned long long s = warp_incl_scan(w, lane);
            warp_tot[lane] = s - w;
            if (lane == 31) block_total = s;
            uint32_t lv = warp_live[lane];
            const uint32_t lw = lv;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t y = __shfl_up_sync(0xffffffffu, lv, o);
                if (lane >= (uint32_t)o) lv += y;
            }
            warp_live[lane] = lv - lw;
            if (lane == 31) live_total = lv;
        }
        __syncthreads();
        const unsigned long long base = carry + warp_tot[warp] + (x - c);
        if (tile < g.tiles) {
            uint4 *o = out + tile;                       // .w belongs to the live list: written below, by another thread
            o->x = (uint32_t)(base & 0x1FFFFFull); o->y = (uint32_t)((base >> 21) & 0x1FFFFFull);
            o->z = (uint32_t)((base >> 42) & 0x1FFFFFull);
            if (live_count != nullptr && c != 0ull)
                out[live_carry + warp_live[warp] + (uint32_t)__popc(live & ((1u << lane) - 1u))].w = (uint32_t)tile;
        }
        __syncthreads();
        if (tid == 0) { carry += block_total; live_carry += live_total; }
        __syncthreads();
    }
    if (live_count != nullptr && tid == 0) live_count[(int64_t)r * g.L + l] = live_carry;

    if (kPack) {
        uint8_t *tm = rblob + lo.tier_map_off + (int64_t)l * n;         // tier map of this layer, verbatim
        for (int64_t j = tid; j < n; j += blockDim.x) tm[j] = tier[j];
        uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
        for (int s = 0; s < 10; ++s) {                                  // zero pads of the ten segments
            const uint64_t beg = lo.seg_off[s] + lo.seg_raw[s];
            const uint64_t end = lo.seg_off[s] + pad256(lo.seg_raw[s]);
            for (uint64_t o = beg + tid; o < end; o += blockDim.x) lbase[o] = 0;
        }
        if (l == 0) {
            if (tid < 64) reinterpret_cast<uint32_t *>(rblob)[tid] = hdr.w[tid];
            const uint64_t beg = lo.tier_map_off + (uint64_t)g.L * (uint64_t)n;
            for (uint64_t o = beg + tid; o < lo.layer0_off; o += blockDim.x) rblob[o] = 0;
        }
    } else if (tier_out != nullptr) {
        uint8_t *tm = tier_out + ((int64_t)r * g.L + l) * n;
        if (g.patch) {                                                   // patch mode: only shipped tokens change tier
            for (int64_t j = tid; j < n; j += blockDim.x) { const uint8_t t = tier[j]; if (t != 0) tm[j] = t; }
        } else {
            for (int64_t j = tid; j < n; j += blockDim.x) tm[j] = tier[j];
        }
    }
}

cudaError_t launch_tile_scan_pack(const Geom &g, const Layout &lo, const uint8_t *tier_map, uint8_t *blob,
                                  uint64_t blob_stride, const Header256 &hdr, uint4 *tile_base, uint32_t *live_count,
                                  cudaStream_t s)
{
    dim3 grid(g.L, g.R);
    tile_scan_kernel<true><<<grid, 1024, 0, s>>>(g, lo, tier_map, blob, blob_stride, hdr, nullptr, tile_base, live_count);
    return cudaGetLastError();
}

cudaError_t launch_tile_scan_unpack(const Geom &g, const Layout &lo, const uint8_t *blob, uint64_t blob_stride,
                                    uint8_t *tier_map_out, uint4 *tile_base, uint32_t *live_count, cudaStream_t s)
{
    dim3 grid(g.L, g.R);
    Header256 hdr = {};
    tile_scan_kernel<false><<<grid, 1024, 0, s>>>(g, lo, nullptr, const_cast<uint8_t *>(blob), blob_stride, hdr,
                                                  tier_map_out, tile_base, live_count);
    return cudaGetLastError();
}

}  // namespace skv
