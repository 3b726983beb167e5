// skv_unpack.cu -- unpack-and-dequantize (decode side, "only lightweight dequantization
// (table lookup) is needed at the decode worker").
//
// Mirror of skv_pack.cu: one warp per token, one CTA per 32-token tile of one (request, layer).  The slot
// of a token is recomputed from the transmitted tier map (tile base + ballot rank; the tile base comes from
// skv_scan.cu, or for n <= kFuseMaxTokens from the CTA's own count of the tier-map bytes below its tile, so
// that unpack is one launch; skv_unpack_patch of a sparse upgrade blob walks the scan's list of live tiles).
// INT8: 8-byte loads per lane -> 8 fp16 (one 16-byte store); INT4: 4-byte loads -> 8 fp16.  y = f16_rn(
// fl32(float(q) * fl32(amax/qmax))); int->float goes through the 2^23 exponent trick (exact), so no I2F.
// Dropped tokens are written as +0.0 (reading P10).  HBM-bound: reads beta*Bytes_FP16, writes Bytes_FP16.
#include "skv_codec.cuh"

namespace skv {

// Fused launch (TileSrc::tile_base == nullptr): the tier map the scan kernel would have copied out (the validity mask);
// in patch mode only the tokens the blob carries change tier.
__device__ __forceinline__ void unpack_metadata(const Geom &g, uint8_t *tier_out, int64_t rl, int64_t j0, uint32_t my_t)
{
    const uint32_t tid = threadIdx.x;
    if (tier_out != nullptr && tid < 32 && j0 + tid < g.n && !(g.patch && my_t == 0u))
        tier_out[rl * g.n + j0 + tid] = (uint8_t)my_t;
}

template <int D, class E, bool SPARSE>
__global__ void __launch_bounds__(256)
unpack_kernel(Geom g, Layout lo, const uint8_t *__restrict__ blob, uint64_t blob_stride,
              __half *__restrict__ K, __half *__restrict__ V, uint8_t *__restrict__ tier_out, TileSrc ts)
{
    using H = typename E::H; using H2 = typename E::H2;
    __shared__ uint32_t sCnt[16];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t n = g.n, rl = (int64_t)r * g.L + l;
    const uint8_t *rblob = blob + (uint64_t)r * blob_stride;
    const uint8_t *tm = rblob + lo.tier_map_off + (int64_t)l * n;
    const uint32_t low = (uint32_t)g.low_code;                       // 4: symmetric INT4, 2: asymmetric 2-bit (NEXT-4)
    const uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
    const int row_elems = g.Hkv * D;
    const int64_t cache_off = (int64_t)r * g.sr + (int64_t)l * g.sl;
    const uint32_t limit = SPARSE ? ts.live_count[rl] : (uint32_t)g.tiles;
    uint32_t idx = blockIdx.x;
    if (SPARSE && idx >= limit) return;

#pragma unroll 1
    do {
    const int64_t tile = SPARSE ? (int64_t)ts.tile_base[rl * g.tiles + idx].w : (int64_t)idx;
    const int64_t j0 = tile * kTileTokens;
    const uint32_t my_t = (j0 + lane < n) ? (uint32_t)tm[j0 + lane] : 0xFFu;
    const uint32_t m16 = __ballot_sync(0xffffffffu, my_t == 16u);
    const uint32_t m8 = __ballot_sync(0xffffffffu, my_t == 8u);
    const uint32_t m4 = __ballot_sync(0xffffffffu, my_t == low);
    uint4 base;
    if (ts.tile_base) base = ts.tile_base[rl * g.tiles + tile];
    else { base = self_tile_base(tm, tile, low, sCnt); unpack_metadata(g, tier_out, rl, j0, my_t); }

    for (uint32_t i = warp; i < (uint32_t)kTileTokens; i += nwarps) {
        const int64_t j = j0 + i;
        if (j >= n) break;
        uint32_t t = __shfl_sync(0xffffffffu, my_t, i);
        const uint32_t below = (1u << i) - 1u;
        __half *krow = K + cache_off + j * g.st;
        __half *vrow = V + cache_off + j * g.st;
        uint32_t slot = 0;
        if (t == 16u) { slot = base.x + __popc(m16 & below); if (slot >= (uint32_t)g.n16) t = 0; }
        else if (t == 8u) { slot = base.y + __popc(m8 & below); if (slot >= (uint32_t)g.n8) t = 0; }
        else if (t == low) { slot = base.z + __popc(m4 & below); if (slot >= (uint32_t)g.n4) t = 0; }
        else t = 0;
        if (t == 0u && g.patch) continue;                             // patch mode (skv_unpack_patch): keep what is there

        if (t == 16u) {
            const uint8_t *ks = lbase + lo.seg_off[0] + (uint64_t)slot * row_elems * 2;
            const uint8_t *vs = lbase + lo.seg_off[1] + (uint64_t)slot * row_elems * 2;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint4 kv[4], vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) { kv[u] = ld_stream(ks + e * 2); vv[u] = ld_stream(vs + e * 2); }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        st_stream(krow + (int64_t)h * g.sh + c, kv[u]);
                        st_stream(vrow + (int64_t)h * g.sh + c, vv[u]);
                    }
                }
            }
        } else if (t == 8u) {
            const uint8_t *ks = lbase + lo.seg_off[2] + (uint64_t)slot * row_elems;
            const uint8_t *vs = lbase + lo.seg_off[3] + (uint64_t)slot * row_elems;
            const H *ka = reinterpret_cast<const H *>(lbase + lo.seg_off[6]) + (uint64_t)slot * g.Hkv;
            const H *va = reinterpret_cast<const H *>(lbase + lo.seg_off[7]) + (uint64_t)slot * g.Hkv;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint2 kv[4], vv[4]; H ak[4], av[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        kv[u] = ld_stream8(ks + e); vv[u] = ld_stream8(vs + e);
                        ak[u] = ka[e / D]; av[u] = va[e / D];
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        st_stream(krow + (int64_t)h * g.sh + c, dequant_int8<E>(kv[u], scale_of(ak[u], 127.0f)));
                        st_stream(vrow + (int64_t)h * g.sh + c, dequant_int8<E>(vv[u], scale_of(av[u], 127.0f)));
                    }
                }
            }
        } else if (t == 2u) {
            const uint8_t *ks = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 4);
            const uint8_t *vs = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 4);
            const int recs = g.low_group ? row_elems / g.low_group : g.Hkv;          // (lo, hi) records per token row
            const H2 *ka = reinterpret_cast<const H2 *>(lbase + lo.seg_off[8]) + (uint64_t)slot * recs;
            const H2 *va = reinterpret_cast<const H2 *>(lbase + lo.seg_off[9]) + (uint64_t)slot * recs;
            for (int c0 = 0; c0 < g.row_chunks; ++c0) {
                const int e = c0 * 256 + lane * 8;
                if (e < row_elems) {
                    const int h = e / D, c = e % D;
                    const int rec = g.low_group ? e / g.low_group : h;             // per head vector, or per 32 elements (P22)
                    const H2 rk = ka[rec], rv = va[rec];            // (lo, hi) records
                    const uint32_t kw = ld_stream2(ks + e / 4), vw = ld_stream2(vs + e / 4);
                    st_stream(krow + (int64_t)h * g.sh + c,
                              dequant_int2<E>(kw, step3_of(range_of(lo_h(rk), hi_h(rk))), to_f(lo_h(rk))));
                    st_stream(vrow + (int64_t)h * g.sh + c,
                              dequant_int2<E>(vw, step3_of(range_of(lo_h(rv), hi_h(rv))), to_f(lo_h(rv))));
                }
            }
        } else if (t == 4u) {
            const uint8_t *ks = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 2);
            const uint8_t *vs = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 2);
            const H *ka = reinterpret_cast<const H *>(lbase + lo.seg_off[8]) + (uint64_t)slot * g.Hkv;
            const H *va = reinterpret_cast<const H *>(lbase + lo.seg_off[9]) + (uint64_t)slot * g.Hkv;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint32_t kv[4], vv[4]; H ak[4], av[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        kv[u] = ld_stream4(ks + e / 2); vv[u] = ld_stream4(vs + e / 2);
                        ak[u] = ka[e / D]; av[u] = va[e / D];
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        st_stream(krow + (int64_t)h * g.sh + c, dequant_int4<E>(kv[u], scale_of(ak[u], 7.0f)));
                        st_stream(vrow + (int64_t)h * g.sh + c, dequant_int4<E>(vv[u], scale_of(av[u], 7.0f)));
                    }
                }
            }
        } else {
            const uint4 z = make_uint4(0, 0, 0, 0);
            for (int c0 = 0; c0 < g.row_chunks; ++c0) {
                const int e = c0 * 256 + lane * 8;
                if (e < row_elems) {
                    const int h = e / D, c = e % D;
                    st_stream(krow + (int64_t)h * g.sh + c, z);
                    st_stream(vrow + (int64_t)h * g.sh + c, z);
                }
            }
        }
    }
    idx += gridDim.x;
    } while (SPARSE && idx < limit);
}

// ------------------------------------------------------------------------------------------------
// Fast path (row_elems % (256*NCH) == 0): fully unrolled; each lane loads the amax record of ONE
// (chunk, head) for K and V, divides twice, and the scales are broadcast with 2*NCH shuffles.
// ------------------------------------------------------------------------------------------------
// SPARSE: the grid strides over the scan's list of live tiles (patch mode only); otherwise one CTA per tile, no loop.
template <int D, int NCH, int MINB, bool LOW2, class E, bool SPARSE>
__global__ void __launch_bounds__(256, MINB)
unpack_fast_kernel(Geom g, Layout lo, const uint8_t *__restrict__ blob, uint64_t blob_stride,
                   __half *__restrict__ K, __half *__restrict__ V, uint8_t *__restrict__ tier_out, TileSrc ts)
{
    using H = typename E::H; using H2 = typename E::H2;
    constexpr int LPV = D / 8;
    constexpr int HPC = 256 / D;
    constexpr uint32_t kLow = LOW2 ? 2u : 4u;
    __shared__ uint32_t sCnt[16];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t n = g.n, rl = (int64_t)r * g.L + l;
    const uint8_t *rblob = blob + (uint64_t)r * blob_stride;
    const uint8_t *tm = rblob + lo.tier_map_off + (int64_t)l * n;
    const uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
    const int row_elems = g.Hkv * D;
    __half *Kb = K + (int64_t)r * g.sr + (int64_t)l * g.sl;
    __half *Vb = V + (int64_t)r * g.sr + (int64_t)l * g.sl;
    const int lane_h = (int)(lane * 8) / D, lane_c = (int)(lane * 8) % D;
    const int my_chunk = held_chunk<LPV, NCH>(lane);
    const uint32_t limit = SPARSE ? ts.live_count[rl] : (uint32_t)g.tiles;
    uint32_t idx = blockIdx.x;
    if (SPARSE && idx >= limit) return;

#pragma unroll 1
    do {
    const int64_t tile = SPARSE ? (int64_t)ts.tile_base[rl * g.tiles + idx].w : (int64_t)idx;
    const int64_t j0 = tile * kTileTokens;
    const uint32_t my_t = (j0 + lane < n) ? (uint32_t)tm[j0 + lane] : 0xFFu;
    const uint32_t m16 = __ballot_sync(0xffffffffu, my_t == 16u);
    const uint32_t m8 = __ballot_sync(0xffffffffu, my_t == 8u);
    const uint32_t m4 = __ballot_sync(0xffffffffu, my_t == kLow);
    uint4 base;
    if (ts.tile_base) base = ts.tile_base[rl * g.tiles + tile];
    else { base = self_tile_base(tm, tile, kLow, sCnt); unpack_metadata(g, tier_out, rl, j0, my_t); }

    for (uint32_t i = warp; i < (uint32_t)kTileTokens; i += 8) {
        const int64_t j = j0 + i;
        if (j >= n) break;
        uint32_t t = __shfl_sync(0xffffffffu, my_t, i);
        const uint32_t below = (1u << i) - 1u;
        __half *krow = Kb + j * g.st + lane_c;
        __half *vrow = Vb + j * g.st + lane_c;
        uint32_t slot = 0;
        if (t == 16u) { slot = base.x + __popc(m16 & below); if (slot >= (uint32_t)g.n16) t = 0; }
        else if (t == 8u) { slot = base.y + __popc(m8 & below); if (slot >= (uint32_t)g.n8) t = 0; }
        else if (t == kLow) { slot = base.z + __popc(m4 & below); if (slot >= (uint32_t)g.n4) t = 0; }
        else t = 0;
        if (t == 0u && g.patch) continue;                             // patch mode (skv_unpack_patch): keep what is there

#pragma unroll 1
        for (int cb = 0; cb < g.row_chunks; cb += NCH) {
            if (t == 16u) {
                const uint8_t *ks = lbase + lo.seg_off[0] + ((uint64_t)slot * row_elems + cb * 256 + lane * 8) * 2;
                const uint8_t *vs = lbase + lo.seg_off[1] + ((uint64_t)slot * row_elems + cb * 256 + lane * 8) * 2;
                uint4 kv[NCH], vv[NCH];
#pragma unroll
                for (int u = 0; u < NCH; ++u) { kv[u] = ld_stream(ks + u * 512); vv[u] = ld_stream(vs + u * 512); }
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                    st_stream(krow + off, kv[u]); st_stream(vrow + off, vv[u]);
                }
            } else if (t == 8u) {
                const uint8_t *ks = lbase + lo.seg_off[2] + (uint64_t)slot * row_elems + cb * 256 + lane * 8;
                const uint8_t *vs = lbase + lo.seg_off[3] + (uint64_t)slot * row_elems + cb * 256 + lane * 8;
                const int head = (cb + my_chunk) * HPC + (int)(lane / LPV);
                uint2 kv[NCH], vv[NCH];
#pragma unroll
                for (int u = 0; u < NCH; ++u) { kv[u] = ld_stream8(ks + u * 256); vv[u] = ld_stream8(vs + u * 256); }
                const H ak = reinterpret_cast<const H *>(lbase + lo.seg_off[6])[(uint64_t)slot * g.Hkv + head];
                const H av = reinterpret_cast<const H *>(lbase + lo.seg_off[7])[(uint64_t)slot * g.Hkv + head];
                const float sK = scale_of(ak, 127.0f), sV = scale_of(av, 127.0f);
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int src = src_lane<LPV, NCH>(lane, u);
                    const float sk = __shfl_sync(0xffffffffu, sK, src), sv = __shfl_sync(0xffffffffu, sV, src);
                    const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                    st_stream(krow + off, dequant_int8<E>(kv[u], sk));
                    st_stream(vrow + off, dequant_int8<E>(vv[u], sv));
                }
            } else if (LOW2 && t == 2u && g.low_group) {
                // group-wise 2-bit (reading P22): the four lanes of a 32-element group read the same (lo, hi) record
                const uint8_t *ks = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                const uint8_t *vs = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                const H2 *ka = reinterpret_cast<const H2 *>(lbase + lo.seg_off[8]) + (uint64_t)slot * (row_elems / 32) + cb * 8 + lane / 4;
                const H2 *va = reinterpret_cast<const H2 *>(lbase + lo.seg_off[9]) + (uint64_t)slot * (row_elems / 32) + cb * 8 + lane / 4;
                uint32_t kv[NCH], vv[NCH]; H2 rk[NCH], rv[NCH];
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    kv[u] = ld_stream2(ks + u * 64); vv[u] = ld_stream2(vs + u * 64);
                    rk[u] = ka[u * 8]; rv[u] = va[u * 8];
                }
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                    st_stream(krow + off, dequant_int2<E>(kv[u], step3_of(range_of(lo_h(rk[u]), hi_h(rk[u]))), to_f(lo_h(rk[u]))));
                    st_stream(vrow + off, dequant_int2<E>(vv[u], step3_of(range_of(lo_h(rv[u]), hi_h(rv[u]))), to_f(lo_h(rv[u]))));
                }
            } else if (LOW2 && t == 2u) {
                const uint8_t *ks = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                const uint8_t *vs = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                const int head = (cb + my_chunk) * HPC + (int)(lane / LPV);
                uint32_t kv[NCH], vv[NCH];
#pragma unroll
                for (int u = 0; u < NCH; ++u) { kv[u] = ld_stream2(ks + u * 64); vv[u] = ld_stream2(vs + u * 64); }
                const H2 rk = reinterpret_cast<const H2 *>(lbase + lo.seg_off[8])[(uint64_t)slot * g.Hkv + head];
                const H2 rv = reinterpret_cast<const H2 *>(lbase + lo.seg_off[9])[(uint64_t)slot * g.Hkv + head];
                const float sK = step3_of(range_of(lo_h(rk), hi_h(rk))), lK = to_f(lo_h(rk));
                const float sV = step3_of(range_of(lo_h(rv), hi_h(rv))), lV = to_f(lo_h(rv));
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int src = src_lane<LPV, NCH>(lane, u);
                    const float sk = __shfl_sync(0xffffffffu, sK, src), sv = __shfl_sync(0xffffffffu, sV, src);
                    const float lk = __shfl_sync(0xffffffffu, lK, src), lv = __shfl_sync(0xffffffffu, lV, src);
                    const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                    st_stream(krow + off, dequant_int2<E>(kv[u], sk, lk));
                    st_stream(vrow + off, dequant_int2<E>(vv[u], sv, lv));
                }
            } else if (!LOW2 && t == 4u) {
                const uint8_t *ks = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 2) + cb * 128 + lane * 4;
                const uint8_t *vs = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 2) + cb * 128 + lane * 4;
                const int head = (cb + my_chunk) * HPC + (int)(lane / LPV);
                uint32_t kv[NCH], vv[NCH];
#pragma unroll
                for (int u = 0; u < NCH; ++u) { kv[u] = ld_stream4(ks + u * 128); vv[u] = ld_stream4(vs + u * 128); }
                const H ak = reinterpret_cast<const H *>(lbase + lo.seg_off[8])[(uint64_t)slot * g.Hkv + head];
                const H av = reinterpret_cast<const H *>(lbase + lo.seg_off[9])[(uint64_t)slot * g.Hkv + head];
                const float sK = scale_of(ak, 7.0f), sV = scale_of(av, 7.0f);
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int src = src_lane<LPV, NCH>(lane, u);
                    const float sk = __shfl_sync(0xffffffffu, sK, src), sv = __shfl_sync(0xffffffffu, sV, src);
                    const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                    st_stream(krow + off, dequant_int4<E>(kv[u], sk));
                    st_stream(vrow + off, dequant_int4<E>(vv[u], sv));
                }
            } else {
                const uint4 z = make_uint4(0, 0, 0, 0);
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                    st_stream(krow + off, z); st_stream(vrow + off, z);
                }
            }
        }
    }
    idx += gridDim.x;
    } while (SPARSE && idx < limit);
}

template <int D, class E>
static cudaError_t launch_unpack_d(const Geom &g, const Layout &lo, const uint8_t *blob, uint64_t blob_stride,
                                   __half *K, __half *V, uint8_t *tier_out, TileSrc ts, dim3 grid, cudaStream_t s)
{
    if ((g.Hkv * D) % 256 == 0) {
        // (a sparse launch never carries a 2-bit tier: skv_host.cu plan_stage)
#define SKV_LAUNCH_UNPACK(NCH)                                                                                                        \
        do {                                                                                                                          \
            if (g.low_code == 2) unpack_fast_kernel<D, NCH, MinBlocks<NCH, true>::value, true, E, false><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tier_out, ts); \
            else if (ts.live_count) unpack_fast_kernel<D, NCH, MinBlocks<NCH, false>::value, false, E, true><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tier_out, ts); \
            else unpack_fast_kernel<D, NCH, MinBlocks<NCH, false>::value, false, E, false><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tier_out, ts); \
        } while (0)
        if (g.row_chunks % 4 == 0) SKV_LAUNCH_UNPACK(4);
        else if (g.row_chunks % 2 == 0) SKV_LAUNCH_UNPACK(2);
        else SKV_LAUNCH_UNPACK(1);
#undef SKV_LAUNCH_UNPACK
    } else if (ts.live_count) {
        unpack_kernel<D, E, true><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tier_out, ts);
    } else {
        unpack_kernel<D, E, false><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tier_out, ts);
    }
    return cudaGetLastError();
}

cudaError_t launch_unpack(const Geom &g, const Layout &lo, const uint8_t *blob, uint64_t blob_stride,
                          __half *K, __half *V, uint8_t *tier_out, TileSrc ts, int grid_x, cudaStream_t s)
{
    const dim3 grid(grid_x, g.L, g.R);
    switch (g.D) {
    case 64: return g.bf16 ? launch_unpack_d<64, ElemBF16>(g, lo, blob, blob_stride, K, V, tier_out, ts, grid, s)
                            : launch_unpack_d<64, ElemF16>(g, lo, blob, blob_stride, K, V, tier_out, ts, grid, s);
    case 128: return g.bf16 ? launch_unpack_d<128, ElemBF16>(g, lo, blob, blob_stride, K, V, tier_out, ts, grid, s)
                            : launch_unpack_d<128, ElemF16>(g, lo, blob, blob_stride, K, V, tier_out, ts, grid, s);
    case 256: return g.bf16 ? launch_unpack_d<256, ElemBF16>(g, lo, blob, blob_stride, K, V, tier_out, ts, grid, s)
                            : launch_unpack_d<256, ElemF16>(g, lo, blob, blob_stride, K, V, tier_out, ts, grid, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace skv
