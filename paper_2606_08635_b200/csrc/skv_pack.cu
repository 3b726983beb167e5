// skv_pack.cu -- quantize-and-pack (Alg. 1 step 4; "standard symmetric").
//
// One warp per token, one CTA per 32-token tile of one (request, layer).  The warp reads the token's K
// row and V row with 16-byte loads (8 fp16 per lane, coalesced; any 16-B aligned strides), reduces the
// |x| max over the lanes of a head vector with shuffles, quantises in fp32 exactly as include/skv.h
// specifies, and stores the codes at the token's slot (tile base + in-tile rank from a ballot).  The tile
// base comes from skv_scan.cu (long sequences) or is counted by the CTA itself (n <= kFuseMaxTokens: pack
// is then ONE launch, metadata included); a sparse blob (cold-tier upgrade) is walked through the scan's
// list of live tiles.  All lanes of a warp share one tier => no divergence.  Dropped tokens are never loaded.
//
// HBM-bound: reads Bytes_FP16, writes beta*Bytes_FP16.
#include "skv_codec.cuh"

namespace skv {

// |x| max of the 8 halves in a uint4, as a half2 with the max in both halves' union (max(lo,hi) taken later)
template <class E>
__device__ __forceinline__ typename E::H2 absmax8(const uint4 &v)
{
    using H2 = typename E::H2;
    const H2 a = __habs2(as_pair<H2>(v.x)), b = __habs2(as_pair<H2>(v.y));
    const H2 c = __habs2(as_pair<H2>(v.z)), d = __habs2(as_pair<H2>(v.w));
    return __hmax2(__hmax2(a, b), __hmax2(c, d));
}

// Fused launch (TileSrc::tile_base == nullptr): the blob metadata tile_scan_kernel would have written.  Every CTA copies
// its 32 tier-map bytes; the CTA of tile 0 zeroes the pads of its layer's ten segments and, in layer 0, writes the
// header and the pad behind the tier map.
__device__ __forceinline__ void pack_metadata(const Geom &g, const Layout &lo, const Header256 &hdr, uint8_t *rblob,
                                              int l, int64_t tile, int64_t j0, uint32_t my_t)
{
    const uint32_t tid = threadIdx.x;
    if (tid < 32 && j0 + tid < g.n) rblob[lo.tier_map_off + (int64_t)l * g.n + j0 + tid] = (uint8_t)my_t;
    if (tile != 0) return;
    uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
    for (int s = 0; s < 10; ++s) {
        const uint64_t beg = lo.seg_off[s] + lo.seg_raw[s], end = lo.seg_off[s] + pad256(lo.seg_raw[s]);
        for (uint64_t o = beg + tid; o < end; o += blockDim.x) lbase[o] = 0;
    }
    if (l == 0) {
        if (tid < 64) reinterpret_cast<uint32_t *>(rblob)[tid] = hdr.w[tid];
        for (uint64_t o = lo.tier_map_off + (uint64_t)g.L * (uint64_t)g.n + tid; o < lo.layer0_off; o += blockDim.x) rblob[o] = 0;
    }
}

template <int D, int QMAX, class E>
__device__ __forceinline__ void quantize_chunk(const uint4 &v, uint32_t lane, typename E::H &amax_out, uint32_t codes[8])
{
    using H = typename E::H; using H2 = typename E::H2;
    constexpr int LPV = D / 8;                        // lanes per head vector
    H2 m2 = absmax8<E>(v);
#pragma unroll
    for (int o = 1; o < LPV; o <<= 1) m2 = __hmax2(m2, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(m2), o)));
    const H amax = __hmax(lo_h(m2), hi_h(m2));
    const float inv = inv_of(amax, (float)QMAX);
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 f = to_f2(as_pair<H2>(w[k]));
        codes[2 * k] = rne_code_bits(f.x, inv);
        codes[2 * k + 1] = rne_code_bits(f.y, inv);
    }
    amax_out = amax;
    (void)lane;
}

template <int D, class E, bool SPARSE>
__global__ void __launch_bounds__(256)
pack_kernel(Geom g, Layout lo, const __half *__restrict__ K, const __half *__restrict__ V,
            const uint8_t *__restrict__ tier_map, uint8_t *__restrict__ blob, uint64_t blob_stride,
            Header256 hdr, TileSrc ts)
{
    using H = typename E::H; using H2 = typename E::H2;
    constexpr int LPV = D / 8;
    __shared__ uint32_t sCnt[16];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t n = g.n, rl = (int64_t)r * g.L + l;
    const uint8_t *tm = tier_map + rl * n;
    const uint32_t low = (uint32_t)g.low_code;                       // 4: symmetric INT4, 2: asymmetric 2-bit (NEXT-4)
    uint8_t *rblob = blob + (uint64_t)r * blob_stride;
    uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
    const int row_elems = g.Hkv * D;
    const int64_t cache_off = (int64_t)r * g.sr + (int64_t)l * g.sl;
    const uint32_t limit = SPARSE ? ts.live_count[rl] : (uint32_t)g.tiles;
    uint32_t idx = blockIdx.x;
    if (SPARSE && idx >= limit) return;

#pragma unroll 1
    do {
    const int64_t tile = SPARSE ? (int64_t)ts.tile_base[rl * g.tiles + idx].w : (int64_t)idx;
    const int64_t j0 = tile * kTileTokens;
    // tiers of the tile: lane i holds token j0+i
    const uint32_t my_t = (j0 + lane < n) ? (uint32_t)tm[j0 + lane] : 0xFFu;
    const uint32_t m16 = __ballot_sync(0xffffffffu, my_t == 16u);
    const uint32_t m8 = __ballot_sync(0xffffffffu, my_t == 8u);
    const uint32_t m4 = __ballot_sync(0xffffffffu, my_t == low);
    uint4 base;
    if (ts.tile_base) base = ts.tile_base[rl * g.tiles + tile];
    else { base = self_tile_base(tm, tile, low, sCnt); pack_metadata(g, lo, hdr, rblob, l, tile, j0, my_t); }

    for (uint32_t i = warp; i < (uint32_t)kTileTokens; i += nwarps) {
        const uint32_t t = __shfl_sync(0xffffffffu, my_t, i);
        if (t != 16u && t != 8u && t != low) continue;                // dropped / tail / invalid: no bytes
        const uint32_t below = (1u << i) - 1u;
        const int64_t j = j0 + i;
        const __half *krow = K + cache_off + j * g.st;
        const __half *vrow = V + cache_off + j * g.st;

        if (t == 16u) {
            const uint32_t slot = base.x + __popc(m16 & below);
            if (slot >= (uint32_t)g.n16) continue;
            uint8_t *kd = lbase + lo.seg_off[0] + (uint64_t)slot * row_elems * 2;
            uint8_t *vd = lbase + lo.seg_off[1] + (uint64_t)slot * row_elems * 2;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint4 kv[4], vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        kv[u] = ld_stream(krow + (int64_t)h * g.sh + c);
                        vv[u] = ld_stream(vrow + (int64_t)h * g.sh + c);
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) { st_stream(kd + e * 2, kv[u]); st_stream(vd + e * 2, vv[u]); }
                }
            }
        } else if (t == 8u) {
            const uint32_t slot = base.y + __popc(m8 & below);
            if (slot >= (uint32_t)g.n8) continue;
            uint8_t *kd = lbase + lo.seg_off[2] + (uint64_t)slot * row_elems;
            uint8_t *vd = lbase + lo.seg_off[3] + (uint64_t)slot * row_elems;
            H *ks = reinterpret_cast<H *>(lbase + lo.seg_off[6]) + (uint64_t)slot * g.Hkv;
            H *vs = reinterpret_cast<H *>(lbase + lo.seg_off[7]) + (uint64_t)slot * g.Hkv;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint4 kv[4], vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    kv[u] = make_uint4(0, 0, 0, 0); vv[u] = kv[u];
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        kv[u] = ld_stream(krow + (int64_t)h * g.sh + c);
                        vv[u] = ld_stream(vrow + (int64_t)h * g.sh + c);
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if ((c0 + u) * 256 >= row_elems) break;            // warp-uniform
                    const int e = (c0 + u) * 256 + lane * 8;
                    H ak, av; uint32_t ck[8], cv[8];
                    quantize_chunk<D, 127, E>(kv[u], lane, ak, ck);
                    quantize_chunk<D, 127, E>(vv[u], lane, av, cv);
                    if (e < row_elems) {
                        st_stream(kd + e, make_uint2(pack4_bytes(ck[0], ck[1], ck[2], ck[3]), pack4_bytes(ck[4], ck[5], ck[6], ck[7])));
                        st_stream(vd + e, make_uint2(pack4_bytes(cv[0], cv[1], cv[2], cv[3]), pack4_bytes(cv[4], cv[5], cv[6], cv[7])));
                        if ((lane % LPV) == 0) { ks[e / D] = ak; vs[e / D] = av; }
                    }
                }
            }
        } else if (low == 2u) {
            const uint32_t slot = base.z + __popc(m4 & below);
            if (slot >= (uint32_t)g.n4) continue;
            uint8_t *kd = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 4);
            uint8_t *vd = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 4);
            const int recs = g.low_group ? row_elems / g.low_group : g.Hkv;          // (lo, hi) records per token row
            H2 *ks = reinterpret_cast<H2 *>(lbase + lo.seg_off[8]) + (uint64_t)slot * recs;
            H2 *vs = reinterpret_cast<H2 *>(lbase + lo.seg_off[9]) + (uint64_t)slot * recs;
            for (int c0 = 0; c0 < g.row_chunks; ++c0) {
                const int e = c0 * 256 + lane * 8;
                const bool in = e < row_elems;
                uint4 kv = make_uint4(0, 0, 0, 0), vv = kv;
                if (in) {
                    const int h = e / D, c = e % D;
                    kv = ld_stream(krow + (int64_t)h * g.sh + c);
                    vv = ld_stream(vrow + (int64_t)h * g.sh + c);
                }
                // lanes past the row hold zeros: they sit in head-vector groups of their own (row_elems % D == 0)
                // quantisation group: the head vector (LPV lanes), or 32 elements = 4 lanes (reading P22)
                const int glanes = g.low_group ? g.low_group / 8 : LPV;
                H2 mk = max_negmin8<E>(kv), mv = max_negmin8<E>(vv);
                for (int o = 1; o < glanes; o <<= 1) {
                    mk = __hmax2(mk, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(mk), o)));
                    mv = __hmax2(mv, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(mv), o)));
                }
                H loK, hiK, loV, hiV;
                lohi_of(mk, loK, hiK); lohi_of(mv, loV, hiV);
                if (in) {
                    st_stream2(kd + e / 4, (uint16_t)quant8_int2<E>(kv, to_f(loK), inv3_of(range_of(loK, hiK))));
                    st_stream2(vd + e / 4, (uint16_t)quant8_int2<E>(vv, to_f(loV), inv3_of(range_of(loV, hiV))));
                    if ((lane % glanes) == 0) {
                        const int rec = g.low_group ? e / g.low_group : e / D;      // record index inside the token's row
                        ks[rec] = pair_h(loK, hiK); vs[rec] = pair_h(loV, hiV);
                    }
                }
            }
        } else {
            const uint32_t slot = base.z + __popc(m4 & below);
            if (slot >= (uint32_t)g.n4) continue;
            uint8_t *kd = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 2);
            uint8_t *vd = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 2);
            H *ks = reinterpret_cast<H *>(lbase + lo.seg_off[8]) + (uint64_t)slot * g.Hkv;
            H *vs = reinterpret_cast<H *>(lbase + lo.seg_off[9]) + (uint64_t)slot * g.Hkv;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint4 kv[4], vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    kv[u] = make_uint4(0, 0, 0, 0); vv[u] = kv[u];
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        kv[u] = ld_stream(krow + (int64_t)h * g.sh + c);
                        vv[u] = ld_stream(vrow + (int64_t)h * g.sh + c);
                    }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    if ((c0 + u) * 256 >= row_elems) break;
                    const int e = (c0 + u) * 256 + lane * 8;
                    H ak, av; uint32_t ck[8], cv[8];
                    quantize_chunk<D, 7, E>(kv[u], lane, ak, ck);
                    quantize_chunk<D, 7, E>(vv[u], lane, av, cv);
                    if (e < row_elems) {
                        uint32_t kb[4], vb[4];
#pragma unroll
                        for (int k = 0; k < 4; ++k) {                  // element 2k low nibble, 2k+1 high nibble
                            kb[k] = (ck[2 * k] & 0xFu) | (ck[2 * k + 1] << 4);
                            vb[k] = (cv[2 * k] & 0xFu) | (cv[2 * k + 1] << 4);
                        }
                        st_stream(kd + e / 2, pack4_bytes(kb[0], kb[1], kb[2], kb[3]));
                        st_stream(vd + e / 2, pack4_bytes(vb[0], vb[1], vb[2], vb[3]));
                        if ((lane % LPV) == 0) { ks[e / D] = ak; vs[e / D] = av; }
                    }
                }
            }
        }
    }
    idx += gridDim.x;
    } while (SPARSE && idx < limit);
}

// ------------------------------------------------------------------------------------------------
// Fast path: the token row is a whole number of NCH-chunk batches (row_elems % (256*NCH) == 0).
// Fully unrolled; the K and V absmax of the NCH chunks are reduced together by the transposed group
// reduction (skv_codec.cuh): NCH-1+log2(LPV/NCH) shuffles and TWO divisions per lane per batch instead
// of 2*NCH*log2(LPV) shuffles and 2*NCH divisions; the reciprocals are then broadcast with 2*NCH shuffles.
// ------------------------------------------------------------------------------------------------
// LOW2 = false: the low tier is symmetric INT4 (tier code 4).  LOW2 = true (NEXT-4): asymmetric 2-bit (tier code 2).
// SPARSE: the grid strides over the scan's list of live tiles (TileSrc::live_count); otherwise one CTA per tile, no loop.
template <int D, int NCH, int MINB, bool LOW2, class E, bool SPARSE>
__global__ void __launch_bounds__(256, MINB)
pack_fast_kernel(Geom g, Layout lo, const __half *__restrict__ K, const __half *__restrict__ V,
                 const uint8_t *__restrict__ tier_map, uint8_t *__restrict__ blob, uint64_t blob_stride,
                 Header256 hdr, TileSrc ts)
{
    using H = typename E::H; using H2 = typename E::H2;
    constexpr int LPV = D / 8;                 // lanes per head vector
    constexpr int HPC = 256 / D;               // head vectors per 256-element chunk
    constexpr uint32_t kLow = LOW2 ? 2u : 4u;
    __shared__ uint32_t sCnt[16];
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t n = g.n, rl = (int64_t)r * g.L + l;
    const uint8_t *tm = tier_map + rl * n;
    uint8_t *rblob = blob + (uint64_t)r * blob_stride;
    uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
    const int row_elems = g.Hkv * D;
    const __half *Kb = K + (int64_t)r * g.sr + (int64_t)l * g.sl;
    const __half *Vb = V + (int64_t)r * g.sr + (int64_t)l * g.sl;
    const int lane_h = (int)(lane * 8) / D, lane_c = (int)(lane * 8) % D;
    const int my_chunk = held_chunk<LPV, NCH>(lane);
    const bool scale_writer = (lane % (LPV / NCH)) == 0;
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
    else { base = self_tile_base(tm, tile, kLow, sCnt); pack_metadata(g, lo, hdr, rblob, l, tile, j0, my_t); }

#pragma unroll 1
    for (uint32_t i = warp; i < (uint32_t)kTileTokens; i += 8) {
        const uint32_t t = __shfl_sync(0xffffffffu, my_t, i);
        if (t != 16u && t != 8u && t != kLow) continue;               // dropped / tail / invalid: no bytes
        const uint32_t below = (1u << i) - 1u;
        const int64_t j = j0 + i;
        const __half *krow = Kb + j * g.st + lane_c;
        const __half *vrow = Vb + j * g.st + lane_c;
        const uint32_t slot = (t == 16u) ? base.x + __popc(m16 & below)
                            : (t == 8u)  ? base.y + __popc(m8 & below) : base.z + __popc(m4 & below);
        const uint32_t cap = (t == 16u) ? (uint32_t)g.n16 : (t == 8u) ? (uint32_t)g.n8 : (uint32_t)g.n4;
        if (slot >= cap) continue;                                    // foreign map that disagrees with counts

#pragma unroll 1
        for (int cb = 0; cb < g.row_chunks; cb += NCH) {
            uint4 kv[NCH], vv[NCH];
#pragma unroll
            for (int u = 0; u < NCH; ++u) {
                const int64_t off = (int64_t)((cb + u) * HPC + lane_h) * g.sh;
                kv[u] = ld_stream(krow + off);
                vv[u] = ld_stream(vrow + off);
            }
            if (t == 16u) {
                uint8_t *kd = lbase + lo.seg_off[0] + ((uint64_t)slot * row_elems + cb * 256 + lane * 8) * 2;
                uint8_t *vd = lbase + lo.seg_off[1] + ((uint64_t)slot * row_elems + cb * 256 + lane * 8) * 2;
#pragma unroll
                for (int u = 0; u < NCH; ++u) { st_stream(kd + u * 512, kv[u]); st_stream(vd + u * 512, vv[u]); }
                continue;
            }
            if (LOW2 && t == 2u && g.low_group) {
                // group-wise 2-bit (reading P22): a group of 32 elements = 4 lanes; every lane ends up with its own
                // group's (max, -min), so nothing is broadcast; one (lo, hi) record per group
                uint8_t *kd = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                uint8_t *vd = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                H2 *ks = reinterpret_cast<H2 *>(lbase + lo.seg_off[8]) + (uint64_t)slot * (row_elems / 32) + cb * 8 + lane / 4;
                H2 *vs = reinterpret_cast<H2 *>(lbase + lo.seg_off[9]) + (uint64_t)slot * (row_elems / 32) + cb * 8 + lane / 4;
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    H2 mk = max_negmin8<E>(kv[u]), mv = max_negmin8<E>(vv[u]);
#pragma unroll
                    for (int o = 1; o < 4; o <<= 1) {
                        mk = __hmax2(mk, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(mk), o)));
                        mv = __hmax2(mv, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(mv), o)));
                    }
                    H loK, hiK, loV, hiV;
                    lohi_of(mk, loK, hiK); lohi_of(mv, loV, hiV);
                    st_stream2(kd + u * 64, (uint16_t)quant8_int2<E>(kv[u], to_f(loK), inv3_of(range_of(loK, hiK))));
                    st_stream2(vd + u * 64, (uint16_t)quant8_int2<E>(vv[u], to_f(loV), inv3_of(range_of(loV, hiV))));
                    if ((lane & 3) == 0) { ks[u * 8] = pair_h(loK, hiK); vs[u * 8] = pair_h(loV, hiV); }
                }
                continue;
            }
            if (LOW2 && t == 2u) {
                // asymmetric 2-bit: (max, -min) of K and of V reduced over the lanes of a head vector, (lo, hi) records,
                // 16 bits of codes per lane and chunk
                H2 mk[NCH], mv[NCH];
#pragma unroll
                for (int u = 0; u < NCH; ++u) { mk[u] = max_negmin8<E>(kv[u]); mv[u] = max_negmin8<E>(vv[u]); }
                const H2 rk = group_absmax<LPV, NCH>(mk, lane), rv = group_absmax<LPV, NCH>(mv, lane);
                H loK, hiK, loV, hiV;
                lohi_of(rk, loK, hiK); lohi_of(rv, loV, hiV);
                const float invK = inv3_of(range_of(loK, hiK)), invV = inv3_of(range_of(loV, hiV));
                const float lKf = to_f(loK), lVf = to_f(loV);
                if (scale_writer) {
                    const int head = (cb + my_chunk) * HPC + (int)(lane / LPV);
                    H2 *ks = reinterpret_cast<H2 *>(lbase + lo.seg_off[8]) + (uint64_t)slot * g.Hkv;
                    H2 *vs = reinterpret_cast<H2 *>(lbase + lo.seg_off[9]) + (uint64_t)slot * g.Hkv;
                    ks[head] = pair_h(loK, hiK);
                    vs[head] = pair_h(loV, hiV);
                }
                uint8_t *kd = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
                uint8_t *vd = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 4) + cb * 64 + lane * 2;
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int src = src_lane<LPV, NCH>(lane, u);
                    const float ik = __shfl_sync(0xffffffffu, invK, src), iv = __shfl_sync(0xffffffffu, invV, src);
                    const float lk = __shfl_sync(0xffffffffu, lKf, src), lv = __shfl_sync(0xffffffffu, lVf, src);
                    st_stream2(kd + u * 64, (uint16_t)quant8_int2<E>(kv[u], lk, ik));
                    st_stream2(vd + u * 64, (uint16_t)quant8_int2<E>(vv[u], lv, iv));
                }
                continue;
            }
            H2 m[NCH];
#pragma unroll
            for (int u = 0; u < NCH; ++u) m[u] = pair_h(absmax8_scalar<E>(kv[u]), absmax8_scalar<E>(vv[u]));
            const H2 a2 = group_absmax<LPV, NCH>(m, lane);      // (K amax, V amax) of chunk cb + my_chunk
            const bool is8 = (t == 8u);
            const float qmax = is8 ? 127.0f : 7.0f;
            const float invK = inv_of(lo_h(a2), qmax), invV = inv_of(hi_h(a2), qmax);
            if (scale_writer) {
                const int head = (cb + my_chunk) * HPC + (int)(lane / LPV);
                H *ks = reinterpret_cast<H *>(lbase + lo.seg_off[is8 ? 6 : 8]) + (uint64_t)slot * g.Hkv;
                H *vs = reinterpret_cast<H *>(lbase + lo.seg_off[is8 ? 7 : 9]) + (uint64_t)slot * g.Hkv;
                ks[head] = lo_h(a2);
                vs[head] = hi_h(a2);
            }
            if (is8) {
                uint8_t *kd = lbase + lo.seg_off[2] + (uint64_t)slot * row_elems + cb * 256 + lane * 8;
                uint8_t *vd = lbase + lo.seg_off[3] + (uint64_t)slot * row_elems + cb * 256 + lane * 8;
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int src = src_lane<LPV, NCH>(lane, u);
                    const float ik = __shfl_sync(0xffffffffu, invK, src), iv = __shfl_sync(0xffffffffu, invV, src);
                    st_stream(kd + u * 256, quant8_int8<E>(kv[u], ik));
                    st_stream(vd + u * 256, quant8_int8<E>(vv[u], iv));
                }
            } else {
                uint8_t *kd = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 2) + cb * 128 + lane * 4;
                uint8_t *vd = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 2) + cb * 128 + lane * 4;
#pragma unroll
                for (int u = 0; u < NCH; ++u) {
                    const int src = src_lane<LPV, NCH>(lane, u);
                    const float ik = __shfl_sync(0xffffffffu, invK, src), iv = __shfl_sync(0xffffffffu, invV, src);
                    st_stream(kd + u * 128, quant8_int4<E>(kv[u], ik));
                    st_stream(vd + u * 128, quant8_int4<E>(vv[u], iv));
                }
            }
        }
    }
    idx += gridDim.x;
    } while (SPARSE && idx < limit);
}

template <int D, int NCH, class E>
static cudaError_t launch_pack_fast(const Geom &g, const Layout &lo, const __half *K, const __half *V,
                                    const uint8_t *tier_map, uint8_t *blob, uint64_t blob_stride,
                                    const Header256 &hdr, TileSrc ts, dim3 grid, cudaStream_t s)
{
    // (a sparse launch never carries a 2-bit tier: skv_host.cu plan_stage)
    if (g.low_code == 2) pack_fast_kernel<D, NCH, MinBlocks<NCH, true>::value, true, E, false><<<grid, 256, 0, s>>>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts);
    else if (ts.live_count) pack_fast_kernel<D, NCH, MinBlocks<NCH, false>::value, false, E, true><<<grid, 256, 0, s>>>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts);
    else pack_fast_kernel<D, NCH, MinBlocks<NCH, false>::value, false, E, false><<<grid, 256, 0, s>>>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts);
    return cudaGetLastError();
}

template <int D, class E>
static cudaError_t launch_pack_d(const Geom &g, const Layout &lo, const __half *K, const __half *V,
                                 const uint8_t *tier_map, uint8_t *blob, uint64_t blob_stride,
                                 const Header256 &hdr, TileSrc ts, dim3 grid, cudaStream_t s)
{
    if ((g.Hkv * D) % 256 == 0) {
        if (g.row_chunks % 4 == 0) return launch_pack_fast<D, 4, E>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s);
        if (g.row_chunks % 2 == 0) return launch_pack_fast<D, 2, E>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s);
        return launch_pack_fast<D, 1, E>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s);
    }
    if (ts.live_count) pack_kernel<D, E, true><<<grid, 256, 0, s>>>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts);
    else pack_kernel<D, E, false><<<grid, 256, 0, s>>>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts);
    return cudaGetLastError();
}

cudaError_t launch_pack(const Geom &g, const Layout &lo, const __half *K, const __half *V, const uint8_t *tier_map,
                        uint8_t *blob, uint64_t blob_stride, const Header256 &hdr, TileSrc ts, int grid_x, cudaStream_t s)
{
    const dim3 grid(grid_x, g.L, g.R);
    switch (g.D) {
    case 64: return g.bf16 ? launch_pack_d<64, ElemBF16>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s)
                            : launch_pack_d<64, ElemF16>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s);
    case 128: return g.bf16 ? launch_pack_d<128, ElemBF16>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s)
                            : launch_pack_d<128, ElemF16>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s);
    case 256: return g.bf16 ? launch_pack_d<256, ElemBF16>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s)
                            : launch_pack_d<256, ElemF16>(g, lo, K, V, tier_map, blob, blob_stride, hdr, ts, grid, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace skv
