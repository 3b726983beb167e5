// skv_unpack.cu -- unpack-and-dequantize (decode side, "only lightweight dequantization
// (table lookup) is needed at the decode worker").
//
// Mirror of skv_pack.cu: one warp per token, one CTA per 32-token tile of one (request, layer).  The slot
// of a token is recomputed from the transmitted tier map (tile base from skv_scan.cu + ballot rank).
// INT8: 8-byte loads per lane -> 8 fp16 (one 16-byte store); INT4: 4-byte loads -> 8 fp16.  y = f16_rn(
// fl32(float(q) * fl32(amax/qmax))); int->float goes through the 2^23 exponent trick (exact), so no I2F.
// Dropped tokens are written as +0.0 (reading P10).  HBM-bound: reads beta*Bytes_FP16, writes Bytes_FP16.
#include "skv_common.cuh"

namespace skv {

__device__ __forceinline__ void st_stream16(void *p, uint4 v)
{
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ uint4 ld_stream16(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ uint2 ld_stream8(const void *p)
{
    uint2 r;
    asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(r.x), "=r"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ uint32_t ld_stream4(const void *p)
{
    uint32_t r;
    asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}

__device__ __forceinline__ float scale_of(__half amax, float qmax)
{
    const float af = __half2float(amax);
    return af != 0.0f ? __fdiv_rn(af, qmax) : 0.0f;
}

__device__ __forceinline__ uint32_t h2_bits(float a, float b)
{
    const __half2 h = __floats2half2_rn(a, b);
    return *reinterpret_cast<const uint32_t *>(&h);
}

// four biased bytes (q+BIAS in each byte of w) -> two half2 words of f16_rn(q*scale)
template <int BIAS>
__device__ __forceinline__ void dequant4(uint32_t w, float scale, uint32_t &o0, uint32_t &o1)
{
    constexpr float kOff = 8388608.0f + (float)BIAS;                  // 2^23 + BIAS, exact
    const float f0 = __fsub_rn(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7540)), kOff);
    const float f1 = __fsub_rn(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7541)), kOff);
    const float f2 = __fsub_rn(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7542)), kOff);
    const float f3 = __fsub_rn(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7543)), kOff);
    o0 = h2_bits(__fmul_rn(f0, scale), __fmul_rn(f1, scale));
    o1 = h2_bits(__fmul_rn(f2, scale), __fmul_rn(f3, scale));
}

__device__ __forceinline__ uint4 dequant_int8(uint2 w, float scale)
{
    uint4 o;
    dequant4<128>(w.x ^ 0x80808080u, scale, o.x, o.y);
    dequant4<128>(w.y ^ 0x80808080u, scale, o.z, o.w);
    return o;
}

__device__ __forceinline__ uint4 dequant_int4(uint32_t w, float scale)
{
    w ^= 0x88888888u;                                   // every nibble becomes q+8 in 1..15
    const uint32_t even = w & 0x0F0F0F0Fu;              // elements 0,2,4,6
    const uint32_t odd = (w >> 4) & 0x0F0F0F0Fu;        // elements 1,3,5,7
    constexpr float kOff = 8388608.0f + 8.0f;
    float f[8];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        f[2 * k] = __fsub_rn(__uint_as_float(__byte_perm(even, 0x4B000000u, 0x7540 + k)), kOff);
        f[2 * k + 1] = __fsub_rn(__uint_as_float(__byte_perm(odd, 0x4B000000u, 0x7540 + k)), kOff);
    }
    uint4 o;
    o.x = h2_bits(__fmul_rn(f[0], scale), __fmul_rn(f[1], scale));
    o.y = h2_bits(__fmul_rn(f[2], scale), __fmul_rn(f[3], scale));
    o.z = h2_bits(__fmul_rn(f[4], scale), __fmul_rn(f[5], scale));
    o.w = h2_bits(__fmul_rn(f[6], scale), __fmul_rn(f[7], scale));
    return o;
}

template <int D>
__global__ void __launch_bounds__(256)
unpack_kernel(Geom g, Layout lo, const uint8_t *__restrict__ blob, uint64_t blob_stride,
              __half *__restrict__ K, __half *__restrict__ V, const uint4 *__restrict__ tile_base)
{
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    const int64_t tile = blockIdx.x;
    const int l = blockIdx.y, r = blockIdx.z;
    const int64_t n = g.n;
    const int64_t j0 = tile * kTileTokens;

    const uint8_t *rblob = blob + (uint64_t)r * blob_stride;
    const uint8_t *tm = rblob + lo.tier_map_off + (int64_t)l * n;
    const uint32_t my_t = (j0 + lane < n) ? (uint32_t)tm[j0 + lane] : 0xFFu;
    const uint32_t m16 = __ballot_sync(0xffffffffu, my_t == 16u);
    const uint32_t m8 = __ballot_sync(0xffffffffu, my_t == 8u);
    const uint32_t m4 = __ballot_sync(0xffffffffu, my_t == 4u);
    const uint4 base = tile_base[((int64_t)r * g.L + l) * g.tiles + tile];

    const uint8_t *lbase = rblob + lo.layer0_off + (uint64_t)l * lo.layer_stride;
    const int row_elems = g.Hkv * D;
    const int64_t cache_off = (int64_t)r * g.sr + (int64_t)l * g.sl;

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
        else if (t == 4u) { slot = base.z + __popc(m4 & below); if (slot >= (uint32_t)g.n4) t = 0; }
        else t = 0;

        if (t == 16u) {
            const uint8_t *ks = lbase + lo.seg_off[0] + (uint64_t)slot * row_elems * 2;
            const uint8_t *vs = lbase + lo.seg_off[1] + (uint64_t)slot * row_elems * 2;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint4 kv[4], vv[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) { kv[u] = ld_stream16(ks + e * 2); vv[u] = ld_stream16(vs + e * 2); }
                }
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const int e = (c0 + u) * 256 + lane * 8;
                    if (e < row_elems) {
                        const int h = e / D, c = e % D;
                        st_stream16(krow + (int64_t)h * g.sh + c, kv[u]);
                        st_stream16(vrow + (int64_t)h * g.sh + c, vv[u]);
                    }
                }
            }
        } else if (t == 8u) {
            const uint8_t *ks = lbase + lo.seg_off[2] + (uint64_t)slot * row_elems;
            const uint8_t *vs = lbase + lo.seg_off[3] + (uint64_t)slot * row_elems;
            const __half *ka = reinterpret_cast<const __half *>(lbase + lo.seg_off[6]) + (uint64_t)slot * g.Hkv;
            const __half *va = reinterpret_cast<const __half *>(lbase + lo.seg_off[7]) + (uint64_t)slot * g.Hkv;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint2 kv[4], vv[4]; __half ak[4], av[4];
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
                        st_stream16(krow + (int64_t)h * g.sh + c, dequant_int8(kv[u], scale_of(ak[u], 127.0f)));
                        st_stream16(vrow + (int64_t)h * g.sh + c, dequant_int8(vv[u], scale_of(av[u], 127.0f)));
                    }
                }
            }
        } else if (t == 4u) {
            const uint8_t *ks = lbase + lo.seg_off[4] + (uint64_t)slot * (row_elems / 2);
            const uint8_t *vs = lbase + lo.seg_off[5] + (uint64_t)slot * (row_elems / 2);
            const __half *ka = reinterpret_cast<const __half *>(lbase + lo.seg_off[8]) + (uint64_t)slot * g.Hkv;
            const __half *va = reinterpret_cast<const __half *>(lbase + lo.seg_off[9]) + (uint64_t)slot * g.Hkv;
            for (int c0 = 0; c0 < g.row_chunks; c0 += 4) {
                uint32_t kv[4], vv[4]; __half ak[4], av[4];
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
                        st_stream16(krow + (int64_t)h * g.sh + c, dequant_int4(kv[u], scale_of(ak[u], 7.0f)));
                        st_stream16(vrow + (int64_t)h * g.sh + c, dequant_int4(vv[u], scale_of(av[u], 7.0f)));
                    }
                }
            }
        } else {
            const uint4 z = make_uint4(0, 0, 0, 0);
            for (int c0 = 0; c0 < g.row_chunks; ++c0) {
                const int e = c0 * 256 + lane * 8;
                if (e < row_elems) {
                    const int h = e / D, c = e % D;
                    st_stream16(krow + (int64_t)h * g.sh + c, z);
                    st_stream16(vrow + (int64_t)h * g.sh + c, z);
                }
            }
        }
    }
}

cudaError_t launch_unpack(const Geom &g, const Layout &lo, const uint8_t *blob, uint64_t blob_stride,
                          __half *K, __half *V, const uint4 *tile_base, cudaStream_t s)
{
    dim3 grid(g.tiles, g.L, g.R);
    switch (g.D) {
    case 64:  unpack_kernel<64><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tile_base); break;
    case 128: unpack_kernel<128><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tile_base); break;
    case 256: unpack_kernel<256><<<grid, 256, 0, s>>>(g, lo, blob, blob_stride, K, V, tile_base); break;
    default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}

}  // namespace skv
