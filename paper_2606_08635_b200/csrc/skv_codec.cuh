// skv_codec.cuh -- device helpers shared by the pack and unpack kernels: streaming loads/stores, the
// per-vector absmax machinery and the exact fp32 quantise / dequantise steps of include/skv.h.
#pragma once
#include <cuda_bf16.h>

#include "skv_common.cuh"

namespace skv {

__device__ __forceinline__ uint4 ld_stream(const void *p)
{
    uint4 r;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
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
__device__ __forceinline__ void st_stream(void *p, uint4 v)
{
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void st_stream(void *p, uint2 v)
{
    asm volatile("st.global.L1::no_allocate.v2.u32 [%0], {%1,%2};" :: "l"(p), "r"(v.x), "r"(v.y) : "memory");
}
__device__ __forceinline__ void st_stream(void *p, uint32_t v)
{
    asm volatile("st.global.L1::no_allocate.u32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

// Resident CTAs per SM the fast pack / unpack kernels are compiled for (register cap 65536 / (256 * value)).  A lane
// keeps 2 * NCH 16-byte loads in flight, so short rows (NCH = 2 or 1: rows of 512 or 256 elements, e.g. 4 KV heads of 128)
// need more resident warps than long ones to cover the HBM latency (C2 pack: 0.75 -> 0.85 of the copy peak from 3 -> 5).
// The 2-bit codec needs more registers: it stays at four.
template <int NCH, bool LOW2> struct MinBlocks {
    static constexpr int value = (NCH >= 4) ? 3 : LOW2 ? 4 : (NCH == 2) ? 5 : 6;
};

// ------------------------------------------------------------------------------------------------
// Fused slot scan (short sequences, n <= kFuseMaxTokens): the whole CTA counts the FP16 / INT8 / low-tier bytes of
// the layer's tier map below its own tile -- the same exclusive counts tile_scan_kernel would have left in
// tile_base[tile] -- so that pack and unpack are ONE launch each.  Every thread returns the counts.  Contains CTA-wide
// barriers: call it from CTA-uniform control flow.  sCnt: 16 words of shared memory.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 self_tile_base(const uint8_t *__restrict__ tm, int64_t tile, uint32_t low, uint32_t *sCnt)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t chunks = tile * (kTileTokens / 16);                 // 16-byte chunks below the tile
    const uint32_t lowrep = low * 0x01010101u;
    uint32_t a = 0 /* #16 | #8 << 16 */, b = 0 /* #low */;
    if ((reinterpret_cast<uintptr_t>(tm) & 15) == 0) {
        for (int64_t c = tid; c < chunks; c += blockDim.x) {
            const uint4 v = reinterpret_cast<const uint4 *>(tm)[c];
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                a += (uint32_t)(__popc(__vcmpeq4(w[k], 0x10101010u)) >> 3) + ((uint32_t)(__popc(__vcmpeq4(w[k], 0x08080808u)) >> 3) << 16);
                b += (uint32_t)(__popc(__vcmpeq4(w[k], lowrep)) >> 3);
            }
        }
    } else {
        for (int64_t c = tid; c < chunks; c += blockDim.x)
            for (int k = 0; k < 16; ++k) {
                const uint32_t t = tm[c * 16 + k];
                a += (t == 16u) + ((uint32_t)(t == 8u) << 16);
                b += (t == low);
            }
    }
    a = __reduce_add_sync(0xffffffffu, a);
    b = __reduce_add_sync(0xffffffffu, b);
    __syncthreads();                                                  // sCnt may still be read by a previous call
    if (lane == 0) { sCnt[warp] = a; sCnt[8 + warp] = b; }
    __syncthreads();
    uint32_t sa = 0, sb = 0;
#pragma unroll
    for (int i = 0; i < 8; ++i) { sa += sCnt[i]; sb += sCnt[8 + i]; }
    return make_uint4(sa & 0xFFFFu, sa >> 16, sb, 0u);
}

// ------------------------------------------------------------------------------------------------
// Element types of a cache: binary16 (the paper's FP16) or bfloat16 (reading P20).  The kernels are
// templates on one of these traits; everything that differs between the two formats is an overload below.
// ------------------------------------------------------------------------------------------------
struct ElemF16  { using H = __half;        using H2 = __half2;        static constexpr bool kBf16 = false; };
struct ElemBF16 { using H = __nv_bfloat16; using H2 = __nv_bfloat162; static constexpr bool kBf16 = true; };

__device__ __forceinline__ uint32_t h2u(__half2 h) { return *reinterpret_cast<uint32_t *>(&h); }
__device__ __forceinline__ uint32_t h2u(__nv_bfloat162 h) { return *reinterpret_cast<uint32_t *>(&h); }
template <class H2> __device__ __forceinline__ H2 as_pair(uint32_t u) { return *reinterpret_cast<H2 *>(&u); }
__device__ __forceinline__ __half2 u2h(uint32_t u) { return as_pair<__half2>(u); }
__device__ __forceinline__ __half lo_h(__half2 v) { return __low2half(v); }
__device__ __forceinline__ __half hi_h(__half2 v) { return __high2half(v); }
__device__ __forceinline__ __nv_bfloat16 lo_h(__nv_bfloat162 v) { return __low2bfloat16(v); }
__device__ __forceinline__ __nv_bfloat16 hi_h(__nv_bfloat162 v) { return __high2bfloat16(v); }
__device__ __forceinline__ __half2 pair_h(__half a, __half b) { return __halves2half2(a, b); }
__device__ __forceinline__ __nv_bfloat162 pair_h(__nv_bfloat16 a, __nv_bfloat16 b) { return __halves2bfloat162(a, b); }
__device__ __forceinline__ float to_f(__half a) { return __half2float(a); }
__device__ __forceinline__ float to_f(__nv_bfloat16 a) { return __bfloat162float(a); }
__device__ __forceinline__ float2 to_f2(__half2 a) { return __half22float2(a); }
__device__ __forceinline__ float2 to_f2(__nv_bfloat162 a) { return __bfloat1622float2(a); }
template <class E> __device__ __forceinline__ uint32_t from_f2(float a, float b);
template <> __device__ __forceinline__ uint32_t from_f2<ElemF16>(float a, float b) { return h2u(__floats2half2_rn(a, b)); }
template <> __device__ __forceinline__ uint32_t from_f2<ElemBF16>(float a, float b) { return h2u(__floats2bfloat162_rn(a, b)); }
template <class H> __device__ __forceinline__ H zero_h() { unsigned short z = 0; return *reinterpret_cast<H *>(&z); }

// |x| max of the 8 halves in a uint4 as one half
template <class E>
__device__ __forceinline__ typename E::H absmax8_scalar(const uint4 &v)
{
    using H2 = typename E::H2;
    const H2 m = __hmax2(__hmax2(__habs2(as_pair<H2>(v.x)), __habs2(as_pair<H2>(v.y))),
                         __hmax2(__habs2(as_pair<H2>(v.z)), __habs2(as_pair<H2>(v.w))));
    return __hmax(lo_h(m), hi_h(m));
}

// round-half-even of the EXACT product x*inv (include/skv.h) in one fused multiply-add with the 1.5*2^23 magic
// constant: |x*inv| <= qmax*(1+2^-23) << 2^22, so x*inv + 1.5*2^23 lies in [2^23, 2^24) where binary32 spacing is 1
// and the FMA's single rounding IS round-half-even to an integer (the constant is even, so parity carries over);
// the low bits of the encoding are the two's-complement code and the clamp of the spec is a no-op.
__device__ __forceinline__ uint32_t rne_code_bits(float x, float inv)
{
    return __float_as_uint(__fmaf_rn(x, inv, 12582912.0f));
}

__device__ __forceinline__ uint32_t pack4_bytes(uint32_t a, uint32_t b, uint32_t c, uint32_t d)
{
    const uint32_t ab = __byte_perm(a, b, 0x0040);    // [a.b0, b.b0, -, -]
    const uint32_t cd = __byte_perm(c, d, 0x0040);
    return __byte_perm(ab, cd, 0x5410);               // [a.b0, b.b0, c.b0, d.b0]
}

// 8 fp16 -> 8 INT8 codes (two words): rne_code_bits on packed pairs (FFMA2: two elements per issue slot)
template <class E>
__device__ __forceinline__ uint2 quant8_int8(const uint4 &v, float inv)
{
    using H2 = typename E::H2;
    const float2 inv2 = make_float2(inv, inv), magic = make_float2(12582912.0f, 12582912.0f);
    const float2 a = __ffma2_rn(to_f2(as_pair<H2>(v.x)), inv2, magic), b = __ffma2_rn(to_f2(as_pair<H2>(v.y)), inv2, magic);
    const float2 c = __ffma2_rn(to_f2(as_pair<H2>(v.z)), inv2, magic), d = __ffma2_rn(to_f2(as_pair<H2>(v.w)), inv2, magic);
    return make_uint2(pack4_bytes(__float_as_uint(a.x), __float_as_uint(a.y), __float_as_uint(b.x), __float_as_uint(b.y)),
                      pack4_bytes(__float_as_uint(c.x), __float_as_uint(c.y), __float_as_uint(d.x), __float_as_uint(d.y)));
}

// 8 fp16 -> 8 INT4 codes (one word; element 2k in the low nibble of byte k).  The codes are built in the mantissas of
// packed float pairs by fused multiply-adds (FFMA2: two elements per issue slot):
//     a <- fma(x_hi, inv, M)              M = 1.5 * 2^23;  a = M + q_hi, the FMA's single rounding is RNE(x * inv)
//     a <- fma(a, 256, -255 * M)          exact: M + 256 q_hi   (255 M = 765 * 2^22 is a binary32 number)
//     a <- fma(x_lo, inv, a)              a = M + q_lo + 256 q_hi   (a is an even integer in [2^23, 2^24) before each
//                                         rounding step, so ties keep rounding to even)
// with (x_lo, x_hi) = elements (e, e + 2) in the .x lane and (e + 1, e + 3) in the .y lane.  The codes are signed, so an
// integer add of 0x0808 to the mantissa makes both fields unsigned (q + 8 in 1..15, no borrows between them); one
// bit-select interleaves the two lanes into four nibbles, and q + 8 -> two's-complement nibble is an XOR with 8.
template <class E>
__device__ __forceinline__ uint32_t quant8_int4(const uint4 &v, float inv)
{
    using H2 = typename E::H2;
    const float2 inv2 = make_float2(inv, inv);
    const float2 first = make_float2(12582912.0f, 12582912.0f);                       // M
    const float2 sh = make_float2(256.0f, 256.0f), back = make_float2(-3208642560.0f, -3208642560.0f);   // -255 M
    float2 a = __ffma2_rn(to_f2(as_pair<H2>(v.y)), inv2, first);                      // elements (2, 3)
    float2 b = __ffma2_rn(to_f2(as_pair<H2>(v.w)), inv2, first);                      // elements (6, 7)
    a = __ffma2_rn(a, sh, back);
    b = __ffma2_rn(b, sh, back);
    a = __ffma2_rn(to_f2(as_pair<H2>(v.x)), inv2, a);                                 // elements (0, 1)
    b = __ffma2_rn(to_f2(as_pair<H2>(v.z)), inv2, b);                                 // elements (4, 5)
    // .x holds nibbles 0 and 2 of a half-word (bits 0-3, 8-11), .y nibbles 1 and 3 once shifted up by 4
    const uint32_t h0 = ((__float_as_uint(a.x) + 0x0808u) & 0x0F0Fu) | (((__float_as_uint(a.y) + 0x0808u) << 4) & 0xF0F0u);
    const uint32_t h1 = ((__float_as_uint(b.x) + 0x0808u) & 0x0F0Fu) | (((__float_as_uint(b.y) + 0x0808u) << 4) & 0xF0F0u);
    return __byte_perm(h0, h1, 0x5410) ^ 0x88888888u;
}

// ------------------------------------------------------------------------------------------------
// Transposed group reduction.  A head vector spans LPV lanes; a warp holds NCH chunks (K and V amax of a
// chunk packed in one half2).  Instead of NCH full butterflies, the first log2(NCH) steps halve the set
// of chunks a lane keeps, so the whole reduction costs NCH-1 + log2(LPV/NCH) shuffles.  Afterwards lane
// holds the reduced value of chunk held_chunk(lane); src_lane(lane, u) is a lane that holds chunk u.
// ------------------------------------------------------------------------------------------------
template <int LPV, int NCH>
__device__ __forceinline__ int held_chunk(uint32_t lane)
{
    if (NCH == 4) return (int)(((lane / (LPV / 2)) & 1) * 2 + ((lane / (LPV / 4)) & 1));
    if (NCH == 2) return (int)((lane / (LPV / 2)) & 1);
    return 0;
}
template <int LPV, int NCH>
__device__ __forceinline__ int src_lane(uint32_t lane, int u)
{
    const int base = (int)(lane & ~(uint32_t)(LPV - 1));
    if (NCH == 4) return base + (u >> 1) * (LPV / 2) + (u & 1) * (LPV / 4);
    if (NCH == 2) return base + u * (LPV / 2);
    return base;
}
template <int LPV, int NCH, class H2>
__device__ __forceinline__ H2 group_absmax(H2 (&m)[NCH], uint32_t lane)
{
    H2 v;
    int o = LPV / 2;
    if (NCH == 4) {
        const bool hi = (lane / (LPV / 2)) & 1;
        const H2 keep0 = hi ? m[2] : m[0], keep1 = hi ? m[3] : m[1];
        const H2 send0 = hi ? m[0] : m[2], send1 = hi ? m[1] : m[3];
        const H2 k0 = __hmax2(keep0, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(send0), LPV / 2)));
        const H2 k1 = __hmax2(keep1, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(send1), LPV / 2)));
        const bool hi2 = (lane / (LPV / 4)) & 1;
        const H2 keep = hi2 ? k1 : k0, send = hi2 ? k0 : k1;
        v = __hmax2(keep, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(send), LPV / 4)));
        o = LPV / 8;
    } else if (NCH == 2) {
        const bool hi = (lane / (LPV / 2)) & 1;
        const H2 keep = hi ? m[1] : m[0], send = hi ? m[0] : m[1];
        v = __hmax2(keep, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(send), LPV / 2)));
        o = LPV / 4;
    } else {
        v = m[0];
    }
#pragma unroll
    for (; o >= 1; o >>= 1) v = __hmax2(v, as_pair<H2>(__shfl_xor_sync(0xffffffffu, h2u(v), o)));
    return v;
}

// ------------------------------------------------------------------------------------------------
// dequantise: biased bytes -> f16_rn(fl32(float(q) * scale)); int->float through the 2^23 exponent trick
// ------------------------------------------------------------------------------------------------
template <int BIAS, class E>
__device__ __forceinline__ void dequant4(uint32_t w, float scale, uint32_t &o0, uint32_t &o1)
{
    constexpr float kOff = -(8388608.0f + (float)BIAS);               // -(2^23 + BIAS), exact
    const float2 off = make_float2(kOff, kOff), sc2 = make_float2(scale, scale);
    // packed pairs (FADD2 / FMUL2: two elements per issue slot); per lane the same two roundings as fsub, fmul
    const float2 a = __fmul2_rn(__fadd2_rn(make_float2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7540)),
                                                       __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7541))), off), sc2);
    const float2 b = __fmul2_rn(__fadd2_rn(make_float2(__uint_as_float(__byte_perm(w, 0x4B000000u, 0x7542)),
                                                       __uint_as_float(__byte_perm(w, 0x4B000000u, 0x7543))), off), sc2);
    o0 = from_f2<E>(a.x, a.y);
    o1 = from_f2<E>(b.x, b.y);
}
template <class E>
__device__ __forceinline__ uint4 dequant_int8(uint2 w, float scale)
{
    uint4 o;
    dequant4<128, E>(w.x ^ 0x80808080u, scale, o.x, o.y);
    dequant4<128, E>(w.y ^ 0x80808080u, scale, o.z, o.w);
    return o;
}
template <class E>
__device__ __forceinline__ uint4 dequant_int4(uint32_t w, float scale)
{
    w ^= 0x88888888u;                                   // every nibble becomes q+8
    const uint32_t even = w & 0x0F0F0F0Fu;              // elements 0,2,4,6
    const uint32_t odd = (w >> 4) & 0x0F0F0F0Fu;        // elements 1,3,5,7
    const float2 off = make_float2(-8388616.0f, -8388616.0f), sc2 = make_float2(scale, scale);      // -(2^23 + 8)
    uint32_t o[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {                        // elements 2k (even nibble of byte k) and 2k+1 (odd nibble), as a packed pair
        const float2 f = make_float2(__uint_as_float(__byte_perm(even, 0x4B000000u, 0x7540 + k)),
                                     __uint_as_float(__byte_perm(odd, 0x4B000000u, 0x7540 + k)));
        const float2 y = __fmul2_rn(__fadd2_rn(f, off), sc2);
        o[k] = from_f2<E>(y.x, y.y);
    }
    return make_uint4(o[0], o[1], o[2], o[3]);
}
// ------------------------------------------------------------------------------------------------
// NEXT-4: asymmetric 2-bit low tier (include/skv.h "2-bit quantiser")
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint16_t ld_stream2(const void *p)
{
    uint16_t r;
    asm volatile("ld.global.nc.L1::no_allocate.u16 %0, [%1];" : "=h"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream2(void *p, uint16_t v)
{
    asm volatile("st.global.L1::no_allocate.u16 [%0], %1;" :: "l"(p), "h"(v) : "memory");
}
// (max, -min) of the 8 halves in a uint4: both halves of the result reduce with hmax2
template <class E>
__device__ __forceinline__ typename E::H2 max_negmin8(const uint4 &v)
{
    using H2 = typename E::H2;
    const H2 a = as_pair<H2>(v.x), b = as_pair<H2>(v.y), c = as_pair<H2>(v.z), d = as_pair<H2>(v.w);
    const H2 mx = __hmax2(__hmax2(a, b), __hmax2(c, d));
    const H2 mn = __hmin2(__hmin2(a, b), __hmin2(c, d));
    return pair_h(__hmax(lo_h(mx), hi_h(mx)), __hneg(__hmin(lo_h(mn), hi_h(mn))));
}
// canonical records from a reduced (max, -min): a zero of either sign is stored as +0
template <class H2, class H>
__device__ __forceinline__ void lohi_of(H2 m, H &lo, H &hi)
{
    hi = lo_h(m);
    lo = __hneg(hi_h(m));
    const H z = zero_h<H>();
    if (__heq(hi, z)) hi = z;
    if (__heq(lo, z)) lo = z;
}
template <class H> __device__ __forceinline__ float range_of(H lo, H hi) { return __fsub_rn(to_f(hi), to_f(lo)); }
// 3/r; a bfloat16 range below ~1e-38 overflows the quotient: such vectors are coded as all-zero codes (P20)
__device__ __forceinline__ float inv3_of(float r)
{
    const float q = r != 0.0f ? __fdiv_rn(3.0f, r) : 0.0f;
    return (q <= 3.402823466e38f) ? q : 0.0f;
}
// r/3; a bfloat16 range beyond FLT_MAX (r = +Inf; the encoder's 3/Inf = 0 gave all-zero codes) takes step = 0, so the vector
// decodes to lo instead of fma(0, Inf, lo) = NaN (P20)
__device__ __forceinline__ float step3_of(float r)
{
    const float q = r != 0.0f ? __fdiv_rn(r, 3.0f) : 0.0f;
    return (q <= 3.402823466e38f) ? q : 0.0f;
}
// 8 fp16 -> 8 two-bit codes (16 bits; element k in bits 2k..2k+1).  q_k = rint(fl32(x_k - lo) * inv), the product exact
// and rounded once: the codes are built in the mantissas of ONE packed pair of floats (even elements in .x, odd ones
// in .y) by a chain of packed fused multiply-adds (FFMA2 / FADD2: two elements per issue slot),
//     a <- fma(dx_k, inv, a)      adds q_k (a is an even integer in [2^23, 2^24), so the FMA's rounding is RNE of the product)
//     a <- fma(a, 16, -15*M)      shifts the partial word four bits up (exact), M = 1.5 * 2^23
// which leaves q_0 q_2 q_4 q_6 at bits 0, 4, 8, 12 of a.x and q_1 q_3 q_5 q_7 likewise in a.y; two logic ops interleave them.
template <class E>
__device__ __forceinline__ uint32_t quant8_int2(const uint4 &v, float lo, float inv)
{
    using H2 = typename E::H2;
    // inv = 0 (zero range, or a bfloat16 range / reciprocal beyond binary32, P20) means "all codes 0"; x - lo may be +Inf
    // there, and Inf * 0 is no code, so the subtraction runs against 0 instead (x is finite: x * 0 = 0)
    lo = (inv != 0.0f) ? lo : 0.0f;
    const float2 nlo = make_float2(-lo, -lo), inv2 = make_float2(inv, inv);
    const float2 sh = make_float2(16.0f, 16.0f), back = make_float2(-188743680.0f, -188743680.0f);     // -15 * 1.5 * 2^23
    float2 a = __ffma2_rn(__fadd2_rn(to_f2(as_pair<H2>(v.w)), nlo), inv2, make_float2(12582912.0f, 12582912.0f));
    a = __ffma2_rn(a, sh, back);
    a = __ffma2_rn(__fadd2_rn(to_f2(as_pair<H2>(v.z)), nlo), inv2, a);
    a = __ffma2_rn(a, sh, back);
    a = __ffma2_rn(__fadd2_rn(to_f2(as_pair<H2>(v.y)), nlo), inv2, a);
    a = __ffma2_rn(a, sh, back);
    a = __ffma2_rn(__fadd2_rn(to_f2(as_pair<H2>(v.x)), nlo), inv2, a);
    return (__float_as_uint(a.x) & 0x3333u) | ((__float_as_uint(a.y) & 0x3333u) << 2);
}
// 16 bits of two-bit codes -> 8 fp16: y = f16_rn(fma(q, step, lo)); int -> float through the 2^23 exponent trick (exact),
// the subtraction and the fused multiply-add in packed form
template <class E>
__device__ __forceinline__ uint4 dequant_int2(uint32_t w, float step, float lo)
{
    const float2 off = make_float2(-8388608.0f, -8388608.0f), st2 = make_float2(step, step), lo2 = make_float2(lo, lo);
    uint32_t o[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float2 f = make_float2(__uint_as_float(0x4B000000u | ((w >> (4 * k)) & 3u)), __uint_as_float(0x4B000000u | ((w >> (4 * k + 2)) & 3u)));
        const float2 y = __ffma2_rn(__fadd2_rn(f, off), st2, lo2);
        o[k] = from_f2<E>(y.x, y.y);
    }
    return make_uint4(o[0], o[1], o[2], o[3]);
}

template <class H>
__device__ __forceinline__ float scale_of(H amax, float qmax)
{
    const float af = to_f(amax);
    return af != 0.0f ? __fdiv_rn(af, qmax) : 0.0f;
}
// qmax/amax; only a bfloat16 amax below ~4e-37 can overflow the quotient: such a vector gets all-zero codes (P20)
__device__ __forceinline__ float inv_of(__half amax, float qmax)
{
    const float af = to_f(amax);
    return af != 0.0f ? __fdiv_rn(qmax, af) : 0.0f;
}
__device__ __forceinline__ float inv_of(__nv_bfloat16 amax, float qmax)
{
    const float af = to_f(amax);
    const float q = af != 0.0f ? __fdiv_rn(qmax, af) : 0.0f;
    return (q <= 3.402823466e38f) ? q : 0.0f;
}

}  // namespace skv
