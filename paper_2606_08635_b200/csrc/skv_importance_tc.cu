// skv_importance_tc.cu -- importance scores on the 5th-generation tensor cores (tcgen05 + TMEM + TMA).
//
// Same mathematics as skv_importance.cu (Eq. 13; logits PAPER.md:109), re-designed for sm_100a:
//   * one persistent, warp-specialised CTA per SM: warp 0 = TMA producer, warp 1 = MMA issuer (one elected
//     thread) and TMEM owner, warps 2..17 = sixteen epilogue warps (four per scheduler, so that the MUFU pipe,
//     which bounds this kernel at d_h = 128, always has an eligible warp);
//   * a quarter of the exponentials is evaluated on the FMA pipe (round-to-nearest range reduction + degree-4
//     minimax polynomial, 2.7e-6 relative) instead of MUFU.EX2, which lifts the 16 ex2/clk/SM ceiling;
//   * operands land in shared memory by TMA (cp.async.bulk.tensor, 128-byte swizzle, mbarrier complete_tx)
//     straight from the strided K cache and the Q window; accumulators live in TMEM (2 stages x 256 columns);
//   * pass 1 (rowstats): D[query row][key] = Q_blk K_tile^T, queries are TMEM lanes, so each epilogue thread owns
//     one query row and keeps its online (max, sum 2^x) entirely in registers -- no shuffles;
//   * pass 2 (colsum):  D[key][query row] = K_tile Q_blk^T, keys are TMEM lanes, so each thread owns one key and
//     sums p = 2^(s - lse2[row]) over its columns in registers -- no shuffles, no atomics; the four column groups
//     of a tile are added through shared memory in a fixed order, the per-(KV head, row block) partial sums go to a
//     workspace and a small finish kernel adds them in a fixed order (deterministic) and applies 1/(Hq w) and the
//     recency decay.
// A work item is (request, layer, KV head, row block, key chunk); items are dealt round-robin to the CTAs.
#include <cuda.h>
#include <string.h>

#include <algorithm>

#include "skv_common.cuh"

namespace skv {

namespace tc {

constexpr int kEpiWarps = 16;
constexpr int kEpiThreads = kEpiWarps * 32;
constexpr int kThreads = 64 + kEpiThreads;   // warps: 0 TMA, 1 MMA/TMEM, 2..17 epilogue
constexpr int kTileKeys = 128;
constexpr float kNegBig = -1.0e30f;

struct Params {
    Geom g;
    int w, causal;
    int chunk_keys, n_chunks;           // key chunk per work item
    int RB, MB, qrows;                  // row blocks per KV head, rows per block, TMA box rows (multiple of 32)
    int halves;                         // pass 1: 128-row MMA halves per row block (1 or 2)
    int n_items;
    int kdim[4];                        // position of (head, token, layer, request) in the K tensor map (1..4)
    float2 *partial;                    // [rows][pchunks]
    int pchunks;                        // n_chunks * (column groups per row in pass 1: 4 / halves)
    const float *lse2;                  // [R][L][Hq*w]
    float *apart;                       // [R][L][S][n], S = Hkv*RB
    int S;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}"
        :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, uint32_t bar, int c0, int c1, int c2)
{
    asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
                 :: "r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void tma_load_5d(uint32_t dst, const CUtensorMap *tm, uint32_t bar, int c0, int c1, int c2, int c3, int c4)
{
    asm volatile("cp.async.bulk.tensor.5d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6, %7}], [%2];"
                 :: "r"(dst), "l"(tm), "r"(bar), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(c4) : "memory");
}

// K-major, 128-byte-swizzled shared-memory operand descriptor (8-row groups 1024 B apart).
__device__ __forceinline__ uint64_t umma_desc(uint32_t smem_addr)
{
    return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) |
           ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// kind::f16 instruction descriptor: fp16 x fp16 (or bf16 x bf16: a_format / b_format = 1) -> fp32, both operands K-major.
__device__ __forceinline__ uint32_t umma_idesc(int M, int N, int bf16)
{
    return (1u << 4) | (bf16 ? ((1u << 7) | (1u << 10)) : 0u) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        :: "r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32])
{
    uint32_t r[32];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
          "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
          "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 32; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&v)[16])
{
    uint32_t r[16];
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}
__device__ __forceinline__ float ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
// 2^x for a PAIR of values on the FMA/ALU pipes with the packed fp32 instructions of sm_100 (FFMA2 / FADD2):
// n = rint(x) through the 1.5*2^23 constant, f = x - n in [-0.5, 0.5], degree-4 minimax polynomial for 2^f (max
// relative error 2.7e-6), exponent patched in with one shift-add per value.  x is clamped to [-125, 128]: anything
// below contributes < 2^-125 of the row's reference term, anything above yields a value the caller's overflow guard
// (a < 1e30 is false for huge, Inf and NaN) rejects.  6 issue slots per value and no MUFU.
__device__ __forceinline__ float2 ex2_fma2(float2 x)
{
    x.x = fminf(fmaxf(x.x, -125.0f), 128.0f);            // upper clamp: x >= 128 must come out as >= 2^127 / Inf / NaN
    x.y = fminf(fmaxf(x.y, -125.0f), 128.0f);            // (never a wrapped exponent), so the overflow guard sees it
    const float2 t = __fadd2_rn(x, make_float2(12582912.0f, 12582912.0f));
    const float2 nf = __fadd2_rn(t, make_float2(-12582912.0f, -12582912.0f));
    const float2 f = __ffma2_rn(nf, make_float2(-1.0f, -1.0f), x);
    float2 q = __ffma2_rn(f, make_float2(0.009570102207362652f, 0.009570102207362652f), make_float2(0.05591785907745361f, 0.05591785907745361f));
    q = __ffma2_rn(q, f, make_float2(0.240247443318367f, 0.240247443318367f));
    q = __ffma2_rn(q, f, make_float2(0.6931217908859253f, 0.6931217908859253f));
    q = __ffma2_rn(q, f, make_float2(0.9999992847442627f, 0.9999992847442627f));
    return make_float2(__int_as_float(__float_as_int(q.x) + (__float_as_int(t.x) << 23)),
                       __int_as_float(__float_as_int(q.y) + (__float_as_int(t.y) << 23)));
}
__device__ __forceinline__ float2 ex2_mufu2(float2 x) { return make_float2(ex2(x.x), ex2(x.y)); }
// which of the 8 value pairs of a 16-wide group go to the FMA pipe (the rest to MUFU.EX2): kFmaPairs of 8
#ifndef SKV_EX2_FMA_PAIRS
#define SKV_EX2_FMA_PAIRS 2
#endif
__device__ __forceinline__ constexpr bool pair_on_fma(int pi)
{
    return SKV_EX2_FMA_PAIRS == 0 ? false
         : SKV_EX2_FMA_PAIRS == 1 ? (pi & 7) == 3
         : SKV_EX2_FMA_PAIRS == 2 ? (pi & 3) == 1
         : SKV_EX2_FMA_PAIRS == 3 ? ((pi & 7) == 1 || (pi & 7) == 4 || (pi & 7) == 6)
         :                          (pi & 1) == 1;
}
template <int PI> __device__ __forceinline__ float2 ex2_pair(float2 x) { return pair_on_fma(PI) ? ex2_fma2(x) : ex2_mufu2(x); }
// sum of 2^(v*sc + add) over a 16-wide group, two packed accumulators
template <int N>
__device__ __forceinline__ void exp_accumulate(const float (&v)[N], float2 sc2, const float2 (&add2)[N / 2], float2 &accA, float2 &accB)
{
#pragma unroll
    for (int pi = 0; pi < N / 2; ++pi) {
        const float2 x = __ffma2_rn(make_float2(v[2 * pi], v[2 * pi + 1]), sc2, add2[pi]);
        const float2 e = pair_on_fma(pi) ? ex2_fma2(x) : ex2_mufu2(x);
        if (pi & 1) accB = __fadd2_rn(accB, e); else accA = __fadd2_rn(accA, e);
    }
}
template <int D> struct ScaleLog2 {   // log2(e) / sqrt(D) as an immediate
    static constexpr float value = (D == 64) ? 0.18033688011112042f : (D == 128) ? 0.12751743082459868f : 0.09016844005556021f;
};
__device__ __forceinline__ void epi_bar_sync() { asm volatile("bar.sync 1, 512;" ::: "memory"); }

}  // namespace tc

namespace tc {

template <int D> struct Cfg {
    static constexpr int KB = D / 64;                                   // 64-element (128-byte) k-blocks
    static constexpr int QROWS_MAX = (D == 256) ? 128 : 256;
    static constexpr int Q_KB_STRIDE = QROWS_MAX * 128;                 // bytes between k-blocks of the Q buffer
    static constexpr int Q_BYTES = KB * Q_KB_STRIDE;
    static constexpr int K_KB_STRIDE = kTileKeys * 128;
    static constexpr int K_BYTES = KB * K_KB_STRIDE;
    static constexpr int STAGES = (D == 64) ? 6 : (D == 128) ? 4 : 2;
    static constexpr int RED_BYTES = 4 * 3 * kTileKeys * 4;            // pass 2: ring of 4 x [column groups 1..3][128 keys]
    static constexpr int SMEM = 1024 + Q_BYTES + STAGES * K_BYTES + 256 * 4 * 2 + RED_BYTES + 256;
};

struct Item { int r, l, g, rb, chunk, gb; };

__device__ __forceinline__ Item decode_item(const Params &p, int item)
{
    Item it;
    it.chunk = item % p.n_chunks;
    int t = item / p.n_chunks;
    const int GB = p.g.Hkv * p.RB;
    it.gb = t % GB; t /= GB;
    it.l = t % p.g.L; it.r = t / p.g.L;
    it.g = it.gb / p.RB; it.rb = it.gb % p.RB;
    return it;
}

template <int D, int PASS>
__global__ void __launch_bounds__(kThreads, 1)
imp_tc_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmQ, const Params p)
{
    using C = Cfg<D>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;       // 1024-B aligned (128-B swizzle atoms)
    uint8_t *gbase = smem_raw + (sbase - smem_u32(smem_raw));
    const uint32_t sQ = sbase;
    const uint32_t sK = sQ + C::Q_BYTES;
    float *sLse = reinterpret_cast<float *>(gbase + C::Q_BYTES + C::STAGES * C::K_BYTES);
    int *sLim = reinterpret_cast<int *>(sLse + 256);
    float *sRed = reinterpret_cast<float *>(sLim + 256);
    const uint32_t sBar = sK + C::STAGES * C::K_BYTES + 256 * 4 * 2 + C::RED_BYTES;
    // barriers (8 bytes each): kfull[S], kempty[S], qfull, qempty, tfull[2], tempty[2]
    const uint32_t kfull = sBar, kempty = sBar + 8 * C::STAGES;
    const uint32_t qfull = sBar + 16 * C::STAGES, qempty = qfull + 8;
    const uint32_t tfull = qempty + 8, tempty = tfull + 16;
    const uint32_t redfull = tempty + 16;                               // 4 barriers: column-group partials landed
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(gbase + (redfull + 32 - sbase));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = p.g.n;

    if (warp == 0 && lane == 0) {
        for (int s = 0; s < C::STAGES; ++s) { mbar_init(kfull + 8 * s, 1); mbar_init(kempty + 8 * s, 1); }
        mbar_init(qfull, 1); mbar_init(qempty, 1);
        for (int a = 0; a < 2; ++a) { mbar_init(tfull + 8 * a, 1); mbar_init(tempty + 8 * a, kEpiWarps); }
        for (int a = 0; a < 4; ++a) mbar_init(redfull + 8 * a, kEpiWarps - 4);
        fence_barrier_init();
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" :: "r"(smem_u32(tmem_slot)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            uint32_t kstage = 0, kphase = 0, qphase = 0;
            for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
                const Item it = decode_item(p, item);
                mbar_wait(qempty, qphase ^ 1); qphase ^= 1;
                mbar_expect_tx(qfull, (uint32_t)(p.qrows * D * 2));
                for (int kb = 0; kb < C::KB; ++kb)
                    tma_load_3d(sQ + kb * C::Q_KB_STRIDE, &tmQ, qfull, kb * 64, it.rb * p.MB, (it.r * p.g.L + it.l) * p.g.Hkv + it.g);
                const int key_beg = it.chunk * p.chunk_keys, key_end = min(n, key_beg + p.chunk_keys);
                for (int k0 = key_beg; k0 < key_end; k0 += kTileKeys) {
                    mbar_wait(kempty + 8 * kstage, kphase ^ 1);
                    mbar_expect_tx(kfull + 8 * kstage, (uint32_t)C::K_BYTES);
                    int c[5]; c[0] = 0;
                    c[p.kdim[0]] = it.g; c[p.kdim[1]] = k0; c[p.kdim[2]] = it.l; c[p.kdim[3]] = it.r;
                    for (int kb = 0; kb < C::KB; ++kb)
                        tma_load_5d(sK + kstage * C::K_BYTES + kb * C::K_KB_STRIDE, &tmK, kfull + 8 * kstage, kb * 64, c[1], c[2], c[3], c[4]);
                    if (++kstage == C::STAGES) { kstage = 0; kphase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            uint32_t kstage = 0, kphase = 0, qphase = 0, astage = 0, aphase = 0;
            const uint32_t idesc = (PASS == 1) ? umma_idesc(128, kTileKeys, p.g.bf16) : umma_idesc(128, p.qrows, p.g.bf16);
            for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
                const Item it = decode_item(p, item);
                mbar_wait(qfull, qphase); qphase ^= 1;
                const int key_beg = it.chunk * p.chunk_keys, key_end = min(n, key_beg + p.chunk_keys);
                for (int k0 = key_beg; k0 < key_end; k0 += kTileKeys) {
                    mbar_wait(tempty + 8 * astage, aphase ^ 1);
                    mbar_wait(kfull + 8 * kstage, kphase);
                    tc_fence_after();
                    const uint32_t kt = sK + kstage * C::K_BYTES;
                    const uint32_t acc = tmem + astage * 256;
                    if (PASS == 1) {
                        for (int hh = 0; hh < p.halves; ++hh)
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks) {
                                const uint32_t koff = (ks >> 2) * 1u, kin = (ks & 3) * 32u;
                                umma_f16(acc + hh * 128, umma_desc(sQ + koff * C::Q_KB_STRIDE + hh * (128 * 128) + kin),
                                         umma_desc(kt + koff * C::K_KB_STRIDE + kin), idesc, ks > 0);
                            }
                    } else {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            const uint32_t koff = (ks >> 2) * 1u, kin = (ks & 3) * 32u;
                            umma_f16(acc, umma_desc(kt + koff * C::K_KB_STRIDE + kin),
                                     umma_desc(sQ + koff * C::Q_KB_STRIDE + kin), idesc, ks > 0);
                        }
                    }
                    umma_commit(kempty + 8 * kstage);          // smem stage free once these MMAs have read it
                    umma_commit(tfull + 8 * astage);           // accumulator ready for the epilogue
                    if (++kstage == C::STAGES) { kstage = 0; kphase ^= 1; }
                    if (++astage == 2) { astage = 0; aphase ^= 1; }
                }
                umma_commit(qempty);                           // Q buffer free once every MMA of the item is done
            }
        }
    } else {
        // ===================== epilogue warps (2..17) =====================
        // TMEM lane window of a warp is fixed by (warp id % 4); grp = which of the four warps on that window.
        const int e = warp - 2, quad = warp & 3, grp = e >> 2;
        const int etid = e * 32 + lane;                                   // 0..511 among the epilogue threads
        constexpr float sc = ScaleLog2<D>::value;                         // log2(e)/sqrt(d)
        const int G = p.g.Hq / p.g.Hkv, M = G * p.w;
        uint32_t astage = 0, aphase = 0, rstage = 0, rphase = 0;
        for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
            const Item it = decode_item(p, item);
            const int key_beg = it.chunk * p.chunk_keys, key_end = min(n, key_beg + p.chunk_keys);
            const int64_t rowbase = ((int64_t)it.r * p.g.L + it.l) * p.g.Hq * p.w + (int64_t)it.g * M;
            const int mrows = min(p.MB, M - it.rb * p.MB);
            if (PASS == 1) {
                // halves == 2: 2 row halves x 2 column groups of 64 keys; halves == 1: 4 column groups of 32 keys
                const int hsel = (p.halves == 2) ? (grp & 1) : 0;
                const int cg = (p.halves == 2) ? (grp >> 1) : grp;
                const int ncols = (p.halves == 2) ? 64 : 32;
                const int col0 = cg * ncols;                              // key offset inside the 128-key tile
                const int row_in_blk = hsel * 128 + quad * 32 + lane;
                const int row_g = it.rb * p.MB + row_in_blk;
                const bool valid = row_in_blk < mrows;
                const int lim = p.causal ? (n - p.w + (row_g % p.w)) : (n - 1);
                float m = kNegBig, z = 0.f;
                for (int k0 = key_beg; k0 < key_end; k0 += kTileKeys) {
                    mbar_wait(tfull + 8 * astage, aphase);
                    tc_fence_after();
                    const bool need_mask = p.causal ? (k0 + kTileKeys - 1 > n - p.w) : (k0 + kTileKeys > n);
                    const uint32_t taddr = tmem + ((uint32_t)(quad * 32) << 16) + astage * 256 + hsel * 128 + col0;
                    for (int cc = 0; cc < ncols; cc += 32) {
                        float v[32];
                        tmem_ld32(taddr + cc, v);
                        const int j0 = k0 + col0 + cc;
                        float tmax = kNegBig;
                        if (!need_mask) {
                            // lazy reference exponent: m is fixed by the first visible group of the row and only an
                            // overflow guard watches it afterwards (the row sum is z * 2^m for ANY m, so no per-
                            // element max is needed); the exact online-max update below is the rare rescue path.
                            if (m < 0.5f * kNegBig) {
#pragma unroll
                                for (int i = 0; i < 32; ++i) tmax = fmaxf(tmax, v[i]);
                                m = tmax * sc;
                            }
                            float2 nm2[16];
#pragma unroll
                            for (int pi = 0; pi < 16; ++pi) nm2[pi] = make_float2(-m, -m);
                            float2 accA = make_float2(0.f, 0.f), accB = accA;
                            exp_accumulate<32>(v, make_float2(sc, sc), nm2, accA, accB);
                            const float2 s2 = __fadd2_rn(accA, accB);
                            const float a = s2.x + s2.y;
                            if (a < 1.0e30f) {
                                z += a;
                                if (!(z < 1.0e30f)) { z *= 0x1p-80f; m += 80.0f; }
                            } else {                                      // a term overflowed: redo the group exactly
#pragma unroll
                                for (int i = 0; i < 32; ++i) tmax = fmaxf(tmax, v[i]);
                                const float mn = fmaxf(m, tmax * sc);
                                float acc = 0.f;
#pragma unroll
                                for (int i = 0; i < 32; ++i) acc += ex2(fmaf(v[i], sc, -mn));
                                z = z * ex2(m - mn) + acc;
                                m = mn;
                            }
                        } else {
#pragma unroll
                            for (int i = 0; i < 32; ++i) if (j0 + i <= lim) tmax = fmaxf(tmax, v[i]);
                            const float mn = fmaxf(m, tmax > 0.5f * kNegBig ? tmax * sc : kNegBig);
                            float acc = 0.f;
#pragma unroll
                            for (int i = 0; i < 32; ++i) acc += (j0 + i <= lim) ? ex2(fmaf(v[i], sc, -mn)) : 0.f;
                            z = z * ex2(m - mn) + acc;
                            m = mn;
                        }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty + 8 * astage);
                    if (++astage == 2) { astage = 0; aphase ^= 1; }
                }
                if (valid) {
                    const int cs = (p.halves == 2) ? 2 : 4;
                    p.partial[(rowbase + row_g) * p.pchunks + it.chunk * cs + cg] = make_float2(m, z);
                }
            } else {
                // per-item column tables: lse2 of the block's query rows and their causal limits
                epi_bar_sync();
                for (int idx = etid; idx < p.qrows; idx += kEpiThreads) {
                    const bool ok = idx < mrows;
                    sLse[idx] = ok ? -p.lse2[rowbase + it.rb * p.MB + idx] : 0.f;      // NEGATED lse2
                    sLim[idx] = ok ? (p.causal ? (n - p.w + ((it.rb * p.MB + idx) % p.w)) : (n - 1)) : -1;
                }
                epi_bar_sync();
                const int qcols = p.qrows >> 2;                           // query columns per group: 16, 32, 48 or 64
                const int cbeg = grp * qcols;
                float *out = p.apart + (((int64_t)it.r * p.g.L + it.l) * p.S + it.gb) * (int64_t)n;
                for (int k0 = key_beg; k0 < key_end; k0 += kTileKeys) {
                    mbar_wait(tfull + 8 * astage, aphase);
                    tc_fence_after();
                    const int j = k0 + quad * 32 + lane;
                    const bool tile_mask = p.causal && (k0 + kTileKeys - 1 > n - p.w);
                    const uint32_t taddr = tmem + ((uint32_t)(quad * 32) << 16) + astage * 256 + cbeg;
                    float2 accA = make_float2(0.f, 0.f), accB = accA;
                    float s0 = 0.f;
                    for (int cc = 0; cc < qcols; cc += 16) {
                        if (cbeg + cc >= mrows) break;                    // warp-uniform: only padding columns left
                        float v[16];
                        tmem_ld16(taddr + cc, v);
                        if (!tile_mask && cbeg + cc + 16 <= mrows) {
                            const float4 *l4 = reinterpret_cast<const float4 *>(sLse + cbeg + cc);
                            float2 nl2[8];
#pragma unroll
                            for (int i = 0; i < 4; ++i) {
                                const float4 L4 = l4[i];
                                nl2[2 * i] = make_float2(L4.x, L4.y);
                                nl2[2 * i + 1] = make_float2(L4.z, L4.w);
                            }
                            exp_accumulate<16>(v, make_float2(sc, sc), nl2, accA, accB);
                        } else {
                            const int *lim = sLim + cbeg + cc;
#pragma unroll
                            for (int i = 0; i < 16; ++i)
                                s0 += (j <= lim[i]) ? ex2(fmaf(v[i], sc, sLse[cbeg + cc + i])) : 0.f;
                        }
                    }
                    const float2 s2 = __fadd2_rn(accA, accB);
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(tempty + 8 * astage);
                    if (++astage == 2) { astage = 0; aphase ^= 1; }
                    // add the four column groups of this tile in a fixed order (deterministic): groups 1..3 drop
                    // their sums into a 4-deep shared-memory ring and arrive on its mbarrier (they never block);
                    // group 0 waits for the slot, adds and stores.  Ring depth 4 > the 2 TMEM stages any warp can
                    // run ahead, so a slot is never overwritten before group 0 has read it.
                    const float mine = (s2.x + s2.y) + s0;
                    float *red = sRed + rstage * (3 * kTileKeys);
                    if (grp != 0) {
                        red[(grp - 1) * kTileKeys + quad * 32 + lane] = mine;
                        __syncwarp();
                        if (lane == 0) mbar_arrive(redfull + 8 * rstage);
                    } else {
                        mbar_wait(redfull + 8 * rstage, rphase);
                        const int k = quad * 32 + lane;
                        if (j < n) out[j] = (mine + red[k]) + (red[kTileKeys + k] + red[2 * kTileKeys + k]);
                    }
                    if (++rstage == 4) { rstage = 0; rphase ^= 1; }
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tmem) : "memory");
    }
}

__global__ void __launch_bounds__(256)
imp_finish_kernel(Geom g, int w, float lambda, int S, const float *__restrict__ apart, float *__restrict__ importance)
{
    const int l = blockIdx.y, r = blockIdx.z;
    const int j = blockIdx.x * 256 + threadIdx.x;
    if (j >= g.n) return;
    const float *a = apart + (((int64_t)r * g.L + l) * S) * (int64_t)g.n + j;
    float sum = 0.f;
    for (int s = 0; s < S; ++s) sum += a[(int64_t)s * g.n];            // fixed order: deterministic
    const float norm = 1.0f / ((float)g.Hq * (float)w);
    importance[((int64_t)r * g.L + l) * g.n + j] = sum * norm * expf(-lambda * (float)(g.n - 1 - j));
}

}  // namespace tc

// ------------------------------------------------------------------------------------------------
// host side: tensor maps, work decomposition, launches
// ------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn get_encode_fn()
{
    void *fn = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
        return nullptr;
    return (EncodeTiledFn)fn;
}

struct TcPlan {
    int QROWS_MAX, RB, MB, qrows, halves, chunk_keys, n_chunks, pchunks, S, n_items;
    size_t partial_bytes, lse_bytes, apart_bytes;
};

static TcPlan tc_plan(const Geom &g, int w)
{
    TcPlan t;
    const int M = (g.Hq / g.Hkv) * w;
    t.QROWS_MAX = (g.D == 256) ? 128 : 256;
    t.RB = (M + t.QROWS_MAX - 1) / t.QROWS_MAX;
    int mb = (M + t.RB - 1) / t.RB;
    mb = ((mb + 63) / 64) * 64;
    if (mb > t.QROWS_MAX) mb = t.QROWS_MAX;
    t.MB = (t.RB == 1) ? M : mb;
    t.qrows = ((std::min(t.MB, M) + 63) / 64) * 64;
    t.halves = t.qrows > 128 ? 2 : 1;
    const long long triples = (long long)g.R * g.L * g.Hkv * t.RB;
    // Key chunk per work item: items are dealt round-robin to one persistent CTA per SM, so the cost of a candidate
    // chunk size is (rounds of items) x (tiles per item + ~3 tiles of per-item overhead: Q load, pipeline fill and
    // drain).  Candidates are multiples of 128 keys from 512 up; ties go to the larger chunk (fewer partials).
    const int npad = ((g.n + 127) / 128) * 128;
    constexpr long long kSMs = 148;                     // B200; also used by the host-only workspace query
    int ck = npad;
    long long best = -1;
    for (int c = std::min(512, npad); c <= npad; c += 128) {
        const long long chunks = (g.n + c - 1) / c;
        const long long rounds = (triples * chunks + kSMs - 1) / kSMs;
        const long long cost = rounds * (c / 128 + 3);
        if (best < 0 || cost <= best) { best = cost; ck = c; }
    }
    t.chunk_keys = ck;
    t.n_chunks = (g.n + ck - 1) / ck;
    t.pchunks = t.n_chunks * (t.halves == 1 ? 4 : 2);
    t.S = g.Hkv * t.RB;
    const long long items = triples * t.n_chunks;
    t.n_items = items > 0x7FFFFFFFll ? -1 : (int)items;                 // -1: does not fit (reported as unsupported)
    const size_t rows = (size_t)g.R * g.L * g.Hq * w;
    t.partial_bytes = (rows * t.pchunks * sizeof(float2) + 255) & ~(size_t)255;
    t.lse_bytes = (rows * sizeof(float) + 255) & ~(size_t)255;
    t.apart_bytes = (size_t)g.R * g.L * t.S * g.n * sizeof(float);
    return t;
}

size_t importance_tc_ws_bytes(const Geom &g, int window)
{
    if (g.Hkv <= 0 || g.Hq < g.Hkv || g.Hq % g.Hkv || window <= 0) return 0;
    const TcPlan t = tc_plan(g, window);
    if (t.n_items < 0) return 0;
    return t.partial_bytes + t.lse_bytes + t.apart_bytes;
}

// lse2[row] = M + log2(sum_c z_c 2^(m_c - M)) over the row's partial (max, sum) pairs
__global__ void imp_tc_combine_kernel(const float2 *__restrict__ partial, int n_chunks, int64_t rows, float *__restrict__ lse2)
{
    const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (row >= rows) return;
    const float2 *q = partial + row * n_chunks;
    float m = tc::kNegBig;
    for (int c = 0; c < n_chunks; ++c) m = fmaxf(m, q[c].x);
    float z = 0.f;
    for (int c = 0; c < n_chunks; ++c) z += q[c].y * exp2f(q[c].x - m);
    lse2[row] = m + log2f(z);
}

template <int D>
static cudaError_t launch_tc_t(const Geom &g, const CUtensorMap &tmK, const CUtensorMap &tmQ, tc::Params p, float lambda,
                               float *importance, int sms, cudaStream_t s)
{
    using C = tc::Cfg<D>;
    cudaError_t e;
    if ((e = cudaFuncSetAttribute(tc::imp_tc_kernel<D, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM)) != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(tc::imp_tc_kernel<D, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM)) != cudaSuccess) return e;
    const int grid = std::min(p.n_items, sms);
    tc::imp_tc_kernel<D, 1><<<grid, tc::kThreads, C::SMEM, s>>>(tmK, tmQ, p);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    const int64_t rows = (int64_t)g.R * g.L * g.Hq * p.w;
    imp_tc_combine_kernel<<<(unsigned)((rows + 255) / 256), 256, 0, s>>>(p.partial, p.pchunks, rows, const_cast<float *>(p.lse2));
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    tc::imp_tc_kernel<D, 2><<<grid, tc::kThreads, C::SMEM, s>>>(tmK, tmQ, p);
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    dim3 gf((g.n + 255) / 256, g.L, g.R);
    tc::imp_finish_kernel<<<gf, 256, 0, s>>>(g, p.w, lambda, p.S, p.apart, importance);
    return cudaGetLastError();
}

// Returns cudaErrorNotSupported when the tensor maps cannot be built (reported as SKV_ERR_CUDA; there is no other path).
cudaError_t launch_importance_tc(const Geom &g, const __half *K, const __half *Q, int window, int causal, float lambda,
                                 float *importance, void *ws, cudaStream_t s)
{
    static EncodeTiledFn encode = get_encode_fn();
    if (!encode) return cudaErrorNotSupported;
    const TcPlan t = tc_plan(g, window);
    const int M = (g.Hq / g.Hkv) * window;

    // K: dim 0 = head_dim (contiguous); the other four dims ordered by ascending stride
    struct Dim { int which; uint64_t size; uint64_t stride; };
    Dim d[4] = {{0, (uint64_t)g.Hkv, (uint64_t)g.sh}, {1, (uint64_t)g.n, (uint64_t)g.st},
                {2, (uint64_t)g.L, (uint64_t)g.sl}, {3, (uint64_t)g.R, (uint64_t)g.sr}};
    for (int i = 0; i < 4; ++i) if (d[i].stride < 8) d[i].stride = 8;
    std::stable_sort(d, d + 4, [](const Dim &a, const Dim &b) { return a.stride < b.stride; });
    tc::Params p;
    memset(&p, 0, sizeof(p));
    cuuint64_t kdims[5] = {(cuuint64_t)g.D, 0, 0, 0, 0}, kstr[4];
    cuuint32_t kbox[5] = {64, 1, 1, 1, 1}, ones[5] = {1, 1, 1, 1, 1};
    for (int i = 0; i < 4; ++i) {
        kdims[i + 1] = d[i].size;
        kstr[i] = d[i].stride * 2;
        if (d[i].which == 1) kbox[i + 1] = tc::kTileKeys;
        p.kdim[d[i].which] = i + 1;
    }
    CUtensorMap tmK, tmQ;
    const CUtensorMapDataType et = g.bf16 ? CU_TENSOR_MAP_DATA_TYPE_BFLOAT16 : CU_TENSOR_MAP_DATA_TYPE_FLOAT16;
    if (encode(&tmK, et, 5, const_cast<__half *>(K), kdims, kstr, kbox, ones,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;
    cuuint64_t qdims[3] = {(cuuint64_t)g.D, (cuuint64_t)M, (cuuint64_t)g.R * g.L * g.Hkv};
    cuuint64_t qstr[2] = {(cuuint64_t)g.D * 2, (cuuint64_t)M * g.D * 2};
    cuuint32_t qbox[3] = {64, (cuuint32_t)t.qrows, 1};
    if (encode(&tmQ, et, 3, const_cast<__half *>(Q), qdims, qstr, qbox, ones,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;

    p.g = g; p.w = window; p.causal = causal;
    p.chunk_keys = t.chunk_keys; p.n_chunks = t.n_chunks; p.RB = t.RB; p.MB = t.MB; p.qrows = t.qrows;
    p.halves = t.halves; p.n_items = t.n_items; p.pchunks = t.pchunks; p.S = t.S;
    uint8_t *w8 = reinterpret_cast<uint8_t *>(ws);
    p.partial = reinterpret_cast<float2 *>(w8);
    p.lse2 = reinterpret_cast<const float *>(w8 + t.partial_bytes);
    p.apart = reinterpret_cast<float *>(w8 + t.partial_bytes + t.lse_bytes);

    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    switch (g.D) {
    case 64:  return launch_tc_t<64>(g, tmK, tmQ, p, lambda, importance, sms, s);
    case 128: return launch_tc_t<128>(g, tmK, tmQ, p, lambda, importance, sms, s);
    case 256: return launch_tc_t<256>(g, tmK, tmQ, p, lambda, importance, sms, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace skv
