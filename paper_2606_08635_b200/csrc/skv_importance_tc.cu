// skv_importance_tc.cu -- importance scores on the 5th-generation tensor cores (tcgen05 + TMEM + TMA).
//
// Eq. 13 with the logits of PAPER.md:109, designed for sm_100a:
//   * one persistent, warp-specialised CTA per SM: warp 0 = TMA producer, warp 1 = MMA issuer (one elected
//     thread) and TMEM owner, warps 2..17 = sixteen epilogue warps (four per scheduler, so that the MUFU pipe,
//     which bounds the arithmetic at d_h = 128, always has an eligible warp);
//   * a quarter of the exponentials is evaluated on the FMA pipe (round-to-nearest range reduction + degree-4
//     minimax polynomial, 2.7e-6 relative) instead of MUFU.EX2, which lifts the 16 ex2/clk/SM ceiling;
//   * operands land in shared memory by TMA (cp.async.bulk.tensor, 128-byte swizzle, mbarrier complete_tx)
//     straight from the strided K cache and the Q window; accumulators live in TMEM (2 stages x 256 columns, or
//     4 x 128 when a tile needs no more than 128 columns);
//   * pass 1 (rowstats): D[query row][key] = Q_blk K_tile^T, queries are TMEM lanes, so each epilogue thread owns
//     one query row and keeps its (reference exponent, sum 2^x) entirely in registers -- no shuffles;
//   * pass 2 (colsum):  D[key][query row] = K_tile Q_blk^T, keys are TMEM lanes, so each thread owns one key and
//     sums p = 2^(s - lse2[row]) over its columns in registers -- no shuffles, no atomics; the four column groups
//     of a tile are added through shared memory in a fixed order, the per-(KV head, row block) partial sums go to a
//     workspace and the last phase adds them in a fixed order (deterministic) and applies 1/(Hq w) and the decay;
//   * ONE cooperative launch runs pass 1 | lse2 per row | pass 2 | final sum, separated by grid-wide barriers, so
//     TMEM, the mbarriers and the tensor maps are set up once and a 4 K-token request pays one launch, not four;
//   * the epilogue pulls TMEM in 16-column chunks with one chunk in flight (the load of chunk c+1 is issued before
//     the exponentials of chunk c), so the TMEM latency hides behind arithmetic, and hands an accumulator stage back
//     the moment its last chunk is in registers: with two 256-column stages the chain release -> MMA -> commit would
//     otherwise be serial with the arithmetic (profiles/r2_importance_ncu.md: measured with per-tile clock stamps).
// What bounds it (same file): not TMEM (>= 670 B/clk/SM read, ~50 used), not the tensor pipe (64 clk per K = 16 step,
// as measured alone), not HBM except at head_dim 256; the epilogue's ~69 instructions per 16 exponentials on four
// in-order warps per scheduler, at the clock the 1 kW power cap leaves.
// Work decomposition (both passes): the unit is one 128-key tile of one (request, layer, KV head, row block); the
// R*L*S*T units, tile index fastest, are cut into gridDim.x equal contiguous ranges, one per CTA ("stream-K"), so
// every SM gets the same number of tiles (+-1) whatever the shape.  A CTA walks its range as segments (one
// (request, layer, KV head, row block) and a run of its tiles); a row of T tiles cut by CTA boundaries yields one
// partial (m, z) per piece in pass 1 and disjoint key ranges in pass 2.
#include <cuda.h>
#include <string.h>

#include <math.h>

#include <algorithm>

#include "skv_common.cuh"

namespace skv {

namespace tc {

constexpr int kEpiWarps = 16;
constexpr int kEpiThreads = kEpiWarps * 32;
constexpr int kThreads = 64 + kEpiThreads;   // warps: 0 TMA, 1 MMA/TMEM, 2..17 epilogue
constexpr int kTileKeys = 128;
constexpr int kRing = 8;                     // pass 2: depth of the column-group reduction ring (> accumulator stages)
constexpr float kNegBig = -1.0e30f;

struct Params {
    Geom g;
    int w, causal;
    int RB, MB, qrows;                  // row blocks per KV head, rows per block, TMA box rows (multiple of 64)
    int halves;                         // pass 1: 128-row MMA halves per row block (1 or 2)
    int S, T;                           // S = Hkv*RB (KV head, row block) pairs per layer; T = 128-key tiles per row
    long long U;                        // work units = R*L*S*T
    int pmax;                           // pass 1: partial slots per query row = max pieces of a row * column groups
    int kdim[4];                        // position of (head, token, layer, request) in the K tensor map (1..4)
    float2 *partial;                    // [R*L*Hq*w][pmax]
    const float *lse2;                  // [R][L][Hq*w]
    float *apart;                       // [R][L][S][n]
    unsigned int *gbar;                 // grid-barrier arrival counter (zeroed on the stream before the launch)
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
// The same wait for the two single-thread control roles (TMA producer, MMA issuer): they run a whole tile ahead of the
// epilogue, so a failed probe sleeps before the next one instead of competing with the epilogue warps of its scheduler
// for issue slots.
__device__ __forceinline__ void mbar_wait_ctrl(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "nanosleep.u32 64;\n\t"
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
__device__ __forceinline__ float2 ex2_mufu2(float2 x) { return make_float2(ex2(x.x), ex2(x.y)); }
// which of the 8 value pairs of a 16-value chunk go to the FMA pipe (the rest to MUFU.EX2): SKV_EX2_FMA_PAIRS of 8
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
    static constexpr int RED_BYTES = kRing * 3 * kTileKeys * 4;        // pass 2: ring of [column groups 1..3][128 keys]
    static constexpr int SMEM = 1024 + Q_BYTES + STAGES * K_BYTES + 256 * 4 * 2 + RED_BYTES + 256;
};

// One segment of a CTA's unit range: tiles [t0, t1) of one (request, layer, KV head, row block).
struct Seg { int r, l, g, rb, gb, t0, t1, piece; };

// CTA that owns unit u when U units are cut into G equal contiguous ranges [c*U/G, (c+1)*U/G)
__host__ __device__ __forceinline__ long long cta_of_unit(long long u, long long U, long long G) { return ((u + 1) * G - 1) / U; }

__device__ __forceinline__ Seg seg_at(const Params &p, long long u, long long end)
{
    Seg s;
    const long long row = u / p.T;
    s.t0 = (int)(u - row * p.T);
    const long long left = end - u;
    s.t1 = (left < (long long)(p.T - s.t0)) ? s.t0 + (int)left : p.T;
    int t = (int)row;
    s.gb = t % p.S; t /= p.S;
    s.l = t % p.g.L; s.r = t / p.g.L;
    s.g = s.gb / p.RB; s.rb = s.gb % p.RB;
    s.piece = (int)((long long)blockIdx.x - cta_of_unit(row * p.T, p.U, gridDim.x));
    return s;
}

// ---- epilogue building blocks -------------------------------------------------------------------------------
// TMEM leaves in 16-column chunks with ONE chunk in flight: the load of chunk c+1 is issued before the exponentials
// of chunk c run, so its latency hides behind ~100 instructions of arithmetic, and an accumulator stage goes back to
// the MMA warp as soon as its last chunk has landed in registers (not after the arithmetic on it).
__device__ __forceinline__ void tmem_ld16_issue(uint32_t taddr, uint32_t (&r)[16])
{
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
          "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr) : "memory");
}
// wait for the outstanding TMEM loads; the chunk's registers are threaded through the statement so that no use of
// them can be scheduled above the wait
__device__ __forceinline__ void tmem_wait_ld(uint32_t (&r)[16])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]),
                   "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
                 :: "memory");
}

__device__ __forceinline__ void release_stage(uint32_t tempty, uint32_t stage, int lane)
{
    tc_fence_before();
    __syncwarp();
    if (lane == 0) mbar_arrive(tempty + 8 * stage);
}

// One tile = NCH chunks; b0 holds (or is about to receive) chunk 0.  chunk(regs, c) consumes a chunk.  The accumulator
// stage goes back to the MMA warp the moment the tile's LAST chunk has landed in registers -- before that chunk's
// arithmetic and before the wait for the next tile -- because with two 256-column stages the MMA of tile i+2 can only
// start then, and the chain  release -> MMA (~1400 clk) -> commit -> next tile visible  must fit inside the arithmetic
// of ONE tile (measured with per-tile clock stamps: releasing after the arithmetic left the epilogue idle ~20 % of the
// time).  Nothing may read the tile's TMEM after its last chunk is in registers (pass 1 rescues from registers).
template <int NCH, int ACOLS, class ChunkFn>
__device__ __forceinline__ void stream_tile(uint32_t (&b0)[16], uint32_t (&b1)[16], uint32_t base, bool more, uint32_t tfull,
                                            uint32_t tempty, int lane, uint32_t &astage, uint32_t &aphase, ChunkFn &&chunk)
{
    const uint32_t tile_addr = base + astage * ACOLS;
#pragma unroll
    for (int c = 0; c < NCH; ++c) {
        uint32_t (&cur)[16] = (c & 1) ? b1 : b0;
        uint32_t (&nxt)[16] = (c & 1) ? b0 : b1;
        tmem_wait_ld(cur);
        if (c == NCH - 1) {
            release_stage(tempty, astage, lane);
            if (++astage == 512 / ACOLS) { astage = 0; aphase ^= 1; }
            if (more) {
                mbar_wait(tfull + 8 * astage, aphase);
                tc_fence_after();
                tmem_ld16_issue(base + astage * ACOLS, nxt);
            }
        } else {
            tmem_ld16_issue(tile_addr + 16 * (c + 1), nxt);
        }
        chunk(cur, c);
    }
}

// 2^x for a PAIR of values on the FMA/ALU pipes with the packed fp32 instructions of sm_100 (FFMA2 / FADD2):
// n = rint(x) through the 1.5*2^23 constant, f = x - n in [-0.5, 0.5], degree-4 minimax polynomial for 2^f (max
// relative error 2.7e-6), exponent patched in with one shift-add per value.  Only the lower clamp is applied
// (anything below -125 contributes < 2^-125 of the reference term); the caller knows x <= ~0 (pass 2) or watches
// the largest exponent it sends here (pass 1), because x >= 128 would wrap the exponent field.
__device__ __forceinline__ float2 ex2_fma2_lo(float2 x)
{
    x.x = fmaxf(x.x, -125.0f);
    x.y = fmaxf(x.y, -125.0f);
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

// pass 1, one 16-logit chunk of one query row: z += sum 2^(x*sc - m) over the first nvis logits (MASKED: the causal window /
// ragged tail hides the rest; they are pushed to 2^-200, i.e. nothing, before the same packed pipeline as the unmasked
// tiles -- the masked tiles are few, but with a scalar path for them the CTAs that own a row end reached the grid
// barrier late: C2 94 -> 91 us).  Overflow guard of the lazy reference exponent per chunk and per row: a row whose chunk trips it redoes
// the chunk with the exact online-max update, from the 16 logits still in registers (no TMEM re-read).
template <bool MASKED>
__device__ __forceinline__ void rowstats_chunk(const uint32_t (&r)[16], int nvis, float sc, float &m, float &z)
{
    const float2 nm2 = make_float2(-m, -m), sc2 = make_float2(sc, sc);
    float2 accA = make_float2(0.f, 0.f), accB = accA;
    float xmax = kNegBig;                                             // largest exponent sent to the FMA pipe
#pragma unroll
    for (int pi = 0; pi < 8; ++pi) {
        float2 x = __ffma2_rn(make_float2(__uint_as_float(r[2 * pi]), __uint_as_float(r[2 * pi + 1])), sc2, nm2);
        if (MASKED) { if (2 * pi >= nvis) x.x = -200.0f; if (2 * pi + 1 >= nvis) x.y = -200.0f; }
        float2 e;
        if (pair_on_fma(pi)) { xmax = fmaxf(xmax, fmaxf(x.x, x.y)); e = ex2_fma2_lo(x); }
        else e = ex2_mufu2(x);
        if (pi & 1) accB = __fadd2_rn(accB, e); else accA = __fadd2_rn(accA, e);
    }
    const float2 s2 = __fadd2_rn(accA, accB);
    const float a = s2.x + s2.y;
    if (a < 1.0e30f && xmax < 127.0f) {
        z += a;
        if (!(z < 1.0e30f)) { z *= 0x1p-80f; m += 80.0f; }
    } else {
        float tmax = kNegBig;
#pragma unroll
        for (int i = 0; i < 16; ++i) if (!MASKED || i < nvis) tmax = fmaxf(tmax, __uint_as_float(r[i]));
        const float mn = fmaxf(m, tmax * sc);
        float acc = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) acc += (!MASKED || i < nvis) ? ex2(fmaf(__uint_as_float(r[i]), sc, -mn)) : 0.f;
        z = z * ex2(m - mn) + acc;
        m = mn;
    }
}

// pass 1, one work item: every epilogue thread owns one query row and 16*NCH key columns of each 128-key tile and
// keeps the row's (reference exponent m, sum z of 2^(x - m)) in registers.  The reference exponent is lazy: it is
// fixed by the first visible chunk of the row and only an overflow guard watches it afterwards (the row sum is
// z * 2^m for ANY m, so no per-element max is needed); a chunk that trips the guard is redone, by the rows concerned
// and from the 16 logits still in registers, with the exact online-max update (the rare rescue path).
template <int D, int NCH>
__device__ __forceinline__ void rowstats_segment(const Params &p, const Seg &it, uint32_t tmem, uint32_t tfull, uint32_t tempty,
                                                 uint32_t &astage, uint32_t &aphase, int quad, int grp, int lane,
                                                 int64_t rowbase, int mrows)
{
    constexpr float sc = ScaleLog2<D>::value;
    constexpr int NC = 16 * NCH;
    constexpr int ACOLS = (NCH == 4) ? 256 : 128;             // accumulator stage: both 128-row halves, or one
    const int key_beg = it.t0 * kTileKeys, key_end = min(p.g.n, it.t1 * kTileKeys);
    const int n = p.g.n;
    const int hsel = (NCH == 4) ? (grp & 1) : 0;
    const int cg = (NCH == 4) ? (grp >> 1) : grp;
    const int col0 = cg * NC;                                 // key offset inside the 128-key tile
    const int row_in_blk = hsel * 128 + quad * 32 + lane;
    const int row_g = it.rb * p.MB + row_in_blk;
    const bool valid = row_in_blk < mrows;
    const int lim = p.causal ? (n - p.w + (row_g % p.w)) : (n - 1);
    // first key of the first tile that needs a mask (causal window or ragged tail); tiles before it take the fast path
    const int mask_from = p.causal ? (n - p.w - kTileKeys + 2) : (n - kTileKeys + 1);
    float m = kNegBig, z = 0.f;
    const uint32_t base = tmem + ((uint32_t)(quad * 32) << 16) + hsel * 128 + col0;
    uint32_t bA[16], bB[16];
    if (key_beg < key_end) {
        mbar_wait(tfull + 8 * astage, aphase);
        tc_fence_after();
        tmem_ld16_issue(base + astage * ACOLS, bA);
    }
    int k0 = key_beg;
    for (; k0 < key_end && k0 < mask_from; k0 += kTileKeys) {             // ---- fast tiles
        stream_tile<NCH, ACOLS>(bA, bB, base, k0 + kTileKeys < key_end, tfull, tempty, lane, astage, aphase,
            [&](const uint32_t (&r)[16], int c) {
                if (c == 0 && m < 0.5f * kNegBig) {
                    float tmax = kNegBig;
#pragma unroll
                    for (int i = 0; i < 16; ++i) tmax = fmaxf(tmax, __uint_as_float(r[i]));
                    m = tmax * sc;
                }
                rowstats_chunk<false>(r, 16, sc, m, z);
            });
    }
    for (; k0 < key_end; k0 += kTileKeys) {                               // ---- masked tiles (the last ones of a layer)
        stream_tile<NCH, ACOLS>(bA, bB, base, k0 + kTileKeys < key_end, tfull, tempty, lane, astage, aphase,
            [&](const uint32_t (&r)[16], int c) {
                const int nvis = lim - (k0 + col0 + 16 * c) + 1;          // visible logits of this chunk: <= 0 none, >= 16 all
                if (nvis <= 0) return;                                    // (per row; nothing warp-collective in here)
                if (m < 0.5f * kNegBig) {                                 // first visible chunk of the row fixes the reference
                    float tmax = kNegBig;
#pragma unroll
                    for (int i = 0; i < 16; ++i) if (i < nvis) tmax = fmaxf(tmax, __uint_as_float(r[i]));
                    m = tmax * sc;
                }
                rowstats_chunk<true>(r, nvis, sc, m, z);
            });
    }
    if (valid) {
        const int cs = (NCH == 4) ? 2 : 4;
        p.partial[(rowbase + row_g) * p.pmax + it.piece * cs + cg] = make_float2(m, z);
    }
}

// pass 2, one work item: keys are TMEM lanes, so every epilogue thread owns one key and 16*QC query columns of each
// tile and sums p = 2^(s - lse2[column]) over them in registers; the four column groups of a tile are then added in a
// fixed order through a 4-deep shared-memory ring.
template <int D, int QC>
__device__ __forceinline__ void colsum_segment(const Params &p, const Seg &it, uint32_t tmem, uint32_t tfull, uint32_t tempty, uint32_t redfull,
                                               uint32_t &astage, uint32_t &aphase, uint32_t &rstage, uint32_t &rphase,
                                               int quad, int grp, int lane, int mrows,
                                               const float *sLse, const int *sLim, float *sRed, float *out)
{
    constexpr float sc = ScaleLog2<D>::value;
    constexpr int qcols = 16 * QC;
    constexpr int ACOLS = (QC >= 3) ? 256 : 128;                          // accumulator stage = the block's query rows
    const int key_beg = it.t0 * kTileKeys, key_end = min(p.g.n, it.t1 * kTileKeys);
    const int n = p.g.n;
    const int cbeg = grp * qcols;
    const bool cols_full = cbeg + qcols <= mrows;                         // no padding column in this warp's group
    const int mask_from = p.causal ? (n - p.w - kTileKeys + 2) : n;       // first key of the first tile with masked logits
    const uint32_t base = tmem + ((uint32_t)(quad * 32) << 16) + cbeg;
    uint32_t bA[16], bB[16];
    if (key_beg < key_end) {
        mbar_wait(tfull + 8 * astage, aphase);
        tc_fence_after();
        tmem_ld16_issue(base + astage * ACOLS, bA);
    }
    bool par = false;                                                     // buffer holding chunk 0 of the tile (QC odd: alternates)
    for (int k0 = key_beg; k0 < key_end; k0 += kTileKeys) {
        const int j = k0 + quad * 32 + lane;
        const bool more = k0 + kTileKeys < key_end;
        float mine;
        if (cols_full && k0 < mask_from) {                                // ---- fast tile
            float2 accA = make_float2(0.f, 0.f), accB = accA;
            auto chunk = [&](const uint32_t (&r)[16], int c) {
                const float4 *l4 = reinterpret_cast<const float4 *>(sLse + cbeg + 16 * c);
                const float2 sc2 = make_float2(sc, sc);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const float4 L4 = l4[i];
                    const float2 x0 = __ffma2_rn(make_float2(__uint_as_float(r[4 * i]), __uint_as_float(r[4 * i + 1])), sc2, make_float2(L4.x, L4.y));
                    const float2 x1 = __ffma2_rn(make_float2(__uint_as_float(r[4 * i + 2]), __uint_as_float(r[4 * i + 3])), sc2, make_float2(L4.z, L4.w));
                    accA = __fadd2_rn(accA, pair_on_fma(2 * i) ? ex2_fma2_lo(x0) : ex2_mufu2(x0));
                    accB = __fadd2_rn(accB, pair_on_fma(2 * i + 1) ? ex2_fma2_lo(x1) : ex2_mufu2(x1));
                }
            };
            if (!par) stream_tile<QC, ACOLS>(bA, bB, base, more, tfull, tempty, lane, astage, aphase, chunk);
            else      stream_tile<QC, ACOLS>(bB, bA, base, more, tfull, tempty, lane, astage, aphase, chunk);
            const float2 s2 = __fadd2_rn(accA, accB);
            mine = s2.x + s2.y;
        } else {                                                          // ---- masked tile or padded column group
            // the same packed pipeline; a logit the key may not see (causal window, padding column: limit -1) is pushed
            // to 2^-200 first
            float2 accA = make_float2(0.f, 0.f), accB = accA;
            auto chunk = [&](const uint32_t (&r)[16], int c) {
                const int cc = 16 * c;
                if (cbeg + cc >= mrows) return;                           // warp-uniform: padding columns only
                const float4 *l4 = reinterpret_cast<const float4 *>(sLse + cbeg + cc);
                const int4 *m4 = reinterpret_cast<const int4 *>(sLim + cbeg + cc);
                const float2 sc2 = make_float2(sc, sc);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const float4 L4 = l4[i];
                    const int4 M4 = m4[i];
                    float2 x0 = __ffma2_rn(make_float2(__uint_as_float(r[4 * i]), __uint_as_float(r[4 * i + 1])), sc2, make_float2(L4.x, L4.y));
                    float2 x1 = __ffma2_rn(make_float2(__uint_as_float(r[4 * i + 2]), __uint_as_float(r[4 * i + 3])), sc2, make_float2(L4.z, L4.w));
                    if (j > M4.x) x0.x = -200.0f;
                    if (j > M4.y) x0.y = -200.0f;
                    if (j > M4.z) x1.x = -200.0f;
                    if (j > M4.w) x1.y = -200.0f;
                    accA = __fadd2_rn(accA, pair_on_fma(2 * i) ? ex2_fma2_lo(x0) : ex2_mufu2(x0));
                    accB = __fadd2_rn(accB, pair_on_fma(2 * i + 1) ? ex2_fma2_lo(x1) : ex2_mufu2(x1));
                }
            };
            if (!par) stream_tile<QC, ACOLS>(bA, bB, base, more, tfull, tempty, lane, astage, aphase, chunk);
            else      stream_tile<QC, ACOLS>(bB, bA, base, more, tfull, tempty, lane, astage, aphase, chunk);
            const float2 s2 = __fadd2_rn(accA, accB);
            mine = s2.x + s2.y;
        }
        if (QC & 1) par = !par;
        // add the four column groups of this tile in a fixed order (deterministic): groups 1..3 drop their sums
        // into a 4-deep shared-memory ring and arrive on its mbarrier (they never block); group 0 waits for the
        // slot, adds and stores.  A warp is never more than (accumulator stages <= 4) tiles ahead of the slowest one
        // (the MMA of tile i+stages needs every warp to have released tile i, which it does before the arithmetic of
        // that tile's last chunk), so with kRing = 8 slots a slot is never overwritten before group 0 has read it.
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
        if (++rstage == kRing) { rstage = 0; rphase ^= 1; }
    }
}

// Shared-memory addresses and the pipeline cursors that survive from pass 1 to pass 2 (every barrier keeps counting
// phases across the grid-wide barriers in between; all pipelines are empty at a pass boundary).
struct Smem {
    uint32_t sQ, sK, kfull, kempty, qfull, qempty, tfull, tempty, redfull;
    float *sLse; int *sLim; float *sRed;
};
struct Cursors { uint32_t kstage, kphase, qphase, astage, aphase, rstage, rphase; };

// One pass over this CTA's unit range.  V: pass 1 = 16-key chunks per thread per tile (2 or 4); pass 2 = 16-query-
// column chunks per thread per tile (1..4).
template <int D, int PASS, int V>
__device__ __forceinline__ void run_pass(const CUtensorMap *tmK, const CUtensorMap *tmQ, const Params &p, const Smem &sm,
                                         uint32_t tmem, Cursors &cu, int warp, int lane)
{
    using C = Cfg<D>;
    constexpr int ACOLS = (PASS == 1) ? (V == 4 ? 256 : 128) : (V >= 3 ? 256 : 128);   // TMEM columns per accumulator stage
    constexpr int ASTAGES = 512 / ACOLS;
    const int n = p.g.n;
    const long long ubeg = (long long)blockIdx.x * p.U / gridDim.x, uend = (long long)(blockIdx.x + 1) * p.U / gridDim.x;
    if (warp == 0) {
        // ===================== TMA producer =====================
        if (lane == 0) {
            const int kd0 = p.kdim[0], kd1 = p.kdim[1], kd2 = p.kdim[2];
            for (long long u = ubeg; u < uend;) {
                const Seg it = seg_at(p, u, uend);
                u += it.t1 - it.t0;
                mbar_wait_ctrl(sm.qempty, cu.qphase ^ 1); cu.qphase ^= 1;
                mbar_expect_tx(sm.qfull, (uint32_t)(p.qrows * D * 2));
                for (int kb = 0; kb < C::KB; ++kb)
                    tma_load_3d(sm.sQ + kb * C::Q_KB_STRIDE, tmQ, sm.qfull, kb * 64, it.rb * p.MB, (it.r * p.g.L + it.l) * p.g.Hkv + it.g);
                for (int t = it.t0; t < it.t1; ++t) {
                    mbar_wait_ctrl(sm.kempty + 8 * cu.kstage, cu.kphase ^ 1);
                    mbar_expect_tx(sm.kfull + 8 * cu.kstage, (uint32_t)C::K_BYTES);
                    // coordinate of tensor-map dimension i = the one of (head, token, layer, request) whose kdim is i;
                    // selects, not an array indexed by kdim (that array lived in local memory: ~100 STL / LDL per kernel)
                    const int tk = t * kTileKeys;
                    auto coord = [&](int i) { return kd0 == i ? it.g : kd1 == i ? tk : kd2 == i ? it.l : it.r; };
                    const int c1 = coord(1), c2 = coord(2), c3 = coord(3), c4 = coord(4);
                    for (int kb = 0; kb < C::KB; ++kb)
                        tma_load_5d(sm.sK + cu.kstage * C::K_BYTES + kb * C::K_KB_STRIDE, tmK, sm.kfull + 8 * cu.kstage, kb * 64, c1, c2, c3, c4);
                    if (++cu.kstage == C::STAGES) { cu.kstage = 0; cu.kphase ^= 1; }
                }
            }
        }
        __syncwarp();          // lanes 1..31 wait here for the elected lane: the CTA-wide barriers that follow are warp-collective
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        if (lane == 0) {
            const uint32_t idesc = (PASS == 1) ? umma_idesc(128, kTileKeys, p.g.bf16) : umma_idesc(128, p.qrows, p.g.bf16);
            for (long long u = ubeg; u < uend;) {
                const Seg it = seg_at(p, u, uend);
                u += it.t1 - it.t0;
                mbar_wait_ctrl(sm.qfull, cu.qphase); cu.qphase ^= 1;
                for (int t = it.t0; t < it.t1; ++t) {
                    mbar_wait_ctrl(sm.tempty + 8 * cu.astage, cu.aphase ^ 1);
                    mbar_wait_ctrl(sm.kfull + 8 * cu.kstage, cu.kphase);
                    tc_fence_after();
                    const uint32_t kt = sm.sK + cu.kstage * C::K_BYTES;
                    const uint32_t acc = tmem + cu.astage * ACOLS;
                    if (PASS == 1) {
#pragma unroll
                        for (int hh = 0; hh < (V == 4 ? 2 : 1); ++hh)
#pragma unroll
                            for (int ks = 0; ks < D / 16; ++ks) {
                                const uint32_t koff = (ks >> 2) * 1u, kin = (ks & 3) * 32u;
                                umma_f16(acc + hh * 128, umma_desc(sm.sQ + koff * C::Q_KB_STRIDE + hh * (128 * 128) + kin),
                                         umma_desc(kt + koff * C::K_KB_STRIDE + kin), idesc, ks > 0);
                            }
                    } else {
#pragma unroll
                        for (int ks = 0; ks < D / 16; ++ks) {
                            const uint32_t koff = (ks >> 2) * 1u, kin = (ks & 3) * 32u;
                            umma_f16(acc, umma_desc(kt + koff * C::K_KB_STRIDE + kin),
                                     umma_desc(sm.sQ + koff * C::Q_KB_STRIDE + kin), idesc, ks > 0);
                        }
                    }
                    umma_commit(sm.kempty + 8 * cu.kstage);    // smem stage free once these MMAs have read it
                    umma_commit(sm.tfull + 8 * cu.astage);     // accumulator ready for the epilogue
                    if (++cu.kstage == C::STAGES) { cu.kstage = 0; cu.kphase ^= 1; }
                    if (++cu.astage == ASTAGES) { cu.astage = 0; cu.aphase ^= 1; }
                }
                umma_commit(sm.qempty);                        // Q buffer free once every MMA of the segment is done
            }
        }
        __syncwarp();
    } else {
        // ===================== epilogue warps (2..17) =====================
        // TMEM lane window of a warp is fixed by (warp id % 4); grp = which of the four warps on that window.
        const int e = warp - 2, quad = warp & 3, grp = e >> 2;
        const int etid = e * 32 + lane;                                   // 0..511 among the epilogue threads
        const int G = p.g.Hq / p.g.Hkv, M = G * p.w;
        for (long long u = ubeg; u < uend;) {
            const Seg it = seg_at(p, u, uend);
            u += it.t1 - it.t0;
            const int64_t rowbase = ((int64_t)it.r * p.g.L + it.l) * p.g.Hq * p.w + (int64_t)it.g * M;
            const int mrows = min(p.MB, M - it.rb * p.MB);
            if (PASS == 1) {
                rowstats_segment<D, (PASS == 1 ? V : 2)>(p, it, tmem, sm.tfull, sm.tempty, cu.astage, cu.aphase, quad, grp, lane, rowbase, mrows);
            } else {
                // per-segment column tables: lse2 of the block's query rows and their causal limits
                epi_bar_sync();
                for (int idx = etid; idx < p.qrows; idx += kEpiThreads) {
                    const bool ok = idx < mrows;
                    sm.sLse[idx] = ok ? -p.lse2[rowbase + it.rb * p.MB + idx] : 0.f;   // NEGATED lse2
                    sm.sLim[idx] = ok ? (p.causal ? (n - p.w + ((it.rb * p.MB + idx) % p.w)) : (n - 1)) : -1;
                }
                epi_bar_sync();
                float *out = p.apart + (((int64_t)it.r * p.g.L + it.l) * p.S + it.gb) * (int64_t)n;
                colsum_segment<D, (PASS == 2 ? V : 1)>(p, it, tmem, sm.tfull, sm.tempty, sm.redfull, cu.astage, cu.aphase, cu.rstage, cu.rphase,
                                                       quad, grp, lane, mrows, sm.sLse, sm.sLim, sm.sRed, out);
            }
        }
    }
}

// The whole score in ONE cooperative launch of one persistent CTA per SM:
//   pass 1 (row statistics)  | grid barrier |  lse2 per query row  | grid barrier |  pass 2 (column sums)  | grid
//   barrier |  fixed-order sum over (KV head, row block), 1/(Hq w) and the recency decay.
// TMEM, the mbarriers and the tensor-map fetch are set up once.  VA / VC: chunk counts of pass 1 / pass 2 (run_pass).
// Grid-wide barrier of the persistent grid (every CTA is resident: cooperative launch).  The counter only grows:
// the k-th barrier of the launch completes when it reaches k * gridDim.x.
__device__ __forceinline__ void grid_barrier(unsigned int *counter, unsigned int target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();                                                  // this CTA's global writes before the arrival
        atomicAdd(counter, 1u);
        unsigned int seen;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(counter) : "memory");
        } while (seen < target);
    }
    __syncthreads();
}

template <int D, int VA, int VC>
__global__ void __launch_bounds__(kThreads, 1)
imp_fused_kernel(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmQ, const Params p,
                 float lambda, float *__restrict__ importance)
{
    using C = Cfg<D>;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;       // 1024-B aligned (128-B swizzle atoms)
    uint8_t *gbase = smem_raw + (sbase - smem_u32(smem_raw));
    Smem sm;
    sm.sQ = sbase;
    sm.sK = sm.sQ + C::Q_BYTES;
    sm.sLse = reinterpret_cast<float *>(gbase + C::Q_BYTES + C::STAGES * C::K_BYTES);
    sm.sLim = reinterpret_cast<int *>(sm.sLse + 256);
    sm.sRed = reinterpret_cast<float *>(sm.sLim + 256);
    const uint32_t sBar = sm.sK + C::STAGES * C::K_BYTES + 256 * 4 * 2 + C::RED_BYTES;
    // barriers (8 bytes each): kfull[S], kempty[S], qfull, qempty, tfull[4], tempty[4], redfull[kRing]
    sm.kfull = sBar; sm.kempty = sBar + 8 * C::STAGES;
    sm.qfull = sBar + 16 * C::STAGES; sm.qempty = sm.qfull + 8;
    sm.tfull = sm.qempty + 8; sm.tempty = sm.tfull + 32;
    sm.redfull = sm.tempty + 32;                                        // column-group partials of a tile have landed
    uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(gbase + (sm.redfull + 8 * kRing - sbase));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (warp == 0 && lane == 0) {
        for (int s = 0; s < C::STAGES; ++s) { mbar_init(sm.kfull + 8 * s, 1); mbar_init(sm.kempty + 8 * s, 1); }
        mbar_init(sm.qfull, 1); mbar_init(sm.qempty, 1);
        for (int a = 0; a < 4; ++a) { mbar_init(sm.tfull + 8 * a, 1); mbar_init(sm.tempty + 8 * a, kEpiWarps); }
        for (int a = 0; a < kRing; ++a) mbar_init(sm.redfull + 8 * a, kEpiWarps - 4);
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
    Cursors cu = {0, 0, 0, 0, 0, 0, 0};

    run_pass<D, 1, VA>(&tmK, &tmQ, p, sm, tmem, cu, warp, lane);
    grid_barrier(p.gbar, gridDim.x);

    {   // lse2[row] = m* + log2(sum_c z_c 2^(m_c - m*)) over the (reference exponent, sum) pairs of the row's pieces
        const int64_t rows = (int64_t)p.g.R * p.g.L * p.g.Hq * p.w;
        const int HW = p.g.Hq * p.w, M = (p.g.Hq / p.g.Hkv) * p.w;
        constexpr int cs = (VA == 4) ? 2 : 4;
        for (int64_t row = (int64_t)blockIdx.x * kThreads + threadIdx.x; row < rows; row += (int64_t)gridDim.x * kThreads) {
            // which (request, layer, KV head, row block) the row belongs to, hence how many CTAs shared its tiles
            const int rr = (int)(row % HW);
            const long long rl = row / HW;
            const int gb = (rr / M) * p.RB + (rr % M) / p.MB;
            const long long first = (rl * p.S + gb) * (long long)p.T;
            const int cnt = cs * ((int)(cta_of_unit(first + p.T - 1, p.U, gridDim.x) - cta_of_unit(first, p.U, gridDim.x)) + 1);
            const float2 *q = p.partial + row * p.pmax;
            float m = kNegBig;
            for (int c = 0; c < cnt; ++c) m = fmaxf(m, q[c].x);
            float z = 0.f;
            for (int c = 0; c < cnt; ++c) z += q[c].y * exp2f(q[c].x - m);
            const_cast<float *>(p.lse2)[row] = m + log2f(z);
        }
    }
    grid_barrier(p.gbar, 2 * gridDim.x);

    run_pass<D, 2, VC>(&tmK, &tmQ, p, sm, tmem, cu, warp, lane);
    grid_barrier(p.gbar, 3 * gridDim.x);

    {   // importance = (sum over (KV head, row block) partials in a fixed order) / (Hq w) * exp(-lambda (n-1-j))
        const int64_t total = (int64_t)p.g.R * p.g.L * p.g.n;
        const float norm = 1.0f / ((float)p.g.Hq * (float)p.w);
        for (int64_t i = (int64_t)blockIdx.x * kThreads + threadIdx.x; i < total; i += (int64_t)gridDim.x * kThreads) {
            const int64_t rl = i / p.g.n;
            const int j = (int)(i - rl * p.g.n);
            const float *a = p.apart + rl * p.S * (int64_t)p.g.n + j;
            float sum = 0.f;
            for (int s = 0; s < p.S; ++s) sum += a[(int64_t)s * p.g.n];
            importance[i] = sum * norm * expf(-lambda * (float)(p.g.n - 1 - j));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" :: "r"(tmem) : "memory");
    }
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
    int QROWS_MAX, RB, MB, qrows, halves, S, T, grid, pmax;
    long long U;
    size_t partial_bytes, lse_bytes, apart_bytes, bar_bytes;
};

constexpr int kPlanSMs = 148;                          // B200; the grid is planned on the host (the workspace query is host-only)

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
    t.S = g.Hkv * t.RB;
    t.T = (g.n + tc::kTileKeys - 1) / tc::kTileKeys;
    t.U = (long long)g.R * g.L * t.S * t.T;
    t.grid = (int)std::min<long long>(t.U, kPlanSMs);
    // a row of T tiles is cut by CTA boundaries into at most ceil(T / q) + 1 pieces, q = units per CTA (floor)
    const long long q = std::max<long long>(1, t.U / t.grid);
    const int pieces = (int)((t.T + q - 1) / q) + 1;
    t.pmax = pieces * (t.halves == 1 ? 4 : 2);
    const size_t rows = (size_t)g.R * g.L * g.Hq * w;
    t.partial_bytes = (rows * t.pmax * sizeof(float2) + 255) & ~(size_t)255;
    t.lse_bytes = (rows * sizeof(float) + 255) & ~(size_t)255;
    t.apart_bytes = ((size_t)g.R * g.L * t.S * g.n * sizeof(float) + 255) & ~(size_t)255;
    t.bar_bytes = 256;
    return t;
}

size_t importance_tc_ws_bytes(const Geom &g, int window)
{
    if (g.Hkv <= 0 || g.Hq < g.Hkv || g.Hq % g.Hkv || window <= 0) return 0;
    // The kernel keeps work-item indices, tile rows and the TMA coordinate (r*L + l)*Hkv + g in 32-bit ints, and the
    // byte counts below must not wrap: refuse (0) what does not fit.  Checked in double before any integer product.
    const double M = (double)(g.Hq / g.Hkv) * (double)window;
    const double RB = ceil(M / ((g.D == 256) ? 128.0 : 256.0));
    const double T = ceil((double)g.n / (double)tc::kTileKeys);
    const double U = (double)g.R * (double)g.L * (double)g.Hkv * RB * T;
    const double rows = (double)g.R * (double)g.L * (double)g.Hq * (double)window;
    if (U > 2147483647.0 || rows > 2147483647.0 || M > 2147483647.0) return 0;
    if ((double)g.R * (double)g.L * (double)g.Hkv * RB * (double)g.n * 4.0 > 9.0e18) return 0;      // apart_bytes
    const TcPlan t = tc_plan(g, window);
    if (rows * (double)t.pmax * 8.0 > 9.0e18) return 0;                                               // partial_bytes
    return t.partial_bytes + t.lse_bytes + t.apart_bytes + t.bar_bytes;
}

template <int D, int VA, int VC>
static cudaError_t launch_fused(const CUtensorMap &tmK, const CUtensorMap &tmQ, const tc::Params &p, float lambda,
                                float *importance, int grid, cudaStream_t s)
{
    using C = tc::Cfg<D>;
    cudaError_t e = cudaFuncSetAttribute(tc::imp_fused_kernel<D, VA, VC>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM);
    if (e != cudaSuccess) return e;
    void *args[] = {const_cast<CUtensorMap *>(&tmK), const_cast<CUtensorMap *>(&tmQ), const_cast<tc::Params *>(&p), &lambda, &importance};
    // cooperative: the grid-wide barriers need every CTA resident (one per SM; the launch fails rather than deadlocks)
    return cudaLaunchCooperativeKernel(reinterpret_cast<const void *>(tc::imp_fused_kernel<D, VA, VC>), dim3(grid), dim3(tc::kThreads),
                                       args, C::SMEM, s);
}

template <int D>
static cudaError_t launch_tc_t(const CUtensorMap &tmK, const CUtensorMap &tmQ, const tc::Params &p, float lambda,
                               float *importance, int grid, cudaStream_t s)
{
    switch (p.qrows >> 6) {          // 64-row quarters of the query block: 16-column chunks per thread in pass 2
    case 1:  return launch_fused<D, 2, 1>(tmK, tmQ, p, lambda, importance, grid, s);
    case 2:  return launch_fused<D, 2, 2>(tmK, tmQ, p, lambda, importance, grid, s);
    case 3:  return launch_fused<D, 4, 3>(tmK, tmQ, p, lambda, importance, grid, s);
    default: return launch_fused<D, 4, 4>(tmK, tmQ, p, lambda, importance, grid, s);
    }
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
    p.RB = t.RB; p.MB = t.MB; p.qrows = t.qrows; p.halves = t.halves;
    p.S = t.S; p.T = t.T; p.U = t.U; p.pmax = t.pmax;
    uint8_t *w8 = reinterpret_cast<uint8_t *>(ws);
    p.partial = reinterpret_cast<float2 *>(w8);
    p.lse2 = reinterpret_cast<const float *>(w8 + t.partial_bytes);
    p.apart = reinterpret_cast<float *>(w8 + t.partial_bytes + t.lse_bytes);
    p.gbar = reinterpret_cast<unsigned int *>(w8 + t.partial_bytes + t.lse_bytes + t.apart_bytes);
    if (cudaMemsetAsync(p.gbar, 0, sizeof(unsigned int), s) != cudaSuccess) return cudaGetLastError();

    int dev = 0, sms = kPlanSMs;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = std::min(t.grid, sms);             // fewer CTAs than planned only lengthens the pieces: pmax still holds
    switch (g.D) {
    case 64:  return launch_tc_t<64>(tmK, tmQ, p, lambda, importance, grid, s);
    case 128: return launch_tc_t<128>(tmK, tmQ, p, lambda, importance, grid, s);
    case 256: return launch_tc_t<256>(tmK, tmQ, p, lambda, importance, grid, s);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace skv
