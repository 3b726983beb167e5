/*
 * skv.h -- C ABI of the B200-native SpectrumKV per-token mixed-precision KV transfer path
 * (arxiv/paper_2606_08635; citations are /root/reference/PAPER.md:<line>).
 *
 * The library implements Algorithm 1 steps 2-4 and the decode-side
 * dequantisation as hand-written CUDA for sm_100a:
 *
 *   skv_importance    Alg. 1 step 2, Eq. 13: I_j = A_j exp(-lambda Delta_j), A_j = softmax
 *                     mass of the last-w prompt queries on key j (logits q.k/sqrt(d)),
 *                     averaged over query heads and window queries
 *   skv_importance_kvnorm   the "KV-norm fallback" of Alg. 1 step 2
 *   skv_tier_counts   Eq. 2-3, Eq. 14-15, SinkProtect,
 *                     2-tier fallback with drop: budget b -> (n16, n8, n4, n0)
 *   skv_assign_tiers  Alg. 1 step 3, Prop. 1: pin protected positions to
 *                     FP16, rank the rest by (importance desc, position asc)
 *   skv_pack          Alg. 1 step 4: quantise K and V independently per the tier map
 *                     ("standard symmetric") and compact into one SKV1 blob
 *   skv_unpack        PAPER.md:202: dequantise and scatter back into a dense FP16 cache
 *   skv_blob_check    decode-side validation of a received blob header (host)
 *   skv_unpack_patch  cold-tier precision upgrade: apply an upgrade blob to a dense cache in place
 *
 * Conventions
 *   - Every pointer is tagged HOST or DEVICE.  DEVICE pointers are plain CUDA device addresses
 *     (e.g. torch.Tensor.data_ptr()); the library never allocates, frees or keeps them.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All work is
 *     enqueued on that stream; no entry point synchronises the host, so a sequence of calls can be captured into a
 *     CUDA graph (tests: test_whole_path_is_cuda_graph_capturable).  Launches per call: skv_importance 1 (cooperative:
 *     it needs the whole GPU, one CTA per SM) + one 4-byte memset node (the grid-barrier counter); skv_assign_tiers 1; skv_pack / skv_unpack 1 for
 *     n_tokens <= 8192 and 2 (slot scan first) beyond or for sparse upgrade blobs; skv_importance_kvnorm 2.
 *   - Every entry returns SKV_OK (0) or a negative skv_status and launches nothing on error.
 *   - The library keeps no mutable global state and is re-entrant.  (Two process-wide constants are set idempotently:
 *     the driver entry point of the tensor-map encoder is looked up once and cached, and kernels that need more than
 *     48 KiB of dynamic shared memory always request the same fixed maximum.)  The one exception is
 *     skv_importance_kvnorm_noalloc, the entry point for callers that cannot allocate: its scratch is a fixed array
 *     inside the library that all its calls on a GPU share (see its declaration for the rules that follow from that).
 *   - fp16 = IEEE binary16.  K/V inputs must be finite (NaN/Inf is undefined behaviour).
 *   - With skv_shape.dtype = SKV_BF16 every "fp16" below reads bfloat16 (caches, queries, amax / (lo, hi) records,
 *     dequantised output); the byte model is unchanged (2 bytes per element).  Only difference in the arithmetic: a
 *     quotient qmax/amax (or 3/r) that overflows binary32 -- possible only for a bfloat16 amax below ~4e-37 -- is
 *     replaced by 0, i.e. such a vector gets all-zero codes (reading P20 of DESIGN.md).
 *
 * Tier codes (bits per element): 16 = FP16, 8 = INT8, 4 = INT4, 0 = dropped (c = 0).
 *
 * Wire format "SKV1" (little endian; one self-contained blob per request; a batch is R blobs back to
 * back at stride skv_blob_bytes(); the paper only says "mixed-precision payload"):
 *
 *   [0,256)  header: 0 u32 magic 0x31564B53 ("SKV1"), 4 u32 version = 1, 8 u32 L, 12 u32 Hkv, 16 u32 d_h,
 *            20 u32 n, 24 u32 n16, 28 u32 n8, 32 u32 n4, 36 u32 n0, 40 u32 flags (bit0 = allow_int4, bit1 = 2-bit low tier,
 *            bit2 = bfloat16, bit3 = INT8 hot tier, bit4 = 2-bit tier quantised in groups of 32 elements),
 *            44 u32 0, 48 u64 budget in quarter-units, 56 u64 tier_map_off (= 256), 64 u64 layer0_off,
 *            72 u64 layer_stride, 80 u64 seg_off[10] (relative to the layer block), 160 u64 total_bytes,
 *            168..255 zero
 *   [256,..) tier map u8[L][n], zero padded to a multiple of 256 B
 *   layer l at layer0_off + l*layer_stride: ten segments, each starting on a 256-B boundary, pads zero:
 *            K16,V16 : f16 [n16][Hkv][d_h]     K8,V8 : i8 [n8][Hkv][d_h]     K4,V4 : u8 [n4][Hkv][d_h/2]
 *            SK8,SV8 : f16 amax [n8][Hkv]      SK4,SV4 : f16 amax [n4][Hkv]
 *   Slot order inside a tier = ascending token position.  INT4 byte i holds element 2i in the low nibble
 *   and 2i+1 in the high nibble (4-bit two's complement).  Dropped tokens occupy no bytes.
 *
 * 2-bit low tier (NEXT-4; "the INT4 tier could use KIVI-style asymmetric 2-bit quantization"): with
 * allow_int4 = 2 the low tier of a blob is coded in 2 bits instead of 4.  Its tier code is 2, header flags = 3,
 * K4/V4 hold four codes per byte (element 4i+k in bits 2k..2k+1 of byte i), SK4/SV4 hold an fp16 (lo, hi) pair per
 * head vector, and the budget runs in EIGHTH-units (8 / 4 / 1 / 0 per token; budget_q4 and spent_q4 are then
 * eighths).  Quantiser: lo = min x, hi = max x (a zero of either sign recorded as +0), r = fl32(hi - lo),
 * inv = fl32(3/r), step = fl32(r/3) (0 when r = 0); q = clamp(rint(fl32(x - lo) * inv), 0, 3), the product exact and
 * rounded once, half to even; y = f16_rn(fma(q, step, lo)).
 *
 * INT8 hot tier (NEXT-4; "the FP16 tier could be further compressed to INT8 (if the model is INT8-safe for high-
 * importance tokens)"; reading P21 of DESIGN.md): with tier_mode bit0 (SKV_MODE_HOT_INT8) nothing ships
 * at FP16.  n16 = 0, the protected positions are pinned to -- and paid at -- INT8 (tier code 8), and the greedy ladder
 * of Eq. 14 runs over the costs 1/2 and 1/4 (1/2 and 1/8 with the 2-bit low tier): R = Q - 2P, m = n - P;
 * R >= 2m: all INT8 (every b >= 1/2); m <= R < 2m: n8 = P + (R - m), n4 = 2m - R; R < m: n8 = P, n4 = R, rest dropped;
 * 2-tier: n8 = P + floor(R/2), rest dropped.  Header flags bit3; K16 / V16 are empty.
 *
 * Group-wise 2-bit low tier (NEXT-4; "KIVI partitions keys and values into separate quantization groups",
 * PAPER.md:623; reading P22): with tier_mode bit1 (SKV_MODE_GROUP2, needs allow_int4 = 2) the 2-bit quantiser above
 * runs on every group of 32 consecutive elements of a head vector instead of on the whole vector (token-local, so a
 * token stays self-contained on the wire); SK4 / SV4 hold d_h/32 (lo, hi) pairs per head vector, in element order.
 * Header flags bit4.  The records cost 1 bit per element on top of the 2 bits of code (scale overhead outside b, as
 * for every tier): a 2-bit token takes 3 bits per element on the wire instead of 2.25 (d_h = 128) or 2.125 (d_h = 256).
 *
 * Quantiser (one group = one head vector of d_h values; qmax = 127 / 7):
 *   amax = max|x| (an fp16 value, stored as the 2-byte scale record);
 *   inv = fl32(qmax/amax), scale = fl32(amax/qmax)   (both 0 when amax = 0);
 *   q = clamp(rint(x*inv), -qmax, qmax): the real product of the fp16 x and the fp32 inv, rounded ONCE, half to
 *   even (a 35-bit product, so no intermediate binary32 rounding);   y = f16_rn(fl32(q*scale)).
 */
#ifndef SKV_H_
#define SKV_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    SKV_OK = 0,
    SKV_ERR_INVALID_ARG = -1,       /* null pointer, dims <= 0, Hq % Hkv != 0, window outside [1,n], b <= 0 or NaN,
                                       range outside [0,n] or begin > end; counts that do not add up to n, carry a
                                       low tier without the allow_int4 flag, or spend more than their budget (such a
                                       blob would fail skv_blob_check); an OUTPUT cache whose layer / request stride
                                       is 0 with more than one layer / request (overlapping writes) */
    SKV_ERR_UNSUPPORTED = -2,       /* head_dim not in {64,128,256}; stride_token/stride_head/stride_layer/
                                       stride_request not multiples of 8 elements; pointer (cache, queries or
                                       workspace) not 16-B aligned (blob: 256-B); skv_importance only: stride_layer = 0
                                       with more than one layer or stride_request = 0 with more than one request (the
                                       tensor map has no broadcast stride); n_tokens > 2^20 (the slot scan packs three 21-bit counters in a word);
                                       n_layers * n_requests > 65535 (grid dimension of the per-layer kernels);
                                       more than 32 disjoint protected intervals after merging sinks and ranges */
    SKV_ERR_BUDGET_INFEASIBLE = -3, /* protected tokens alone exceed the budget (4P > floor(4bn)) */
    SKV_ERR_BUFFER_TOO_SMALL = -4,  /* blob capacity or workspace */
    SKV_ERR_BAD_BLOB = -5,          /* skv_blob_check: magic / version / dims / offsets / total_bytes mismatch */
    SKV_ERR_CUDA = -6,              /* a CUDA runtime call or kernel launch failed */
    SKV_ERR_NOALLOC_LIMIT = -7      /* skv_importance_kvnorm_noalloc only: the problem needs more scratch than the
                                       SKV_NOALLOC_SCRATCH_BYTES built into the library; use skv_importance_kvnorm
                                       with a workspace of your own, or split the batch */
} skv_status;

/* One batch of dense caches.  Strides are in ELEMENTS (fp16) and apply to both K and V; the head
 * dimension is contiguous.  Token-major default: stride_head = d_h, stride_token = Hkv*d_h,
 * stride_layer = n*Hkv*d_h, stride_request = L*n*Hkv*d_h.  The HF layout [L][Hkv][n][d_h] is
 * stride_token = d_h, stride_head = n*d_h.  All requests of a batch have the same n_tokens. */
typedef struct {
    int32_t n_layers, n_q_heads, n_kv_heads, head_dim, n_tokens, n_requests;
    int64_t stride_request, stride_layer, stride_token, stride_head;
    int32_t dtype;            /* element type of K, V, Q and of the scale records: 0 = fp16 (SKV_F16, the paper's
                                 cache), 1 = bfloat16 (SKV_BF16, NEXT-4); header flags bit2 */
    int32_t reserved;         /* must be 0 */
} skv_shape;
#define SKV_F16 0
#define SKV_BF16 1

/* Transfer policy (PAPER.md:51-58 b; :216, :230 sinks; :25 protected positions; :234 allow_int4). */
typedef struct {
    double  budget;           /* b in (0,1]; values > 1 are clamped to 1 */
    int32_t n_sink;           /* s: positions [0,s) forced FP16 */
    int32_t n_ranges;         /* number of protected ranges */
    const int32_t *ranges;    /* HOST, n_ranges x [begin,end) half-open, forced FP16; read during the call only */
    int32_t allow_int4;       /* probe result: 1 = 3-tier, 0 = 2-tier FP16+INT8(+drop);
                                 2 = 3-tier whose low tier is asymmetric 2-bit (NEXT-4) */
    int32_t tier_mode;        /* NEXT-4 bit flags, 0 = the paper's tiers: SKV_MODE_HOT_INT8, SKV_MODE_GROUP2 */
} skv_policy;
#define SKV_MODE_HOT_INT8 1   /* the hot tier ships INT8: no FP16 on the wire, protected positions pinned to INT8 (P21) */
#define SKV_MODE_GROUP2 2     /* the 2-bit low tier is quantised in groups of 32 elements (P22); needs allow_int4 = 2 */

/* Tier populations of ONE layer of ONE request (identical for every layer and request of a batch,
 * because n, b and the protected set are).  budget_q4 = floor(4bn + 1e-6), spent_q4 = 4n16+2n8+n4; with
 * allow_int4 = 2, n4 is the population of the 2-bit tier and both are in eighths: floor(8bn + 1e-6), 8n16+4n8+n4. */
typedef struct {
    int32_t n16, n8, n4, n0;
    int32_t allow_int4, tier_mode;   /* tier_mode: the policy's NEXT-4 flags (0 = default); with SKV_MODE_HOT_INT8, n16 = 0 */
    int64_t budget_q4, spent_q4;
} skv_counts;

/* HOST only.  Closed form of Eq. 14-15 with sink/range pinning paid out of the budget. */
int skv_tier_counts(const skv_shape *shape, const skv_policy *policy, skv_counts *counts_out);

/* HOST only.  Bytes of ONE request's SKV1 blob (a multiple of 256); 0 on invalid arguments. */
size_t skv_blob_bytes(const skv_shape *shape, const skv_counts *counts);

/* HOST only.  Workspace (DEVICE bytes) sufficient for any entry point on this shape with the given
 * observation window (pass window = 0 if skv_importance is not used).  0 on invalid arguments (dims <= 0; with
 * window > 0 also Hq % Hkv != 0 or window > n) and on shapes skv_importance reports as unsupported (its work
 * decomposition -- R*L*Hkv*row-blocks*key-tiles items, R*L*Hq*window query rows -- must fit 32-bit counters).
 * The workspace passed to any entry point must be 16-byte aligned (SKV_ERR_UNSUPPORTED otherwise). */
size_t skv_workspace_bytes(const skv_shape *shape, int32_t window);

/* HOST only.  Validates the first 256 bytes of a received blob (HOST memory) against blob_bytes and
 * returns the dims (strides zero) and counts it declares.  SKV_ERR_BAD_BLOB on any mismatch. */
int skv_blob_check(const void *header_host, size_t blob_bytes, skv_shape *shape_out, skv_counts *counts_out);

/* DEVICE.  K_dev: fp16, addressed by `shape` strides.  Q_dev: fp16 [R][L][Hq][window][d_h] contiguous,
 * window query i of a request sits at position n - window + i.  causal != 0 excludes keys beyond the
 * query position.  importance_dev: f32 [R][L][n].  Accumulation in fp32 (tensor cores, fp16 inputs);
 * agreement with the float64 definition is ~1e-5 relative (contract: 1e-3). */
int skv_importance(const skv_shape *shape, const void *K_dev, const void *Q_dev, int32_t window,
                   int32_t causal, float lambda, float *importance_dev,
                   void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* DEVICE.  KV-norm fallback score: A_j = mean over KV heads of ||k_j||_2, normalised to sum 1 per layer,
 * times the same decay.  importance_dev: f32 [R][L][n]. */
int skv_importance_kvnorm(const skv_shape *shape, const void *K_dev, float lambda, float *importance_dev,
                          void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* DEVICE.  skv_importance_kvnorm for a caller that cannot allocate device memory: same inputs, same output (bit for
 * bit -- the same two kernels run), no workspace argument.
 *
 * For whom: code embedded in a serving engine (a prefill-side plug-in, a custom op written against the engine's C
 * interface) that is handed the key cache and the output tensor and nothing else.  The engine's memory pool has
 * already claimed the GPU's memory, so the plug-in's own cudaMalloc fails (or, on a hot loop, is forbidden because it
 * stalls the whole device), and the pool is not reachable from C.  Such a caller cannot produce the `workspace_dev`
 * the other entry points ask for.
 *
 * How: the scratch the two KV-norm kernels share -- one f32 per (request, layer, token) plus one f64 per 64 tokens --
 * is a fixed SKV_NOALLOC_SCRATCH_BYTES (4.25 MiB) array inside the library image.  Every GPU that loads the library
 * carries it from load to process exit.  The call performs no cudaMalloc / cudaFree and calls nothing that allocates.
 *
 * Limit: n_requests * n_layers * n_tokens <= 1 Mi scores is always enough room as long as n_tokens >= 64 per layer
 * (precisely: 4*R*L*n rounded up to 256, plus 8*R*L*ceil(n/64), must not exceed SKV_NOALLOC_SCRATCH_BYTES) -- one
 * 32-layer request of 32768 tokens, or four of 8192.  Anything larger returns SKV_ERR_NOALLOC_LIMIT and launches
 * nothing.  Other argument errors are those of skv_importance_kvnorm.
 *
 * First call on each GPU: the entry point asks the CUDA runtime for the array's address on the device that is current
 * at that moment (this may also be the moment the driver loads the library's device code), and caches it per device
 * ordinal.  Make that first call during start-up -- with the right device current, and before any stream capture is
 * begun -- so that later calls are kernel launches only.  The device that is current at every call must be the one
 * `cuda_stream`, K_dev and importance_dev belong to.  At most 64 device ordinals (SKV_ERR_UNSUPPORTED beyond).
 *
 * Sharing: all calls on one GPU use the same array -- from every stream and every host thread.  Two calls whose
 * kernels can be in flight at the same time (different streams without an event between them) overwrite each other's
 * partial results and return garbage without any error; order them on one stream or with events.  Nothing needs to be
 * cleared between calls: each call writes every scratch word it later reads, so the previous call's leftovers (of
 * whatever shape) are never read. */
#define SKV_NOALLOC_SCRATCH_BYTES (4352u * 1024u)
int skv_importance_kvnorm_noalloc(const skv_shape *shape, const void *K_dev, float lambda, float *importance_dev,
                                  void *cuda_stream);

/* DEVICE.  importance_dev f32 [R][L][n] -> tier_map_dev u8 [R][L][n].  NaN / negative / -0 scores rank as
 * +0; equal scores are ranked by ascending position.  counts_out_host (HOST, nullable) receives the
 * closed-form counts; no device->host transfer takes place. */
int skv_assign_tiers(const skv_shape *shape, const skv_policy *policy, const float *importance_dev,
                     uint8_t *tier_map_dev, skv_counts *counts_out_host,
                     void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* DEVICE.  The same selection with EXPLICIT tier populations instead of a budget (ablation policies of PAPER.md:271,
 * :503 -- e.g. "Balanced", whose fractions the paper does not define; Random_Tier is skv_assign_tiers with random
 * scores).  counts: from skv_counts_from_populations(); positions [0,n_sink) and the n_ranges half-open ranges (HOST)
 * are FP16 and count towards n16 (INT8 and n8 with SKV_MODE_HOT_INT8; SKV_ERR_BUDGET_INFEASIBLE if they exceed it).  The rest is ranked as in
 * skv_assign_tiers: top n16-P -> 16, next n8 -> 8, next n4 -> low tier, rest -> 0. */
int skv_assign_tiers_counts(const skv_shape *shape, const skv_counts *counts, int32_t n_sink, int32_t n_ranges,
                            const int32_t *ranges, const float *importance_dev, uint8_t *tier_map_dev,
                            void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* DEVICE.  Writes n_requests blobs at blob_dev + r*skv_blob_bytes(); every byte of each blob is written
 * (pads zero) so blobs are memcmp-comparable.  blob_dev must be 256-B aligned.  `counts` must match the
 * tier map of every layer (maps produced by skv_assign_tiers always do); on a mismatch slots are clamped
 * to the segment capacity (memory safe) and the blob is meaningless. */
int skv_pack(const skv_shape *shape, const void *K_dev, const void *V_dev, const uint8_t *tier_map_dev,
             const skv_counts *counts, void *blob_dev, size_t blob_capacity,
             void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* DEVICE.  blob_dev holds n_requests blobs of blob_bytes each (as validated by skv_blob_check on the
 * host copy).  `shape` gives dims, OUTPUT strides and the element type, which must be the one the header declares
 * (skv_blob_check reports it in shape_out->dtype).  Writes every element of K_out/V_out (dropped
 * tokens -> +0.0) and, if tier_map_out_dev != NULL, the tier map u8 [R][L][n] (the validity mask). */
int skv_unpack(const skv_shape *shape, const void *blob_dev, size_t blob_bytes, const skv_counts *counts,
               void *K_out_dev, void *V_out_dev, uint8_t *tier_map_out_dev,
               void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* DEVICE.  Cold-tier precision upgrade, decode side ("a cold-tier fetch only needs to
 * upgrade the precision"; described there, never implemented).  The prefill side builds an UPGRADE
 * blob with skv_pack() from an upgrade map u8 [R][L][n] that holds the new tier (normally 16) at the tokens to
 * upgrade and 0 everywhere else, with counts from skv_counts_from_populations() (the same number of upgraded
 * tokens in every layer).  skv_unpack_patch() applies it in place: tokens the blob carries are overwritten in
 * K_inout/V_inout exactly as skv_unpack() would write them, tokens it does not carry (tier 0 in the blob) are left
 * untouched, and tier_map_inout_dev (nullable) is updated at the carried tokens only.  The replacement rows are
 * shipped whole (2 B per element at tier 16): a lossless residual against the INT4 codes does not fit the paper's
 * s16 - s4 figure (NEXT-3). */
int skv_unpack_patch(const skv_shape *shape, const void *blob_dev, size_t blob_bytes, const skv_counts *counts,
                     void *K_inout_dev, void *V_inout_dev, uint8_t *tier_map_inout_dev,
                     void *workspace_dev, size_t workspace_bytes, void *cuda_stream);

/* HOST only.  Counts for explicit tier populations (upgrade blobs, ablation policies): n0 = n - n16 - n8 - n4,
 * budget_q4 = spent_q4 = 4 n16 + 2 n8 + n4.  SKV_ERR_INVALID_ARG if the populations exceed n or n4 > 0 without
 * allow_int4.  tier_mode of the result is 0; a caller that wants group-wise 2-bit codes or an INT8 hot tier (n16 = 0)
 * sets counts_out->tier_mode itself. */
int skv_counts_from_populations(const skv_shape *shape, int32_t n16, int32_t n8, int32_t n4, int32_t allow_int4,
                                skv_counts *counts_out);

const char *skv_strerror(int status);

/* Library build tag, e.g. "skv 0.1 sm_100a". */
const char *skv_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SKV_H_ */
