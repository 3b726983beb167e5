// skv_host.cu -- the C ABI of libskv (include/skv.h): argument validation, the closed-form tier counts
// (Eq. 14-15; SinkProtect PAPER.md:230; 2-tier drop PAPER.md:543), the SKV1 layout
// arithmetic, and kernel launches on the caller's stream.  No allocation, no global state, no host sync.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "skv_common.cuh"

namespace skv {

// low_bits: 4 = the low tier holds symmetric INT4 codes (two per byte, one fp16 amax record per head vector);
// 2 = asymmetric 2-bit codes (four per byte, an fp16 (lo, hi) pair per head vector) -- NEXT-4.
// low_group (2-bit tier only): 0 = one record per head vector, 32 = one per group of 32 elements (reading P22).
Layout make_layout(int L, int Hkv, int D, int64_t n, int64_t n16, int64_t n8, int64_t n4, int low_bits, int low_group)
{
    Layout lo;
    const uint64_t H = (uint64_t)Hkv, d = (uint64_t)D;
    const uint64_t cpb = low_bits == 2 ? 4 : 2;
    const uint64_t rec = low_bits == 2 ? (low_group ? d / (uint64_t)low_group : 1) * 4 : 2;     // record bytes per head vector
    const uint64_t raw[10] = {
        (uint64_t)n16 * H * d * 2, (uint64_t)n16 * H * d * 2,
        (uint64_t)n8 * H * d,      (uint64_t)n8 * H * d,
        (uint64_t)n4 * H * d / cpb, (uint64_t)n4 * H * d / cpb,
        (uint64_t)n8 * H * 2,      (uint64_t)n8 * H * 2,
        (uint64_t)n4 * H * rec,    (uint64_t)n4 * H * rec};
    lo.tier_map_off = 256;
    lo.layer0_off = 256 + pad256((uint64_t)L * (uint64_t)n);
    uint64_t off = 0;
    for (int s = 0; s < 10; ++s) { lo.seg_off[s] = off; lo.seg_raw[s] = raw[s]; off += pad256(raw[s]); }
    lo.layer_stride = off;
    lo.total_bytes = lo.layer0_off + (uint64_t)L * lo.layer_stride;
    return lo;
}

static bool dims_ok(const skv_shape *s)
{
    return s && s->n_layers > 0 && s->n_kv_heads > 0 && s->head_dim > 0 && s->n_tokens > 0 && s->n_requests > 0;
}

static int check_dims_supported(const skv_shape *s)
{
    if (!dims_ok(s)) return SKV_ERR_INVALID_ARG;
    if (s->head_dim != 64 && s->head_dim != 128 && s->head_dim != 256) return SKV_ERR_UNSUPPORTED;
    if (s->n_tokens > (1 << 20)) return SKV_ERR_UNSUPPORTED;
    if ((s->dtype != SKV_F16 && s->dtype != SKV_BF16) || s->reserved != 0) return SKV_ERR_INVALID_ARG;
    if (s->n_layers > 65535 || s->n_requests > 65535 || (int64_t)s->n_layers * s->n_requests > 65535) return SKV_ERR_UNSUPPORTED;
    return SKV_OK;
}

// is_output: the cache is written (skv_unpack / skv_unpack_patch), so a zero layer / request stride with more than one
// layer / request would make the writes overlap; for inputs a zero stride is a harmless broadcast.
static int check_cache(const skv_shape *s, const void *K, const void *V, bool is_output = false)
{
    int rc = check_dims_supported(s);
    if (rc) return rc;
    if (!K || !V) return SKV_ERR_INVALID_ARG;
    if (s->stride_head <= 0 || s->stride_token <= 0 || s->stride_layer < 0 || s->stride_request < 0) return SKV_ERR_INVALID_ARG;
    if (is_output && ((s->n_layers > 1 && s->stride_layer == 0) || (s->n_requests > 1 && s->stride_request == 0)))
        return SKV_ERR_INVALID_ARG;
    if ((s->stride_head % 8) || (s->stride_token % 8) || (s->stride_layer % 8) || (s->stride_request % 8)) return SKV_ERR_UNSUPPORTED;
    if (((uintptr_t)K & 15) || ((uintptr_t)V & 15)) return SKV_ERR_UNSUPPORTED;
    return SKV_OK;
}

// every workspace layout starts with 16-byte (uint4 / float2 / double) records: a misaligned base would fault in the kernel
static bool ws_misaligned(const void *ws) { return ((uintptr_t)ws & 15) != 0; }

static Geom make_geom(const skv_shape *s, const skv_counts *c)
{
    Geom g;
    g.L = s->n_layers; g.Hq = s->n_q_heads; g.Hkv = s->n_kv_heads; g.D = s->head_dim; g.n = s->n_tokens; g.R = s->n_requests;
    g.sr = s->stride_request; g.sl = s->stride_layer; g.st = s->stride_token; g.sh = s->stride_head;
    g.n16 = c ? c->n16 : 0; g.n8 = c ? c->n8 : 0; g.n4 = c ? c->n4 : 0; g.n0 = c ? c->n0 : 0;
    g.row_chunks = (g.Hkv * g.D + 255) / 256;
    g.tiles = (g.n + kTileTokens - 1) / kTileTokens;
    g.patch = 0;
    g.low_code = (c && c->allow_int4 == 2) ? 2 : 4;
    g.bf16 = s->dtype == SKV_BF16 ? 1 : 0;
    g.low_group = (c && c->allow_int4 == 2 && (c->tier_mode & SKV_MODE_GROUP2)) ? 32 : 0;
    return g;
}

static bool counts_ok(const skv_shape *s, const skv_counts *c)
{
    return c && c->n16 >= 0 && c->n8 >= 0 && c->n4 >= 0 && c->n0 >= 0 &&
           (int64_t)c->n16 + c->n8 + c->n4 + c->n0 == (int64_t)s->n_tokens;
}

// what skv_blob_check would refuse on the decode side: a low tier without the flag, or a budget the populations exceed
static bool counts_wire_ok(const skv_shape *s, const skv_counts *c)
{
    if (!counts_ok(s, c) || c->allow_int4 < 0 || c->allow_int4 > 2 || (c->tier_mode & ~3)) return false;
    if (c->allow_int4 == 0 && c->n4 != 0) return false;
    if ((c->tier_mode & SKV_MODE_HOT_INT8) && c->n16 != 0) return false;        // INT8 hot tier: nothing ships at FP16
    if ((c->tier_mode & SKV_MODE_GROUP2) && c->allow_int4 != 2) return false;   // groups exist only in the 2-bit tier
    const int64_t unit = c->allow_int4 == 2 ? 8 : 4;
    const int64_t spent = unit * c->n16 + (unit / 2) * c->n8 + c->n4;
    return c->budget_q4 >= spent && c->budget_q4 <= unit * (int64_t)s->n_tokens;
}

// workspace of pack / unpack: the tile prefix table uint4[R][L][tiles] (.w = the list of live tiles of a sparse blob),
// then the live-tile counts u32[R][L]
static size_t scan_table_bytes(const skv_shape *s)
{
    const size_t tiles = ((size_t)s->n_tokens + kTileTokens - 1) / kTileTokens;
    return (size_t)s->n_requests * s->n_layers * tiles * sizeof(uint4);
}
static size_t scan_ws_bytes(const skv_shape *s)
{
    return scan_table_bytes(s) + (size_t)s->n_requests * s->n_layers * sizeof(uint32_t);
}

// How a pack / unpack stage is launched (skv_common.cuh: TileSrc).
//   fused  (n <= kFuseMaxTokens): one launch, every CTA counts the tiers below its own tile;
//   sparse (fewer than 1 token in 8 is shipped, no 2-bit tier, and empty tiles need no work: pack, unpack_patch): the scan emits the
//          list of live tiles and the grid strides over it -- a cold-tier upgrade of 1024 tokens of a 32 K-token layer
//          touches at most 1024 of its tiles, typically a few dozen;
//   otherwise the scan kernel, then one CTA per tile.
struct StagePlan { bool fused, sparse; int grid_x; };
static StagePlan plan_stage(const Geom &g, bool empty_tiles_skippable)
{
    StagePlan p;
    const int64_t shipped = (int64_t)g.n16 + g.n8 + g.n4;
    p.sparse = empty_tiles_skippable && shipped * 8 <= (int64_t)g.n && g.tiles > 1 && g.low_code != 2;
    p.fused = !p.sparse && g.n <= kFuseMaxTokens;
    p.grid_x = g.tiles;
    if (p.sparse) {
        const int64_t live_max = std::max<int64_t>(1, std::min<int64_t>(g.tiles, shipped));
        const int64_t want = std::max<int64_t>(1, 4096 / ((int64_t)g.L * g.R));      // ~9 waves of CTAs in total
        p.grid_x = (int)std::min(live_max, want);
    }
    return p;
}

// merged, sorted protected intervals = [0,s) U ranges; returns P (their total size) or <0 on error
static int64_t merge_protected(const skv_shape *s, const skv_policy *p, std::vector<std::pair<int32_t, int32_t>> &out)
{
    const int32_t n = s->n_tokens;
    if (p->n_sink < 0 || p->n_ranges < 0 || (p->n_ranges > 0 && !p->ranges)) return -1;
    std::vector<std::pair<int32_t, int32_t>> iv;
    if (p->n_sink > 0) iv.emplace_back(0, std::min(p->n_sink, n));
    for (int i = 0; i < p->n_ranges; ++i) {
        const int32_t b = p->ranges[2 * i], e = p->ranges[2 * i + 1];
        if (b < 0 || e > n || b > e) return -1;
        if (e > b) iv.emplace_back(b, e);
    }
    std::sort(iv.begin(), iv.end());
    out.clear();
    for (auto &x : iv) {
        if (!out.empty() && x.first <= out.back().second) out.back().second = std::max(out.back().second, x.second);
        else out.push_back(x);
    }
    int64_t P = 0;
    for (auto &x : out) P += x.second - x.first;
    return P;
}

static int tier_counts_impl(const skv_shape *s, const skv_policy *p, skv_counts *c,
                            std::vector<std::pair<int32_t, int32_t>> &prot)
{
    if (!dims_ok(s) || !p || !c) return SKV_ERR_INVALID_ARG;
    double b = p->budget;
    if (!(b > 0.0)) return SKV_ERR_INVALID_ARG;           // also rejects NaN
    if (b > 1.0) b = 1.0;
    const int64_t P = merge_protected(s, p, prot);
    if (P < 0) return SKV_ERR_INVALID_ARG;
    const int64_t n = s->n_tokens;
    if (p->allow_int4 != 0 && p->allow_int4 != 1 && p->allow_int4 != 2) return SKV_ERR_INVALID_ARG;
    if ((p->tier_mode & ~3) || ((p->tier_mode & SKV_MODE_GROUP2) && p->allow_int4 != 2)) return SKV_ERR_INVALID_ARG;
    if (p->tier_mode & SKV_MODE_HOT_INT8) {
        // NEXT-4, reading P21: the hot tier ships INT8.  Costs c8 (INT8) and 1 (low tier) in quarter- or eighth-units.
        const int64_t unit = p->allow_int4 == 2 ? 8 : 4, c8 = unit / 2;
        const int64_t Q = (int64_t)floor((double)unit * b * (double)n + 1e-6);
        const int64_t m = n - P, R = Q - c8 * P;
        if (R < 0) return SKV_ERR_BUDGET_INFEASIBLE;
        int64_t n8 = P, nl = 0, n0 = 0;
        if (R >= c8 * m) n8 = n;
        else if (!p->allow_int4) { n8 = P + R / c8; n0 = n - n8; }
        else if (R >= m) { const int64_t up = (R - m) / (c8 - 1); n8 = P + up; nl = m - up; }
        else { nl = R; n0 = m - R; }
        c->n16 = 0; c->n8 = (int32_t)n8; c->n4 = (int32_t)nl; c->n0 = (int32_t)n0;
        c->allow_int4 = p->allow_int4; c->tier_mode = p->tier_mode;
        c->budget_q4 = Q; c->spent_q4 = c8 * n8 + nl;
        return SKV_OK;
    }
    if (p->allow_int4 == 2) {
        // NEXT-4: 2-bit low tier, c = 1/8 -> the same greedy ladder in EIGHTH-units, 8 / 4 / 1 / 0 per token
        const int64_t Q8 = (int64_t)floor(8.0 * b * (double)n + 1e-6);
        const int64_t m8 = n - P, R8 = Q8 - 8 * P;
        if (R8 < 0) return SKV_ERR_BUDGET_INFEASIBLE;
        int64_t a16 = P, a8 = 0, a2 = 0, a0 = 0;
        if (R8 >= 8 * m8) a16 = n;
        else if (R8 >= 4 * m8) { const int64_t up = (R8 - 4 * m8) / 4; a16 = P + up; a8 = m8 - up; }
        else if (R8 >= m8) { a8 = (R8 - m8) / 3; a2 = m8 - a8; }
        else { a2 = R8; a0 = m8 - R8; }
        c->n16 = (int32_t)a16; c->n8 = (int32_t)a8; c->n4 = (int32_t)a2; c->n0 = (int32_t)a0;
        c->allow_int4 = 2; c->tier_mode = p->tier_mode;
        c->budget_q4 = Q8; c->spent_q4 = 8 * a16 + 4 * a8 + a2;
        return SKV_OK;
    }
    const int64_t Q = (int64_t)floor(4.0 * b * (double)n + 1e-6);     // quarter-units: 4 / 2 / 1 / 0 per token
    const int64_t m = n - P, R = Q - 4 * P;
    if (R < 0) return SKV_ERR_BUDGET_INFEASIBLE;
    int64_t n16 = P, n8 = 0, n4 = 0, n0 = 0;
    if (R >= 4 * m) n16 = n;
    else if (R >= 2 * m) { const int64_t up = (R - 2 * m) / 2; n16 = P + up; n8 = m - up; }
    else if (p->allow_int4) {
        if (R >= m) { n8 = R - m; n4 = m - n8; }
        else { n4 = R; n0 = m - R; }
    } else { n8 = R / 2; n0 = m - n8; }
    c->n16 = (int32_t)n16; c->n8 = (int32_t)n8; c->n4 = (int32_t)n4; c->n0 = (int32_t)n0;
    c->allow_int4 = p->allow_int4 ? 1 : 0; c->tier_mode = 0;
    c->budget_q4 = Q; c->spent_q4 = 4 * n16 + 2 * n8 + n4;
    return SKV_OK;
}

static void put32(uint8_t *p, uint32_t v) { memcpy(p, &v, 4); }
static void put64(uint8_t *p, uint64_t v) { memcpy(p, &v, 8); }
static uint32_t get32(const uint8_t *p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint64_t get64(const uint8_t *p) { uint64_t v; memcpy(&v, p, 8); return v; }

}  // namespace skv

using namespace skv;

extern "C" {

int skv_tier_counts(const skv_shape *shape, const skv_policy *policy, skv_counts *counts_out)
{
    std::vector<std::pair<int32_t, int32_t>> prot;
    return tier_counts_impl(shape, policy, counts_out, prot);
}

size_t skv_blob_bytes(const skv_shape *shape, const skv_counts *counts)
{
    if (!dims_ok(shape) || !counts_ok(shape, counts)) return 0;
    const bool low2 = counts->allow_int4 == 2;
    return (size_t)make_layout(shape->n_layers, shape->n_kv_heads, shape->head_dim, shape->n_tokens,
                               counts->n16, counts->n8, counts->n4, low2 ? 2 : 4,
                               (low2 && (counts->tier_mode & SKV_MODE_GROUP2)) ? 32 : 0).total_bytes;
}

size_t skv_workspace_bytes(const skv_shape *shape, int32_t window)
{
    if (!dims_ok(shape)) return 0;
    const Geom g = make_geom(shape, nullptr);
    size_t need = scan_ws_bytes(shape);
    need = std::max(need, (size_t)shape->n_requests * shape->n_layers * shape->n_tokens * sizeof(uint32_t));  // assign keys
    need = std::max(need, kvnorm_ws_bytes(g));
    if (window > 0) {
        // the importance plan divides by (Hq / Hkv) * window: refuse what skv_importance itself refuses
        if (shape->n_q_heads <= 0 || shape->n_q_heads % shape->n_kv_heads || window > shape->n_tokens) return 0;
        const size_t imp = importance_tc_ws_bytes(g, window);
        if (imp == 0) return 0;                                          // work decomposition does not fit 32-bit counters
        need = std::max(need, imp);
    }
    return (need + 255) & ~(size_t)255;
}

int skv_blob_check(const void *header_host, size_t blob_bytes, skv_shape *shape_out, skv_counts *counts_out)
{
    if (!header_host) return SKV_ERR_INVALID_ARG;
    if (blob_bytes < 256) return SKV_ERR_BAD_BLOB;
    const uint8_t *h = (const uint8_t *)header_host;
    if (get32(h) != 0x31564B53u || get32(h + 4) != 1u) return SKV_ERR_BAD_BLOB;
    const uint32_t L = get32(h + 8), Hkv = get32(h + 12), D = get32(h + 16), n = get32(h + 20);
    const uint32_t n16 = get32(h + 24), n8 = get32(h + 28), n4 = get32(h + 32), n0 = get32(h + 36);
    const uint32_t flags = get32(h + 40);
    if (L == 0 || Hkv == 0 || n == 0 || L > 65535u || n > (1u << 20) || Hkv > 65535u) return SKV_ERR_BAD_BLOB;
    if (D != 64 && D != 128 && D != 256) return SKV_ERR_BAD_BLOB;
    if ((uint64_t)n16 + n8 + n4 + n0 != n || (flags & ~31u) || (flags & 3u) == 2u || get32(h + 44) != 0) return SKV_ERR_BAD_BLOB;
    if (!(flags & 1u) && n4 != 0) return SKV_ERR_BAD_BLOB;
    const bool low2 = (flags & 2u) != 0;                    // bit1: the low tier is asymmetric 2-bit (budget in eighths)
    if ((flags & 8u) && n16 != 0) return SKV_ERR_BAD_BLOB;  // bit3: INT8 hot tier, nothing ships at FP16
    if ((flags & 16u) && !low2) return SKV_ERR_BAD_BLOB;    // bit4: 2-bit groups of 32 elements
    const Layout lo = make_layout((int)L, (int)Hkv, (int)D, n, n16, n8, n4, low2 ? 2 : 4, (flags & 16u) ? 32 : 0);
    if (get64(h + 56) != lo.tier_map_off || get64(h + 64) != lo.layer0_off || get64(h + 72) != lo.layer_stride ||
        get64(h + 160) != lo.total_bytes || lo.total_bytes != blob_bytes) return SKV_ERR_BAD_BLOB;
    for (int s = 0; s < 10; ++s) if (get64(h + 80 + 8 * s) != lo.seg_off[s]) return SKV_ERR_BAD_BLOB;
    for (int o = 168; o < 256; ++o) if (h[o]) return SKV_ERR_BAD_BLOB;
    const uint64_t Q = get64(h + 48);
    const uint64_t unit = low2 ? 8ull : 4ull;
    const uint64_t spent = unit * n16 + (unit / 2) * n8 + n4;
    if (Q > unit * n || spent > Q) return SKV_ERR_BAD_BLOB;
    if (shape_out) {
        memset(shape_out, 0, sizeof(*shape_out));
        shape_out->n_layers = (int32_t)L; shape_out->n_kv_heads = (int32_t)Hkv; shape_out->head_dim = (int32_t)D;
        shape_out->n_tokens = (int32_t)n; shape_out->n_requests = 1;
        shape_out->dtype = (flags & 4u) ? SKV_BF16 : SKV_F16;
    }
    if (counts_out) {
        counts_out->n16 = (int32_t)n16; counts_out->n8 = (int32_t)n8; counts_out->n4 = (int32_t)n4; counts_out->n0 = (int32_t)n0;
        counts_out->allow_int4 = low2 ? 2 : (int32_t)(flags & 1u);
        counts_out->tier_mode = ((flags & 8u) ? SKV_MODE_HOT_INT8 : 0) | ((flags & 16u) ? SKV_MODE_GROUP2 : 0);
        counts_out->budget_q4 = (int64_t)Q; counts_out->spent_q4 = (int64_t)spent;
    }
    return SKV_OK;
}

int skv_importance(const skv_shape *shape, const void *K_dev, const void *Q_dev, int32_t window, int32_t causal,
                   float lambda, float *importance_dev, void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_cache(shape, K_dev, K_dev);
    if (rc) return rc;
    if (!Q_dev || !importance_dev || !ws) return SKV_ERR_INVALID_ARG;
    if (shape->n_q_heads <= 0 || shape->n_q_heads % shape->n_kv_heads) return SKV_ERR_INVALID_ARG;
    if (window < 1 || window > shape->n_tokens) return SKV_ERR_INVALID_ARG;
    if (!(lambda >= 0.0f)) return SKV_ERR_INVALID_ARG;
    if (((uintptr_t)Q_dev & 15) || ws_misaligned(ws)) return SKV_ERR_UNSUPPORTED;
    // the K tensor map cannot express a broadcast (zero) stride over a dimension that has more than one entry
    if ((shape->n_layers > 1 && shape->stride_layer == 0) || (shape->n_requests > 1 && shape->stride_request == 0))
        return SKV_ERR_UNSUPPORTED;
    const Geom g = make_geom(shape, nullptr);
    const size_t need = importance_tc_ws_bytes(g, window);
    if (need == 0) return SKV_ERR_UNSUPPORTED;                            // R*L*Hkv*key-chunk items overflow 32 bits
    if (ws_bytes < need) return SKV_ERR_BUFFER_TOO_SMALL;
    cudaError_t e = launch_importance_tc(g, (const __half *)K_dev, (const __half *)Q_dev, window, causal ? 1 : 0, lambda,
                                         importance_dev, ws, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? SKV_OK : SKV_ERR_CUDA;
}

int skv_importance_kvnorm(const skv_shape *shape, const void *K_dev, float lambda, float *importance_dev,
                          void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_cache(shape, K_dev, K_dev);
    if (rc) return rc;
    if (!importance_dev || !ws || !(lambda >= 0.0f)) return SKV_ERR_INVALID_ARG;
    if (ws_misaligned(ws)) return SKV_ERR_UNSUPPORTED;
    const Geom g = make_geom(shape, nullptr);
    if (ws_bytes < kvnorm_ws_bytes(g)) return SKV_ERR_BUFFER_TOO_SMALL;
    cudaError_t e = launch_importance_kvnorm(g, (const __half *)K_dev, lambda, importance_dev, ws, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? SKV_OK : SKV_ERR_CUDA;
}

static int assign_launch(const skv_shape *shape, const skv_counts &c, const std::vector<std::pair<int32_t, int32_t>> &prot,
                         const float *importance_dev, uint8_t *tier_map_dev, void *ws, size_t ws_bytes, void *cuda_stream)
{
    if (prot.size() > 32) return SKV_ERR_UNSUPPORTED;    // more than 32 disjoint protected intervals
    const size_t key_bytes = (size_t)shape->n_requests * shape->n_layers * shape->n_tokens * sizeof(uint32_t);
    const bool need_ws = (size_t)shape->n_tokens * 4 > 200 * 1024;
    if (need_ws && (!ws || ws_bytes < key_bytes)) return SKV_ERR_BUFFER_TOO_SMALL;
    if (ws && ws_misaligned(ws)) return SKV_ERR_UNSUPPORTED;
    Intervals iv;
    memset(&iv, 0, sizeof(iv));
    iv.count = (int32_t)prot.size();
    for (size_t i = 0; i < prot.size(); ++i) { iv.lo[i] = prot[i].first; iv.hi[i] = prot[i].second; }
    const Geom g = make_geom(shape, &c);
    cudaError_t e = launch_assign(g, iv, importance_dev, tier_map_dev, (uint32_t *)ws, (cudaStream_t)cuda_stream);
    return e == cudaSuccess ? SKV_OK : SKV_ERR_CUDA;
}

int skv_assign_tiers(const skv_shape *shape, const skv_policy *policy, const float *importance_dev,
                     uint8_t *tier_map_dev, skv_counts *counts_out_host, void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_dims_supported(shape);
    if (rc) return rc;
    if (!policy || !importance_dev || !tier_map_dev) return SKV_ERR_INVALID_ARG;
    skv_counts c;
    std::vector<std::pair<int32_t, int32_t>> prot;
    rc = tier_counts_impl(shape, policy, &c, prot);
    if (rc) return rc;
    rc = assign_launch(shape, c, prot, importance_dev, tier_map_dev, ws, ws_bytes, cuda_stream);
    if (rc) return rc;
    if (counts_out_host) *counts_out_host = c;
    return SKV_OK;
}

int skv_assign_tiers_counts(const skv_shape *shape, const skv_counts *counts, int32_t n_sink, int32_t n_ranges,
                            const int32_t *ranges, const float *importance_dev, uint8_t *tier_map_dev,
                            void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_dims_supported(shape);
    if (rc) return rc;
    if (!importance_dev || !tier_map_dev || !counts_ok(shape, counts)) return SKV_ERR_INVALID_ARG;
    skv_policy pol;
    memset(&pol, 0, sizeof(pol));
    pol.budget = 1.0; pol.n_sink = n_sink; pol.n_ranges = n_ranges; pol.ranges = ranges;
    std::vector<std::pair<int32_t, int32_t>> prot;
    const int64_t P = merge_protected(shape, &pol, prot);
    if (P < 0) return SKV_ERR_INVALID_ARG;
    // the protected positions all sit in the hot tier (FP16, or INT8 with SKV_MODE_HOT_INT8)
    if (P > ((counts->tier_mode & SKV_MODE_HOT_INT8) ? counts->n8 : counts->n16)) return SKV_ERR_BUDGET_INFEASIBLE;
    if ((counts->tier_mode & SKV_MODE_HOT_INT8) && counts->n16 != 0) return SKV_ERR_INVALID_ARG;
    return assign_launch(shape, *counts, prot, importance_dev, tier_map_dev, ws, ws_bytes, cuda_stream);
}

int skv_pack(const skv_shape *shape, const void *K_dev, const void *V_dev, const uint8_t *tier_map_dev,
             const skv_counts *counts, void *blob_dev, size_t blob_capacity, void *ws, size_t ws_bytes, void *cuda_stream)
{
    int rc = check_cache(shape, K_dev, V_dev);
    if (rc) return rc;
    if (!tier_map_dev || !blob_dev || !ws || !counts_wire_ok(shape, counts)) return SKV_ERR_INVALID_ARG;
    if (((uintptr_t)blob_dev & 255) || ws_misaligned(ws)) return SKV_ERR_UNSUPPORTED;
    const Geom g = make_geom(shape, counts);
    const Layout lo = make_layout(g.L, g.Hkv, g.D, g.n, g.n16, g.n8, g.n4, g.low_code, g.low_group);
    if (blob_capacity < (size_t)lo.total_bytes * (size_t)g.R) return SKV_ERR_BUFFER_TOO_SMALL;
    if (ws_bytes < scan_ws_bytes(shape)) return SKV_ERR_BUFFER_TOO_SMALL;

    Header256 hdr;
    memset(&hdr, 0, sizeof(hdr));
    uint8_t *h = reinterpret_cast<uint8_t *>(hdr.w);
    put32(h + 0, 0x31564B53u); put32(h + 4, 1u);
    put32(h + 8, (uint32_t)g.L); put32(h + 12, (uint32_t)g.Hkv); put32(h + 16, (uint32_t)g.D); put32(h + 20, (uint32_t)g.n);
    put32(h + 24, (uint32_t)g.n16); put32(h + 28, (uint32_t)g.n8); put32(h + 32, (uint32_t)g.n4); put32(h + 36, (uint32_t)g.n0);
    put32(h + 40, (counts->allow_int4 ? 1u : 0u) | (counts->allow_int4 == 2 ? 2u : 0u) | (g.bf16 ? 4u : 0u) |
                  ((counts->tier_mode & SKV_MODE_HOT_INT8) ? 8u : 0u) | (g.low_group ? 16u : 0u));
    put64(h + 48, (uint64_t)counts->budget_q4);
    put64(h + 56, lo.tier_map_off); put64(h + 64, lo.layer0_off); put64(h + 72, lo.layer_stride);
    for (int s = 0; s < 10; ++s) put64(h + 80 + 8 * s, lo.seg_off[s]);
    put64(h + 160, lo.total_bytes);

    cudaStream_t st = (cudaStream_t)cuda_stream;
    const StagePlan plan = plan_stage(g, true);
    uint32_t *live = plan.sparse ? reinterpret_cast<uint32_t *>((uint8_t *)ws + scan_table_bytes(shape)) : nullptr;
    TileSrc ts = {plan.fused ? nullptr : (const uint4 *)ws, live};
    if (!plan.fused) {
        cudaError_t e = launch_tile_scan_pack(g, lo, tier_map_dev, (uint8_t *)blob_dev, lo.total_bytes, hdr, (uint4 *)ws, live, st);
        if (e != cudaSuccess) return SKV_ERR_CUDA;
    }
    cudaError_t e = launch_pack(g, lo, (const __half *)K_dev, (const __half *)V_dev, tier_map_dev, (uint8_t *)blob_dev,
                                lo.total_bytes, hdr, ts, plan.grid_x, st);
    return e == cudaSuccess ? SKV_OK : SKV_ERR_CUDA;
}

static int unpack_impl(const skv_shape *shape, const void *blob_dev, size_t blob_bytes, const skv_counts *counts,
                       void *K_out_dev, void *V_out_dev, uint8_t *tier_map_out_dev, void *ws, size_t ws_bytes,
                       void *cuda_stream, int patch)
{
    int rc = check_cache(shape, K_out_dev, V_out_dev, true);
    if (rc) return rc;
    if (!blob_dev || !ws || !counts_wire_ok(shape, counts)) return SKV_ERR_INVALID_ARG;
    if (((uintptr_t)blob_dev & 255) || ws_misaligned(ws)) return SKV_ERR_UNSUPPORTED;
    Geom g = make_geom(shape, counts);
    g.patch = patch;
    const Layout lo = make_layout(g.L, g.Hkv, g.D, g.n, g.n16, g.n8, g.n4, g.low_code, g.low_group);
    if (blob_bytes != (size_t)lo.total_bytes) return SKV_ERR_BAD_BLOB;
    if (ws_bytes < scan_ws_bytes(shape)) return SKV_ERR_BUFFER_TOO_SMALL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const StagePlan plan = plan_stage(g, patch != 0);               // a full unpack writes zeros into the empty tiles too
    uint32_t *live = plan.sparse ? reinterpret_cast<uint32_t *>((uint8_t *)ws + scan_table_bytes(shape)) : nullptr;
    TileSrc ts = {plan.fused ? nullptr : (const uint4 *)ws, live};
    if (!plan.fused) {
        cudaError_t e = launch_tile_scan_unpack(g, lo, (const uint8_t *)blob_dev, lo.total_bytes, tier_map_out_dev, (uint4 *)ws, live, st);
        if (e != cudaSuccess) return SKV_ERR_CUDA;
    }
    cudaError_t e = launch_unpack(g, lo, (const uint8_t *)blob_dev, lo.total_bytes, (__half *)K_out_dev, (__half *)V_out_dev,
                                  tier_map_out_dev, ts, plan.grid_x, st);
    return e == cudaSuccess ? SKV_OK : SKV_ERR_CUDA;
}

int skv_unpack(const skv_shape *shape, const void *blob_dev, size_t blob_bytes, const skv_counts *counts,
               void *K_out_dev, void *V_out_dev, uint8_t *tier_map_out_dev, void *ws, size_t ws_bytes, void *cuda_stream)
{
    return unpack_impl(shape, blob_dev, blob_bytes, counts, K_out_dev, V_out_dev, tier_map_out_dev, ws, ws_bytes, cuda_stream, 0);
}

int skv_unpack_patch(const skv_shape *shape, const void *blob_dev, size_t blob_bytes, const skv_counts *counts,
                     void *K_inout_dev, void *V_inout_dev, uint8_t *tier_map_inout_dev, void *ws, size_t ws_bytes,
                     void *cuda_stream)
{
    return unpack_impl(shape, blob_dev, blob_bytes, counts, K_inout_dev, V_inout_dev, tier_map_inout_dev, ws, ws_bytes, cuda_stream, 1);
}

int skv_counts_from_populations(const skv_shape *shape, int32_t n16, int32_t n8, int32_t n4, int32_t allow_int4,
                                skv_counts *counts_out)
{
    if (!dims_ok(shape) || !counts_out || n16 < 0 || n8 < 0 || n4 < 0) return SKV_ERR_INVALID_ARG;
    if ((int64_t)n16 + n8 + n4 > (int64_t)shape->n_tokens || (n4 > 0 && !allow_int4)) return SKV_ERR_INVALID_ARG;
    memset(counts_out, 0, sizeof(*counts_out));
    counts_out->n16 = n16; counts_out->n8 = n8; counts_out->n4 = n4;
    counts_out->n0 = shape->n_tokens - n16 - n8 - n4;
    if (allow_int4 < 0 || allow_int4 > 2) return SKV_ERR_INVALID_ARG;
    counts_out->allow_int4 = allow_int4;
    counts_out->spent_q4 = allow_int4 == 2 ? 8LL * n16 + 4LL * n8 + n4 : 4LL * n16 + 2LL * n8 + n4;
    counts_out->budget_q4 = counts_out->spent_q4;
    return SKV_OK;
}

const char *skv_strerror(int status)
{
    switch (status) {
    case SKV_OK: return "ok";
    case SKV_ERR_INVALID_ARG: return "invalid argument";
    case SKV_ERR_UNSUPPORTED: return "unsupported shape, stride or alignment";
    case SKV_ERR_BUDGET_INFEASIBLE: return "protected tokens alone exceed the transfer budget";
    case SKV_ERR_BUFFER_TOO_SMALL: return "blob capacity or workspace too small";
    case SKV_ERR_BAD_BLOB: return "malformed SKV1 blob";
    case SKV_ERR_CUDA: return "CUDA runtime error";
    case SKV_ERR_NOALLOC_LIMIT: return "problem exceeds the scratch built into the library (SKV_NOALLOC_SCRATCH_BYTES); pass a workspace to skv_importance_kvnorm instead";
    default: return "unknown status";
    }
}

const char *skv_version(void) { return "skv 0.1 sm_100a"; }

}  // extern "C"
