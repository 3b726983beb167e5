// skv_common.cuh -- internal declarations shared by the CUDA translation units of libskv.
// (Product code; shares nothing with oracle/.)
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/skv.h"

namespace skv {

// SKV1 layout of one request's blob (include/skv.h, "Wire format").  Segment order:
// K16 V16 K8 V8 K4 V4 SK8 SV8 SK4 SV4.
struct Layout {
    uint64_t tier_map_off, layer0_off, layer_stride, total_bytes;
    uint64_t seg_off[10];
    uint64_t seg_raw[10];
};

// Dense-cache geometry handed to kernels by value.
struct Geom {
    int32_t L, Hq, Hkv, D, n, R;
    int64_t sr, sl, st, sh;      // strides in elements
    int32_t n16, n8, n4, n0;
    int32_t row_chunks;          // ceil(Hkv*D / 256): 16-byte-per-lane warp chunks in one token row
    int32_t tiles;               // ceil(n / kTileTokens)
    int32_t patch;               // unpack only: 1 = tokens the blob does not carry (tier 0) are left untouched
    int32_t low_code;            // tier code of the low tier: 4 (symmetric INT4) or 2 (asymmetric 2-bit, NEXT-4)
    int32_t bf16;                // element type of the dense caches and of the scale records: 0 = fp16, 1 = bfloat16
    int32_t low_group;           // 2-bit low tier: 0 = one (lo, hi) record per head vector, 32 = one per 32 elements (P22)
};

constexpr int kTileTokens = 32;  // tokens per pack/unpack tile (one ballot word)
#ifndef SKV_FUSE_MAX_TOKENS
#define SKV_FUSE_MAX_TOKENS 8192
#endif
constexpr int kFuseMaxTokens = SKV_FUSE_MAX_TOKENS;   // up to this n a pack / unpack CTA counts the tiers below its tile itself (one launch)
static_assert(kFuseMaxTokens >= kTileTokens && kFuseMaxTokens <= 65535,
              "self_tile_base (skv_codec.cuh) packs two tier counts into the 16-bit halves of one word");

// Where a pack / unpack CTA gets its tiles and their slot bases from.
//   tile_base != nullptr: from tile_scan_kernel (skv_scan.cu), [R][L][tiles]; nullptr = "fused": the CTA counts the
//                         tier-map bytes below its tile itself and also writes the stage's metadata;
//   live_count != nullptr: sparse blob -- only the live_count[r][l] tiles listed in tile_base[r][l][idx].w carry
//                         tokens, and the grid strides over that list.
struct TileSrc { const uint4 *tile_base; const uint32_t *live_count; };

struct Header256 { uint32_t w[64]; };   // the 256-byte SKV1 header image, built on the host

static inline __host__ __device__ uint64_t pad256(uint64_t x) { return (x + 255ull) & ~255ull; }

// host helpers (skv_host.cu)
Layout make_layout(int L, int Hkv, int D, int64_t n, int64_t n16, int64_t n8, int64_t n4, int low_bits, int low_group = 0);

// launchers (one per .cu)
cudaError_t launch_tile_scan_pack(const Geom &g, const Layout &lo, const uint8_t *tier_map, uint8_t *blob,
                                  uint64_t blob_stride, const Header256 &hdr, uint4 *tile_base, uint32_t *live_count,
                                  cudaStream_t s);
// grid_x: CTAs per (layer, request) -- the number of tiles, or fewer when the grid strides over a sparse live list
cudaError_t launch_pack(const Geom &g, const Layout &lo, const __half *K, const __half *V, const uint8_t *tier_map,
                        uint8_t *blob, uint64_t blob_stride, const Header256 &hdr, TileSrc ts, int grid_x, cudaStream_t s);
cudaError_t launch_tile_scan_unpack(const Geom &g, const Layout &lo, const uint8_t *blob, uint64_t blob_stride,
                                    uint8_t *tier_map_out, uint4 *tile_base, uint32_t *live_count, cudaStream_t s);
cudaError_t launch_unpack(const Geom &g, const Layout &lo, const uint8_t *blob, uint64_t blob_stride,
                          __half *K, __half *V, uint8_t *tier_map_out, TileSrc ts, int grid_x, cudaStream_t s);

struct Intervals { int32_t count; int32_t lo[32]; int32_t hi[32]; };   // merged protected ranges (incl. sinks)
cudaError_t launch_assign(const Geom &g, const Intervals &prot, const float *importance, uint8_t *tier_map,
                          uint32_t *key_ws, cudaStream_t s);

cudaError_t launch_importance_tc(const Geom &g, const __half *K, const __half *Q, int window, int causal, float lambda,
                                 float *importance, void *ws, cudaStream_t s);
size_t importance_tc_ws_bytes(const Geom &g, int window);      // 0: the work decomposition does not fit
cudaError_t launch_importance_kvnorm(const Geom &g, const __half *K, float lambda, float *importance, void *ws,
                                     cudaStream_t s);
size_t kvnorm_ws_bytes(const Geom &g);

}  // namespace skv
