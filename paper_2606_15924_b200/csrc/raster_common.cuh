// Shared pieces of the two raster kernels: the per-warp staged Gaussian batch, the conservative
// warp-level cull and the work-unit scheduler.
//
// Work decomposition (both kernels): a WORK UNIT is one group of 32 consecutive sampled pixels of
// one sampled tile (PAPER.md:156 -- pixels are listed tile by tile).  Warps are persistent and pull
// units from a global atomic counter, so a tile with a long Gaussian range does not pin a whole
// block, and a launch with few sampled tiles still spreads over all SMs.  Each warp walks its
// tile's depth-ordered range in batches of 32: every lane loads one Gaussian record (float4 loads),
// tests it against the bounding box of the warp's 32 pixels, and the survivors are compacted into
// the warp's shared-memory slice in range order; the inner loop then runs over survivors only.
//
// The cull is conservative: it only drops a Gaussian when NO pixel of the box can reach
// alpha >= 1/255 (so the result is identical to walking the full range).
#pragma once
#include "common.cuh"

namespace tgs {

constexpr int kRasterWarps = 8;                 // warps per block
constexpr int kRasterThreads = kRasterWarps * 32;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLnAlphaMin = -5.541263545158426f;  // ln(1/255)

struct WarpBatch {
    float4 a[32];    // mx, my, -A/2, -B
    float2 b[32];    // -C/2, thr = ln(1/(255 o))  (blend needs thr <= power <= 0)
    float4 c[32];    // opacity, r, g, b
    uint32_t p[32];  // 1-based position in the tile range (fwd) / Gaussian id (bwd)
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Canonical power: fma(fma(-B, dy, (-A/2) dx), dx, ((-C/2) dy) dy)
__device__ __forceinline__ float splat_power(float nA, float nB, float nC, float dx, float dy) {
    return __fmaf_rn(__fmaf_rn(nB, dy, __fmul_rn(nA, dx)), dx, __fmul_rn(__fmul_rn(nC, dy), dy));
}

// Conservative test: can the splat reach alpha >= 1/255 anywhere in the pixel box [bx0,bx1]x[by0,by1]?
// The region {power >= thr} is the ellipse d^T M d <= 2|thr| (M = conic); its axis-aligned half
// extents are sqrt(2|thr| C/det), sqrt(2|thr| A/det).  Slack: 0.1 % + 0.05 px.
__device__ __forceinline__ bool splat_may_touch(float mx, float my, float A, float B, float C, float thr,
                                                float bx0, float by0, float bx1, float by1) {
    if (thr > 0.0f) return false;  // opacity < 1/255: never blends
    const float det = A * C - B * B;
    const float s = -2.0f * thr / det;
    const float ex = sqrtf(s * C) * 1.001f + 0.05f;
    const float ey = sqrtf(s * A) * 1.001f + 0.05f;
    // written so that NaN anywhere keeps the Gaussian
    return !(mx + ex < bx0 || mx - ex > bx1 || my + ey < by0 || my - ey > by1);
}

struct UnitInfo {
    uint32_t start, end;   // tile range in gid_sorted
    uint32_t pix0, npix;   // this warp's pixels: global list index of lane 0, count (1..32)
};

// unit u -> (sampled tile u/8, pixel group u%8); returns false if the group is empty
__device__ __forceinline__ bool decode_unit(uint32_t u, const uint32_t* __restrict__ tiles,
                                            const uint32_t* __restrict__ tile_offsets,
                                            const uint32_t* __restrict__ tpo, UnitInfo& ui) {
    const uint32_t it = u >> 3, gi = u & 7u;
    const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
    if (gi * 32u >= m) return false;
    const uint32_t t = tiles[it];
    ui.start = tile_offsets[t];
    ui.end = tile_offsets[t + 1];
    ui.pix0 = p0 + gi * 32u;
    ui.npix = min(32u, m - gi * 32u);
    return true;
}

}  // namespace tgs
