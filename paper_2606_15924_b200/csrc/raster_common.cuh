// Shared pieces of the two raster kernels: the per-warp staged Gaussian batch, the conservative
// warp-level cull and the work-unit decoding.
//
// Work decomposition (both kernels): a WORK UNIT is one group of 32 sampled pixels of one sampled
// tile (PAPER.md:156 -- pixels are listed tile by tile).  Warps are persistent and pull units from
// a global atomic counter, so a tile with a long Gaussian range does not pin a whole block, and a
// launch with few sampled tiles still spreads over all SMs.  Each warp walks its tile's
// depth-ordered range in batches of 32: every lane loads one Gaussian record (float4 loads, ids
// prefetched two batches ahead, records one batch ahead), tests it against the bounding box of the
// warp's 32 pixels, and the survivors are compacted into the warp's shared-memory slice in range
// order; the inner loop then runs over survivors only.
//
// The cull is conservative: it only drops a Gaussian when NO point of the box can reach
// alpha >= 1/255 (so the result is identical to walking the full range).
#pragma once
#include "common.cuh"

namespace tgs {

constexpr int kRasterWarps = 8;                 // warps per block
constexpr int kRasterThreads = kRasterWarps * 32;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kLnAlphaMin = -5.541263545158426f;  // ln(1/255)

struct WarpBatch {
    float4 a[32];  // mx, my, -A/2, -B
    float4 b[32];  // -C/2, thr = ln(1/(255 o)) - 1e-5, opacity, bits: 1-based range position (fwd) / 0-based (bwd)
    float4 c[32];  // r, g, b, bits: Gaussian id
};

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
    float y;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Canonical power: fma(fma(-B, dy, (-A/2) dx), dx, ((-C/2) dy) dy)
__device__ __forceinline__ float splat_power(float nA, float nB, float nC, float dx, float dy) {
    return __fmaf_rn(__fmaf_rn(nB, dy, __fmul_rn(nA, dx)), dx, __fmul_rn(__fmul_rn(nC, dy), dy));
}

// blend threshold on power: alpha >= 1/255  <=>  power >= ln(1/(255 o)); lowered a hair so that
// rounding never rejects a Gaussian the exact alpha test (still applied afterwards) keeps
__device__ __forceinline__ float blend_threshold(float opacity) {
    return (kLnAlphaMin - kLn2 * lg2_approx(opacity)) - 1e-5f;
}

struct PixelBox { float x0, y0, x1, y1; };

// Conservative test: can the splat reach alpha >= 1/255 anywhere in the pixel box?
// q(d) = A dx^2 + 2 B dx dy + C dy^2 is minimised over the box exactly (the minimum of a convex
// quadratic over a box that does not contain its centre lies on an edge facing the centre: two 1-D
// minimisations with clamping); the splat may touch iff q_min <= 2 |thr|.  Slack 0.1 % + 1e-3.
__device__ __forceinline__ bool splat_may_touch(float mx, float my, float A, float B, float C, float thr,
                                                const PixelBox& bx) {
    if (thr > 0.0f) return false;  // opacity < 1/255: never blends
    const float X0 = bx.x0 - mx, X1 = bx.x1 - mx, Y0 = bx.y0 - my, Y1 = bx.y1 - my;
    const float dxc = fminf(fmaxf(0.0f, X0), X1), dyc = fminf(fmaxf(0.0f, Y0), Y1);
    const float xs = fminf(fmaxf(-B * dyc * rcp_approx(A), X0), X1);
    const float ys = fminf(fmaxf(-B * dxc * rcp_approx(C), Y0), Y1);
    const float q1 = A * xs * xs + 2.0f * B * xs * dyc + C * dyc * dyc;
    const float q2 = A * dxc * dxc + 2.0f * B * dxc * ys + C * ys * ys;
    const float lim = -2.002f * thr + 1e-3f;
    return !(fminf(q1, q2) > lim);  // NaN anywhere keeps the Gaussian
}

struct UnitInfo {
    uint32_t start, end;  // tile range in gid_sorted
    uint32_t slot;        // this lane's index in the sampled-pixel list (valid if active)
    bool active;
};

// unit u -> (sampled tile u/8, pixel group u%8).  A full tile (256 pixels) is cut into 8x4-pixel
// blocks (compact boxes cull better); a partial tile into runs of 32 consecutive list entries.
__device__ __forceinline__ bool decode_unit(uint32_t u, int lane, const uint32_t* __restrict__ tiles,
                                            const uint32_t* __restrict__ tile_offsets,
                                            const uint32_t* __restrict__ tpo, UnitInfo& ui) {
    const uint32_t it = u >> 3, gi = u & 7u;
    const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
    if (gi * 32u >= m) return false;
    const uint32_t t = tiles[it];
    ui.start = tile_offsets[t];
    ui.end = tile_offsets[t + 1];
    if (m == 256u) {
        const uint32_t local = (((gi >> 1) * 4u + ((uint32_t)lane >> 3)) << 4) + (gi & 1u) * 8u + ((uint32_t)lane & 7u);
        ui.slot = p0 + local;
        ui.active = true;
    } else {
        ui.slot = p0 + gi * 32u + (uint32_t)lane;
        ui.active = gi * 32u + (uint32_t)lane < m;
    }
    return true;
}

// box of the warp's active pixels
__device__ __forceinline__ PixelBox warp_pixel_box(bool active, int ipx, int ipy) {
    PixelBox b;
    b.x0 = (float)__reduce_min_sync(0xffffffffu, active ? ipx : 0x7fffffff);
    b.y0 = (float)__reduce_min_sync(0xffffffffu, active ? ipy : 0x7fffffff);
    b.x1 = (float)__reduce_max_sync(0xffffffffu, active ? ipx : -1);
    b.y1 = (float)__reduce_max_sync(0xffffffffu, active ? ipy : -1);
    return b;
}

// the last warp to leave re-arms the scheduler counters for the next launch
__device__ __forceinline__ void scheduler_leave(uint32_t* sched, int lane) {
    if (lane == 0) {
        const uint32_t total = gridDim.x * kRasterWarps;
        if (atomicAdd(&sched[1], 1u) == total - 1u) {
            sched[0] = 0u;
            sched[1] = 0u;
            __threadfence();
        }
    }
}

}  // namespace tgs
