// Shared pieces of the two raster kernels: work decomposition, the producer warp that stages a
// sampled tile's depth-ordered Gaussians through a shared-memory ring, the conservative per-warp
// cull and the unit decoding.
//
// Work decomposition (both kernels).  A thread block is persistent and handles one SAMPLED TILE at
// a time (sampled pixels are listed tile by tile; tile-parallel execution).  It has
// one PRODUCER warp and eight CONSUMER warps:
//   * consumer w owns unit w of the tile = 32 sampled pixels (an 8x4 block of a full tile, or 32
//     consecutive entries of a partial tile's pixel list), so warps stay full on a sparse pixel set;
//   * the producer pulls tiles from a global atomic counter, walks the tile's range in gid_sorted
//     and gathers each Gaussian's 48-byte splat record ONCE per tile into a ring of shared-memory
//     stages (kStages x 64..128 records), pre-scaled for the inner loops.  Full / empty
//     mbarriers per stage decouple it from the consumers, and the consumers from each other, by up
//     to kStages stages; it runs ahead into the next tile while the consumers finish the current one.
//     (profiles/r1b: with every warp gathering its own records the L1 LSU data pipe was ~70-80 %
//     busy, mostly on 32-line gathers repeated by the 8 warps of a tile, and was the limiter.)
//   * each consumer reads a stage 32 records at a time (conflict-free float4 planes), tests them
//     against the bounding box of ITS 32 pixels, compacts the survivors into its private slice in
//     range order and runs its inner loop over survivors only.
//   * the stream of stages carries the control flow: a stage's header names the sampled tile it
//     starts (or "continuation" / "end of work"), so only the producer talks to the scheduler.
//   * forward early termination: a consumer whose pixels are all saturated publishes the tile's
//     sequence number; the producer stops a tile's stream as soon as all eight have.
//
// The cull is conservative: it only drops a Gaussian when NO point of the box can reach
// alpha >= 1/255 (so the result is identical to walking the full range).
#pragma once
#include "common.cuh"

namespace tgs {

constexpr int kConsumers = 8;                        // consumer warps per block = units per tile
constexpr int kRasterThreads = (kConsumers + 1) * 32;  // + 1 producer warp
constexpr uint32_t kLitePixels = 32;  // tiles with at most this many sampled pixels go to the warp-per-tile kernels (raster_lite.cu)
constexpr uint32_t kHdrCont = 0xfffffffeu, kHdrEnd = 0xffffffffu;
constexpr float kLog2e = 1.4426950408889634f;
constexpr float kLn2 = 0.6931471805599453f;
constexpr float kLnAlphaMin = -5.541263545158426f;  // ln(1/255)

// One staged record, split into planes so that every consumer access is as narrow as its use (profiles/r2b: both
// raster kernels are bound by shared-memory wavefronts -- a warp-wide broadcast LDS.128 costs 2, LDS.64 / LDS.32 1):
//   p0 = mx, my, -A/2, -B      p1 = -C/2, opacity, red, green      ct = -C/2, thr = ln(1/(255 o)) - 1e-5 (cull only)
//   bl = blue                  id = Gaussian id                     dz = depth (statistics forward only)
// Entry ENTRIES of every plane is a DUMMY record (opacity 0, id 0xffffffff) that never blends: lists of survivor
// indices are padded with it to a multiple of four.
struct StageInfo {
    uint32_t cnt;   // valid records in this stage
    uint32_t hdr;   // index into tiles[] of the sampled tile this stage STARTS, kHdrCont, or kHdrEnd
    uint32_t base;  // range position (0-based) of record 0; forward ascending, backward descending
    uint32_t rowmajor;  // backward, on a tile's first stage: 1 = the tile lists 256 pixels in row-major order (else 0)
};
template <int ENTRIES, bool DEPTH = false>
struct Stage {
    float4 p0[ENTRIES + 4];
    float4 p1[ENTRIES + 4];
    float2 ct[ENTRIES + 4];
    float bl[ENTRIES + 4];
    uint32_t id[ENTRIES + 4];
};
// DEPTH = true (statistics forward, which copies its survivors into a private batch and needs the depth): three
// float4 planes   p0 = mx, my, -A/2, -B      p1 = -C/2, thr, opacity, red      p2 = green, blue, bits: Gaussian id, depth
template <int ENTRIES>
struct Stage<ENTRIES, true> {
    float4 p0[ENTRIES];
    float4 p1[ENTRIES];
    float4 p2[ENTRIES];
};
template <int ENTRIES, bool DEPTH = false, int STAGES = 4>
struct Ring {
    static constexpr int kEntries = ENTRIES;
    static constexpr bool kDepth = DEPTH;
    static constexpr int kStages = STAGES;
    Stage<ENTRIES, DEPTH> st[kStages];
    unsigned long long full[kStages], empty[kStages];
    StageInfo info[kStages];
    uint32_t done_seq[kConsumers];  // consumer w needs nothing more of the block's done_seq[w]-th tile
};

// a consumer's private list of the stage entries that survived its cull, in range order (block-per-tile kernels)
template <int ENTRIES>
struct WarpList {
    uint32_t idx[ENTRIES + 4];
};

// a warp's private survivors of one 32-record batch (warp-per-tile kernels, raster_lite.cu)
struct WarpBatch {
    float4 a[32];  // mx, my, -A/2, -B
    float4 b[32];  // -C/2, thr, opacity, bits: range position (fwd: 1-based, bwd: 0-based)
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

// ---- mbarrier (shared::cta) ------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {  // release.cta
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, uint32_t parity) {  // acquire.cta
    const uint32_t a = smem_u32(bar);
    // A warp that waits (its pixels are saturated, it has no contributor left, or the producer is behind) must not
    // take issue slots from the warps that work: profiles/r2b, r2c -- with a fixed 128 ns sleep, and likewise with
    // try_wait's suspend-time hint (which the hardware caps far below a stage's duration), the polling loop was
    // 16-18 % of all executed instructions while `not selected` was the top stall.  Exponential back-off: a short
    // wait wakes within tens of ns, a long one (waiting for the other warps of the tile) polls every 2 us.  (Letting a
    // warp with nothing left in its tile start at 2 us was slower: its late arrival on `empty` stalls the producer.)
    uint32_t ns = 32;
    for (;;) {
        uint32_t ok;
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(a), "r"(parity)
            : "memory");
        if (ok) break;
        __nanosleep(ns);
        ns = min(ns * 2u, 2048u);
    }
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
// power(d) = nA dx^2 + nB dx dy + nC dy^2 (nA = -A/2, nB = -B, nC = -C/2) is maximised over the box
// exactly (the maximum of a concave quadratic over a box that does not contain its centre lies on
// an edge facing the centre: two 1-D maximisations with clamping); the splat may touch iff
// power_max >= thr.  Slack 0.1 % + 5e-4.
__device__ __forceinline__ bool splat_may_touch(float mx, float my, float nA, float nB, float nC, float thr,
                                                const PixelBox& bx) {
    if (thr > 0.0f) return false;  // opacity < 1/255: never blends
    const float X0 = bx.x0 - mx, X1 = bx.x1 - mx, Y0 = bx.y0 - my, Y1 = bx.y1 - my;
    const float dxc = fminf(fmaxf(0.0f, X0), X1), dyc = fminf(fmaxf(0.0f, Y0), Y1);
    const float xs = fminf(fmaxf(-0.5f * nB * dyc * rcp_approx(nA), X0), X1);
    const float ys = fminf(fmaxf(-0.5f * nB * dxc * rcp_approx(nC), Y0), Y1);
    const float h1 = nA * xs * xs + nB * xs * dyc + nC * dyc * dyc;
    const float h2 = nA * dxc * dxc + nB * dxc * ys + nC * ys * ys;
    const float lim = 1.001f * thr - 5e-4f;
    return !(fmaxf(h1, h2) < lim);  // NaN anywhere keeps the Gaussian
}

struct UnitInfo {
    uint32_t start, end;  // tile range in gid_sorted
    uint32_t slot;        // this lane's index in the sampled-pixel list (valid if active)
    bool active;
    bool full;            // the tile lists all 256 pixels: the unit is slots of an 8x4 block -- lane j at (j & 7, j >> 3) from
                          // lane 0 IF the list is row-major (StageInfo::rowmajor)
};

// (sampled tile `it`, pixel group `gi`).  A full tile (256 pixels) is cut into 8x4-pixel blocks
// (compact boxes cull better); a partial tile into runs of 32 consecutive list entries.
__device__ __forceinline__ bool decode_unit(uint32_t it, uint32_t gi, int lane, const uint32_t* __restrict__ tiles,
                                            const uint32_t* __restrict__ tile_offsets,
                                            const uint32_t* __restrict__ tpo, UnitInfo& ui) {
    const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
    if (gi * 32u >= m) return false;
    const uint32_t t = tiles[it];
    ui.start = tile_offsets[t];
    ui.end = tile_offsets[t + 1];
    ui.full = m == 256u;
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

template <class RingT>
__device__ __forceinline__ void ring_init(RingT& R) {
    if (threadIdx.x == 0) {
        for (int s = 0; s < RingT::kStages; ++s) {
            mbar_init(&R.full[s], 1u);
            mbar_init(&R.empty[s], (uint32_t)kConsumers);
        }
        for (int w = 0; w < kConsumers; ++w) R.done_seq[w] = 0u;
        if constexpr (!RingT::kDepth) {
            for (int s = 0; s < RingT::kStages; ++s) {  // the dummy record of every stage
                auto& st = R.st[s];
                constexpr int E = RingT::kEntries;
                st.p0[E] = make_float4(0.f, 0.f, 0.f, 0.f);
                st.p1[E] = make_float4(0.f, 0.f, 0.f, 0.f);
                st.ct[E] = make_float2(0.f, 1.f);
                st.bl[E] = 0.f;
                st.id[E] = 0xffffffffu;
            }
        }
    }
    __syncthreads();
}

// The producer warp.  BWD = false: ranges front to back, stops a tile early once every consumer is
// saturated.  BWD = true: from the tile's deepest contributor (max n_contrib) back to front.
template <bool BWD, class RingT>
__device__ __forceinline__ void producer_loop(RingT& R, const float4* __restrict__ splats,
                                              const uint32_t* __restrict__ tile_offsets,
                                              const uint32_t* __restrict__ gid_sorted, uint32_t k,
                                              const uint32_t* __restrict__ tiles, const uint32_t* __restrict__ tpo,
                                              const uint32_t* __restrict__ n_contrib, uint32_t* __restrict__ sched,
                                              int lane, uint32_t lite_max = 0u,
                                              const uint32_t* __restrict__ pix = nullptr, uint32_t W = 0u) {
    uint32_t gchunk = 0, seq = 0;
    for (;;) {
        uint32_t it = 0;
        if (lane == 0) it = atomicAdd(&sched[0], 1u);
        it = __shfl_sync(0xffffffffu, it, 0);
        if (it >= k) break;
        if (lite_max != 0u && tpo[it + 1] - tpo[it] <= lite_max) continue;  // a warp-per-tile kernel's tile
        ++seq;
        const uint32_t t = tiles[it];
        const uint32_t start = tile_offsets[t];
        uint32_t len = tile_offsets[t + 1] - start;
        uint32_t rowmajor = 0u;
        if (BWD) {
            const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
            uint32_t mx = 0;
            for (uint32_t i = lane; i < m; i += 32) mx = max(mx, n_contrib[p0 + i]);
            len = __reduce_max_sync(0xffffffffu, mx);
            // The backward's separable phase 2 takes a unit's pixels from lane 0's pixel plus a fixed 8x4 offset, which
            // holds when the tile's 256 pixels are listed row-major (as tgs_sample writes them).  A caller's own list may
            // be in any order, so the producer -- which has registers to spare and walks the tile's slots anyway --
            // verifies it once per tile; any other order takes the general phase 2, which reads px, py per pixel.
            if (m == 256u && pix != nullptr) {
                const uint32_t id0 = pix[p0];
                bool ok = id0 % W + 15u < W;  // no wrap into the next image row
#pragma unroll
                for (uint32_t i = lane; i < 256u; i += 32)
                    ok = ok && pix[p0 + i] == id0 + (i >> 4) * W + (i & 15u);
                rowmajor = __all_sync(0xffffffffu, ok) ? 1u : 0u;
            }
        }
        uint32_t produced = 0;
        bool first = true;
        do {
            if (!BWD && !first) {
                const uint32_t d = lane < kConsumers ? *(volatile uint32_t*)&R.done_seq[lane] : seq;
                if (__all_sync(0xffffffffu, d >= seq)) break;
            }
            const uint32_t s = gchunk % RingT::kStages;
            mbar_wait(&R.empty[s], ((gchunk / RingT::kStages) & 1u) ^ 1u);
            constexpr int kStageEntries = RingT::kEntries;
            const uint32_t cnt = min((uint32_t)kStageEntries, len - produced);
            auto& st = R.st[s];
            // two batches of 32 records at a time: six independent gathers in flight per lane
#pragma unroll 1
            for (int h = 0; h < kStageEntries / 64; ++h) {
                if ((uint32_t)h * 64u >= cnt) break;
                uint32_t g[2];
                float4 r0[2], r1[2];
                float2 r2x[2];  // blue, depth
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    const uint32_t i = h * 64 + j * 32 + lane;
                    const uint32_t pos = BWD ? (len - 1u - produced - i) : (produced + i);
                    g[j] = i < cnt ? gid_sorted[start + pos] : 0xffffffffu;
                }
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    if (g[j] != 0xffffffffu) {
                        r0[j] = splats[3 * (size_t)g[j]];
                        r1[j] = splats[3 * (size_t)g[j] + 1];
                        r2x[j] = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(splats) + (size_t)g[j] * kSplatWords + 8);
                    }
                }
#pragma unroll
                for (int j = 0; j < 2; ++j) {
                    if (g[j] != 0xffffffffu) {
                        const int i = h * 64 + j * 32 + lane;
                        const float nC = -0.5f * r1[j].x;
                        st.p0[i] = make_float4(r0[j].x, r0[j].y, -0.5f * r0[j].z, -r0[j].w);
                        if constexpr (RingT::kDepth) {
                            st.p1[i] = make_float4(nC, blend_threshold(r1[j].y), r1[j].y, r1[j].z);
                            st.p2[i] = make_float4(r1[j].w, r2x[j].x, __uint_as_float(g[j]), r2x[j].y);
                        } else {
                            st.p1[i] = make_float4(nC, r1[j].y, r1[j].z, r1[j].w);
                            st.ct[i] = make_float2(nC, blend_threshold(r1[j].y));
                            st.bl[i] = r2x[j].x;
                            st.id[i] = g[j];
                        }
                    }
                }
            }
            if (lane == 0) {
                StageInfo inf;
                inf.cnt = cnt;
                inf.hdr = first ? it : kHdrCont;
                inf.base = BWD ? (len - 1u - produced) : produced;
                inf.rowmajor = rowmajor;
                R.info[s] = inf;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(&R.full[s]);
            ++gchunk;
            produced += cnt;
            first = false;
        } while (produced < len);
    }
    // end of work
    const uint32_t s = gchunk % RingT::kStages;
    mbar_wait(&R.empty[s], ((gchunk / RingT::kStages) & 1u) ^ 1u);
    if (lane == 0) {
        StageInfo inf;
        inf.cnt = 0; inf.hdr = kHdrEnd; inf.base = 0; inf.rowmajor = 0;
        R.info[s] = inf;
        mbar_arrive(&R.full[s]);
        // the last producer to leave re-arms the scheduler counters for the next launch
        if (atomicAdd(&sched[1], 1u) == gridDim.x - 1u) {
            sched[0] = 0u;
            sched[1] = 0u;
            __threadfence();
        }
    }
}

}  // namespace tgs
