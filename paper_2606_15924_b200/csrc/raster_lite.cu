// Sparse-list variants of the two raster kernels: ONE WARP PER SAMPLED TILE, for tiles that hold at most
// 32 sampled pixels (one unit) -- the paper's own regime, N_pix ~ 25 pixels in EVERY tile (PAPER.md:130,
// 470; tgs_sample_paper).  The block-per-tile kernels (raster_fwd.cu / raster_bwd.cu) give such a tile a
// whole block of which one consumer warp works and seven idle, and the producer's staging buys nothing
// because nobody shares the records (measured: 25 pixels per tile cost as much as 256).  Here every warp
// of a block walks its OWN tile: it gathers the tile's records itself, 32 at a time (ids prefetched two
// batches ahead, records one), culls them against the box of its pixels, compacts the survivors into its
// private shared-memory slice and runs the same inner loops as the block kernels' consumers.  Warps are
// persistent and pull tiles from a global counter.
//
// The two families split the tiles of one call between them by the tile's pixel count (<= 32: here),
// so a call always launches both; each skips the other's tiles.
#include "raster_common.cuh"

namespace tgs {

namespace {

constexpr int kLiteWarps = 8;

struct LiteRec {  // one gathered record, pre-scaled like the staged ones
    float4 p0;    // mx, my, -A/2, -B
    float4 p1;    // -C/2, thr, opacity, red
    float4 p2;    // green, blue, bits: Gaussian id, depth
};

__device__ __forceinline__ LiteRec lite_load(const float4* __restrict__ splats, uint32_t g) {
    LiteRec r;
    r.p0 = make_float4(0.f, 0.f, 0.f, 0.f); r.p1 = r.p0; r.p2 = r.p0;
    if (g != 0xffffffffu) {
        const float4 a = splats[3 * (size_t)g];
        const float4 b = splats[3 * (size_t)g + 1];
        const float2 c = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(splats) + (size_t)g * kSplatWords + 8);
        r.p0 = make_float4(a.x, a.y, -0.5f * a.z, -a.w);
        r.p1 = make_float4(-0.5f * b.x, blend_threshold(b.y), b.y, b.z);
        r.p2 = make_float4(b.w, c.x, __uint_as_float(g), c.y);
    }
    return r;
}

// persistent-warp scheduler: tiles come from sched[0]; the last warp to leave re-arms both words
__device__ __forceinline__ uint32_t lite_next(uint32_t* sched, int lane) {
    uint32_t it = 0;
    if (lane == 0) it = atomicAdd(&sched[0], 1u);
    return __shfl_sync(0xffffffffu, it, 0);
}
__device__ __forceinline__ void lite_leave(uint32_t* sched, int lane) {
    if (lane == 0) {
        const uint32_t total = gridDim.x * kLiteWarps;
        if (atomicAdd(&sched[1], 1u) == total - 1u) {
            sched[0] = 0u;
            sched[1] = 0u;
            __threadfence();
        }
    }
}

template <bool COUNT>
__global__ void __launch_bounds__(kLiteWarps * 32)
raster_fwd_lite_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                       const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                       const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                       float* __restrict__ out_color, float* __restrict__ out_T, uint32_t* __restrict__ n_contrib,
                       uint32_t* __restrict__ n_walked, uint32_t* __restrict__ n_blended, uint32_t* __restrict__ sched) {
    __shared__ __align__(16) WarpBatch batch[kLiteWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpBatch& sb = batch[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    for (;;) {
        const uint32_t it = lite_next(sched, lane);
        if (it >= (uint32_t)k) break;
        const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
        if (m == 0u || m > kLitePixels) continue;  // the block kernel's tile
        const uint32_t t = tiles[it];
        const uint32_t start = tile_offsets[t], len = tile_offsets[t + 1] - start;
        const bool active = (uint32_t)lane < m;
        const uint32_t slot = p0 + (uint32_t)lane;
        int ipx = 0, ipy = 0;
        if (active) {
            const uint32_t id = pix[slot];
            ipx = (int)(id % (uint32_t)cam.W);
            ipy = (int)(id / (uint32_t)cam.W);
        }
        const PixelBox box = warp_pixel_box(active, ipx, ipy);
        const float px = (float)ipx;
        bool alive = active;  // sampled and not yet terminated: gates the blend decision only (no loop-carried chain through px)
        const float py = (float)ipy;
        float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
        uint32_t last = 0, walked = len, blended = 0;

        auto gid_at = [&](uint32_t pos) { return pos < len ? gid_sorted[start + pos] : 0xffffffffu; };
        uint32_t g_next = gid_at((uint32_t)lane + 32u);
        LiteRec cur = lite_load(splats, gid_at((uint32_t)lane));
        for (uint32_t b0 = 0; b0 < len; b0 += 32) {
            const LiteRec nxt = lite_load(splats, g_next);  // records of the next batch, ids of the one after
            g_next = gid_at(b0 + 64u + (uint32_t)lane);
            // ---- cull this batch against the pixel box, compact survivors in range order ----
            const bool have = b0 + (uint32_t)lane < len;
            const bool pass = have && splat_may_touch(cur.p0.x, cur.p0.y, cur.p0.z, cur.p0.w, cur.p1.x, cur.p1.y, box);
            const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
            const int cnt = __popc(ballot);
            __syncwarp();
            if (pass) {
                const int s = __popc(ballot & lt_mask);
                sb.a[s] = cur.p0;
                sb.b[s] = make_float4(cur.p1.x, cur.p1.y, cur.p1.z, __uint_as_float(b0 + (uint32_t)lane + 1u));
                sb.c[s] = make_float4(cur.p1.w, cur.p2.x, cur.p2.y, 0.f);
            }
            __syncwarp();
#pragma unroll 4
            for (int e = 0; e < cnt; ++e) {
                const float4 a = sb.a[e];
                const float4 b = sb.b[e];
                const float4 c = sb.c[e];
                const float dx = a.x - px, dy = a.y - py;
                const float power = splat_power(a.z, a.w, b.x, dx, dy);
                const float alpha = fminf(kAlphaMax, __fmul_rn(b.z, ex2_approx(power * kLog2e)));
                const bool blend = alive && (power <= 0.0f) && !(alpha < kAlphaMin);
                const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                const bool term = blend && (Tn < kTMin);
                const bool upd = blend && !term;
                const float w = upd ? alpha * T : 0.0f;
                C0 = fmaf(c.x, w, C0); C1 = fmaf(c.y, w, C1); C2 = fmaf(c.z, w, C2);
                T = upd ? Tn : T;
                last = upd ? __float_as_uint(b.w) : last;
                if (COUNT) {
                    blended += upd ? 1u : 0u;
                    walked = term ? __float_as_uint(b.w) : walked;
                }
                alive = alive && !term;
            }
            if (!__any_sync(0xffffffffu, alive)) break;
            cur = nxt;
        }
        if (active) {
            out_color[3 * (size_t)slot] = fmaf(T, cam.bg[0], C0);
            out_color[3 * (size_t)slot + 1] = fmaf(T, cam.bg[1], C1);
            out_color[3 * (size_t)slot + 2] = fmaf(T, cam.bg[2], C2);
            out_T[slot] = T;
            n_contrib[slot] = last;
            if (COUNT) {
                if (n_walked) n_walked[slot] = walked;
                if (n_blended) n_blended[slot] = blended;
            }
        }
    }
    lite_leave(sched, lane);
}

// ---- backward ---------------------------------------------------------------------------------------
__device__ __forceinline__ void red_add_v4(float4* p, float x, float y, float z, float w) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

constexpr int kSlots = 16;     // Gaussians per transposed tile
constexpr int kTStride = 33;   // float2 row stride: conflict-free for both phases

struct LiteXpose {
    float2 v[kSlots * kTStride];  // [slot][pixel] = (dpow, w)
    float4 ma[kSlots];            // mx, my, -A/2, -B
    float4 mb[kSlots];            // -C/2, opacity, bits: Gaussian id, unused
    float4 pa[32];                // per pixel: px, py, g0, g1
    float pb[32];                 // per pixel: g2
};

struct LiteBwdShared {
    WarpBatch batch[kLiteWarps];
    LiteXpose xpose[kLiteWarps];
};

__global__ void __launch_bounds__(kLiteWarps * 32)
raster_bwd_lite_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                       const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                       const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                       const float* __restrict__ out_T, const uint32_t* __restrict__ n_contrib,
                       const float* __restrict__ dL_dcolor, float* __restrict__ dL_dsplats, uint32_t* __restrict__ sched) {
    extern __shared__ __align__(16) unsigned char lite_smem_raw[];  // > 48 KB: dynamic, opted in by the launcher
    LiteBwdShared& sm = *reinterpret_cast<LiteBwdShared*>(lite_smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpBatch& sb = sm.batch[warp];
    LiteXpose& sx = sm.xpose[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int slot2 = lane & (kSlots - 1), half = lane >> 4;  // phase-2 role of this lane
    int m = 0;  // Gaussians pending in the transposed tile

    // ---- phase 2: lane = (Gaussian slot2, pixel half); nine sums over 16 pixels in registers ----
    auto flush = [&]() {
        __syncwarp();
        const float4 ga = sx.ma[slot2];
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f, a5 = 0.f, a6 = 0.f, a7 = 0.f, a8 = 0.f;
        const float2* vrow = sx.v + slot2 * kTStride + half * 16;
        const float4* prow = sx.pa + half * 16;
        const float* qrow = sx.pb + half * 16;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float2 v = vrow[i];
            const float4 q = prow[i];
            const float h2 = qrow[i];
            const float dx = ga.x - q.x, dy = ga.y - q.y;
            const float t0 = v.x * dx, t1 = v.x * dy;
            a0 += t0; a1 += t1;
            a2 = fmaf(t0, dx, a2); a3 = fmaf(t0, dy, a3); a4 = fmaf(t1, dy, a4);
            a5 += v.x;
            a6 = fmaf(v.y, q.z, a6); a7 = fmaf(v.y, q.w, a7); a8 = fmaf(v.y, h2, a8);
        }
        a0 += __shfl_xor_sync(0xffffffffu, a0, 16); a1 += __shfl_xor_sync(0xffffffffu, a1, 16);
        a2 += __shfl_xor_sync(0xffffffffu, a2, 16); a3 += __shfl_xor_sync(0xffffffffu, a3, 16);
        a4 += __shfl_xor_sync(0xffffffffu, a4, 16); a5 += __shfl_xor_sync(0xffffffffu, a5, 16);
        a6 += __shfl_xor_sync(0xffffffffu, a6, 16); a7 += __shfl_xor_sync(0xffffffffu, a7, 16);
        a8 += __shfl_xor_sync(0xffffffffu, a8, 16);
        if (slot2 < m) {
            const float4 gb = sx.mb[slot2];
            float4* dst = reinterpret_cast<float4*>(dL_dsplats + (size_t)__float_as_uint(gb.z) * kSplatWords);
            const float dmx = fmaf(2.0f * ga.z, a0, ga.w * a1), dmy = fmaf(2.0f * gb.x, a1, ga.w * a0);
            const float dop = a5 / gb.y;
            if (half == 0) {
                red_add_v4(dst + 0, dmx, dmy, -0.5f * a2, -a3);
                red_add_v4(dst + 2, a8, 0.f, 0.f, 0.f);
            } else {
                red_add_v4(dst + 1, -0.5f * a4, dop, a6, a7);
            }
        }
        m = 0;
        __syncwarp();
    };

    for (;;) {
        const uint32_t it = lite_next(sched, lane);
        if (it >= (uint32_t)k) break;
        const uint32_t p0 = tpo[it], np = tpo[it + 1] - p0;
        if (np == 0u || np > kLitePixels) continue;  // the block kernel's tile
        const uint32_t t = tiles[it];
        const uint32_t start = tile_offsets[t];
        const bool active = (uint32_t)lane < np;
        int ipx = 0, ipy = 0;
        float Tf = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f;
        uint32_t last = 0;
        if (active) {
            const uint32_t o = p0 + (uint32_t)lane;
            const uint32_t id = pix[o];
            ipx = (int)(id % (uint32_t)cam.W);
            ipy = (int)(id / (uint32_t)cam.W);
            Tf = out_T[o];
            last = n_contrib[o];
            g0 = dL_dcolor[3 * (size_t)o]; g1 = dL_dcolor[3 * (size_t)o + 1]; g2 = dL_dcolor[3 * (size_t)o + 2];
        }
        const uint32_t len = __reduce_max_sync(0xffffffffu, last);  // deepest contributor of the tile's pixels
        if (len == 0u) continue;
        const PixelBox box = warp_pixel_box(active, ipx, ipy);
        const float px = (float)ipx, py = (float)ipy;
        const float bgdot = (cam.bg[0] * g0 + cam.bg[1] * g1 + cam.bg[2] * g2) * Tf;
        float T = Tf, Sg = 0.f;
        __syncwarp();
        sx.pa[lane] = make_float4(px, py, g0, g1);
        sx.pb[lane] = g2;

        // batch b holds range positions len-1-32b-lane (descending)
        auto gid_at = [&](uint32_t i) { return i < len ? gid_sorted[start + (len - 1u - i)] : 0xffffffffu; };
        uint32_t g_next = gid_at((uint32_t)lane + 32u);
        LiteRec cur = lite_load(splats, gid_at((uint32_t)lane));
        for (uint32_t b0 = 0; b0 < len; b0 += 32) {
            const LiteRec nxt = lite_load(splats, g_next);
            g_next = gid_at(b0 + 64u + (uint32_t)lane);
            const uint32_t i = b0 + (uint32_t)lane;
            const bool have = i < len;
            const bool pass = have && splat_may_touch(cur.p0.x, cur.p0.y, cur.p0.z, cur.p0.w, cur.p1.x, cur.p1.y, box);
            const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
            const int cnt = __popc(ballot);
            __syncwarp();
            if (pass) {
                const int s = __popc(ballot & lt_mask);
                sb.a[s] = cur.p0;
                sb.b[s] = make_float4(cur.p1.x, cur.p1.y, cur.p1.z, __uint_as_float(len - 1u - i));  // 0-based range position
                sb.c[s] = make_float4(cur.p1.w, cur.p2.x, cur.p2.y, cur.p2.z);
            }
            __syncwarp();
            int e = 0;
            while (e < cnt) {
                // ---- phase 1: replay the next survivors (as many as fit in the transposed tile), branch free ----
                const int take = min(cnt - e, kSlots - m);
                const float4* sa = sb.a + e;
                float2* vdst = sx.v + m * kTStride + lane;
                float4* mdst = sx.ma + m;
#pragma unroll 2
                for (int ii = 0; ii < take; ++ii) {
                    const float4 a = sa[ii];
                    const float4 b = sa[32 + ii];
                    const float4 c = sa[64 + ii];
                    const float dx = a.x - px, dy = a.y - py;
                    const float power = splat_power(a.z, a.w, b.x, dx, dy);
                    const float G = ex2_approx(fminf(power, 0.0f) * kLog2e);
                    const float oG = __fmul_rn(b.z, G);
                    const float alpha = fminf(kAlphaMax, oG);
                    const bool valid = (__float_as_uint(b.w) < last) && (power <= 0.0f) && !(alpha < kAlphaMin);
                    const float om = 1.0f - alpha;
                    const float rom = rcp_approx(om);
                    const float Tk = T * rom;  // T_k
                    const float cg = fmaf(c.z, g2, fmaf(c.y, g1, c.x * g0));
                    const float dL_dalpha = fmaf(cg - Sg, Tk, -bgdot * rom);
                    const float dpow = (valid && oG < kAlphaMax) ? oG * dL_dalpha : 0.0f;  // dL/dpower
                    const float w = valid ? alpha * Tk : 0.0f;
                    T = valid ? Tk : T;
                    Sg = valid ? fmaf(alpha, cg, om * Sg) : Sg;
                    vdst[ii * kTStride] = make_float2(dpow, w);
                }
                if (lane < take) {  // the Gaussians' parameters for phase 2: one parallel copy per group
                    const float4 b = sa[32 + lane];
                    mdst[lane] = sa[lane];
                    mdst[kSlots + lane] = make_float4(b.x, b.z, sa[64 + lane].w, 0.f);
                }
                e += take;
                m += take;
                if (m == kSlots) flush();
            }
            cur = nxt;
        }
        if (m > 0) flush();  // tail of this tile (the per-pixel arrays change with the next one)
    }
    lite_leave(sched, lane);
}

// ---- statistics forward (tgs_raster_stats_sparse) -----------------------------------------------------
struct LiteStatXpose {
    float v[kSlots * kTStride];  // [slot][pixel] = w  (row stride 33)
    float4 ma[kSlots];           // mx, my, -A/2, -B
    float2 mb[kSlots];           // -C/2, bits: Gaussian id
    float4 pa[32];               // per pixel: px, py, e(p), unused
};
struct LiteStatShared {
    WarpBatch batch[kLiteWarps];
    LiteStatXpose xpose[kLiteWarps];
};

__global__ void __launch_bounds__(kLiteWarps * 32)
raster_stats_lite_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                         const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                         const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                         const float* __restrict__ pix_err, float* __restrict__ stats, float* __restrict__ out_depth,
                         uint32_t* __restrict__ sched) {
    __shared__ __align__(16) LiteStatShared sm;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpBatch& sb = sm.batch[warp];
    LiteStatXpose& sx = sm.xpose[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int slot2 = lane & (kSlots - 1), half = lane >> 4;
    int m = 0;

    auto flush = [&]() {
        __syncwarp();
        const float4 ga = sx.ma[slot2];
        const float2 gb = sx.mb[slot2];
        float E = 0.f, D = 0.f, Wt = 0.f;
        const float* vrow = sx.v + slot2 * kTStride + half * 16;
        const float4* prow = sx.pa + half * 16;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float w = vrow[i];
            const float4 q = prow[i];
            const float pw = splat_power(ga.z, ga.w, gb.x, ga.x - q.x, ga.y - q.y);
            Wt += w;
            E = fmaf(w, q.z, E);
            D = fmaf(w, -2.0f * pw, D);
        }
        E += __shfl_xor_sync(0xffffffffu, E, 16);
        D += __shfl_xor_sync(0xffffffffu, D, 16);
        Wt += __shfl_xor_sync(0xffffffffu, Wt, 16);
        if (slot2 < m && half == 0) red_add_v4(reinterpret_cast<float4*>(stats) + __float_as_uint(gb.y), E, D, Wt, 0.f);
        m = 0;
        __syncwarp();
    };

    for (;;) {
        const uint32_t it = lite_next(sched, lane);
        if (it >= (uint32_t)k) break;
        const uint32_t p0 = tpo[it], np = tpo[it + 1] - p0;
        if (np == 0u || np > kLitePixels) continue;  // the block kernel's tile
        const uint32_t t = tiles[it];
        const uint32_t start = tile_offsets[t], len = tile_offsets[t + 1] - start;
        const bool active = (uint32_t)lane < np;
        const uint32_t slot = p0 + (uint32_t)lane;
        int ipx = 0, ipy = 0;
        float e_p = 0.f;
        if (active) {
            const uint32_t id = pix[slot];
            ipx = (int)(id % (uint32_t)cam.W);
            ipy = (int)(id / (uint32_t)cam.W);
            e_p = pix_err[slot];
        }
        const PixelBox box = warp_pixel_box(active, ipx, ipy);
        const float px = (float)ipx;
        bool alive = active;  // sampled and not yet terminated: gates the blend decision only (no loop-carried chain through px)
        const float py = (float)ipy;
        float T = 1.0f, zacc = 0.f;
        __syncwarp();
        sx.pa[lane] = make_float4((float)ipx, (float)ipy, e_p, 0.f);

        auto gid_at = [&](uint32_t pos) { return pos < len ? gid_sorted[start + pos] : 0xffffffffu; };
        uint32_t g_next = gid_at((uint32_t)lane + 32u);
        LiteRec cur = lite_load(splats, gid_at((uint32_t)lane));
        for (uint32_t b0 = 0; b0 < len; b0 += 32) {
            const LiteRec nxt = lite_load(splats, g_next);
            g_next = gid_at(b0 + 64u + (uint32_t)lane);
            const bool have = b0 + (uint32_t)lane < len;
            const bool pass = have && splat_may_touch(cur.p0.x, cur.p0.y, cur.p0.z, cur.p0.w, cur.p1.x, cur.p1.y, box);
            const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
            const int cnt = __popc(ballot);
            __syncwarp();
            if (pass) {
                const int s = __popc(ballot & lt_mask);
                sb.a[s] = cur.p0;
                sb.b[s] = make_float4(cur.p1.x, cur.p1.y, cur.p1.z, 0.f);
                sb.c[s] = make_float4(cur.p2.w, cur.p2.z, 0.f, 0.f);  // depth, bits: Gaussian id
            }
            __syncwarp();
            int e = 0;
            while (e < cnt) {
                const int take = min(cnt - e, kSlots - m);
                const float4* sa = sb.a + e;
                float* vdst = sx.v + m * kTStride + lane;
#pragma unroll 2
                for (int ii = 0; ii < take; ++ii) {
                    const float4 a = sa[ii];
                    const float4 b = sa[32 + ii];
                    const float dx = a.x - px, dy = a.y - py;
                    const float power = splat_power(a.z, a.w, b.x, dx, dy);
                    const float alpha = fminf(kAlphaMax, __fmul_rn(b.z, ex2_approx(power * kLog2e)));
                    const bool blend = alive && (power <= 0.0f) && !(alpha < kAlphaMin);
                    const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                    const bool term = blend && (Tn < kTMin);
                    const bool upd = blend && !term;
                    const float w = upd ? alpha * T : 0.0f;
                    zacc = fmaf(w, sa[64 + ii].x, zacc);
                    T = upd ? Tn : T;
                    alive = alive && !term;
                    vdst[ii * kTStride] = w;
                }
                if (lane < take) {
                    sx.ma[m + lane] = sa[lane];
                    sx.mb[m + lane] = make_float2(sa[32 + lane].x, sa[64 + lane].y);
                }
                e += take;
                m += take;
                if (m == kSlots) flush();
            }
            if (!__any_sync(0xffffffffu, alive)) break;
            cur = nxt;
        }
        if (m > 0) flush();  // before the per-pixel array changes
        if (active && out_depth) out_depth[slot] = zacc;
    }
    lite_leave(sched, lane);
}

}  // namespace

cudaError_t launch_raster_stats_lite(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                                     const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                     const uint32_t* pix, const float* pix_err, float* stats, float* out_depth,
                                     uint32_t* sched, int num_sms, cudaStream_t s) {
    if (k <= 0) return cudaSuccess;
    int blocks = num_sms * 5;
    if (blocks > (k + kLiteWarps - 1) / kLiteWarps) blocks = (k + kLiteWarps - 1) / kLiteWarps;
    raster_stats_lite_kernel<<<blocks, kLiteWarps * 32, 0, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                               gid_sorted, k, tiles, tpo, pix, pix_err, stats, out_depth, sched);
    count_launches(1);
    return cudaGetLastError();
}

cudaError_t launch_raster_fwd_lite(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                                   const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                   const uint32_t* pix, float* out_color, float* out_T, uint32_t* n_contrib,
                                   uint32_t* n_walked, uint32_t* n_blended, uint32_t* sched, int num_sms, cudaStream_t s) {
    if (k <= 0) return cudaSuccess;
    int blocks = num_sms * 6;  // persistent warps; 48 resident warps per SM
    if (blocks > (k + kLiteWarps - 1) / kLiteWarps) blocks = (k + kLiteWarps - 1) / kLiteWarps;
    const float4* sp = reinterpret_cast<const float4*>(splats);
    if (n_walked || n_blended)
        raster_fwd_lite_kernel<true><<<blocks, kLiteWarps * 32, 0, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                        out_color, out_T, n_contrib, n_walked, n_blended, sched);
    else
        raster_fwd_lite_kernel<false><<<blocks, kLiteWarps * 32, 0, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                         out_color, out_T, n_contrib, n_walked, n_blended, sched);
    count_launches(1);
    return cudaGetLastError();
}

cudaError_t launch_raster_bwd_lite(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                                   const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                   const uint32_t* pix, const float* out_T, const uint32_t* n_contrib,
                                   const float* dL_dcolor, float* dL_dsplats, uint32_t* sched, int num_sms, cudaStream_t s) {
    if (k <= 0) return cudaSuccess;
    int blocks = num_sms * 4;  // 54 KB of shared memory per block
    if (blocks > (k + kLiteWarps - 1) / kLiteWarps) blocks = (k + kLiteWarps - 1) / kLiteWarps;
    static SmemOptIn opt;  // per device
    cudaError_t e = opt.ensure((const void*)raster_bwd_lite_kernel, sizeof(LiteBwdShared));
    if (e != cudaSuccess) return e;
    raster_bwd_lite_kernel<<<blocks, kLiteWarps * 32, sizeof(LiteBwdShared), s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                             gid_sorted, k, tiles, tpo, pix, out_T, n_contrib, dL_dcolor,
                                                             dL_dsplats, sched);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
