// tgs_raster_bwd_sparse, raster half: back-to-front replay of Eq. 1 over the sampled
// pixels only, producing dL/d(mean2D, conic, opacity, rgb) per Gaussian.
//
// Same decomposition as the forward (raster_common.cuh): persistent warps, one (tile, 32-pixel
// group) unit at a time, the tile's range walked from the warp's deepest contributor backwards in
// batches of 32 with the per-warp cull.  The gradient of one Gaussian is a sum over pixels; summing
// it with a shuffle tree per Gaussian costs more issue slots than the math itself (profiles/r1b),
// so the warp TRANSPOSES instead:
//   phase 1 (lane = pixel): per surviving Gaussian every lane replays its pixel and stores only the
//            two per-(pixel, Gaussian) scalars everything else is linear in -- dpow = dL/dpower and
//            w = alpha * T_k -- into a [16 Gaussians][32 pixels] shared-memory tile;
//   phase 2 (lane = Gaussian): when 16 Gaussians are pending, lane e (and lane e + 16 for the other
//            half of the pixels) sums Gaussian e's nine gradient components over the pixels in
//            registers -- plain FMAs, no shuffles -- and issues the global float atomics.
// So the per-Gaussian gradients are reduced over the warp's 32 pixels before any global atomic
// (north_star), with 9 shuffles per 16 Gaussians instead of 14 per Gaussian.
#include "raster_common.cuh"

namespace tgs {

namespace {

__device__ __forceinline__ void red_add_v4(float4* p, float x, float y, float z, float w) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

constexpr int kSlots = 16;     // Gaussians per transposed tile
constexpr int kTStride = 33;   // float2 row stride: conflict-free for both phases

struct WarpXpose {
    float2 v[kSlots * kTStride];  // [slot][pixel] = (dpow, w)
    float4 ma[kSlots];            // mx, my, -A/2, -B
    float4 mb[kSlots];            // -C/2, opacity, bits: Gaussian id, unused
    float4 pa[32];                // per pixel: px, py, g0, g1
    float pb[32];                 // per pixel: g2
};

__global__ void __launch_bounds__(kRasterThreads, 3)
raster_bwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  const float* __restrict__ out_T, const uint32_t* __restrict__ n_contrib,
                  const float* __restrict__ dL_dcolor, float* __restrict__ dL_dsplats, uint32_t* __restrict__ sched) {
    extern __shared__ __align__(16) unsigned char smem_raw[];  // > 48 KB: dynamic, opted in by the launcher
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpBatch& sb = reinterpret_cast<WarpBatch*>(smem_raw)[warp];
    WarpXpose& sx = reinterpret_cast<WarpXpose*>(smem_raw + kRasterWarps * sizeof(WarpBatch))[warp];
    const uint32_t num_units = (uint32_t)k * 8u;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int slot2 = lane & (kSlots - 1), half = lane >> 4;  // phase-2 role of this lane

    for (;;) {
        uint32_t u = 0;
        if (lane == 0) u = atomicAdd(&sched[0], 1u);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= num_units) break;
        UnitInfo ui;
        if (!decode_unit(u, lane, tiles, tile_offsets, tpo, ui)) continue;

        int ipx = 0, ipy = 0;
        float Tf = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f;
        uint32_t last = 0;
        if (ui.active) {
            const uint32_t o = ui.slot;
            const uint32_t id = pix[o];
            ipx = (int)(id % (uint32_t)cam.W);
            ipy = (int)(id / (uint32_t)cam.W);
            Tf = out_T[o];
            last = n_contrib[o];
            g0 = dL_dcolor[3 * (size_t)o]; g1 = dL_dcolor[3 * (size_t)o + 1]; g2 = dL_dcolor[3 * (size_t)o + 2];
        }
        const uint32_t wmax = __reduce_max_sync(0xffffffffu, last);
        if (wmax == 0) continue;
        const PixelBox box = warp_pixel_box(ui.active, ipx, ipy);
        const float px = (float)ipx, py = (float)ipy;
        const float bgdot = (cam.bg[0] * g0 + cam.bg[1] * g1 + cam.bg[2] * g2) * Tf;
        float T = Tf, S0 = 0.f, S1 = 0.f, S2 = 0.f;
        sx.pa[lane] = make_float4(px, py, g0, g1);
        sx.pb[lane] = g2;

        // lane l of a batch owns range position hi-1-l: survivors stay in descending position order
        float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
        float r2x = 0.f;
        uint32_t gcur = 0, g_next = 0;
        if ((uint32_t)lane < wmax) {
            gcur = gid_sorted[ui.start + wmax - 1 - lane];
            r0 = splats[3 * (size_t)gcur]; r1 = splats[3 * (size_t)gcur + 1];
            r2x = reinterpret_cast<const float*>(splats)[(size_t)gcur * kSplatWords + 8];
        }
        if ((uint32_t)lane + 32 < wmax) g_next = gid_sorted[ui.start + wmax - 33 - lane];

        uint32_t hi = wmax;  // entries [0, hi) of the range are still to be staged
        int cnt = 0, e = 0;  // survivors staged in sb / next one to replay
        int m = 0;           // Gaussians pending in the transposed tile
        bool done = false;
        while (!done) {
            // ---- phase 1: replay survivors until kSlots Gaussians are pending or the range is exhausted ----
            while (m < kSlots) {
                if (e == cnt) {
                    if (hi == 0) { done = true; break; }
                    __syncwarp();
                    // stage the next 32 range entries: cull against the pixel box, compact the survivors
                    const bool have = (uint32_t)lane < hi;
                    const float thr = blend_threshold(r1.y);
                    const bool pass = have && splat_may_touch(r0.x, r0.y, r0.z, r0.w, r1.x, thr, box);
                    const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
                    cnt = __popc(ballot);
                    e = 0;
                    if (pass) {
                        const int slot = __popc(ballot & lt_mask);
                        sb.a[slot] = make_float4(r0.x, r0.y, -0.5f * r0.z, -r0.w);
                        sb.b[slot] = make_float4(-0.5f * r1.x, thr, r1.y, __uint_as_float(hi - 1 - lane));
                        sb.c[slot] = make_float4(r1.z, r1.w, r2x, __uint_as_float(gcur));
                    }
                    __syncwarp();
                    if ((uint32_t)lane + 32 < hi) {
                        gcur = g_next;
                        r0 = splats[3 * (size_t)gcur]; r1 = splats[3 * (size_t)gcur + 1];
                        r2x = reinterpret_cast<const float*>(splats)[(size_t)gcur * kSplatWords + 8];
                    }
                    if ((uint32_t)lane + 64 < hi) g_next = gid_sorted[ui.start + hi - 65 - lane];
                    hi = hi > 32 ? hi - 32 : 0;
                    continue;
                }
                // replay the next survivors (as many as fit in the transposed tile), branch free
                const int take = min(cnt - e, kSlots - m);
                const float4* sa = sb.a + e;
                float2* vdst = sx.v + m * kTStride + lane;
                float4* mdst = sx.ma + m;
#pragma unroll 2
                for (int i = 0; i < take; ++i) {
                    const float4 a = sa[i];
                    const float4 b = sa[32 + i];
                    const float4 c = sa[64 + i];
                    const float dx = a.x - px, dy = a.y - py;
                    const float power = splat_power(a.z, a.w, b.x, dx, dy);
                    // power is clamped for the exp only: G stays finite on lanes that fail the tests (no inf * 0)
                    const float G = ex2_approx(fminf(power, 0.0f) * kLog2e);
                    const float oG = __fmul_rn(b.z, G);
                    const float alpha = fminf(kAlphaMax, oG);
                    const bool valid = (__float_as_uint(b.w) < last) && (power >= b.y) && (power <= 0.0f) &&
                                       !(alpha < kAlphaMin);
                    const float om = 1.0f - alpha;
                    const float rom = rcp_approx(om);
                    const float Tk = T * rom;  // T_k
                    const float dL_dalpha = ((c.x - S0) * g0 + (c.y - S1) * g1 + (c.z - S2) * g2) * Tk - bgdot * rom;
                    // zero derivative through the active 0.99 clamp; invalid lanes contribute exact zeros
                    const float dpow = (valid && oG < kAlphaMax) ? oG * dL_dalpha : 0.0f;  // dL/dpower
                    const float w = valid ? alpha * Tk : 0.0f;
                    T = valid ? Tk : T;
                    S0 = valid ? fmaf(alpha, c.x, om * S0) : S0;
                    S1 = valid ? fmaf(alpha, c.y, om * S1) : S1;
                    S2 = valid ? fmaf(alpha, c.z, om * S2) : S2;
                    vdst[i * kTStride] = make_float2(dpow, w);
                    if (lane == 0) {  // predicated single-lane stores: one wavefront each
                        mdst[i] = a;
                        mdst[kSlots + i] = make_float4(b.x, b.z, c.w, 0.f);
                    }
                }
                e += take;
                m += take;
            }
            if (m == 0) break;
            __syncwarp();
            // ---- phase 2: lane = (Gaussian slot2, pixel half); nine sums over 16 pixels in registers ----
            {
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
                // moments -> gradients:  dL/dmx = sum dpow (-A dx - B dy),  dL/dA = -1/2 sum dpow dx^2, ...
                // 16-byte vector reductions (red.global.add.v4.f32): 3 per Gaussian instead of 9 scalar ones
                if (slot2 < m) {
                    const float4 gb = sx.mb[slot2];
                    float4* dst = reinterpret_cast<float4*>(dL_dsplats + (size_t)__float_as_uint(gb.z) * kSplatWords);
                    const float dmx = fmaf(2.0f * ga.z, a0, ga.w * a1), dmy = fmaf(2.0f * gb.x, a1, ga.w * a0);
                    const float dop = a5 / gb.y;  // dL/dopacity = sum G dL/dalpha = (sum dpow) / o
                    if (half == 0) {
                        red_add_v4(dst + 0, dmx, dmy, -0.5f * a2, -a3);
                        red_add_v4(dst + 2, a8, 0.f, 0.f, 0.f);
                    } else {
                        red_add_v4(dst + 1, -0.5f * a4, dop, a6, a7);
                    }
                }
            }
            m = 0;
            __syncwarp();
        }
        __syncwarp();
    }
    scheduler_leave(sched, lane);
}

}  // namespace

cudaError_t launch_raster_bwd(const CamK& cam, int N, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, const float* out_T, const uint32_t* n_contrib,
                              const float* dL_dcolor, float* dL_dsplats, uint32_t* sched, int num_sms, cudaStream_t s) {
    cudaError_t e = cudaMemsetAsync(dL_dsplats, 0, (size_t)N * kSplatWords * sizeof(float), s);
    if (e != cudaSuccess) return e;
    if (k <= 0) return cudaSuccess;
    int blocks = num_sms * 3;
    const int need = (k * 8 + kRasterWarps - 1) / kRasterWarps;
    if (blocks > need) blocks = need;
    constexpr size_t smem = kRasterWarps * (sizeof(WarpBatch) + sizeof(WarpXpose));
    static bool opted_in = false;  // attribute of the function, set once per process
    if (!opted_in) {
        e = cudaFuncSetAttribute(raster_bwd_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        opted_in = true;
    }
    raster_bwd_kernel<<<blocks, kRasterThreads, smem, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                        gid_sorted, k, tiles, tpo, pix, out_T, n_contrib, dL_dcolor,
                                                        dL_dsplats, sched);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
