// tgs_raster_fwd_sparse: front-to-back alpha compositing (Eq. 1) for the SAMPLED
// pixels only (Fig. 6: sampled pixels listed tile by tile, tile-wise pixel
// offsets by prefix sum, tile-parallel execution).
//
// B200 design (raster_common.cuh): persistent warps pull (tile, 32-pixel group) units from an
// atomic counter; each warp stages its tile's depth-ordered Gaussians 32 at a time (one float4
// record load per lane, prefetched into registers while the current batch is consumed), culls them
// against the bounding box of its own 32 pixels and walks only the survivors with a branch-free,
// unrolled inner loop (per survivor: three shared loads, ~25 FP32/ALU ops, one MUFU.EX2).
//
// power uses the one fixed fused sequence of DESIGN.md "canonical arithmetic", so `power > 0` is
// decided on the same bits as the oracle; alpha itself is o * ex2.approx(power * log2 e).
#include "raster_common.cuh"

namespace tgs {

namespace {

template <bool COUNT>
__global__ void __launch_bounds__(kRasterThreads, 5)
raster_fwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  float* __restrict__ out_color, float* __restrict__ out_T, uint32_t* __restrict__ n_contrib,
                  uint32_t* __restrict__ n_walked, uint32_t* __restrict__ n_blended, uint32_t* __restrict__ sched) {
    __shared__ WarpBatch s_batch[kRasterWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpBatch& sb = s_batch[warp];
    const uint32_t num_units = (uint32_t)k * 8u;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const float kNaN = __int_as_float(0x7fc00000);

    for (;;) {
        uint32_t u = 0;
        if (lane == 0) u = atomicAdd(&sched[0], 1u);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= num_units) break;
        UnitInfo ui;
        if (!decode_unit(u, lane, tiles, tile_offsets, tpo, ui)) continue;

        int ipx = 0, ipy = 0;
        if (ui.active) {
            const uint32_t id = pix[ui.slot];
            ipx = (int)(id % (uint32_t)cam.W);
            ipy = (int)(id / (uint32_t)cam.W);
        }
        const PixelBox box = warp_pixel_box(ui.active, ipx, ipy);
        // a finished (or inactive) lane carries px = NaN: power becomes NaN and every test fails
        float px = ui.active ? (float)ipx : kNaN;
        const float py = (float)ipy;

        float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
        uint32_t last = 0, walked = ui.end - ui.start, blended = 0;

        // software pipeline: ids two batches ahead, records one batch ahead
        float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
        float r2x = 0.f;
        uint32_t g_next = 0;
        {
            const uint32_t j = ui.start + lane;
            if (j < ui.end) {
                const uint32_t g = gid_sorted[j];
                r0 = splats[3 * (size_t)g]; r1 = splats[3 * (size_t)g + 1];
                r2x = reinterpret_cast<const float*>(splats)[(size_t)g * kSplatWords + 8];
            }
            if (j + 32 < ui.end) g_next = gid_sorted[j + 32];
        }
        for (uint32_t base = ui.start; base < ui.end; base += 32) {
            // ---- stage: cull against the pixel box, compact survivors in range order ----
            const bool have = base + lane < ui.end;
            const float thr = blend_threshold(r1.y);
            const bool pass = have && splat_may_touch(r0.x, r0.y, r0.z, r0.w, r1.x, thr, box);
            const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
            const int cnt = __popc(ballot);
            if (pass) {
                const int slot = __popc(ballot & lt_mask);
                sb.a[slot] = make_float4(r0.x, r0.y, -0.5f * r0.z, -r0.w);
                sb.b[slot] = make_float4(-0.5f * r1.x, thr, r1.y, __uint_as_float((base - ui.start) + lane + 1));
                sb.c[slot] = make_float4(r1.z, r1.w, r2x, 0.f);
            }
            __syncwarp();
            // ---- prefetch ----
            {
                const uint32_t j = base + 32 + lane;
                if (j < ui.end) {
                    r0 = splats[3 * (size_t)g_next]; r1 = splats[3 * (size_t)g_next + 1];
                    r2x = reinterpret_cast<const float*>(splats)[(size_t)g_next * kSplatWords + 8];
                }
                if (j + 32 < ui.end) g_next = gid_sorted[j + 32];
            }
            // ---- walk the survivors (branch free) ----
#pragma unroll 4
            for (int e = 0; e < cnt; ++e) {
                const float4 a = sb.a[e];
                const float4 b = sb.b[e];
                const float4 c = sb.c[e];
                const float dx = a.x - px, dy = a.y - py;
                const float power = splat_power(a.z, a.w, b.x, dx, dy);
                const float alpha = fminf(kAlphaMax, __fmul_rn(b.z, ex2_approx(power * kLog2e)));
                const bool blend = (power >= b.y) && (power <= 0.0f) && !(alpha < kAlphaMin);
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
                px = term ? kNaN : px;
            }
            if (__all_sync(0xffffffffu, px != px)) break;
            __syncwarp();  // the batch slice is rewritten next iteration
        }
        if (ui.active) {
            const uint32_t o = ui.slot;
            out_color[3 * (size_t)o] = fmaf(T, cam.bg[0], C0);
            out_color[3 * (size_t)o + 1] = fmaf(T, cam.bg[1], C1);
            out_color[3 * (size_t)o + 2] = fmaf(T, cam.bg[2], C2);
            out_T[o] = T;
            n_contrib[o] = last;
            if (COUNT) {
                if (n_walked) n_walked[o] = walked;
                if (n_blended) n_blended[o] = blended;
            }
        }
        __syncwarp();
    }
    scheduler_leave(sched, lane);
}

}  // namespace

cudaError_t launch_raster_fwd(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, float* out_color, float* out_T, uint32_t* n_contrib,
                              uint32_t* n_walked, uint32_t* n_blended, uint32_t* sched, int num_sms, cudaStream_t s) {
    if (k <= 0) return cudaSuccess;
    const bool count = n_walked || n_blended;
    // persistent grid: never more warps than units
    int blocks = num_sms * 5;
    const int need = (k * 8 + kRasterWarps - 1) / kRasterWarps;
    if (blocks > need) blocks = need;
    const float4* sp = reinterpret_cast<const float4*>(splats);
    if (count)
        raster_fwd_kernel<true><<<blocks, kRasterThreads, 0, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                  out_color, out_T, n_contrib, n_walked, n_blended, sched);
    else
        raster_fwd_kernel<false><<<blocks, kRasterThreads, 0, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                   out_color, out_T, n_contrib, n_walked, n_blended, sched);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
