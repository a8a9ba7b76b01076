// tgs_raster_bwd_sparse, raster half: back-to-front replay of Eq. 1 over the sampled
// pixels only, producing dL/d(mean2D, conic, opacity, rgb) per Gaussian.
//
// Same decomposition as the forward (raster_common.cuh): persistent warps, one (tile, 32-pixel
// group) unit at a time, the tile's range walked from the warp's deepest contributor backwards in
// batches of 32 with the per-warp cull.  Per surviving Gaussian each lane forms nine partial sums
// for its pixel -- three colour terms, dL/dopacity and the five moments dpow*(dx, dy, dx^2, dx dy,
// dy^2) from which the mean2D / conic gradients follow linearly -- which are summed across the warp
// with a butterfly (8 values in 9 shuffles + the 9th in 5) into the warp's shared-memory slice;
// after the batch each lane turns ONE Gaussian's sums into its nine gradient components and issues
// the global float atomics: 9 atomic instructions per 32 Gaussians instead of per Gaussian
// (north_star: "warp-shuffle reduction of per-Gaussian gradients before global atomics").
#include "raster_common.cuh"

namespace tgs {

namespace {

struct WarpAcc {
    float v[32][9];  // row stride 9 words: conflict-free when lane e reads row e
};

// keep/send exchange of one butterfly step: lanes with `hi` keep b and send a, the others keep a
__device__ __forceinline__ float bfly(float a, float b, bool hi, int mask) {
    const float send = hi ? a : b;
    const float keep = hi ? b : a;
    return keep + __shfl_xor_sync(0xffffffffu, send, mask);
}

// Sums v[0..8] over the 32 lanes and stores the nine totals to row[0..8].
__device__ __forceinline__ void warp_reduce9_store(const float (&v)[9], float* row, int lane) {
    const bool h16 = lane & 16, h8 = lane & 8, h4 = lane & 4;
    const float a0 = bfly(v[0], v[4], h16, 16), a1 = bfly(v[1], v[5], h16, 16);
    const float a2 = bfly(v[2], v[6], h16, 16), a3 = bfly(v[3], v[7], h16, 16);
    const float b0 = bfly(a0, a2, h8, 8), b1 = bfly(a1, a3, h8, 8);
    float c0 = bfly(b0, b1, h4, 4);
    c0 += __shfl_xor_sync(0xffffffffu, c0, 2);
    c0 += __shfl_xor_sync(0xffffffffu, c0, 1);
    float e = v[8];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
    // lane L (L % 4 == 0) holds quantity 4*bit4 + 2*bit3 + bit2 = L >> 2
    if ((lane & 3) == 0) row[lane >> 2] = c0;
    if (lane == 1) row[8] = e;
}

__global__ void __launch_bounds__(kRasterThreads, 4)
raster_bwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  const float* __restrict__ out_T, const uint32_t* __restrict__ n_contrib,
                  const float* __restrict__ dL_dcolor, float* __restrict__ dL_dsplats, uint32_t* __restrict__ sched) {
    __shared__ WarpBatch s_batch[kRasterWarps];
    __shared__ WarpAcc s_acc[kRasterWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    WarpBatch& sb = s_batch[warp];
    WarpAcc& sa = s_acc[warp];
    const uint32_t num_units = (uint32_t)k * 8u;
    const uint32_t lt_mask = (1u << lane) - 1u;

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
        for (uint32_t hi = wmax; hi > 0; hi = hi > 32 ? hi - 32 : 0) {
            const bool have = (uint32_t)lane < hi;
            const float thr = blend_threshold(r1.y);
            const bool pass = have && splat_may_touch(r0.x, r0.y, r0.z, r0.w, r1.x, thr, box);
            const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
            const int cnt = __popc(ballot);
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

            uint32_t touched = 0;
#pragma unroll 2
            for (int e = 0; e < cnt; ++e) {
                const float4 a = sb.a[e];
                const float4 b = sb.b[e];
                const float4 c = sb.c[e];
                const float dx = a.x - px, dy = a.y - py;
                const float power = splat_power(a.z, a.w, b.x, dx, dy);
                // power is clamped for the exp only: G stays finite on lanes that fail the tests (no inf * 0)
                const float G = ex2_approx(fminf(power, 0.0f) * kLog2e);
                const float oG = __fmul_rn(b.z, G);
                const float alpha = fminf(kAlphaMax, oG);
                const bool valid = (__float_as_uint(b.w) < last) && (power >= b.y) && (power <= 0.0f) &&
                                   !(alpha < kAlphaMin);
                if (!__any_sync(0xffffffffu, valid)) continue;
                touched |= 1u << e;
                float v[9];
                {
                    const float om = 1.0f - alpha;
                    const float rom = rcp_approx(om);
                    const float Tk = T * rom;  // T_k
                    const float w = valid ? alpha * Tk : 0.0f;
                    v[6] = w * g0; v[7] = w * g1; v[8] = w * g2;
                    float dL_dalpha = ((c.x - S0) * g0 + (c.y - S1) * g1 + (c.z - S2) * g2) * Tk - bgdot * rom;
                    dL_dalpha = valid ? dL_dalpha : 0.0f;
                    if (valid) {
                        T = Tk;
                        S0 = fmaf(alpha, c.x, om * S0); S1 = fmaf(alpha, c.y, om * S1); S2 = fmaf(alpha, c.z, om * S2);
                    }
                    // zero derivative through the active 0.99 clamp
                    const float dLa = (oG < kAlphaMax) ? dL_dalpha : 0.0f;
                    v[5] = G * dLa;               // dL/dopacity
                    const float dpow = oG * dLa;  // dL/dpower
                    v[0] = dpow * dx; v[1] = dpow * dy;
                    v[2] = v[0] * dx; v[3] = v[0] * dy; v[4] = v[1] * dy;
                }
                warp_reduce9_store(v, sa.v[e], lane);
            }
            __syncwarp();
            // flush: lane e owns staged entry e; moments -> gradients
            //   dL/dmx = sum dpow (-A dx - B dy),  dL/dA = -1/2 sum dpow dx^2,  dL/dB = -sum dpow dx dy, ...
            if (lane < cnt && (touched >> lane) & 1u) {
                const float4 a = sb.a[lane];
                const float nC = sb.b[lane].x;
                const float* m = sa.v[lane];
                float* dst = dL_dsplats + (size_t)__float_as_uint(sb.c[lane].w) * kSplatWords;
                atomicAdd(dst + 0, fmaf(2.0f * a.z, m[0], a.w * m[1]));
                atomicAdd(dst + 1, fmaf(2.0f * nC, m[1], a.w * m[0]));
                atomicAdd(dst + 2, -0.5f * m[2]);
                atomicAdd(dst + 3, -m[3]);
                atomicAdd(dst + 4, -0.5f * m[4]);
                atomicAdd(dst + 5, m[5]);
                atomicAdd(dst + 6, m[6]);
                atomicAdd(dst + 7, m[7]);
                atomicAdd(dst + 8, m[8]);
            }
            __syncwarp();
        }
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
    int blocks = num_sms * 4;
    const int need = (k * 8 + kRasterWarps - 1) / kRasterWarps;
    if (blocks > need) blocks = need;
    raster_bwd_kernel<<<blocks, kRasterThreads, 0, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                        gid_sorted, k, tiles, tpo, pix, out_T, n_contrib, dL_dcolor,
                                                        dL_dsplats, sched);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
