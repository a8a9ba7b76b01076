// tgs_raster_bwd_sparse, raster half: back-to-front replay of Eq. 1 over the sampled
// pixels only, producing dL/d(mean2D, conic, opacity, rgb) per Gaussian.
//
// Same decomposition as the forward (raster_common.cuh): persistent block per sampled tile, a
// producer warp stages the tile's records from its deepest contributor backwards through the
// shared-memory ring, eight consumer warps (32 sampled pixels each) cull per warp and replay.
// The gradient of one Gaussian is a sum over pixels; summing it with a shuffle tree per Gaussian
// costs more issue slots and LSU traffic than the math itself (profiles/r1b), so the warp
// TRANSPOSES instead:
//   phase 1 (lane = pixel): per surviving Gaussian every lane replays its pixel and stores only the
//            two per-(pixel, Gaussian) scalars everything else is linear in -- dpow = dL/dpower and
//            w = alpha * T_k -- into a [16 Gaussians][32 pixels] shared-memory tile;
//   phase 2 (lane = Gaussian): when 16 Gaussians are pending, lane e (and lane e + 16 for the other
//            half of the pixels) sums Gaussian e's nine gradient components over the pixels in
//            registers -- plain FMAs, no shuffles -- and issues three 16-byte vector reductions
//            (red.global.add.v4.f32) into the Gaussian's gradient record.
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
    float4 org;                   // x, y of lane 0's pixel; z != 0: the unit is an 8x4 block of a row-major full tile (separable phase 2)
};

constexpr int kBwdStageEntries = 128;
using BwdRing = Ring<kBwdStageEntries, false, 4>;

struct BwdShared {
    BwdRing ring;
    WarpList<kBwdStageEntries> list[kConsumers];
    WarpXpose xpose[kConsumers];
};

__global__ void __launch_bounds__(kRasterThreads, 3)
raster_bwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  const float* __restrict__ out_T, const uint32_t* __restrict__ n_contrib,
                  const float* __restrict__ dL_dcolor, float* __restrict__ dL_dsplats, uint32_t* __restrict__ sched) {
    extern __shared__ __align__(16) unsigned char smem_raw[];  // > 48 KB: dynamic, opted in by the launcher
    BwdShared& sm = *reinterpret_cast<BwdShared*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ring_init(sm.ring);
    if (warp == kConsumers) {
        producer_loop<true>(sm.ring, splats, tile_offsets, gid_sorted, (uint32_t)k, tiles, tpo, n_contrib, sched, lane, kLitePixels,
                            pix, (uint32_t)cam.W);
        return;
    }
    BwdRing& R = sm.ring;
    uint32_t* const idx = sm.list[warp].idx;
    WarpXpose& sx = sm.xpose[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int slot2 = lane & (kSlots - 1), half = lane >> 4;  // phase-2 role of this lane

    // per-tile state of this consumer's 32 pixels
    float px = 0.f, py = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f, bgdot = 0.f;
    float T = 0.f, Sg = 0.f;
    uint32_t last = 0, wmax = 0;
    int m = 0;  // Gaussians pending in the transposed tile
    uint32_t gchunk = 0;

    // ---- phase 2: lane = (Gaussian slot2, pixel half); nine sums over 16 pixels in registers ----
    auto flush = [&]() {
        __syncwarp();
        const float4 ga = sx.ma[slot2];
        float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f, a4 = 0.f, a5 = 0.f, a6 = 0.f, a7 = 0.f, a8 = 0.f;
        const float2* vrow = sx.v + slot2 * kTStride + half * 16;
        const float4* prow = sx.pa + half * 16;
        const float* qrow = sx.pb + half * 16;
        const float4 org = sx.org;
        if (org.z != 0.f) {
            // full 8x4 block: pixel i of this half sits at (org.x + (i & 7), org.y + 2 half + (i >> 3)), so the moments
            // separate -- per row  s0 = sum d, s1 = sum d dx, s2 = sum d dx^2  (4 operations per pixel instead of 9),
            // then  a1 += s0 dy, a3 += s1 dy, a4 += s0 dy^2  once per row
            const float gxo = ga.x - org.x;
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                const float dy = ga.y - (org.y + (float)(2 * half + r));
                float s0 = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int i = 8 * r + u;
                    const float2 v = vrow[i];
                    const float2 gq = *reinterpret_cast<const float2*>(&prow[i].z);
                    const float h2 = qrow[i];
                    const float dx = gxo - (float)u;
                    const float t0 = v.x * dx;
                    s0 += v.x; s1 += t0; s2 = fmaf(t0, dx, s2);
                    a6 = fmaf(v.y, gq.x, a6); a7 = fmaf(v.y, gq.y, a7); a8 = fmaf(v.y, h2, a8);
                }
                const float s0y = s0 * dy;
                a0 += s1; a1 += s0y; a2 += s2; a3 = fmaf(s1, dy, a3); a4 = fmaf(s0y, dy, a4); a5 += s0;
            }
        } else {
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
        }
        a0 += __shfl_xor_sync(0xffffffffu, a0, 16); a1 += __shfl_xor_sync(0xffffffffu, a1, 16);
        a2 += __shfl_xor_sync(0xffffffffu, a2, 16); a3 += __shfl_xor_sync(0xffffffffu, a3, 16);
        a4 += __shfl_xor_sync(0xffffffffu, a4, 16); a5 += __shfl_xor_sync(0xffffffffu, a5, 16);
        a6 += __shfl_xor_sync(0xffffffffu, a6, 16); a7 += __shfl_xor_sync(0xffffffffu, a7, 16);
        a8 += __shfl_xor_sync(0xffffffffu, a8, 16);
        // moments -> gradients:  dL/dmx = sum dpow (-A dx - B dy),  dL/dA = -1/2 sum dpow dx^2, ...
        const float4 gb = sx.mb[slot2];
        if (slot2 < m && __float_as_uint(gb.z) != 0xffffffffu) {  // (a padding slot holds the stage's dummy record)
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
        m = 0;
        __syncwarp();
    };

    for (;;) {
        const uint32_t s = gchunk % BwdRing::kStages;
        mbar_wait(&R.full[s], (gchunk / BwdRing::kStages) & 1u);
        const StageInfo inf = R.info[s];
        if (inf.hdr != kHdrCont) {
            if (m > 0) flush();  // tail of the previous tile
            if (inf.hdr == kHdrEnd) break;
            UnitInfo ui;
            wmax = 0;
            if (decode_unit(inf.hdr, (uint32_t)warp, lane, tiles, tile_offsets, tpo, ui)) {
                int ipx = 0, ipy = 0;
                float Tf = 0.f;
                g0 = 0.f; g1 = 0.f; g2 = 0.f; last = 0;
                if (ui.active) {
                    const uint32_t o = ui.slot;
                    const uint32_t id = pix[o];
                    ipx = (int)(id % (uint32_t)cam.W);
                    ipy = (int)(id / (uint32_t)cam.W);
                    Tf = out_T[o];
                    last = n_contrib[o];
                    g0 = dL_dcolor[3 * (size_t)o]; g1 = dL_dcolor[3 * (size_t)o + 1]; g2 = dL_dcolor[3 * (size_t)o + 2];
                }
                wmax = __reduce_max_sync(0xffffffffu, last);
                px = (float)ipx; py = (float)ipy;
                bgdot = (cam.bg[0] * g0 + cam.bg[1] * g1 + cam.bg[2] * g2) * Tf;
                T = Tf; Sg = 0.f;
                sx.pa[lane] = make_float4(px, py, g0, g1);
                sx.pb[lane] = g2;
                if (lane == 0) sx.org = make_float4(px, py, inf.rowmajor ? 1.f : 0.f, 0.f);  // 256 pixels, verified row-major
            }
        }
        if (wmax > 0) {
            const Stage<kBwdStageEntries>& st = R.st[s];
            // the box of THIS stage: only the pixels whose deepest contributor lies in or in front of it (a record at
            // position p can only contribute to pixels with n_contrib > p); it grows to the warp's full box towards the front
            const uint32_t lowpos = inf.base - (inf.cnt - 1u);  // the front-most position staged here
            const PixelBox box = warp_pixel_box(last > lowpos, (int)px, (int)py);
            // ---- cull the stage against that box; survivors' indices in range order (descending position) ----
            uint32_t n = 0;
            for (uint32_t b0 = 0; b0 < inf.cnt; b0 += 32) {
                // records of this batch sit at range positions base-b0 .. base-b0-31 (descending)
                if (inf.base - b0 >= wmax + 31u && inf.base >= b0 + 31u) continue;  // all beyond this warp's deepest contributor
                const uint32_t i = b0 + lane;
                const float4 q0 = st.p0[i];
                const float2 c2 = st.ct[i];
                const bool pass = i < inf.cnt && splat_may_touch(q0.x, q0.y, q0.z, q0.w, c2.x, c2.y, box);
                const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
                if (pass) idx[n + __popc(ballot & lt_mask)] = i;
                n += __popc(ballot);
            }
            // pad the list to a multiple of four with the stage's dummy record: groups stay aligned and m stays a
            // multiple of four, so a group never straddles a flush
            if (lane < 3) idx[n + lane] = (uint32_t)kBwdStageEntries;
            n = (n + 3u) & ~3u;
            __syncwarp();
            for (uint32_t e = 0; e < n; e += 4) {
                // ---- phase 1: replay four survivors in place, branch free ----
                const uint4 j4 = *reinterpret_cast<const uint4*>(idx + e);
                float2* vdst = sx.v + m * kTStride + lane;
#pragma unroll
                for (int ii = 0; ii < 4; ++ii) {
                    const uint32_t i = ii == 0 ? j4.x : (ii == 1 ? j4.y : (ii == 2 ? j4.z : j4.w));
                    const float4 a = st.p0[i];
                    const float4 b = st.p1[i];  // -C/2, opacity, red, green
                    const float blue = st.bl[i];
                    const float dx = a.x - px, dy = a.y - py;
                    const float power = splat_power(a.z, a.w, b.x, dx, dy);
                    const float G = ex2_approx(power * kLog2e);
                    const float oG = __fmul_rn(b.y, G);
                    const float alpha = fminf(kAlphaMax, oG);
                    // (power >= thr is implied by the alpha test; thr only serves the cull); every use of a quantity
                    // of an invalid lane below is a select, never a product: G may be inf there
                    const bool valid = (inf.base - i < last) && (power <= 0.0f) && !(alpha < kAlphaMin);
                    const float om = 1.0f - alpha;
                    const float rom = rcp_approx(om);
                    const float Tk = T * rom;  // T_k
                    // only the projection of the colour behind onto dL/dcolor is needed: one scalar
                    // recurrence Sg = S . g instead of three
                    const float cg = fmaf(blue, g2, fmaf(b.w, g1, b.z * g0));
                    const float dL_dalpha = fmaf(cg - Sg, Tk, -bgdot * rom);
                    // zero derivative through the active 0.99 clamp; invalid lanes contribute exact zeros
                    const float dpow = (valid && oG < kAlphaMax) ? oG * dL_dalpha : 0.0f;  // dL/dpower
                    const float w = valid ? alpha * Tk : 0.0f;
                    T = valid ? Tk : T;
                    Sg = valid ? fmaf(alpha, cg, om * Sg) : Sg;
                    vdst[ii * kTStride] = make_float2(dpow, w);
                }
                if (lane < 4) {  // the Gaussians' parameters for phase 2: one parallel copy per group
                    const uint32_t i = idx[e + lane];
                    const float4 b = st.p1[i];
                    sx.ma[m + lane] = st.p0[i];
                    sx.mb[m + lane] = make_float4(b.x, b.y, __uint_as_float(st.id[i]), 0.f);
                }
                m += 4;
                if (m == kSlots) flush();
            }
            __syncwarp();  // the list is rewritten at the next stage
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&R.empty[s]);
        ++gchunk;
    }
}

}  // namespace

cudaError_t launch_raster_bwd(const CamK& cam, int N, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, const float* out_T, const uint32_t* n_contrib,
                              const float* dL_dcolor, float* dL_dsplats, uint32_t* sched, int num_sms, cudaStream_t s,
                              const SideStream* side) {
    cudaError_t e = cudaMemsetAsync(dL_dsplats, 0, (size_t)N * kSplatWords * sizeof(float), s);
    if (e != cudaSuccess) return e;
    if (k <= 0) return cudaSuccess;
    // fork (after the memset): the warp-per-tile kernel for tiles with <= kLitePixels sampled pixels runs on the
    // side stream, concurrently with the block-per-tile kernel; both accumulate with atomics
    e = cudaEventRecord(side->fork, s);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(side->aux, side->fork, 0);
    if (e == cudaSuccess)
        e = launch_raster_bwd_lite(cam, splats, tile_offsets, gid_sorted, k, tiles, tpo, pix, out_T, n_contrib, dL_dcolor,
                                   dL_dsplats, sched + 2, num_sms, side->aux);
    if (e == cudaSuccess) e = cudaEventRecord(side->join, side->aux);
    if (e != cudaSuccess) return e;
    int blocks = num_sms * 3;
    if (blocks > k) blocks = k;
    constexpr size_t smem = sizeof(BwdShared);
    static SmemOptIn opt;  // per device
    e = opt.ensure((const void*)raster_bwd_kernel, smem);
    if (e != cudaSuccess) return e;
    raster_bwd_kernel<<<blocks, kRasterThreads, smem, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                          gid_sorted, k, tiles, tpo, pix, out_T, n_contrib, dL_dcolor,
                                                          dL_dsplats, sched);
    count_launches(1);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return cudaStreamWaitEvent(s, side->join, 0);  // join
}

}  // namespace tgs
