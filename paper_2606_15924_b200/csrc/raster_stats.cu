// tgs_raster_stats_sparse: statistics forward (Sec. 3.8 Eq. 12,
// Alg. 1 step 11 "rasterize_forward_pixels"): the forward walk of Eq. 1 over the sampled pixels, but
// instead of colours every composited (pixel, Gaussian) pair with weight w = T alpha is projected back
// onto its Gaussian:   E_i += e(p) w,   D_i += (d^T Sigma'^-1 d) w,   W_i += w,
// plus the expected depth sum_i w z_i of every sampled pixel.
//
// Same decomposition as the raster kernels (raster_common.cuh): persistent block per sampled tile, a
// producer warp stages the tile's records front to back through the mbarrier ring and stops once all
// eight consumers are saturated; each consumer culls against the box of its 32 pixels and walks the
// survivors.  The per-Gaussian sums use the backward's transpose: phase 1 (lane = pixel) stores only
// w into a [16 Gaussians][32 pixels] shared tile, phase 2 (lane = Gaussian) sums E, D, W over the
// pixels in registers (D is recomputed from the Gaussian and the pixel) and issues ONE 16-byte vector
// reduction per (warp, Gaussian).
#include "raster_common.cuh"

namespace tgs {

namespace {

__device__ __forceinline__ void red_add_v4(float4* p, float x, float y, float z, float w) {
    asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(p), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

constexpr int kSlots = 16;    // Gaussians per transposed tile
constexpr int kVStride = 33;  // row stride of the w tile: conflict-free for both phases

struct StatXpose {
    float v[kSlots * kVStride];  // [slot][pixel] = w
    float4 ma[kSlots];           // mx, my, -A/2, -B
    float2 mb[kSlots];           // -C/2, bits: Gaussian id
    float4 pa[32];               // per pixel: px, py, e(p), unused
};

constexpr int kStatStageEntries = 128;
using StatRing = Ring<kStatStageEntries, true>;  // with the depth plane

struct StatShared {
    StatRing ring;
    WarpBatch batch[kConsumers];
    StatXpose xpose[kConsumers];
};

__global__ void __launch_bounds__(kRasterThreads, 3)
raster_stats_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                    const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                    const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                    const float* __restrict__ pix_err, float* __restrict__ stats, float* __restrict__ out_depth,
                    uint32_t* __restrict__ sched) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    StatShared& sm = *reinterpret_cast<StatShared*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ring_init(sm.ring);
    if (warp == kConsumers) {
        producer_loop<false>(sm.ring, splats, tile_offsets, gid_sorted, (uint32_t)k, tiles, tpo, nullptr, sched, lane, kLitePixels);
        return;
    }
    StatRing& R = sm.ring;
    WarpBatch& sb = sm.batch[warp];
    StatXpose& sx = sm.xpose[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    const int slot2 = lane & (kSlots - 1), half = lane >> 4;  // phase-2 role of this lane

    UnitInfo ui;
    ui.start = ui.end = ui.slot = 0; ui.active = false;
    PixelBox box = {0.f, 0.f, 0.f, 0.f};
    const float kNaN = __int_as_float(0x7fc00000);
    // (a finished or inactive lane carries px = NaN here: the alive flag of the forward kernel costs this kernel a
    // register it does not have at 3 blocks / SM -- 90 bytes of spills in the inner loop, 0.87 instead of 0.74 ms)
    float px = kNaN, py = 0.f, T = 1.0f, zacc = 0.f;
    bool open = false;
    int m = 0;  // Gaussians pending in the transposed tile
    uint32_t gchunk = 0, seq = 0;

    // ---- phase 2: lane = (Gaussian slot2, pixel half); three sums over 16 pixels in registers ----
    auto flush = [&]() {
        __syncwarp();
        const float4 ga = sx.ma[slot2];
        const float2 gb = sx.mb[slot2];
        float E = 0.f, D = 0.f, Wt = 0.f;
        const float* vrow = sx.v + slot2 * kVStride + half * 16;
        const float4* prow = sx.pa + half * 16;
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float w = vrow[i];
            const float4 q = prow[i];
            const float dx = ga.x - q.x, dy = ga.y - q.y;
            const float pw = splat_power(ga.z, ga.w, gb.x, dx, dy);
            Wt += w;
            E = fmaf(w, q.z, E);
            D = fmaf(w, -2.0f * pw, D);
        }
        E += __shfl_xor_sync(0xffffffffu, E, 16);
        D += __shfl_xor_sync(0xffffffffu, D, 16);
        Wt += __shfl_xor_sync(0xffffffffu, Wt, 16);
        if (slot2 < m && half == 0)
            red_add_v4(reinterpret_cast<float4*>(stats) + __float_as_uint(gb.y), E, D, Wt, 0.f);
        m = 0;
        __syncwarp();
    };
    auto finalize = [&]() {
        if (m > 0) flush();
        if (ui.active && out_depth) out_depth[ui.slot] = zacc;
        open = false;
        if (lane == 0) *(volatile uint32_t*)&R.done_seq[warp] = seq;
    };

    for (;;) {
        const uint32_t s = gchunk % StatRing::kStages;
        mbar_wait(&R.full[s], (gchunk / StatRing::kStages) & 1u);
        const StageInfo inf = R.info[s];
        if (inf.hdr != kHdrCont) {
            if (open) finalize();
            if (inf.hdr == kHdrEnd) break;
            ++seq;
            open = decode_unit(inf.hdr, (uint32_t)warp, lane, tiles, tile_offsets, tpo, ui);
            if (!open) {
                if (lane == 0) *(volatile uint32_t*)&R.done_seq[warp] = seq;
            } else {
                int ipx = 0, ipy = 0;
                float e = 0.f;
                if (ui.active) {
                    const uint32_t id = pix[ui.slot];
                    ipx = (int)(id % (uint32_t)cam.W);
                    ipy = (int)(id / (uint32_t)cam.W);
                    e = pix_err[ui.slot];
                }
                box = warp_pixel_box(ui.active, ipx, ipy);
                px = ui.active ? (float)ipx : kNaN;  // NaN: power becomes NaN and every test fails
                py = (float)ipy;
                T = 1.0f; zacc = 0.f;
                sx.pa[lane] = make_float4((float)ipx, (float)ipy, e, 0.f);
            }
        }
        if (open) {
            // (survivors are copied into the warp's private batch, from three float4 planes, as in round 1: the
            // in-place index list of the forward / backward kernels measured 0.83 instead of 0.74 ms in this kernel)
            const Stage<kStatStageEntries, true>& st = R.st[s];
            for (uint32_t b0 = 0; b0 < inf.cnt; b0 += 32) {
                // ---- cull this batch against the pixel box, compact survivors in range order ----
                const uint32_t i = b0 + lane;
                const bool have = i < inf.cnt;
                const float4 q0 = st.p0[i];
                const float4 q1 = st.p1[i];
                const bool pass = have && splat_may_touch(q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, box);
                const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
                const int cnt = __popc(ballot);
                __syncwarp();
                if (pass) {
                    const int slot = __popc(ballot & lt_mask);
                    const float4 q2 = st.p2[i];
                    sb.a[slot] = q0;
                    sb.b[slot] = make_float4(q1.x, q1.y, q1.z, 0.f);  // -C/2, thr, opacity
                    sb.c[slot] = make_float4(q2.w, q2.z, 0.f, 0.f);    // depth, bits: Gaussian id
                }
                __syncwarp();
                int e = 0;
                while (e < cnt) {
                    // ---- phase 1: walk the next survivors (as many as fit in the transposed tile), branch free ----
                    const int take = min(cnt - e, kSlots - m);
                    const float4* sa = sb.a + e;
                    float* vdst = sx.v + m * kVStride + lane;
#pragma unroll 2
                    for (int ii = 0; ii < take; ++ii) {
                        const float4 a = sa[ii];
                        const float4 b = sa[32 + ii];
                        const float dx = a.x - px, dy = a.y - py;
                        const float power = splat_power(a.z, a.w, b.x, dx, dy);
                        const float alpha = fminf(kAlphaMax, __fmul_rn(b.z, ex2_approx(power * kLog2e)));
                        const bool blend = (power <= 0.0f) && !(alpha < kAlphaMin);
                        const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                        const bool term = blend && (Tn < kTMin);
                        const bool upd = blend && !term;
                        const float w = upd ? alpha * T : 0.0f;
                        zacc = fmaf(w, sa[64 + ii].x, zacc);
                        T = upd ? Tn : T;
                        px = term ? kNaN : px;
                        vdst[ii * kVStride] = w;
                    }
                    if (lane < take) {  // the Gaussians' parameters for phase 2: one parallel copy per group
                        sx.ma[m + lane] = sa[lane];
                        sx.mb[m + lane] = make_float2(sa[32 + lane].x, sa[64 + lane].y);
                    }
                    e += take;
                    m += take;
                    if (m == kSlots) flush();
                }
                if (__all_sync(0xffffffffu, px != px)) {
                    finalize();
                    break;
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&R.empty[s]);
        ++gchunk;
    }
}

}  // namespace

cudaError_t launch_raster_stats(const CamK& cam, int N, const float* splats, const uint32_t* tile_offsets,
                                const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                const uint32_t* pix, const float* pix_err, float* stats, float* out_depth,
                                uint32_t* sched, int num_sms, cudaStream_t s, const SideStream* side) {
    cudaError_t e = cudaMemsetAsync(stats, 0, (size_t)N * 4 * sizeof(float), s);
    if (e != cudaSuccess) return e;
    if (k <= 0) return cudaSuccess;
    // fork (after the memset): tiles with <= kLitePixels sampled pixels go to the warp-per-tile kernel on the side stream
    e = cudaEventRecord(side->fork, s);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(side->aux, side->fork, 0);
    if (e == cudaSuccess)
        e = launch_raster_stats_lite(cam, splats, tile_offsets, gid_sorted, k, tiles, tpo, pix, pix_err, stats, out_depth,
                                     sched + 2, num_sms, side->aux);
    if (e == cudaSuccess) e = cudaEventRecord(side->join, side->aux);
    if (e != cudaSuccess) return e;
    int blocks = num_sms * 3;
    if (blocks > k) blocks = k;
    constexpr size_t smem = sizeof(StatShared);
    static SmemOptIn opt;  // per device
    e = opt.ensure((const void*)raster_stats_kernel, smem);
    if (e != cudaSuccess) return e;
    raster_stats_kernel<<<blocks, kRasterThreads, smem, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                            gid_sorted, k, tiles, tpo, pix, pix_err, stats, out_depth, sched);
    count_launches(1);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return cudaStreamWaitEvent(s, side->join, 0);  // join
}

}  // namespace tgs
