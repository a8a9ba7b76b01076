// tgs_raster_fwd_sparse: front-to-back alpha compositing (Eq. 1) for the SAMPLED
// pixels only (Fig. 6: sampled pixels listed tile by tile, tile-wise pixel
// offsets by prefix sum, tile-parallel execution).
//
// B200 design (raster_common.cuh): one persistent block per sampled tile at a time; a producer warp
// gathers the tile's depth-ordered splat records once into a shared-memory stage ring (mbarrier
// full/empty), eight consumer warps each own 32 of the tile's sampled pixels, cull every staged
// stage against the bounding box of their own pixels, keep the INDICES of the survivors in a private
// list and walk only those with a branch-free inner loop that reads the records in place from the
// stage (per survivor: a quarter of a 16-byte index load, LDS.128 + LDS.128 + LDS.32 = 5 shared-memory
// wavefronts, ~25 FP32/ALU ops, one MUFU.EX2).  profiles/r2b: the kernel is bound by shared-memory
// wavefronts; copying the survivors into a private slice (three STS.128 + three LDS.128 of 2 wavefronts
// each per survivor) cost 57 wavefronts per 32 staged records against 37 now.
//
// power uses the one fixed fused sequence of DESIGN.md "canonical arithmetic", so `power > 0` is
// decided on the same bits as the oracle; alpha itself is o * ex2.approx(power * log2 e).
#include "raster_common.cuh"

namespace tgs {

namespace {

constexpr int kFwdStageEntries = 128;
using FwdRing = Ring<kFwdStageEntries, false, 4>;

struct FwdShared {
    FwdRing ring;
    WarpList<kFwdStageEntries> list[kConsumers];
};

template <bool COUNT>
__global__ void __launch_bounds__(kRasterThreads, 4)
raster_fwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  float* __restrict__ out_color, float* __restrict__ out_T, uint32_t* __restrict__ n_contrib,
                  uint32_t* __restrict__ n_walked, uint32_t* __restrict__ n_blended, uint32_t* __restrict__ sched) {
    extern __shared__ __align__(16) unsigned char smem_raw[];  // > 48 KB: dynamic, opted in by the launcher
    FwdShared& sm = *reinterpret_cast<FwdShared*>(smem_raw);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ring_init(sm.ring);
    if (warp == kConsumers) {
        producer_loop<false>(sm.ring, splats, tile_offsets, gid_sorted, (uint32_t)k, tiles, tpo, nullptr, sched, lane, kLitePixels);
        return;
    }
    FwdRing& R = sm.ring;
    uint32_t* const idx = sm.list[warp].idx;
    const uint32_t lt_mask = (1u << lane) - 1u;

    // per-tile state of this consumer's 32 pixels
    UnitInfo ui;
    ui.start = ui.end = ui.slot = 0; ui.active = false;
    PixelBox box = {0.f, 0.f, 0.f, 0.f};
    float px = 0.f, py = 0.f, T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
    bool alive = false;  // this lane's pixel is sampled and not yet terminated
    uint32_t last = 0, walked = 0, blended = 0;
    bool open = false;  // a tile is in progress and its outputs are not written yet
    uint32_t gchunk = 0, seq = 0;

    auto finalize = [&]() {
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
        open = false;
        if (lane == 0) *(volatile uint32_t*)&R.done_seq[warp] = seq;
    };

    for (;;) {
        const uint32_t s = gchunk % FwdRing::kStages;
        mbar_wait(&R.full[s], (gchunk / FwdRing::kStages) & 1u);
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
                if (ui.active) {
                    const uint32_t id = pix[ui.slot];
                    ipx = (int)(id % (uint32_t)cam.W);
                    ipy = (int)(id / (uint32_t)cam.W);
                }
                box = warp_pixel_box(ui.active, ipx, ipy);
                // `alive` gates the blend decision only, so that the evaluation of the next survivor never waits
                // for this one's termination test (it did while a finished lane was marked by px = NaN: a
                // loop-carried chain through the whole evaluation)
                px = (float)ipx;
                py = (float)ipy;
                alive = ui.active;
                T = 1.0f; C0 = 0.f; C1 = 0.f; C2 = 0.f;
                last = 0; walked = ui.end - ui.start; blended = 0;
            }
        }
        if (open) {
            const Stage<kFwdStageEntries>& st = R.st[s];
            // the box shrinks with the pixels that are still alive: a Gaussian that only reaches terminated pixels is culled
            if (inf.hdr == kHdrCont) box = warp_pixel_box(alive, (int)px, (int)py);
            // ---- cull the stage against the pixel box; survivors' indices in range order ----
            uint32_t n = 0;
            for (uint32_t b0 = 0; b0 < inf.cnt; b0 += 32) {
                const uint32_t i = b0 + lane;
                const float4 q0 = st.p0[i];
                const float2 c2 = st.ct[i];
                const bool pass = i < inf.cnt && splat_may_touch(q0.x, q0.y, q0.z, q0.w, c2.x, c2.y, box);
                const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
                if (pass) idx[n + __popc(ballot & lt_mask)] = i;
                n += __popc(ballot);
            }
            __syncwarp();
            // ---- walk the survivors in place (branch free) ----
            auto eval = [&](uint32_t i) {
                const float4 a = st.p0[i];
                const float4 b = st.p1[i];   // -C/2, opacity, red, green
                const float blue = st.bl[i];
                const float dx = a.x - px, dy = a.y - py;
                const float power = splat_power(a.z, a.w, b.x, dx, dy);
                const float alpha = fminf(kAlphaMax, __fmul_rn(b.y, ex2_approx(power * kLog2e)));
                const bool blend = alive && (power <= 0.0f) && !(alpha < kAlphaMin);
                const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                const bool term = blend && (Tn < kTMin);
                const bool upd = blend && !term;
                const float w = upd ? alpha * T : 0.0f;
                C0 = fmaf(b.z, w, C0); C1 = fmaf(b.w, w, C1); C2 = fmaf(blue, w, C2);
                T = upd ? Tn : T;
                const uint32_t pos = inf.base + i + 1u;   // 1-based range position
                last = upd ? pos : last;
                if (COUNT) {
                    blended += upd ? 1u : 0u;
                    walked = term ? pos : walked;
                }
                alive = alive && !term;
            };
            uint32_t e = 0;
            for (; e + 4 <= n; e += 4) {
                const uint4 j = *reinterpret_cast<const uint4*>(idx + e);
                eval(j.x); eval(j.y); eval(j.z); eval(j.w);
            }
            for (; e < n; ++e) eval(idx[e]);
            __syncwarp();  // the list is rewritten at the next stage
            if (!__any_sync(0xffffffffu, alive)) finalize();
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&R.empty[s]);
        ++gchunk;
    }
}

}  // namespace

cudaError_t launch_raster_fwd(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, float* out_color, float* out_T, uint32_t* n_contrib,
                              uint32_t* n_walked, uint32_t* n_blended, uint32_t* sched, int num_sms, cudaStream_t s,
                              const SideStream* side) {
    if (k <= 0) return cudaSuccess;
    // fork: tiles with <= kLitePixels sampled pixels go to the warp-per-tile kernel (raster_lite.cu; its own
    // counters at sched + 2) on the context's side stream, concurrently with the block-per-tile kernel
    cudaError_t e = cudaEventRecord(side->fork, s);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(side->aux, side->fork, 0);
    if (e == cudaSuccess)
        e = launch_raster_fwd_lite(cam, splats, tile_offsets, gid_sorted, k, tiles, tpo, pix, out_color, out_T, n_contrib,
                                   n_walked, n_blended, sched + 2, num_sms, side->aux);
    if (e == cudaSuccess) e = cudaEventRecord(side->join, side->aux);
    if (e != cudaSuccess) return e;
    const bool count = n_walked || n_blended;
    // persistent grid: one block per sampled tile at a time
    int blocks = num_sms * 4;
    if (blocks > k) blocks = k;
    const float4* sp = reinterpret_cast<const float4*>(splats);
    constexpr size_t smem = sizeof(FwdShared);
    static SmemOptIn opt_count, opt_plain;  // per device
    e = count ? opt_count.ensure((const void*)raster_fwd_kernel<true>, smem) : opt_plain.ensure((const void*)raster_fwd_kernel<false>, smem);
    if (e != cudaSuccess) return e;
    if (count)
        raster_fwd_kernel<true><<<blocks, kRasterThreads, smem, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                  out_color, out_T, n_contrib, n_walked, n_blended, sched);
    else
        raster_fwd_kernel<false><<<blocks, kRasterThreads, smem, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                   out_color, out_T, n_contrib, n_walked, n_blended, sched);
    count_launches(1);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return cudaStreamWaitEvent(s, side->join, 0);  // join
}

}  // namespace tgs
