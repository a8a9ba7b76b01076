// tgs_raster_fwd_sparse: front-to-back alpha compositing (Eq. 1) for the SAMPLED
// pixels only (Fig. 6: sampled pixels listed tile by tile, tile-wise pixel
// offsets by prefix sum, tile-parallel execution).
//
// B200 design (raster_common.cuh): one persistent block per sampled tile at a time; a producer warp
// gathers the tile's depth-ordered splat records once into a shared-memory stage ring (mbarrier
// full/empty), eight consumer warps each own 32 of the tile's sampled pixels, cull every staged
// batch against the bounding box of their own pixels and walk only the survivors with a
// branch-free, unrolled inner loop (per survivor: three shared loads, ~25 FP32/ALU ops, one
// MUFU.EX2).
//
// power uses the one fixed fused sequence of DESIGN.md "canonical arithmetic", so `power > 0` is
// decided on the same bits as the oracle; alpha itself is o * ex2.approx(power * log2 e).
#include "raster_common.cuh"

namespace tgs {

namespace {

struct FwdShared {
    Ring<128> ring;
    WarpBatch batch[kConsumers];
};

template <bool COUNT>
__global__ void __launch_bounds__(kRasterThreads, 4)
raster_fwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  float* __restrict__ out_color, float* __restrict__ out_T, uint32_t* __restrict__ n_contrib,
                  uint32_t* __restrict__ n_walked, uint32_t* __restrict__ n_blended, uint32_t* __restrict__ sched) {
    __shared__ __align__(16) FwdShared sm;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    ring_init(sm.ring);
    if (warp == kConsumers) {
        producer_loop<false>(sm.ring, splats, tile_offsets, gid_sorted, (uint32_t)k, tiles, tpo, nullptr, sched, lane, kLitePixels);
        return;
    }
    Ring<128>& R = sm.ring;
    WarpBatch& sb = sm.batch[warp];
    const uint32_t lt_mask = (1u << lane) - 1u;
    const float kNaN = __int_as_float(0x7fc00000);

    // per-tile state of this consumer's 32 pixels
    UnitInfo ui;
    ui.start = ui.end = ui.slot = 0; ui.active = false;
    PixelBox box = {0.f, 0.f, 0.f, 0.f};
    float px = kNaN, py = 0.f, T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
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
        const uint32_t s = gchunk % kStages;
        mbar_wait(&R.full[s], (gchunk / kStages) & 1u);
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
                // a finished (or inactive) lane carries px = NaN: power becomes NaN and every test fails
                px = ui.active ? (float)ipx : kNaN;
                py = (float)ipy;
                T = 1.0f; C0 = 0.f; C1 = 0.f; C2 = 0.f;
                last = 0; walked = ui.end - ui.start; blended = 0;
            }
        }
        if (open) {
            const Stage<128>& st = R.st[s];
            for (uint32_t b0 = 0; b0 < inf.cnt; b0 += 32) {
                // ---- cull this batch against the pixel box, compact survivors in range order ----
                const uint32_t i = b0 + lane;
                const bool have = i < inf.cnt;
                const float4 q0 = st.p0[i];
                const float4 q1 = st.p1[i];
                const bool pass = have && splat_may_touch(q0.x, q0.y, q0.z, q0.w, q1.x, q1.y, box);
                const uint32_t ballot = __ballot_sync(0xffffffffu, pass);
                const int cnt = __popc(ballot);
                if (pass) {
                    const float4 q2 = st.p2[i];
                    const int slot = __popc(ballot & lt_mask);
                    sb.a[slot] = q0;
                    sb.b[slot] = make_float4(q1.x, q1.y, q1.z, __uint_as_float(inf.base + i + 1u));
                    sb.c[slot] = make_float4(q1.w, q2.x, q2.y, 0.f);
                }
                __syncwarp();
                // ---- walk the survivors (branch free) ----
#pragma unroll 4
                for (int e = 0; e < cnt; ++e) {
                    const float4 a = sb.a[e];
                    const float4 b = sb.b[e];
                    const float4 c = sb.c[e];
                    const float dx = a.x - px, dy = a.y - py;
                    const float power = splat_power(a.z, a.w, b.x, dx, dy);
                    const float alpha = fminf(kAlphaMax, __fmul_rn(b.z, ex2_approx(power * kLog2e)));
                    const bool blend = (power <= 0.0f) && !(alpha < kAlphaMin);  // thr (b.y) only serves the cull
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
                __syncwarp();  // the batch slice is rewritten next iteration
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
    if (count)
        raster_fwd_kernel<true><<<blocks, kRasterThreads, 0, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                  out_color, out_T, n_contrib, n_walked, n_blended, sched);
    else
        raster_fwd_kernel<false><<<blocks, kRasterThreads, 0, s>>>(cam, sp, tile_offsets, gid_sorted, k, tiles, tpo, pix,
                                                                   out_color, out_T, n_contrib, n_walked, n_blended, sched);
    count_launches(1);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return cudaStreamWaitEvent(s, side->join, 0);  // join
}

}  // namespace tgs
