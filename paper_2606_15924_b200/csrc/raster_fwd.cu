// tgs_raster_fwd_sparse: front-to-back alpha compositing (Eq. 1) for the SAMPLED
// pixels only, one thread block per valid sampled tile (Fig. 6), Gaussian
// records of the tile's depth-ordered range staged through shared memory in batches.
//
// power is evaluated with one fixed fused sequence:
//   power = fma(fma(-B, dy, (-A/2) dx), dx, ((-C/2) dy) dy)
// so that the skip decisions (power > 0, alpha < 1/255, T < 1e-4) are taken on the same bits as the
// oracle's; only exp differs (ex2.approx vs libm), within tolerance.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kFwdThreads = 256;
constexpr int kBatch = 256;

__global__ void __launch_bounds__(kFwdThreads)
raster_fwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  float* __restrict__ out_color, float* __restrict__ out_T, uint32_t* __restrict__ n_contrib,
                  uint32_t* __restrict__ n_walked, uint32_t* __restrict__ n_blended) {
    __shared__ float4 s_a[kBatch];  // mx, my, -A/2, -B
    __shared__ float4 s_b[kBatch];  // -C/2, opacity, r, g
    __shared__ float s_c[kBatch];   // b

    for (int it = blockIdx.x; it < k; it += gridDim.x) {
        const uint32_t t = tiles[it];
        const uint32_t start = tile_offsets[t], end = tile_offsets[t + 1];
        const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
        const bool active = threadIdx.x < m;
        float px = 0.f, py = 0.f;
        if (active) {
            const uint32_t id = pix[p0 + threadIdx.x];
            px = (float)(id % (uint32_t)cam.W);
            py = (float)(id / (uint32_t)cam.W);
        }
        float T = 1.0f, C0 = 0.f, C1 = 0.f, C2 = 0.f;
        uint32_t last = 0, walked = 0, blended = 0;
        bool done = !active;

        for (uint32_t b0 = start; b0 < end; b0 += kBatch) {
            if (__syncthreads_count(done) == kFwdThreads) break;
            const uint32_t j = b0 + threadIdx.x;
            if (j < end) {
                const uint32_t g = gid_sorted[j];
                const float4 r0 = splats[3 * (size_t)g], r1 = splats[3 * (size_t)g + 1];
                const float bl = reinterpret_cast<const float*>(splats)[(size_t)g * kSplatWords + 8];
                s_a[threadIdx.x] = make_float4(r0.x, r0.y, -0.5f * r0.z, -r0.w);
                s_b[threadIdx.x] = make_float4(-0.5f * r1.x, r1.y, r1.z, r1.w);
                s_c[threadIdx.x] = bl;
            }
            __syncthreads();
            if (!done) {
                const uint32_t cnt = min((uint32_t)kBatch, end - b0);
                for (uint32_t jj = 0; jj < cnt; ++jj) {
                    ++walked;
                    const float4 a = s_a[jj];
                    const float dx = a.x - px, dy = a.y - py;
                    const float power = __fmaf_rn(__fmaf_rn(a.w, dy, __fmul_rn(a.z, dx)), dx,
                                                  __fmul_rn(__fmul_rn(s_b[jj].x, dy), dy));
                    if (power > 0.0f) continue;
                    const float4 bb = s_b[jj];
                    const float alpha = fminf(kAlphaMax, __fmul_rn(bb.y, __expf(power)));
                    if (alpha < kAlphaMin) continue;
                    const float Tn = __fmul_rn(T, __fsub_rn(1.0f, alpha));
                    if (Tn < kTMin) { done = true; break; }
                    const float w = alpha * T;
                    C0 = fmaf(bb.z, w, C0); C1 = fmaf(bb.w, w, C1); C2 = fmaf(s_c[jj], w, C2);
                    T = Tn;
                    ++blended;
                    last = (b0 - start) + jj + 1;
                }
            }
        }
        if (active) {
            const uint32_t o = p0 + threadIdx.x;
            out_color[3 * (size_t)o] = fmaf(T, cam.bg[0], C0);
            out_color[3 * (size_t)o + 1] = fmaf(T, cam.bg[1], C1);
            out_color[3 * (size_t)o + 2] = fmaf(T, cam.bg[2], C2);
            out_T[o] = T;
            n_contrib[o] = last;
            if (n_walked) n_walked[o] = walked;
            if (n_blended) n_blended[o] = blended;
        }
        __syncthreads();  // shared batch buffers are reused by the next tile
    }
}

}  // namespace

cudaError_t launch_raster_fwd(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, float* out_color, float* out_T, uint32_t* n_contrib,
                              uint32_t* n_walked, uint32_t* n_blended, int num_sms, cudaStream_t s) {
    (void)num_sms;
    if (k <= 0) return cudaSuccess;
    raster_fwd_kernel<<<k, kFwdThreads, 0, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                gid_sorted, k, tiles, tpo, pix, out_color, out_T, n_contrib,
                                                n_walked, n_blended);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
