// tgs_raster_bwd_sparse, raster half: back-to-front replay of Eq. 1 over the sampled
// pixels only, producing dL/d(mean2D, conic, opacity, rgb) per Gaussian.
// One block per sampled tile; per-Gaussian partials are reduced across the warp with shuffles and
// one lane issues the global atomics (north_star: "warp-shuffle reduction of per-Gaussian gradients
// before global atomics").
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kBwdThreads = 256;
constexpr int kBatch = 256;

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(kBwdThreads)
raster_bwd_kernel(const CamK cam, const float4* __restrict__ splats, const uint32_t* __restrict__ tile_offsets,
                  const uint32_t* __restrict__ gid_sorted, int k, const uint32_t* __restrict__ tiles,
                  const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                  const float* __restrict__ out_T, const uint32_t* __restrict__ n_contrib,
                  const float* __restrict__ dL_dcolor, float* __restrict__ dL_dsplats) {
    __shared__ float4 s_a[kBatch];  // mx, my, -A/2, -B
    __shared__ float4 s_b[kBatch];  // -C/2, opacity, r, g
    __shared__ float s_c[kBatch];   // b
    __shared__ uint32_t s_g[kBatch];
    __shared__ uint32_t s_max;

    const int lane = threadIdx.x & 31;
    for (int it = blockIdx.x; it < k; it += gridDim.x) {
        const uint32_t t = tiles[it];
        const uint32_t start = tile_offsets[t];
        const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0;
        const bool active = threadIdx.x < m;
        float px = 0.f, py = 0.f, Tf = 0.f, g0 = 0.f, g1 = 0.f, g2 = 0.f;
        uint32_t last = 0;
        if (active) {
            const uint32_t o = p0 + threadIdx.x;
            const uint32_t id = pix[o];
            px = (float)(id % (uint32_t)cam.W);
            py = (float)(id / (uint32_t)cam.W);
            Tf = out_T[o];
            last = n_contrib[o];
            g0 = dL_dcolor[3 * (size_t)o]; g1 = dL_dcolor[3 * (size_t)o + 1]; g2 = dL_dcolor[3 * (size_t)o + 2];
        }
        if (threadIdx.x == 0) s_max = 0;
        __syncthreads();
        {
            uint32_t wm = __reduce_max_sync(0xffffffffu, last);
            if (lane == 0 && wm) atomicMax(&s_max, wm);
        }
        __syncthreads();
        const uint32_t max_last = s_max;
        const float bgdot = (cam.bg[0] * g0 + cam.bg[1] * g1 + cam.bg[2] * g2) * Tf;
        float T = Tf, S0 = 0.f, S1 = 0.f, S2 = 0.f;

        // batches of the range [0, max_last), from the back
        for (uint32_t hi = max_last; hi > 0;) {
            const uint32_t cnt = min((uint32_t)kBatch, hi);
            const uint32_t b0 = hi - cnt;
            __syncthreads();
            if (threadIdx.x < cnt) {
                const uint32_t g = gid_sorted[start + b0 + threadIdx.x];
                const float4 r0 = splats[3 * (size_t)g], r1 = splats[3 * (size_t)g + 1];
                const float bl = reinterpret_cast<const float*>(splats)[(size_t)g * kSplatWords + 8];
                s_a[threadIdx.x] = make_float4(r0.x, r0.y, -0.5f * r0.z, -r0.w);
                s_b[threadIdx.x] = make_float4(-0.5f * r1.x, r1.y, r1.z, r1.w);
                s_c[threadIdx.x] = bl;
                s_g[threadIdx.x] = g;
            }
            __syncthreads();
            for (int jj = (int)cnt - 1; jj >= 0; --jj) {
                const uint32_t pos = b0 + (uint32_t)jj;
                const float4 a = s_a[jj];
                const float4 bb = s_b[jj];
                const float dx = a.x - px, dy = a.y - py;
                const float power = __fmaf_rn(__fmaf_rn(a.w, dy, __fmul_rn(a.z, dx)), dx,
                                              __fmul_rn(__fmul_rn(bb.x, dy), dy));
                const float G = __expf(power);
                const float oG = __fmul_rn(bb.y, G);
                const float alpha = fminf(kAlphaMax, oG);
                const bool valid = active && pos < last && !(power > 0.0f) && !(alpha < kAlphaMin);
                if (!__any_sync(0xffffffffu, valid)) continue;
                float d_mx = 0.f, d_my = 0.f, d_A = 0.f, d_B = 0.f, d_C = 0.f, d_o = 0.f, d_r = 0.f, d_g = 0.f, d_b = 0.f;
                if (valid) {
                    const float om = 1.0f - alpha;
                    const float rom = __frcp_rn(om);
                    T = T * rom;  // T_k
                    const float w = alpha * T;
                    const float cb = s_c[jj];
                    d_r = w * g0; d_g = w * g1; d_b = w * g2;
                    float dL_dalpha = ((bb.z - S0) * g0 + (bb.w - S1) * g1 + (cb - S2) * g2) * T - bgdot * rom;
                    S0 = fmaf(alpha, bb.z, om * S0); S1 = fmaf(alpha, bb.w, om * S1); S2 = fmaf(alpha, cb, om * S2);
                    if (oG < kAlphaMax) {  // zero derivative through the active 0.99 clamp
                        const float dpow = oG * dL_dalpha;
                        d_o = G * dL_dalpha;
                        // -A dx - B dy = 2(-A/2) dx + (-B) dy ; -C dy - B dx = 2(-C/2) dy + (-B) dx
                        d_mx = dpow * fmaf(2.0f * a.z, dx, a.w * dy);
                        d_my = dpow * fmaf(2.0f * bb.x, dy, a.w * dx);
                        d_A = -0.5f * dx * dx * dpow;
                        d_B = -dx * dy * dpow;
                        d_C = -0.5f * dy * dy * dpow;
                    }
                }
                d_mx = warp_sum(d_mx); d_my = warp_sum(d_my); d_A = warp_sum(d_A); d_B = warp_sum(d_B);
                d_C = warp_sum(d_C); d_o = warp_sum(d_o); d_r = warp_sum(d_r); d_g = warp_sum(d_g); d_b = warp_sum(d_b);
                if (lane == 0) {
                    float* dst = dL_dsplats + (size_t)s_g[jj] * kSplatWords;
                    atomicAdd(dst + 0, d_mx); atomicAdd(dst + 1, d_my); atomicAdd(dst + 2, d_A);
                    atomicAdd(dst + 3, d_B); atomicAdd(dst + 4, d_C); atomicAdd(dst + 5, d_o);
                    atomicAdd(dst + 6, d_r); atomicAdd(dst + 7, d_g); atomicAdd(dst + 8, d_b);
                }
            }
            hi = b0;
        }
        __syncthreads();
    }
}

}  // namespace

cudaError_t launch_raster_bwd(const CamK& cam, int N, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, const float* out_T, const uint32_t* n_contrib,
                              const float* dL_dcolor, float* dL_dsplats, int num_sms, cudaStream_t s) {
    (void)num_sms;
    cudaError_t e = cudaMemsetAsync(dL_dsplats, 0, (size_t)N * kSplatWords * sizeof(float), s);
    if (e != cudaSuccess) return e;
    if (k <= 0) return cudaSuccess;
    raster_bwd_kernel<<<k, kBwdThreads, 0, s>>>(cam, reinterpret_cast<const float4*>(splats), tile_offsets,
                                                gid_sorted, k, tiles, tpo, pix, out_T, n_contrib, dL_dcolor,
                                                dL_dsplats);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
