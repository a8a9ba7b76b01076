// tgs_loss_sparse: sparse supervision on the sampled pixels (PAPER.md:168-208
// Sec. 3.7 Eq. 9-11, Eq. 17-18): Charbonnier pixel term, tile-level sparse NCC term,
// gradient-balanced lambda per tile; writes dL/dcolor for tgs_raster_bwd_sparse, the per-pixel error
// (Eq. 2) and per-tile statistics, in ONE pass over the sampled pixels.
//
// The paper gives a block per tile with block-level reductions.  A tile holds at most
// 256 sampled pixels, so here a WARP owns a tile: 8 pixels per lane live in registers across the
// three dependent reductions (means -> centred moments and the l1 statistics -> NCC gradient norm),
// every reduction is a fixed xor-butterfly (bit-reproducible), and there is no shared memory or
// barrier at all.  HBM-bound: 12 B colour + 12 B gathered target + 4 B index read, 12 + 4 B written
// per sampled pixel.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kPerLane = kTilePixels / 32;  // 8

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

__global__ void __launch_bounds__(256)
loss_sparse_kernel(int k, const uint32_t* __restrict__ tpo, const uint32_t* __restrict__ pix,
                   const float* __restrict__ color, const float* __restrict__ target, float eps_l1, float eps_ncc,
                   float eps_lam, float* __restrict__ dL_dcolor, float* __restrict__ pix_err,
                   float* __restrict__ tile_stats) {
    const int lane = threadIdx.x & 31;
    const int it = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5);
    if (it >= k) return;
    const uint32_t p0 = tpo[it], m = tpo[it + 1] - p0, n = tpo[k];
    if (m == 0) {  // an empty tile (never produced by the library's samplers): no pixel, no term
        if (lane < 3) tile_stats[3 * (size_t)it + lane] = 0.f;
        return;
    }
    const float inv_m = 1.0f / (float)m, inv_n = 1.0f / (float)n;

    float x[kPerLane][3], y[kPerLane][3];
    float sx[3] = {0.f, 0.f, 0.f}, sy[3] = {0.f, 0.f, 0.f};
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const uint32_t i = (uint32_t)lane + 32u * j;
        const bool on = i < m;
        const uint32_t s = p0 + (on ? i : 0u);
        const uint32_t id = pix[s];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            x[j][c] = on ? color[3 * (size_t)s + c] : 0.f;
            y[j][c] = on ? target[3 * (size_t)id + c] : 0.f;
            sx[c] += x[j][c];
            sy[c] += y[j][c];
        }
    }
    float mux[3], muy[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        mux[c] = warp_sum(sx[c]) * inv_m;
        muy[c] = warp_sum(sy[c]) * inv_m;
    }
    // centred moments, Charbonnier sum and its gradient 1-norm
    float vx[3] = {0.f, 0.f, 0.f}, vy[3] = {0.f, 0.f, 0.f}, cxy[3] = {0.f, 0.f, 0.f};
    float l1sum = 0.f, g1abs = 0.f;
    const float e1sq = eps_l1 * eps_l1;
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const bool on = (uint32_t)lane + 32u * j < m;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float dx = x[j][c] - mux[c], dy = y[j][c] - muy[c];
            const float d = x[j][c] - y[j][c];
            const float ch = sqrtf(d * d + e1sq);
            if (on) {
                vx[c] += dx * dx; vy[c] += dy * dy; cxy[c] += dx * dy;
                l1sum += ch;
                g1abs += fabsf(d / ch);
            }
        }
    }
    float ncc[3], rden[3], kx[3], Lncc = 0.f;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const float a = warp_sum(vx[c]) * inv_m, b = warp_sum(vy[c]) * inv_m, ab = warp_sum(cxy[c]) * inv_m;
        const float den = a * b + eps_ncc;
        rden[c] = 1.0f / sqrtf(den);
        ncc[c] = ab * rden[c];
        kx[c] = ncc[c] * b / den;  // coefficient of (x - mu_x) in Eq. 17
        Lncc += (1.0f - ncc[c]);
    }
    Lncc *= (1.0f / 3.0f);
    l1sum = warp_sum(l1sum) * (1.0f / 3.0f);
    const float g1bar = warp_sum(g1abs) * (1.0f / 3.0f) * inv_m;
    // NCC gradient 1-norm (Eq. 10), then lambda (Eq. 18)
    float gNabs = 0.f;
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const bool on = (uint32_t)lane + 32u * j < m;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const float gN = -((y[j][c] - muy[c]) * rden[c] - kx[c] * (x[j][c] - mux[c])) * (1.0f / 3.0f);
            if (on) gNabs += fabsf(gN);
        }
    }
    const float gNbar = warp_sum(gNabs) * inv_m;
    const float lam = fminf(1.0f, fmaxf(0.0f, g1bar / (gNbar + eps_lam)));
    // outputs
#pragma unroll
    for (int j = 0; j < kPerLane; ++j) {
        const uint32_t i = (uint32_t)lane + 32u * j;
        if (i < m) {
            const uint32_t s = p0 + i;
            float e = 0.f;
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const float d = x[j][c] - y[j][c];
                const float g1 = (d / sqrtf(d * d + e1sq)) * (1.0f / 3.0f);
                const float gN = -((y[j][c] - muy[c]) * rden[c] - kx[c] * (x[j][c] - mux[c])) * (1.0f / 3.0f);
                dL_dcolor[3 * (size_t)s + c] = (g1 + lam * gN) * inv_n;
                e += fabsf(d);
            }
            pix_err[s] = e;
        }
    }
    if (lane == 0) {
        tile_stats[3 * (size_t)it] = l1sum;
        tile_stats[3 * (size_t)it + 1] = Lncc;
        tile_stats[3 * (size_t)it + 2] = lam;
    }
}

// loss[0] = 1/n sum_p l1(p), loss[1] = 1/n sum_tau lambda m L_ncc (Eq. 11): one block, fixed summation order
__global__ void __launch_bounds__(1024)
loss_reduce_kernel(int k, const uint32_t* __restrict__ tpo, const float* __restrict__ tile_stats, float* __restrict__ loss) {
    __shared__ double s0[32], s1[32];
    double a = 0.0, b = 0.0;
    for (int t = threadIdx.x; t < k; t += blockDim.x) {
        a += (double)tile_stats[3 * (size_t)t];
        b += (double)tile_stats[3 * (size_t)t + 2] * (double)(tpo[t + 1] - tpo[t]) * (double)tile_stats[3 * (size_t)t + 1];
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_xor_sync(0xffffffffu, a, o);
        b += __shfl_xor_sync(0xffffffffu, b, o);
    }
    if ((threadIdx.x & 31) == 0) { s0[threadIdx.x >> 5] = a; s1[threadIdx.x >> 5] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double A = 0.0, B = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { A += s0[w]; B += s1[w]; }
        const double n = (double)tpo[k];
        loss[0] = n > 0.0 ? (float)(A / n) : 0.f;
        loss[1] = n > 0.0 ? (float)(B / n) : 0.f;
    }
}

}  // namespace

cudaError_t launch_loss_sparse(int k, const uint32_t* tpo, const uint32_t* pix, const float* color, const float* target,
                               float eps_l1, float eps_ncc, float eps_lam, float* dL_dcolor, float* pix_err,
                               float* tile_stats, float* loss, cudaStream_t s) {
    if (k > 0) {
        loss_sparse_kernel<<<(k + 7) / 8, 256, 0, s>>>(k, tpo, pix, color, target, eps_l1, eps_ncc, eps_lam, dL_dcolor,
                                                       pix_err, tile_stats);
        count_launches(1);
    }
    if (loss) {
        loss_reduce_kernel<<<1, 1024, 0, s>>>(k, tpo, tile_stats, loss);
        count_launches(1);
    }
    return cudaGetLastError();
}

}  // namespace tgs
