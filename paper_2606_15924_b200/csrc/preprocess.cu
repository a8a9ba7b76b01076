// tgs_preprocess: EWA projection of 3D Gaussians to 2D splat records (
// PAPER.md:62-64 "3DGS projects Gaussians to the image plane", 75 "the original rasterization
// kernels").
//
// THIS TRANSLATION UNIT IS COMPILED WITH -fmad=false.  Tile rects, depth keys and mean2D decide
// integers downstream (sort keys, tile ranges), so every product and sum below is rounded once,
// in the order written; '/' and sqrtf are IEEE (no fast-math).
// The kernel is HBM-bound (236 B in + 53 B out per Gaussian at degree 3), so this costs nothing.
#include "common.cuh"

namespace tgs {

namespace {

constexpr float SH_C0 = 0.28209479177387814f;
constexpr float SH_C1 = 0.4886025119029199f;
constexpr float SH_C2A = 1.0925484305920792f;
constexpr float SH_C2B = 0.31539156525252005f;
constexpr float SH_C2C = 0.5462742152960396f;
constexpr float SH_C3A = 0.5900435899266435f;
constexpr float SH_C3B = 2.890611442640554f;
constexpr float SH_C3C = 0.4570457994644658f;
constexpr float SH_C3D = 0.3731763325901154f;
constexpr float SH_C3E = 1.445305721320277f;

template <int D>
__device__ __forceinline__ void sh_basis(float x, float y, float z, float* B) {
    B[0] = SH_C0;
    if (D >= 1) {
        B[1] = (-SH_C1) * y;
        B[2] = SH_C1 * z;
        B[3] = (-SH_C1) * x;
    }
    if (D >= 2) {
        float xx = x * x, yy = y * y, zz = z * z, xy = x * y, yz = y * z, xz = x * z;
        B[4] = SH_C2A * xy;
        B[5] = (-SH_C2A) * yz;
        B[6] = SH_C2B * ((2.0f * zz - xx) - yy);
        B[7] = (-SH_C2A) * xz;
        B[8] = SH_C2C * (xx - yy);
        if (D >= 3) {
            B[9] = ((-SH_C3A) * y) * (3.0f * xx - yy);
            B[10] = (SH_C3B * xy) * z;
            B[11] = ((-SH_C3C) * y) * ((4.0f * zz - xx) - yy);
            B[12] = (SH_C3D * z) * ((2.0f * zz - 3.0f * xx) - 3.0f * yy);
            B[13] = ((-SH_C3C) * x) * ((4.0f * zz - xx) - yy);
            B[14] = (SH_C3E * z) * (xx - yy);
            B[15] = ((-SH_C3A) * x) * (xx - 3.0f * yy);
        }
    }
}

template <int D>
__global__ void __launch_bounds__(128)
preprocess_kernel(const CamK cam, int N, const float* __restrict__ mu, const float* __restrict__ sc,
                  const float* __restrict__ qt, const float* __restrict__ op, const float* __restrict__ sh,
                  float4* __restrict__ splats, int32_t* __restrict__ radii, uint8_t* __restrict__ clamped) {
    constexpr int K = (D + 1) * (D + 1);
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;

    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0, r2 = r0;
    int rad_out = 0;
    uint8_t cl = 0;

    const float m0 = mu[3 * i], m1 = mu[3 * i + 1], m2 = mu[3 * i + 2];
    const float* W = cam.R;
    const float t0 = ((W[0] * m0 + W[1] * m1) + W[2] * m2) + cam.t[0];
    const float t1 = ((W[3] * m0 + W[4] * m1) + W[5] * m2) + cam.t[1];
    const float tz = ((W[6] * m0 + W[7] * m1) + W[8] * m2) + cam.t[2];
    if (tz > cam.znear) {
        const float limx = kJClamp * ((0.5f * (float)cam.W) / cam.fx);
        const float limy = kJClamp * ((0.5f * (float)cam.H) / cam.fy);
        const float txtz = t0 / tz, tytz = t1 / tz;
        float cxr = txtz, cyr = tytz;
        if (cxr > limx) cxr = limx; else if (cxr < -limx) cxr = -limx;
        if (cyr > limy) cyr = limy; else if (cyr < -limy) cyr = -limy;
        const float txc = cxr * tz, tyc = cyr * tz;
        const float tz2 = tz * tz;
        const float J00 = cam.fx / tz;
        const float J02 = -(cam.fx * txc) / tz2;
        const float J11 = cam.fy / tz;
        const float J12 = -(cam.fy * tyc) / tz2;
        float Tm[6];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Tm[c] = J00 * W[c] + J02 * W[6 + c];
            Tm[3 + c] = J11 * W[3 + c] + J12 * W[6 + c];
        }
        // Sigma = M M^T, M = R(q) diag(s)
        const float4 q = reinterpret_cast<const float4*>(qt)[i];
        const float w = q.x, x = q.y, y = q.z, z = q.w;
        float Rq[9];
        Rq[0] = 1.0f - 2.0f * (y * y + z * z);
        Rq[1] = 2.0f * (x * y - w * z);
        Rq[2] = 2.0f * (x * z + w * y);
        Rq[3] = 2.0f * (x * y + w * z);
        Rq[4] = 1.0f - 2.0f * (x * x + z * z);
        Rq[5] = 2.0f * (y * z - w * x);
        Rq[6] = 2.0f * (x * z - w * y);
        Rq[7] = 2.0f * (y * z + w * x);
        Rq[8] = 1.0f - 2.0f * (x * x + y * y);
        const float s0 = sc[3 * i], s1 = sc[3 * i + 1], s2 = sc[3 * i + 2];
        float M[9];
#pragma unroll
        for (int r = 0; r < 3; ++r) {
            M[3 * r] = Rq[3 * r] * s0; M[3 * r + 1] = Rq[3 * r + 1] * s1; M[3 * r + 2] = Rq[3 * r + 2] * s2;
        }
        float Sg[9];
#pragma unroll
        for (int r = 0; r < 3; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                Sg[3 * r + c] = M[3 * r] * M[3 * c] + M[3 * r + 1] * M[3 * c + 1] + M[3 * r + 2] * M[3 * c + 2];
        float V[6];
#pragma unroll
        for (int r = 0; r < 2; ++r)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                V[3 * r + c] = Tm[3 * r] * Sg[c] + Tm[3 * r + 1] * Sg[3 + c] + Tm[3 * r + 2] * Sg[6 + c];
        const float c00 = V[0] * Tm[0] + V[1] * Tm[1] + V[2] * Tm[2];
        const float c01 = V[0] * Tm[3] + V[1] * Tm[4] + V[2] * Tm[5];
        const float c11 = V[3] * Tm[3] + V[4] * Tm[4] + V[5] * Tm[5];
        const float a = c00 + kLowpass, b = c01, c = c11 + kLowpass;
        const float det = a * c - b * b;
        if (det > 0.0f) {
            const float A = c / det, B = (-b) / det, C = a / det;
            const float mid = 0.5f * (a + c);
            const float lam = mid + sqrtf(fmaxf(0.1f, mid * mid - det));
            const float rad = ceilf(3.0f * sqrtf(lam));
            const float mx = (cam.fx * txtz + cam.cx) - 0.5f;
            const float my = (cam.fy * tytz + cam.cy) - 0.5f;
            const float fgx = (float)cam.gx, fgy = (float)cam.gy;
            const int x0 = (int)fminf(fmaxf(floorf((mx - rad) / 16.0f), 0.0f), fgx);
            const int x1 = (int)fminf(fmaxf(floorf(((mx + rad) + 15.0f) / 16.0f), 0.0f), fgx);
            const int y0 = (int)fminf(fmaxf(floorf((my - rad) / 16.0f), 0.0f), fgy);
            const int y1 = (int)fminf(fmaxf(floorf(((my + rad) + 15.0f) / 16.0f), 0.0f), fgy);
            if ((x1 - x0) > 0 && (y1 - y0) > 0) {
                // view-dependent colour: d = (mu - o_cam)/|mu - o_cam|, o_cam = -R^T t
                const float o0 = -((W[0] * cam.t[0] + W[3] * cam.t[1]) + W[6] * cam.t[2]);
                const float o1 = -((W[1] * cam.t[0] + W[4] * cam.t[1]) + W[7] * cam.t[2]);
                const float o2 = -((W[2] * cam.t[0] + W[5] * cam.t[1]) + W[8] * cam.t[2]);
                const float v0 = m0 - o0, v1 = m1 - o1, v2 = m2 - o2;
                const float len = sqrtf((v0 * v0 + v1 * v1) + v2 * v2);
                float Bk[K];
                sh_basis<D>(v0 / len, v1 / len, v2 / len, Bk);
                float acc[3];
                const float* s_i = sh + (size_t)i * (K * 3);
                if (D == 1 || D == 3) {
                    // K*3 floats = 12 or 48: whole float4s, 16-byte aligned records
                    float buf[K * 3];
                    const float4* s4 = reinterpret_cast<const float4*>(s_i);
#pragma unroll
                    for (int v = 0; v < (K * 3) / 4; ++v) {
                        float4 f = __ldg(s4 + v);
                        buf[4 * v] = f.x; buf[4 * v + 1] = f.y; buf[4 * v + 2] = f.z; buf[4 * v + 3] = f.w;
                    }
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) {
                        float a_ = Bk[0] * buf[ch];
#pragma unroll
                        for (int k = 1; k < K; ++k) a_ = a_ + Bk[k] * buf[3 * k + ch];
                        acc[ch] = a_;
                    }
                } else {
#pragma unroll
                    for (int ch = 0; ch < 3; ++ch) {
                        float a_ = Bk[0] * __ldg(s_i + ch);
#pragma unroll
                        for (int k = 1; k < K; ++k) a_ = a_ + Bk[k] * __ldg(s_i + 3 * k + ch);
                        acc[ch] = a_;
                    }
                }
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    acc[ch] = acc[ch] + 0.5f;
                    if (acc[ch] < 0.0f) { acc[ch] = 0.0f; cl |= (uint8_t)(1u << ch); }
                }
                r0 = make_float4(mx, my, A, B);
                r1 = make_float4(C, op[i], acc[0], acc[1]);
                r2 = make_float4(acc[2], tz, __uint_as_float((uint32_t)x0 | ((uint32_t)x1 << 16)),
                                 __uint_as_float((uint32_t)y0 | ((uint32_t)y1 << 16)));
                rad_out = (int)rad;
            }
        }
    }
    splats[3 * (size_t)i] = r0;
    splats[3 * (size_t)i + 1] = r1;
    splats[3 * (size_t)i + 2] = r2;
    radii[i] = rad_out;
    clamped[i] = cl;
}

}  // namespace

cudaError_t launch_preprocess(const CamK& cam, int N, int D, const float* mu, const float* sc, const float* qt,
                              const float* op, const float* sh, float* splats, int32_t* radii,
                              uint8_t* clamped, cudaStream_t s) {
    const int threads = 128;
    const int blocks = (N + threads - 1) / threads;
    float4* sp = reinterpret_cast<float4*>(splats);
    switch (D) {
        case 0: preprocess_kernel<0><<<blocks, threads, 0, s>>>(cam, N, mu, sc, qt, op, sh, sp, radii, clamped); break;
        case 1: preprocess_kernel<1><<<blocks, threads, 0, s>>>(cam, N, mu, sc, qt, op, sh, sp, radii, clamped); break;
        case 2: preprocess_kernel<2><<<blocks, threads, 0, s>>>(cam, N, mu, sc, qt, op, sh, sp, radii, clamped); break;
        default: preprocess_kernel<3><<<blocks, threads, 0, s>>>(cam, N, mu, sc, qt, op, sh, sp, radii, clamped); break;
    }
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
