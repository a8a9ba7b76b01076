// tgs_raster_bwd_sparse, projection half: chains dL/d(mean2D, conic, opacity, rgb) of every
// Gaussian through the EWA projection and the SH colour to dL/d(mean3D, scale, quaternion,
// opacity, SH) ("This pipeline is differentiable", 441).
// One thread per Gaussian, no atomics; HBM-bound (reads 236 + 48 + 20 B, writes 236 B at degree 3).
// A Gaussian whose raster gradient record is all zero (not listed in any sampled tile, or listed with a zero
// gradient) has a zero result -- the chain is linear in that record: only its 48-byte record is read, nothing else,
// and (SPARSE, `touched` given) nothing is written but touched[i] = 0; without `touched` its rows are written as
// zeros.  With 5 % of the tiles sampled that is 85 % of the Gaussians.
// The SH block (192 B in, 192 B out per Gaussian -- three quarters of the traffic) moves through
// shared memory: the block's 128 x K x 3 coefficients are one contiguous span in HBM, copied with
// coalesced float4 accesses into rows of odd stride (conflict-free for one-row-per-thread access),
// overwritten in place by dL/dsh and copied back the same way.
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

// basis values B[k] and their gradients dB[k][0..2] w.r.t. the direction components
template <int D>
__device__ __forceinline__ void sh_basis_and_grad(float x, float y, float z, float* B, float (*dB)[3]) {
    constexpr int K = (D + 1) * (D + 1);
#pragma unroll
    for (int k = 0; k < K; ++k) { dB[k][0] = 0.f; dB[k][1] = 0.f; dB[k][2] = 0.f; }
    B[0] = SH_C0;
    if (D >= 1) {
        B[1] = -SH_C1 * y; dB[1][1] = -SH_C1;
        B[2] = SH_C1 * z;  dB[2][2] = SH_C1;
        B[3] = -SH_C1 * x; dB[3][0] = -SH_C1;
    }
    if (D >= 2) {
        const float xx = x * x, yy = y * y, zz = z * z;
        B[4] = SH_C2A * x * y;  dB[4][0] = SH_C2A * y;  dB[4][1] = SH_C2A * x;
        B[5] = -SH_C2A * y * z; dB[5][1] = -SH_C2A * z; dB[5][2] = -SH_C2A * y;
        B[6] = SH_C2B * (2.f * zz - xx - yy);
        dB[6][0] = -2.f * SH_C2B * x; dB[6][1] = -2.f * SH_C2B * y; dB[6][2] = 4.f * SH_C2B * z;
        B[7] = -SH_C2A * x * z; dB[7][0] = -SH_C2A * z; dB[7][2] = -SH_C2A * x;
        B[8] = SH_C2C * (xx - yy); dB[8][0] = 2.f * SH_C2C * x; dB[8][1] = -2.f * SH_C2C * y;
        if (D >= 3) {
            B[9] = -SH_C3A * y * (3.f * xx - yy);
            dB[9][0] = -6.f * SH_C3A * x * y; dB[9][1] = -3.f * SH_C3A * (xx - yy);
            B[10] = SH_C3B * x * y * z;
            dB[10][0] = SH_C3B * y * z; dB[10][1] = SH_C3B * x * z; dB[10][2] = SH_C3B * x * y;
            B[11] = -SH_C3C * y * (4.f * zz - xx - yy);
            dB[11][0] = 2.f * SH_C3C * x * y; dB[11][1] = -SH_C3C * (4.f * zz - xx - 3.f * yy);
            dB[11][2] = -8.f * SH_C3C * y * z;
            B[12] = SH_C3D * z * (2.f * zz - 3.f * xx - 3.f * yy);
            dB[12][0] = -6.f * SH_C3D * x * z; dB[12][1] = -6.f * SH_C3D * y * z;
            dB[12][2] = 3.f * SH_C3D * (2.f * zz - xx - yy);
            B[13] = -SH_C3C * x * (4.f * zz - xx - yy);
            dB[13][0] = -SH_C3C * (4.f * zz - 3.f * xx - yy); dB[13][1] = 2.f * SH_C3C * x * y;
            dB[13][2] = -8.f * SH_C3C * x * z;
            B[14] = SH_C3E * z * (xx - yy);
            dB[14][0] = 2.f * SH_C3E * x * z; dB[14][1] = -2.f * SH_C3E * y * z; dB[14][2] = SH_C3E * (xx - yy);
            B[15] = -SH_C3A * x * (xx - 3.f * yy);
            dB[15][0] = -3.f * SH_C3A * (xx - yy); dB[15][1] = 6.f * SH_C3A * x * y;
        }
    }
}

constexpr int kPBThreads = 128;

template <int D, bool SPARSE>
__global__ void __launch_bounds__(kPBThreads)
project_bwd_kernel(const CamK cam, int N, const float* __restrict__ mu, const float* __restrict__ sc,
                   const float* __restrict__ qt, const float* __restrict__ sh, const int32_t* __restrict__ radii,
                   const uint8_t* __restrict__ clamped, const float4* __restrict__ spl, const float4* __restrict__ dsp,
                   float* __restrict__ dmu, float* __restrict__ dsc, float* __restrict__ dqt,
                   float* __restrict__ dop, float* __restrict__ dsh, int32_t* __restrict__ touched) {
    constexpr int K = (D + 1) * (D + 1);
    constexpr int KC = K * 3;                       // floats per Gaussian
    constexpr int STRIDE = (KC % 2) ? KC : KC + 1;  // odd row stride: lane i -> bank (STRIDE * i + j) % 32, all distinct
    __shared__ float s_sh[kPBThreads * STRIDE];
    __shared__ unsigned char s_on[kPBThreads];
    const int base = blockIdx.x * kPBThreads;
    const int nvalid = min(kPBThreads, N - base);
    const int i = base + threadIdx.x;
    // the raster gradient record decides whether this Gaussian has anything to chain
    float4 d0 = make_float4(0.f, 0.f, 0.f, 0.f), d1 = d0, d2 = d0;
    bool on = false;
    if (i < N && radii[i] > 0) {
        d0 = dsp[3 * (size_t)i]; d1 = dsp[3 * (size_t)i + 1]; d2 = dsp[3 * (size_t)i + 2];
        on = d0.x != 0.f || d0.y != 0.f || d0.z != 0.f || d0.w != 0.f || d1.x != 0.f || d1.y != 0.f || d1.z != 0.f ||
             d1.w != 0.f || d2.x != 0.f;
    }
    s_on[threadIdx.x] = on;
    if (!__syncthreads_or(on)) {   // nothing to chain in this block of 128 Gaussians
        if (i < N) {
            if (SPARSE) { touched[i] = 0; return; }
            dmu[3 * i] = 0.f; dmu[3 * i + 1] = 0.f; dmu[3 * i + 2] = 0.f;
            dsc[3 * i] = 0.f; dsc[3 * i + 1] = 0.f; dsc[3 * i + 2] = 0.f;
            reinterpret_cast<float4*>(dqt)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
            dop[i] = 0.f;
        }
        if (!SPARSE) {
            const int total = nvalid * KC;
            float* dst = dsh + (size_t)base * KC;
            float4* dst4 = reinterpret_cast<float4*>(dst);
            for (int v = threadIdx.x; v < total / 4; v += kPBThreads) dst4[v] = make_float4(0.f, 0.f, 0.f, 0.f);
            for (int e = (total / 4) * 4 + threadIdx.x; e < total; e += kPBThreads) dst[e] = 0.f;
        }
        return;
    }
    {   // coalesced copy in of the rows that are needed: float4 body (the span starts 16-byte aligned), scalar tail
        const int total = nvalid * KC;
        const float* src = sh + (size_t)base * KC;
        const float4* src4 = reinterpret_cast<const float4*>(src);
        for (int v = threadIdx.x; v < total / 4; v += kPBThreads) {
            const int e = 4 * v;
            if (!(s_on[e / KC] | s_on[(e + 3) / KC])) continue;
            const float4 f = __ldg(src4 + v);
            const float vals[4] = {f.x, f.y, f.z, f.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) s_sh[((e + c) / KC) * STRIDE + (e + c) % KC] = vals[c];
        }
        for (int e = (total / 4) * 4 + threadIdx.x; e < total; e += kPBThreads)
            if (s_on[e / KC]) s_sh[(e / KC) * STRIDE + e % KC] = __ldg(src + e);
    }
    __syncthreads();
    if (i < N) {
    float gmu[3] = {0.f, 0.f, 0.f}, gs[3] = {0.f, 0.f, 0.f}, gq[4] = {0.f, 0.f, 0.f, 0.f}, gop = 0.f;
    float* gsh = s_sh + threadIdx.x * STRIDE;  // SH in, dL/dsh out (in place)
    bool live = on;
    const float* W = cam.R;
    float m0 = 0.f, m1 = 0.f, m2 = 0.f, t0 = 0.f, t1 = 0.f, tz = 1.f;
    if (live) {
        m0 = mu[3 * i]; m1 = mu[3 * i + 1]; m2 = mu[3 * i + 2];
        t0 = W[0] * m0 + W[1] * m1 + W[2] * m2 + cam.t[0];
        t1 = W[3] * m0 + W[4] * m1 + W[5] * m2 + cam.t[1];
        tz = W[6] * m0 + W[7] * m1 + W[8] * m2 + cam.t[2];
        live = tz > cam.znear;
    }
    if (!live) {
        if (!SPARSE) {
#pragma unroll
            for (int e = 0; e < K * 3; ++e) gsh[e] = 0.f;
        }
    } else {
        const float4 f0 = spl[3 * (size_t)i];
        const float A = f0.z, B = f0.w, C = spl[3 * (size_t)i + 1].x;  // the forward's conic
        const float gmx = d0.x, gmy = d0.y, gA = d0.z, gB = d0.w, gC = d1.x;
        gop = d1.y;
        const float grgb[3] = {d1.z, d1.w, d2.x};
        // ---- forward intermediates ----
        const float limx = kJClamp * ((0.5f * (float)cam.W) / cam.fx);
        const float limy = kJClamp * ((0.5f * (float)cam.H) / cam.fy);
        const float txtz = t0 / tz, tytz = t1 / tz;
        float cxr = txtz, cyr = tytz;
        int clx = 0, cly = 0;
        if (cxr > limx) { cxr = limx; clx = 1; } else if (cxr < -limx) { cxr = -limx; clx = -1; }
        if (cyr > limy) { cyr = limy; cly = 1; } else if (cyr < -limy) { cyr = -limy; cly = -1; }
        const float tz2 = tz * tz, itz = 1.0f / tz, itz2 = 1.0f / tz2;
        const float J00 = cam.fx * itz, J02 = -(cam.fx * cxr * tz) * itz2;
        const float J11 = cam.fy * itz, J12 = -(cam.fy * cyr * tz) * itz2;
        float Tm[6];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            Tm[c] = J00 * W[c] + J02 * W[6 + c];
            Tm[3 + c] = J11 * W[3 + c] + J12 * W[6 + c];
        }
        const float4 q = reinterpret_cast<const float4*>(qt)[i];
        const float w = q.x, x = q.y, y = q.z, z = q.w;
        float Rq[9];
        Rq[0] = 1.f - 2.f * (y * y + z * z); Rq[1] = 2.f * (x * y - w * z); Rq[2] = 2.f * (x * z + w * y);
        Rq[3] = 2.f * (x * y + w * z); Rq[4] = 1.f - 2.f * (x * x + z * z); Rq[5] = 2.f * (y * z - w * x);
        Rq[6] = 2.f * (x * z - w * y); Rq[7] = 2.f * (y * z + w * x); Rq[8] = 1.f - 2.f * (x * x + y * y);
        const float s[3] = {sc[3 * i], sc[3 * i + 1], sc[3 * i + 2]};
        // The conic (A, B, C) is the forward's own (splat record words 2..4).  With Sigma' = sum_k s_k^2 v_k v_k^T + 0.3 I,
        // v_k = Tm R_k the projected k-th axis, everything downstream of dL/dSigma' = H = -M Ghat M (M = conic,
        // Ghat = [[gA, gB/2], [gB/2, gC]]) only needs H v_k.  It is formed axis by axis as
        //     y_k = M v_k,  w_k = Ghat y_k,  z_k = M w_k = -H v_k
        // and H itself never: for a needle (condition number kappa of Sigma' large) the entries of H are ~kappa^2 larger
        // than v^T H v along the long axis, so a gradient formed from H cancels kappa^2 of fp32 rounding; y_k = M v_k
        // cancels only kappa, the sensitivity the 2x2 inverse has anyway.
        //     dL/ds_k     = 2 s_k v_k^T H v_k            = -2 s_k (y_k . w_k)
        //     dL/dM[:,k]  = 2 s_k Tm^T H v_k             = -2 s_k Tm^T z_k        (M = R diag(s), Sigma = M M^T)
        //     dL/dTm      = 2 H Tm Sigma = 2 sum_k s_k^2 (H v_k) R_k^T = -2 sum_k s_k^2 z_k R_k^T
        const float hB = 0.5f * gB;
        float dR[9], dTm[6] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const float v0 = Tm[0] * Rq[k] + Tm[1] * Rq[3 + k] + Tm[2] * Rq[6 + k];
            const float v1 = Tm[3] * Rq[k] + Tm[4] * Rq[3 + k] + Tm[5] * Rq[6 + k];
            const float y0 = A * v0 + B * v1, y1 = B * v0 + C * v1;
            const float w0 = gA * y0 + hB * y1, w1 = hB * y0 + gC * y1;
            const float z0 = A * w0 + B * w1, z1 = B * w0 + C * w1;
            gs[k] = -2.f * s[k] * (y0 * w0 + y1 * w1);
            const float m2s2 = -2.f * s[k] * s[k];
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                dR[3 * r + k] = m2s2 * (Tm[r] * z0 + Tm[3 + r] * z1);  // dL/dM[r][k] * s_k
                dTm[r] = fmaf(m2s2 * z0, Rq[3 * r + k], dTm[r]);
                dTm[3 + r] = fmaf(m2s2 * z1, Rq[3 * r + k], dTm[3 + r]);
            }
        }
        const float dJ00 = dTm[0] * W[0] + dTm[1] * W[1] + dTm[2] * W[2];
        const float dJ02 = dTm[0] * W[6] + dTm[1] * W[7] + dTm[2] * W[8];
        const float dJ11 = dTm[3] * W[3] + dTm[4] * W[4] + dTm[5] * W[5];
        const float dJ12 = dTm[3] * W[6] + dTm[4] * W[7] + dTm[5] * W[8];
        float dt0 = 0.f, dt1 = 0.f, dt2 = 0.f;
        dt2 += -(cam.fx * itz2) * dJ00 - (cam.fy * itz2) * dJ11;
        if (clx == 0) { dt0 += -(cam.fx * itz2) * dJ02; dt2 += (2.f * cam.fx * t0 * itz2 * itz) * dJ02; }
        else dt2 += ((float)clx * cam.fx * limx * itz2) * dJ02;
        if (cly == 0) { dt1 += -(cam.fy * itz2) * dJ12; dt2 += (2.f * cam.fy * t1 * itz2 * itz) * dJ12; }
        else dt2 += ((float)cly * cam.fy * limy * itz2) * dJ12;
        dt0 += gmx * cam.fx * itz;
        dt1 += gmy * cam.fy * itz;
        dt2 += -gmx * cam.fx * t0 * itz2 - gmy * cam.fy * t1 * itz2;
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) gmu[cc] = W[cc] * dt0 + W[3 + cc] * dt1 + W[6 + cc] * dt2;
        gq[0] = 2.f * (z * (dR[3] - dR[1]) + y * (dR[2] - dR[6]) + x * (dR[7] - dR[5]));
        gq[1] = 2.f * (y * (dR[1] + dR[3]) + z * (dR[2] + dR[6]) + w * (dR[7] - dR[5])) - 4.f * x * (dR[4] + dR[8]);
        gq[2] = 2.f * (x * (dR[1] + dR[3]) + w * (dR[2] - dR[6]) + z * (dR[5] + dR[7])) - 4.f * y * (dR[0] + dR[8]);
        gq[3] = 2.f * (w * (dR[3] - dR[1]) + x * (dR[2] + dR[6]) + y * (dR[5] + dR[7])) - 4.f * z * (dR[0] + dR[4]);
        // ---- colour ----
        const float o0 = -(W[0] * cam.t[0] + W[3] * cam.t[1] + W[6] * cam.t[2]);
        const float o1 = -(W[1] * cam.t[0] + W[4] * cam.t[1] + W[7] * cam.t[2]);
        const float o2 = -(W[2] * cam.t[0] + W[5] * cam.t[1] + W[8] * cam.t[2]);
        const float v0 = m0 - o0, v1 = m1 - o1, v2 = m2 - o2;
        const float len = sqrtf(v0 * v0 + v1 * v1 + v2 * v2), ilen = 1.0f / len;
        const float d[3] = {v0 * ilen, v1 * ilen, v2 * ilen};
        float Bk[K], dB[K][3];
        sh_basis_and_grad<D>(d[0], d[1], d[2], Bk, dB);
        const uint8_t cl = clamped[i];
        float gch[3];
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) gch[ch] = (cl & (1u << ch)) ? 0.f : grgb[ch];
        float dd[3] = {0.f, 0.f, 0.f};
#pragma unroll
        for (int k = 0; k < K; ++k) {
#pragma unroll
            for (int ch = 0; ch < 3; ++ch) {
                const float sv = gsh[3 * k + ch] * gch[ch];
                gsh[3 * k + ch] = Bk[k] * gch[ch];
                dd[0] = fmaf(dB[k][0], sv, dd[0]); dd[1] = fmaf(dB[k][1], sv, dd[1]); dd[2] = fmaf(dB[k][2], sv, dd[2]);
            }
        }
        const float dot = d[0] * dd[0] + d[1] * dd[1] + d[2] * dd[2];
#pragma unroll
        for (int cc = 0; cc < 3; ++cc) gmu[cc] += (dd[cc] - d[cc] * dot) * ilen;
    }
    // (a Gaussian with a record but behind znear cannot occur: radii > 0 implies t_z > znear; if it did, `live`
    // is false here and its rows are zeros / untouched like any other)
    if (SPARSE) touched[i] = live ? 1 : 0;
    if (!SPARSE || live) {
        dmu[3 * i] = gmu[0]; dmu[3 * i + 1] = gmu[1]; dmu[3 * i + 2] = gmu[2];
        dsc[3 * i] = gs[0]; dsc[3 * i + 1] = gs[1]; dsc[3 * i + 2] = gs[2];
        reinterpret_cast<float4*>(dqt)[i] = make_float4(gq[0], gq[1], gq[2], gq[3]);
        dop[i] = gop;
    }
    if (SPARSE) s_on[threadIdx.x] = live;
    }
    __syncthreads();
    {   // coalesced copy out (SPARSE: of the chained rows only; a float4 that straddles two rows is written by parts)
        const int total = nvalid * KC;
        float* dst = dsh + (size_t)base * KC;
        float4* dst4 = reinterpret_cast<float4*>(dst);
        for (int v = threadIdx.x; v < total / 4; v += kPBThreads) {
            const int e = 4 * v;
            float vals[4];
#pragma unroll
            for (int c = 0; c < 4; ++c) vals[c] = s_sh[((e + c) / KC) * STRIDE + (e + c) % KC];
            if (!SPARSE) {
                dst4[v] = make_float4(vals[0], vals[1], vals[2], vals[3]);
            } else {
                const bool a = s_on[e / KC], b = s_on[(e + 3) / KC];
                if (a & b) dst4[v] = make_float4(vals[0], vals[1], vals[2], vals[3]);
                else if (a | b) {
#pragma unroll
                    for (int c = 0; c < 4; ++c) if (s_on[(e + c) / KC]) dst[e + c] = vals[c];
                }
            }
        }
        for (int e = (total / 4) * 4 + threadIdx.x; e < total; e += kPBThreads)
            if (!SPARSE || s_on[e / KC]) dst[e] = s_sh[(e / KC) * STRIDE + e % KC];
    }
}

}  // namespace

cudaError_t launch_project_bwd(const CamK& cam, int N, int D, const float* mu, const float* sc, const float* qt,
                               const float* sh, const int32_t* radii, const uint8_t* clamped, const float* splats,
                               const float* dL_dsplats, float* dmu, float* dsc, float* dqt, float* dop,
                               float* dsh, int32_t* touched, cudaStream_t s) {
    const int threads = kPBThreads, blocks = (N + threads - 1) / threads;
    const float4* dsp = reinterpret_cast<const float4*>(dL_dsplats);
    const float4* spl = reinterpret_cast<const float4*>(splats);
#define TGS_PB(DD)                                                                                                          \
    if (touched) project_bwd_kernel<DD, true><<<blocks, threads, 0, s>>>(cam, N, mu, sc, qt, sh, radii, clamped, spl, dsp, dmu, dsc, dqt, dop, dsh, touched); \
    else project_bwd_kernel<DD, false><<<blocks, threads, 0, s>>>(cam, N, mu, sc, qt, sh, radii, clamped, spl, dsp, dmu, dsc, dqt, dop, dsh, touched)
    switch (D) {
        case 0: TGS_PB(0); break;
        case 1: TGS_PB(1); break;
        case 2: TGS_PB(2); break;
        default: TGS_PB(3); break;
    }
#undef TGS_PB
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
