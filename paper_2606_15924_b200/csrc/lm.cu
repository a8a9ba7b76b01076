// f4: the moment-damped LM solve, PAPER.md:231-239 (Eq. 14), 483-490 (Eq. 19), Alg. 1 steps 9-10.
//
// Two kernels, split by the ARRAYS they touch (the paper also uses two):
//   lm_geo_kernel     the geometry block (position, scale, rotation; 10 x 10): one thread per Gaussian, the lower
//                     triangle of J^T J + diag(sqrt(v) + eps) in 55 fp64 registers, Cholesky by rsqrt (no division).
//                     Reads / writes means3D, scales, quats only.
//   lm_app_sh_kernel  everything that lives in sh[] and opacities[]: thread i of a block of 128 solves the appearance
//                     block (RGB DC + opacity; 4 x 4, fp64 registers) of Gaussian 128 b + i, and the block's
//                     128 K 3 floats of the SH arrays are swept with coalesced 16-byte accesses for the Adam branch
//                     (fp32).  The two parts touch disjoint elements (the DC band sh[:,0,:] belongs to the
//                     appearance block): no barrier, no shared memory; having them in ONE kernel keeps the 32-byte
//                     sectors that hold a Gaussian's DC term (12 B of 192) in L1 / L2 between their two uses, so the
//                     DRAM traffic stays the algorithmic (V + 2) x 236 B read + (2 + outputs) x 236 B written per
//                     Gaussian (ncu: 5.64 GB against 5.66 GB at N = 3 M, V = 3).
// HBM bound; a first version with both blocks and the sweep in one kernel ran at 168 registers / 12 warps per SM and
// 2.4 TB/s -- the 10 x 10 block's registers starved the sweep of loads in flight.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kLmThreads = 128;

// In-register Cholesky solve of (A + diag(sqrt(vb) + eps)) x = -mb for one SPD system of size D, A = J^T J given
// as its lower triangle (row major, idx(i, j) = i (i + 1) / 2 + j).  Every loop has constant bounds and is fully
// unrolled, so A, inv and x live in registers.  inv[j] = 1 / L_jj comes from rsqrt: no division, no sqrt of the pivot.
template <int D>
__device__ __forceinline__ void chol_solve(double (&A)[D * (D + 1) / 2], const double (&vb)[D], const double (&mb)[D],
                                           double eps, double (&x)[D]) {
    double inv[D];
#pragma unroll
    for (int i = 0; i < D; ++i) A[i * (i + 1) / 2 + i] += sqrt(vb[i]) + eps;
#pragma unroll
    for (int j = 0; j < D; ++j) {
        double s = A[j * (j + 1) / 2 + j];
#pragma unroll
        for (int k = 0; k < j; ++k) s = fma(-A[j * (j + 1) / 2 + k], A[j * (j + 1) / 2 + k], s);
        inv[j] = rsqrt(s);
#pragma unroll
        for (int i = j + 1; i < D; ++i) {
            double r = A[i * (i + 1) / 2 + j];
#pragma unroll
            for (int k = 0; k < j; ++k) r = fma(-A[i * (i + 1) / 2 + k], A[j * (j + 1) / 2 + k], r);
            A[i * (i + 1) / 2 + j] = r * inv[j];
        }
    }
    // L y = -m, then L^T x = y
#pragma unroll
    for (int i = 0; i < D; ++i) {
        double s = -mb[i];
#pragma unroll
        for (int k = 0; k < i; ++k) s = fma(-A[i * (i + 1) / 2 + k], x[k], s);
        x[i] = s * inv[i];
    }
#pragma unroll
    for (int i = D - 1; i >= 0; --i) {
        double s = x[i];
#pragma unroll
        for (int k = i + 1; k < D; ++k) s = fma(-A[k * (k + 1) / 2 + i], x[k], s);
        x[i] = s * inv[i];
    }
}

// One LM block of one Gaussian.  off[c] / ptr selection is done by the caller through the small accessor below:
// element c of the block lives at base(c)[n * stride(c) + sub(c)] of a parameter set.
template <int D, int kViewBatch, bool VT, class Acc>
__device__ __forceinline__ void lm_block(const LmArgs& a, const Acc acc, int n, unsigned long long views) {
    double A[D * (D + 1) / 2];
    double gb[D];
#pragma unroll
    for (int i = 0; i < D * (D + 1) / 2; ++i) A[i] = 0.0;
#pragma unroll
    for (int c = 0; c < D; ++c) gb[c] = 0.0;
    // the moments' loads are issued before the views' so that one latency covers both
    float m0[D], v0[D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        m0[c] = acc.ptr(a.m, c)[acc.off(c, n)];
        v0[c] = acc.ptr(a.v, c)[acc.off(c, n)];
    }
    // views in batches of kViewBatch: all loads of a batch are in flight before the first is consumed
    for (int vw0 = 0; vw0 < a.V; vw0 += kViewBatch) {
        float gf[kViewBatch][D];
#pragma unroll
        for (int u = 0; u < kViewBatch; ++u)
#pragma unroll
            for (int c = 0; c < D; ++c)
                gf[u][c] = (vw0 + u < a.V && (!VT || ((views >> (vw0 + u)) & 1ull)))
                               ? __ldg(acc.view(a.g, c, vw0 + u, a.N) + acc.off(c, n)) : 0.f;
#pragma unroll
        for (int u = 0; u < kViewBatch; ++u) {
            if (vw0 + u >= a.V) break;
            double g[D];
#pragma unroll
            for (int c = 0; c < D; ++c) { g[c] = (double)gf[u][c]; gb[c] += g[c]; }
#pragma unroll
            for (int i = 0; i < D; ++i)
#pragma unroll
                for (int j = 0; j <= i; ++j) A[i * (i + 1) / 2 + j] = fma(g[i], g[j], A[i * (i + 1) / 2 + j]);
        }
    }
    double mb[D], vb[D], x[D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        mb[c] = a.b1 * (double)m0[c] + (1.0 - a.b1) * gb[c];
        vb[c] = a.b2 * (double)v0[c] + (1.0 - a.b2) * gb[c] * gb[c];
        acc.ptr(a.m, c)[acc.off(c, n)] = (float)mb[c];
        acc.ptr(a.v, c)[acc.off(c, n)] = (float)vb[c];
    }
    chol_solve<D>(A, vb, mb, a.eps, x);
#pragma unroll
    for (int c = 0; c < D; ++c) {
        const float dx = (float)x[c];
        if (a.d.mu) acc.ptr(a.d, c)[acc.off(c, n)] = dx;
        if (a.p.mu) { float* pp = acc.ptr(a.p, c) + acc.off(c, n); *pp = (float)((double)*pp + x[c]); }
    }
}

struct GeoAcc {  // (position 3, scale 3, rotation 4)
    __device__ __forceinline__ float* ptr(const LmSet& s, int c) const { return c < 3 ? s.mu : (c < 6 ? s.sc : s.qt); }
    __device__ __forceinline__ const float* view(const LmSet& s, int c, int vw, int N) const {
        return c < 3 ? s.mu + (size_t)vw * N * 3 : (c < 6 ? s.sc + (size_t)vw * N * 3 : s.qt + (size_t)vw * N * 4);
    }
    __device__ __forceinline__ size_t off(int c, int n) const {
        return c < 3 ? (size_t)n * 3 + c : (c < 6 ? (size_t)n * 3 + (c - 3) : (size_t)n * 4 + (c - 6));
    }
};
struct AppAcc {  // (RGB DC 3, opacity 1)
    int K;
    __device__ __forceinline__ float* ptr(const LmSet& s, int c) const { return c < 3 ? s.sh : s.op; }
    __device__ __forceinline__ const float* view(const LmSet& s, int c, int vw, int N) const {
        return c < 3 ? s.sh + (size_t)vw * N * K * 3 : s.op + (size_t)vw * N;
    }
    __device__ __forceinline__ size_t off(int c, int n) const { return c < 3 ? (size_t)n * K * 3 + c : (size_t)n; }
};

// Adam branch of Eq. 19 for one coefficient, in fp32 (the storage precision; IEEE sqrt and division).
__device__ __forceinline__ void adam_one(const LmArgs& a, float gbar, float& m, float& v, float& dlt) {
    m = fmaf(a.b1f, m, a.omb1f * gbar);
    v = fmaf(a.b2f, v, (a.omb2f * gbar) * gbar);
    const float mh = m * a.ibc1f;
    const float vh = v * a.ibc2f;
    dlt = -a.eta * mh / (sqrtf(vh) + a.epsf);
}

// VEC = 4: K * 3 is a multiple of 4 (degrees 1 and 3) and the block's span is swept with float4 accesses;
// VEC = 1: degree 2 (27 floats per Gaussian), scalar accesses.
template <int VEC> struct Vec;
template <> struct Vec<4> { using T = float4; };
template <> struct Vec<1> { using T = float; };
__device__ __forceinline__ float comp(const float4& q, int i) { return i == 0 ? q.x : (i == 1 ? q.y : (i == 2 ? q.z : q.w)); }
__device__ __forceinline__ float comp(const float& q, int) { return q; }
__device__ __forceinline__ float& comp(float4& q, int i) { return i == 0 ? q.x : (i == 1 ? q.y : (i == 2 ? q.z : q.w)); }
__device__ __forceinline__ float& comp(float& q, int) { return q; }

template <int VEC, int kViewBatch, int kSpanBatch, int MINB, bool VT>
__global__ void __launch_bounds__(kLmThreads, MINB) lm_app_sh_kernel(const LmArgs a) {
    using T = typename Vec<VEC>::T;
    const int n = blockIdx.x * kLmThreads + threadIdx.x;
    // ---- Adam branch over the block's span of the SH arrays (coalesced; skips the DC band) ----
    const int row = a.K * 3;                        // floats per Gaussian
    if (a.K > 1) {
        const size_t span0 = (size_t)blockIdx.x * kLmThreads * row;
        const size_t total = (size_t)a.N * row;     // also the distance between two views of grads.sh
        const int per_block = kLmThreads * row / VEC;
        for (int j0 = threadIdx.x; j0 < per_block; j0 += kSpanBatch * kLmThreads) {
            size_t e[kSpanBatch];
            bool ok[kSpanBatch], on[kSpanBatch];
            int r[kSpanBatch];
            unsigned long long views[kSpanBatch];
            T m4[kSpanBatch], v4[kSpanBatch];
            float gs[kSpanBatch][VEC];
#pragma unroll
            for (int u = 0; u < kSpanBatch; ++u) {
                const int j = j0 + u * kLmThreads;
                e[u] = span0 + (size_t)j * VEC;
                ok[u] = j < per_block && e[u] < total;
                const int gn = ok[u] ? (int)(e[u] / row) : 0;
                r[u] = (int)(e[u] - (size_t)gn * row);   // first element's position inside the Gaussian's row
                views[u] = ok[u] ? lm_views<VT>(a, gn) : 0ull;
                on[u] = views[u] != 0ull;
                if (VEC == 1 && r[u] < 3) on[u] = ok[u] = false;   // DC band: appearance block
#pragma unroll
                for (int i = 0; i < VEC; ++i) gs[u][i] = 0.f;
            }
#pragma unroll
            for (int u = 0; u < kSpanBatch; ++u)
                if (on[u]) {
                    m4[u] = *reinterpret_cast<const T*>(a.m.sh + e[u]);
                    v4[u] = *reinterpret_cast<const T*>(a.v.sh + e[u]);
                }
            for (int vw0 = 0; vw0 < a.V; vw0 += kViewBatch) {
                T g4[kViewBatch][kSpanBatch];
#pragma unroll
                for (int w = 0; w < kViewBatch; ++w)
#pragma unroll
                    for (int u = 0; u < kSpanBatch; ++u)
                        if (on[u] && vw0 + w < a.V && (!VT || ((views[u] >> (vw0 + w)) & 1ull)))
                            g4[w][u] = __ldg(reinterpret_cast<const T*>(a.g.sh + (size_t)(vw0 + w) * total + e[u]));
                        else if (VT)
                            g4[w][u] = T{};
#pragma unroll
                for (int w = 0; w < kViewBatch; ++w)
#pragma unroll
                    for (int u = 0; u < kSpanBatch; ++u)
                        if (on[u] && vw0 + w < a.V) {
#pragma unroll
                            for (int i = 0; i < VEC; ++i) gs[u][i] += comp(g4[w][u], i);
                        }
            }
#pragma unroll
            for (int u = 0; u < kSpanBatch; ++u) {
                if (!ok[u]) continue;
                const bool dc = VEC == 4 && r[u] == 0;   // x y z of this vector are the DC band: only .w is an Adam coefficient
                T d4;
#pragma unroll
                for (int i = 0; i < VEC; ++i) comp(d4, i) = 0.f;
                if (on[u]) {
#pragma unroll
                    for (int i = 0; i < VEC; ++i)
                        if (!(dc && i < 3)) adam_one(a, gs[u][i], comp(m4[u], i), comp(v4[u], i), comp(d4, i));
                    if (dc) {
                        a.m.sh[e[u] + 3] = comp(m4[u], 3);
                        a.v.sh[e[u] + 3] = comp(v4[u], 3);
                        if (a.p.mu) a.p.sh[e[u] + 3] += comp(d4, 3);
                    } else {
                        *reinterpret_cast<T*>(a.m.sh + e[u]) = m4[u];
                        *reinterpret_cast<T*>(a.v.sh + e[u]) = v4[u];
                        if (a.p.mu) {
                            T p4 = *reinterpret_cast<const T*>(a.p.sh + e[u]);
#pragma unroll
                            for (int i = 0; i < VEC; ++i) comp(p4, i) += comp(d4, i);
                            *reinterpret_cast<T*>(a.p.sh + e[u]) = p4;
                        }
                    }
                }
                if (a.d.mu) {
                    if (dc) a.d.sh[e[u] + 3] = comp(d4, 3);
                    else *reinterpret_cast<T*>(a.d.sh + e[u]) = d4;
                }
            }
        }
    }
    // ---- the appearance block of Gaussian n (Eq. 14): RGB DC + opacity ----
    if (n >= a.N) return;
    const unsigned long long nviews = lm_views<VT>(a, n);
    if (nviews == 0ull) {
        if (a.d.mu) {
            const AppAcc aa{a.K};
#pragma unroll
            for (int c = 0; c < 4; ++c) aa.ptr(a.d, c)[aa.off(c, n)] = 0.f;
        }
        return;
    }
    lm_block<4, kViewBatch, VT>(a, AppAcc{a.K}, n, nviews);
}

// The geometry block (position, scale, rotation) of Eq. 14: one thread per Gaussian, the 55 entries of the lower
// triangle in fp64 registers.  Touches means3D / scales / quats only, so it runs beside lm_app_sh_kernel.
template <int kViewBatch, int MINB, bool VT>
__global__ void __launch_bounds__(kLmThreads, MINB) lm_geo_kernel(const LmArgs a) {
    const int n = blockIdx.x * kLmThreads + threadIdx.x;
    if (n >= a.N) return;
    const unsigned long long nviews = lm_views<VT>(a, n);
    if (nviews == 0ull) {
        if (a.d.mu) {
            const GeoAcc ga;
#pragma unroll
            for (int c = 0; c < 10; ++c) ga.ptr(a.d, c)[ga.off(c, n)] = 0.f;
        }
        return;
    }
    lm_block<10, kViewBatch, VT>(a, GeoAcc(), n, nviews);
}

}  // namespace

cudaError_t launch_lm_solve(const LmArgs& a, cudaStream_t s) {
    if (a.N <= 0) return cudaSuccess;
    const int blocks = (a.N + kLmThreads - 1) / kLmThreads;
    // batching measured on B200 at N = 3 M, V = 3 (profiles/r2_lm.md): geometry 4 views per batch at 2 blocks / SM
    // (248 registers), SH sweep 4 pieces of the span per thread, one view at a time (109 registers, 4 blocks / SM)
    // (the per-view masks are a template flag: with them as a run-time test the unmasked call ran 40 % slower)
    if (a.vt) {
        lm_geo_kernel<4, 2, true><<<blocks, kLmThreads, 0, s>>>(a);
        if ((a.K * 3) % 4 == 0) lm_app_sh_kernel<4, 1, 4, 1, true><<<blocks, kLmThreads, 0, s>>>(a);
        else lm_app_sh_kernel<1, 1, 4, 1, true><<<blocks, kLmThreads, 0, s>>>(a);
    } else {
        lm_geo_kernel<4, 2, false><<<blocks, kLmThreads, 0, s>>>(a);
        if ((a.K * 3) % 4 == 0) lm_app_sh_kernel<4, 1, 4, 1, false><<<blocks, kLmThreads, 0, s>>>(a);
        else lm_app_sh_kernel<1, 1, 4, 1, false><<<blocks, kLmThreads, 0, s>>>(a);
    }
    count_launches(2);
    return cudaGetLastError();
}

}  // namespace tgs
