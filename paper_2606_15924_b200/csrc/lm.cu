// f4: the moment-damped LM solve, PAPER.md:231-239 (Eq. 14), 483-490 (Eq. 19), Alg. 1 steps 9-10.
//
// ONE fused kernel (the paper uses two): thread i of a block of 128 owns Gaussian n = 128 b + i for the
// two Cholesky blocks (geometry 10 x 10, appearance 4 x 4) and, independently, the block's 128 K 3 floats of the SH
// arrays are swept with coalesced 16-byte accesses for the Adam branch.  The two parts touch disjoint elements
// (the DC band sh[:,0,:] belongs to the appearance block), so there is no barrier and no shared memory; fusing
// them keeps the 32-byte sectors that hold a Gaussian's DC term (12 B of 192) in L2 between their two uses, so
// that the DRAM traffic is the algorithmic (V + 2) x 236 B read + (2 + outputs) x 236 B written per Gaussian.
// HBM bound: the fp64 factorisation (about 700 DFMA per Gaussian) hides behind the loads.
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
template <int D, class Acc>
__device__ __forceinline__ void lm_block(const LmArgs& a, const Acc acc, int n) {
    double A[D * (D + 1) / 2];
    double gb[D];
#pragma unroll
    for (int i = 0; i < D * (D + 1) / 2; ++i) A[i] = 0.0;
#pragma unroll
    for (int c = 0; c < D; ++c) gb[c] = 0.0;
    for (int vw = 0; vw < a.V; ++vw) {
        float gf[D];
#pragma unroll
        for (int c = 0; c < D; ++c) gf[c] = __ldg(acc.view(a.g, c, vw, a.N) + acc.off(c, n));
        double g[D];
#pragma unroll
        for (int c = 0; c < D; ++c) { g[c] = (double)gf[c]; gb[c] += g[c]; }
#pragma unroll
        for (int i = 0; i < D; ++i)
#pragma unroll
            for (int j = 0; j <= i; ++j) A[i * (i + 1) / 2 + j] = fma(g[i], g[j], A[i * (i + 1) / 2 + j]);
    }
    double mb[D], vb[D], x[D];
#pragma unroll
    for (int c = 0; c < D; ++c) {
        float* pm = acc.ptr(a.m, c) + acc.off(c, n);
        float* pv = acc.ptr(a.v, c) + acc.off(c, n);
        mb[c] = a.b1 * (double)*pm + (1.0 - a.b1) * gb[c];
        vb[c] = a.b2 * (double)*pv + (1.0 - a.b2) * gb[c] * gb[c];
        *pm = (float)mb[c];
        *pv = (float)vb[c];
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

// Adam branch of Eq. 19 for one coefficient: the moment sums in fp64 (cheap, and the stored moments are then the
// correctly rounded ones), the quotient in fp32.
__device__ __forceinline__ void adam_one(const LmArgs& a, double gbar, float& m, float& v, float& dlt) {
    const double mn = a.b1 * (double)m + (1.0 - a.b1) * gbar;
    const double vn = a.b2 * (double)v + (1.0 - a.b2) * gbar * gbar;
    m = (float)mn;
    v = (float)vn;
    const float mh = (float)(mn * a.inv_bc1);
    const float vh = (float)(vn * a.inv_bc2);
    dlt = -a.eta * mh / (sqrtf(vh) + a.epsf);
}

// VEC = 4: K * 3 is a multiple of 4 (degrees 1 and 3) and the block's span is swept with float4 accesses;
// VEC = 1: degree 2 (27 floats per Gaussian), scalar accesses.
template <int VEC>
__global__ void __launch_bounds__(kLmThreads) lm_solve_kernel(const LmArgs a) {
    const int n = blockIdx.x * kLmThreads + threadIdx.x;
    // ---- Adam branch over the block's span of the SH arrays (coalesced; skips the DC band) ----
    const int row = a.K * 3;                        // floats per Gaussian
    if (a.K > 1) {
        const size_t span0 = (size_t)blockIdx.x * kLmThreads * row;
        const size_t total = (size_t)a.N * row;
        const size_t vstride = total;               // floats between two views of grads.sh
        const int per_block = kLmThreads * row / VEC;
        for (int j = threadIdx.x; j < per_block; j += kLmThreads) {
            const size_t e = span0 + (size_t)j * VEC;
            if (e >= total) break;
            const int gn = (int)(e / row);
            const int r = (int)(e - (size_t)gn * row);   // first element's position inside the Gaussian's row
            const bool on = a.update == nullptr || __ldg(a.update + gn) != 0;
            if (VEC == 4) {
                float4 d4 = make_float4(0.f, 0.f, 0.f, 0.f);
                if (on) {
                    double gs[4] = {0.0, 0.0, 0.0, 0.0};
                    for (int vw = 0; vw < a.V; ++vw) {
                        const float4 g4 = __ldg(reinterpret_cast<const float4*>(a.g.sh + vw * vstride + e));
                        gs[0] += (double)g4.x; gs[1] += (double)g4.y; gs[2] += (double)g4.z; gs[3] += (double)g4.w;
                    }
                    float4 m4 = *reinterpret_cast<const float4*>(a.m.sh + e);
                    float4 v4 = *reinterpret_cast<const float4*>(a.v.sh + e);
                    if (r == 0) {  // x y z are the DC band (appearance block): only .w is an Adam coefficient
                        adam_one(a, gs[3], m4.w, v4.w, d4.w);
                        a.m.sh[e + 3] = m4.w;
                        a.v.sh[e + 3] = v4.w;
                        if (a.d.mu) a.d.sh[e + 3] = d4.w;
                        if (a.p.mu) a.p.sh[e + 3] += d4.w;
                    } else {
                        adam_one(a, gs[0], m4.x, v4.x, d4.x);
                        adam_one(a, gs[1], m4.y, v4.y, d4.y);
                        adam_one(a, gs[2], m4.z, v4.z, d4.z);
                        adam_one(a, gs[3], m4.w, v4.w, d4.w);
                        *reinterpret_cast<float4*>(a.m.sh + e) = m4;
                        *reinterpret_cast<float4*>(a.v.sh + e) = v4;
                        if (a.d.mu) *reinterpret_cast<float4*>(a.d.sh + e) = d4;
                        if (a.p.mu) {
                            float4 p4 = *reinterpret_cast<const float4*>(a.p.sh + e);
                            p4.x += d4.x; p4.y += d4.y; p4.z += d4.z; p4.w += d4.w;
                            *reinterpret_cast<float4*>(a.p.sh + e) = p4;
                        }
                    }
                } else if (a.d.mu) {
                    if (r == 0) a.d.sh[e + 3] = 0.f;
                    else *reinterpret_cast<float4*>(a.d.sh + e) = d4;
                }
            } else {
                if (r < 3) continue;
                float dl = 0.f;
                if (on) {
                    double gs = 0.0;
                    for (int vw = 0; vw < a.V; ++vw) gs += (double)__ldg(a.g.sh + vw * vstride + e);
                    float mm = a.m.sh[e], vv = a.v.sh[e];
                    adam_one(a, gs, mm, vv, dl);
                    a.m.sh[e] = mm;
                    a.v.sh[e] = vv;
                    if (a.p.mu) a.p.sh[e] += dl;
                }
                if (a.d.mu) a.d.sh[e] = dl;
            }
        }
    }
    // ---- the two LM blocks of Gaussian n (Eq. 14) ----
    if (n >= a.N) return;
    if (a.update != nullptr && __ldg(a.update + n) == 0) {
        if (a.d.mu) {
            const GeoAcc ga;
            const AppAcc aa{a.K};
#pragma unroll
            for (int c = 0; c < 10; ++c) ga.ptr(a.d, c)[ga.off(c, n)] = 0.f;
#pragma unroll
            for (int c = 0; c < 4; ++c) aa.ptr(a.d, c)[aa.off(c, n)] = 0.f;
        }
        return;
    }
    lm_block<4>(a, AppAcc{a.K}, n);
    lm_block<10>(a, GeoAcc(), n);
}

}  // namespace

cudaError_t launch_lm_solve(const LmArgs& a, cudaStream_t s) {
    if (a.N <= 0) return cudaSuccess;
    const int blocks = (a.N + kLmThreads - 1) / kLmThreads;
    if ((a.K * 3) % 4 == 0) lm_solve_kernel<4><<<blocks, kLmThreads, 0, s>>>(a);
    else lm_solve_kernel<1><<<blocks, kLmThreads, 0, s>>>(a);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
