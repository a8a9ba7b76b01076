// Internal declarations shared by the CUDA translation units of libtgs (never by the oracle).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/tgs.h"

namespace tgs {

constexpr int kTile = 16;
constexpr int kTilePixels = 256;
constexpr int kSplatWords = TGS_SPLAT_WORDS;

// Readings of the paper (R2/R3): constants of the 3DGS kernels TurboGS modifies.
constexpr float kLowpass = 0.3f;
constexpr float kJClamp = 1.3f;
constexpr float kAlphaMin = 0.00392156862745098f;  // 1/255
constexpr float kAlphaMax = 0.99f;
constexpr float kTMin = 0.0001f;

// A second stream of the context: the warp-per-tile raster kernel of a call runs on it, concurrently with the
// block-per-tile kernel on the caller's stream (fork / join by events; capturable in a CUDA graph).
struct SideStream {
    cudaStream_t aux;
    cudaEvent_t fork, join;
};

struct ctx_impl {
    int device;
    int num_sms;
    uint32_t* sched;  // device, 8 words: work-unit counters of the persistent raster kernels (self re-arming)
    SideStream side;
    char err[512];
};

// Kernel-side copy of the camera (same fields as tgs_camera; passed by value).
struct CamK {
    int W, H, gx, gy;
    float fx, fy, cx, cy;
    float R[9];
    float t[3];
    float znear;
    float bg[3];
};

inline CamK make_camk(const tgs_camera* c) {
    CamK k;
    k.W = c->width; k.H = c->height;
    k.gx = (c->width + kTile - 1) / kTile; k.gy = (c->height + kTile - 1) / kTile;
    k.fx = c->fx; k.fy = c->fy; k.cx = c->cx; k.cy = c->cy;
    for (int i = 0; i < 9; ++i) k.R[i] = c->R[i];
    for (int i = 0; i < 3; ++i) { k.t[i] = c->t[i]; k.bg[i] = c->bg[i]; }
    k.znear = c->znear;
    return k;
}

__device__ __forceinline__ void unpack_rect(uint32_t rx, uint32_t ry, int& x0, int& y0, int& x1, int& y1) {
    x0 = (int)(rx & 0xffffu); x1 = (int)(rx >> 16);
    y0 = (int)(ry & 0xffffu); y1 = (int)(ry >> 16);
}

// Every kernel launch of the library is counted (tgs_launch_count).
void count_launches(int n);

// Kernels with more than 48 KB of shared memory opt in through a function attribute, which is PER DEVICE: one flag
// per (kernel, device), set on the first launch on that device (a race between threads only sets it twice).
constexpr int kMaxDevices = 64;
struct SmemOptIn {
    unsigned char done[kMaxDevices] = {};
    cudaError_t ensure(const void* fn, size_t bytes) {
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) return e;
        if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
        if (!done[dev]) {
            e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
            if (e != cudaSuccess) return e;
            done[dev] = 1;
        }
        return cudaSuccess;
    }
};

// ---- launchers (one per translation unit) ---------------------------------------------------
cudaError_t launch_preprocess(const CamK& cam, int N, int D, const float* mu, const float* sc, const float* qt,
                              const float* op, const float* sh, float* splats, int32_t* radii,
                              uint8_t* clamped, cudaStream_t s);

size_t binsort_workspace_bytes(int N, int64_t Pcap, int T);
cudaError_t launch_bin_sort(const CamK& cam, int N, const float* splats, const uint32_t* tile_select, int64_t Pcap,
                            uint64_t* keys_sorted,
                            uint32_t* gid_sorted, uint32_t* tile_offsets, int64_t* P_dev, void* ws,
                            size_t ws_bytes, int num_sms, cudaStream_t s, const SideStream* side);

size_t sample_workspace_bytes(int T);
cudaError_t launch_sample(const CamK& cam, const float* err, const float* render, const float* target, int k,
                          int mode, int rnum, int rden, uint64_t seed, uint64_t* tile_score, uint32_t* tiles,
                          uint32_t* tpo, uint32_t* pix, uint32_t* tile_select, int32_t* kn_dev, void* ws,
                          cudaStream_t s);

// tgs_sample_static: launch_sample with its scratch in a static device array of sample.cu (no workspace argument)
int sample_static_max_tiles();
cudaError_t launch_sample_static(int device, const CamK& cam, const float* err, const float* render, const float* target,
                                 int k, int mode, int rnum, int rden, uint64_t seed, uint64_t* tile_score,
                                 uint32_t* tiles, uint32_t* tpo, uint32_t* pix, uint32_t* tile_select, int32_t* kn_dev,
                                 cudaStream_t s);

cudaError_t launch_raster_fwd(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, float* out_color, float* out_T, uint32_t* n_contrib,
                              uint32_t* n_walked, uint32_t* n_blended, uint32_t* sched, int num_sms, cudaStream_t s,
                              const SideStream* side);

cudaError_t launch_raster_bwd(const CamK& cam, int N, const float* splats, const uint32_t* tile_offsets,
                              const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                              const uint32_t* pix, const float* out_T, const uint32_t* n_contrib,
                              const float* dL_dcolor, float* dL_dsplats, uint32_t* sched, int num_sms, cudaStream_t s,
                              const SideStream* side);

cudaError_t launch_raster_fwd_lite(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                                   const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                   const uint32_t* pix, float* out_color, float* out_T, uint32_t* n_contrib,
                                   uint32_t* n_walked, uint32_t* n_blended, uint32_t* sched, int num_sms, cudaStream_t s);
cudaError_t launch_raster_bwd_lite(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                                   const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                   const uint32_t* pix, const float* out_T, const uint32_t* n_contrib,
                                   const float* dL_dcolor, float* dL_dsplats, uint32_t* sched, int num_sms, cudaStream_t s);

cudaError_t launch_raster_stats_lite(const CamK& cam, const float* splats, const uint32_t* tile_offsets,
                                     const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                     const uint32_t* pix, const float* pix_err, float* stats, float* out_depth,
                                     uint32_t* sched, int num_sms, cudaStream_t s);

cudaError_t launch_project_bwd(const CamK& cam, int N, int D, const float* mu, const float* sc, const float* qt,
                               const float* sh, const int32_t* radii, const uint8_t* clamped, const float* splats,
                               const float* dL_dsplats, float* dmu, float* dsc, float* dqt, float* dop,
                               float* dsh, int32_t* touched, cudaStream_t s);

cudaError_t launch_sample_paper(const CamK& cam, const uint16_t* E_half, const uint16_t* age, int n_pix, int n_hard,
                                int n_stable, uint64_t seed, uint32_t* tiles, uint32_t* tpo, uint32_t* pix,
                                int32_t* kn_dev, void* ws, cudaStream_t s);
cudaError_t launch_maps_update(const CamK& cam, uint16_t* E_half, uint16_t* age, const int32_t* kn_dev,
                               const uint32_t* pix, const float* pix_err, float beta, int num_sms, cudaStream_t s);

cudaError_t launch_raster_stats(const CamK& cam, int N, const float* splats, const uint32_t* tile_offsets,
                                const uint32_t* gid_sorted, int k, const uint32_t* tiles, const uint32_t* tpo,
                                const uint32_t* pix, const float* pix_err, float* stats, float* out_depth,
                                uint32_t* sched, int num_sms, cudaStream_t s, const SideStream* side);

cudaError_t launch_loss_sparse(int k, const uint32_t* tpo, const uint32_t* pix, const float* color, const float* target,
                               float eps_l1, float eps_ncc, float eps_lam, float* dL_dcolor, float* pix_err,
                               float* tile_stats, float* loss, cudaStream_t s);

// f4: parameter sets of tgs_lm_solve (device pointers in the parameter layouts).
struct LmSet {
    float* mu; float* sc; float* qt; float* op; float* sh;
};

struct LmArgs {
    LmSet g, m, v, d, p;   // g: [V, N, ...] read only; d / p nullable as a whole (d.mu == nullptr, p.mu == nullptr)
    const int32_t* update; // nullable [N]
    const int32_t* vt;     // nullable [V, N]: per-view touched masks; a view's gradient rows are read only where set
    int N, K, V;
    double b1, b2, eps;    // Eq. 14
    double inv_bc1, inv_bc2;  // 1 / (1 - beta^t), Eq. 19 right
    float eta, epsf;
    float b1f, b2f, omb1f, omb2f, ibc1f, ibc2f;  // fp32 copies for the Adam branch (1 - beta and 1 / (1 - beta^t) rounded once)
};

cudaError_t launch_lm_solve(const LmArgs& a, cudaStream_t s);

// Which views touch Gaussian n (bit v; all ones without per-view masks), 0 if the call does not update it at all:
// update[n] == 0, or touched in no view.  All mask words are loaded before any gradient (one latency, not one per view).
template <bool VT>
__device__ __forceinline__ unsigned long long lm_views(const LmArgs& a, int n) {
    if (a.update != nullptr && __ldg(a.update + n) == 0) return 0ull;
    if (!VT) return ~0ull;
    unsigned long long bits = 0ull;
    for (int vw = 0; vw < a.V; ++vw) bits |= (unsigned long long)(__ldg(a.vt + (size_t)vw * a.N + n) != 0) << vw;
    return bits;
}

}  // namespace tgs
