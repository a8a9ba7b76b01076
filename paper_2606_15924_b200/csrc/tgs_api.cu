// C-ABI entry points of libtgs (include/tgs.h): argument validation, error reporting and launch
// order.  No arithmetic of the method lives here.
#include <math.h>
#include <stdarg.h>
#include <string.h>

#include <atomic>
#include <new>

#include "common.cuh"

using namespace tgs;

namespace tgs {
static std::atomic<uint64_t> g_launches{0};
void count_launches(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }
}  // namespace tgs

struct tgs_ctx : public ctx_impl {};

namespace {

int fail(tgs_ctx* ctx, int code, const char* fmt, ...) {
    if (ctx) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(ctx->err, sizeof(ctx->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

int cuda_fail(tgs_ctx* ctx, const char* where, cudaError_t e) {
    return fail(ctx, TGS_ERR_CUDA, "%s: %s", where, cudaGetErrorString(e));
}

constexpr size_t kCtxDeviceBytes = 8 * sizeof(uint32_t) + 256;

// Every entry point makes its context's device current: a process may hold contexts on several GPUs.
bool on_device(tgs_ctx* ctx, const char* where) {
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e == cudaSuccess) return true;
    cuda_fail(ctx, where, e);
    return false;
}

bool cam_ok(const tgs_camera* c) {
    return c && c->width > 0 && c->height > 0 && c->fx > 0.f && c->fy > 0.f;
}

int num_tiles(const tgs_camera* c) {
    return ((c->width + kTile - 1) / kTile) * ((c->height + kTile - 1) / kTile);
}

}  // namespace

extern "C" {

const char* tgs_version(void) { return "tgs 0.1 (sm_100a)"; }

uint64_t tgs_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

int tgs_create(tgs_ctx** out, int device) {
    if (!out) return TGS_ERR_INVALID_ARG;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || device < 0 || device >= count) return TGS_ERR_CUDA;  // no GPU, no fallback
    tgs_ctx* c = new (std::nothrow) tgs_ctx();
    if (!c) return TGS_ERR_INVALID_ARG;
    c->device = device;
    c->err[0] = 0;
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, device);
    if (e != cudaSuccess) { delete c; return TGS_ERR_CUDA; }
    c->num_sms = prop.multiProcessorCount;
    e = cudaSetDevice(device);
    if (e != cudaSuccess) { delete c; return TGS_ERR_CUDA; }
    // the only allocation the library ever makes: scheduler counters + a scratch line, once per context
    e = cudaMalloc((void**)&c->sched, kCtxDeviceBytes);  // 8 counter words + 256 B scratch (tgs_fp32_peak)
    if (e == cudaSuccess) e = cudaMemset(c->sched, 0, kCtxDeviceBytes);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->side.aux, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->side.fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->side.join, cudaEventDisableTiming);
    if (e != cudaSuccess) { delete c; return TGS_ERR_CUDA; }
    *out = c;
    return TGS_OK;
}

int tgs_destroy(tgs_ctx* ctx) {
    if (ctx && ctx->sched) {
        cudaFree(ctx->sched);
        cudaEventDestroy(ctx->side.fork);
        cudaEventDestroy(ctx->side.join);
        cudaStreamDestroy(ctx->side.aux);
    }
    delete ctx;
    return TGS_OK;
}

const char* tgs_last_error(const tgs_ctx* ctx) { return ctx ? ctx->err : "null context"; }

// ---- diagnostic: FFMA-only micro-benchmark (roofline denominator of the ALU-bound kernels) ----
namespace {
__global__ void __launch_bounds__(256) ffma_peak_kernel(float* out, float a, float b, int iters) {
    float x0 = threadIdx.x, x1 = x0 + 1.f, x2 = x0 + 2.f, x3 = x0 + 3.f, x4 = x0 + 4.f, x5 = x0 + 5.f, x6 = x0 + 6.f, x7 = x0 + 7.f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            x0 = fmaf(x0, a, b); x1 = fmaf(x1, a, b); x2 = fmaf(x2, a, b); x3 = fmaf(x3, a, b);
            x4 = fmaf(x4, a, b); x5 = fmaf(x5, a, b); x6 = fmaf(x6, a, b); x7 = fmaf(x7, a, b);
        }
    }
    const float r = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
    if (r == 123.456f) out[0] = r;  // keeps the chains alive
}
}  // namespace

int tgs_fp32_peak(tgs_ctx* ctx, int reps, double* tflops, void* stream) {
    if (!ctx || !tflops || reps < 1) return TGS_ERR_INVALID_ARG;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_fp32_peak", e);
    float* d = reinterpret_cast<float*>(ctx->sched + 8);  // the context's scratch line
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int blocks = ctx->num_sms * 8, iters = 4096;
    const double flop = 2.0 * 8 * 16 * (double)iters * 256.0 * blocks;
    double best = 0.0;
    for (int r = 0; r < reps + 2; ++r) {  // two warm-up launches
        cudaEventRecord(e0, s);
        ffma_peak_kernel<<<blocks, 256, 0, s>>>(d, 0.999f, 0.001f, iters);
        cudaEventRecord(e1, s);
        e = cudaEventSynchronize(e1);
        if (e != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (r >= 2 && ms > 0.f) best = fmax(best, flop / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_fp32_peak", e);
    *tflops = best;
    return TGS_OK;
}

int tgs_preprocess(tgs_ctx* ctx, const tgs_camera* cam, int N, int sh_degree, const float* means3D,
                   const float* scales, const float* quats, const float* opacities, const float* sh,
                   float* splats, int32_t* radii, uint8_t* clamped, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_preprocess")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_preprocess: bad camera");
    if (N < 0) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_preprocess: N < 0");
    if (sh_degree < 0 || sh_degree > 3) return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_preprocess: sh_degree %d not in 0..3", sh_degree);
    if (num_tiles(cam) > (1 << 20) || cam->width > 65535 * kTile || cam->height > 65535 * kTile)
        return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_preprocess: image too large (T > 2^20)");
    if (N == 0) return TGS_OK;
    if (!means3D || !scales || !quats || !opacities || !sh || !splats || !radii || !clamped)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_preprocess: null pointer");
    if (((uintptr_t)sh & 15) || ((uintptr_t)quats & 15) || ((uintptr_t)splats & 15))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_preprocess: sh, quats and splats must be 16-byte aligned");
    cudaError_t e = launch_preprocess(make_camk(cam), N, sh_degree, means3D, scales, quats, opacities, sh, splats,
                                      radii, clamped, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_preprocess", e);
    return TGS_OK;
}

int tgs_bin_sort_workspace_bytes(int N, int64_t P_capacity, int T, size_t* bytes) {
    if (!bytes || N < 0 || P_capacity < 0 || T <= 0) return TGS_ERR_INVALID_ARG;
    *bytes = binsort_workspace_bytes(N, P_capacity, T);
    return TGS_OK;
}

int tgs_bin_sort(tgs_ctx* ctx, const tgs_camera* cam, int N, const float* splats, const uint32_t* tile_select,
                 int64_t P_capacity,
                 uint64_t* keys_sorted, uint32_t* gid_sorted, uint32_t* tile_offsets, int64_t* P_dev,
                 int64_t* P_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_bin_sort")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_bin_sort: bad camera");
    if (N < 0 || P_capacity < 0) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_bin_sort: negative size");
    if (P_capacity >= (1ll << 30) || (int64_t)N >= (1ll << 30))
        return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_bin_sort: N and P_capacity must be < 2^30");
    const int T = num_tiles(cam);
    if (T > (1 << 20)) return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_bin_sort: T > 2^20");
    if (!gid_sorted || !tile_offsets || !P_dev || !workspace || (N > 0 && !splats))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_bin_sort: null pointer");
    const size_t need = binsort_workspace_bytes(N, P_capacity, T);
    if (workspace_bytes < need)
        return fail(ctx, TGS_ERR_CAPACITY, "tgs_bin_sort: workspace %zu B < required %zu B", workspace_bytes, need);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = launch_bin_sort(make_camk(cam), N, splats, tile_select, P_capacity, keys_sorted, gid_sorted, tile_offsets,
                                    P_dev, workspace, workspace_bytes, ctx->num_sms, s, &ctx->side);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_bin_sort", e);
    if (P_host) {
        int64_t h[2];
        e = cudaMemcpyAsync(h, P_dev, sizeof(h), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return cuda_fail(ctx, "tgs_bin_sort (P readback)", e);
        *P_host = h[0];
        if (h[1]) return fail(ctx, TGS_ERR_CAPACITY, "tgs_bin_sort: P = %lld exceeds P_capacity = %lld",
                              (long long)h[0], (long long)P_capacity);
    }
    return TGS_OK;
}

int tgs_sample_num_tiles(const tgs_camera* cam, int num, int den) {
    if (!cam_ok(cam) || den <= 0 || num < 0) return -1;
    const int T = num_tiles(cam);
    int64_t k = ((int64_t)num * T) / den;
    if (k < 1) k = 1;
    if (k > T) k = T;
    return (int)k;
}

int tgs_sample_workspace_bytes(const tgs_camera* cam, size_t* bytes) {
    if (!cam_ok(cam) || !bytes) return TGS_ERR_INVALID_ARG;
    *bytes = sample_workspace_bytes(num_tiles(cam));
    return TGS_OK;
}

int tgs_sample(tgs_ctx* ctx, const tgs_camera* cam, const float* err, const float* render, const float* target,
               int tile_pct_num, int tile_pct_den, int pixel_mode, int pix_rate_num, int pix_rate_den,
               uint64_t seed, uint64_t* tile_score, uint32_t* tiles, uint32_t* tile_pix_offsets, uint32_t* pix,
               uint32_t* tile_select, int32_t* kn_dev, int32_t* kn_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_sample")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample: bad camera");
    if (tile_pct_den <= 0 || tile_pct_num < 0 || tile_pct_num > tile_pct_den)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample: tile fraction %d/%d not in [0,1]", tile_pct_num, tile_pct_den);
    if (pixel_mode != TGS_PIXELS_ALL && pixel_mode != TGS_PIXELS_BERNOULLI_ERR)
        return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_sample: pixel_mode %d", pixel_mode);
    if (pixel_mode == TGS_PIXELS_BERNOULLI_ERR &&
        (pix_rate_den <= 0 || pix_rate_den > 255 || pix_rate_num < 0 || pix_rate_num > 255))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample: pixel rate %d/%d outside 0..255", pix_rate_num, pix_rate_den);
    if (!err && !(render && target)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample: need err or render+target");
    if (!tile_score || !tiles || !tile_pix_offsets || !pix || !kn_dev || !workspace)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample: null pointer");
    const int T = num_tiles(cam);
    if (T > (1 << 20)) return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_sample: T > 2^20");
    const size_t need = sample_workspace_bytes(T);
    if (workspace_bytes < need)
        return fail(ctx, TGS_ERR_CAPACITY, "tgs_sample: workspace %zu B < required %zu B", workspace_bytes, need);
    const int k = tgs_sample_num_tiles(cam, tile_pct_num, tile_pct_den);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = launch_sample(make_camk(cam), err, render, target, k, pixel_mode, pix_rate_num, pix_rate_den, seed,
                                  tile_score, tiles, tile_pix_offsets, pix, tile_select, kn_dev, workspace, s);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_sample", e);
    if (kn_host) {
        e = cudaMemcpyAsync(kn_host, kn_dev, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return cuda_fail(ctx, "tgs_sample (k,n readback)", e);
    }
    return TGS_OK;
}

// tgs_sample without a context or a workspace (include/tgs.h: for callers that cannot allocate device memory).
// Validation mirrors tgs_sample; messages go to the caller's buffer because there is no context to keep them in.
// Nothing on this path allocates: no cudaMalloc / cudaFree, no stream or event creation, no new / malloc.
int tgs_sample_static(int device, const tgs_camera* cam, const float* err, const float* render, const float* target,
                      int tile_pct_num, int tile_pct_den, int pixel_mode, int pix_rate_num, int pix_rate_den,
                      uint64_t seed, uint64_t* tile_score, uint32_t* tiles, uint32_t* tile_pix_offsets, uint32_t* pix,
                      uint32_t* tile_select, int32_t* kn_dev, int32_t* kn_host, char* err_msg, size_t err_msg_bytes,
                      void* stream) {
    auto say = [&](int code, const char* fmt, auto... a) {
        if (err_msg && err_msg_bytes) snprintf(err_msg, err_msg_bytes, fmt, a...);
        return code;
    };
    if (err_msg && err_msg_bytes) err_msg[0] = 0;
    if (device < 0) return say(TGS_ERR_INVALID_ARG, "tgs_sample_static: device %d", device);
    cudaError_t e = cudaSetDevice(device);
    if (e != cudaSuccess) return say(TGS_ERR_CUDA, "tgs_sample_static: cudaSetDevice(%d): %s", device, cudaGetErrorString(e));
    if (!cam_ok(cam)) return say(TGS_ERR_INVALID_ARG, "%s", "tgs_sample_static: bad camera");
    if (tile_pct_den <= 0 || tile_pct_num < 0 || tile_pct_num > tile_pct_den)
        return say(TGS_ERR_INVALID_ARG, "tgs_sample_static: tile fraction %d/%d not in [0,1]", tile_pct_num, tile_pct_den);
    if (pixel_mode != TGS_PIXELS_ALL && pixel_mode != TGS_PIXELS_BERNOULLI_ERR)
        return say(TGS_ERR_UNSUPPORTED, "tgs_sample_static: pixel_mode %d", pixel_mode);
    if (pixel_mode == TGS_PIXELS_BERNOULLI_ERR &&
        (pix_rate_den <= 0 || pix_rate_den > 255 || pix_rate_num < 0 || pix_rate_num > 255))
        return say(TGS_ERR_INVALID_ARG, "tgs_sample_static: pixel rate %d/%d outside 0..255", pix_rate_num, pix_rate_den);
    if (!err && !(render && target)) return say(TGS_ERR_INVALID_ARG, "%s", "tgs_sample_static: need err or render+target");
    if (!tile_score || !tiles || !tile_pix_offsets || !pix || !kn_dev)
        return say(TGS_ERR_INVALID_ARG, "%s", "tgs_sample_static: null pointer");
    // 64-bit tile count: the camera is unchecked user input and the limit must hold before anything is launched
    const int64_t T = (int64_t)((cam->width + kTile - 1) / kTile) * (int64_t)((cam->height + kTile - 1) / kTile);
    if (T > (int64_t)sample_static_max_tiles())
        return say(TGS_ERR_CAPACITY,
                   "tgs_sample_static: a %d x %d image has %lld tiles, the static scratch holds %d "
                   "(TGS_SAMPLE_STATIC_MAX_TILES); use tgs_sample with a workspace",
                   cam->width, cam->height, (long long)T, sample_static_max_tiles());
    const int k = tgs_sample_num_tiles(cam, tile_pct_num, tile_pct_den);
    cudaStream_t s = (cudaStream_t)stream;
    e = launch_sample_static(device, make_camk(cam), err, render, target, k, pixel_mode, pix_rate_num, pix_rate_den, seed,
                             tile_score, tiles, tile_pix_offsets, pix, tile_select, kn_dev, s);
    if (e != cudaSuccess) return say(TGS_ERR_CUDA, "tgs_sample_static: %s", cudaGetErrorString(e));
    if (kn_host) {
        e = cudaMemcpyAsync(kn_host, kn_dev, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return say(TGS_ERR_CUDA, "tgs_sample_static (k,n readback): %s", cudaGetErrorString(e));
    }
    return TGS_OK;
}

int tgs_raster_fwd_sparse(tgs_ctx* ctx, const tgs_camera* cam, int N, const float* splats,
                          const uint32_t* tile_offsets, const uint32_t* gid_sorted, int k, const uint32_t* tiles,
                          const uint32_t* tile_pix_offsets, const uint32_t* pix, float* out_color, float* out_T,
                          uint32_t* n_contrib, uint32_t* n_walked, uint32_t* n_blended, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_raster_fwd_sparse")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_fwd_sparse: bad camera");
    if (N < 0 || k < 0 || k > num_tiles(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_fwd_sparse: bad N or k");
    if (k == 0) return TGS_OK;
    if (!splats || !tile_offsets || !gid_sorted || !tiles || !tile_pix_offsets || !pix || !out_color || !out_T || !n_contrib)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_fwd_sparse: null pointer");
    cudaError_t e = launch_raster_fwd(make_camk(cam), splats, tile_offsets, gid_sorted, k, tiles, tile_pix_offsets, pix,
                                      out_color, out_T, n_contrib, n_walked, n_blended, ctx->sched, ctx->num_sms, (cudaStream_t)stream,
                                      &ctx->side);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_raster_fwd_sparse", e);
    return TGS_OK;
}

int tgs_raster_bwd_sparse(tgs_ctx* ctx, const tgs_camera* cam, int N, int sh_degree, const float* splats,
                          const uint32_t* tile_offsets, const uint32_t* gid_sorted, int k, const uint32_t* tiles,
                          const uint32_t* tile_pix_offsets, const uint32_t* pix, const float* out_T,
                          const uint32_t* n_contrib, const float* dL_dcolor, const float* means3D,
                          const float* scales, const float* quats, const float* sh, const int32_t* radii,
                          const uint8_t* clamped, float* dL_dsplats, float* dL_dmeans3D, float* dL_dscales,
                          float* dL_dquats, float* dL_dopacities, float* dL_dsh, int32_t* touched, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_raster_bwd_sparse")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_bwd_sparse: bad camera");
    if (N < 0 || k < 0 || k > num_tiles(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_bwd_sparse: bad N or k");
    if (sh_degree < 0 || sh_degree > 3) return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_raster_bwd_sparse: sh_degree %d", sh_degree);
    if (N == 0) return TGS_OK;
    if (!splats || !dL_dsplats) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_bwd_sparse: null pointer");
    if (k > 0 && (!tile_offsets || !gid_sorted || !tiles || !tile_pix_offsets || !pix || !out_T || !n_contrib || !dL_dcolor))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_bwd_sparse: null pointer");
    cudaStream_t s = (cudaStream_t)stream;
    const CamK ck = make_camk(cam);
    cudaError_t e = launch_raster_bwd(ck, N, splats, tile_offsets, gid_sorted, k, tiles, tile_pix_offsets, pix, out_T,
                                      n_contrib, dL_dcolor, dL_dsplats, ctx->sched + 4, ctx->num_sms, s, &ctx->side);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_raster_bwd_sparse (raster)", e);
    if (dL_dmeans3D) {
        if (!dL_dscales || !dL_dquats || !dL_dopacities || !dL_dsh || !means3D || !scales || !quats || !sh || !radii || !clamped)
            return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_bwd_sparse: null pointer (projection half)");
        if (((uintptr_t)quats & 15) || ((uintptr_t)dL_dquats & 15) || ((uintptr_t)dL_dsplats & 15) || ((uintptr_t)sh & 15) ||
            ((uintptr_t)dL_dsh & 15))
            return fail(ctx, TGS_ERR_INVALID_ARG,
                        "tgs_raster_bwd_sparse: quats, sh, dL_dquats, dL_dsh, dL_dsplats must be 16-byte aligned");
        e = launch_project_bwd(ck, N, sh_degree, means3D, scales, quats, sh, radii, clamped, splats, dL_dsplats, dL_dmeans3D,
                               dL_dscales, dL_dquats, dL_dopacities, dL_dsh, touched, s);
        if (e != cudaSuccess) return cuda_fail(ctx, "tgs_raster_bwd_sparse (projection)", e);
    }
    return TGS_OK;
}

int tgs_loss_sparse(tgs_ctx* ctx, const tgs_camera* cam, int k, const uint32_t* tile_pix_offsets, const uint32_t* pix,
                    const float* color, const float* target, float eps_l1, float eps_ncc, float eps_lambda,
                    float* dL_dcolor, float* pix_err, float* tile_stats, float* loss, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_loss_sparse")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_loss_sparse: bad camera");
    if (k < 0 || k > num_tiles(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_loss_sparse: k = %d outside 0..T", k);
    if (!(eps_l1 > 0.f) || !(eps_ncc > 0.f) || !(eps_lambda > 0.f))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_loss_sparse: the three eps must be positive");
    if (!tile_pix_offsets || !pix || !color || !target || !dL_dcolor || !pix_err || !tile_stats)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_loss_sparse: null pointer");
    cudaError_t e = launch_loss_sparse(k, tile_pix_offsets, pix, color, target, eps_l1, eps_ncc, eps_lambda, dL_dcolor,
                                       pix_err, tile_stats, loss, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_loss_sparse", e);
    return TGS_OK;
}

int tgs_raster_stats_sparse(tgs_ctx* ctx, const tgs_camera* cam, int N, const float* splats,
                            const uint32_t* tile_offsets, const uint32_t* gid_sorted, int k, const uint32_t* tiles,
                            const uint32_t* tile_pix_offsets, const uint32_t* pix, const float* pix_err, float* stats,
                            float* out_depth, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_raster_stats_sparse")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_stats_sparse: bad camera");
    if (N < 0 || k < 0 || k > num_tiles(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_stats_sparse: bad N or k");
    if (!stats || (N > 0 && !splats) || (k > 0 && (!tile_offsets || !gid_sorted || !tiles || !tile_pix_offsets || !pix || !pix_err)))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_stats_sparse: null pointer");
    if (((uintptr_t)splats & 15) || ((uintptr_t)stats & 15))
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_raster_stats_sparse: splats and stats must be 16-byte aligned");
    cudaError_t e = launch_raster_stats(make_camk(cam), N, splats, tile_offsets, gid_sorted, k, tiles, tile_pix_offsets, pix,
                                        pix_err, stats, out_depth, ctx->sched, ctx->num_sms, (cudaStream_t)stream, &ctx->side);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_raster_stats_sparse", e);
    return TGS_OK;
}

int tgs_sample_paper(tgs_ctx* ctx, const tgs_camera* cam, const uint16_t* E_half, const uint16_t* age, int n_pix,
                     int n_hard, int n_stable, uint64_t seed, uint32_t* tiles, uint32_t* tile_pix_offsets, uint32_t* pix,
                     int32_t* kn_dev, int32_t* kn_host, void* workspace, size_t workspace_bytes, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_sample_paper")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample_paper: bad camera");
    if (n_pix < 1 || n_pix > 256 || n_hard < 0 || n_stable < 0 || n_hard + n_stable > n_pix)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample_paper: need 1 <= n_pix <= 256 and n_hard + n_stable <= n_pix (got %d, %d, %d)",
                    n_pix, n_hard, n_stable);
    if (!E_half || !age || !tiles || !tile_pix_offsets || !pix || !kn_dev || !workspace)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_sample_paper: null pointer");
    const int T = num_tiles(cam);
    if (T > (1 << 20)) return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_sample_paper: T > 2^20");
    const size_t need = sample_workspace_bytes(T);
    if (workspace_bytes < need)
        return fail(ctx, TGS_ERR_CAPACITY, "tgs_sample_paper: workspace %zu B < required %zu B", workspace_bytes, need);
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e = launch_sample_paper(make_camk(cam), E_half, age, n_pix, n_hard, n_stable, seed, tiles, tile_pix_offsets,
                                        pix, kn_dev, workspace, s);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_sample_paper", e);
    if (kn_host) {
        e = cudaMemcpyAsync(kn_host, kn_dev, 2 * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) return cuda_fail(ctx, "tgs_sample_paper (k, n readback)", e);
    }
    return TGS_OK;
}

int tgs_maps_update(tgs_ctx* ctx, const tgs_camera* cam, uint16_t* E_half, uint16_t* age, const int32_t* kn_dev,
                    const uint32_t* pix, const float* pix_err, float beta, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_maps_update")) return TGS_ERR_CUDA;
    if (!cam_ok(cam)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_maps_update: bad camera");
    if (!(beta >= 0.f && beta <= 1.f)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_maps_update: beta outside [0, 1]");
    if (!E_half || !age || !kn_dev || !pix || !pix_err) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_maps_update: null pointer");
    cudaError_t e = launch_maps_update(make_camk(cam), E_half, age, kn_dev, pix, pix_err, beta, ctx->num_sms, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_maps_update", e);
    return TGS_OK;
}

int tgs_lm_solve(tgs_ctx* ctx, int N, int sh_degree, int V, const tgs_params* grads, const int32_t* update,
                 const int32_t* view_touched, float beta1,
                 float beta2, float eps, float eta_sh, int t, const tgs_params* m, const tgs_params* v,
                 const tgs_params* delta, const tgs_params* params, void* stream) {
    if (!ctx) return TGS_ERR_INVALID_ARG;
    if (!on_device(ctx, "tgs_lm_solve")) return TGS_ERR_CUDA;
    if (N < 0) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_lm_solve: N < 0");
    if (sh_degree < 0 || sh_degree > 3) return fail(ctx, TGS_ERR_UNSUPPORTED, "tgs_lm_solve: sh_degree %d not in 0..3", sh_degree);
    if (V < 1 || V > 64) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_lm_solve: V = %d outside 1..64", V);
    if (!(beta1 >= 0.f && beta1 < 1.f) || !(beta2 >= 0.f && beta2 < 1.f) || !(eps > 0.f) || t < 1)
        return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_lm_solve: need 0 <= beta < 1, eps > 0, t >= 1");
    if (!grads || !m || !v || (!delta && !params)) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_lm_solve: null parameter set");
    if (N == 0) return TGS_OK;
    const tgs_params* sets[5] = {grads, m, v, delta, params};
    LmArgs a;
    LmSet* dst[5] = {&a.g, &a.m, &a.v, &a.d, &a.p};
    for (int i = 0; i < 5; ++i) {
        const tgs_params* q = sets[i];
        if (!q) { *dst[i] = LmSet{nullptr, nullptr, nullptr, nullptr, nullptr}; continue; }
        if (!q->means3D || !q->scales || !q->quats || !q->opacities || !q->sh)
            return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_lm_solve: null pointer in parameter set %d", i);
        if ((uintptr_t)q->sh & 15) return fail(ctx, TGS_ERR_INVALID_ARG, "tgs_lm_solve: sh pointers must be 16-byte aligned");
        *dst[i] = LmSet{q->means3D, q->scales, q->quats, q->opacities, q->sh};
    }
    a.update = update;
    a.vt = view_touched;
    a.N = N; a.K = (sh_degree + 1) * (sh_degree + 1); a.V = V;
    a.b1 = (double)beta1; a.b2 = (double)beta2; a.eps = (double)eps;
    // bias corrections of Eq. 19 (right) are scalars of the call, formed in double on the host (pow: O(1) in t)
    const double p1 = pow(a.b1, (double)t), p2 = pow(a.b2, (double)t);
    a.inv_bc1 = 1.0 / (1.0 - p1); a.inv_bc2 = 1.0 / (1.0 - p2);
    a.eta = eta_sh; a.epsf = eps;
    a.b1f = beta1; a.b2f = beta2; a.omb1f = (float)(1.0 - a.b1); a.omb2f = (float)(1.0 - a.b2);
    a.ibc1f = (float)a.inv_bc1; a.ibc2f = (float)a.inv_bc2;
    cudaError_t e = launch_lm_solve(a, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(ctx, "tgs_lm_solve", e);
    return TGS_OK;
}

}  // extern "C"
