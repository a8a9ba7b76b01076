// tgs_sample: per-tile error reduction, top-k tile selection and tile-ordered sampled-pixel
// lists ("sampled pixels are ordered by their tile indices",
// 93 Eq. 2, 128-150 Sec. 3.5, 156 "tile-wise pixel offsets via prefix-sum").  Selection is done in
// integers on a fixed-point copy of the error so that it is order independent and bit exact.
#include <cuda_fp16.h>

#include <atomic>

#include "common.cuh"

// Scratch of tgs_sample_static (include/tgs.h): the per-tile keep masks and selection flags that tgs_sample keeps
// in a caller-allocated workspace live here instead, in memory that is part of the loaded library image, so that the
// call works for a host program that has no way to allocate device memory.  Sized for
// TGS_SAMPLE_STATIC_MAX_TILES = 16384 tiles (36 B + 4 B per tile, each part rounded up to 256 B): 640 KiB, held by
// every GPU that loads libtgs from the moment the module is loaded until the process exits.
// In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and is never
// passed to a kernel; static_scratch_on() below turns it into one, per device.
constexpr size_t kStaticScratchBytes = 640u * 1024u;
static __device__ __align__(256) unsigned char g_sample_static_scratch[kStaticScratchBytes];

namespace tgs {

namespace {

constexpr float kErrClamp = 15.999f;
constexpr float kErrScale = 1048576.0f;  // 2^20

struct TileMeta {       // per tile, written by the reduction kernel
    uint32_t mask[8];   // keep decision of each of the 256 local pixels (bit = local index)
    uint32_t npix;      // number of kept pixels (>= 1)
};

__device__ __forceinline__ uint64_t mix64(uint64_t seed, uint64_t idx) {
    uint64_t z = seed + (idx + 1ull) * 0x9E3779B97F4A7C15ull;
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ull;
    z ^= z >> 27; z *= 0x94D049BB133111EBull;
    z ^= z >> 31;
    return z;
}

__device__ __forceinline__ uint32_t quant_err(float e) {
    if (!(e > 0.0f)) return 0u;  // negative, zero, NaN
    e = fminf(e, kErrClamp);
    return (uint32_t)(e * kErrScale);  // exact: multiplication by 2^20, truncation
}

// One warp per tile.  Lane l owns local pixels 8l .. 8l+7 (row l/2, columns 8(l%2) .. +7).
__global__ void __launch_bounds__(256)
tile_reduce_kernel(const CamK cam, const float* __restrict__ err, const float* __restrict__ render,
                   const float* __restrict__ target, int mode, int rnum, int rden, uint64_t seed,
                   uint64_t* __restrict__ tile_score, TileMeta* __restrict__ meta) {
    const int T = cam.gx * cam.gy;
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= T) return;
    const int lane = threadIdx.x & 31;
    const int tx = t % cam.gx, ty = t / cam.gx;
    const int y = ty * kTile + (lane >> 1);
    const int xb = tx * kTile + (lane & 1) * 8;
    uint32_t q[8];
    uint32_t cnt = 0, qmax = 0, imax = 0xffffffffu;
    uint64_t sum = 0;
    uint32_t s16 = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const int x = xb + j;
        q[j] = 0;
        if (x < cam.W && y < cam.H) {
            const size_t p = (size_t)y * cam.W + x;
            float e;
            if (err) e = err[p];
            else e = (fabsf(render[3 * p] - target[3 * p]) + fabsf(render[3 * p + 1] - target[3 * p + 1])) +
                     fabsf(render[3 * p + 2] - target[3 * p + 2]);
            q[j] = quant_err(e);
            ++cnt; sum += q[j]; s16 += q[j] >> 8;
            const uint32_t li = (uint32_t)(lane * 8 + j);
            if (imax == 0xffffffffu || q[j] > qmax) { qmax = q[j]; imax = li; }
        }
    }
    // warp reductions: count, sums, argmax (max q, lowest local index on ties)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
        sum += __shfl_xor_sync(0xffffffffu, sum, o);
        s16 += __shfl_xor_sync(0xffffffffu, s16, o);
        const uint32_t oq = __shfl_xor_sync(0xffffffffu, qmax, o);
        const uint32_t oi = __shfl_xor_sync(0xffffffffu, imax, o);
        if (oi != 0xffffffffu && (imax == 0xffffffffu || oq > qmax || (oq == qmax && oi < imax))) { qmax = oq; imax = oi; }
    }
    // keep decisions of this lane's 8 pixels
    uint32_t bits = 0;
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        const int x = xb + j;
        if (x < cam.W && y < cam.H) {
            bool keep = true;
            if (mode != TGS_PIXELS_ALL) {
                const uint64_t p = (uint64_t)y * cam.W + x;
                const uint64_t u16 = mix64(seed, p) >> 48;
                const uint64_t q16 = q[j] >> 8;
                keep = (u16 * (uint64_t)s16 * (uint64_t)rden) < ((uint64_t)rnum * cnt * q16 * 65536ull);
            }
            if (keep) bits |= 1u << j;
        }
    }
    uint32_t npix = __popc(bits);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) npix += __shfl_xor_sync(0xffffffffu, npix, o);
    if (npix == 0) {  // N_pix >= 1: keep the max-error pixel
        if ((int)(imax >> 3) == lane) bits |= 1u << (imax & 7);
        npix = 1;
    }
    // pack: word w holds local pixels 32w .. 32w+31 = lanes 4w .. 4w+3
    uint32_t word = bits << ((lane & 3) * 8);
    word |= __shfl_xor_sync(0xffffffffu, word, 1);
    word |= __shfl_xor_sync(0xffffffffu, word, 2);
    if ((lane & 3) == 0) meta[t].mask[lane >> 2] = word;
    if (lane == 0) {
        meta[t].npix = npix;
        tile_score[t] = (sum << 8) / cnt;  // cnt >= 1: every tile of the grid has an in-image pixel
    }
}

// Block-wide exclusive scan of one 64-bit value per thread (1024 threads); wsum holds 33 words.  Ends with a barrier.
__device__ __forceinline__ uint64_t block_excl_scan_u64(uint64_t v, uint64_t* wsum, uint64_t& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint64_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint64_t yv = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += yv;
    }
    if (lane == 31) wsum[warp] = x;
    __syncthreads();
    if (warp == 0) {
        const uint64_t w = wsum[lane];
        uint64_t xs = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint64_t yv = __shfl_up_sync(0xffffffffu, xs, o);
            if (lane >= o) xs += yv;
        }
        wsum[lane] = xs - w;
        if (lane == 31) wsum[32] = xs;
    }
    __syncthreads();
    const uint64_t r = wsum[warp] + (x - v);
    total = wsum[32];
    __syncthreads();
    return r;
}

// single block: top-k selection, compaction of the selected tiles (ascending id) and exclusive prefix sum of
// their pixel counts.
//   Selection: tile t is selected iff fewer than k tiles precede it in the order (score descending, tile id
//   ascending).  The k-th largest score s* is found by an MSD radix select on the 64-bit scores (5 passes of
//   8 bits over the 40 significant bits, a 256-bin shared histogram over the tiles that still match the prefix): O(T) work for any T (the
//   first version ranked every tile against every other, O(T^2)).  Tiles with score > s* are selected, and of
//   those with score == s* the first (k - #greater) in tile order.
//   Compaction: a 64-bit scan carries both results: count << 40 | pixels.
__global__ void __launch_bounds__(1024)
tile_select_compact_kernel(int T, int k, const uint64_t* __restrict__ tile_score, const TileMeta* __restrict__ meta,
                           uint32_t* __restrict__ selected, uint32_t* __restrict__ tiles, uint32_t* __restrict__ tpo,
                           int32_t* __restrict__ kn_dev) {
    __shared__ uint64_t wsum[33];
    __shared__ uint64_t carry_s, s_prefix;
    __shared__ uint32_t hist[256], wtot[8];
    __shared__ uint32_t s_kk, carry_eq;
    if (threadIdx.x == 0) { carry_s = 0; carry_eq = 0; s_prefix = 0; s_kk = (uint32_t)k; }
    __syncthreads();
    // ---- the k-th largest score ----
    // scores are (sum of <= 256 fixed-point errors < 2^24, << 8) / count < 2^40 (R11): bytes 7..5 are zero
    constexpr int kTopByte = 4;
    for (int p = kTopByte; p >= 0; --p) {
        if (threadIdx.x < 256) hist[threadIdx.x] = 0u;
        __syncthreads();
        const uint64_t prefix = s_prefix;
        for (int t = threadIdx.x; t < T; t += 1024) {
            const uint64_t sc = tile_score[t];
            if ((sc >> (8 * (p + 1))) == prefix) atomicAdd(&hist[(uint32_t)(sc >> (8 * p)) & 255u], 1u);
        }
        __syncthreads();
        // the digit d with  #(digits > d) < kk <= #(digits >= d): a scan over the bins from the top (threads 0..255)
        const uint32_t kk = s_kk;
        uint32_t h = 0, incl = 0;
        if (threadIdx.x < 256) {
            h = hist[255 - threadIdx.x];
            incl = h;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t yv = __shfl_up_sync(0xffffffffu, incl, o);
                if ((threadIdx.x & 31) >= o) incl += yv;
            }
            if ((threadIdx.x & 31) == 31) wtot[threadIdx.x >> 5] = incl;
        }
        __syncthreads();
        if (threadIdx.x < 256) {
            for (int w = 0; w < (int)(threadIdx.x >> 5); ++w) incl += wtot[w];
            const uint32_t excl = incl - h;
            if (excl < kk && kk <= incl) { s_prefix = (prefix << 8) | (uint64_t)(255 - threadIdx.x); s_kk = kk - excl; }
        }
        __syncthreads();
    }
    const uint64_t sstar = s_prefix;
    const uint32_t need_eq = s_kk;  // how many of the tiles with score == s* are selected (the first ones in tile order)
    // ---- selection flags and compaction, 1024 tiles at a time ----
    for (int b0 = 0; b0 < T; b0 += 1024) {
        const int t = b0 + threadIdx.x;
        const uint64_t sc = t < T ? tile_score[t] : 0ull;
        const bool gt = t < T && sc > sstar, eq = t < T && sc == sstar;
        uint64_t tot_eq;
        const uint64_t eq_rank = (uint64_t)carry_eq + block_excl_scan_u64(eq ? 1ull : 0ull, wsum, tot_eq);
        const bool sel = gt || (eq && eq_rank < (uint64_t)need_eq);
        if (t < T) selected[t] = sel ? 1u : 0u;
        const uint64_t v = sel ? ((1ull << 40) | (uint64_t)meta[t].npix) : 0ull;
        uint64_t tot;
        const uint64_t excl = carry_s + block_excl_scan_u64(v, wsum, tot);
        if (sel) {
            const uint32_t pos = (uint32_t)(excl >> 40);
            tiles[pos] = (uint32_t)t;
            tpo[pos] = (uint32_t)(excl & ((1ull << 40) - 1));
        }
        __syncthreads();
        if (threadIdx.x == 0) { carry_s += tot; carry_eq += (uint32_t)tot_eq; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const uint32_t kk = (uint32_t)(carry_s >> 40), nn = (uint32_t)(carry_s & ((1ull << 40) - 1));
        tpo[kk] = nn;
        kn_dev[0] = (int32_t)kk;
        kn_dev[1] = (int32_t)nn;
    }
}

// compaction alone (every tile selected): the paper's sampler
__global__ void __launch_bounds__(1024)
tile_compact_kernel(int T, const uint32_t* __restrict__ selected, const TileMeta* __restrict__ meta,
                    uint32_t* __restrict__ tiles, uint32_t* __restrict__ tpo, int32_t* __restrict__ kn_dev) {
    __shared__ uint64_t wsum[33];
    __shared__ uint64_t carry_s;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < T; b0 += 1024) {
        const int t = b0 + threadIdx.x;
        const bool sel = t < T && selected[t];
        const uint64_t v = sel ? ((1ull << 40) | (uint64_t)meta[t].npix) : 0ull;
        uint64_t tot;
        const uint64_t excl = carry_s + block_excl_scan_u64(v, wsum, tot);
        if (sel) {
            const uint32_t pos = (uint32_t)(excl >> 40);
            tiles[pos] = (uint32_t)t;
            tpo[pos] = (uint32_t)(excl & ((1ull << 40) - 1));
        }
        __syncthreads();
        if (threadIdx.x == 0) carry_s += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const uint32_t kk = (uint32_t)(carry_s >> 40), nn = (uint32_t)(carry_s & ((1ull << 40) - 1));
        tpo[kk] = nn;
        kn_dev[0] = (int32_t)kk;
        kn_dev[1] = (int32_t)nn;
    }
}

// One warp per selected tile: expand the keep mask into global pixel indices, ascending local index.
__global__ void __launch_bounds__(256)
write_pix_kernel(const CamK cam, int k, const uint32_t* __restrict__ tiles, const uint32_t* __restrict__ tpo,
                 const TileMeta* __restrict__ meta, uint32_t* __restrict__ pix) {
    const int i = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (i >= k) return;
    const int lane = threadIdx.x & 31;
    const uint32_t t = tiles[i];
    const int tx = t % cam.gx, ty = t / cam.gx;
    const uint32_t word = meta[t].mask[lane >> 2];
    const uint32_t bits = (word >> ((lane & 3) * 8)) & 0xffu;
    const uint32_t c = __popc(bits);
    uint32_t x = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t yv = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += yv;
    }
    uint32_t o = tpo[i] + (x - c);
    const int y = ty * kTile + (lane >> 1);
    const int xb = tx * kTile + (lane & 1) * 8;
#pragma unroll
    for (int j = 0; j < 8; ++j)
        if (bits & (1u << j)) pix[o++] = (uint32_t)(y * cam.W + xb + j);
}

// ---- f2: the paper's own sampler (Sec. 3.5 Eq. 7-8) and its maps (Eq. 3-4) ----
// One warp per tile, every tile sampled.  Lane l owns local pixels 8l .. 8l+7.  All decisions are integer
// (R26-R29): weight q = 1 + trunc(min(E, 15.999) * 2^16) from the fp16 error map; hard draw d takes
// the pixel whose running sum of q first exceeds mix64(seed, t << 16 | d) mod (sum of remaining q) and removes
// it (sequential multinomial sampling without replacement: a warp scan per draw); the stable set is the TopK of
// the age map over the rest (a warp max per pick; ties: lower local index); the remainder is uniform.
__device__ __forceinline__ uint32_t half_weight(uint16_t h) {
    float e = __half2float(__ushort_as_half(h));
    if (!(e > 0.0f)) return 1u;  // zero, negative, NaN
    e = fminf(e, kErrClamp);
    return 1u + (uint32_t)(e * 65536.0f);
}

__device__ __forceinline__ uint32_t warp_incl_scan_u32(uint32_t v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += y;
    }
    return v;
}

__global__ void __launch_bounds__(256)
paper_tile_kernel(const CamK cam, const uint16_t* __restrict__ E_half, const uint16_t* __restrict__ age, int n_pix,
                  int n_hard, int n_stable, uint64_t seed, TileMeta* __restrict__ meta, uint32_t* __restrict__ selected) {
    const int T = cam.gx * cam.gy;
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= T) return;
    const int lane = threadIdx.x & 31;
    const int tx = t % cam.gx, ty = t / cam.gx;
    const int y = ty * kTile + (lane >> 1), xb = tx * kTile + (lane & 1) * 8;
    uint32_t q[8], ag[8];
    uint32_t avail = 0;  // bit j: pixel j of this lane is inside the image and not chosen yet
#pragma unroll
    for (int j = 0; j < 8; ++j) {
        q[j] = 0u; ag[j] = 0u;
        if (y < cam.H && xb + j < cam.W) {
            const size_t p = (size_t)y * cam.W + xb + j;
            q[j] = half_weight(E_half[p]);
            ag[j] = age[p];
            avail |= 1u << j;
        }
    }
    uint32_t chosen = 0;
    const int cnt = (int)__reduce_add_sync(0xffffffffu, (uint32_t)__popc(avail));
    const int N = min(n_pix, cnt), Nh = min(n_hard, N), Ns = min(n_stable, N - Nh), Nr = N - Nh - Ns;
    const uint64_t tkey = (uint64_t)(uint32_t)t << 16;
    // ---- Eq. 7: hard pixels ----
    for (int d = 0; d < Nh; ++d) {
        uint32_t sum = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j) sum += ((avail >> j) & 1u) ? q[j] : 0u;
        const uint32_t incl = warp_incl_scan_u32(sum, lane);
        const uint32_t S = __shfl_sync(0xffffffffu, incl, 31);
        const uint32_t r = (uint32_t)(mix64(seed, tkey | (uint64_t)d) % (uint64_t)S);
        uint32_t acc = incl - sum;
        if (r >= acc && r < incl) {  // exactly one lane
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                if ((avail >> j) & 1u) {
                    acc += q[j];
                    if (r < acc) { avail &= ~(1u << j); chosen |= 1u << j; acc = 0xffffffffu; break; }
                }
            }
        }
    }
    // ---- Eq. 8: the oldest of the rest ----
    for (int d = 0; d < Ns; ++d) {
        uint32_t best = 0;  // (age + 1) << 8 | 255 - local index; 0 = nothing available
#pragma unroll
        for (int j = 0; j < 8; ++j)
            if ((avail >> j) & 1u) best = max(best, ((ag[j] + 1u) << 8) | (uint32_t)(255 - (lane * 8 + j)));
        const uint32_t win = __reduce_max_sync(0xffffffffu, best);
        const int l = 255 - (int)(win & 255u);
        if ((l >> 3) == lane) { avail &= ~(1u << (l & 7)); chosen |= 1u << (l & 7); }
    }
    // ---- remainder: uniform over what is left ----
    for (int d = 0; d < Nr; ++d) {
        const uint32_t c = (uint32_t)__popc(avail);
        const uint32_t incl = warp_incl_scan_u32(c, lane);
        const uint32_t R = __shfl_sync(0xffffffffu, incl, 31);
        const uint32_t r = (uint32_t)(mix64(seed ^ 0x5bd1e995a5a5a5a5ull, tkey | (uint64_t)d) % (uint64_t)R);
        const uint32_t excl = incl - c;
        if (r >= excl && r < incl) {
            const int j = __fns(avail, 0, (int)(r - excl) + 1);  // the (r - excl)-th set bit
            avail &= ~(1u << j);
            chosen |= 1u << j;
        }
    }
    // keep mask: word w holds local indices 32w .. 32w+31 = the bytes of lanes 4w .. 4w+3
    uint32_t v = chosen << ((lane & 3) * 8);
    v |= __shfl_xor_sync(0xffffffffu, v, 1);
    v |= __shfl_xor_sync(0xffffffffu, v, 2);
    if ((lane & 3) == 0) meta[t].mask[lane >> 2] = v;
    if (lane == 0) { meta[t].npix = (uint32_t)N; selected[t] = 1u; }
}

// Eq. 4: every age + 1 (saturating at 65535); the sampled pixels are reset by maps_sampled_kernel
__global__ void __launch_bounds__(256) age_increment_kernel(size_t npix, uint16_t* __restrict__ age) {
    for (size_t p = (size_t)blockIdx.x * blockDim.x + threadIdx.x; p < npix; p += (size_t)gridDim.x * blockDim.x) {
        const uint16_t a = age[p];
        if (a != 0xffffu) age[p] = (uint16_t)(a + 1u);
    }
}

// Eq. 3 at the sampled pixels: E <- fp16((1 - beta) E + beta e), three fp32 roundings; age <- 0
__global__ void __launch_bounds__(256)
maps_sampled_kernel(const int32_t* __restrict__ kn_dev, const uint32_t* __restrict__ pix, const float* __restrict__ pix_err,
                    float beta, uint16_t* __restrict__ E_half, uint16_t* __restrict__ age) {
    const int n = kn_dev[1];
    const float omb = __fsub_rn(1.0f, beta);
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const uint32_t p = pix[i];
        const float a = __fmul_rn(omb, __half2float(__ushort_as_half(E_half[p])));
        const float b = __fmul_rn(beta, pix_err[i]);
        E_half[p] = __half_as_ushort(__float2half_rn(__fadd_rn(a, b)));
        age[p] = 0;
    }
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

size_t sample_workspace_bytes(int T) {
    return align256((size_t)T * sizeof(TileMeta)) + align256((size_t)T * 4);
}

cudaError_t launch_sample(const CamK& cam, const float* err, const float* render, const float* target, int k,
                          int mode, int rnum, int rden, uint64_t seed, uint64_t* tile_score, uint32_t* tiles,
                          uint32_t* tpo, uint32_t* pix, uint32_t* tile_select, int32_t* kn_dev, void* ws,
                          cudaStream_t s) {
    const int T = cam.gx * cam.gy;
    TileMeta* meta = (TileMeta*)ws;
    uint32_t* selected = tile_select ? tile_select : (uint32_t*)((char*)ws + align256((size_t)T * sizeof(TileMeta)));
    tile_reduce_kernel<<<(T + 7) / 8, 256, 0, s>>>(cam, err, render, target, mode, rnum, rden, seed, tile_score, meta);
    tile_select_compact_kernel<<<1, 1024, 0, s>>>(T, k, tile_score, meta, selected, tiles, tpo, kn_dev);
    write_pix_kernel<<<(k + 7) / 8, 256, 0, s>>>(cam, k, tiles, tpo, meta, pix);
    count_launches(3);
    return cudaGetLastError();
}

// ---- tgs_sample_static: the same three kernels, scratch in g_sample_static_scratch ----
namespace {

constexpr int kStaticMaxTiles = TGS_SAMPLE_STATIC_MAX_TILES;
static_assert(sizeof(TileMeta) == 36, "TileMeta is 36 B per tile");
static_assert(((size_t)kStaticMaxTiles * sizeof(TileMeta) + 255) / 256 * 256 + ((size_t)kStaticMaxTiles * 4 + 255) / 256 * 256
                  <= kStaticScratchBytes, "static scratch too small for TGS_SAMPLE_STATIC_MAX_TILES");

constexpr int kStaticDevSlots = 64;
std::atomic<void*> g_static_scratch_dev[kStaticDevSlots];  // device address of the array on device d, once resolved

// Device address of g_sample_static_scratch on `device`, which must be the current device.  Every GPU has its own
// copy of the array, so the address is looked up once per device and remembered (two threads racing here both get
// the same answer).  The look-up may load the library's device code on that GPU: that is the set-up step the header
// asks callers to get out of the way before they start capturing a stream.
cudaError_t static_scratch_on(int device, void** out) {
    void* p = device < kStaticDevSlots ? g_static_scratch_dev[device].load(std::memory_order_acquire) : nullptr;
    if (!p) {
        cudaError_t e = cudaGetSymbolAddress(&p, g_sample_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        if (device < kStaticDevSlots) g_static_scratch_dev[device].store(p, std::memory_order_release);
    }
    *out = p;
    return cudaSuccess;
}

}  // namespace

int sample_static_max_tiles() { return kStaticMaxTiles; }

// Same launches as launch_sample, scratch = the static array.  Nothing in the scratch has to start at zero: for the
// T tiles of this call, tile_reduce_kernel writes all nine words of meta[t] and tile_select_compact_kernel writes
// selected[t] before any kernel reads them, and no kernel reads beyond tile T-1, so whatever an earlier (possibly
// larger) call left behind is never seen.
cudaError_t launch_sample_static(int device, const CamK& cam, const float* err, const float* render, const float* target,
                                 int k, int mode, int rnum, int rden, uint64_t seed, uint64_t* tile_score,
                                 uint32_t* tiles, uint32_t* tpo, uint32_t* pix, uint32_t* tile_select, int32_t* kn_dev,
                                 cudaStream_t s) {
    const int T = cam.gx * cam.gy;
    if (T > kStaticMaxTiles) return cudaErrorInvalidValue;  // the ABI glue has already said so in words
    void* ws = nullptr;
    cudaError_t e = static_scratch_on(device, &ws);
    if (e != cudaSuccess) return e;
    TileMeta* meta = (TileMeta*)ws;
    uint32_t* selected = tile_select ? tile_select : (uint32_t*)((char*)ws + align256((size_t)kStaticMaxTiles * sizeof(TileMeta)));
    tile_reduce_kernel<<<(T + 7) / 8, 256, 0, s>>>(cam, err, render, target, mode, rnum, rden, seed, tile_score, meta);
    tile_select_compact_kernel<<<1, 1024, 0, s>>>(T, k, tile_score, meta, selected, tiles, tpo, kn_dev);
    write_pix_kernel<<<(k + 7) / 8, 256, 0, s>>>(cam, k, tiles, tpo, meta, pix);
    count_launches(3);
    return cudaGetLastError();
}

cudaError_t launch_sample_paper(const CamK& cam, const uint16_t* E_half, const uint16_t* age, int n_pix, int n_hard,
                                int n_stable, uint64_t seed, uint32_t* tiles, uint32_t* tpo, uint32_t* pix,
                                int32_t* kn_dev, void* ws, cudaStream_t s) {
    const int T = cam.gx * cam.gy;
    TileMeta* meta = (TileMeta*)ws;
    uint32_t* selected = (uint32_t*)((char*)ws + align256((size_t)T * sizeof(TileMeta)));
    paper_tile_kernel<<<(T + 7) / 8, 256, 0, s>>>(cam, E_half, age, n_pix, n_hard, n_stable, seed, meta, selected);
    tile_compact_kernel<<<1, 1024, 0, s>>>(T, selected, meta, tiles, tpo, kn_dev);
    write_pix_kernel<<<(T + 7) / 8, 256, 0, s>>>(cam, T, tiles, tpo, meta, pix);
    count_launches(3);
    return cudaGetLastError();
}

cudaError_t launch_maps_update(const CamK& cam, uint16_t* E_half, uint16_t* age, const int32_t* kn_dev,
                               const uint32_t* pix, const float* pix_err, float beta, int num_sms, cudaStream_t s) {
    const size_t npix = (size_t)cam.W * (size_t)cam.H;
    int blocks = (int)((npix + 255) / 256);
    if (blocks > num_sms * 16) blocks = num_sms * 16;
    age_increment_kernel<<<blocks, 256, 0, s>>>(npix, age);
    maps_sampled_kernel<<<blocks, 256, 0, s>>>(kn_dev, pix, pix_err, beta, E_half, age);
    count_launches(2);
    return cudaGetLastError();
}

}  // namespace tgs
