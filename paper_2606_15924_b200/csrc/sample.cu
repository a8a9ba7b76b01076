// tgs_sample: per-tile error reduction, top-k tile selection and tile-ordered sampled-pixel
// lists ("sampled pixels are ordered by their tile indices",
// 93 Eq. 2, 128-150 Sec. 3.5, 156 "tile-wise pixel offsets via prefix-sum").  Selection is done in
// integers on a fixed-point copy of the error so that it is order independent and bit exact.
#include "common.cuh"

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

// rank by counting: tile t is selected iff fewer than k tiles precede it in the order
// (score descending, tile id ascending).  One warp per tile, lanes stride over all T scores:
// O(T^2) compares spread over the whole GPU, no sort needed for T of a few thousand.
__global__ void __launch_bounds__(256)
tile_select_kernel(int T, int k, const uint64_t* __restrict__ tile_score, uint32_t* __restrict__ selected) {
    const int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (t >= T) return;
    const int lane = threadIdx.x & 31;
    const uint64_t mine = tile_score[t];
    uint32_t rank = 0;
    for (int j = lane; j < T; j += 32) {
        const uint64_t o = __ldg(tile_score + j);
        rank += (o > mine || (o == mine && j < t)) ? 1u : 0u;
    }
    rank = __reduce_add_sync(0xffffffffu, rank);
    if (lane == 0) selected[t] = rank < (uint32_t)k ? 1u : 0u;
}

// single block: compaction of the selected tiles (ascending id) and exclusive prefix sum of their
// pixel counts.  A 64-bit scan carries both: count << 40 | pixels.
__global__ void __launch_bounds__(1024)
tile_compact_kernel(int T, const uint32_t* __restrict__ selected, const TileMeta* __restrict__ meta,
                    uint32_t* __restrict__ tiles, uint32_t* __restrict__ tpo, int32_t* __restrict__ kn_dev) {
    __shared__ uint64_t wsum[33];
    __shared__ uint64_t carry_s;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry_s = 0;
    __syncthreads();
    for (int b0 = 0; b0 < T; b0 += 1024) {
        const int t = b0 + threadIdx.x;
        const bool sel = t < T && selected[t];
        const uint64_t v = sel ? ((1ull << 40) | (uint64_t)meta[t].npix) : 0ull;
        uint64_t x = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint64_t yv = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += yv;
        }
        if (lane == 31) wsum[warp] = x;
        __syncthreads();
        if (warp == 0) {
            uint64_t w = wsum[lane], xs = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                uint64_t yv = __shfl_up_sync(0xffffffffu, xs, o);
                if (lane >= o) xs += yv;
            }
            wsum[lane] = xs - w;
            if (lane == 31) wsum[32] = xs;
        }
        __syncthreads();
        const uint64_t excl = carry_s + wsum[warp] + (x - v);
        if (sel) {
            const uint32_t pos = (uint32_t)(excl >> 40);
            tiles[pos] = (uint32_t)t;
            tpo[pos] = (uint32_t)(excl & ((1ull << 40) - 1));
        }
        __syncthreads();
        if (threadIdx.x == 0) carry_s += wsum[32];
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
    tile_select_kernel<<<(T + 7) / 8, 256, 0, s>>>(T, k, tile_score, selected);
    tile_compact_kernel<<<1, 1024, 0, s>>>(T, selected, meta, tiles, tpo, kn_dev);
    write_pix_kernel<<<(k + 7) / 8, 256, 0, s>>>(cam, k, tiles, tpo, meta, pix);
    count_launches(4);
    return cudaGetLastError();
}

}  // namespace tgs
