// tgs_bin_sort: tile-overlap duplication, hand-written stable LSD radix sort on (tile, depth)
// keys, per-tile CSR ranges ("K(p) ... sorted by depth").
//
// The 64-bit key is tile_id<<32 | float_bits(depth).  Its low 32 bits depend on the Gaussian
// only, so the four depth-digit passes of the LSD sort run on the N Gaussians BEFORE
// duplication; duplication then emits pairs in depth order and only the tile-id digits
// (ceil(log2 T) bits, two passes) run on the P pairs.  LSD stability makes the result identical
// to sorting all 64-bit keys: order = (tile_id, depth bits, Gaussian id).
//
// Every kernel reads its element count from device memory (P is data dependent), so the whole
// call is asynchronous and graph-capturable.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kRadixThreads = 256;
constexpr int kRadixIPT = 16;
constexpr int kRadixItems = kRadixThreads * kRadixIPT;  // 4096 items per block
constexpr int kScanThreads = 1024;

__device__ __forceinline__ int64_t eff_count(const int64_t* n_dev, int64_t n_host) {
    if (n_dev == nullptr) return n_host;
    return n_dev[1] ? 0 : n_dev[0];  // overflow -> process nothing
}

__device__ __forceinline__ uint32_t warp_excl_scan(uint32_t v, uint32_t& total) {
    const int lane = threadIdx.x & 31;
    uint32_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    total = __shfl_sync(0xffffffffu, x, 31);
    return x - v;
}

// Block-wide exclusive scan of one value per thread (blockDim.x multiple of 32, <= 1024).
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* smem33, uint32_t& block_total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    uint32_t wt;
    uint32_t e = warp_excl_scan(v, wt);
    if (lane == 31) smem33[warp] = wt;
    __syncthreads();
    if (warp == 0) {
        uint32_t t = lane < nw ? smem33[lane] : 0, tt;
        uint32_t ex = warp_excl_scan(t, tt);
        smem33[lane] = ex;
        if (lane == 0) smem33[32] = tt;
    }
    __syncthreads();
    uint32_t r = e + smem33[warp];
    block_total = smem33[32];
    __syncthreads();
    return r;
}

// ---- step A: depth keys of the N Gaussians -------------------------------------------------
__global__ void depth_keys_kernel(int N, const float4* __restrict__ splats, uint32_t* __restrict__ keys,
                                  uint32_t* __restrict__ vals) {
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float4 r2 = splats[3 * (size_t)i + 2];
    int x0, y0, x1, y1;
    unpack_rect(__float_as_uint(r2.z), __float_as_uint(r2.w), x0, y0, x1, y1);
    bool vis = (x1 - x0) > 0 && (y1 - y0) > 0;
    keys[i] = vis ? __float_as_uint(r2.y) : 0xffffffffu;  // depth > 0: raw bits order like the value
    vals[i] = (uint32_t)i;
}

// ---- one LSD radix pass = histogram, per-digit scan, stable scatter --------------------------
__global__ void __launch_bounds__(kRadixThreads)
radix_hist_kernel(const uint32_t* __restrict__ keys, const int64_t* n_dev, int64_t n_host, int shift,
                  uint32_t mask, uint32_t* __restrict__ hist /* [256][gridDim.x] */) {
    __shared__ uint32_t h[256];
    const int64_t n = eff_count(n_dev, n_host);
    const int64_t base = (int64_t)blockIdx.x * kRadixItems;
    if (base >= n) return;  // columns >= ceil(n/items) are never read
    h[threadIdx.x] = 0;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kRadixIPT; ++i) {
        int64_t idx = base + (int64_t)i * kRadixThreads + threadIdx.x;
        if (idx < n) atomicAdd(&h[(keys[idx] >> shift) & mask], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x] = h[threadIdx.x];
}

// One block per digit: exclusive scan of that digit's per-block counts; total -> digit_tot.
__global__ void __launch_bounds__(kScanThreads)
radix_scan_kernel(uint32_t* __restrict__ hist, int stride, const int64_t* n_dev, int64_t n_host,
                  uint32_t* __restrict__ digit_tot) {
    __shared__ uint32_t sm[33];
    const int64_t n = eff_count(n_dev, n_host);
    const int nb = (int)((n + kRadixItems - 1) / kRadixItems);
    uint32_t* row = hist + (size_t)blockIdx.x * stride;
    uint32_t carry = 0;
    for (int b0 = 0; b0 < nb; b0 += kScanThreads) {
        int b = b0 + threadIdx.x;
        uint32_t v = b < nb ? row[b] : 0, tot;
        uint32_t e = block_excl_scan(v, sm, tot);
        if (b < nb) row[b] = carry + e;
        carry += tot;
    }
    if (threadIdx.x == 0) digit_tot[blockIdx.x] = carry;
}

__global__ void __launch_bounds__(kRadixThreads)
radix_scatter_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                     uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, const int64_t* n_dev,
                     int64_t n_host, int shift, uint32_t mask, const uint32_t* __restrict__ hist,
                     const uint32_t* __restrict__ digit_tot) {
    __shared__ uint32_t wcnt[kRadixThreads / 32][256];
    __shared__ uint32_t gbase[256];
    __shared__ uint32_t sm[33];
    const int64_t n = eff_count(n_dev, n_host);
    const int64_t base = (int64_t)blockIdx.x * kRadixItems;
    if (base >= n) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    // digit base = exclusive scan of the 256 digit totals
    {
        uint32_t tot;
        uint32_t e = block_excl_scan(digit_tot[threadIdx.x], sm, tot);
        gbase[threadIdx.x] = e + hist[(size_t)threadIdx.x * gridDim.x + blockIdx.x];
    }
#pragma unroll
    for (int w = 0; w < kRadixThreads / 32; ++w) wcnt[w][threadIdx.x] = 0;
    __syncthreads();

    uint32_t key[kRadixIPT], val[kRadixIPT], rnk[kRadixIPT];
    const int64_t wbase = base + (int64_t)warp * (32 * kRadixIPT);
#pragma unroll
    for (int i = 0; i < kRadixIPT; ++i) {
        const int64_t idx = wbase + i * 32 + lane;
        const bool valid = idx < n;
        key[i] = valid ? keys_in[idx] : 0u;
        val[i] = valid ? vals_in[idx] : 0u;
        const uint32_t d = valid ? ((key[i] >> shift) & mask) : 256u;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (lane == leader && valid) {
            old = wcnt[warp][d];
            wcnt[warp][d] = old + __popc(peers);
        }
        old = __shfl_sync(0xffffffffu, old, leader);
        rnk[i] = old + __popc(peers & ((1u << lane) - 1u));
        __syncwarp();
    }
    __syncthreads();
    {   // per-digit exclusive scan across the warps of this block
        uint32_t run = 0;
#pragma unroll
        for (int w = 0; w < kRadixThreads / 32; ++w) {
            uint32_t c = wcnt[w][threadIdx.x];
            wcnt[w][threadIdx.x] = run;
            run += c;
        }
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < kRadixIPT; ++i) {
        const int64_t idx = wbase + i * 32 + lane;
        if (idx < n) {
            const uint32_t d = (key[i] >> shift) & mask;
            const uint32_t dst = gbase[d] + wcnt[warp][d] + rnk[i];
            keys_out[dst] = key[i];
            vals_out[dst] = val[i];
        }
    }
}

// ---- step B: tiles touched in depth order, exclusive scan ------------------------------------
__global__ void __launch_bounds__(kScanThreads)
counts_kernel(int N, const uint32_t* __restrict__ order, const float4* __restrict__ splats,
              uint32_t* __restrict__ cnt, uint32_t* __restrict__ bsum) {
    __shared__ uint32_t sm[33];
    int r = blockIdx.x * kScanThreads + threadIdx.x;
    uint32_t c = 0;
    if (r < N) {
        const float2 rc = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(splats) +
                                                             (size_t)order[r] * kSplatWords + 10);
        int x0, y0, x1, y1;
        unpack_rect(__float_as_uint(rc.x), __float_as_uint(rc.y), x0, y0, x1, y1);
        c = (uint32_t)((x1 - x0) * (y1 - y0));
        cnt[r] = c;
    }
    uint32_t tot;
    block_excl_scan(c, sm, tot);
    if (threadIdx.x == 0) bsum[blockIdx.x] = tot;
}

// single block: exclusive scan of the block sums (64-bit running total), writes P and the overflow flag
__global__ void __launch_bounds__(kScanThreads)
bsum_scan_kernel(int nb, uint32_t* __restrict__ bsum, int64_t Pcap, int64_t* __restrict__ P_dev) {
    __shared__ uint32_t sm[33];
    __shared__ unsigned long long carry_s;
    if (threadIdx.x == 0) carry_s = 0ull;
    __syncthreads();
    for (int b0 = 0; b0 < nb; b0 += kScanThreads) {
        int b = b0 + threadIdx.x;
        uint32_t v = b < nb ? bsum[b] : 0, tot;
        uint32_t e = block_excl_scan(v, sm, tot);
        unsigned long long c = carry_s;
        // offsets are 32-bit: a total beyond capacity (< 2^32) is flagged below and nothing is written
        if (b < nb) bsum[b] = (uint32_t)(c + e);
        __syncthreads();
        if (threadIdx.x == 0) carry_s = c + tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        P_dev[0] = (int64_t)carry_s;
        P_dev[1] = ((int64_t)carry_s > Pcap) ? 1 : 0;
    }
}

__global__ void __launch_bounds__(kScanThreads)
offsets_kernel(int N, const uint32_t* __restrict__ cnt, const uint32_t* __restrict__ bsum,
               uint32_t* __restrict__ off) {
    __shared__ uint32_t sm[33];
    int r = blockIdx.x * kScanThreads + threadIdx.x;
    uint32_t c = r < N ? cnt[r] : 0, tot;
    uint32_t e = block_excl_scan(c, sm, tot);
    if (r < N) off[r] = bsum[blockIdx.x] + e;
}

// ---- step C: duplication, in depth order -----------------------------------------------------
__global__ void duplicate_kernel(int N, int gx, const uint32_t* __restrict__ order,
                                 const uint32_t* __restrict__ off, const float4* __restrict__ splats,
                                 const int64_t* __restrict__ P_dev, uint32_t* __restrict__ tkey,
                                 uint32_t* __restrict__ tval) {
    int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= N || P_dev[1]) return;
    const uint32_t g = order[r];
    const float2 rc = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(splats) +
                                                         (size_t)g * kSplatWords + 10);
    int x0, y0, x1, y1;
    unpack_rect(__float_as_uint(rc.x), __float_as_uint(rc.y), x0, y0, x1, y1);
    uint32_t o = off[r];
    for (int ty = y0; ty < y1; ++ty)
        for (int tx = x0; tx < x1; ++tx) {
            tkey[o] = (uint32_t)(ty * gx + tx);
            tval[o] = g;
            ++o;
        }
}

// ---- step E: CSR ranges from the sorted tile ids ---------------------------------------------
__global__ void ranges_kernel(const uint32_t* __restrict__ tkey, const int64_t* __restrict__ P_dev, int T,
                              uint32_t* __restrict__ tile_offsets) {
    const int64_t P = eff_count(P_dev, 0);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j <= P; j += stride) {
        // tiles in (prev, cur] start at j
        const int64_t prev = j > 0 ? (int64_t)tkey[j - 1] : -1;
        const int64_t cur = j < P ? (int64_t)tkey[j] : (int64_t)T;
        for (int64_t t = prev + 1; t <= cur; ++t) tile_offsets[t] = (uint32_t)j;
    }
}

__global__ void keys64_kernel(const uint32_t* __restrict__ tkey, const uint32_t* __restrict__ gid,
                              const float4* __restrict__ splats, const int64_t* __restrict__ P_dev,
                              uint64_t* __restrict__ keys_sorted) {
    const int64_t P = eff_count(P_dev, 0);
    const int64_t stride = (int64_t)gridDim.x * blockDim.x;
    for (int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; j < P; j += stride) {
        const float d = reinterpret_cast<const float*>(splats)[(size_t)gid[j] * kSplatWords + 9];
        keys_sorted[j] = ((uint64_t)tkey[j] << 32) | (uint64_t)__float_as_uint(d);
    }
}

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Workspace {
    uint32_t *kA, *vA, *kB, *vB;   // N-sized ping-pong for the depth sort
    uint32_t *cnt, *off, *bsum;    // N, N, ceil(N/1024)
    uint32_t *tkA, *tkB, *tvB;     // Pcap-sized: tile keys ping-pong, second value buffer
    uint32_t *hist, *dtot;         // 256 * max blocks, 256
    size_t total;
};

Workspace carve(void* base, int N, int64_t Pcap) {
    Workspace w;
    size_t o = 0;
    char* p = (char*)base;
    auto take = [&](size_t bytes) { uint32_t* r = (uint32_t*)(p + o); o += align256(bytes); return r; };
    const size_t n = (size_t)(N > 0 ? N : 1), pc = (size_t)(Pcap > 0 ? Pcap : 1);
    w.kA = take(n * 4); w.vA = take(n * 4); w.kB = take(n * 4); w.vB = take(n * 4);
    w.cnt = take(n * 4); w.off = take(n * 4); w.bsum = take(((n + kScanThreads - 1) / kScanThreads) * 4);
    w.tkA = take(pc * 4); w.tkB = take(pc * 4); w.tvB = take(pc * 4);
    const size_t maxItems = n > pc ? n : pc;
    const size_t nb = (maxItems + kRadixItems - 1) / kRadixItems;
    w.hist = take(256 * nb * 4); w.dtot = take(256 * 4);
    w.total = o;
    return w;
}

void radix_pass(const uint32_t* kin, const uint32_t* vin, uint32_t* kout, uint32_t* vout, const int64_t* n_dev,
                int64_t n_host_or_cap, int shift, int bits, const Workspace& w, cudaStream_t s) {
    const int nb = (int)((n_host_or_cap + kRadixItems - 1) / kRadixItems);
    if (nb == 0) return;
    const uint32_t mask = (1u << bits) - 1u;
    radix_hist_kernel<<<nb, kRadixThreads, 0, s>>>(kin, n_dev, n_host_or_cap, shift, mask, w.hist);
    radix_scan_kernel<<<256, kScanThreads, 0, s>>>(w.hist, nb, n_dev, n_host_or_cap, w.dtot);
    radix_scatter_kernel<<<nb, kRadixThreads, 0, s>>>(kin, vin, kout, vout, n_dev, n_host_or_cap, shift, mask,
                                                      w.hist, w.dtot);
    count_launches(3);
}

}  // namespace

size_t binsort_workspace_bytes(int N, int64_t Pcap, int T) {
    (void)T;
    return carve(nullptr, N, Pcap).total;
}

cudaError_t launch_bin_sort(const CamK& cam, int N, const float* splats_f, int64_t Pcap, uint64_t* keys_sorted,
                            uint32_t* gid_sorted, uint32_t* tile_offsets, int64_t* P_dev, void* ws,
                            size_t ws_bytes, int num_sms, cudaStream_t s) {
    (void)ws_bytes;
    const Workspace w = carve(ws, N, Pcap);
    const float4* splats = reinterpret_cast<const float4*>(splats_f);
    const int T = cam.gx * cam.gy;

    // A: depth sort of the Gaussians (4 x 8-bit passes, ends in kA/vA)
    depth_keys_kernel<<<(N + 255) / 256, 256, 0, s>>>(N, splats, w.kA, w.vA);
    radix_pass(w.kA, w.vA, w.kB, w.vB, nullptr, N, 0, 8, w, s);
    radix_pass(w.kB, w.vB, w.kA, w.vA, nullptr, N, 8, 8, w, s);
    radix_pass(w.kA, w.vA, w.kB, w.vB, nullptr, N, 16, 8, w, s);
    radix_pass(w.kB, w.vB, w.kA, w.vA, nullptr, N, 24, 8, w, s);

    // B: tiles touched per Gaussian in depth order -> exclusive offsets, P
    const int nbs = (N + kScanThreads - 1) / kScanThreads;
    counts_kernel<<<nbs, kScanThreads, 0, s>>>(N, w.vA, splats, w.cnt, w.bsum);
    bsum_scan_kernel<<<1, kScanThreads, 0, s>>>(nbs, w.bsum, Pcap, P_dev);
    offsets_kernel<<<nbs, kScanThreads, 0, s>>>(N, w.cnt, w.bsum, w.off);

    // C + D: duplicate in depth order, then stable sort on the tile-id bits only
    int tbits = 1;
    while ((1 << tbits) < T) ++tbits;
    const int npass = (tbits + 7) / 8;
    const int bits_per = (tbits + npass - 1) / npass;
    // ping-pong (tkA, gid_sorted) <-> (tkB, tvB); start so that the result lands in (tkA, gid_sorted)
    uint32_t* k0 = (npass % 2 == 0) ? w.tkA : w.tkB;
    uint32_t* v0 = (npass % 2 == 0) ? gid_sorted : w.tvB;
    uint32_t* k1 = (npass % 2 == 0) ? w.tkB : w.tkA;
    uint32_t* v1 = (npass % 2 == 0) ? w.tvB : gid_sorted;
    duplicate_kernel<<<(N + 127) / 128, 128, 0, s>>>(N, cam.gx, w.vA, w.off, splats, P_dev, k0, v0);
    for (int p = 0; p < npass; ++p) {
        radix_pass(k0, v0, k1, v1, P_dev, Pcap, p * bits_per, bits_per, w, s);
        uint32_t* tk = k0; k0 = k1; k1 = tk;
        uint32_t* tv = v0; v0 = v1; v1 = tv;
    }
    // E: CSR ranges (+ optional 64-bit keys)
    const int rb = num_sms * 8;
    ranges_kernel<<<rb, 256, 0, s>>>(w.tkA, P_dev, T, tile_offsets);
    if (keys_sorted) keys64_kernel<<<rb, 256, 0, s>>>(w.tkA, gid_sorted, splats, P_dev, keys_sorted);
    count_launches(6 + (keys_sorted ? 1 : 0));  // depth_keys, counts, bsum_scan, offsets, duplicate, ranges
    return cudaGetLastError();
}

}  // namespace tgs
