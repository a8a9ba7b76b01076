// tgs_bin_sort: tile-overlap duplication, hand-written stable LSD radix sort on (tile, depth)
// keys, per-tile CSR ranges ("K(p) ... sorted by depth").
//
// The 64-bit key is tile_id<<32 | float_bits(depth).  Its low 32 bits depend on the Gaussian
// only, so the four depth-digit passes of the LSD sort run on the N Gaussians BEFORE
// duplication; duplication then emits pairs in depth order and only the tile-id digits
// (ceil(log2 T) bits, two passes) run on the P pairs.  LSD stability makes the result identical
// to sorting all 64-bit keys: order = (tile_id, depth bits, Gaussian id).
//
// Each radix pass is ONE kernel ("onesweep"): digit histograms of all passes are accumulated up
// front (fused into key generation / duplication), and the pass itself ranks its block's keys
// (warp match-any ranking, stable), obtains the block's per-digit global offset by decoupled
// look-back over the status words of the preceding blocks (blocks take their index from an atomic
// ticket, so every predecessor is resident: no deadlock) and scatters.  The exclusive scan of the
// tiles-touched counts uses the same look-back.  11 launches per call instead of 24.
//
// Every kernel reads its element count from device memory (P is data dependent), so the whole
// call is asynchronous and graph-capturable.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kRadixThreads = 256;
constexpr int kScanThreads = 1024;
constexpr uint32_t kFlagAgg = 1u << 30, kFlagIncl = 2u << 30, kValMask = (1u << 30) - 1u;

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

__device__ __forceinline__ uint32_t ld_volatile(const uint32_t* p) { return *reinterpret_cast<const volatile uint32_t*>(p); }
__device__ __forceinline__ void st_volatile(uint32_t* p, uint32_t v) { *reinterpret_cast<volatile uint32_t*>(p) = v; }

// ---- step A: depth keys of the N Gaussians + histograms of the four depth digits ------------
__global__ void __launch_bounds__(256)
depth_keys_kernel(int N, const float4* __restrict__ splats, uint32_t* __restrict__ keys,
                  uint32_t* __restrict__ vals, uint32_t* __restrict__ ghist /* [4][256] */) {
    __shared__ uint32_t h[4][256];
#pragma unroll
    for (int p = 0; p < 4; ++p) h[p][threadIdx.x] = 0;
    __syncthreads();
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        float4 r2 = splats[3 * (size_t)i + 2];
        int x0, y0, x1, y1;
        unpack_rect(__float_as_uint(r2.z), __float_as_uint(r2.w), x0, y0, x1, y1);
        const bool vis = (x1 - x0) > 0 && (y1 - y0) > 0;
        const uint32_t key = vis ? __float_as_uint(r2.y) : 0xffffffffu;  // depth > 0: raw bits order like the value
        keys[i] = key;
        vals[i] = (uint32_t)i;
#pragma unroll
        for (int p = 0; p < 4; ++p) atomicAdd(&h[p][(key >> (8 * p)) & 255u], 1u);
    }
    __syncthreads();
#pragma unroll
    for (int p = 0; p < 4; ++p) {
        const uint32_t c = h[p][threadIdx.x];
        if (c) atomicAdd(&ghist[p * 256 + threadIdx.x], c);
    }
}

// ---- one LSD radix pass in one kernel --------------------------------------------------------
// status[b][d]: 2 flag bits | 30-bit count.  ticket: dynamic block index.
template <int IPT>
__global__ void __launch_bounds__(kRadixThreads)
onesweep_kernel(const uint32_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                uint32_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, const int64_t* n_dev,
                int64_t n_host, int shift, uint32_t mask, const uint32_t* __restrict__ ghist /* [256] */,
                uint32_t* __restrict__ status, uint32_t* __restrict__ ticket) {
    constexpr int kItems = kRadixThreads * IPT;
    __shared__ uint32_t wcnt[kRadixThreads / 32][256];
    __shared__ uint32_t gbase[256];
    __shared__ uint32_t sm[33];
    __shared__ uint32_t s_block;
    const int64_t n = eff_count(n_dev, n_host);
    if (threadIdx.x == 0) s_block = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t b = s_block;
    const int64_t base = (int64_t)b * kItems;
    if (base >= n) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t digit_base;
    {
        uint32_t tot;
        digit_base = block_excl_scan(ghist[threadIdx.x], sm, tot);
    }
#pragma unroll
    for (int w = 0; w < kRadixThreads / 32; ++w) wcnt[w][threadIdx.x] = 0;
    __syncthreads();

    uint32_t key[IPT], val[IPT], rnk[IPT];
    const int64_t wbase = base + (int64_t)warp * (32 * IPT);
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
        const int64_t idx = wbase + i * 32 + lane;
        const bool valid = idx < n;
        key[i] = valid ? keys_in[idx] : 0u;
        val[i] = valid ? vals_in[idx] : 0u;
    }
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
        const bool valid = wbase + i * 32 + lane < n;
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
    // per-digit exclusive scan across the warps of this block; thread d owns digit d
    uint32_t total = 0;
#pragma unroll
    for (int w = 0; w < kRadixThreads / 32; ++w) {
        const uint32_t c = wcnt[w][threadIdx.x];
        wcnt[w][threadIdx.x] = total;
        total += c;
    }
    // decoupled look-back for digit d = threadIdx.x
    uint32_t* my = status + (size_t)b * 256 + threadIdx.x;
    uint32_t prefix = 0;
    if (b == 0) {
        st_volatile(my, kFlagIncl | total);
    } else {
        st_volatile(my, kFlagAgg | total);
        for (int64_t p = (int64_t)b - 1; p >= 0; --p) {
            const uint32_t* ps = status + (size_t)p * 256 + threadIdx.x;
            uint32_t s;
            do { s = ld_volatile(ps); } while ((s >> 30) == 0u);
            prefix += s & kValMask;
            if (s & kFlagIncl) break;
        }
        st_volatile(my, kFlagIncl | (prefix + total));
    }
    gbase[threadIdx.x] = digit_base + prefix;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < IPT; ++i) {
        const int64_t idx = wbase + i * 32 + lane;
        if (idx < n) {
            const uint32_t d = (key[i] >> shift) & mask;
            const uint32_t dst = gbase[d] + wcnt[warp][d] + rnk[i];
            keys_out[dst] = key[i];
            vals_out[dst] = val[i];
        }
    }
}

// ---- step B: tiles touched in depth order, exclusive scan (single pass, decoupled look-back) ---
// status64[b]: 2 flag bits | 62-bit sum
__global__ void __launch_bounds__(kScanThreads)
offsets_kernel(int N, const uint32_t* __restrict__ order, const float4* __restrict__ splats,
               uint32_t* __restrict__ cnt_out, uint32_t* __restrict__ off, unsigned long long* __restrict__ status64,
               uint32_t* __restrict__ ticket, int64_t Pcap, int64_t* __restrict__ P_dev) {
    __shared__ uint32_t sm[33];
    __shared__ uint32_t s_block;
    __shared__ unsigned long long s_prefix;
    if (threadIdx.x == 0) s_block = atomicAdd(ticket, 1u);
    __syncthreads();
    const uint32_t b = s_block;
    const int r = (int)(b * kScanThreads + threadIdx.x);
    uint32_t c = 0;
    if (r < N) {
        const float2 rc = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(splats) +
                                                             (size_t)order[r] * kSplatWords + 10);
        int x0, y0, x1, y1;
        unpack_rect(__float_as_uint(rc.x), __float_as_uint(rc.y), x0, y0, x1, y1);
        c = (uint32_t)((x1 - x0) * (y1 - y0));
        cnt_out[r] = c;
    }
    uint32_t tot;
    const uint32_t e = block_excl_scan(c, sm, tot);
    if (threadIdx.x == 0) {
        const unsigned long long AGG = 1ull << 62, INCL = 2ull << 62, VM = (1ull << 62) - 1ull;
        volatile unsigned long long* st = status64;
        unsigned long long prefix = 0;
        if (b == 0) {
            st[0] = INCL | (unsigned long long)tot;
        } else {
            st[b] = AGG | (unsigned long long)tot;
            for (int64_t p = (int64_t)b - 1; p >= 0; --p) {
                unsigned long long s;
                do { s = st[p]; } while ((s >> 62) == 0ull);
                prefix += s & VM;
                if (s & INCL) break;
            }
            st[b] = INCL | (prefix + tot);
        }
        s_prefix = prefix;
        if ((int64_t)(b + 1) * kScanThreads >= N) {  // last block: total
            const unsigned long long P = prefix + tot;
            P_dev[0] = (int64_t)P;
            P_dev[1] = ((int64_t)P > Pcap) ? 1 : 0;
        }
    }
    __syncthreads();
    // offsets are 32-bit: a total beyond capacity (< 2^30) is flagged above and nothing is written downstream
    if (r < N) off[r] = (uint32_t)(s_prefix + e);
}

// ---- step C: duplication in depth order + histograms of the tile-id digits ---------------------
__global__ void __launch_bounds__(256)
duplicate_kernel(int N, int gx, const uint32_t* __restrict__ order, const uint32_t* __restrict__ off,
                 const float4* __restrict__ splats, const int64_t* __restrict__ P_dev, uint32_t* __restrict__ tkey,
                 uint32_t* __restrict__ tval, int npass, int bits_per, uint32_t* __restrict__ ghist /* [npass][256] */) {
    __shared__ uint32_t h[3][256];
    h[0][threadIdx.x] = 0; h[1][threadIdx.x] = 0; h[2][threadIdx.x] = 0;
    __syncthreads();
    const uint32_t mask = (1u << bits_per) - 1u;
    if (!P_dev[1]) {
        for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < N; r += gridDim.x * blockDim.x) {
            const uint32_t g = order[r];
            const float2 rc = *reinterpret_cast<const float2*>(reinterpret_cast<const float*>(splats) +
                                                                 (size_t)g * kSplatWords + 10);
            int x0, y0, x1, y1;
            unpack_rect(__float_as_uint(rc.x), __float_as_uint(rc.y), x0, y0, x1, y1);
            uint32_t o = off[r];
            for (int ty = y0; ty < y1; ++ty)
                for (int tx = x0; tx < x1; ++tx) {
                    const uint32_t t = (uint32_t)(ty * gx + tx);
                    tkey[o] = t;
                    tval[o] = g;
                    ++o;
                    atomicAdd(&h[0][t & mask], 1u);
                    if (npass > 1) atomicAdd(&h[1][(t >> bits_per) & mask], 1u);
                    if (npass > 2) atomicAdd(&h[2][(t >> (2 * bits_per)) & mask], 1u);
                }
        }
    }
    __syncthreads();
    for (int p = 0; p < npass; ++p) {
        const uint32_t c = h[p][threadIdx.x];
        if (c) atomicAdd(&ghist[p * 256 + threadIdx.x], c);
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
inline int ipt_for(int64_t n) { return n <= (1 << 18) ? 4 : (n <= (1 << 22) ? 8 : 16); }
inline int64_t blocks_for(int64_t n) {
    const int64_t items = (int64_t)kRadixThreads * ipt_for(n);
    return (n + items - 1) / items;
}

struct Workspace {
    uint32_t *kA, *vA, *kB, *vB;   // N-sized ping-pong for the depth sort
    uint32_t *cnt, *off;           // N, N
    uint32_t *tkA, *tkB, *tvB;     // Pcap-sized: tile keys ping-pong, second value buffer
    // zeroed at the start of every call (one memset): histograms, tickets, look-back status
    char* zero_begin;
    uint32_t *ghist;               // [7][256]: 4 depth digits, up to 3 tile-id digits
    uint32_t *ticket;              // [8]
    unsigned long long* scan_status;  // ceil(N/1024)
    uint32_t *statusN;             // 4 passes x blocks_for(N) x 256
    uint32_t *statusP;             // 3 passes x blocks_for(Pcap) x 256
    size_t zero_bytes;
    size_t total;
};

Workspace carve(void* base, int N, int64_t Pcap) {
    Workspace w;
    size_t o = 0;
    char* p = (char*)base;
    auto take = [&](size_t bytes) { char* r = p + o; o += align256(bytes); return r; };
    const size_t n = (size_t)(N > 0 ? N : 1), pc = (size_t)(Pcap > 0 ? Pcap : 1);
    w.kA = (uint32_t*)take(n * 4); w.vA = (uint32_t*)take(n * 4); w.kB = (uint32_t*)take(n * 4); w.vB = (uint32_t*)take(n * 4);
    w.cnt = (uint32_t*)take(n * 4); w.off = (uint32_t*)take(n * 4);
    w.tkA = (uint32_t*)take(pc * 4); w.tkB = (uint32_t*)take(pc * 4); w.tvB = (uint32_t*)take(pc * 4);
    const size_t z0 = o;
    w.zero_begin = p + o;
    w.ghist = (uint32_t*)take(7 * 256 * 4);
    w.ticket = (uint32_t*)take(8 * 4);
    w.scan_status = (unsigned long long*)take(((n + kScanThreads - 1) / kScanThreads) * 8);
    w.statusN = (uint32_t*)take(4 * (size_t)blocks_for((int64_t)n) * 256 * 4);
    w.statusP = (uint32_t*)take(3 * (size_t)blocks_for((int64_t)pc) * 256 * 4);
    w.zero_bytes = o - z0;
    w.total = o;
    return w;
}

void radix_pass(const uint32_t* kin, const uint32_t* vin, uint32_t* kout, uint32_t* vout, const int64_t* n_dev,
                int64_t n_cap, int shift, int bits, const uint32_t* ghist, uint32_t* status, uint32_t* ticket,
                cudaStream_t s) {
    const int nb = (int)blocks_for(n_cap);
    if (nb == 0) return;
    const uint32_t mask = (1u << bits) - 1u;
    switch (ipt_for(n_cap)) {
        case 4: onesweep_kernel<4><<<nb, kRadixThreads, 0, s>>>(kin, vin, kout, vout, n_dev, n_cap, shift, mask, ghist, status, ticket); break;
        case 8: onesweep_kernel<8><<<nb, kRadixThreads, 0, s>>>(kin, vin, kout, vout, n_dev, n_cap, shift, mask, ghist, status, ticket); break;
        default: onesweep_kernel<16><<<nb, kRadixThreads, 0, s>>>(kin, vin, kout, vout, n_dev, n_cap, shift, mask, ghist, status, ticket); break;
    }
    count_launches(1);
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
    cudaError_t e = cudaMemsetAsync(w.zero_begin, 0, w.zero_bytes, s);
    if (e != cudaSuccess) return e;

    // A: depth sort of the Gaussians (4 x 8-bit passes, ends in kA/vA)
    const int nbN = (int)blocks_for(N);
    int kb = (N + 255) / 256;
    if (kb > num_sms * 8) kb = num_sms * 8;
    if (kb < 1) kb = 1;
    depth_keys_kernel<<<kb, 256, 0, s>>>(N, splats, w.kA, w.vA, w.ghist);
    count_launches(1);
    const size_t stN = (size_t)nbN * 256;
    radix_pass(w.kA, w.vA, w.kB, w.vB, nullptr, N, 0, 8, w.ghist + 0 * 256, w.statusN + 0 * stN, w.ticket + 0, s);
    radix_pass(w.kB, w.vB, w.kA, w.vA, nullptr, N, 8, 8, w.ghist + 1 * 256, w.statusN + 1 * stN, w.ticket + 1, s);
    radix_pass(w.kA, w.vA, w.kB, w.vB, nullptr, N, 16, 8, w.ghist + 2 * 256, w.statusN + 2 * stN, w.ticket + 2, s);
    radix_pass(w.kB, w.vB, w.kA, w.vA, nullptr, N, 24, 8, w.ghist + 3 * 256, w.statusN + 3 * stN, w.ticket + 3, s);

    // B: tiles touched per Gaussian in depth order -> exclusive offsets, P
    const int nbs = (N + kScanThreads - 1) / kScanThreads;
    if (nbs > 0) {
        offsets_kernel<<<nbs, kScanThreads, 0, s>>>(N, w.vA, splats, w.cnt, w.off, w.scan_status, w.ticket + 7, Pcap, P_dev);
        count_launches(1);
    } else {
        e = cudaMemsetAsync(P_dev, 0, 2 * sizeof(int64_t), s);
        if (e != cudaSuccess) return e;
    }

    // C + D: duplicate in depth order, then stable sort on the tile-id bits only
    int tbits = 1;
    while ((1 << tbits) < T) ++tbits;
    const int npass = (tbits + 7) / 8;  // T <= 2^20: at most 3; in practice 1 or 2 (tickets 4..6, scan ticket 7)
    const int bits_per = (tbits + npass - 1) / npass;
    // ping-pong (tkA, gid_sorted) <-> (tkB, tvB); start so that the result lands in (tkA, gid_sorted)
    uint32_t* k0 = (npass % 2 == 0) ? w.tkA : w.tkB;
    uint32_t* v0 = (npass % 2 == 0) ? gid_sorted : w.tvB;
    uint32_t* k1 = (npass % 2 == 0) ? w.tkB : w.tkA;
    uint32_t* v1 = (npass % 2 == 0) ? w.tvB : gid_sorted;
    duplicate_kernel<<<kb, 256, 0, s>>>(N, cam.gx, w.vA, w.off, splats, P_dev, k0, v0, npass, bits_per, w.ghist + 4 * 256);
    count_launches(1);
    const size_t stP = (size_t)blocks_for(Pcap) * 256;
    for (int p = 0; p < npass; ++p) {
        radix_pass(k0, v0, k1, v1, P_dev, Pcap, p * bits_per, bits_per, w.ghist + (4 + p) * 256, w.statusP + (size_t)p * stP,
                   w.ticket + 4 + p, s);
        uint32_t* tk = k0; k0 = k1; k1 = tk;
        uint32_t* tv = v0; v0 = v1; v1 = tv;
    }
    // E: CSR ranges (+ optional 64-bit keys)
    const int rb = num_sms * 8;
    ranges_kernel<<<rb, 256, 0, s>>>(w.tkA, P_dev, T, tile_offsets);
    count_launches(1);
    if (keys_sorted) {
        keys64_kernel<<<rb, 256, 0, s>>>(w.tkA, gid_sorted, splats, P_dev, keys_sorted);
        count_launches(1);
    }
    return cudaGetLastError();
}

}  // namespace tgs
