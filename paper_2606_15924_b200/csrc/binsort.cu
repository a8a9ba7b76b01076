// tgs_bin_sort: tile-overlap duplication, hand-written radix sort of the (tile, depth) keys and
// per-tile CSR ranges ("K(p) ... sorted by depth").
//
// Required result: all (tile, Gaussian) pairs ordered by (tile_id, depth bits, Gaussian id) --
// i.e. the 64-bit keys tile_id<<32 | float_bits(depth) sorted, ties by Gaussian id.  The key has
// structure a generic 64-bit sort does not use: its high word is a BIN (a few thousand tiles) and
// only the low word needs ordering, inside one bin at a time.  So the sort is an MSD radix sort
// whose first digit is the whole tile id, done as a counting sort, followed by an independent
// LSD radix sort of every tile's segment in SHARED MEMORY:
//
//   K1 bin_count    per Gaussian, per covered (selected) tile: count.  Counts are privatised in a
//                   shared-memory histogram per block (hot tiles of a clustered scene would
//                   serialise same-address global atomics).  The last block to finish turns the
//                   counts into the CSR tile_offsets[T+1], P, and the list of oversized tiles.
//   K2 bin_scatter  same walk; a block reserves its share of every tile's segment with one global
//                   atomic per (block, tile) and its threads take slots with shared-memory atomics;
//                   writes (depth bits, Gaussian id) into the tile's segment, in arbitrary order.
//   K3 seg_sort     persistent blocks pull tiles; a segment is loaded into shared memory, sorted by
//                   LSD radix passes over the VARYING depth bits only (per-warp private histograms,
//                   match-any ranking: stable), and written out as gid_sorted.  Only the top
//                   ~log2(m)+5 varying bits are radix-sorted (usually 2 passes of <= 9 bits); the
//                   few elements that still tie on those bits are ordered by a local full
//                   (depth, id) comparison.  A segment whose ties run longer than 32 falls back to
//                   the full LSD sort on all 64 bits (id digits first).  Segments larger than the
//                   shared-memory capacity are sorted by a second launch with 1024-thread blocks
//                   (shared memory up to 8192 entries, global ping-pong beyond).
//
// The final order is unique, so the result is deterministic although K2's intra-segment order is
// not.  With `tile_select` (written by tgs_sample) only pairs of selected tiles are counted and
// scattered: every cost after reading the 16 rect/depth bytes per Gaussian scales with the sampled
// tile fraction (R14).
//
// Every kernel reads its element counts from device memory (P is data dependent), so the whole
// call is asynchronous and graph-capturable.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kBinThreads = 256;
constexpr int kSmemTilesMax = 12288;   // tile histogram kept in shared memory up to this many tiles (48 KB)
constexpr int kSmallRect = 6;          // rects up to this many tiles are walked by their own thread
constexpr int kMaxDigitBits = 9;
constexpr int kTieRun = 32;            // longest tie run resolved by local comparison

// zeroed words at the head of the workspace
struct Counters {
    uint32_t done_count;     // K1 blocks finished
    uint32_t n_big;          // tiles with more than the small kernel's capacity
    uint32_t sched_small;    // work tickets of the two seg_sort launches
    uint32_t sched_big;
    uint32_t done_small;     // blocks finished (self re-arm is not needed: zeroed per call)
    uint32_t pad[3];
};

__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v) {
    const int lane = threadIdx.x & 31;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += y;
    }
    return v;
}

// Block-wide exclusive scan of one value per thread; `ws` holds 33 words.  Returns the exclusive
// prefix, `total` = block sum.  Ends with a barrier (ws reusable).
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* ws, uint32_t& total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const uint32_t inc = warp_incl_scan(v);
    if (lane == 31) ws[warp] = inc;
    __syncthreads();
    if (warp == 0) {
        const uint32_t t = lane < nw ? ws[lane] : 0u;
        const uint32_t ti = warp_incl_scan(t);
        ws[lane] = ti - t;
        if (lane == 31) ws[32] = ti;
    }
    __syncthreads();
    const uint32_t r = inc - v + ws[warp];
    total = ws[32];
    __syncthreads();
    return r;
}

// ---- the walk shared by K1 and K2: every (Gaussian, covered selected tile) pair of a chunk -------
// f(tile, gid, depth_bits) is called once per pair.  Small rects are walked by their own thread,
// large ones by the whole warp (a 30x30-tile splat must not stall 31 lanes).
template <class F>
__device__ __forceinline__ void walk_pairs(int begin, int end, int gx, const float4* __restrict__ splats,
                                           const uint32_t* __restrict__ tile_select, F f) {
    const int lane = threadIdx.x & 31;
    for (int i0 = begin + (int)(threadIdx.x & ~31u); i0 < end; i0 += blockDim.x) {
        const int i = i0 + lane;
        int x0 = 0, y0 = 0, x1 = 0, y1 = 0;
        uint32_t dbits = 0;
        if (i < end) {
            const float4 r2 = splats[3 * (size_t)i + 2];
            unpack_rect(__float_as_uint(r2.z), __float_as_uint(r2.w), x0, y0, x1, y1);
            dbits = __float_as_uint(r2.y);
        }
        const int w = x1 - x0, h = y1 - y0;
        const int area = (w > 0 && h > 0) ? w * h : 0;
        if (area > 0 && area <= kSmallRect) {
            for (int ty = y0; ty < y1; ++ty)
                for (int tx = x0; tx < x1; ++tx) {
                    const uint32_t t = (uint32_t)(ty * gx + tx);
                    if (tile_select == nullptr || tile_select[t]) f(t, (uint32_t)i, dbits);
                }
        }
        uint32_t big = __ballot_sync(0xffffffffu, area > kSmallRect);
        while (big) {
            const int src = __ffs(big) - 1;
            big &= big - 1;
            const int bx0 = __shfl_sync(0xffffffffu, x0, src), by0 = __shfl_sync(0xffffffffu, y0, src);
            const int bw = __shfl_sync(0xffffffffu, w, src), ba = __shfl_sync(0xffffffffu, area, src);
            const uint32_t bd = __shfl_sync(0xffffffffu, dbits, src);
            for (int j = lane; j < ba; j += 32) {
                const int ty = by0 + j / bw, tx = bx0 + j % bw;
                const uint32_t t = (uint32_t)(ty * gx + tx);
                if (tile_select == nullptr || tile_select[t]) f(t, (uint32_t)(i0 + src), bd);
            }
        }
    }
}

// ---- K1: per-tile pair counts, then (last block) CSR offsets, P and the oversized-tile list -----
template <bool SMEM_HIST>
__global__ void __launch_bounds__(kBinThreads)
bin_count_kernel(int N, int chunk, int gx, int T, const float4* __restrict__ splats,
                 const uint32_t* __restrict__ tile_select, uint32_t* __restrict__ tile_count,
                 uint32_t* __restrict__ tile_offsets, int64_t Pcap, int64_t* __restrict__ P_dev,
                 Counters* __restrict__ ctr, uint32_t* __restrict__ big_list, uint32_t small_cap) {
    extern __shared__ __align__(16) uint32_t hist[];  // [T] when SMEM_HIST
    __shared__ uint32_t ws[33];
    __shared__ uint32_t s_last;
    __shared__ unsigned long long s_carry;
    if (SMEM_HIST) {
        for (int t = threadIdx.x; t < T; t += blockDim.x) hist[t] = 0;
        __syncthreads();
    }
    const int begin = min(N, (int)blockIdx.x * chunk), end = min(N, begin + chunk);
    if (SMEM_HIST)
        walk_pairs(begin, end, gx, splats, tile_select, [&](uint32_t t, uint32_t, uint32_t) { atomicAdd(&hist[t], 1u); });
    else
        walk_pairs(begin, end, gx, splats, tile_select, [&](uint32_t t, uint32_t, uint32_t) { atomicAdd(&tile_count[t], 1u); });
    __syncthreads();
    if (SMEM_HIST) {
        for (int t = threadIdx.x; t < T; t += blockDim.x) {
            const uint32_t c = hist[t];
            if (c) atomicAdd(&tile_count[t], c);
        }
    }
    // ---- last block: exclusive scan of the counts ----
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = (atomicAdd(&ctr->done_count, 1u) == gridDim.x - 1u) ? 1u : 0u;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (threadIdx.x == 0) s_carry = 0ull;
    __syncthreads();
    // each thread owns kPer consecutive tiles of a span of blockDim * kPer tiles
    constexpr int kPer = 8;
    for (int b0 = 0; b0 < T; b0 += kBinThreads * kPer) {
        const int t0 = b0 + (int)threadIdx.x * kPer;
        uint32_t c[kPer], sum = 0;
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            c[j] = (t0 + j < T) ? __ldcg(tile_count + t0 + j) : 0u;
            sum += c[j];
        }
        uint32_t tot;
        const uint32_t ex = block_excl_scan(sum, ws, tot);
        unsigned long long run = s_carry + ex;
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            if (t0 + j < T) {
                // offsets are 32-bit; beyond capacity (< 2^30) nothing downstream runs
                tile_offsets[t0 + j] = (uint32_t)(run < (1ull << 32) ? run : 0xffffffffull);
                if (c[j] > small_cap) big_list[atomicAdd(&ctr->n_big, 1u)] = (uint32_t)(t0 + j);
            }
            run += c[j];
        }
        __syncthreads();
        if (threadIdx.x == 0) s_carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const unsigned long long P = s_carry;
        tile_offsets[T] = (uint32_t)(P < (1ull << 32) ? P : 0xffffffffull);
        P_dev[0] = (int64_t)P;
        P_dev[1] = ((int64_t)P > Pcap) ? 1 : 0;
    }
}

// ---- K2: scatter (depth bits, Gaussian id) into the tile segments ---------------------------------
template <bool SMEM_HIST>
__global__ void __launch_bounds__(kBinThreads)
bin_scatter_kernel(int N, int chunk, int gx, int T, const float4* __restrict__ splats,
                   const uint32_t* __restrict__ tile_select, const uint32_t* __restrict__ tile_offsets,
                   uint32_t* __restrict__ cursor, const int64_t* __restrict__ P_dev, uint2* __restrict__ pairs) {
    extern __shared__ __align__(16) uint32_t hist[];
    if (P_dev[1]) return;  // over capacity: nothing is written
    const int begin = min(N, (int)blockIdx.x * chunk), end = min(N, begin + chunk);
    if (SMEM_HIST) {
        for (int t = threadIdx.x; t < T; t += blockDim.x) hist[t] = 0;
        __syncthreads();
        walk_pairs(begin, end, gx, splats, tile_select, [&](uint32_t t, uint32_t, uint32_t) { atomicAdd(&hist[t], 1u); });
        __syncthreads();
        // reserve this block's share of every segment it touches; hist[t] becomes the absolute cursor
        for (int t = threadIdx.x; t < T; t += blockDim.x) {
            const uint32_t c = hist[t];
            if (c) hist[t] = tile_offsets[t] + atomicAdd(&cursor[t], c);
        }
        __syncthreads();
        walk_pairs(begin, end, gx, splats, tile_select, [&](uint32_t t, uint32_t g, uint32_t d) {
            const uint32_t slot = atomicAdd(&hist[t], 1u);
            pairs[slot] = make_uint2(d, g);
        });
    } else {
        walk_pairs(begin, end, gx, splats, tile_select, [&](uint32_t t, uint32_t g, uint32_t d) {
            const uint32_t slot = tile_offsets[t] + atomicAdd(&cursor[t], 1u);
            pairs[slot] = make_uint2(d, g);
        });
    }
}

// ---- K3: per-tile segment sort ----------------------------------------------------------------------
// One stable LSD pass src -> dst over `bits` bits at `shift` of word `word` (0 = depth, 1 = id).
// Warp w owns the contiguous sub-range [w*per_warp, ...) and a private histogram row wh[w][*]:
// count, scan in (digit, warp) order, then rank in range order with match-any.
template <int THREADS>
__device__ __forceinline__ void radix_pass(const uint2* src, uint2* dst, uint32_t m, int word, int shift, int bits,
                                           uint32_t* wh, uint32_t* ws) {
    constexpr int W = THREADS / 32;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t nb = 1u << bits, mask = nb - 1u, lt_mask = (1u << lane) - 1u;
    for (uint32_t i = threadIdx.x; i < (uint32_t)W * nb; i += THREADS) wh[i] = 0u;
    __syncthreads();
    const uint32_t per_warp = (((m + W - 1) / W) + 31u) & ~31u;
    const uint32_t lo = min(m, (uint32_t)warp * per_warp), hi = min(m, lo + per_warp);
    uint32_t* row = wh + (uint32_t)warp * nb;
    for (uint32_t i0 = lo; i0 < hi; i0 += 32) {
        const uint32_t i = i0 + lane;
        const bool valid = i < hi;
        uint2 kv = make_uint2(0u, 0u);
        if (valid) kv = src[i];
        const uint32_t d = valid ? (((word ? kv.y : kv.x) >> shift) & mask) : 0xffffffffu;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        if (valid && lane == __ffs(peers) - 1) row[d] += __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    uint32_t carry = 0;
    for (uint32_t d0 = 0; d0 < nb; d0 += THREADS) {
        const uint32_t d = d0 + threadIdx.x;
        uint32_t tot = 0;
        if (d < nb) {
#pragma unroll 4
            for (int w = 0; w < W; ++w) {
                const uint32_t c = wh[w * nb + d];
                wh[w * nb + d] = tot;
                tot += c;
            }
        }
        uint32_t total;
        const uint32_t base = carry + block_excl_scan(tot, ws, total);
        if (d < nb) {
#pragma unroll 4
            for (int w = 0; w < W; ++w) wh[w * nb + d] += base;
        }
        carry += total;
    }
    __syncthreads();
    for (uint32_t i0 = lo; i0 < hi; i0 += 32) {
        const uint32_t i = i0 + lane;
        const bool valid = i < hi;
        uint2 kv = make_uint2(0u, 0u);
        if (valid) kv = src[i];
        const uint32_t d = valid ? (((word ? kv.y : kv.x) >> shift) & mask) : 0xffffffffu;
        const uint32_t peers = __match_any_sync(0xffffffffu, d);
        const int leader = __ffs(peers) - 1;
        uint32_t old = 0;
        if (valid && lane == leader) {
            old = row[d];
            row[d] = old + __popc(peers);
        }
        old = __shfl_sync(0xffffffffu, old, leader);
        if (valid) dst[old + __popc(peers & lt_mask)] = kv;
        __syncwarp();
    }
    __syncthreads();
}

__device__ __forceinline__ int ceil_log2_u32(uint32_t v) { return v <= 1u ? 0 : 32 - __clz(v - 1u); }

template <int THREADS, int CAP, bool BIG>
__global__ void __launch_bounds__(THREADS)
seg_sort_kernel(int T, const uint32_t* __restrict__ tile_offsets, uint2* pairs, uint2* tmp,
                uint32_t* __restrict__ gid_sorted, uint64_t* __restrict__ keys_sorted,
                const int64_t* __restrict__ P_dev, Counters* __restrict__ ctr, const uint32_t* __restrict__ big_list,
                uint32_t small_cap, int gid_bits) {
    constexpr int W = THREADS / 32;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint2* smA = reinterpret_cast<uint2*>(smem_raw);
    uint2* smB = smA + CAP;
    uint32_t* wh = reinterpret_cast<uint32_t*>(smB + CAP);  // [W][1 << kMaxDigitBits]
    __shared__ uint32_t ws[33];
    __shared__ uint32_t s_ticket[2];
    __shared__ uint32_t s_diff, s_flag;
    if (P_dev[1]) return;
    uint32_t* sched = BIG ? &ctr->sched_big : &ctr->sched_small;
    const uint32_t n_work = BIG ? *reinterpret_cast<volatile uint32_t*>(&ctr->n_big) : (uint32_t)T;
    const int lane = threadIdx.x & 31;
    if (threadIdx.x == 0) s_ticket[0] = atomicAdd(sched, 1u);
    __syncthreads();
    for (uint32_t it = 0;; ++it) {
        const uint32_t ticket = s_ticket[it & 1u];
        if (ticket >= n_work) break;
        if (threadIdx.x == 0) {  // prefetch the next ticket: its latency hides behind this tile
            s_ticket[(it + 1u) & 1u] = atomicAdd(sched, 1u);
            s_diff = 0u;
            s_flag = 0u;
        }
        const uint32_t t = BIG ? big_list[ticket] : ticket;
        const uint32_t start = tile_offsets[t], m = tile_offsets[t + 1] - start;
        __syncthreads();
        if (m == 0u || (!BIG && m > small_cap)) { __syncthreads(); continue; }
        const bool in_smem = BIG ? (m <= (uint32_t)CAP) : true;  // small kernel: always shared (address space known statically)
        uint2* A = in_smem ? smA : pairs + start;
        uint2* B = in_smem ? smB : tmp + start;
        // ---- load (shared-memory path) and find the varying depth bits ----
        {
            const uint32_t k0 = pairs[start].x;
            uint32_t diff = 0;
            for (uint32_t i = threadIdx.x; i < m; i += THREADS) {
                const uint2 kv = pairs[start + i];
                if (in_smem) smA[i] = kv;
                diff |= kv.x ^ k0;
            }
            diff = __reduce_or_sync(0xffffffffu, diff);
            if (lane == 0 && diff) atomicOr(&s_diff, diff);
        }
        __syncthreads();
        const int nbits = 32 - __clz(s_diff);  // depth bits [0, nbits) vary inside this tile
        int sb = min(nbits, max(8, min(27, ceil_log2_u32(m) + 5)));
        int npass = (sb + kMaxDigitBits - 1) / kMaxDigitBits;
        int bits = npass ? (sb + npass - 1) / npass : 0;
        const int shift0 = max(0, nbits - npass * bits);  // bits below shift0 are left to the tie step
        for (int p = 0; p < npass; ++p) {
            radix_pass<THREADS>(A, B, m, 0, shift0 + p * bits, bits, wh, ws);
            uint2* x = A; A = B; B = x;
        }
        // ---- ties on the sorted bits: local full (depth, id) comparison ----
        for (uint32_t i = threadIdx.x; i < m; i += THREADS) {
            const uint2 kv = A[i];
            const uint32_t sk = shift0 < 32 ? (kv.x >> shift0) : 0u;
            uint32_t s = i, e = i + 1;
            while (s > 0 && i - s <= (uint32_t)kTieRun && (A[s - 1].x >> shift0) == sk) --s;
            while (e < m && e - i <= (uint32_t)kTieRun && (A[e].x >> shift0) == sk) ++e;
            if (i - s > (uint32_t)kTieRun || e - i > (uint32_t)kTieRun) {
                s_flag = 1u;
                continue;
            }
            uint32_t rank = 0;
            for (uint32_t j = s; j < e; ++j) {
                const uint2 o = A[j];
                rank += (o.x < kv.x || (o.x == kv.x && o.y < kv.y)) ? 1u : 0u;
            }
            gid_sorted[start + s + rank] = kv.y;
            if (keys_sorted) keys_sorted[start + s + rank] = ((uint64_t)t << 32) | (uint64_t)kv.x;
        }
        __syncthreads();
        if (s_flag) {
            // ---- fallback: full LSD sort on (depth, id): id digits first, then every varying depth bit ----
            int np = (gid_bits + kMaxDigitBits - 1) / kMaxDigitBits, bt = (gid_bits + np - 1) / np;
            for (int p = 0; p < np; ++p) {
                radix_pass<THREADS>(A, B, m, 1, p * bt, bt, wh, ws);
                uint2* x = A; A = B; B = x;
            }
            np = (nbits + kMaxDigitBits - 1) / kMaxDigitBits;
            bt = np ? (nbits + np - 1) / np : 0;
            for (int p = 0; p < np; ++p) {
                radix_pass<THREADS>(A, B, m, 0, p * bt, bt, wh, ws);
                uint2* x = A; A = B; B = x;
            }
            for (uint32_t i = threadIdx.x; i < m; i += THREADS) {
                const uint2 kv = A[i];
                gid_sorted[start + i] = kv.y;
                if (keys_sorted) keys_sorted[start + i] = ((uint64_t)t << 32) | (uint64_t)kv.x;
            }
            __syncthreads();
        }
    }
}

constexpr int kSmallThreads = 256, kSmallCap = 3072;
constexpr int kBigThreads = 1024, kBigCap = 8192;
constexpr size_t kSmallSmem = 2 * (size_t)kSmallCap * sizeof(uint2) + (kSmallThreads / 32) * (sizeof(uint32_t) << kMaxDigitBits);
constexpr size_t kBigSmem = 2 * (size_t)kBigCap * sizeof(uint2) + (kBigThreads / 32) * (sizeof(uint32_t) << kMaxDigitBits);

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Workspace {
    // zeroed at the start of every call (one memset): counters, tile counts, scatter cursors
    Counters* ctr;
    uint32_t *tile_count, *cursor;
    size_t zero_bytes;
    uint32_t* big_list;   // [T]
    uint2 *pairs, *tmp;   // [Pcap] each: unsorted segments; ping-pong partner for oversized segments
    size_t total;
};

Workspace carve(void* base, int T, int64_t Pcap) {
    Workspace w;
    size_t o = 0;
    char* p = (char*)base;
    auto take = [&](size_t bytes) { char* r = p + o; o += align256(bytes); return r; };
    const size_t nt = (size_t)(T > 0 ? T : 1), pc = (size_t)(Pcap > 0 ? Pcap : 1);
    w.ctr = (Counters*)take(sizeof(Counters));
    w.tile_count = (uint32_t*)take(nt * 4);
    w.cursor = (uint32_t*)take(nt * 4);
    w.zero_bytes = o;
    w.big_list = (uint32_t*)take(nt * 4);
    w.pairs = (uint2*)take(pc * 8);
    w.tmp = (uint2*)take(pc * 8);
    w.total = o;
    return w;
}

}  // namespace

size_t binsort_workspace_bytes(int N, int64_t Pcap, int T) {
    (void)N;
    return carve(nullptr, T, Pcap).total;
}

cudaError_t launch_bin_sort(const CamK& cam, int N, const float* splats_f, const uint32_t* tile_select, int64_t Pcap,
                            uint64_t* keys_sorted, uint32_t* gid_sorted, uint32_t* tile_offsets, int64_t* P_dev,
                            void* ws, size_t ws_bytes, int num_sms, cudaStream_t s) {
    (void)ws_bytes;
    const int T = cam.gx * cam.gy;
    const Workspace w = carve(ws, T, Pcap);
    const float4* splats = reinterpret_cast<const float4*>(splats_f);
    cudaError_t e = cudaMemsetAsync(w.ctr, 0, w.zero_bytes, s);
    if (e != cudaSuccess) return e;

    static bool opted_in = false;  // function attributes, set once per process
    if (!opted_in) {
        e = cudaFuncSetAttribute(seg_sort_kernel<kSmallThreads, kSmallCap, false>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmallSmem);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(seg_sort_kernel<kBigThreads, kBigCap, true>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kBigSmem);
        if (e != cudaSuccess) return e;
        opted_in = true;
    }

    // K1 / K2: a block owns a contiguous chunk of Gaussians
    int blocks = (N + kBinThreads - 1) / kBinThreads;
    if (blocks > num_sms * 4) blocks = num_sms * 4;
    if (blocks < 1) blocks = 1;
    const int chunk = (N + blocks - 1) / blocks;
    const bool smem_hist = T <= kSmemTilesMax;
    const size_t hist_bytes = smem_hist ? (size_t)T * 4 : 0;
    if (smem_hist) {
        bin_count_kernel<true><<<blocks, kBinThreads, hist_bytes, s>>>(N, chunk, cam.gx, T, splats, tile_select,
            w.tile_count, tile_offsets, Pcap, P_dev, w.ctr, w.big_list, (uint32_t)kSmallCap);
        bin_scatter_kernel<true><<<blocks, kBinThreads, hist_bytes, s>>>(N, chunk, cam.gx, T, splats, tile_select,
            tile_offsets, w.cursor, P_dev, w.pairs);
    } else {
        bin_count_kernel<false><<<blocks, kBinThreads, 0, s>>>(N, chunk, cam.gx, T, splats, tile_select,
            w.tile_count, tile_offsets, Pcap, P_dev, w.ctr, w.big_list, (uint32_t)kSmallCap);
        bin_scatter_kernel<false><<<blocks, kBinThreads, 0, s>>>(N, chunk, cam.gx, T, splats, tile_select,
            tile_offsets, w.cursor, P_dev, w.pairs);
    }
    count_launches(2);

    // K3: oversized segments first (1024-thread blocks), then everything else
    int gid_bits = 1;
    while (gid_bits < 30 && (1ll << gid_bits) < (long long)N) ++gid_bits;
    if (Pcap > kSmallCap) {  // otherwise no segment can be oversized
        int bb = num_sms < T ? num_sms : T;
        seg_sort_kernel<kBigThreads, kBigCap, true><<<bb, kBigThreads, kBigSmem, s>>>(T, tile_offsets, w.pairs, w.tmp,
            gid_sorted, keys_sorted, P_dev, w.ctr, w.big_list, (uint32_t)kSmallCap, gid_bits);
        count_launches(1);
    }
    int sb = num_sms * 3;
    if (sb > T) sb = T;
    seg_sort_kernel<kSmallThreads, kSmallCap, false><<<sb, kSmallThreads, kSmallSmem, s>>>(T, tile_offsets, w.pairs,
        w.tmp, gid_sorted, keys_sorted, P_dev, w.ctr, w.big_list, (uint32_t)kSmallCap, gid_bits);
    count_launches(1);
    return cudaGetLastError();
}

}  // namespace tgs
