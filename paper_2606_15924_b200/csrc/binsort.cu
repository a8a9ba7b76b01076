// tgs_bin_sort: tile-overlap duplication, hand-written sort of the (tile, depth) keys and per-tile
// CSR ranges ("K(p) ... sorted by depth").
//
// Required result: all (tile, Gaussian) pairs ordered by (tile_id, depth bits, Gaussian id) --
// i.e. the 64-bit keys tile_id<<32 | float_bits(depth) sorted, ties by Gaussian id.  The key has
// structure a generic 64-bit sort does not use: its high word is a BIN (a few thousand tiles), only
// the low word needs ordering inside one bin, and the bins a Gaussian falls into form a small
// rectangle.  Shared-memory and global atomics cost ~2 cycles per LANE on this machine, i.e. one
// atomic per pair is as expensive as all the memory traffic of the sort, so the design avoids
// per-pair atomics altogether:
//
//   Ks select_sat     (one block, only with tile_select) summed-area table of the selection.
//   K0 topleft_count  every rect is cut into pieces of at most 4x4 tiles; histogram of the pieces'
//                     top-left tiles (pieces without a selected tile are dropped), privatised in
//                     shared memory per block; P = sum of the pieces' selected tiles.
//   K1 bin_scan       (one block) exclusive scan of that histogram; publishes P and the capacity flag.
//   K2 reorder        a 16-byte record {depth bits, id, piece rect} per piece, grouped by top-left
//                     tile (slots from the block's private cursors: no global atomic).  From here on
//                     a warp's 32 records are neighbours on screen.
//   K3 pair_count     per warp: the lanes that share a top ROW span a window of a few tiles; each
//                     lane holds its coverage of the window as a 32-bit mask, ONE ballot per window
//                     tile gives the covering lanes, so the warp issues one RED per (warp, tile)
//                     instead of one per pair.
//   K4 tile_scan      (one block) CSR tile_offsets[T+1] and the work lists of the sort by size.
//   K5 pair_scatter   same walk as K3: one ATOM per (warp, tile) reserves a run of the tile's
//                     segment, the covering lanes write (depth bits, id) at consecutive slots.
//   K6 giant_split    segments above the shared-memory capacity are split by depth: 1024 fine
//                     buckets (monotone interpolation between the segment's min and max key) merged
//                     into sub-segments of ~2k elements.
//   K7 seg_sort       (three launches: <= 2048 / 4096 / 8192 elements with 256 / 1024 / 1024 threads; four elements
//                     per thread in the middle class: a segment's latency, not throughput, sets the time when few
//                     tiles are sampled -- 0.131 -> 0.122 ms at 5 % of config 5's tiles) a block sorts a segment in
//                     shared memory in ONE distribution step: bucket = monotone interpolation of the
//                     depth bits between the segment's min and max (about two buckets per element);
//                     the slot inside a bucket comes from one write-then-check round on a 16-bit
//                     table (the last writer wins slot 0: no atomic for ~80 % of the elements) and a
//                     shared-memory atomic for the losers; buckets are then ordered by counting,
//                     inside each bucket, the elements with a smaller (depth, id).  A segment whose
//                     keys pile up (> 512 in a bucket: equal depths) falls back to a stable LSD radix
//                     sort on (id, depth) in global memory.
//
// The final order is unique, so the result is deterministic although the slot assignment of K2/K5
// is not.  With `tile_select` (written by tgs_sample) only pairs of selected tiles are counted and
// scattered: everything after K2 scales with the sampled tile fraction (R14).
//
// Every kernel reads its element counts from device memory (P is data dependent), so the whole
// call is asynchronous and graph-capturable.
#include "common.cuh"

namespace tgs {

namespace {

constexpr int kScanThreads = 1024;
constexpr int kWalkThreads = 256;
constexpr int kSmemTilesMax = 12288;     // top-left histogram kept in shared memory up to this many tiles (48 KB)
constexpr int kRegroupBlocksMax = 160;   // blocks of K0 / K2 (one per SM)
constexpr int kSmallW = 4, kSmallH = 4;  // rects up to this size go through the ballot window
constexpr int kRounds = 1;               // write-then-check rounds before the atomic fallback
constexpr uint32_t kMaxOcc = 512;        // bucket occupancy above which a segment takes the radix fallback
constexpr int kFbBits = 8;               // digit width of the fallback radix sort
constexpr uint32_t kSubTarget = 2048;    // expected sub-segment size of a giant split
constexpr int kCoarseMax = 1024;         // sub-segments per giant tile (one per thread of giant_split)

// zeroed words at the head of the workspace
struct Counters {
    uint32_t n_vis;                       // records written by K2 (rects of at most 4x4 tiles)
    uint32_t n_small, n_medium, n_large, n_giant;   // lengths of the work lists
    uint32_t sched_small, sched_medium, sched_large, sched_giant;  // work tickets
    uint32_t pad[3];
    unsigned long long p_total;           // P, known after K0 (sum of the records' selected tiles)
};

struct Seg {            // one unit of sort work
    uint32_t start;     // offset in pairs / tmp / gid_sorted
    uint32_t len;
    uint32_t tile;
    uint32_t in_tmp;    // 1: the unsorted pairs are in tmp (a sub-segment written by giant_split)
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

__device__ __forceinline__ void load_rect(const float4* __restrict__ splats, int i, int gx, int gy, int& x0, int& y0,
                                          int& x1, int& y1, uint32_t& dbits) {
    const float4 r2 = splats[3 * (size_t)i + 2];
    unpack_rect(__float_as_uint(r2.z), __float_as_uint(r2.w), x0, y0, x1, y1);
    x1 = min(x1, gx);
    y1 = min(y1, gy);
    dbits = __float_as_uint(r2.y);
}

// Selected tiles inside [x0,x1) x [y0,y1): from the summed-area table, or the area when every tile counts.
__device__ __forceinline__ uint32_t rect_pairs(const uint32_t* __restrict__ sat, int sx, int x0, int y0, int x1, int y1) {
    if (sat == nullptr) return (uint32_t)((x1 - x0) * (y1 - y0));
    return sat[(size_t)y1 * sx + x1] - sat[(size_t)y0 * sx + x1] - sat[(size_t)y1 * sx + x0] + sat[(size_t)y0 * sx + x0];
}

// A rect is cut into pieces of at most kSmallW x kSmallH tiles; f(px0, py0, px1, py1, pairs) is called
// for every piece that holds a selected tile.  (Most rects are one piece.)
template <class F>
__device__ __forceinline__ void for_each_piece(const uint32_t* __restrict__ sat, int gx, int x0, int y0, int x1, int y1, F f) {
    for (int py = y0; py < y1; py += kSmallH)
        for (int px = x0; px < x1; px += kSmallW) {
            const int qx = min(px + kSmallW, x1), qy = min(py + kSmallH, y1);
            const uint32_t np = rect_pairs(sat, gx + 1, px, py, qx, qy);
            if (np) f(px, py, qx, qy, np);
        }
}

// ---- K0: histogram of the top-left tile ---------------------------------------------------------
// A block owns a contiguous chunk of Gaussians.  SMEM: the block counts into a private shared-memory
// histogram (scattered global REDs are one L2 transaction each and ~5x slower), then adds its counts
// to the global histogram with coalesced atomics whose RETURN value is the block's offset inside
// every bin (blk_base[block][T]): K2 then needs no global atomic at all.
template <bool SMEM>
__global__ void __launch_bounds__(1024)
topleft_count_kernel(int N, int chunk, int gx, int gy, const float4* __restrict__ splats,
                     const uint32_t* __restrict__ sat, uint32_t* __restrict__ bin_count,
                     uint32_t* __restrict__ blk_base, Counters* __restrict__ ctr) {
    extern __shared__ __align__(16) uint32_t hist[];  // [T] when SMEM
    __shared__ unsigned long long s_pairs;
    const int T = gx * gy;
    const int begin = min(N, (int)blockIdx.x * chunk), end = min(N, begin + chunk);
    if (threadIdx.x == 0) s_pairs = 0ull;
    if (SMEM)
        for (int t = threadIdx.x; t < T; t += blockDim.x) hist[t] = 0u;
    __syncthreads();
    unsigned long long pairs = 0ull;
    for (int i = begin + (int)threadIdx.x; i < end; i += blockDim.x) {
        int x0, y0, x1, y1;
        uint32_t d;
        load_rect(splats, i, gx, gy, x0, y0, x1, y1, d);
        for_each_piece(sat, gx, x0, y0, x1, y1, [&](int px, int py, int, int, uint32_t np) {
            atomicAdd(SMEM ? &hist[py * gx + px] : &bin_count[py * gx + px], 1u);
            pairs += np;
        });
    }
    // P = sum of the pieces' selected tiles: one 64-bit atomic per block
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) pairs += __shfl_xor_sync(0xffffffffu, pairs, o);
    if ((threadIdx.x & 31) == 0 && pairs) atomicAdd(&s_pairs, pairs);
    __syncthreads();
    if (threadIdx.x == 0 && s_pairs) atomicAdd(&ctr->p_total, s_pairs);
    if (SMEM) {
        uint32_t* mine = blk_base + (size_t)blockIdx.x * T;
        for (int t = threadIdx.x; t < T; t += blockDim.x) {
            const uint32_t c = hist[t];
            mine[t] = c ? atomicAdd(&bin_count[t], c) : 0u;
        }
    }
}

// ---- Ks: summed-area table of tile_select (one block; only when a selection is given) -----------
// sat[(gy+1) x (gx+1)]: sat[y][x] = number of selected tiles with ty < y and tx < x.
__global__ void __launch_bounds__(kScanThreads)
select_sat_kernel(int gx, int gy, const uint32_t* __restrict__ tile_select, uint32_t* sat) {
    // row prefixes (a warp per row), then column sums (a thread per column)
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, sx = gx + 1;
    for (int x = threadIdx.x; x <= gx; x += kScanThreads) sat[x] = 0u;
    for (int y = warp; y < gy; y += kScanThreads / 32) {
        uint32_t running = 0;
        if (lane == 0) sat[(size_t)(y + 1) * sx] = 0u;
        for (int xb = 0; xb < gx; xb += 32) {
            const int x = xb + lane;
            const uint32_t v = (x < gx && tile_select[y * gx + x]) ? 1u : 0u;
            const uint32_t inc = warp_incl_scan(v) + running;
            if (x < gx) sat[(size_t)(y + 1) * sx + x + 1] = inc;
            running = __shfl_sync(0xffffffffu, inc, 31);
        }
    }
    __syncthreads();
    for (int x = 1 + (int)threadIdx.x; x <= gx; x += kScanThreads) {
        uint32_t acc = 0;
#pragma unroll 8
        for (int y = 1; y <= gy; ++y) {
            acc += sat[(size_t)y * sx + x];
            sat[(size_t)y * sx + x] = acc;
        }
    }
}

// ---- K1: scan of the top-left histogram; P and the capacity flag -----------------------------------
__global__ void __launch_bounds__(kScanThreads)
bin_scan_kernel(int T, const uint32_t* __restrict__ bin_count, uint32_t* __restrict__ bin_offset,
                Counters* __restrict__ ctr, int64_t Pcap, int64_t* __restrict__ P_dev) {
    __shared__ uint32_t ws[33];
    __shared__ uint32_t s_carry;
    if (threadIdx.x == 0) s_carry = 0u;
    __syncthreads();
    constexpr int kPer = 4;
    for (int b0 = 0; b0 < T; b0 += kScanThreads * kPer) {
        const int t0 = b0 + (int)threadIdx.x * kPer;
        uint32_t c[kPer], sum = 0;
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            c[j] = (t0 + j < T) ? bin_count[t0 + j] : 0u;
            sum += c[j];
        }
        uint32_t tot;
        uint32_t run = s_carry + block_excl_scan(sum, ws, tot);
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            if (t0 + j < T) bin_offset[t0 + j] = run;
            run += c[j];
        }
        __syncthreads();
        if (threadIdx.x == 0) s_carry += tot;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        // every record holds at least one pair, so records <= P <= Pcap whenever the call can proceed
        const unsigned long long P = ctr->p_total;
        ctr->n_vis = s_carry;
        P_dev[0] = (int64_t)P;
        P_dev[1] = ((int64_t)P > Pcap) ? 1 : 0;
    }
}

// ---- K2: records grouped by top-left tile -----------------------------------------------------------
template <bool SMEM>
__global__ void __launch_bounds__(1024)
reorder_kernel(int N, int chunk, int gx, int gy, const float4* __restrict__ splats,
               const uint32_t* __restrict__ bin_offset, uint32_t* __restrict__ bin_cursor,
               const uint32_t* __restrict__ blk_base, const uint32_t* __restrict__ sat,
               const int64_t* __restrict__ P_dev, uint4* __restrict__ rec) {
    extern __shared__ __align__(16) uint32_t cur[];  // [T] when SMEM: this block's next slot in every bin
    if (P_dev[1]) return;  // over capacity (the record buffer holds P_capacity records)
    const int T = gx * gy;
    const int begin = min(N, (int)blockIdx.x * chunk), end = min(N, begin + chunk);
    if (SMEM) {
        const uint32_t* mine = blk_base + (size_t)blockIdx.x * T;
        for (int t = threadIdx.x; t < T; t += blockDim.x) cur[t] = bin_offset[t] + mine[t];
        __syncthreads();
    }
    for (int i = begin + (int)threadIdx.x; i < end; i += blockDim.x) {
        int x0, y0, x1, y1;
        uint32_t d;
        load_rect(splats, i, gx, gy, x0, y0, x1, y1, d);
        for_each_piece(sat, gx, x0, y0, x1, y1, [&](int px, int py, int qx, int qy, uint32_t) {
            const int t0 = py * gx + px;
            const uint32_t slot = SMEM ? atomicAdd(&cur[t0], 1u) : bin_offset[t0] + atomicAdd(&bin_cursor[t0], 1u);
            rec[slot] = make_uint4(d, (uint32_t)i, (uint32_t)px | ((uint32_t)qx << 16), (uint32_t)py | ((uint32_t)qy << 16));
        });
    }
}

// ---- K3 / K5: the pair walk over the regrouped records ------------------------------------------
// SCATTER = false: tile_count[t] += pairs of tile t.  SCATTER = true: (depth bits, id) of every pair
// is written into its tile's segment (arbitrary order inside the segment).
template <bool SCATTER>
__global__ void __launch_bounds__(kWalkThreads)
pair_walk_kernel(int gx, const uint4* __restrict__ rec, const Counters* __restrict__ ctr,
                 const uint32_t* __restrict__ tile_select, uint32_t* __restrict__ tile_count,
                 const uint32_t* __restrict__ tile_offsets, uint32_t* __restrict__ cursor,
                 const int64_t* __restrict__ P_dev, uint2* __restrict__ pairs) {
    if (P_dev[1]) return;  // over capacity: nothing is written
    const uint32_t n = ctr->n_vis;
    const int lane = threadIdx.x & 31;
    const uint32_t lt_mask = (1u << lane) - 1u;
    const uint32_t gwarp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nwarps = (gridDim.x * blockDim.x) >> 5;
    for (uint32_t base = gwarp * 32u; base < n; base += nwarps * 32u) {
        const uint32_t i = base + lane;
        uint4 r = make_uint4(0u, 0u, 0u, 0u);
        if (i < n) r = rec[i];
        int x0, y0, x1, y1;
        unpack_rect(r.z, r.w, x0, y0, x1, y1);
        const int w = x1 - x0, h = y1 - y0;
        const bool live = w > 0 && h > 0;
        const bool small = live;  // K2 cuts every rect into pieces of at most kSmallW x kSmallH tiles
        // ---- small rects: lanes with the same top row share a window of tiles ----
        uint32_t todo = __ballot_sync(0xffffffffu, small);
        while (todo) {
            const int row = __shfl_sync(0xffffffffu, y0, __ffs(todo) - 1);
            const bool in = small && y0 == row;
            todo &= ~__ballot_sync(0xffffffffu, in);
            const int X0 = __reduce_min_sync(0xffffffffu, in ? x0 : 0x7fffffff);
            const int X1 = __reduce_max_sync(0xffffffffu, in ? x1 : 0);
            const int Hw = __reduce_max_sync(0xffffffffu, in ? h : 0);
            const int Ww = X1 - X0, win = Ww * Hw;
            if (win <= 32) {
                // ---- fast path: the whole window fits one 32-bit mask per lane ----
                uint32_t cover = 0;  // bit c = this lane's rect covers window tile c (row-major, Ww wide)
                if (in) {
                    const uint32_t rowmask = ((1u << w) - 1u) << (x0 - X0);
#pragma unroll
                    for (int rr = 0; rr < kSmallH; ++rr)
                        if (rr < h) cover |= rowmask << (rr * Ww);
                }
                uint32_t mine = 0;  // lane j: the lanes whose rect covers window tile j
                for (int j = 0; j < win; ++j) {
                    const uint32_t bal = __ballot_sync(0xffffffffu, (cover >> j) & 1u);
                    if (lane == j) mine = bal;
                }
                int ty = 0, tx = lane;  // lane's own window tile (win <= 32: at most 4 rows)
#pragma unroll
                for (int rr = 1; rr < kSmallH; ++rr)
                    if (lane >= rr * Ww) { ty = rr; tx = lane - rr * Ww; }
                const uint32_t t = (uint32_t)((row + ty) * gx + X0 + tx);
                bool has = lane < win && mine != 0u;
                if (has && tile_select != nullptr && tile_select[t] == 0u) has = false;
                if (!SCATTER) {
                    if (has) atomicAdd(&tile_count[t], (uint32_t)__popc(mine));
                } else {
                    uint32_t b = 0xffffffffu;
                    if (has) b = tile_offsets[t] + atomicAdd(&cursor[t], (uint32_t)__popc(mine));
                    // every lane walks ITS covered tiles; the run base and the covering mask come from the tile's lane
                    const int most = __reduce_max_sync(0xffffffffu, __popc(cover));
                    uint32_t left = cover;
                    for (int q = 0; q < most; ++q) {
                        const int j = left ? __ffs(left) - 1 : 0;
                        const uint32_t mj = __shfl_sync(0xffffffffu, mine, j);
                        const uint32_t bj = __shfl_sync(0xffffffffu, b, j);
                        if (left && bj != 0xffffffffu) pairs[bj + (uint32_t)__popc(mj & lt_mask)] = make_uint2(r.x, r.y);
                        left &= left - 1u;
                    }
                }
                continue;
            }
            for (int c0 = 0; c0 < win; c0 += 32) {
                const int cnt = min(32, win - c0);
                int tyj = row + c0 / Ww, txj = X0 + c0 % Ww;
                uint32_t mine = 0;  // lane j: the lanes whose rect covers window tile c0 + j
                for (int j = 0; j < cnt; ++j) {
                    const bool cov = in && txj >= x0 && txj < x1 && tyj < y1;
                    const uint32_t bal = __ballot_sync(0xffffffffu, cov);
                    if (lane == j) mine = bal;
                    if (++txj == X1) { txj = X0; ++tyj; }
                }
                const int c = c0 + lane;
                const uint32_t t = (uint32_t)((row + c / Ww) * gx + X0 + c % Ww);
                bool has = c < win && mine != 0u;
                if (has && tile_select != nullptr && tile_select[t] == 0u) has = false;
                if (!SCATTER) {
                    if (has) atomicAdd(&tile_count[t], (uint32_t)__popc(mine));
                } else {
                    uint32_t b = 0;
                    if (has) b = tile_offsets[t] + atomicAdd(&cursor[t], (uint32_t)__popc(mine));
                    uint32_t act = __ballot_sync(0xffffffffu, has);
                    while (act) {
                        const int j = __ffs(act) - 1;
                        act &= act - 1u;
                        const uint32_t mj = __shfl_sync(0xffffffffu, mine, j);
                        const uint32_t bj = __shfl_sync(0xffffffffu, b, j);
                        if ((mj >> lane) & 1u) pairs[bj + (uint32_t)__popc(mj & lt_mask)] = make_uint2(r.x, r.y);
                    }
                }
            }
        }
    }
}

// ---- K4: CSR offsets, P, capacity flag and the work lists of the sort -------------------------------
__global__ void __launch_bounds__(kScanThreads)
tile_scan_kernel(int T, const uint32_t* __restrict__ tile_count, uint32_t* __restrict__ tile_offsets, int64_t Pcap,
                 int64_t* __restrict__ P_dev, Counters* __restrict__ ctr, Seg* __restrict__ small_list,
                 Seg* __restrict__ medium_list, Seg* __restrict__ large_list, Seg* __restrict__ giant_list,
                 uint32_t small_cap, uint32_t medium_cap, uint32_t large_cap) {
    __shared__ uint32_t ws[33];
    __shared__ unsigned long long s_carry;
    if (threadIdx.x == 0) s_carry = 0ull;
    __syncthreads();
    constexpr int kPer = 4;
    for (int b0 = 0; b0 < T; b0 += kScanThreads * kPer) {
        const int t0 = b0 + (int)threadIdx.x * kPer;
        uint32_t c[kPer], sum = 0;
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            c[j] = (t0 + j < T) ? tile_count[t0 + j] : 0u;
            sum += c[j];
        }
        uint32_t tot;
        const uint32_t ex = block_excl_scan(sum, ws, tot);
        unsigned long long run = s_carry + ex;
#pragma unroll
        for (int j = 0; j < kPer; ++j) {
            if (t0 + j < T) {
                // offsets are 32-bit; beyond capacity (< 2^30) nothing downstream runs
                const uint32_t st = (uint32_t)(run < (1ull << 32) ? run : 0xffffffffull);
                tile_offsets[t0 + j] = st;
                if (c[j] > 0u) {
                    Seg sg;
                    sg.start = st; sg.len = c[j]; sg.tile = (uint32_t)(t0 + j); sg.in_tmp = 0u;
                    if (c[j] <= small_cap) small_list[atomicAdd(&ctr->n_small, 1u)] = sg;
                    else if (c[j] <= medium_cap) medium_list[atomicAdd(&ctr->n_medium, 1u)] = sg;
                    else if (c[j] <= large_cap) large_list[atomicAdd(&ctr->n_large, 1u)] = sg;
                    else giant_list[atomicAdd(&ctr->n_giant, 1u)] = sg;
                }
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
        (void)Pcap;  // P and the capacity flag were published by K1 (over capacity, K3 counted nothing)
        (void)P_dev;
    }
}

// ---- monotone bucket map ------------------------------------------------------------------------
// key in [kmin, kmax] -> bucket in [0, nb): every step (uint->float, multiply by a positive
// constant, truncate, clamp) is non-decreasing, so bucket order never contradicts key order.
__device__ __forceinline__ float bucket_scale(uint32_t kmin, uint32_t kmax, uint32_t nb) {
    return (float)nb / ((float)(kmax - kmin) + 1.0f);
}
__device__ __forceinline__ uint32_t bucket_of(uint32_t key, uint32_t kmin, float scale, uint32_t nb) {
    return min(nb - 1u, __float2uint_rz(__uint2float_rz(key - kmin) * scale));
}

// block-wide min / max of the depth bits; ws holds 66 words.  Ends with a barrier.
__device__ __forceinline__ void block_minmax(uint32_t& lo, uint32_t& hi, uint32_t* ws) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    lo = __reduce_min_sync(0xffffffffu, lo);
    hi = __reduce_max_sync(0xffffffffu, hi);
    if (lane == 0) { ws[warp] = lo; ws[33 + warp] = hi; }
    __syncthreads();
    lo = __reduce_min_sync(0xffffffffu, lane < nw ? ws[lane] : 0xffffffffu);
    hi = __reduce_max_sync(0xffffffffu, lane < nw ? ws[33 + lane] : 0u);
    __syncthreads();
}

// ---- K6: split the segments that exceed the shared-memory capacity ---------------------------------
__global__ void __launch_bounds__(kCoarseMax)
giant_split_kernel(const Seg* __restrict__ giant_list, Seg* __restrict__ large_list, Counters* __restrict__ ctr,
                   const uint2* __restrict__ pairs, uint2* __restrict__ tmp, const int64_t* __restrict__ P_dev) {
    __shared__ uint32_t hist[kCoarseMax];
    __shared__ uint32_t gstart[kCoarseMax];
    __shared__ uint32_t ws[66];
    __shared__ uint32_t s_ticket;
    if (P_dev[1]) return;
    const uint32_t n_work = *reinterpret_cast<volatile uint32_t*>(&ctr->n_giant);
    if (n_work == 0u) return;
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_ticket = atomicAdd(&ctr->sched_giant, 1u);
        __syncthreads();
        const uint32_t ticket = s_ticket;
        if (ticket >= n_work) break;
        const Seg sg = giant_list[ticket];
        const uint2* src = pairs + sg.start;
        uint32_t lo = 0xffffffffu, hi = 0u;
        for (uint32_t i = threadIdx.x; i < sg.len; i += kCoarseMax) {
            const uint32_t k = src[i].x;
            lo = min(lo, k);
            hi = max(hi, k);
        }
        block_minmax(lo, hi, ws);
        // always kCoarseMax fine buckets; runs of consecutive buckets are then merged into sub-segments
        // of about S elements, so a depth cluster is cut as finely as the bucket map allows
        const uint32_t nb = (uint32_t)kCoarseMax;
        const float scale = bucket_scale(lo, hi, nb);
        hist[threadIdx.x] = 0u;
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < sg.len; i += kCoarseMax) atomicAdd(&hist[bucket_of(src[i].x, lo, scale, nb)], 1u);
        __syncthreads();
        const uint32_t c = hist[threadIdx.x];
        uint32_t tot;
        const uint32_t off = block_excl_scan(c, ws, tot);
        __syncthreads();
        hist[threadIdx.x] = off;  // becomes the bucket's cursor
        // bucket b opens a sub-segment when its offset enters a new block of S elements (S > len / 1024)
        const uint32_t S = max(kSubTarget, sg.len / (uint32_t)kCoarseMax + 1u);  // off / S < kCoarseMax even for off == len
        gstart[threadIdx.x] = 0xffffffffu;
        __syncthreads();
        const uint32_t q = off / S;
        const bool opens = threadIdx.x == 0 || hist[threadIdx.x - 1] / S != q;
        if (opens) gstart[q] = off;  // q < kCoarseMax; one opener per q
        __syncthreads();
        const bool closes = threadIdx.x == kCoarseMax - 1 || hist[threadIdx.x + 1] / S != q;
        if (closes) {
            const uint32_t st = gstart[q], en = off + c;
            if (en > st) {
                Seg sub;
                sub.start = sg.start + st; sub.len = en - st; sub.tile = sg.tile; sub.in_tmp = 1u;
                large_list[atomicAdd(&ctr->n_large, 1u)] = sub;
            }
        }
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < sg.len; i += kCoarseMax) {
            const uint2 kv = src[i];
            tmp[sg.start + atomicAdd(&hist[bucket_of(kv.x, lo, scale, nb)], 1u)] = kv;
        }
    }
}

// ---- fallback: one stable LSD pass src -> dst over `bits` bits at `shift` of word `word` ------------
// (0 = depth, 1 = id).  Warp w owns the contiguous sub-range [w*per_warp, ...) and a private
// histogram row wh[w][*]: count, scan in (digit, warp) order, then rank in range order with match-any.
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

// ---- K7: per-segment sort -----------------------------------------------------------------------------
__device__ __forceinline__ bool pair_less(const uint2 a, const uint2 b) {
    return (((unsigned long long)a.x << 32) | a.y) < (((unsigned long long)b.x << 32) | b.y);
}

template <int CAP, int NBMAX>
struct SortSmem {
    union {
        uint2 B[CAP];             // the segment grouped by bucket (after the rounds)
        uint16_t tab[2][NBMAX];   // write-then-check tables of the rounds
    } u;
    uint32_t cnt[NBMAX + 4];      // bucket counts -> exclusive offsets; histogram rows of the fallback
};

// KEEP: the segment's pairs stay in registers between the passes (otherwise they are re-read, L2 hits).
template <int THREADS, int CAP, int NBMAX, bool KEEP, int MINB>
__global__ void __launch_bounds__(THREADS, MINB)
seg_sort_kernel(const Seg* __restrict__ list, const uint32_t* n_work_ptr, uint32_t* sched, uint2* pairs, uint2* tmp,
                uint32_t* __restrict__ gid_sorted, uint64_t* __restrict__ keys_sorted,
                const int64_t* __restrict__ P_dev, int gid_bits) {
    constexpr int EPT = CAP / THREADS, PER = NBMAX / THREADS, W = THREADS / 32;
    static_assert(PER % 4 == 0 && CAP <= 65535 && NBMAX <= 32768, "layout");
    static_assert(sizeof(uint32_t) * (NBMAX + 4) >= sizeof(uint32_t) * W * (1 << kFbBits), "fallback histogram rows");
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem<CAP, NBMAX>& sm = *reinterpret_cast<SortSmem<CAP, NBMAX>*>(smem_raw);
    __shared__ uint32_t ws[66];
    __shared__ uint32_t s_ticket[2];
    if (P_dev[1]) return;
    const uint32_t n_work = *reinterpret_cast<const volatile uint32_t*>(n_work_ptr);
    if (n_work == 0u) return;  // nothing of this size class: skip the ticket round trip
    const uint32_t tid = threadIdx.x;
    if (tid == 0) s_ticket[0] = atomicAdd(sched, 1u);
    __syncthreads();
    for (uint32_t it = 0;; ++it) {
        const uint32_t ticket = s_ticket[it & 1u];
        if (ticket >= n_work) break;
        if (tid == 0) s_ticket[(it + 1u) & 1u] = atomicAdd(sched, 1u);  // prefetch: its latency hides behind this segment
        const Seg sg = list[ticket];
        uint2* src = (sg.in_tmp ? tmp : pairs) + sg.start;
        uint2* oth = (sg.in_tmp ? pairs : tmp) + sg.start;
        const uint32_t m = sg.len;
        const int nE = (int)((m + THREADS - 1u) / THREADS);  // element slots in use per thread
        bool fb = m > (uint32_t)CAP;  // block-uniform from here on
        uint2 kv[KEEP ? EPT : 1];
        uint32_t lo = 0xffffffffu, hi = 0u;
        if (!fb) {
#pragma unroll
            for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                const uint32_t i = (uint32_t)e * THREADS + tid;
                if (i < m) {
                    const uint2 v = src[i];
                    if (KEEP) kv[KEEP ? e : 0] = v;
                    lo = min(lo, v.x);
                    hi = max(hi, v.x);
                }
            }
        } else {
            for (uint32_t i = tid; i < m; i += THREADS) {
                const uint32_t k = src[i].x;
                lo = min(lo, k);
                hi = max(hi, k);
            }
        }
        block_minmax(lo, hi, ws);  // (its barriers also separate this segment's shared memory from the last one's)
        if (lo == hi && m > kMaxOcc) fb = true;
        if (!fb) {
            uint32_t nb = 32u;
            while (nb < 2u * m && nb < (uint32_t)NBMAX) nb <<= 1;
            const float scale = bucket_scale(lo, hi, nb);
            const uint32_t cbase = tid * PER;
            if (cbase < nb) {
#pragma unroll
                for (int j = 0; j < PER; j += 4) *reinterpret_cast<uint4*>(&sm.cnt[cbase + j]) = make_uint4(0u, 0u, 0u, 0u);
            }
            // state of an element: bucket << 16 | slot inside the bucket (0xffff = pending); 0xffffffff = no element
            uint32_t st[EPT];
#pragma unroll
            for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                const uint32_t i = (uint32_t)e * THREADS + tid;
                st[e] = 0xffffffffu;
                if (i < m) st[e] = (bucket_of(KEEP ? kv[KEEP ? e : 0].x : src[i].x, lo, scale, nb) << 16) | 0xffffu;
            }
            // ---- rounds: the last writer of a bucket's table entry takes the bucket's next slot ----
            for (int r = 0; r < kRounds; ++r) {
                uint16_t* tab = sm.u.tab[r & 1];
                bool any = false;
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                    if (st[e] != 0xffffffffu && (st[e] & 0xffffu) == 0xffffu) {
                        tab[st[e] >> 16] = (uint16_t)((uint32_t)e * THREADS + tid);
                        any = true;
                    }
                }
                if (!__syncthreads_or(any)) break;
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                    if (st[e] != 0xffffffffu && (st[e] & 0xffffu) == 0xffffu) {
                        const uint32_t b = st[e] >> 16;
                        if (tab[b] == (uint16_t)((uint32_t)e * THREADS + tid)) {
                            st[e] = (b << 16) | (uint32_t)r;
                            sm.cnt[b] = (uint32_t)r + 1u;
                        }
                    }
                }
            }
            __syncthreads();
            // crowded buckets: the elements still pending take their slots with atomics
#pragma unroll
            for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                if (st[e] != 0xffffffffu && (st[e] & 0xffffu) == 0xffffu) {
                    const uint32_t b = st[e] >> 16;
                    st[e] = (b << 16) | min(0xfffeu, atomicAdd(&sm.cnt[b], 1u));
                }
            }
            __syncthreads();
            // ---- counts -> exclusive offsets (in place), largest bucket ----
            uint32_t c[PER], sum = 0, mx = 0;
            if (cbase < nb) {
#pragma unroll
                for (int j = 0; j < PER; j += 4) {
                    const uint4 q = *reinterpret_cast<const uint4*>(&sm.cnt[cbase + j]);
                    c[j] = q.x; c[j + 1] = q.y; c[j + 2] = q.z; c[j + 3] = q.w;
                }
#pragma unroll
                for (int j = 0; j < PER; ++j) {
                    sum += c[j];
                    mx = max(mx, c[j]);
                }
            }
            uint32_t tot;
            uint32_t run = block_excl_scan(sum, ws, tot);
            if (cbase < nb) {
#pragma unroll
                for (int j = 0; j < PER; ++j) {
                    sm.cnt[cbase + j] = run;
                    run += c[j];
                }
            }
            if (tid == 0) sm.cnt[nb] = m;
            fb = __syncthreads_or(mx > kMaxOcc) != 0;
            if (!fb) {
                // ---- place by bucket, then order every bucket by counting smaller (depth, id) ----
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                    if (st[e] != 0xffffffffu) {
                        const uint2 v = KEEP ? kv[KEEP ? e : 0] : src[(uint32_t)e * THREADS + tid];
                        sm.u.B[sm.cnt[st[e] >> 16] + (st[e] & 0xffffu)] = v;
                    }
                }
                __syncthreads();
#pragma unroll
                for (int e = 0; e < EPT; ++e) {
                if (e >= nE) break;  // block-uniform
                    const uint32_t i = (uint32_t)e * THREADS + tid;
                    if (i < m) {
                        const uint2 v = sm.u.B[i];
                        const uint32_t b = bucket_of(v.x, lo, scale, nb);
                        const uint32_t s = sm.cnt[b], t = sm.cnt[b + 1];
                        uint32_t rank = s;
                        for (uint32_t j = s; j < t; ++j) rank += pair_less(sm.u.B[j], v) ? 1u : 0u;
                        gid_sorted[sg.start + rank] = v.y;
                        if (keys_sorted) keys_sorted[sg.start + rank] = ((uint64_t)sg.tile << 32) | (uint64_t)v.x;
                    }
                }
            }
        }
        if (fb) {
            // ---- fallback: stable LSD radix sort on (depth, id) in global memory: id digits first,
            //      then every varying depth bit ----
            __syncthreads();
            uint32_t* wh = sm.cnt;
            uint2 *A = src, *Bq = oth;
            int np = (gid_bits + kFbBits - 1) / kFbBits, bt = (gid_bits + np - 1) / np;
            for (int p = 0; p < np; ++p) {
                radix_pass<THREADS>(A, Bq, m, 1, p * bt, bt, wh, ws);
                uint2* x = A; A = Bq; Bq = x;
            }
            const int nbits = 32 - __clz(lo ^ hi);  // depth bits [0, nbits) vary inside this segment
            np = (nbits + kFbBits - 1) / kFbBits;
            bt = np ? (nbits + np - 1) / np : 0;
            for (int p = 0; p < np; ++p) {
                radix_pass<THREADS>(A, Bq, m, 0, p * bt, bt, wh, ws);
                uint2* x = A; A = Bq; Bq = x;
            }
            for (uint32_t i = tid; i < m; i += THREADS) {
                const uint2 v = A[i];
                gid_sorted[sg.start + i] = v.y;
                if (keys_sorted) keys_sorted[sg.start + i] = ((uint64_t)sg.tile << 32) | (uint64_t)v.x;
            }
        }
    }
}

constexpr int kSmallThreads = 256, kSmallCap = 2048, kSmallNb = 4096;
constexpr int kMediumThreads = 1024, kMediumCap = 4096, kMediumNb = 8192;
constexpr int kLargeThreads = 1024, kLargeCap = 8192, kLargeNb = 8192;
constexpr size_t kSmallSmem = sizeof(SortSmem<kSmallCap, kSmallNb>);
constexpr size_t kMediumSmem = sizeof(SortSmem<kMediumCap, kMediumNb>);
constexpr size_t kLargeSmem = sizeof(SortSmem<kLargeCap, kLargeNb>);

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

struct Workspace {
    // zeroed at the start of every call (one memset): counters, histograms, cursors
    Counters* ctr;
    uint32_t *bin_count, *bin_cursor, *tile_count, *cursor;
    size_t zero_bytes;
    uint32_t *bin_offset, *sat, *blk_base;     // blk_base: [regroup blocks][T] when the tile histogram fits shared memory
    uint4* rec;                                // [N] regrouped records
    Seg *small_list, *medium_list, *large_list, *giant_list;
    uint2 *pairs, *tmp;                        // [Pcap] each: unsorted segments; scratch of giant_split / the fallback
    size_t total;
};

Workspace carve(void* base, int N, int T_, int64_t Pcap) {
    Workspace w;
    size_t o = 0;
    char* p = (char*)base;
    auto take = [&](size_t bytes) { char* r = p + o; o += align256(bytes); return r; };
    const size_t nt = (size_t)(T_ > 0 ? T_ : 1), pc = (size_t)(Pcap > 0 ? Pcap : 1), nn = (size_t)(N > 0 ? N : 1);
    w.ctr = (Counters*)take(sizeof(Counters));
    w.bin_count = (uint32_t*)take(nt * 4);
    w.bin_cursor = (uint32_t*)take(nt * 4);
    w.tile_count = (uint32_t*)take(nt * 4);
    w.cursor = (uint32_t*)take(nt * 4);
    w.zero_bytes = o;
    w.bin_offset = (uint32_t*)take(nt * 4);
    w.sat = (uint32_t*)take((2 * nt + 2) * 4);  // (gx+1)(gy+1) <= 2T+2
    w.blk_base = (uint32_t*)take(nt <= (size_t)kSmemTilesMax ? (size_t)kRegroupBlocksMax * nt * 4 : 4);
    w.rec = (uint4*)take(pc * 16);  // every record holds at least one pair: records <= P <= Pcap
    w.small_list = (Seg*)take(nt * sizeof(Seg));
    w.medium_list = (Seg*)take(nt * sizeof(Seg));
    w.large_list = (Seg*)take((2 * nt + pc / kSubTarget + 16) * sizeof(Seg));
    w.giant_list = (Seg*)take(nt * sizeof(Seg));
    w.pairs = (uint2*)take(pc * 8);
    w.tmp = (uint2*)take(pc * 8);
    w.total = o;
    return w;
}

}  // namespace

size_t binsort_workspace_bytes(int N, int64_t Pcap, int T) { return carve(nullptr, N, T, Pcap).total; }

cudaError_t launch_bin_sort(const CamK& cam, int N, const float* splats_f, const uint32_t* tile_select, int64_t Pcap,
                            uint64_t* keys_sorted, uint32_t* gid_sorted, uint32_t* tile_offsets, int64_t* P_dev,
                            void* ws, size_t ws_bytes, int num_sms, cudaStream_t s, const SideStream* side) {
    (void)ws_bytes;
    const int gx = cam.gx, gy = cam.gy, T = gx * gy;
    const Workspace w = carve(ws, N, T, Pcap);
    const float4* splats = reinterpret_cast<const float4*>(splats_f);
    cudaError_t e = cudaMemsetAsync(w.ctr, 0, w.zero_bytes, s);
    if (e != cudaSuccess) return e;

    static SmemOptIn opt[3];  // per device
    e = opt[0].ensure((const void*)seg_sort_kernel<kSmallThreads, kSmallCap, kSmallNb, true, 4>, kSmallSmem);
    if (e != cudaSuccess) return e;
    e = opt[1].ensure((const void*)seg_sort_kernel<kMediumThreads, kMediumCap, kMediumNb, true, 1>, kMediumSmem);
    if (e != cudaSuccess) return e;
    e = opt[2].ensure((const void*)seg_sort_kernel<kLargeThreads, kLargeCap, kLargeNb, true, 1>, kLargeSmem);
    if (e != cudaSuccess) return e;

    // Ks, K0-K2: cut the rects into pieces and regroup them by top-left tile
    int nblk = (N + 255) / 256;
    if (nblk > num_sms * 8) nblk = num_sms * 8;
    if (nblk < 1) nblk = 1;
    uint32_t* sat = nullptr;
    if (tile_select) {
        sat = w.sat;
        select_sat_kernel<<<1, kScanThreads, 0, s>>>(gx, gy, tile_select, sat);
        count_launches(1);
    }
    if (T <= kSmemTilesMax) {
        int rb = num_sms < kRegroupBlocksMax ? num_sms : kRegroupBlocksMax;
        if (rb > (N + 1023) / 1024) rb = (N + 1023) / 1024;
        if (rb < 1) rb = 1;
        const int chunk = (N + rb - 1) / rb;
        const size_t hb = (size_t)T * 4;
        topleft_count_kernel<true><<<rb, 1024, hb, s>>>(N, chunk, gx, gy, splats, sat, w.bin_count, w.blk_base, w.ctr);
        bin_scan_kernel<<<1, kScanThreads, 0, s>>>(T, w.bin_count, w.bin_offset, w.ctr, Pcap, P_dev);
        reorder_kernel<true><<<rb, 1024, hb, s>>>(N, chunk, gx, gy, splats, w.bin_offset, w.bin_cursor, w.blk_base, sat,
                                                   P_dev, w.rec);
    } else {
        const int chunk = (N + nblk - 1) / nblk;
        topleft_count_kernel<false><<<nblk, 256, 0, s>>>(N, chunk, gx, gy, splats, sat, w.bin_count, nullptr, w.ctr);
        bin_scan_kernel<<<1, kScanThreads, 0, s>>>(T, w.bin_count, w.bin_offset, w.ctr, Pcap, P_dev);
        reorder_kernel<false><<<nblk, 256, 0, s>>>(N, chunk, gx, gy, splats, w.bin_offset, w.bin_cursor, nullptr, sat,
                                                    P_dev, w.rec);
    }
    // K3-K5: pair counts, CSR offsets, scatter
    pair_walk_kernel<false><<<nblk, kWalkThreads, 0, s>>>(gx, w.rec, w.ctr, tile_select, w.tile_count, nullptr, nullptr,
                                                          P_dev, nullptr);
    tile_scan_kernel<<<1, kScanThreads, 0, s>>>(T, w.tile_count, tile_offsets, Pcap, P_dev, w.ctr, w.small_list,
                                                w.medium_list, w.large_list, w.giant_list, (uint32_t)kSmallCap,
                                                (uint32_t)kMediumCap, (uint32_t)kLargeCap);
    pair_walk_kernel<true><<<nblk, kWalkThreads, 0, s>>>(gx, w.rec, w.ctr, tile_select, nullptr, tile_offsets, w.cursor,
                                                         P_dev, w.pairs);
    count_launches(6);

    // K6-K7: sort the segments.  The three classes write disjoint ranges: the long ones (giant split, large,
    // medium) run on the context's side stream, concurrently with the short ones on the caller's stream (when a class
    // is empty its launch hides behind the others instead of adding to the call)
    int gid_bits = 1;
    while (gid_bits < 30 && (1ll << gid_bits) < (long long)N) ++gid_bits;
    const bool long_classes = Pcap > kSmallCap;
    if (long_classes) {
        e = cudaEventRecord(side->fork, s);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(side->aux, side->fork, 0);
        if (e != cudaSuccess) return e;
        cudaStream_t a = side->aux;
        if (Pcap > kMediumCap) {  // otherwise no segment is that long
            if (Pcap > kLargeCap) {
                int gb = num_sms < T ? num_sms : T;
                giant_split_kernel<<<gb, kCoarseMax, 0, a>>>(w.giant_list, w.large_list, w.ctr, w.pairs, w.tmp, P_dev);
                count_launches(1);
            }
            int lb = num_sms < T ? num_sms : T;
            seg_sort_kernel<kLargeThreads, kLargeCap, kLargeNb, true, 1><<<lb, kLargeThreads, kLargeSmem, a>>>(
                w.large_list, &w.ctr->n_large, &w.ctr->sched_large, w.pairs, w.tmp, gid_sorted, keys_sorted, P_dev, gid_bits);
            count_launches(1);
        }
        int mb = num_sms < T ? num_sms : T;
        seg_sort_kernel<kMediumThreads, kMediumCap, kMediumNb, true, 1><<<mb, kMediumThreads, kMediumSmem, a>>>(
            w.medium_list, &w.ctr->n_medium, &w.ctr->sched_medium, w.pairs, w.tmp, gid_sorted, keys_sorted, P_dev, gid_bits);
        count_launches(1);
        e = cudaEventRecord(side->join, a);
        if (e != cudaSuccess) return e;
    }
    int sb = num_sms * 6 < T ? num_sms * 6 : T;
    seg_sort_kernel<kSmallThreads, kSmallCap, kSmallNb, true, 4><<<sb, kSmallThreads, kSmallSmem, s>>>(
        w.small_list, &w.ctr->n_small, &w.ctr->sched_small, w.pairs, w.tmp, gid_sorted, keys_sorted, P_dev, gid_bits);
    count_launches(1);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (long_classes) e = cudaStreamWaitEvent(s, side->join, 0);
    return e;
}

}  // namespace tgs