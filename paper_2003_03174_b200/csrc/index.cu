// index.cu -- the tracklet index of trd_load_tracklets.
//
//   a1  tracklet_key     key = ((sector, layer), z row, y bin) from (chamber, z, y)
//   a2  radix_*          stable LSD radix sort of (key, position), 8 bits per pass:
//                        per-tile digit histogram -> per-digit scan over tiles -> stable scatter
//       gather_store     sorted store: one float4 (y, z, dy/dx, position) per tracklet
//   a3  (in gather_store) first sorted position of every bin (plus sentinel), z extent of every row
//
// Large loads take a counting sort instead of the radix passes (same result): the key kernel also counts every bin
// and keeps the value the count had as the tracklet's rank inside its bin (one byte; the atomics run in the caller's
// order, block after block, so a bin is filled almost in that order), one inclusive scan turns the counts into first
// positions, partition_tracklets groups the tracklets by the leading digit of the key so that the placement that follows
// writes complete lines in L2, place_tracklets puts every tracklet at first(bin) + rank without an atomic, and
// order_bins restores the caller's order inside every bin where the ranks did not give it (insertion sort by position,
// one thread per bin) and records the z extents.  A bin longer than kMaxBin sets a device flag: the placement kernels
// return at once and the one-launch sort of small loads (small_index), enqueued behind them and gated on the same
// flag, builds the index instead -- no host round trip.  Loads of up to 2^18 tracklets take small_index directly.
//
// north_star: "device-side sort and index by chamber and local-y bin ... a radix sort plus
// per-chamber y-bin offsets"; the 18 x 5 x 6 segmentation is PAPER.md:50.  The key also
// carries the z row (SURVEY.md 8(d).3 "design consequence"), and it uses (sector, layer)
// rather than the chamber's stack, because the z window may straddle two stacks (reading R12).
// All of it is HBM-streaming integer work; no tensor cores.
#include <cooperative_groups.h>

#include "trd_internal.cuh"

namespace trd {

namespace {

constexpr int kRadixBits = 8;
constexpr int kRadix = 1 << kRadixBits;
constexpr int kSortThreads = 256;
constexpr int kSortWarps = kSortThreads / 32;
constexpr int kItems = 16;                          // keys per thread and tile
constexpr int kTile = kSortThreads * kItems;        // 4096 keys per tile

// also packs (y, z, dy/dx, chamber) into one 16-byte record so that the gather after the sort reads
// one sector per tracklet instead of three
// a1: bin key of one tracklet; unusable tracklets (chamber or interaction out of range, y or z not finite) get n_bins
// and sort behind every bin
__device__ __forceinline__ uint32_t key_of(const IndexGeom& g, float yy, float zz, int ch, int ia) {
    if (ch >= 0 && ch < g.n_chambers && isfinite(yy) && isfinite(zz) && ia >= 0 && ia < g.n_ia) {
        const int sector = ch / g.per_sector, layer = ch % g.n_layers;
        const uint32_t cell = (uint32_t)((ia * g.n_sectors + sector) * g.n_layers + layer);
        return ((cell * (uint32_t)g.nz + (uint32_t)zrow_of(g, zz)) << g.nb_shift) + (uint32_t)ybin_of(g, yy);
    }
    return g.n_bins;
}

constexpr int kKeyItems = 8;                        // tracklets per thread
__global__ void __launch_bounds__(256) tracklet_key(const float* __restrict__ y, const float* __restrict__ z,
                                                    const float* __restrict__ dydx, const int32_t* __restrict__ chamber,
                                                    const int32_t* __restrict__ interaction, uint32_t* __restrict__ key,
                                                    float4* __restrict__ packed, int64_t n, IndexGeom g,
                                                    uint32_t* __restrict__ digit_tot, int shift,
                                                    uint32_t* __restrict__ count, uint8_t* __restrict__ rank) {
    // digit_tot (counting sort): how many keys carry each leading digit, for the partition that follows
    __shared__ uint32_t cnt[kRadix];
    if (digit_tot) {
        cnt[threadIdx.x] = 0;
        __syncthreads();
    }
    const int64_t i0 = (int64_t)blockIdx.x * kKeyItems * 256 + threadIdx.x;
    float yy[kKeyItems], zz[kKeyItems], dd[kKeyItems];
    int ch[kKeyItems], ia[kKeyItems];
    uint32_t k[kKeyItems], rk[kKeyItems];
#pragma unroll
    for (int u = 0; u < kKeyItems; ++u) {
        const int64_t i = i0 + u * 256;
        yy[u] = zz[u] = dd[u] = 0.0f;
        ch[u] = -1;
        ia[u] = 0;
        if (i < n) {
            yy[u] = __ldcs(y + i); zz[u] = __ldcs(z + i); dd[u] = __ldcs(dydx + i);   // streamed: the count table stays in L2
            ch[u] = __ldcs(chamber + i);
            if (g.n_ia > 1) ia[u] = __ldcs(interaction + i);            // time-frame association: the interaction leads the key
        }
    }
#pragma unroll
    for (int u = 0; u < kKeyItems; ++u) {
        k[u] = key_of(g, yy[u], zz[u], ch[u], ia[u]);
        rk[u] = 0u;
        if (count && i0 + u * 256 < n) rk[u] = atomicAdd(count + k[u] + 1, 1u);   // all in flight before the first is used
    }
#pragma unroll
    for (int u = 0; u < kKeyItems; ++u) {
        const int64_t i = i0 + u * 256;
        if (i < n) {
            __stcs(packed + i, make_float4(yy[u], zz[u], dd[u], __int_as_float(ch[u])));
            __stcs(key + i, k[u]);
            if (digit_tot) atomicAdd(&cnt[(k[u] >> shift) & (kRadix - 1)], 1u);
            if (count) __stcs(rank + i, (uint8_t)min(rk[u], 255u));
        }
    }
    if (digit_tot) {
        __syncthreads();
        if (cnt[threadIdx.x]) atomicAdd(digit_tot + threadIdx.x, cnt[threadIdx.x]);
    }
}

// per-tile histogram of one digit; hist[d * n_tiles + tile]
// gate: when given, the kernel runs only if *gate != 0 (the counting sort gave up, see the header)
__global__ void __launch_bounds__(kSortThreads) radix_hist(const uint32_t* __restrict__ key, uint32_t* __restrict__ hist,
                                                           int64_t n, int n_tiles, int shift, const int* __restrict__ gate) {
    __shared__ uint32_t cnt[kRadix];
    if (gate && *gate == 0) return;
    cnt[threadIdx.x] = 0;
    __syncthreads();
    const int64_t base = (int64_t)blockIdx.x * kTile;
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
        const int64_t i = base + r * kSortThreads + threadIdx.x;
        if (i < n) atomicAdd(&cnt[(key[i] >> shift) & (kRadix - 1)], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * n_tiles + blockIdx.x] = cnt[threadIdx.x];
}

__device__ inline uint32_t block_exclusive_scan(uint32_t v, uint32_t* warp_sums, uint32_t* total) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t incl = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        uint32_t w = (lane < (int)(blockDim.x >> 5)) ? warp_sums[lane] : 0u;
        uint32_t wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        warp_sums[lane] = wi - w;                  // exclusive warp offsets; [31] unused beyond n warps
        if (lane == 31) *total = wi;
    }
    __syncthreads();
    return warp_sums[warp] + incl - v;
}

// one block per digit: exclusive scan of that digit's counts over the tiles, total to digit_tot[d]
__global__ void __launch_bounds__(kSortThreads) radix_rowscan(uint32_t* __restrict__ hist, uint32_t* __restrict__ digit_tot,
                                                              int n_tiles, const int* __restrict__ gate) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    if (gate && *gate == 0) return;
    uint32_t* row = hist + (size_t)blockIdx.x * n_tiles;
    uint32_t carry = 0;
    for (int t0 = 0; t0 < n_tiles; t0 += kSortThreads) {
        const int t = t0 + threadIdx.x;
        const uint32_t v = (t < n_tiles) ? row[t] : 0u;
        const uint32_t ex = block_exclusive_scan(v, warp_sums, &total);
        if (t < n_tiles) row[t] = carry + ex;
        carry += total;
        __syncthreads();
    }
    if (threadIdx.x == 0) digit_tot[blockIdx.x] = carry;
}

// stable scatter of one tile.  Order inside a tile is (warp, round, lane): warp w owns the
// contiguous keys [w * kItems * 32, (w + 1) * kItems * 32) of the tile.  The tile is first reordered by
// digit in shared memory so that the global writes go out as contiguous runs per digit.
__global__ void __launch_bounds__(kSortThreads, 3) radix_scatter(const uint32_t* __restrict__ key_in,
                                                              const uint32_t* __restrict__ val_in,
                                                              uint32_t* __restrict__ key_out, uint32_t* __restrict__ val_out,
                                                              const uint32_t* __restrict__ hist,
                                                              const uint32_t* __restrict__ digit_tot, int64_t n, int n_tiles,
                                                              int shift, const int* __restrict__ gate) {
    __shared__ uint32_t warp_cnt[kSortWarps][kRadix];
    if (gate && *gate == 0) return;
    __shared__ uint32_t digit_base[kRadix];    // global position of the tile's first key with digit d
    __shared__ uint32_t tile_off[kRadix];      // position inside the reordered tile of its first key with digit d
    __shared__ uint32_t s_key[kTile], s_val[kTile];
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lt = (1u << lane) - 1u;
#pragma unroll
    for (int w = 0; w < kSortWarps; ++w) warp_cnt[w][threadIdx.x] = 0;
    // global base of digit d for this tile = (keys with a smaller digit) + (same digit in earlier tiles)
    const uint32_t ex = block_exclusive_scan(digit_tot[threadIdx.x], warp_sums, &total);   // syncs
    digit_base[threadIdx.x] = ex + hist[(size_t)threadIdx.x * n_tiles + blockIdx.x];

    const int64_t tile_base = (int64_t)blockIdx.x * kTile;
    const int64_t base = tile_base + (int64_t)warp * (kItems * 32);
    uint32_t k[kItems], v[kItems], rank[kItems];
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
        const int64_t i = base + r * 32 + lane;
        const bool ok = i < n;
        k[r] = ok ? key_in[i] : 0u;
        v[r] = ok ? (val_in ? val_in[i] : (uint32_t)i) : 0u;
    }
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
        const bool ok = base + r * 32 + lane < n;
        const uint32_t d = (k[r] >> shift) & (kRadix - 1);
        // lanes holding the same digit: one ballot per digit bit (fixed cost, unlike MATCH.ANY whose
        // latency grows with the number of distinct values)
        uint32_t peers = __ballot_sync(0xffffffffu, ok);
#pragma unroll
        for (int b = 0; b < kRadixBits; ++b) {
            const uint32_t m = __ballot_sync(0xffffffffu, (d >> b) & 1u);
            peers &= ((d >> b) & 1u) ? m : ~m;
        }
        uint32_t prior = 0;
        if (ok) prior = warp_cnt[warp][d];
        __syncwarp();
        rank[r] = prior + __popc(peers & lt);
        if (ok && (peers & lt) == 0) warp_cnt[warp][d] = prior + __popc(peers);
        __syncwarp();
    }
    __syncthreads();
    uint32_t mine = 0;
    {   // exclusive scan over the warps, per digit
#pragma unroll
        for (int w = 0; w < kSortWarps; ++w) {
            const uint32_t c = warp_cnt[w][threadIdx.x];
            warp_cnt[w][threadIdx.x] = mine;
            mine += c;
        }
    }
    tile_off[threadIdx.x] = block_exclusive_scan(mine, warp_sums, &total);                  // syncs
    __syncthreads();
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
        if (base + r * 32 + lane < n) {
            const uint32_t d = (k[r] >> shift) & (kRadix - 1);
            const uint32_t lp = tile_off[d] + warp_cnt[warp][d] + rank[r];
            s_key[lp] = k[r];
            s_val[lp] = v[r];
        }
    }
    __syncthreads();
    const int n_here = (int)min((int64_t)kTile, n - tile_base);
#pragma unroll
    for (int r = 0; r < kItems; ++r) {
        const int j = r * kSortThreads + threadIdx.x;
        if (j < n_here) {
            const uint32_t kk = s_key[j];
            const uint32_t d = (kk >> shift) & (kRadix - 1);
            const uint32_t dst = digit_base[d] + ((uint32_t)j - tile_off[d]);
            key_out[dst] = kk;
            val_out[dst] = s_val[j];
        }
    }
}

// Counting sort of large loads: partition by the leading digit of the key, the tracklet itself travelling along (rec_out
// gets (y, z, dy/dx, position), dx_out the radial offset of its chamber, rank_out its rank inside its bin), so that the
// placement that follows finds the tracklets of one bucket, and their bins, close together in L2.  The order inside a
// bucket is free, hence no stable ranking: ranks inside the tile and the tile's place inside the bucket come from atomic
// counters; the tile is reordered in shared memory so that the global writes are runs per digit.
struct Partition {
    const float4* packed;
    float4* rec_out;
    const float* chamber_dx;
    float* dx_out;
    uint32_t* count;
    const uint8_t* rank_in; // place of the tracklet inside its bin (the value the count had when the key kernel counted it)
    uint8_t* rank_out;
    int n_chambers;
};
constexpr int kPartItems = 8;
constexpr int kPartTile = 256 * kPartItems;
constexpr size_t kPartSmem = (size_t)kPartTile * (sizeof(float4) + 2 * sizeof(uint32_t) + 1);

__global__ void __launch_bounds__(256) partition_tracklets(const uint32_t* __restrict__ key_in, uint32_t* __restrict__ key_out,
                                                           const Partition pl, const uint32_t* __restrict__ digit_tot,
                                                           uint32_t* __restrict__ cursor, int64_t n, int shift) {
    extern __shared__ float4 s_dyn[];
    float4* const s_rec = s_dyn;
    uint32_t* const s_key = reinterpret_cast<uint32_t*>(s_rec + kPartTile);
    uint32_t* const s_pos = s_key + kPartTile;
    uint8_t* const s_rank = reinterpret_cast<uint8_t*>(s_pos + kPartTile);
    __shared__ uint32_t s_cnt[kRadix], s_base[kRadix], s_off[kRadix];
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    s_cnt[threadIdx.x] = 0;
    const uint32_t start = block_exclusive_scan(digit_tot[threadIdx.x], warp_sums, &total);     // syncs
    const int64_t tile_base = (int64_t)blockIdx.x * kPartTile;
    uint32_t k[kPartItems], rank[kPartItems];
    uint8_t rb[kPartItems];
    float4 r[kPartItems];
#pragma unroll
    for (int u = 0; u < kPartItems; ++u) {
        const int64_t i = tile_base + u * 256 + threadIdx.x;
        k[u] = 0u;
        rb[u] = 0;
        r[u] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (i < n) {
            k[u] = key_in[i];
            r[u] = pl.packed[i];
            rb[u] = pl.rank_in[i];
        }
    }
#pragma unroll
    for (int u = 0; u < kPartItems; ++u) {
        rank[u] = 0u;
        if (tile_base + u * 256 + threadIdx.x < n) rank[u] = atomicAdd(&s_cnt[(k[u] >> shift) & (kRadix - 1)], 1u);
    }
    __syncthreads();
    const uint32_t c = s_cnt[threadIdx.x];
    s_base[threadIdx.x] = start + (c ? atomicAdd(cursor + threadIdx.x, c) : 0u);
    s_off[threadIdx.x] = block_exclusive_scan(c, warp_sums, &total);                             // syncs
    __syncthreads();
#pragma unroll
    for (int u = 0; u < kPartItems; ++u) {
        const int64_t i = tile_base + u * 256 + threadIdx.x;
        if (i < n) {
            const uint32_t lp = s_off[(k[u] >> shift) & (kRadix - 1)] + rank[u];
            s_rec[lp] = r[u];
            s_key[lp] = k[u];
            s_pos[lp] = (uint32_t)i;
            s_rank[lp] = rb[u];
        }
    }
    __syncthreads();
    const int n_here = (int)min((int64_t)kPartTile, n - tile_base);
#pragma unroll
    for (int u = 0; u < kPartItems; ++u) {
        const int j = u * 256 + threadIdx.x;
        if (j < n_here) {
            const uint32_t kk = s_key[j];
            const uint32_t d = (kk >> shift) & (kRadix - 1);
            const uint32_t dst = s_base[d] + ((uint32_t)j - s_off[d]);
            const float4 tl = s_rec[j];
            key_out[dst] = kk;
            pl.rec_out[dst] = make_float4(tl.x, tl.y, tl.z, __uint_as_float(s_pos[j]));
            if (pl.dx_out) {
                const int ch = __float_as_int(tl.w);
                pl.dx_out[dst] = (ch >= 0 && ch < pl.n_chambers) ? __ldg(pl.chamber_dx + ch) : 0.0f;
            }
            pl.rank_out[dst] = s_rank[j];
        }
    }
}

// also records the z extent of every (cell, z row): row_ext[row] = (min, max) of the encoded z.  The keys are
// sorted, so a warp almost always lies inside one row: one warp reduction and two atomics per warp.  Each
// thread handles kGather tracklets (independent random 16-byte reads in flight), strided by the block size.
constexpr int kGather = 4;

__global__ void __launch_bounds__(256) gather_store(const uint32_t* __restrict__ pos, const uint32_t* __restrict__ key,
                                                    const float4* __restrict__ packed, float4* __restrict__ store,
                                                    uint2* __restrict__ row_ext, int32_t* __restrict__ bin_first,
                                                    const float* __restrict__ chamber_dx, float* __restrict__ store_dx,
                                                    int n_chambers, int64_t n, uint32_t n_bins, int nb_shift,
                                                    const int* __restrict__ gate) {
    if (gate && *gate == 0) return;
    const int64_t base = (int64_t)blockIdx.x * (256 * kGather) + threadIdx.x;
    float4 tl[kGather];
    uint32_t k[kGather], kprev[kGather], p[kGather];
#pragma unroll
    for (int u = 0; u < kGather; ++u) {
        const int64_t i = base + u * 256;
        if (i < n) {
            p[u] = pos[i];
            tl[u] = __ldg(packed + p[u]);
            k[u] = key[i];
            kprev[u] = (i == 0) ? 0u : key[i - 1];
        }
    }
#pragma unroll
    for (int u = 0; u < kGather; ++u) {
        const int64_t i = base + u * 256;
        const bool ok = i < n;
        uint32_t row = 0xffffffffu, zlo = 0xffffffffu, zhi = 0u;
        if (ok) {
            const int ch = __float_as_int(tl[u].w);
            store[i] = make_float4(tl[u].x, tl[u].y, tl[u].z, __uint_as_float(p[u]));      // (y, z, dy/dx, position)
            if (store_dx) store_dx[i] = (ch >= 0 && ch < n_chambers) ? __ldg(chamber_dx + ch) : 0.0f;
            {   // a3: bin_first[b] = first sorted position whose key is >= b, for b = 0..n_bins (boundary detection)
                const uint32_t kc = min(k[u], n_bins);
                const int64_t lo = (i == 0) ? 0 : (int64_t)min(kprev[u], n_bins) + 1;
                for (int64_t b = lo; b <= (int64_t)kc; ++b) bin_first[b] = (int32_t)i;
                if (i == n - 1)
                    for (int64_t b = (int64_t)kc + 1; b <= (int64_t)n_bins; ++b) bin_first[b] = (int32_t)n;
            }
            if (row_ext && k[u] < n_bins) {
                row = k[u] >> nb_shift;
                zlo = zhi = ext_encode(tl[u].y);
            }
        }
        const uint32_t row0 = __shfl_sync(0xffffffffu, row, 0);
        if (__all_sync(0xffffffffu, row == row0)) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                zlo = min(zlo, __shfl_xor_sync(0xffffffffu, zlo, o));
                zhi = max(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
            }
            if ((threadIdx.x & 31) == 0 && row != 0xffffffffu) {
                atomicMin(&row_ext[row].x, zlo);
                atomicMax(&row_ext[row].y, zhi);
            }
        } else if (row != 0xffffffffu) {
            atomicMin(&row_ext[row].x, zlo);
            atomicMax(&row_ext[row].y, zhi);
        }
    }
}

// ---- counting sort of large loads (see the header) ---------------------------------------------------------------
constexpr int kMaxBin = 32;                         // longest bin order_bins sorts; longer -> radix path
constexpr int kScanItems = 16;
constexpr int kScanChunk = 256 * kScanItems;        // table entries per block

// sum of every chunk of the count table; flags a bin (entries 1 .. n_bins; the unusable tracklets behind them
// are never read and need no order) longer than kMaxBin
__global__ void __launch_bounds__(256) count_reduce(const uint32_t* __restrict__ tab, uint32_t* __restrict__ partial, int64_t m,
                                                    int64_t n_bins, int* __restrict__ flag) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
    uint32_t sum = 0, longest = 0;
#pragma unroll
    for (int q = 0; q < kScanItems / 4; ++q) {
        const int64_t j = base + 4 * q;
        uint32_t v[4] = {0u, 0u, 0u, 0u};
        if (j + 3 < m) {
            const uint4 t = *reinterpret_cast<const uint4*>(tab + j);
            v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (j + u < m) v[u] = tab[j + u];
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            sum += v[u];
            if (j + u >= 1 && j + u < n_bins + 1) longest = max(longest, v[u]);
        }
    }
    if (longest > (uint32_t)kMaxBin) *flag = 1;
    block_exclusive_scan(sum, warp_sums, &total);
    if (threadIdx.x == 0) partial[blockIdx.x] = total;
}

// exclusive scan of the chunk sums, one block
__global__ void __launch_bounds__(1024) count_scan_partials(uint32_t* __restrict__ partial, int n_chunks) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    uint32_t carry = 0;
    for (int t0 = 0; t0 < n_chunks; t0 += 1024) {
        const int t = t0 + threadIdx.x;
        const uint32_t v = (t < n_chunks) ? partial[t] : 0u;
        const uint32_t ex = block_exclusive_scan(v, warp_sums, &total);
        if (t < n_chunks) partial[t] = carry + ex;
        carry += total;
        __syncthreads();
    }
}

// inclusive scan of the table in place
__global__ void __launch_bounds__(256) count_apply(uint32_t* __restrict__ tab, const uint32_t* __restrict__ partial, int64_t m) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    const int64_t base = (int64_t)blockIdx.x * kScanChunk + (int64_t)threadIdx.x * kScanItems;
    uint32_t v[kScanItems];
#pragma unroll
    for (int q = 0; q < kScanItems / 4; ++q) {
        const int64_t j = base + 4 * q;
        if (j + 3 < m) {
            const uint4 t = *reinterpret_cast<const uint4*>(tab + j);
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u) v[4 * q + u] = (j + u < m) ? tab[j + u] : 0u;
        }
    }
#pragma unroll
    for (int u = 1; u < kScanItems; ++u) v[u] += v[u - 1];
    const uint32_t off = partial[blockIdx.x] + block_exclusive_scan(v[kScanItems - 1], warp_sums, &total);
#pragma unroll
    for (int q = 0; q < kScanItems / 4; ++q) {
        const int64_t j = base + 4 * q;
        if (j + 3 < m) {
            *reinterpret_cast<uint4*>(tab + j) = make_uint4(v[4 * q] + off, v[4 * q + 1] + off, v[4 * q + 2] + off, v[4 * q + 3] + off);
        } else {
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (j + u < m) tab[j + u] = v[4 * q + u] + off;
        }
    }
}

// every tracklet to its place: tab[k] = first sorted position whose key is >= k (the table the match kernel reads), rank
// from the key kernel.  The input is partitioned by the leading key digit (partition_tracklets): the blocks running at
// one time work on a few buckets, whose table entries and store lines stay in L2 until they are complete.
__global__ void __launch_bounds__(256) place_tracklets(const uint32_t* __restrict__ key, const uint8_t* __restrict__ rank,
                                                       const float4* __restrict__ rec, const float* __restrict__ rec_dx,
                                                       const uint32_t* __restrict__ tab, uint32_t* __restrict__ cursor,
                                                       float4* __restrict__ store, float* __restrict__ store_dx, int64_t n,
                                                       uint32_t n_bins, const int* __restrict__ flag) {
    if (*flag != 0) return;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t k = key[i];
    // usable tracklets: first position of the bin + the rank taken when the bin was counted (bins are at most kMaxBin long
    // here); the unusable ones behind the last bin, in any order
    const uint32_t pos = __ldg(tab + k) + (k < n_bins ? (uint32_t)rank[i] : atomicAdd(cursor, 1u));
    store[pos] = rec[i];
    if (store_dx) store_dx[pos] = rec_dx[i];
}

// one thread per bin: the caller's order inside the bin (what the stable radix sort gives; the match kernel breaks
// score ties of duplicate tracklets by store position, reading R6), and the z extent of every (cell, z row)
__global__ void __launch_bounds__(256) order_bins(const uint32_t* __restrict__ tab, float4* __restrict__ store,
                                                  float* __restrict__ store_dx, uint2* __restrict__ row_ext, int64_t n_bins,
                                                  int nb_shift, const int* __restrict__ flag) {
    if (*flag != 0) return;
    const int64_t b = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t row = 0xffffffffu, zlo = 0xffffffffu, zhi = 0u;
    if (b < n_bins) {
        const uint32_t a = tab[b], e = tab[b + 1];
        if (e > a) {
            float4 prev = store[a];
            row = (uint32_t)(b >> nb_shift);
            zlo = zhi = ext_encode(prev.y);
            for (uint32_t i = a + 1; i < e; ++i) {
                float4 v = store[i];
                const uint32_t z = ext_encode(v.y);
                zlo = min(zlo, z);
                zhi = max(zhi, z);
                if (__float_as_uint(prev.w) > __float_as_uint(v.w)) {       // out of order: sink v
                    const float dxv = store_dx ? store_dx[i] : 0.0f;
                    uint32_t j = i;
                    while (j > a) {
                        const float4 u = store[j - 1];
                        if (__float_as_uint(u.w) < __float_as_uint(v.w)) break;
                        store[j] = u;
                        if (store_dx) store_dx[j] = store_dx[j - 1];
                        --j;
                    }
                    store[j] = v;
                    if (store_dx) store_dx[j] = dxv;
                    v = store[i];
                }
                prev = v;
            }
        }
    }
    if (!row_ext) return;
    const uint32_t row0 = __reduce_min_sync(0xffffffffu, row);      // empty bins carry 0xffffffff and neutral extents
    if (__all_sync(0xffffffffu, row == row0 || row == 0xffffffffu)) {
        zlo = __reduce_min_sync(0xffffffffu, zlo);
        zhi = __reduce_max_sync(0xffffffffu, zhi);
        if ((threadIdx.x & 31) == 0 && row0 != 0xffffffffu) {
            atomicMin(&row_ext[row0].x, zlo);
            atomicMax(&row_ext[row0].y, zhi);
        }
    } else if (row != 0xffffffffu) {
        atomicMin(&row_ext[row].x, zlo);
        atomicMax(&row_ext[row].y, zhi);
    }
}

// ---- small loads: the whole index in ONE cooperative launch ---------------------------------------------------------
// An event of the paper's size (about 2000 tracks, here 7 000 - 240 000 tracklets) is launch bound: the
// radix path is eleven launches of a few microseconds each.  This kernel runs the counting sort of the large loads as
// phases of one grid, separated by grid barriers: zero the tables | key + count per bin | scan (three steps) | place
// (atomic cursor per bin) | order every bin by the caller's position and record the z extents | long bins.  There is
// no radix fallback behind it: a bin longer than kMaxBin is put in order by a whole block -- up to kSmallBitonic
// tracklets by a bitonic sort in shared memory, longer ones (at most n / kSmallBitonic of them) by walking the caller's
// arrays in order and writing the bin's members as they come.
constexpr int64_t kSmallMax = 1 << 18;              // loads up to this many tracklets
constexpr int kSmallThreads = 512;
constexpr int kSmallScan = 8;                       // table entries per thread and chunk
constexpr int kSmallChunk = kSmallThreads * kSmallScan;
constexpr int kSmallBitonic = 4096;

struct SmallIndex {
    const float *y, *z, *dydx;
    const int32_t *chamber, *interaction;
    uint32_t* key;          // caller order (trd_copy_index)
    float4* packed;         // caller order (trd_refit)
    float4* store;
    float* store_dx;
    const float* chamber_dx;
    uint32_t *tab, *cursor, *partial, *long_list, *long_count;
    const int* gate;        // when given, the kernel runs only if *gate != 0 (fallback of the multi-kernel counting sort)
    uint2* row_ext;
    int64_t n;
    uint32_t n_rows;
    IndexGeom g;
};

__device__ __forceinline__ void row_extent(uint2* row_ext, uint32_t row, uint32_t zlo, uint32_t zhi) {
    // called by whole warps; lanes without a row carry 0xffffffff and neutral extents
    const uint32_t row0 = __reduce_min_sync(0xffffffffu, row);
    if (__all_sync(0xffffffffu, row == row0 || row == 0xffffffffu)) {
        zlo = __reduce_min_sync(0xffffffffu, zlo);
        zhi = __reduce_max_sync(0xffffffffu, zhi);
        if ((threadIdx.x & 31) == 0 && row0 != 0xffffffffu) {
            atomicMin(&row_ext[row0].x, zlo);
            atomicMax(&row_ext[row0].y, zhi);
        }
    } else if (row != 0xffffffffu) {
        atomicMin(&row_ext[row].x, zlo);
        atomicMax(&row_ext[row].y, zhi);
    }
}

__global__ void __launch_bounds__(kSmallThreads) small_index(const SmallIndex a) {
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
    __shared__ unsigned long long s_sort[kSmallBitonic];       // (position << 32 | slot) of a long bin
    if (a.gate && *a.gate == 0) return;                        // every block: nobody reaches a grid barrier
    const IndexGeom& g = a.g;
    const int64_t tid = (int64_t)blockIdx.x * kSmallThreads + threadIdx.x, n_thr = (int64_t)gridDim.x * kSmallThreads;
    const int64_t m = (int64_t)g.n_bins + 3;                   // table entries; counts live at [key + 1]
    const int n_chunks = (int)((m + kSmallChunk - 1) / kSmallChunk);
    // ---- zero the tables
    for (int64_t j = tid; j < m; j += n_thr) {
        a.tab[j] = 0;
        a.cursor[j] = 0;
    }
    if (a.row_ext)
        for (int64_t j = tid; j < a.n_rows; j += n_thr) a.row_ext[j] = make_uint2(0xffffffffu, 0u);   // empty: min > max
    if (tid == 0) *a.long_count = 0;
    grid.sync();
    // ---- a1: key, packed copy, count per bin
    for (int64_t i = tid; i < a.n; i += n_thr) {
        const float yy = a.y[i], zz = a.z[i];
        const int ch = a.chamber[i];
        const uint32_t k = key_of(g, yy, zz, ch, (g.n_ia > 1) ? a.interaction[i] : 0);
        a.key[i] = k;
        a.packed[i] = make_float4(yy, zz, a.dydx[i], __int_as_float(ch));
        atomicAdd(a.tab + k + 1, 1u);
    }
    grid.sync();
    // ---- a3: inclusive scan of the table -> tab[k] = first sorted position whose key is >= k
    for (int c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const int64_t base = (int64_t)c * kSmallChunk + (int64_t)threadIdx.x * kSmallScan;
        uint32_t sum = 0;
#pragma unroll
        for (int u = 0; u < kSmallScan; ++u) sum += (base + u < m) ? a.tab[base + u] : 0u;
        block_exclusive_scan(sum, warp_sums, &total);
        if (threadIdx.x == 0) a.partial[c] = total;
        __syncthreads();
    }
    grid.sync();
    if (blockIdx.x == 0) {
        uint32_t carry = 0;
        for (int t0 = 0; t0 < n_chunks; t0 += kSmallThreads) {
            const int t = t0 + threadIdx.x;
            const uint32_t v = (t < n_chunks) ? a.partial[t] : 0u;
            const uint32_t ex = block_exclusive_scan(v, warp_sums, &total);
            if (t < n_chunks) a.partial[t] = carry + ex;
            carry += total;
            __syncthreads();
        }
    }
    grid.sync();
    for (int c = blockIdx.x; c < n_chunks; c += gridDim.x) {
        const int64_t base = (int64_t)c * kSmallChunk + (int64_t)threadIdx.x * kSmallScan;
        uint32_t v[kSmallScan];
#pragma unroll
        for (int u = 0; u < kSmallScan; ++u) v[u] = (base + u < m) ? a.tab[base + u] : 0u;
#pragma unroll
        for (int u = 1; u < kSmallScan; ++u) v[u] += v[u - 1];
        const uint32_t off = a.partial[c] + block_exclusive_scan(v[kSmallScan - 1], warp_sums, &total);
#pragma unroll
        for (int u = 0; u < kSmallScan; ++u)
            if (base + u < m) a.tab[base + u] = v[u] + off;
        __syncthreads();
    }
    grid.sync();
    // ---- a2: every tracklet to the next free place of its bin (order inside the bin restored below)
    for (int64_t i = tid; i < a.n; i += n_thr) {
        const uint32_t k = a.key[i];
        const uint32_t pos = a.tab[k] + atomicAdd(a.cursor + k, 1u);
        const float4 tl = a.packed[i];
        a.store[pos] = make_float4(tl.x, tl.y, tl.z, __uint_as_float((uint32_t)i));
        if (a.store_dx) {
            const int ch = __float_as_int(tl.w);
            a.store_dx[pos] = (ch >= 0 && ch < g.n_chambers) ? __ldg(a.chamber_dx + ch) : 0.0f;
        }
    }
    grid.sync();
    // ---- the caller's order inside every bin, z extent of every row; long bins go on a list
    const int64_t n_bins_up = ((int64_t)g.n_bins + 31) / 32 * 32;
    for (int64_t b = tid; b < n_bins_up; b += n_thr) {
        uint32_t row = 0xffffffffu, zlo = 0xffffffffu, zhi = 0u;
        if (b < g.n_bins) {
            const uint32_t s0 = a.tab[b], e = a.tab[b + 1];
            if (e - s0 > (uint32_t)kMaxBin) {
                a.long_list[atomicAdd(a.long_count, 1u)] = (uint32_t)b;
            } else if (e > s0) {
                float4 prev = a.store[s0];
                row = (uint32_t)(b >> g.nb_shift);
                zlo = zhi = ext_encode(prev.y);
                for (uint32_t i = s0 + 1; i < e; ++i) {
                    float4 v = a.store[i];
                    const uint32_t z = ext_encode(v.y);
                    zlo = min(zlo, z);
                    zhi = max(zhi, z);
                    if (__float_as_uint(prev.w) > __float_as_uint(v.w)) {       // out of order: sink v
                        const float dxv = a.store_dx ? a.store_dx[i] : 0.0f;
                        uint32_t j = i;
                        while (j > s0) {
                            const float4 u = a.store[j - 1];
                            if (__float_as_uint(u.w) < __float_as_uint(v.w)) break;
                            a.store[j] = u;
                            if (a.store_dx) a.store_dx[j] = a.store_dx[j - 1];
                            --j;
                        }
                        a.store[j] = v;
                        if (a.store_dx) a.store_dx[j] = dxv;
                        v = a.store[i];
                    }
                    prev = v;
                }
            }
        }
        if (a.row_ext) row_extent(a.row_ext, row, zlo, zhi);
    }
    grid.sync();
    // ---- long bins: one block each
    const uint32_t n_long = *a.long_count;
    for (uint32_t q = blockIdx.x; q < n_long; q += gridDim.x) {
        const uint32_t b = a.long_list[q];
        const uint32_t s0 = a.tab[b], c = a.tab[b + 1] - s0;
        if (a.row_ext) {                                             // z extent of the bin's row
            for (uint32_t i0 = 0; i0 < c; i0 += kSmallThreads) {
                const uint32_t i = i0 + threadIdx.x;
                uint32_t zlo = 0xffffffffu, zhi = 0u, row = 0xffffffffu;
                if (i < c) {
                    zlo = zhi = ext_encode(a.store[s0 + i].y);
                    row = b >> g.nb_shift;
                }
                row_extent(a.row_ext, row, zlo, zhi);
            }
        }
        if (c <= (uint32_t)kSmallBitonic) {
            // (position, slot) pairs sorted in shared memory; then every place takes the record of its rank
            for (uint32_t i = threadIdx.x; i < (uint32_t)kSmallBitonic; i += kSmallThreads)
                s_sort[i] = (i < c) ? (((unsigned long long)__float_as_uint(a.store[s0 + i].w) << 32) | i) : ~0ull;
            __syncthreads();
            for (uint32_t k2 = 2; k2 <= (uint32_t)kSmallBitonic; k2 <<= 1)
                for (uint32_t j = k2 >> 1; j > 0; j >>= 1) {
                    for (uint32_t i = threadIdx.x; i < (uint32_t)kSmallBitonic; i += kSmallThreads) {
                        const uint32_t l = i ^ j;
                        if (l > i) {
                            const unsigned long long x = s_sort[i], w = s_sort[l];
                            if (((i & k2) == 0) ? (x > w) : (x < w)) {
                                s_sort[i] = w;
                                s_sort[l] = x;
                            }
                        }
                    }
                    __syncthreads();
                }
            // gather: rank r takes the record that sits in slot (s_sort[r] & 0xffffffff); read all, sync, write all
            float4 rec[kSmallBitonic / kSmallThreads];
            float dxs[kSmallBitonic / kSmallThreads];
#pragma unroll
            for (int u = 0; u < kSmallBitonic / kSmallThreads; ++u) {
                const uint32_t r = u * kSmallThreads + threadIdx.x;
                if (r < c) {
                    const uint32_t slot = (uint32_t)(s_sort[r] & 0xffffffffull);
                    rec[u] = a.store[s0 + slot];
                    dxs[u] = a.store_dx ? a.store_dx[s0 + slot] : 0.0f;
                }
            }
            __syncthreads();
#pragma unroll
            for (int u = 0; u < kSmallBitonic / kSmallThreads; ++u) {
                const uint32_t r = u * kSmallThreads + threadIdx.x;
                if (r < c) {
                    a.store[s0 + r] = rec[u];
                    if (a.store_dx) a.store_dx[s0 + r] = dxs[u];
                }
            }
            __syncthreads();
        } else {
            // walk the caller's arrays in order: the members of the bin come out in the caller's order
            uint32_t done = 0;
            for (int64_t i0 = 0; i0 < a.n; i0 += kSmallThreads) {
                const int64_t i = i0 + threadIdx.x;
                const bool mine = i < a.n && a.key[i] == b;
                const uint32_t ex = block_exclusive_scan(mine ? 1u : 0u, warp_sums, &total);
                if (mine) {
                    const float4 tl = a.packed[i];
                    a.store[s0 + done + ex] = make_float4(tl.x, tl.y, tl.z, __uint_as_float((uint32_t)i));
                    if (a.store_dx) {
                        const int ch = __float_as_int(tl.w);
                        a.store_dx[s0 + done + ex] = (ch >= 0 && ch < g.n_chambers) ? __ldg(a.chamber_dx + ch) : 0.0f;
                    }
                }
                done += total;
                __syncthreads();
            }
        }
    }
}

// trd_copy_index after a counting sort: the sorted positions and keys the radix path leaves behind
__global__ void __launch_bounds__(256) export_sorted(const float4* __restrict__ store, const uint32_t* __restrict__ key,
                                                     uint32_t* __restrict__ sorted_pos, uint32_t* __restrict__ sorted_key, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint32_t p = __float_as_uint(store[i].w);
    sorted_pos[i] = p;
    sorted_key[i] = key[p];
}

constexpr int64_t kCountingMin = 1 << 18;           // index_sort = 0: loads of at least this many tracklets are counting-sorted

inline int ceil_log2(uint64_t v) {
    int b = 0;
    while ((1ull << b) < v) ++b;
    return b;
}

}  // namespace

#define TRD_TRY(expr)                              \
    do {                                           \
        cudaError_t e_ = (expr);                   \
        if (e_ != cudaSuccess) return e_;          \
    } while (0)

cudaError_t reserve(Buffer& b, size_t bytes, cudaStream_t stream) {
    if (bytes <= b.bytes) return cudaSuccess;
    if (b.p) {
        TRD_TRY(cudaStreamSynchronize(stream));
        TRD_TRY(cudaFree(b.p));
        b.p = nullptr;
        b.bytes = 0;
    }
    const size_t want = bytes + bytes / 8 + 256;    // a little head room against regrowth
    TRD_TRY(cudaMalloc(&b.p, want));
    b.bytes = want;
    return cudaSuccess;
}

int radix_tiles(int64_t n) { return (int)((n + kTile - 1) / kTile); }

// stable LSD radix sort of (key, position) pairs, 8 bits per pass; positions start as 0..n-1.
// key0/val0 and key1/val1 ping-pong; *side tells which pair holds the result.
cudaError_t radix_sort_pairs(uint32_t* key0, uint32_t* key1, uint32_t* val0, uint32_t* val1, uint32_t* tile_hist,
                             uint32_t* digit_tot, int64_t n, int n_passes, cudaStream_t stream, int* side_out,
                             int64_t* launches, const int* gate) {
    const int n_tiles = radix_tiles(n);
    uint32_t* key[2] = {key0, key1};
    uint32_t* val[2] = {val0, val1};
    int side = 0;
    for (int p = 0; p < n_passes; ++p) {
        const int sh = p * kRadixBits;
        const uint32_t* kin = key[side];
        const uint32_t* vin = (p == 0) ? nullptr : val[side];
        radix_hist<<<n_tiles, kSortThreads, 0, stream>>>(kin, tile_hist, n, n_tiles, sh, gate);
        radix_rowscan<<<kRadix, kSortThreads, 0, stream>>>(tile_hist, digit_tot, n_tiles, gate);
        radix_scatter<<<n_tiles, kSortThreads, 0, stream>>>(kin, vin, key[side ^ 1], val[side ^ 1], tile_hist, digit_tot, n,
                                                           n_tiles, sh, gate);
        *launches += 3;
        side ^= 1;
    }
    *side_out = side;
    return cudaGetLastError();
}

// trd_copy_index: sorted positions and keys into val[sorted_side] / key[sorted_side] when the counting sort built the store
cudaError_t export_sorted_index(trd_handle* h, cudaStream_t stream) {
    if ((h->sort_kind != 1 && h->sort_kind != 3) || h->n_tracklets == 0) return cudaSuccess;
    int flag = 0;
    if (h->sort_kind == 1) {
    TRD_TRY(cudaMemcpyAsync(&flag, h->sort_flag.p, sizeof(int), cudaMemcpyDeviceToHost, stream));
    TRD_TRY(cudaStreamSynchronize(stream));
    if (flag != 0) h->sort_kind = 2;                   // a bin was too long: the one-launch sort did the work
    }
    const int64_t n = h->n_tracklets;
    h->sorted_side = 1;
    export_sorted<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>((const float4*)h->store.p, (const uint32_t*)h->key[0].p,
                                                                  (uint32_t*)h->val[1].p, (uint32_t*)h->key[1].p, n);
    TRD_TRY(cudaGetLastError());
    return cudaStreamSynchronize(stream);
}

// the whole index in one cooperative launch; with `gate` the launch is the fallback of the multi-kernel counting sort
// and does nothing unless the device flag is set
static cudaError_t launch_small_index(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx, const int32_t* d_chamber,
                                      const int32_t* d_interaction, int64_t n, size_t n_tab, int64_t n_cells, const int* gate,
                                      cudaStream_t stream) {
    const IndexGeom& g = h->mp.g;
    const bool has_dx = h->mp.dx_max > 0.0f;
    TRD_TRY(reserve(h->store, ((size_t)n + kStorePad) * sizeof(float4), stream));
    TRD_TRY(reserve(h->packed, (size_t)n * sizeof(float4), stream));
    if (has_dx) TRD_TRY(reserve(h->store_dx, ((size_t)n + kStorePad) * sizeof(float), stream));
    for (int sd = 0; sd < 2; ++sd) {                                  // [0]: keys in caller order / list of long bins;
        TRD_TRY(reserve(h->key[sd], (size_t)n * sizeof(uint32_t), stream));   // [1]: trd_copy_index exports into these
        TRD_TRY(reserve(h->val[sd], (size_t)n * sizeof(uint32_t), stream));
    }
    TRD_TRY(reserve(h->tile_hist, n_tab * sizeof(uint32_t), stream));               // placement cursors
    const int n_chunks = (int)((n_tab + kSmallChunk - 1) / kSmallChunk);
    TRD_TRY(reserve(h->scan_partial, (size_t)n_chunks * sizeof(uint32_t), stream));
    TRD_TRY(reserve(h->sort_flag, 2 * sizeof(int), stream));
    if (h->small_grid == 0) {
        int per_sm = 0;
        TRD_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, small_index, kSmallThreads, 0));
        h->small_grid = per_sm * h->sm_count;
        if (h->small_grid < 1) return cudaErrorLaunchOutOfResources;
    }
    SmallIndex a;
    a.y = d_y; a.z = d_z; a.dydx = d_dydx; a.chamber = d_chamber; a.interaction = d_interaction;
    a.key = (uint32_t*)h->key[0].p;
    a.packed = (float4*)h->packed.p;
    a.store = (float4*)h->store.p;
    a.store_dx = has_dx ? (float*)h->store_dx.p : nullptr;
    a.chamber_dx = has_dx ? (const float*)h->chamber_dx.p : nullptr;
    a.tab = (uint32_t*)h->bin_first.p;
    a.cursor = (uint32_t*)h->tile_hist.p;
    a.partial = (uint32_t*)h->scan_partial.p;
    a.long_list = (uint32_t*)h->val[0].p;
    a.long_count = (uint32_t*)h->sort_flag.p + 1;
    a.gate = gate;
    a.row_ext = h->use_row_ext ? (uint2*)h->row_ext.p : nullptr;
    a.n = n;
    a.n_rows = (uint32_t)(n_cells * g.nz);
    a.g = g;
    const int64_t work = n_tab > (size_t)n ? (int64_t)n_tab : n;
    int grid = (int)((work + kSmallThreads - 1) / kSmallThreads);
    if (grid > h->small_grid) grid = h->small_grid;
    void* args[] = {&a};
    TRD_TRY(cudaLaunchCooperativeKernel((const void*)small_index, dim3((unsigned)grid), dim3(kSmallThreads), args, 0, stream));
    h->launches++;
    return cudaSuccess;
}

cudaError_t build_index(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx,
                        const int32_t* d_chamber, const int32_t* d_interaction, int n_interactions, int64_t n,
                        cudaStream_t stream) {
    const trd_config& c = h->cfg;
    IndexGeom& g = h->mp.g;
    // ---- geometry of the bins for this load ----
    g.n_ia = (d_interaction && n_interactions > 1) ? n_interactions : 1;
    const int64_t n_cells = (int64_t)g.n_ia * c.n_sectors * c.n_layers;
    const int half_rows = (int)ceil(c.z_max / c.pad_length) + 1;
    g.nz = 2 * half_rows;
    g.z_off = (float)(half_rows * c.pad_length);
    g.inv_pad = (float)(1.0 / c.pad_length);
    g.z_bias = (float)((double)half_rows);
    g.zrow_max = g.nz - 1;
    const double x_out = c.layer_x[c.n_layers - 1];
    const double y_half = x_out * tan(M_PI / c.n_sectors) * 1.02 + 1.0;
    int shift;
    if (c.ybin_width > 0.0) {
        shift = ceil_log2((uint64_t)ceil(2.0 * y_half / c.ybin_width));
    } else {
        // about two tracklets per bin on average, y bins between 8 and 1024 per row
        const double per_row = (double)n / ((double)n_cells * g.nz);
        shift = ceil_log2((uint64_t)fmax(per_row / 2.0, 1.0));
    }
    if (shift < 3 && g.n_ia == 1) shift = 3;             // with association a z row of one interaction is nearly empty
    if (shift < 0) shift = 0;
    if (shift > 10) shift = 10;
    while (shift > 0 && (uint64_t)n_cells * g.nz * (1ull << shift) >= (1ull << 28)) --shift;
    g.nb_shift = shift;
    g.ybin_max = (1 << shift) - 1;
    g.y_half = (float)y_half;
    g.inv_w = (float)((double)(1 << shift) / (2.0 * y_half));
    g.y_bias = (float)((double)(1 << shift) / 2.0);
    if ((uint64_t)n_cells * g.nz >= (1ull << 28)) return cudaErrorInvalidValue;     // too many interactions for the key
    g.n_bins = (uint32_t)n_cells * (uint32_t)g.nz * (1u << shift);
    h->ybin_width = 2.0 * y_half / (double)(1 << shift);
    h->key_bits = ceil_log2((uint64_t)g.n_bins + 1);
    h->n_passes = (h->key_bits + kRadixBits - 1) / kRadixBits;
    h->n_tracklets = n;
    h->index_loaded = false;

    // counting sort: when asked for, or for loads large enough that the radix passes cost more than its extra launches
    const bool counting = c.index_sort > 0 || (c.index_sort == 0 && n >= kCountingMin);
    h->sort_kind = counting ? 1 : 0;
    const size_t n_tab = (size_t)g.n_bins + 3;           // counts live at [key + 1] (tracklet_key, small_index)
    TRD_TRY(reserve(h->bin_first, n_tab * sizeof(int32_t), stream));
    // z extents per row only without association (with it a row holds a couple of tracklets and the table would be large)
    h->use_row_ext = g.n_ia == 1;
    if (h->use_row_ext) {
        const size_t n_rows = (size_t)n_cells * g.nz;
        TRD_TRY(reserve(h->row_ext, n_rows * sizeof(uint2), stream));
    }
    if (n == 0) {
        TRD_TRY(cudaMemsetAsync(h->bin_first.p, 0, n_tab * sizeof(int32_t), stream));
        h->sort_kind = 0;
        h->index_loaded = true;
        return cudaSuccess;
    }
    if (c.index_sort == 0 && n <= kSmallMax) {
        // small load: the whole index in one cooperative launch (small_index)
        TRD_TRY(launch_small_index(h, d_y, d_z, d_dydx, d_chamber, d_interaction, n, n_tab, n_cells, nullptr, stream));
        h->sort_kind = 3;
        h->sorted_side = 1;
        h->index_loaded = true;
        return cudaSuccess;
    }
    if (h->use_row_ext) {                                 // empty rows: min = 0xffffffff > max = 0
        const size_t n_rows = (size_t)n_cells * g.nz;
        TRD_TRY(cudaMemset2DAsync(h->row_ext.p, sizeof(uint2), 0xff, sizeof(uint32_t), n_rows, stream));
        TRD_TRY(cudaMemset2DAsync((char*)h->row_ext.p + sizeof(uint32_t), sizeof(uint2), 0x00, sizeof(uint32_t), n_rows, stream));
    }
    const int n_tiles = (int)((n + kTile - 1) / kTile);
    TRD_TRY(reserve(h->store, ((size_t)n + kStorePad) * sizeof(float4), stream));
    TRD_TRY(reserve(h->packed, (size_t)n * sizeof(float4), stream));
    const bool has_dx = h->mp.dx_max > 0.0f;
    if (has_dx) TRD_TRY(reserve(h->store_dx, ((size_t)n + kStorePad) * sizeof(float), stream));
    for (int s = 0; s < 2; ++s) {
        TRD_TRY(reserve(h->key[s], (size_t)n * sizeof(uint32_t), stream));
        TRD_TRY(reserve(h->val[s], (size_t)n * sizeof(uint32_t), stream));
    }
    TRD_TRY(reserve(h->tile_hist, (size_t)kRadix * n_tiles * sizeof(uint32_t), stream));
    TRD_TRY(reserve(h->digit_tot, 2 * kRadix * sizeof(uint32_t), stream));

    const int* gate = nullptr;
    // the counting sort first partitions by the leading digit of the key
    const int sh = h->key_bits > kRadixBits ? h->key_bits - kRadixBits : 0;
    if (counting) {
        TRD_TRY(cudaMemsetAsync(h->digit_tot.p, 0, 2 * kRadix * sizeof(uint32_t), stream));   // totals, cursors
        TRD_TRY(cudaMemsetAsync(h->bin_first.p, 0, n_tab * sizeof(uint32_t), stream));
    }
    tracklet_key<<<(unsigned)((n + 256 * kKeyItems - 1) / (256 * kKeyItems)), 256, 0, stream>>>(
        d_y, d_z, d_dydx, d_chamber, d_interaction, (uint32_t*)h->key[0].p, (float4*)h->packed.p, n, g,
        counting ? (uint32_t*)h->digit_tot.p : nullptr, sh, counting ? (uint32_t*)h->bin_first.p : nullptr,
        counting ? (uint8_t*)h->val[1].p : nullptr);
    h->launches++;
    if (counting) {
        const int n_chunks = (int)((n_tab + kScanChunk - 1) / kScanChunk);
        TRD_TRY(reserve(h->sort_flag, 2 * sizeof(int), stream));
        TRD_TRY(reserve(h->scan_partial, (size_t)n_chunks * sizeof(uint32_t), stream));
        TRD_TRY(reserve(h->part_rec, (size_t)n * sizeof(float4), stream));
        if (has_dx) TRD_TRY(reserve(h->part_dx, (size_t)n * sizeof(float), stream));
        TRD_TRY(cudaMemsetAsync(h->sort_flag.p, 0, 2 * sizeof(int), stream));      // flag, cursor of the unusable tracklets
        uint32_t* tab = (uint32_t*)h->bin_first.p;
        int* flag = (int*)h->sort_flag.p;
        Partition pl;
        pl.packed = (const float4*)h->packed.p;
        pl.rec_out = (float4*)h->part_rec.p;
        pl.chamber_dx = has_dx ? (const float*)h->chamber_dx.p : nullptr;
        pl.dx_out = has_dx ? (float*)h->part_dx.p : nullptr;
        pl.count = tab;
        pl.rank_in = (const uint8_t*)h->val[1].p;
        pl.rank_out = (uint8_t*)h->val[0].p;
        pl.n_chambers = g.n_chambers;
        TRD_TRY(cudaFuncSetAttribute(partition_tracklets, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kPartSmem));
        partition_tracklets<<<(unsigned)((n + kPartTile - 1) / kPartTile), 256, kPartSmem, stream>>>(
            (const uint32_t*)h->key[0].p, (uint32_t*)h->key[1].p, pl, (const uint32_t*)h->digit_tot.p, (uint32_t*)h->digit_tot.p + kRadix, n, sh);
        count_reduce<<<n_chunks, 256, 0, stream>>>(tab, (uint32_t*)h->scan_partial.p, (int64_t)n_tab, (int64_t)g.n_bins, flag);
        count_scan_partials<<<1, 1024, 0, stream>>>((uint32_t*)h->scan_partial.p, n_chunks);
        count_apply<<<n_chunks, 256, 0, stream>>>(tab, (const uint32_t*)h->scan_partial.p, (int64_t)n_tab);
        place_tracklets<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>((const uint32_t*)h->key[1].p, (const uint8_t*)h->val[0].p,
                                                                         (const float4*)h->part_rec.p, has_dx ? (const float*)h->part_dx.p : nullptr,
                                                                         tab, (uint32_t*)h->sort_flag.p + 1, (float4*)h->store.p,
                                                                         has_dx ? (float*)h->store_dx.p : nullptr, n, g.n_bins, flag);
        order_bins<<<(unsigned)(((int64_t)g.n_bins + 255) / 256), 256, 0, stream>>>(tab, (float4*)h->store.p, has_dx ? (float*)h->store_dx.p : nullptr,
                                                                                    h->use_row_ext ? (uint2*)h->row_ext.p : nullptr,
                                                                                    (int64_t)g.n_bins, g.nb_shift, flag);
        h->launches += 6;
        TRD_TRY(cudaGetLastError());
        gate = flag;                                     // the radix kernels below run only if a bin was too long
    }
    if (gate) {
        // a bin longer than kMaxBin made the counting kernels return: the one-launch sort, which orders long bins itself,
        // does the load again (gated on the same device flag: one idle launch otherwise)
        TRD_TRY(launch_small_index(h, d_y, d_z, d_dydx, d_chamber, d_interaction, n, n_tab, n_cells, gate, stream));
        h->sorted_side = 1;
        h->index_loaded = true;
        return cudaSuccess;
    }
    int side = 0;
    TRD_TRY(radix_sort_pairs((uint32_t*)h->key[0].p, (uint32_t*)h->key[1].p, (uint32_t*)h->val[0].p, (uint32_t*)h->val[1].p,
                             (uint32_t*)h->tile_hist.p, (uint32_t*)h->digit_tot.p, n, h->n_passes, stream, &side, &h->launches, nullptr));
    h->sorted_side = side;
    gather_store<<<(unsigned)((n + 256 * kGather - 1) / (256 * kGather)), 256, 0, stream>>>((const uint32_t*)h->val[side].p, (const uint32_t*)h->key[side].p,
                                           (const float4*)h->packed.p, (float4*)h->store.p, h->use_row_ext ? (uint2*)h->row_ext.p : nullptr,
                                           (int32_t*)h->bin_first.p, has_dx ? (const float*)h->chamber_dx.p : nullptr,
                                           has_dx ? (float*)h->store_dx.p : nullptr, g.n_chambers, n, g.n_bins, g.nb_shift, nullptr);
    h->launches += 1;
    TRD_TRY(cudaGetLastError());
    h->index_loaded = true;
    return cudaSuccess;
}

}  // namespace trd
