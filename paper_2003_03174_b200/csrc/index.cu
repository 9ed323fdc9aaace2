// index.cu -- the tracklet index of trd_load_tracklets.
//
//   a1  tracklet_key     key = ((sector, layer), z row, y bin) from (chamber, z, y)
//   a2  radix_*          stable LSD radix sort of (key, position), 8 bits per pass:
//                        per-tile digit histogram -> per-digit scan over tiles -> stable scatter
//       gather_store     sorted store: one float4 (y, z, dy/dx, position) per tracklet
//   a3  (in gather_store) first sorted position of every bin (plus sentinel), z extent of every row
//
// north_star: "device-side sort and index by chamber and local-y bin ... a radix sort plus
// per-chamber y-bin offsets"; the 18 x 5 x 6 segmentation is PAPER.md:50.  The key also
// carries the z row (SURVEY.md 8(d).3 "design consequence"), and it uses (sector, layer)
// rather than the chamber's stack, because the z window may straddle two stacks (reading R12).
// All of it is HBM-streaming integer work; no tensor cores.
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
__global__ void __launch_bounds__(256) tracklet_key(const float* __restrict__ y, const float* __restrict__ z,
                                                    const float* __restrict__ dydx, const int32_t* __restrict__ chamber,
                                                    const int32_t* __restrict__ interaction, uint32_t* __restrict__ key,
                                                    float4* __restrict__ packed, int64_t n, IndexGeom g) {
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const float yy = y[i], zz = z[i];
    packed[i] = make_float4(yy, zz, dydx[i], __int_as_float(chamber[i]));
    const int ch = chamber[i];
    uint32_t k = g.n_bins;                          // unusable: behind every bin
    const int ia = (g.n_ia > 1) ? interaction[i] : 0;      // time-frame association: the interaction leads the key
    if (ch >= 0 && ch < g.n_chambers && isfinite(yy) && isfinite(zz) && ia >= 0 && ia < g.n_ia) {
        const int sector = ch / g.per_sector, layer = ch % g.n_layers;
        const uint32_t cell = (uint32_t)((ia * g.n_sectors + sector) * g.n_layers + layer);
        k = ((cell * (uint32_t)g.nz + (uint32_t)zrow_of(g, zz)) << g.nb_shift) + (uint32_t)ybin_of(g, yy);
    }
    key[i] = k;
}

// per-tile histogram of one digit; hist[d * n_tiles + tile]
__global__ void __launch_bounds__(kSortThreads) radix_hist(const uint32_t* __restrict__ key, uint32_t* __restrict__ hist,
                                                           int64_t n, int n_tiles, int shift) {
    __shared__ uint32_t cnt[kRadix];
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
                                                              int n_tiles) {
    __shared__ uint32_t warp_sums[32];
    __shared__ uint32_t total;
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
                                                              int shift) {
    __shared__ uint32_t warp_cnt[kSortWarps][kRadix];
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

__device__ __forceinline__ uint32_t ext_encode(float f) {          // order-preserving float -> uint
    const uint32_t b = __float_as_uint(f);
    return (b & 0x80000000u) ? ~b : (b ^ 0x80000000u);
}

// also records the z extent of every (cell, z row): row_ext[row] = (min, max) of the encoded z.  The keys are
// sorted, so a warp almost always lies inside one row: one warp reduction and two atomics per warp.  Each
// thread handles kGather tracklets (independent random 16-byte reads in flight), strided by the block size.
constexpr int kGather = 4;

__global__ void __launch_bounds__(256) gather_store(const uint32_t* __restrict__ pos, const uint32_t* __restrict__ key,
                                                    const float4* __restrict__ packed, float4* __restrict__ store,
                                                    uint2* __restrict__ row_ext, int32_t* __restrict__ bin_first,
                                                    const float* __restrict__ chamber_dx, float* __restrict__ store_dx,
                                                    int n_chambers, int64_t n, uint32_t n_bins, int nb_shift) {
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
                             int64_t* launches) {
    const int n_tiles = radix_tiles(n);
    uint32_t* key[2] = {key0, key1};
    uint32_t* val[2] = {val0, val1};
    int side = 0;
    for (int p = 0; p < n_passes; ++p) {
        const int sh = p * kRadixBits;
        const uint32_t* kin = key[side];
        const uint32_t* vin = (p == 0) ? nullptr : val[side];
        radix_hist<<<n_tiles, kSortThreads, 0, stream>>>(kin, tile_hist, n, n_tiles, sh);
        radix_rowscan<<<kRadix, kSortThreads, 0, stream>>>(tile_hist, digit_tot, n_tiles);
        radix_scatter<<<n_tiles, kSortThreads, 0, stream>>>(kin, vin, key[side ^ 1], val[side ^ 1], tile_hist, digit_tot, n,
                                                           n_tiles, sh);
        *launches += 3;
        side ^= 1;
    }
    *side_out = side;
    return cudaGetLastError();
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
    g.y_half = (float)y_half;
    g.inv_w = (float)((double)(1 << shift) / (2.0 * y_half));
    if ((uint64_t)n_cells * g.nz >= (1ull << 28)) return cudaErrorInvalidValue;     // too many interactions for the key
    g.n_bins = (uint32_t)n_cells * (uint32_t)g.nz * (1u << shift);
    h->ybin_width = 2.0 * y_half / (double)(1 << shift);
    h->key_bits = ceil_log2((uint64_t)g.n_bins + 1);
    h->n_passes = (h->key_bits + kRadixBits - 1) / kRadixBits;
    h->n_tracklets = n;
    h->index_loaded = false;

    TRD_TRY(reserve(h->bin_first, ((size_t)g.n_bins + 1) * sizeof(int32_t), stream));
    // z extents per row only without association (with it a row holds a couple of tracklets and the table would be large)
    h->use_row_ext = g.n_ia == 1;
    if (h->use_row_ext) {
        const size_t n_rows = (size_t)n_cells * g.nz;
        TRD_TRY(reserve(h->row_ext, n_rows * sizeof(uint2), stream));
        // empty rows: min = 0xffffffff > max = 0
        TRD_TRY(cudaMemset2DAsync(h->row_ext.p, sizeof(uint2), 0xff, sizeof(uint32_t), n_rows, stream));
        TRD_TRY(cudaMemset2DAsync((char*)h->row_ext.p + sizeof(uint32_t), sizeof(uint2), 0x00, sizeof(uint32_t), n_rows, stream));
    }
    if (n == 0) {
        TRD_TRY(cudaMemsetAsync(h->bin_first.p, 0, ((size_t)g.n_bins + 1) * sizeof(int32_t), stream));
        h->index_loaded = true;
        return cudaSuccess;
    }
    const int n_tiles = (int)((n + kTile - 1) / kTile);
    TRD_TRY(reserve(h->store, (size_t)n * sizeof(float4), stream));
    TRD_TRY(reserve(h->packed, (size_t)n * sizeof(float4), stream));
    const bool has_dx = h->mp.dx_max > 0.0f;
    if (has_dx) TRD_TRY(reserve(h->store_dx, (size_t)n * sizeof(float), stream));
    for (int s = 0; s < 2; ++s) {
        TRD_TRY(reserve(h->key[s], (size_t)n * sizeof(uint32_t), stream));
        TRD_TRY(reserve(h->val[s], (size_t)n * sizeof(uint32_t), stream));
    }
    TRD_TRY(reserve(h->tile_hist, (size_t)kRadix * n_tiles * sizeof(uint32_t), stream));
    TRD_TRY(reserve(h->digit_tot, kRadix * sizeof(uint32_t), stream));

    const unsigned n_blk = (unsigned)((n + 255) / 256);
    tracklet_key<<<n_blk, 256, 0, stream>>>(d_y, d_z, d_dydx, d_chamber, d_interaction, (uint32_t*)h->key[0].p,
                                            (float4*)h->packed.p, n, g);
    h->launches++;
    int side = 0;
    TRD_TRY(radix_sort_pairs((uint32_t*)h->key[0].p, (uint32_t*)h->key[1].p, (uint32_t*)h->val[0].p, (uint32_t*)h->val[1].p,
                             (uint32_t*)h->tile_hist.p, (uint32_t*)h->digit_tot.p, n, h->n_passes, stream, &side, &h->launches));
    h->sorted_side = side;
    gather_store<<<(unsigned)((n + 256 * kGather - 1) / (256 * kGather)), 256, 0, stream>>>((const uint32_t*)h->val[side].p, (const uint32_t*)h->key[side].p,
                                           (const float4*)h->packed.p, (float4*)h->store.p, h->use_row_ext ? (uint2*)h->row_ext.p : nullptr,
                                           (int32_t*)h->bin_first.p, has_dx ? (const float*)h->chamber_dx.p : nullptr,
                                           has_dx ? (float*)h->store_dx.p : nullptr, g.n_chambers, n, g.n_bins, g.nb_shift);
    h->launches += 1;
    TRD_TRY(cudaGetLastError());
    h->index_loaded = true;
    return cudaSuccess;
}

}  // namespace trd
