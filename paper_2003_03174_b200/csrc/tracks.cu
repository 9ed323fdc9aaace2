// tracks.cu -- track binning around the match kernel ("track pre-binning").
//
// Tracks arrive in arbitrary order, so neighbouring sub-warps of the match kernel would touch
// unrelated bins of the tracklet index and re-read it from HBM many times.  For large batches
// trd_match therefore (1) packs every track into one 96-byte record and computes a locality key
// (sector, z row, coarse y of the straight-line prediction at the middle TRD layer), (2) orders the
// tracks by key -- a counting sort (histogram by atomics in the pack kernel, one-block scan, placement
// by atomics; the order inside a key is arbitrary and irrelevant) when the key has at most 16 bits,
// else the radix sort of index.cu --, (3) runs the match kernel over the permutation, gathering whole
// records and scattering whole 128-byte result records, (4) unpacks the results to the caller's
// SoA arrays.  The key only decides the processing order; no result depends on it.
#include "trd_internal.cuh"

namespace trd {

namespace {

constexpr int kThreads = 128;
constexpr int kYBits = 4;                      // 16 coarse y bins per (sector, z row)

// SoA -> records through shared memory so that both sides are coalesced
__global__ void __launch_bounds__(kThreads) pack_kernel(const trd_tracks_in in, int64_t n, float* __restrict__ rec,
                                                        uint32_t* __restrict__ key, IndexGeom g, float x_mid, float edge_mid,
                                                        int nz, uint32_t* __restrict__ hist) {
    __shared__ float sm[kThreads][kRecIn + 1];
    const int64_t base = (int64_t)blockIdx.x * kThreads;
    const int64_t i = base + threadIdx.x;
    if (i < n) {
        float* r = sm[threadIdx.x];
#pragma unroll
        for (int k = 0; k < 5; ++k) r[k] = in.par[k][i];
#pragma unroll
        for (int k = 0; k < 15; ++k) r[5 + k] = in.cov[k][i];
        const float x = in.x[i];
        const int sector = in.sector[i];
        r[20] = x;
        r[21] = __int_as_float(sector);
        const int ia = (g.n_ia > 1) ? in.interaction[i] : 0;
        r[22] = __int_as_float(ia);
        r[23] = 0.0f;
        // locality key from the straight-line prediction at x_mid
        const float s = fminf(fmaxf(r[2], -0.99f), 0.99f);
        const float inv_c = rsqrtf((1.0f - s) * (1.0f + s));
        const float dx = x_mid - x;
        float yp = fmaf(dx, s * inv_c, r[0]);
        const float zp = fmaf(dx, r[3] * inv_c, r[1]);
        int sec = sector;
        if (yp > edge_mid) { sec += 1; yp -= 2.0f * edge_mid; }
        if (yp < -edge_mid) { sec -= 1; yp += 2.0f * edge_mid; }
        sec = ((sec % g.n_sectors) + g.n_sectors) % g.n_sectors;
        float fy = floorf((yp + edge_mid) / (2.0f * edge_mid) * (float)(1 << kYBits));
        fy = fminf(fmaxf(fy, 0.0f), (float)((1 << kYBits) - 1));
        const int zr = isfinite(zp) ? zrow_of(g, zp) : 0;
        uint32_t kk;
        if (g.n_ia > 1) {      // with association the interaction leads, as in the tracklet index
            const int a = min(max(ia, 0), g.n_ia - 1);
            kk = ((uint32_t)a * (uint32_t)g.n_sectors + (uint32_t)sec) * (uint32_t)nz + (uint32_t)zr;
        } else {
            kk = (((uint32_t)sec * (uint32_t)nz + (uint32_t)zr) << kYBits) + (uint32_t)(isfinite(fy) ? (int)fy : 0);
        }
        key[i] = kk;
        if (hist) atomicAdd(hist + kk, 1u);
    }
    __syncthreads();
    const int64_t n_here = min((int64_t)kThreads, n - base);
    const int64_t n_f4 = n_here * (kRecIn / 4);
    float4* dst = reinterpret_cast<float4*>(rec + base * kRecIn);
    for (int64_t j = threadIdx.x; j < n_f4; j += kThreads) {
        const int f = (int)j * 4, t = f / kRecIn, w = f % kRecIn;
        dst[j] = make_float4(sm[t][w], sm[t][w + 1], sm[t][w + 2], sm[t][w + 3]);
    }
}

// result records (caller's order) -> SoA
__global__ void __launch_bounds__(kThreads) unpack_kernel(const float* __restrict__ rec, const trd_tracks_out out, int64_t n,
                                                          int n_layers) {
    __shared__ float sm[kThreads][kRecOut + 1];
    const int64_t base = (int64_t)blockIdx.x * kThreads;
    const int64_t n_here = min((int64_t)kThreads, n - base);
    const int64_t n_f4 = n_here * (kRecOut / 4);
    const float4* src = reinterpret_cast<const float4*>(rec + base * kRecOut);
    for (int64_t j = threadIdx.x; j < n_f4; j += kThreads) {
        const float4 v = src[j];
        const int f = (int)j * 4, t = f / kRecOut, w = f % kRecOut;
        sm[t][w] = v.x; sm[t][w + 1] = v.y; sm[t][w + 2] = v.z; sm[t][w + 3] = v.w;
    }
    __syncthreads();
    const int64_t i = base + threadIdx.x;
    if (i >= n) return;
    const float* r = sm[threadIdx.x];
#pragma unroll
    for (int l = 0; l < TRD_MAX_LAYERS; ++l) out.tracklet_idx[l][i] = (l < n_layers) ? __float_as_int(r[l]) : -1;
#pragma unroll
    for (int k = 0; k < 5; ++k) out.par[k][i] = r[6 + k];
#pragma unroll
    for (int k = 0; k < 15; ++k) out.cov[k][i] = r[11 + k];
    out.x[i] = r[26];
    out.sector[i] = __float_as_int(r[27]);
    out.chi2[i] = r[28];
    out.n_matched[i] = __float_as_int(r[29]);
    if (out.n_cand_evals) out.n_cand_evals[i] = __float_as_int(r[30]);
}

// counting sort, step 2: exclusive scan of the key histogram in place.  One block per tile of 4096 keys (1 to 16 blocks);
// a block publishes its tile's sum in status[tile] (bit 31 = published; pack_tracks cleared the words together with the
// histogram) and adds up the sums of the tiles before it, spinning until they are there: those blocks have lower
// indices and were scheduled first, so they are running.  (One block for the whole table took 15.5 us per call.)
constexpr int kScanThreads = 256;
constexpr int kScanPer = 16;                                       // keys per thread
constexpr int kScanTile = kScanThreads * kScanPer;                 // 4096 = the smallest table (track_key_bits >= 12)
constexpr int kScanMaxTiles = (1 << kCountingBits) / kScanTile;    // 16 status words
constexpr uint32_t kPublished = 0x80000000u;
constexpr int kStatusWords = 64;                                   // 256 bytes in front of the histogram (kTrackHistBytes)
__global__ void __launch_bounds__(kScanThreads) scan_hist(uint32_t* __restrict__ hist, uint32_t* __restrict__ status) {
    __shared__ uint32_t warp_sums[kScanThreads / 32];
    __shared__ uint32_t s_before;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint4* mine = reinterpret_cast<uint4*>(hist) + ((size_t)blockIdx.x * kScanThreads + threadIdx.x) * (kScanPer / 4);
    uint4 c[kScanPer / 4];
#pragma unroll
    for (int k = 0; k < kScanPer / 4; ++k) c[k] = mine[k];
    uint32_t sum = 0;
#pragma unroll
    for (int k = 0; k < kScanPer / 4; ++k) sum += c[k].x + c[k].y + c[k].z + c[k].w;
    uint32_t incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) warp_sums[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        const uint32_t w = lane < kScanThreads / 32 ? warp_sums[lane] : 0u;
        uint32_t wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        if (lane < kScanThreads / 32) warp_sums[lane] = wi - w;
        const uint32_t total = __shfl_sync(0xffffffffu, wi, 31);
        volatile uint32_t* st = status;
        if (lane == 0) st[blockIdx.x] = kPublished | total;        // at most 2^31 - 1 tracks per call
        uint32_t before = 0;                                       // tiles before this one: at most 15, one lane each
        if (lane < (int)blockIdx.x) {
            uint32_t v;
            do { v = st[lane]; } while (!(v & kPublished));
            before = v & ~kPublished;
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xffffffffu, before, o);
        if (lane == 0) s_before = before;
    }
    __syncthreads();
    uint32_t run = s_before + warp_sums[warp] + incl - sum;
#pragma unroll
    for (int k = 0; k < kScanPer / 4; ++k) {
        uint4 o;
        o.x = run; run += c[k].x;
        o.y = run; run += c[k].y;
        o.z = run; run += c[k].z;
        o.w = run; run += c[k].w;
        mine[k] = o;
    }
}
static_assert(kScanMaxTiles <= 32 && kScanMaxTiles <= kStatusWords, "one lane per earlier tile");

// counting sort, step 3: every track takes the next free place of its key
__global__ void __launch_bounds__(256) place_tracks(const uint32_t* __restrict__ key, uint32_t* __restrict__ next,
                                                    uint32_t* __restrict__ perm, int64_t n) {
    const int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (i < n) perm[atomicAdd(next + key[i], 1u)] = (uint32_t)i;
}

}  // namespace

cudaError_t pack_tracks(trd_handle* h, const trd_tracks_in& in, int64_t n, float* rec, uint32_t* key, int* key_bits,
                        uint32_t* hist, cudaStream_t stream) {
    const trd_config& c = h->cfg;
    const IndexGeom& g = h->mp.g;
    const int mid = c.n_layers / 2;
    const float x_mid = (float)c.layer_x[mid];
    const float edge_mid = (float)(c.layer_x[mid] * tan(M_PI / c.n_sectors));
    const unsigned grid = (unsigned)((n + kThreads - 1) / kThreads);
    const int bits = track_key_bits(h);
    if (bits > kCountingBits) hist = nullptr;
    if (hist) {
        // the status words of scan_hist and, behind them, the histogram
        cudaError_t e = cudaMemsetAsync(hist, 0, kStatusWords * sizeof(uint32_t) + (sizeof(uint32_t) << bits), stream);
        if (e != cudaSuccess) return e;
    }
    pack_kernel<<<grid, kThreads, 0, stream>>>(in, n, rec, key, g, x_mid, edge_mid, g.nz, hist ? hist + kStatusWords : nullptr);
    h->launches++;
    *key_bits = bits;
    return cudaGetLastError();
}

int track_key_bits(const trd_handle* h) {
    const trd_config& c = h->cfg;
    const IndexGeom& g = h->mp.g;
    const uint64_t n_keys = g.n_ia > 1 ? (uint64_t)g.n_ia * c.n_sectors * g.nz : ((uint64_t)c.n_sectors * g.nz) << kYBits;
    int bits = 0;
    while ((1ull << bits) < n_keys) ++bits;
    return bits < 12 ? 12 : bits;        // the one-block scan of the counting sort wants at least 4 keys per thread
}

// counting sort of the tracks by the key histogram pack_tracks filled: perm[place] = track
cudaError_t place_tracks_by_key(trd_handle* h, const uint32_t* key, uint32_t* hist, uint32_t* perm, int key_bits, int64_t n,
                                cudaStream_t stream) {
    scan_hist<<<(1 << key_bits) / kScanTile, kScanThreads, 0, stream>>>(hist + kStatusWords, hist);
    place_tracks<<<(unsigned)((n + 255) / 256), 256, 0, stream>>>(key, hist + kStatusWords, perm, n);
    h->launches += 2;
    return cudaGetLastError();
}

cudaError_t unpack_tracks(trd_handle* h, const float* rec_out, const trd_tracks_out& out, int64_t n, cudaStream_t stream) {
    const unsigned grid = (unsigned)((n + kThreads - 1) / kThreads);
    unpack_kernel<<<grid, kThreads, 0, stream>>>(rec_out, out, n, h->cfg.n_layers);
    h->launches++;
    return cudaGetLastError();
}

}  // namespace trd
