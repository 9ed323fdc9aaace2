// trd_internal.cuh -- shared declarations of the CUDA path (not part of the C ABI).
// Nothing here is used by, or uses, anything under oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include <string>

#include "trdmatch.h"

namespace trd {

// ---- geometry of the tracklet index ----------------
// bin key = (((sector * n_layers + layer) * nz + zrow) << nb_shift) + ybin
struct IndexGeom {
    int n_sectors, n_layers, per_sector, n_chambers;
    int n_ia;          // interactions of the loaded time frame (1 = no association)
    int nz;            // z rows per (sector, layer)
    int nb_shift;      // log2(y bins per z row)
    float z_off, inv_pad;
    float y_half, inv_w;
    float z_bias, y_bias;       // z_off * inv_pad, y_half * inv_w: row = floor(z * inv_pad + z_bias), bin likewise
    int zrow_max, ybin_max;     // nz - 1, y bins per row - 1: the clamps of the two bin functions
    uint32_t n_bins;   // also the key of an unusable tracklet (sorts behind every bin)
};

// Both bin functions are monotone in their argument and clamp, so a window query [lo, hi] covers every tracklet whose
// coordinate lies in it; the index build and the match kernel share them.  One FFMA, one F2I.FLOOR, two integer clamps.
__device__ __forceinline__ int zrow_of(const IndexGeom& g, float z) {
    return min(max(__float2int_rd(fmaf(z, g.inv_pad, g.z_bias)), 0), g.zrow_max);
}

__device__ __forceinline__ int ybin_of(const IndexGeom& g, float y) {
    return min(max(__float2int_rd(fmaf(y, g.inv_w, g.y_bias)), 0), g.ybin_max);
}

// order-preserving float -> uint (the z extent of a row is kept by atomicMin / atomicMax on these, index.cu; the match
// kernel compares the encoded bounds of its z window with them)
__host__ __device__ inline uint32_t ext_encode(float f) {
#ifdef __CUDA_ARCH__
    const uint32_t b = __float_as_uint(f);
#else
    uint32_t b;
    memcpy(&b, &f, sizeof b);
#endif
    return (b & 0x80000000u) ? ~b : (b ^ 0x80000000u);
}

// ---- constants of the match kernel, float32, derived in double on the host -------------------
struct MatchParams {
    IndexGeom g;
    int n_hyp;
    float layer_x[TRD_MAX_LAYERS];
    float edge[TRD_MAX_LAYERS];      // layer_x * tan(pi / n_sectors): the sector edge in y
    float b;                         // kappa = b * q/pT
    float cb_hi, sb_hi;              // cos / sin of the sector width, float32 (Jacobian of the frame change)
    double cbd, sbd;                 // the same in double (the point and sin(phi) in the new frame)
    double bd;                       // b in double: sin(phi) advances by bd * q/pT * dx
    float sig_y2, sig_z2;
    float n_sigma_road, half_pad;
    float veto;                      // n_sigma_angle * sigma_dydx
    float chi2_cut, chi2_penalty, max_snp;
    // measurement model (res_model = 1: PAPER.md:62, 66)
    int res_model;
    float n_sigma_angle, sy_c0, sy_c2, sd_c0, sd_c2, sin_lorentz, tan_tilt;
    // two-stage propagation: largest |radial chamber offset|, 0 = all chambers on their nominal plane
    float dx_max;
    // trd_refit
    float tan_half;                  // tan(pi / n_sectors): sector edge in y = x * tan_half
    float x_ref, refit_var[5];
    // material in front of every layer (R32-R34)
    int material;                    // 0: none
    float ms_k;                      // 0.0136^2 * x/X0
    float eloss, eloss_fluct, mass, mass2;
    // field inhomogeneity Bz (1 + bz_r2 r^2 + bz_z2 z^2) (R35)
    int field;                       // 0: uniform
    float bz_r2, bz_z2;
};

struct Buffer {
    void* p = nullptr;
    size_t bytes = 0;
};

}  // namespace trd

struct trd_handle {
    trd_config cfg;
    trd::MatchParams mp;
    int device = 0;
    int sm_count = 0;
    bool index_loaded = false;
    bool use_row_ext = true;
    int64_t n_tracklets = 0;
    int key_bits = 0, n_passes = 0;
    double ybin_width = 0.0;
    int64_t launches = 0;
    static constexpr int kEvRing = 64;               // event pairs around the match kernels of the last 64 trd_match calls
    cudaEvent_t ev_match[kEvRing][2] = {};
    int64_t ev_count = 0;                            // trd_match calls that recorded events so far
    std::string err;
    // device buffers owned by the handle
    trd::Buffer store;      // float4 per sorted tracklet: y, z, dy/dx, original position (bits)
    trd::Buffer packed;     // float4 per tracklet in the caller's order (gather source)
    trd::Buffer key[2];     // uint32 keys, ping-pong
    trd::Buffer val[2];     // uint32 original positions, ping-pong; counting sort: one rank byte per tracklet, [1] in the
                            // caller's order, [0] partitioned
    trd::Buffer tile_hist;  // [256][n_tiles] digit counts per tile
    trd::Buffer digit_tot;  // [256]
    trd::Buffer bin_first;  // [n_bins + 1]
    trd::Buffer row_ext;    // uint2 per (cell, z row): encoded min and max z of the row
    trd::Buffer chamber_dx; // float per chamber: radial offset from the nominal layer plane (trd_set_chamber_dx)
    trd::Buffer store_dx;   // float per sorted tracklet: the offset of its chamber (only when offsets are set)
    int sorted_side = 0;    // which of key[]/val[] holds the sorted result
    int sort_kind = 0;      // last load: 0 = radix sort, 1 = counting sort, 2 = counting sort gave up (long bin), radix did it,
                            // 3 = counting sort in one cooperative launch (small loads)
    int small_grid = 0;     // blocks of the cooperative launch (occupancy x SMs), found on first use
    trd::Buffer sort_flag;  // int: set by the counting sort when a bin is too long for it
    trd::Buffer scan_partial;  // chunk sums of the count table
    trd::Buffer part_rec;   // counting sort: float4 per tracklet, partitioned by the leading key digit
    trd::Buffer part_dx;    // counting sort: chamber offset per partitioned tracklet (only when offsets are set)
    // staging for the *_host entry points
    trd::Buffer stage_tl;   // tracklets
    // pipelined host entry points (host_api.cu): own copy streams, a ring of staging slots
    static constexpr int kRing = 4;
    cudaStream_t s_in = nullptr, s_out = nullptr;        // host->device and device->host copy streams
    trd::Buffer stage_in[kRing], stage_out[kRing];       // tracks in / out per ring slot
    cudaEvent_t ev_in[kRing] = {}, ev_done[kRing] = {}, ev_out[kRing] = {};   // copied in / matched / copied out
    bool slot_busy[kRing] = {};
    cudaEvent_t ev_tl_in = nullptr, ev_tl_used = nullptr;  // tracklets copied in / consumed by the index build
    bool tl_pending = false;
    int ring_next = 0;
    // track binning (trd_match on large batches): packed records and the permutation
    trd::Buffer trk_rec;    // kRecIn floats per track, caller's order
    trd::Buffer trk_out;    // kRecOut floats per track, caller's order
    trd::Buffer trk_key[2]; // uint32 bin keys, ping-pong
    trd::Buffer trk_val[2]; // uint32 track positions, ping-pong
    trd::Buffer trk_hist;   // [256][n_tiles]
    trd::Buffer trk_tot;    // [256]
};

namespace trd {

// returns cudaSuccess or the first error; counts launches into h->launches
cudaError_t build_index(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx,
                        const int32_t* d_chamber, const int32_t* d_interaction, int n_interactions, int64_t n,
                        cudaStream_t stream);
cudaError_t launch_match(trd_handle* h, const trd_tracks_in& in, const trd_tracks_out& out, int64_t n,
                         cudaStream_t stream);
cudaError_t launch_refit(trd_handle* h, const trd_tracks_out& matched, const trd_refit_out& out, int64_t n,
                         cudaStream_t stream);
// trd_match_static (match.cu): the binned path with its scratch in a file-scope device array, no allocation of any kind
cudaError_t launch_match_static(trd_handle* h, const trd_tracks_in& in, const trd_tracks_out& out, int64_t n,
                                cudaStream_t stream);

// packed track records used when a batch is binned before matching (tracks.cu, match.cu)
// the match kernel reads the sorted store four tracklets at a time without looking at the end of the run (what lies behind
// it is masked out afterwards): the store and its companion arrays are allocated this many entries longer
constexpr int kStorePad = 4;

constexpr int kRecIn = 24;    // y z s t c | 15 cov | x | sector bits | 2 pad          (96 bytes)
constexpr int kRecOut = 32;   // 6 idx | 5 par | 15 cov | x sector chi2 n_matched n_evals | pad   (128 bytes)

int radix_tiles(int64_t n);
cudaError_t radix_sort_pairs(uint32_t* key0, uint32_t* key1, uint32_t* val0, uint32_t* val1, uint32_t* tile_hist,
                             uint32_t* digit_tot, int64_t n, int n_passes, cudaStream_t stream, int* side_out,
                             int64_t* launches, const int* gate = nullptr);
// after a counting sort: fills val[sorted_side] / key[sorted_side] for trd_copy_index (synchronises)
cudaError_t export_sorted_index(trd_handle* h, cudaStream_t stream);
// tracks.cu: SoA -> packed records + locality key; packed results -> SoA
constexpr int kCountingBits = 16;     // track keys up to this many bits are counting-sorted (tracks.cu)
// 256 bytes of status words of the scan (tracks.cu scan_hist) + the key histogram of that sort
constexpr size_t kTrackHistBytes = (sizeof(uint32_t) << kCountingBits) + 256;
int track_key_bits(const trd_handle* h);
cudaError_t pack_tracks(trd_handle* h, const trd_tracks_in& in, int64_t n, float* rec, uint32_t* key, int* key_bits,
                        uint32_t* hist, cudaStream_t stream);
cudaError_t place_tracks_by_key(trd_handle* h, const uint32_t* key, uint32_t* hist, uint32_t* perm, int key_bits, int64_t n,
                                cudaStream_t stream);
cudaError_t unpack_tracks(trd_handle* h, const float* rec_out, const trd_tracks_out& out, int64_t n, cudaStream_t stream);

// Every entry point works on the device the handle was created on, whatever device is current in the calling thread:
// the guard switches to it and restores the caller's device on the way out.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const trd_handle* h) {
        if (h && cudaGetDevice(&prev) == cudaSuccess && prev != h->device) switched = cudaSetDevice(h->device) == cudaSuccess;
    }
    ~DeviceGuard() {
        if (switched) cudaSetDevice(prev);
    }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};

int fail(trd_handle* h, int code, const std::string& what);
int fail_cuda(trd_handle* h, cudaError_t e, const char* where);
void host_pipeline_destroy(trd_handle* h);

// grows b to at least `bytes` (contents lost); synchronises `stream` before freeing
cudaError_t reserve(Buffer& b, size_t bytes, cudaStream_t stream);

}  // namespace trd
