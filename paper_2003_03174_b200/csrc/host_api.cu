// host_api.cu -- the *_host entry points of include/trdmatch.h: staging and copy/compute overlap.
// Three streams: s_in (host->device copies), the caller's stream (all kernels), s_out (device->host
// copies), chained by events.  Tracks use a ring of four staging slots so that the copy-in of batch k+1 and
// the copy-out of batch k-1 run while batch k is matched.  No arithmetic of the method lives here.
#include "trd_internal.cuh"

namespace trd {

namespace {

constexpr int kInArrays = 5 + 15 + 1 + 1;                    // par, cov, x, sector
constexpr int kOutArrays = TRD_MAX_LAYERS + 5 + 15 + 5;      // idx, par, cov, x, sector, chi2, n_matched, n_cand_evals

#define TRD_TRY(expr)                              \
    do {                                           \
        cudaError_t e_ = (expr);                   \
        if (e_ != cudaSuccess) return e_;          \
    } while (0)

cudaError_t ensure_pipeline(trd_handle* h) {
    if (h->s_in) return cudaSuccess;
    TRD_TRY(cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking));
    TRD_TRY(cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking));
    for (int k = 0; k < trd_handle::kRing; ++k) {
        TRD_TRY(cudaEventCreateWithFlags(&h->ev_in[k], cudaEventDisableTiming));
        TRD_TRY(cudaEventCreateWithFlags(&h->ev_done[k], cudaEventDisableTiming));
        TRD_TRY(cudaEventCreateWithFlags(&h->ev_out[k], cudaEventDisableTiming));
    }
    TRD_TRY(cudaEventCreateWithFlags(&h->ev_tl_in, cudaEventDisableTiming));
    TRD_TRY(cudaEventCreateWithFlags(&h->ev_tl_used, cudaEventDisableTiming));
    return cudaSuccess;
}

// wait (on the host) until ring slot k is free again
cudaError_t retire_slot(trd_handle* h, int k) {
    if (!h->slot_busy[k]) return cudaSuccess;
    TRD_TRY(cudaEventSynchronize(h->ev_out[k]));
    h->slot_busy[k] = false;
    return cudaSuccess;
}

// a staging buffer may only be re-allocated when nothing queued on any of the three streams uses it
cudaError_t reserve_idle(trd_handle* h, Buffer& b, size_t bytes, cudaStream_t stream) {
    if (bytes <= b.bytes) return cudaSuccess;
    TRD_TRY(cudaStreamSynchronize(h->s_in));
    TRD_TRY(cudaStreamSynchronize(h->s_out));
    return reserve(b, bytes, stream);
}

cudaError_t load_host(trd_handle* h, const float* y, const float* z, const float* dydx, const int32_t* chamber, int64_t n,
                      cudaStream_t st) {
    TRD_TRY(ensure_pipeline(h));
    const size_t bytes = (size_t)n * 4;
    TRD_TRY(reserve_idle(h, h->stage_tl, 4 * bytes + 16, st));
    // the previous load's kernels must have consumed the staging buffer before it is overwritten
    if (h->tl_pending) TRD_TRY(cudaStreamWaitEvent(h->s_in, h->ev_tl_used, 0));
    char* base = (char*)h->stage_tl.p;
    const void* src[4] = {y, z, dydx, chamber};
    for (int k = 0; k < 4 && n > 0;) {
        int m = 1;
        while (k + m < 4 && (const char*)src[k + m] == (const char*)src[k] + (size_t)m * bytes) ++m;
        TRD_TRY(cudaMemcpyAsync(base + k * bytes, src[k], (size_t)m * bytes, cudaMemcpyHostToDevice, h->s_in));
        k += m;
    }
    TRD_TRY(cudaEventRecord(h->ev_tl_in, h->s_in));
    TRD_TRY(cudaStreamWaitEvent(st, h->ev_tl_in, 0));
    TRD_TRY(build_index(h, (const float*)base, (const float*)(base + bytes), (const float*)(base + 2 * bytes),
                        (const int32_t*)(base + 3 * bytes), nullptr, 1, n, st));
    TRD_TRY(cudaEventRecord(h->ev_tl_used, st));
    h->tl_pending = true;
    return cudaSuccess;
}

cudaError_t match_host_async(trd_handle* h, const trd_tracks_in& in, const trd_tracks_out& out, int64_t n, cudaStream_t st) {
    TRD_TRY(ensure_pipeline(h));
    const int k = h->ring_next;
    h->ring_next = (k + 1) % trd_handle::kRing;
    TRD_TRY(retire_slot(h, k));
    const size_t bytes = (size_t)n * 4;
    TRD_TRY(reserve_idle(h, h->stage_in[k], kInArrays * bytes, st));
    TRD_TRY(reserve_idle(h, h->stage_out[k], kOutArrays * bytes, st));
    char* bi = (char*)h->stage_in[k].p;
    char* bo = (char*)h->stage_out[k].p;
    trd_tracks_in din;
    trd_tracks_out dout;
    const void* src[kInArrays];
    void* dst[kOutArrays];
    int a = 0;
    for (int j = 0; j < 5; ++j) { src[a] = in.par[j]; din.par[j] = (const float*)(bi + a * bytes); ++a; }
    for (int j = 0; j < 15; ++j) { src[a] = in.cov[j]; din.cov[j] = (const float*)(bi + a * bytes); ++a; }
    src[a] = in.x; din.x = (const float*)(bi + a * bytes); ++a;
    src[a] = in.sector; din.sector = (const int32_t*)(bi + a * bytes); ++a;
    din.interaction = nullptr;
    int b = 0;
    for (int l = 0; l < TRD_MAX_LAYERS; ++l) { dst[b] = out.tracklet_idx[l]; dout.tracklet_idx[l] = (int32_t*)(bo + b * bytes); ++b; }
    for (int j = 0; j < 5; ++j) { dst[b] = out.par[j]; dout.par[j] = (float*)(bo + b * bytes); ++b; }
    for (int j = 0; j < 15; ++j) { dst[b] = out.cov[j]; dout.cov[j] = (float*)(bo + b * bytes); ++b; }
    dst[b] = out.x; dout.x = (float*)(bo + b * bytes); ++b;
    dst[b] = out.sector; dout.sector = (int32_t*)(bo + b * bytes); ++b;
    dst[b] = out.chi2; dout.chi2 = (float*)(bo + b * bytes); ++b;
    dst[b] = out.n_matched; dout.n_matched = (int32_t*)(bo + b * bytes); ++b;
    dst[b] = out.n_cand_evals; dout.n_cand_evals = out.n_cand_evals ? (int32_t*)(bo + b * bytes) : nullptr; ++b;
    // copy in (s_in) -> kernels (caller's stream) -> copy out (s_out)
    // rows that follow each other in the caller's memory (the rows of one (5, n) or (15, n) array) go as one copy
    for (int j = 0; j < kInArrays;) {
        int m = 1;
        while (j + m < kInArrays && (const char*)src[j + m] == (const char*)src[j] + (size_t)m * bytes) ++m;
        TRD_TRY(cudaMemcpyAsync(bi + j * bytes, src[j], (size_t)m * bytes, cudaMemcpyHostToDevice, h->s_in));
        j += m;
    }
    TRD_TRY(cudaEventRecord(h->ev_in[k], h->s_in));
    TRD_TRY(cudaStreamWaitEvent(st, h->ev_in[k], 0));
    TRD_TRY(launch_match(h, din, dout, n, st));
    TRD_TRY(cudaEventRecord(h->ev_done[k], st));
    TRD_TRY(cudaStreamWaitEvent(h->s_out, h->ev_done[k], 0));
    for (int j = 0; j < kOutArrays;) {
        int m = 1;
        if (dst[j]) {
            while (j + m < kOutArrays && dst[j + m] && (char*)dst[j + m] == (char*)dst[j] + (size_t)m * bytes) ++m;
            TRD_TRY(cudaMemcpyAsync(dst[j], bo + j * bytes, (size_t)m * bytes, cudaMemcpyDeviceToHost, h->s_out));
        }
        j += m;
    }
    TRD_TRY(cudaEventRecord(h->ev_out[k], h->s_out));
    h->slot_busy[k] = true;
    return cudaSuccess;
}

cudaError_t wait_host(trd_handle* h, cudaStream_t st) {
    if (!h->s_in) return cudaSuccess;
    for (int k = 0; k < trd_handle::kRing; ++k) TRD_TRY(retire_slot(h, k));
    TRD_TRY(cudaStreamSynchronize(h->s_in));
    TRD_TRY(cudaStreamSynchronize(st));
    TRD_TRY(cudaStreamSynchronize(h->s_out));
    h->tl_pending = false;
    return cudaSuccess;
}

}  // namespace

void host_pipeline_destroy(trd_handle* h) {
    auto rel = [](Buffer& b) { if (b.p) cudaFree(b.p); b.p = nullptr; b.bytes = 0; };
    rel(h->stage_tl);
    for (int k = 0; k < trd_handle::kRing; ++k) {
        rel(h->stage_in[k]);
        rel(h->stage_out[k]);
        if (h->ev_in[k]) cudaEventDestroy(h->ev_in[k]);
        if (h->ev_done[k]) cudaEventDestroy(h->ev_done[k]);
        if (h->ev_out[k]) cudaEventDestroy(h->ev_out[k]);
    }
    if (h->ev_tl_in) cudaEventDestroy(h->ev_tl_in);
    if (h->ev_tl_used) cudaEventDestroy(h->ev_tl_used);
    if (h->s_in) cudaStreamDestroy(h->s_in);
    if (h->s_out) cudaStreamDestroy(h->s_out);
}

}  // namespace trd

extern "C" {

int trd_load_tracklets_host(trd_handle* h, const float* y, const float* z, const float* dydx,
                            const int32_t* chamber, int64_t n, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (n < 0 || n >= (1 << 29) - 1) return trd::fail(h, TRD_E_ARG, "trd_load_tracklets_host: n out of range (must be < 2^29 - 1)");
    if (n > 0 && (!y || !z || !dydx || !chamber)) return trd::fail(h, TRD_E_ARG, "trd_load_tracklets_host: NULL array");
    const cudaError_t e = trd::load_host(h, y, z, dydx, chamber, n, (cudaStream_t)stream);
    if (e != cudaSuccess) return trd::fail_cuda(h, e, "trd_load_tracklets_host");
    return TRD_OK;
}

int trd_match_host_async(trd_handle* h, const trd_tracks_in* in, const trd_tracks_out* out, int64_t n, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (!in || !out || n < 0) return trd::fail(h, TRD_E_ARG, "trd_match_host: NULL struct or negative n_tracks");
    if (!h->index_loaded) return trd::fail(h, TRD_E_STATE, "trd_match_host: no tracklets loaded");
    if (h->mp.g.n_ia > 1) return trd::fail(h, TRD_E_STATE, "trd_match_host: the index carries interactions; use trd_match");
    if (n == 0) return TRD_OK;
    for (int k = 0; k < 5; ++k)
        if (!in->par[k] || !out->par[k]) return trd::fail(h, TRD_E_ARG, "trd_match_host: NULL par array");
    for (int k = 0; k < 15; ++k)
        if (!in->cov[k] || !out->cov[k]) return trd::fail(h, TRD_E_ARG, "trd_match_host: NULL cov array");
    for (int l = 0; l < TRD_MAX_LAYERS; ++l)
        if (!out->tracklet_idx[l]) return trd::fail(h, TRD_E_ARG, "trd_match_host: NULL tracklet_idx array");
    if (!in->x || !in->sector || !out->x || !out->sector || !out->chi2 || !out->n_matched)
        return trd::fail(h, TRD_E_ARG, "trd_match_host: NULL array");
    const cudaError_t e = trd::match_host_async(h, *in, *out, n, (cudaStream_t)stream);
    if (e != cudaSuccess) return trd::fail_cuda(h, e, "trd_match_host");
    return TRD_OK;
}

int trd_wait_host(trd_handle* h, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    const cudaError_t e = trd::wait_host(h, (cudaStream_t)stream);
    if (e != cudaSuccess) return trd::fail_cuda(h, e, "trd_wait_host");
    return TRD_OK;
}

int trd_match_host(trd_handle* h, const trd_tracks_in* in, const trd_tracks_out* out, int64_t n, void* stream) {
    const int rc = trd_match_host_async(h, in, out, n, stream);
    if (rc != TRD_OK) return rc;
    return trd_wait_host(h, stream);
}

}  // extern "C"
