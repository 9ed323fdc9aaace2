// api.cu -- the extern "C" entry points declared in include/trdmatch.h: argument checks,
// constants, buffer ownership, the host-buffer variants.  All arithmetic of the method lives in
// index.cu and match.cu.
#include <math.h>
#include <string.h>

#include <new>

#include "trd_internal.cuh"

namespace trd {

int fail(trd_handle* h, int code, const std::string& what) {
    if (h) h->err = what;
    return code;
}

int fail_cuda(trd_handle* h, cudaError_t e, const char* where) {
    cudaGetLastError();   // clear the sticky-less error state
    const int code = (e == cudaErrorMemoryAllocation) ? TRD_E_NOMEM : TRD_E_CUDA;
    return fail(h, code, std::string(where) + ": " + cudaGetErrorString(e));
}

}  // namespace trd

namespace {

using trd::fail;
using trd::fail_cuda;

bool derive_params(const trd_config& c, trd::MatchParams& mp) {
    memset(&mp, 0, sizeof mp);
    trd::IndexGeom& g = mp.g;
    g.n_sectors = c.n_sectors;
    g.n_layers = c.n_layers;
    g.per_sector = c.n_stacks * c.n_layers;
    g.n_chambers = c.n_sectors * g.per_sector;
    mp.n_hyp = c.n_hyp;
    const double half = M_PI / c.n_sectors;
    for (int l = 0; l < c.n_layers; ++l) {
        mp.layer_x[l] = (float)c.layer_x[l];
        mp.edge[l] = (float)(c.layer_x[l] * tan(half));
    }
    mp.bd = -0.00299792458 * c.bz_tesla;
    mp.b = (float)mp.bd;
    const double cb = cos(2.0 * half), sb = sin(2.0 * half);
    mp.cb_hi = (float)cb;
    mp.sb_hi = (float)sb;
    mp.cbd = cb;
    mp.sbd = sb;
    mp.sig_y2 = (float)(c.sigma_y * c.sigma_y);
    mp.sig_z2 = (float)(c.sigma_z * c.sigma_z);
    mp.n_sigma_road = (float)c.n_sigma_road;
    mp.half_pad = (float)(0.5 * c.pad_length);
    mp.veto = (float)(c.n_sigma_angle * c.sigma_dydx);
    mp.chi2_cut = (float)c.chi2_cut;
    mp.chi2_penalty = (float)c.chi2_penalty;
    mp.max_snp = (float)c.max_snp;
    mp.res_model = c.res_model;
    mp.n_sigma_angle = (float)c.n_sigma_angle;
    mp.sy_c0 = (float)c.sy_c0;
    mp.sy_c2 = (float)c.sy_c2;
    mp.sd_c0 = (float)c.sd_c0;
    mp.sd_c2 = (float)c.sd_c2;
    mp.sin_lorentz = (float)c.sin_lorentz;
    mp.tan_tilt = (float)c.tan_tilt;
    mp.tan_half = (float)tan(half);
    mp.x_ref = (float)c.x_ref;
    for (int k = 0; k < 5; ++k) mp.refit_var[k] = (float)c.refit_var[k];
    mp.material = (c.x_over_x0 > 0.0 || c.eloss > 0.0) ? 1 : 0;
    mp.ms_k = (float)(0.0136 * 0.0136 * c.x_over_x0);
    mp.eloss = (float)c.eloss;
    mp.eloss_fluct = (float)c.eloss_fluct;
    mp.mass = (float)c.mass;
    mp.mass2 = (float)(c.mass * c.mass);
    mp.field = (c.bz_r2 != 0.0 || c.bz_z2 != 0.0) ? 1 : 0;
    mp.bz_r2 = (float)c.bz_r2;
    mp.bz_z2 = (float)c.bz_z2;
    return true;
}

const char* check_config(const trd_config& c) {
    if (c.struct_size != sizeof(trd_config)) return "trd_config.struct_size does not match this library";
    if (c.n_sectors < 1 || c.n_sectors > 64) return "n_sectors out of range";
    if (c.n_stacks < 1 || c.n_stacks > 64) return "n_stacks out of range";
    if (c.n_layers < 1 || c.n_layers > TRD_MAX_LAYERS) return "n_layers out of range";
    if (c.n_hyp < 1 || c.n_hyp > TRD_MAX_HYP) return "n_hyp out of range";
    for (int l = 0; l < c.n_layers; ++l) {
        if (!(c.layer_x[l] > 0.0) || !isfinite(c.layer_x[l])) return "layer_x must be positive";
        if (l > 0 && !(c.layer_x[l] > c.layer_x[l - 1])) return "layer_x must increase";
    }
    if (!(c.z_max > 0.0) || !(c.pad_length > 0.0)) return "z_max and pad_length must be positive";
    if (c.z_max / c.pad_length > 4096.0) return "too many pad rows";
    if (!isfinite(c.bz_tesla)) return "bz_tesla not finite";
    if (!(c.sigma_y > 0.0) || !(c.sigma_z > 0.0) || !(c.sigma_dydx > 0.0)) return "sigmas must be positive";
    if (!(c.n_sigma_road > 0.0) || !(c.n_sigma_angle > 0.0)) return "n_sigma_* must be positive";
    if (!(c.chi2_cut > 0.0) || !(c.chi2_penalty >= 0.0)) return "chi2_cut / chi2_penalty out of range";
    if (!(c.max_snp > 0.0) || !(c.max_snp < 1.0)) return "max_snp must be in (0, 1)";
    if (!(c.ybin_width >= 0.0)) return "ybin_width must be >= 0";
    if (c.track_binning < -1 || c.track_binning > 1) return "track_binning must be -1, 0 or 1";
    if (c.index_sort < -1 || c.index_sort > 1) return "index_sort must be -1, 0 or 1";
    if (c.res_model != 0 && c.res_model != 1) return "res_model must be 0 or 1";
    if (c.res_model == 1) {
        if (!(c.sy_c0 > 0.0) || !(c.sd_c0 > 0.0) || !(c.sy_c2 >= 0.0) || !(c.sd_c2 >= 0.0)) return "resolution coefficients out of range";
        if (!(fabs(c.sin_lorentz) < 1.0) || !(fabs(c.tan_tilt) < 1.0)) return "sin_lorentz / tan_tilt out of range";
    }
    if (!(c.x_over_x0 >= 0.0) || !(c.eloss >= 0.0) || !(c.eloss_fluct >= 0.0) || !(c.mass >= 0.0) || !isfinite(c.x_over_x0) ||
        !isfinite(c.eloss) || !isfinite(c.eloss_fluct) || !isfinite(c.mass))
        return "x_over_x0, eloss, eloss_fluct and mass must be finite and >= 0";
    if (!isfinite(c.bz_r2) || !isfinite(c.bz_z2)) return "bz_r2 / bz_z2 not finite";
    {   // the field factor must stay well above zero inside the detector
        const double xl = c.layer_x[c.n_layers - 1], half = M_PI / c.n_sectors;
        const double r2 = xl * xl * (1.0 + tan(half) * tan(half));
        const double lo = 1.0 + (c.bz_r2 < 0.0 ? c.bz_r2 * r2 : 0.0) + (c.bz_z2 < 0.0 ? c.bz_z2 * c.z_max * c.z_max : 0.0);
        if (!(lo > 0.5)) return "bz_r2 / bz_z2 take more than half of the field away inside the detector";
    }
    return nullptr;
}

void release(trd::Buffer& b) {
    if (b.p) cudaFree(b.p);
    b.p = nullptr;
    b.bytes = 0;
}


}  // namespace

extern "C" {

int trd_version(void) { return TRD_VERSION; }

int trd_create(const trd_config* cfg, trd_handle** out) {
    if (!cfg || !out) return TRD_E_ARG;
    *out = nullptr;
    if (check_config(*cfg)) return TRD_E_ARG;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return TRD_E_CUDA;                                   // no device: there is no CPU fallback
    }
    trd_handle* h = new (std::nothrow) trd_handle();
    if (!h) return TRD_E_NOMEM;
    h->cfg = *cfg;
    h->device = dev;
    derive_params(h->cfg, h->mp);
    cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, dev);
    *out = h;
    return TRD_OK;
}

void trd_destroy(trd_handle* h) {
    if (!h) return;
    const trd::DeviceGuard on_device(h);
    cudaDeviceSynchronize();
    release(h->store);
    release(h->packed);
    for (int s = 0; s < 2; ++s) {
        release(h->key[s]);
        release(h->val[s]);
    }
    release(h->tile_hist);
    release(h->digit_tot);
    release(h->bin_first);
    release(h->sort_flag);
    release(h->scan_partial);
    release(h->part_rec);
    release(h->part_dx);
    release(h->row_ext);
    release(h->chamber_dx);
    release(h->store_dx);
    trd::host_pipeline_destroy(h);
    release(h->trk_rec);
    release(h->trk_out);
    for (int s = 0; s < 2; ++s) {
        release(h->trk_key[s]);
        release(h->trk_val[s]);
    }
    release(h->trk_hist);
    release(h->trk_tot);
    for (int r = 0; r < trd_handle::kEvRing; ++r)
        for (int k = 0; k < 2; ++k)
            if (h->ev_match[r][k]) cudaEventDestroy(h->ev_match[r][k]);
    delete h;
}

int trd_load_tracklets(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx,
                       const int32_t* d_chamber, int64_t n, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (n < 0 || n >= (1 << 29) - 1) return fail(h, TRD_E_ARG, "trd_load_tracklets: n out of range (must be < 2^29 - 1)");
    if (n > 0 && (!d_y || !d_z || !d_dydx || !d_chamber)) return fail(h, TRD_E_ARG, "trd_load_tracklets: NULL array");
    const cudaError_t e = trd::build_index(h, d_y, d_z, d_dydx, d_chamber, nullptr, 1, n, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_load_tracklets");
    return TRD_OK;
}

int trd_load_tracklets_tf(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx,
                          const int32_t* d_chamber, const int32_t* d_interaction, int32_t n_interactions, int64_t n,
                          void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (n < 0 || n >= (1 << 29) - 1) return fail(h, TRD_E_ARG, "trd_load_tracklets_tf: n out of range (must be < 2^29 - 1)");
    if (n > 0 && (!d_y || !d_z || !d_dydx || !d_chamber)) return fail(h, TRD_E_ARG, "trd_load_tracklets_tf: NULL array");
    if (n_interactions > (1 << 20)) return fail(h, TRD_E_ARG, "trd_load_tracklets_tf: too many interactions");
    const cudaError_t e = trd::build_index(h, d_y, d_z, d_dydx, d_chamber, d_interaction, n_interactions, n, (cudaStream_t)stream);
    if (e == cudaErrorInvalidValue) return fail(h, TRD_E_ARG, "trd_load_tracklets_tf: interactions x rows exceed the key range");
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_load_tracklets_tf");
    return TRD_OK;
}

int trd_set_chamber_dx(trd_handle* h, const float* dx, int32_t n_chambers, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    cudaStream_t st = (cudaStream_t)stream;
    if (!dx || n_chambers == 0) {                        // back to the nominal planes
        h->mp.dx_max = 0.0f;
        h->index_loaded = false;
        return TRD_OK;
    }
    if (n_chambers != h->mp.g.n_chambers) return fail(h, TRD_E_ARG, "trd_set_chamber_dx: n_chambers does not match the geometry");
    float mx = 0.0f;
    for (int c = 0; c < n_chambers; ++c) {
        if (!isfinite(dx[c])) return fail(h, TRD_E_ARG, "trd_set_chamber_dx: offset not finite");
        mx = fmaxf(mx, fabsf(dx[c]));
    }
    cudaError_t e = trd::reserve(h->chamber_dx, (size_t)n_chambers * sizeof(float), st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(h->chamber_dx.p, dx, (size_t)n_chambers * sizeof(float), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);  // dx may be pageable and freed by the caller
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_set_chamber_dx");
    h->mp.dx_max = mx;
    h->index_loaded = false;                             // the next trd_load_tracklets picks the offsets up
    return TRD_OK;
}

int trd_refit(trd_handle* h, const trd_tracks_out* m, const trd_refit_out* out, int64_t n, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (!m || !out || n < 0) return fail(h, TRD_E_ARG, "trd_refit: NULL struct or negative n_tracks");
    if (!h->index_loaded) return fail(h, TRD_E_STATE, "trd_refit: no tracklets loaded");
    if (!(h->cfg.x_ref > 0.0)) return fail(h, TRD_E_ARG, "trd_refit: trd_config.x_ref must be positive");
    for (int k = 0; k < 5; ++k)
        if (!(h->cfg.refit_var[k] > 0.0)) return fail(h, TRD_E_ARG, "trd_refit: trd_config.refit_var must be positive");
    if (n == 0) return TRD_OK;
    for (int k = 0; k < 5; ++k)
        if (!m->par[k] || !out->par[k]) return fail(h, TRD_E_ARG, "trd_refit: NULL par array");
    for (int k = 0; k < 15; ++k)
        if (!m->cov[k] || !out->cov[k]) return fail(h, TRD_E_ARG, "trd_refit: NULL cov array");
    for (int l = 0; l < TRD_MAX_LAYERS; ++l)
        if (!m->tracklet_idx[l]) return fail(h, TRD_E_ARG, "trd_refit: NULL tracklet_idx array");
    if (!m->x || !m->sector || !out->x || !out->sector || !out->chi2 || !out->n_used)
        return fail(h, TRD_E_ARG, "trd_refit: NULL array");
    const cudaError_t e = trd::launch_refit(h, *m, *out, n, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_refit");
    return TRD_OK;
}

int trd_match(trd_handle* h, const trd_tracks_in* in, const trd_tracks_out* out, int64_t n_tracks, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (!in || !out || n_tracks < 0) return fail(h, TRD_E_ARG, "trd_match: NULL struct or negative n_tracks");
    if (!h->index_loaded) return fail(h, TRD_E_STATE, "trd_match: no tracklets loaded");
    if (n_tracks == 0) return TRD_OK;
    for (int k = 0; k < 5; ++k)
        if (!in->par[k] || !out->par[k]) return fail(h, TRD_E_ARG, "trd_match: NULL par array");
    for (int k = 0; k < 15; ++k)
        if (!in->cov[k] || !out->cov[k]) return fail(h, TRD_E_ARG, "trd_match: NULL cov array");
    for (int l = 0; l < TRD_MAX_LAYERS; ++l)
        if (!out->tracklet_idx[l]) return fail(h, TRD_E_ARG, "trd_match: NULL tracklet_idx array");
    if (!in->x || !in->sector || !out->x || !out->sector || !out->chi2 || !out->n_matched)
        return fail(h, TRD_E_ARG, "trd_match: NULL array");
    if (h->mp.g.n_ia > 1 && !in->interaction)
        return fail(h, TRD_E_ARG, "trd_match: the index carries interactions but trd_tracks_in.interaction is NULL");
    const cudaError_t e = trd::launch_match(h, *in, *out, n_tracks, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_match");
    return TRD_OK;
}

int trd_match_static(trd_handle* h, const trd_tracks_in* in, const trd_tracks_out* out, int64_t n_tracks, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (!in || !out || n_tracks < 0) return fail(h, TRD_E_ARG, "trd_match_static: NULL struct or negative n_tracks");
    if (n_tracks > TRD_STATIC_MAX_TRACKS)
        return fail(h, TRD_E_ARG, "trd_match_static: n_tracks = " + std::to_string(n_tracks) + " exceeds TRD_STATIC_MAX_TRACKS = " +
                                      std::to_string(TRD_STATIC_MAX_TRACKS) + " (the static scratch array holds no more; use trd_match)");
    if (!h->index_loaded) return fail(h, TRD_E_STATE, "trd_match_static: no tracklets loaded");
    if (trd::track_key_bits(h) > trd::kCountingBits)
        return fail(h, TRD_E_ARG, "trd_match_static: the track locality key of this configuration is wider than 16 bits (use trd_match)");
    if (n_tracks == 0) return TRD_OK;
    for (int k = 0; k < 5; ++k)
        if (!in->par[k] || !out->par[k]) return fail(h, TRD_E_ARG, "trd_match_static: NULL par array");
    for (int k = 0; k < 15; ++k)
        if (!in->cov[k] || !out->cov[k]) return fail(h, TRD_E_ARG, "trd_match_static: NULL cov array");
    for (int l = 0; l < TRD_MAX_LAYERS; ++l)
        if (!out->tracklet_idx[l]) return fail(h, TRD_E_ARG, "trd_match_static: NULL tracklet_idx array");
    if (!in->x || !in->sector || !out->x || !out->sector || !out->chi2 || !out->n_matched)
        return fail(h, TRD_E_ARG, "trd_match_static: NULL array");
    if (h->mp.g.n_ia > 1 && !in->interaction)
        return fail(h, TRD_E_ARG, "trd_match_static: the index carries interactions but trd_tracks_in.interaction is NULL");
    const cudaError_t e = trd::launch_match_static(h, *in, *out, n_tracks, (cudaStream_t)stream);
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_match_static");
    return TRD_OK;
}

int trd_get_index_info(const trd_handle* h, trd_index_info* info) {
    if (!h || !info) return TRD_E_ARG;
    if (!h->index_loaded) return TRD_E_STATE;
    info->n_tracklets = h->n_tracklets;
    info->n_zrows = h->mp.g.nz;
    info->n_ybins = 1 << h->mp.g.nb_shift;
    info->n_bins = h->mp.g.n_bins;
    info->ybin_width = h->ybin_width;
    info->key_bits = h->key_bits;
    info->n_passes = h->n_passes;
    info->n_interactions = h->mp.g.n_ia;
    info->sort_kind = h->sort_kind;
    return TRD_OK;
}

int trd_copy_index(trd_handle* h, int32_t* sorted_pos, uint32_t* sorted_key, int32_t* bin_first, void* stream) {
    if (!h) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (!h->index_loaded) return fail(h, TRD_E_STATE, "trd_copy_index: no tracklets loaded");
    cudaStream_t st = (cudaStream_t)stream;
    cudaError_t e = cudaStreamSynchronize(st);
    const size_t n = (size_t)h->n_tracklets;
    if (e == cudaSuccess) e = trd::export_sorted_index(h, st);
    if (e == cudaSuccess && sorted_pos && n)
        e = cudaMemcpy(sorted_pos, h->val[h->sorted_side].p, n * 4, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && sorted_key && n)
        e = cudaMemcpy(sorted_key, h->key[h->sorted_side].p, n * 4, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess && bin_first)
        e = cudaMemcpy(bin_first, h->bin_first.p, ((size_t)h->mp.g.n_bins + 1) * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return fail_cuda(h, e, "trd_copy_index");
    return TRD_OK;
}

const char* trd_last_error(const trd_handle* h) { return h ? h->err.c_str() : "NULL handle"; }

int64_t trd_device_bytes(const trd_handle* h) {
    if (!h) return 0;
    size_t t = h->store.bytes + h->packed.bytes + h->part_rec.bytes + h->part_dx.bytes + h->scan_partial.bytes + h->tile_hist.bytes + h->digit_tot.bytes + h->bin_first.bytes + h->row_ext.bytes + h->chamber_dx.bytes + h->store_dx.bytes + h->stage_tl.bytes + h->trk_rec.bytes + h->trk_out.bytes + h->trk_hist.bytes +
               h->trk_tot.bytes;
    for (int s = 0; s < 2; ++s) t += h->key[s].bytes + h->val[s].bytes + h->trk_key[s].bytes + h->trk_val[s].bytes;
    return (int64_t)t;
}

int64_t trd_kernel_launches(const trd_handle* h) { return h ? h->launches : 0; }

int trd_match_kernel_ms(trd_handle* h, float* ms, int32_t n) {
    if (!h || !ms || n < 1) return TRD_E_ARG;
    const trd::DeviceGuard on_device(h);
    if (n > trd_handle::kEvRing || n > h->ev_count) return fail(h, TRD_E_STATE, "trd_match_kernel_ms: fewer trd_match calls on record");
    for (int k = 0; k < n; ++k) {                     // ms[n - 1] is the most recent call
        cudaEvent_t* ev = h->ev_match[(h->ev_count - n + k) % trd_handle::kEvRing];
        cudaError_t e = cudaEventSynchronize(ev[1]);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms[k], ev[0], ev[1]);
        if (e != cudaSuccess) return fail_cuda(h, e, "trd_match_kernel_ms");
    }
    return TRD_OK;
}

int trd_last_match_kernel_ms(trd_handle* h, float* ms) { return trd_match_kernel_ms(h, ms, 1); }

}  // extern "C"
