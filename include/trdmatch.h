/* trdmatch.h -- C ABI of the B200-native online TRD tracking step of arXiv 2003.03174.
 *
 * The operation: PAPER.md section 3 (L46-66) and Fig. 2 (L40).  ITS-TPC seed tracks
 * (y, z, sin(phi), tan(lambda), q/pT with a 5x5 covariance) are extrapolated to each of the
 * TRD layers, the TRD tracklets inside a search road derived from the track
 * covariance are scored by a chi2 built from y and z only, tracklets whose
 * inclination is more than n_sigma_angle sigma off the track inclination are excluded
 * (PAPER.md:60), the best n_hyp hypotheses per layer are kept (Fig. 2) and updated
 * with a Kalman filter.  The paper prints no equation for any of this; the
 * readings taken are listed in DESIGN.md ("Readings", R1..R35).
 *
 * Conventions: cm, Tesla, GeV/c.  Sector frame s is rotated by (s + 1/2) * 2pi/n_sectors about
 * the beam axis; the state at local x is (y, z, sin(phi), tan(lambda), q/pT); curvature
 * kappa = -0.00299792458 * bz_tesla * q/pT per cm.  A covariance is 15 floats, the lower
 * triangle row by row: yy, zy, zz, sy, sz, ss, ty, tz, ts, tt, cy, cz, cs, ct, cc.
 * chamber = sector * (n_stacks * n_layers) + stack * n_layers + layer.
 *
 * All arrays are structure-of-arrays, one contiguous array per component.  Pointers named
 * d_* or placed in trd_tracks_in / trd_tracks_out are DEVICE pointers owned by the caller
 * (the Python binding allocates them with torch); the *_host entry points take HOST pointers
 * instead and do the copies themselves.  `stream` is a cudaStream_t passed as void* (NULL =
 * the legacy default stream).  Device entry points are asynchronous on `stream` and never
 * call cudaDeviceSynchronize; they synchronise `stream` only when an internal buffer has to
 * grow.  Calls on one handle are not thread-safe; several handles may coexist.
 *
 * Every int-returning call returns TRD_OK (0) or a negative trd_status; nothing throws or
 * aborts.  trd_last_error() gives the text of the last failure on a handle.
 * There is no CPU fallback: without a CUDA device trd_create fails with TRD_E_CUDA.
 */
#ifndef TRDMATCH_H_
#define TRDMATCH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TRD_MAX_LAYERS 6
#define TRD_MAX_HYP 8
#define TRD_VERSION 100

typedef enum trd_status {
    TRD_OK = 0,
    TRD_E_ARG = -1,    /* NULL pointer, bad size, bad config field */
    TRD_E_CUDA = -2,   /* a CUDA runtime call failed (text in trd_last_error) */
    TRD_E_NOMEM = -3,  /* device or host allocation failed */
    TRD_E_STATE = -4   /* trd_match before any trd_load_tracklets */
} trd_status;

/* Geometry, field and cuts (BASELINE.json configs[0]; readings R2-R5, R8, R10-R12, R14).
 * struct_size must be sizeof(trd_config). */
typedef struct trd_config {
    uint32_t struct_size;
    int32_t n_sectors;               /* 18; 1..64 */
    int32_t n_stacks;                /* 5; only used to decode `chamber` */
    int32_t n_layers;                /* 6; 1..TRD_MAX_LAYERS */
    int32_t n_hyp;                   /* N_candidates of PAPER.md:60; 1..TRD_MAX_HYP */
    double layer_x[TRD_MAX_LAYERS];  /* local x of the layer planes, increasing */
    double z_max;                    /* half length of the detector along z (350) */
    double pad_length;               /* pad-row pitch along z (8) */
    double bz_tesla;                 /* uniform solenoid field */
    double sigma_y;                  /* tracklet y resolution (0.04) */
    double sigma_z;                  /* tracklet z resolution (pad_length / sqrt(12)) */
    double sigma_dydx;               /* tracklet inclination resolution (0.02) */
    double n_sigma_road;             /* road half width in sigma (3 or 5) */
    double n_sigma_angle;            /* inclination veto in sigma (4) */
    double chi2_cut;                 /* per-layer chi2 increment cut (15) */
    double chi2_penalty;             /* score added for a layer without tracklet (15) */
    double max_snp;                  /* a hypothesis dies at |sin(phi)| >= max_snp (0.95) */
    double ybin_width;               /* local-y bin width of the tracklet index; 0 = chosen per load */
    int32_t track_binning;           /* trd_match bins the tracks of a batch by predicted (sector, z row, y)
                                        before matching, for cache locality: 0 = when it pays (large batch
                                        against a large index), 1 = always, -1 = never.  Results do not
                                        depend on it. */
    int32_t res_model;               /* measurement model.  0: constant sigma_y, sigma_dydx, no pad tilt (the configs).
                                        1 (Fig. 3): sigma_y and sigma_dydx are second-order
                                        polynomials of the track's sin(phi), c0 + c2 (sin(phi) - sin_lorentz)^2, and the
                                        pads of layer l are tilted by +tilt (l even) / -tilt (l odd): tracklet covariance
                                        R = Rot(tau) diag(sigma_y^2, sigma_z^2) Rot(tau)^T, y road on the residual corrected
                                        with the extrapolated z, r_y - tan(tau) r_z */
    double sy_c0, sy_c2;             /* sigma_y(s)    [cm]    (res_model = 1) */
    double sd_c0, sd_c2;             /* sigma_dydx(s)         (res_model = 1) */
    double sin_lorentz;              /* optimum of both polynomials, sin of the Lorentz angle (about +-8 degrees) */
    double tan_tilt;                 /* tan of the pad tilt (2 degrees) */
    double x_ref;                    /* trd_refit: local x of the reference plane (247: the TPC outer wall of the configs) */
    double refit_var[5];             /* trd_refit: variances the covariance is reset to (y, z, sin(phi), tan(lambda), q/pT) */
    /* Material ("taking into account ... energy loss"; R32-R34): one thin slab in front of every
     * layer plane, crossed after the propagation to the plane and before the road (trd_refit crosses it inward after
     * the update).  With path = sqrt((1 + tan(lambda)^2) / (1 - sin(phi)^2)), p = sqrt(1 + tan(lambda)^2) / |q/pT|,
     * E^2 = p^2 + mass^2: scattering width theta0 = 0.0136 / (beta p) sqrt(x_over_x0 path) added to the covariance of
     * (sin(phi), tan(lambda), q/pT); mean loss dE = eloss path / beta^2 taken from E (q/pT rescaled, direction kept), its
     * fluctuation eloss_fluct dE added to the q/pT variance.  A particle with E - dE <= mass stops (the hypothesis
     * only skips from then on).  x_over_x0 = eloss = 0: no material (the configs). */
    double x_over_x0;                /* radiation lengths per layer at normal incidence, >= 0 */
    double eloss;                    /* mean energy loss per layer [GeV] at normal incidence and beta = 1, >= 0 */
    double eloss_fluct;              /* relative width of the energy-loss fluctuation, >= 0 */
    double mass;                     /* mass hypothesis [GeV], >= 0 (0.13957 for pions) */
    /* Field inhomogeneity ("taking into account inhomogenities of the magnetic field"; R35):
     * Bz(r, z) = bz_tesla (1 + bz_r2 r^2 + bz_z2 z^2), r^2 = x^2 + y^2, in cm.  Every propagation stays one helix step,
     * with the field at the middle of the straight line from its start point.  Both zero: uniform field (the configs).
     * The factor must stay positive inside the detector: 1 + bz_r2 R^2 + bz_z2 z_max^2 > 0.5 with R the last layer's
     * outer corner. */
    double bz_r2, bz_z2;             /* [1/cm^2] */
    int32_t index_sort;              /* how trd_load_tracklets orders the tracklets by bin: 0 = counting sort (count per bin,
                                        scan, placement, caller's order restored inside every bin): several kernels for
                                        loads above 2^18 tracklets, one cooperative launch up to that size; 1 = the
                                        several-kernel counting sort always; -1 = 8-bit radix passes always.  A bin of more
                                        than 32 tracklets sends a large load through the one-launch sort, which orders
                                        long bins itself (decided on the device).  The index is the same either way,
                                        except for the order of the unusable tracklets behind the last bin, which
                                        nothing reads. */
    int32_t reserved_;
} trd_config;

/* Input tracks of one batch: device pointers, each of length n_tracks. */
typedef struct trd_tracks_in {
    const float* par[5];    /* y, z, sin(phi), tan(lambda), q/pT at local x */
    const float* cov[15];   /* lower triangle, order above */
    const float* x;         /* local x of the state (247 in the configs) */
    const int32_t* sector;  /* sector frame of the state, 0..n_sectors-1 */
    const int32_t* interaction; /* interaction (collision) of the track, 0..n_interactions-1; read only when the
                                   index was built by trd_load_tracklets_tf with n_interactions > 1, else may be NULL */
} trd_tracks_in;

/* Output of one batch: caller-allocated device pointers, each of length n_tracks.  The best
 * hypothesis after the last layer: tracklet_idx[l] is the position of the attached tracklet
 * in the arrays given to trd_load_tracklets (-1 = none); state, covariance, x and sector are
 * those at the last layer plane the hypothesis reached alive; chi2 is the sum of the chi2
 * increments (no penalties).  n_cand_evals (may be NULL) counts, over all layers and
 * hypotheses of the track, the tracklets found inside both road windows and past the
 * inclination veto.  out->par[k] may alias in->par[k] (same for cov, x, sector). */
typedef struct trd_tracks_out {
    int32_t* tracklet_idx[TRD_MAX_LAYERS];
    float* par[5];
    float* cov[15];
    float* x;
    int32_t* sector;
    float* chi2;
    int32_t* n_matched;
    int32_t* n_cand_evals;
} trd_tracks_out;

/* Output of trd_refit: caller-allocated device pointers, each of length n_tracks. */
typedef struct trd_refit_out {
    float* par[5];
    float* cov[15];
    float* x;           /* x_ref for a refitted track */
    int32_t* sector;
    float* chi2;        /* sum of the chi2 increments of the refit */
    int32_t* n_used;    /* tracklets used; 0 = not refitted, the matcher's state was copied through */
} trd_refit_out;

/* What trd_load_tracklets built (for tests and traffic accounting). */
typedef struct trd_index_info {
    int64_t n_tracklets;   /* tracklets given */
    int32_t n_zrows;       /* z rows per (sector, layer) */
    int32_t n_ybins;       /* y bins per z row (power of two) */
    int64_t n_bins;        /* n_sectors * n_layers * n_zrows * n_ybins */
    double ybin_width;     /* cm */
    int32_t key_bits;      /* radix-sorted key width */
    int32_t n_passes;      /* 8-bit radix passes */
    int32_t n_interactions; /* 1 = no time-frame association */
    int32_t sort_kind;     /* 0 = radix sort, 1 = counting sort, 2 = counting sort met a long bin and the one-launch
                              sort did the work (known only after a trd_copy_index of this load; 1 until then), 3 = the
                              counting sort of small loads (up to 2^18 tracklets, index_sort = 0): one cooperative launch */
} trd_index_info;

typedef struct trd_handle trd_handle;

int trd_version(void);

/* The matcher for one geometry and one set of cuts: the 18 x 5 x 6 segmentation and layer planes of PAPER.md:50
 * (section 3, second paragraph), the search road and the chi2 from y and z only of PAPER.md:52 (n_sigma_road, chi2_cut),
 * the 4 sigma inclination veto and the N hypotheses kept per layer of PAPER.md:60 (n_sigma_angle, n_hyp).
 * Validates and copies *cfg, derives the float32 constants.  Allocates nothing proportional
 * to data.  The library owns *out until trd_destroy. */
int trd_create(const trd_config* cfg, trd_handle** out);

/* Frees everything the handle owns (synchronises the device first).  NULL is a no-op.  (Housekeeping: no passage of
 * the paper defines it.) */
void trd_destroy(trd_handle* h);

/* Builds the tracklet index on the device (north_star: "device-side sort and index by chamber
 * and local-y bin"; PAPER.md:50 for the 18 x 5 x 6 segmentation): key = ((sector, layer), z row,
 * y bin) -> stable LSD radix sort of (key, position) -> gather of (y, z, dy/dx, position) into
 * the sorted store -> first-position table per bin.  Tracklets with a chamber outside
 * 0..n_chambers-1 or a non-finite y or z are never candidates.  Replaces any previous index.
 * The four input arrays (length n, n >= 0) are only read, and only until the work queued on
 * `stream` by this call has run. */
int trd_load_tracklets(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx,
                       const int32_t* d_chamber, int64_t n, void* stream);

/* Time-frame variant (tracklets are matched only to tracks of the same interaction): as
 * trd_load_tracklets, with the interaction id of every tracklet (device array, 0..n_interactions-1; other values
 * make the tracklet unusable).  The id leads the bin key, so a track only ever scans tracklets of its own
 * interaction.  trd_match then reads trd_tracks_in.interaction; a track whose id is out of range is propagated
 * but attaches nothing.  n_interactions <= 1 or d_interaction == NULL is trd_load_tracklets.  Device arrays only
 * (the *_host entry points do not carry interaction ids in this version). */
int trd_load_tracklets_tf(trd_handle* h, const float* d_y, const float* d_z, const float* d_dydx,
                          const int32_t* d_chamber, const int32_t* d_interaction, int32_t n_interactions, int64_t n,
                          void* stream);

/* Two-stage propagation: radial offset [cm] of every chamber from its nominal layer plane, HOST
 * array of n_chambers = n_sectors * n_stacks * n_layers floats (copied; NULL or 0 chambers = all nominal).  A
 * hypothesis is extrapolated to the nominal plane ("average radius"); its (y, z) are extrapolated linearly to
 * x_layer + dx of each candidate's chamber for the road and the chi2; a selected child is re-propagated exactly to
 * that radius before the Kalman update, so the output x is x_layer + dx of the last attached chamber.  Takes effect
 * with the NEXT trd_load_tracklets (the loaded index is dropped). */
int trd_set_chamber_dx(trd_handle* h, const float* dx, int32_t n_chambers, void* stream);

/* The tracking step for one batch (n_tracks >= 0) against the loaded index -- PAPER.md:52-64 (section 3, paragraphs 3-5)
 * and Fig. 2: every track is extrapolated to each TRD layer (L52, L64), the tracklets inside the search
 * road derived from its covariance are its candidates (L52), those whose inclination is more than 4 sigma off are
 * excluded (L60), chi2 is computed from y and z only (L52), the best n_hyp hypotheses per layer are kept (L60) and
 * updated with a Kalman filter (L9, L40); tracks are independent (L86).
 * Device memory: the handle's buffers only grow.  The first call of a size allocates (cudaMalloc, which synchronises the
 * device); calls of the same or a smaller size allocate nothing, only enqueue work on `stream`, and can be captured in a
 * CUDA graph together with trd_load_tracklets (trd_last_match_kernel_ms then reads the events of the captured call as the
 * last replay recorded them). */
int trd_match(trd_handle* h, const trd_tracks_in* in, const trd_tracks_out* out, int64_t n_tracks,
              void* stream);

/* trd_match for callers that cannot allocate device memory (code under CUDA graph capture, serving loops, harnesses
 * that forbid cudaMalloc): the same tracking step (as trd_match above), on the track-binned path, with
 * every scratch buffer (packed track and result records, locality keys, permutation, key histogram) in ONE file-scope
 * device array of TRD_STATIC_SCRATCH_BYTES (7.5 MiB) that is part of the library's device image: every GPU that loads
 * the library holds it until the process exits.  The call allocates and frees nothing -- no cudaMalloc, cudaFree,
 * event or stream creation, no allocating library routine -- and only enqueues a memset and five kernels on `stream`.
 *   in, out     device arrays as for trd_match (the caller's; same layout, same ownership); results are those of
 *               trd_match on the same input (the order in which tracks are processed changes no result)
 *   n_tracks    0 .. TRD_STATIC_MAX_TRACKS; more is refused with TRD_E_ARG and a text in trd_last_error
 *   index       the tracklets must have been loaded before (trd_load_tracklets allocates; this call does not)
 * TRD_E_ARG also when the track locality key of this configuration is wider than 16 bits (time-frame association with
 * more than about 40 interactions): use trd_match there.
 * The array is shared by every call, handle and host thread of the process on that GPU and keeps the last call's
 * contents (the library clears the part that must start at zero): calls that overlap on the GPU -- different streams,
 * or different handles on the same device -- race on it.  Serialise them on one stream or with events. */
#define TRD_STATIC_MAX_TRACKS 32768
#define TRD_STATIC_SCRATCH_BYTES 7864576   /* 32768 x (96 + 128 + 4 + 4) + 4 x 65536 + 256 */
int trd_match_static(trd_handle* h, const trd_tracks_in* in, const trd_tracks_out* out, int64_t n_tracks,
                     void* stream);

/* TRD-only refit of the matched chains (calibration step 3: refits "ignoring the TPC clusters";
 * PAPER.md:9): for every track with at least two attached tracklets the matcher's final state is taken
 * as the starting point, its covariance is reset to diag(refit_var), the Kalman filter runs INWARD over the attached
 * tracklets only (same propagation, sector rule and measurement model as trd_match) and the result is propagated
 * to x_ref.  `matched` is what trd_match wrote (device arrays; the tracklets it refers to must still be the loaded
 * ones); a tracklet attached in another sector frame than the state's is skipped; tracks that cannot be refitted
 * are copied through with n_used = 0.  out->par etc. may alias matched->par etc. */
int trd_refit(trd_handle* h, const trd_tracks_out* matched, const trd_refit_out* out, int64_t n_tracks, void* stream);

/* The same two calls with HOST arrays (pinned memory makes the copies asynchronous; pageable memory works
 * too).  The library stages through its own device buffers and pipelines on two internal copy streams:
 * host->device copies, the kernels (on `stream`) and device->host copies of consecutive calls overlap.
 *   trd_load_tracklets_host   returns once the copies and kernels are queued; the arrays must stay valid
 *                             until trd_wait_host has returned;
 *   trd_match_host_async      queues copy-in, trd_match and copy-out of one batch and returns; the results
 *                             are in `out_host` only after trd_wait_host.  At most four batches are in flight:
 *                             a fifth call first waits for the oldest;
 *   trd_wait_host             blocks until everything queued by *_host calls has completed;
 *   trd_match_host            = trd_match_host_async + trd_wait_host. */
int trd_load_tracklets_host(trd_handle* h, const float* y, const float* z, const float* dydx,
                            const int32_t* chamber, int64_t n, void* stream);
int trd_match_host_async(trd_handle* h, const trd_tracks_in* in_host, const trd_tracks_out* out_host,
                         int64_t n_tracks, void* stream);
int trd_wait_host(trd_handle* h, void* stream);
int trd_match_host(trd_handle* h, const trd_tracks_in* in_host, const trd_tracks_out* out_host,
                   int64_t n_tracks, void* stream);

/* Diagnostics.  trd_copy_index copies the sorted tracklet positions (n_tracklets int32), the
 * sorted keys (n_tracklets uint32) and the first-position table (n_bins + 1 int32) to HOST
 * arrays (any may be NULL) after synchronising `stream`. */
int trd_get_index_info(const trd_handle* h, trd_index_info* info);
int trd_copy_index(trd_handle* h, int32_t* sorted_pos, uint32_t* sorted_key, int32_t* bin_first, void* stream);
const char* trd_last_error(const trd_handle* h);
int64_t trd_device_bytes(const trd_handle* h);   /* device memory currently owned by the handle (SURVEY.md 8(b) calls it
                                                     trd_scratch_bytes; renamed because it also counts the sorted store) */
int64_t trd_kernel_launches(const trd_handle* h); /* kernels launched through this handle so far */
/* Device time of the match kernel alone in the most recent trd_match (CUDA events recorded on the call's
 * stream around that one launch; waits for the end event).  TRD_E_STATE if no trd_match has run. */
int trd_last_match_kernel_ms(trd_handle* h, float* ms);
/* The same for the n most recent trd_match calls (n <= 64; ms[n - 1] is the latest): the library keeps a ring of event
 * pairs, so a timed loop can run without any synchronisation and be read afterwards. */
int trd_match_kernel_ms(trd_handle* h, float* ms, int32_t n);

#ifdef __cplusplus
}
#endif
#endif /* TRDMATCH_H_ */
