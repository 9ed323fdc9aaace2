// trd_oracle.cpp -- ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, double-precision CPU implementation of the online TRD tracking step of
// arXiv 2003.03174 (section 3, Fig. 2 L40): ITS-TPC seed tracks are
// propagated through the six TRD layers, the tracklets inside a search road are scored by
// chi2, the best N hypotheses are kept per layer and updated with a Kalman filter.
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
// may build, load or call this file.  It shares no code, header, table or helper with the
// CUDA path under paper_2003_03174_b200/csrc/ and includes nothing from include/.
//
// The method is a heuristic beam search, so this file is the algorithm written out step by
// step; full 5x5 matrices, std::sort, std::lower_bound, no blocking
// or fusion.  The paper prints no equation for the track model, road, chi2, gain or ranking;
// every reading taken is listed in DESIGN.md ("Readings") and referenced as [R#] below.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"): closed-form straight line at Bz = 0,
// analytic circle crossing, composition and inverse of propagation, finite-difference
// Jacobians, information-form Kalman update via numpy.linalg, batch least squares, exact
// recovery on noise-free input, unit pulls and <chi2> = ndf on smeared input, index ==
// brute force, beam search == exhaustive chain enumeration, nHyp = 1 == greedy matcher.
// No function here is "parity unpinned".
//
// Conventions [R1]: sector frame s rotated by (s + 1/2) * 20 deg about z; state at local x is
// p = (y, z, sin(phi), tan(lambda), q/pT [c/GeV]); cos(phi) > 0 implied; curvature
// kappa = b * q/pT with b = -0.00299792458 * Bz[T] per cm; cm, Tesla, GeV/c.  Covariance is
// the symmetric 5x5 matrix; the 15-element interface order is the lower triangle row by row
// (yy, zy, zz, sy, sz, ss, ty, tz, ts, tt, cy, cz, cs, ct, cc).

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <deque>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

constexpr int kMaxLayers = 6;
constexpr double kLoose = 1e-2;   // slack used only to decide which margins are worth recording

struct Config {
    int32_t n_sectors, n_stacks, n_layers, n_hyp;
    double layer_x[kMaxLayers];
    double z_max, pad_length, bz_tesla;
    double sigma_y, sigma_z, sigma_dydx;
    double n_sigma_road, n_sigma_angle;
    double chi2_cut, chi2_penalty, max_snp;
    // measurement model of PAPER.md:62 (Fig. 3) and PAPER.md:66, readings [R24-R26]; res_model = 0: constants
    double sy_c0, sy_c2, sd_c0, sd_c2, sin_lorentz, tan_tilt;
    int32_t res_model, pad_;
    // TRD-only refit (PAPER.md:33 step 3) [R31]: reference plane and the variances the covariance is reset to
    double x_ref, refit_var[5];
    // material in front of every layer plane ("taking into account ... energy loss") [R32, R33]:
    // thickness in radiation lengths and mean energy loss [GeV] at normal incidence and beta = 1, relative width of
    // the energy-loss fluctuation, particle mass [GeV].  All zero = no material (the configs).
    double x_over_x0, eloss, eloss_fluct, mass;
    // field inhomogeneity ("taking into account inhomogenities of the magnetic field") [R35]:
    // Bz(r, z) = bz_tesla (1 + bz_r2 r^2 + bz_z2 z^2), r^2 = x^2 + y^2 [cm^2].  Both zero = uniform field (the configs).
    double bz_r2, bz_z2;
};

struct Hyp {
    double p[5];
    double C[5][5];
    double x;
    int sector;
    double score;      // sum of chi2 increments + penalty * skipped layers   [R5]
    double chi2;       // sum of chi2 increments only
    int idx[kMaxLayers];
    int n_matched;
    bool alive;
    int ia;            // interaction of the track [R27]
};

struct Tracklet {
    double y, z, dydx;
    int index;         // position in the caller's arrays
    int ia;            // interaction (collision) the tracklet belongs to; 0 without time-frame association [R27]
    double dx;         // radial offset of the tracklet's chamber from the nominal layer plane [R28]
};

struct Counters {
    int64_t n_prop = 0, n_rot = 0, n_road = 0, n_cand = 0, n_upd = 0, n_scanned = 0;
    unsigned char* touched = nullptr;   // optional, one byte per tracklet: set for every tracklet found inside a road
};

// kappa = b q/pT; b from the field at the point (x, y, z) of the current sector frame (r^2 = x^2 + y^2 in any frame) [R35]
inline double curvature_factor(const Config& cfg, double x, double y, double z) {
    return -0.00299792458 * cfg.bz_tesla * (1.0 + cfg.bz_r2 * (x * x + y * y) + cfg.bz_z2 * z * z);
}

// ---- fragile decisions (R23: "several results are correct") ---------------------------
// Every discrete decision of the algorithm compares a quantity with a threshold.  note() records the smallest relative
// distance of any of them from its threshold: the per-track `margin`.  A float32 implementation may take a decision
// whose distance is below its rounding the other way, and the result it then reaches is as legitimate as this one.
// To check such a result (orc_match_alternatives) a track is replayed with chosen decisions taken the other way:
// while a Replay is active, note() numbers the decisions closer than eps to their threshold in the order they are met
// and returns true for those the replay flips.  Nothing else changes: with no Replay (every normal run) note() only
// records the margin and returns false.
constexpr int kMaxDecisions = 64;
struct Replay {
    double eps = 0.0;
    int n_forced = 0;                           // decisions 0 .. n_forced-1 take forced[], later ones their natural outcome
    unsigned char forced[kMaxDecisions] = {};   // 1 = the other way
    int n_seen = 0;                             // fragile decisions met by the run
};
thread_local Replay* t_replay = nullptr;

inline bool note(double* margin, double value, double threshold) {
    // relative distance of a quantity from the threshold it is compared with
    if (!margin && !t_replay) return false;
    const double m = std::fabs(value - threshold) / std::fabs(threshold);
    if (margin && m < *margin) *margin = m;
    if (t_replay && m < t_replay->eps) {
        const int k = t_replay->n_seen++;
        if (k < t_replay->n_forced && k < kMaxDecisions) return t_replay->forced[k] != 0;
    }
    return false;
}

// (asin(w) - w) / w^2, with its series near 0
inline double q_of(double w) {
    if (std::fabs(w) < 1e-2) {
        double w2 = w * w;
        return w * (1.0 / 6.0 + w2 * (3.0 / 40.0 + w2 * (15.0 / 336.0 + w2 * (105.0 / 3456.0))));
    }
    return (std::asin(w) - w) / (w * w);
}

// ---- propagation x0 -> x1 inside one sector frame: one helix step in the field at its middle ---------------
// PAPER.md:52 ("extrapolated to the first TRD layer"); formulas SURVEY.md 8(c).3.
// Returns false (state untouched) if |sin(phi)| would reach max_snp [R14].  F, if given,
// receives the 5x5 Jacobian d(y',z',s',t',c')/d(y,z,s,t,c).
bool propagate_state(const Config& cfg, const double p[5], double x0, double x1, double out[5],
                     double F[5][5], double* margin) {
    const double dx = x1 - x0;
    const double y = p[0], z = p[1], s = p[2], t = p[3], c = p[4];
    if (std::fabs(s) >= 1.0) return false;
    // one helix step with the field taken at the middle of the straight line from the start point [R35]
    const double r0 = std::sqrt(1.0 - s * s);
    const double b = curvature_factor(cfg, x0 + 0.5 * dx, y + 0.5 * dx * s / r0, z + 0.5 * dx * t / r0);
    const double kappa = b * c;
    const double u = kappa * dx;
    const double f1 = s, f2 = s + u;
    const bool flip = note(margin, std::fabs(f2), cfg.max_snp);
    if (std::fabs(f1) >= 1.0 || std::fabs(f2) >= 1.0 || ((std::fabs(f2) >= cfg.max_snp) != flip)) return false;
    const double r1 = std::sqrt(1.0 - f1 * f1), r2 = std::sqrt(1.0 - f2 * f2);
    const double cosd = r1 * r2 + f1 * f2;               // cos of the turning angle
    const double g = (1.0 + cosd) / (r1 + r2);
    const double w = u * g;                              // sin of the turning angle
    const double asw = (std::fabs(w) < 1e-8) ? 1.0 : std::asin(w) / w;
    const double ell = dx * g * asw;                     // xy path length
    out[0] = y + dx * (f1 + f2) / (r1 + r2);
    out[1] = z + t * ell;
    out[2] = f2;
    out[3] = t;
    out[4] = c;
    if (F) {
        for (int i = 0; i < 5; ++i)
            for (int j = 0; j < 5; ++j) F[i][j] = (i == j) ? 1.0 : 0.0;
        const double h = f2 * g / (r2 * (r1 + r2)) - g * g * q_of(w);
        F[0][2] = dx * g / (r1 * r2);
        F[0][4] = b * dx * dx * g / (r2 * (r1 + r2));
        F[1][2] = t * dx * (f1 + f2) / (r1 * r2 * (r1 + r2));
        F[1][3] = ell;
        F[1][4] = b * t * dx * dx * h;
        F[2][4] = b * dx;
    }
    return true;
}

void similarity(const double A[5][5], double C[5][5]) {   // C <- A C A^T, full matrices
    double T[5][5], R[5][5];
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j < 5; ++j) {
            double acc = 0.0;
            for (int k = 0; k < 5; ++k) acc += A[i][k] * C[k][j];
            T[i][j] = acc;
        }
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j < 5; ++j) {
            double acc = 0.0;
            for (int k = 0; k < 5; ++k) acc += T[i][k] * A[j][k];
            R[i][j] = acc;
        }
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j < 5; ++j) C[i][j] = 0.5 * (R[i][j] + R[j][i]);
}

bool propagate(const Config& cfg, Hyp& h, double x1, double* margin, Counters* cnt) {
    double out[5], F[5][5];
    if (cnt) cnt->n_prop++;
    if (!propagate_state(cfg, h.p, h.x, x1, out, F, margin)) return false;
    std::memcpy(h.p, out, sizeof out);
    similarity(F, h.C);
    h.x = x1;
    return true;
}

// ---- rotation of the frame by beta about z at the current point ------
// Same physical point and direction, new frame; the Jacobian brings a perturbed track back
// to the plane x' = const of the new frame.
bool rotate_state(const Config& cfg, const double p[5], double x, double beta, double out[5],
                  double* x_out, double J[5][5], double* margin) {
    const double cb = std::cos(beta), sb = std::sin(beta);
    const double y = p[0], s = p[2], t = p[3];
    if (std::fabs(s) >= 1.0) return false;
    const double r = std::sqrt(1.0 - s * s);
    const double s2 = s * cb - r * sb;
    const double c2 = r * cb + s * sb;                    // cos(phi) in the new frame
    const bool flip = note(margin, std::fabs(s2), cfg.max_snp);
    if (std::fabs(s2) >= 1.0 || ((std::fabs(s2) >= cfg.max_snp) != flip) || c2 <= 0.0) return false;
    const double r2 = std::sqrt(1.0 - s2 * s2);
    *x_out = x * cb + y * sb;
    out[0] = -x * sb + y * cb;
    out[1] = p[1];
    out[2] = s2;
    out[3] = p[3];
    out[4] = p[4];
    if (J) {
        const double kappa = curvature_factor(cfg, x, y, p[1]) * p[4];
        for (int i = 0; i < 5; ++i)
            for (int j = 0; j < 5; ++j) J[i][j] = (i == j) ? 1.0 : 0.0;
        J[0][0] = r / r2;
        J[1][0] = -t * sb / r2;
        J[2][0] = -kappa * sb;
        J[2][2] = r2 / r;
    }
    return true;
}

bool rotate(const Config& cfg, Hyp& h, double beta, double* margin, Counters* cnt) {
    double out[5], J[5][5], xn;
    if (cnt) cnt->n_rot++;
    if (!rotate_state(cfg, h.p, h.x, beta, out, &xn, J, margin)) return false;
    std::memcpy(h.p, out, sizeof out);
    similarity(J, h.C);
    h.x = xn;
    return true;
}

// ---- material: a thin slab crossed at the current point ("energy loss and
// multiple scattering as process noise", C' = F C F^T + Q) [R32, R33].  dir = +1 going outward (the particle loses
// energy), -1 going inward (the refit runs against the flight direction and gives the energy back).
//   path factor      ell = sqrt((1 + t^2) / (1 - s^2))          (slab normal to the local x axis)
//   momentum         p = sqrt(1 + t^2) / |c|,  E = sqrt(p^2 + m^2),  beta = p / E
//   scattering       theta0 = 0.0136 GeV / (beta p) sqrt(x/X0 ell)   (Highland's width without the log term)
//                    two independent angles: theta1 changes lambda, theta2 / cos(lambda) changes phi, |p| stays:
//                    ds = sqrt(1 - s^2) sqrt(1 + t^2) theta2,  dt = (1 + t^2) theta1,  dc = c t theta1
//                    Q_ss = th0^2 (1 - s^2)(1 + t^2), Q_tt = th0^2 (1 + t^2)^2, Q_tc = th0^2 c t (1 + t^2), Q_cc = th0^2 c^2 t^2
//   energy loss      dE = eloss ell / beta^2,  E' = E - dir dE,  p' = sqrt(E'^2 - m^2),  c' = c p / p'  (direction kept);
//                    fluctuation sigma_E = eloss_fluct dE, d(c)/dE = c E / p^2:  Q_cc += (c E / p^2 sigma_E)^2
// Position and covariance of (y, z) are untouched (thin slab); the covariance gets only the additive Q (the
// Jacobian of the mean energy-loss correction, 1 + O(dE / E), is neglected).  Returns false if the particle stops.
inline bool has_material(const Config& cfg) { return cfg.x_over_x0 > 0.0 || cfg.eloss > 0.0; }

bool apply_material(const Config& cfg, Hyp& h, int dir, double* margin) {
    const double s = h.p[2], t = h.p[3], c = h.p[4];
    if (c == 0.0 || std::fabs(s) >= 1.0) return true;           // infinite momentum: nothing happens
    const double ell = std::sqrt((1.0 + t * t) / (1.0 - s * s));
    const double p2 = (1.0 + t * t) / (c * c);
    const double e2 = p2 + cfg.mass * cfg.mass;
    const double beta2 = p2 / e2;
    const double E = std::sqrt(e2);
    const double dE = cfg.eloss * ell / beta2;
    const double E1 = E - dir * dE;
    if (dE > 0.0) {
        const bool flip = note(margin, E1, cfg.mass);
        if ((E1 <= cfg.mass) != flip) return false;             // stopped in the slab: state untouched
    }
    const double th2 = 0.0136 * 0.0136 * cfg.x_over_x0 * ell / (beta2 * p2);
    h.C[2][2] += th2 * (1.0 - s * s) * (1.0 + t * t);
    h.C[3][3] += th2 * (1.0 + t * t) * (1.0 + t * t);
    h.C[3][4] += th2 * c * t * (1.0 + t * t);
    h.C[4][3] = h.C[3][4];
    h.C[4][4] += th2 * c * c * t * t;
    if (dE > 0.0) {
        const double sigE = cfg.eloss_fluct * dE;
        const double dcdE = c * E / p2;
        h.C[4][4] += dcdE * dcdE * sigE * sigE;
        h.p[4] = c * std::sqrt(p2 / (E1 * E1 - cfg.mass * cfg.mass));
    }
    return true;
}

// propagate to the layer plane x = X; change sector while |y| is beyond the sector edge
// X tan(10 deg), at most twice [R14].  On failure the hypothesis is left untouched.
bool propagate_to_layer(const Config& cfg, Hyp& h, double X, double* margin, Counters* cnt) {
    Hyp w = h;
    const double half = M_PI / cfg.n_sectors;
    const double edge = X * std::tan(half);
    if (!propagate(cfg, w, X, margin, cnt)) return false;
    for (int n_rot = 0;; ++n_rot) {
        const bool flip = note(margin, std::fabs(w.p[0]), edge);
        if ((std::fabs(w.p[0]) <= edge) != flip) break;
        if (n_rot == 2) return false;
        const double beta = (w.p[0] > 0.0 ? 2.0 : -2.0) * half;
        if (!rotate(cfg, w, beta, margin, cnt)) return false;
        w.sector = (w.sector + (beta > 0.0 ? 1 : cfg.n_sectors - 1)) % cfg.n_sectors;
        if (!propagate(cfg, w, X, margin, cnt)) return false;
    }
    h = w;
    return true;
}

// ---- measurement model: m = (y, z), H = first two rows of I [R3]
// res_model = 0: R = diag(sy^2, sz^2), constant sigma_dydx, no tilt [R10, R19].
// res_model = 1 (PAPER.md:62 + Fig. 3 L58) [R24-R26]: sigma_y and sigma_dydx are second-order
// polynomials of the track's sin(phi) with their optimum at the Lorentz angle, c0 + c2 (s - sL)^2; the pads of
// layer L are tilted by tau_L = +-tilt (alternating), so the precise coordinate (sigma_y) is across the pad and
// the coarse one (sigma_z) along it: R = Rot(tau) diag(sy^2, sz^2) Rot(tau)^T, i.e. correlated y-z errors.  The
// y road is applied to the residual corrected with the extrapolated z, r'_y = r_y - tan(tau) r_z, whose
// variance is (A S A^T)_yy with A = [[1, -tan(tau)], [0, 1]]; chi2 = r^T S^-1 r is invariant under A.
// Two-stage propagation [R28-R30]: the hypothesis sits at the nominal ("average") radius of the layer;
// for the road and chi2 its (y, z) are extrapolated linearly to the radius of each tracklet's chamber,
// y + dx tan(phi), z + dx tan(lambda) / cos(phi); a kept child is re-propagated exactly to that radius before the
// Kalman update.
struct Road {
    double Sinv[2][2];
    double road_y, road_z, tanphi;
    double tan_tilt, veto;
    double zslope;     // dz/dx of the track = tan(lambda) / cos(phi)
};

Road make_road(const Config& cfg, const Hyp& h, int layer) {
    Road rd;
    double Ryy = cfg.sigma_y * cfg.sigma_y, Ryz = 0.0, Rzz = cfg.sigma_z * cfg.sigma_z;
    rd.tan_tilt = 0.0;
    rd.veto = cfg.n_sigma_angle * cfg.sigma_dydx;
    if (cfg.res_model != 0) {
        const double ds = h.p[2] - cfg.sin_lorentz;
        const double sy = cfg.sy_c0 + cfg.sy_c2 * ds * ds;
        const double sd = cfg.sd_c0 + cfg.sd_c2 * ds * ds;
        const double t = (layer % 2 == 0) ? cfg.tan_tilt : -cfg.tan_tilt;
        const double c2 = 1.0 / (1.0 + t * t), sz2 = cfg.sigma_z * cfg.sigma_z;
        Ryy = c2 * (sy * sy + t * t * sz2);
        Ryz = c2 * t * (sz2 - sy * sy);
        Rzz = c2 * (t * t * sy * sy + sz2);
        rd.tan_tilt = t;
        rd.veto = cfg.n_sigma_angle * sd;
    }
    const double S00 = h.C[0][0] + Ryy;
    const double S01 = h.C[1][0] + Ryz;
    const double S11 = h.C[1][1] + Rzz;
    const double det = S00 * S11 - S01 * S01;
    rd.Sinv[0][0] = S11 / det;
    rd.Sinv[0][1] = rd.Sinv[1][0] = -S01 / det;
    rd.Sinv[1][1] = S00 / det;
    const double t = rd.tan_tilt;
    rd.road_y = cfg.n_sigma_road * std::sqrt(S00 - 2.0 * t * S01 + t * t * S11);     // [R2], of the corrected residual
    rd.road_z = cfg.n_sigma_road * std::sqrt(h.C[1][1]) + 0.5 * cfg.pad_length;      // [R2]
    rd.tanphi = h.p[2] / std::sqrt(1.0 - h.p[2] * h.p[2]);
    rd.zslope = h.p[3] / std::sqrt(1.0 - h.p[2] * h.p[2]);
    return rd;
}

inline double chi2_of(const Road& rd, double ry, double rz) {
    return ry * (rd.Sinv[0][0] * ry + rd.Sinv[0][1] * rz) + rz * (rd.Sinv[1][0] * ry + rd.Sinv[1][1] * rz);
}

// Kalman update with the measurement (ym, zm), plain gain form
double kalman_update(const Config& cfg, Hyp& h, int layer, double ym, double zm) {
    const Road rd = make_road(cfg, h, layer);
    const double r[2] = {ym - h.p[0], zm - h.p[1]};
    const double chi2inc = chi2_of(rd, r[0], r[1]);
    double K[5][2];
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j < 2; ++j) K[i][j] = h.C[i][0] * rd.Sinv[0][j] + h.C[i][1] * rd.Sinv[1][j];
    for (int i = 0; i < 5; ++i) h.p[i] += K[i][0] * r[0] + K[i][1] * r[1];
    double N[5][5];
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j < 5; ++j) N[i][j] = h.C[i][j] - (K[i][0] * h.C[0][j] + K[i][1] * h.C[1][j]);
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j < 5; ++j) h.C[i][j] = 0.5 * (N[i][j] + N[j][i]);
    return chi2inc;
}

// ---- tracklet store: one list per (sector, layer), sorted by y --------------------------
// Time-frame association ("only those tracklets which belong to the same interaction") [R27]:
// with n_ia > 1 every tracklet and track carries an interaction id in 0..n_ia-1 and only equal ids match.  The
// sorted store keeps one y-sorted list per (interaction, sector, layer); the brute-force store keeps one list
// per (sector, layer) and compares the ids tracklet by tracklet -- the two must give identical results.
struct Store {
    int n_sectors = 0, n_layers = 0, n_ia = 1;
    double dx_max = 0.0;                       // largest |chamber offset| [R28]
    std::vector<std::vector<Tracklet>> cell;   // [(ia *) sector * n_layers + layer]
    bool sorted = false, by_ia = false;
};

void build_store(const Config& cfg, const float* y, const float* z, const float* dydx, const int32_t* chamber,
                 const int32_t* ia, int n_ia, const double* chamber_dx, int64_t n, bool sort_by_y, Store& st) {
    st.dx_max = 0.0;
    if (chamber_dx)
        for (int c = 0; c < cfg.n_sectors * cfg.n_stacks * cfg.n_layers; ++c) st.dx_max = std::max(st.dx_max, std::fabs(chamber_dx[c]));
    st.n_sectors = cfg.n_sectors;
    st.n_layers = cfg.n_layers;
    st.n_ia = (ia && n_ia > 1) ? n_ia : 1;
    st.by_ia = sort_by_y && st.n_ia > 1;
    st.cell.assign((size_t)(st.by_ia ? st.n_ia : 1) * cfg.n_sectors * cfg.n_layers, {});
    const int per_sector = cfg.n_stacks * cfg.n_layers;
    for (int64_t i = 0; i < n; ++i) {
        const int ch = chamber[i];
        if (ch < 0 || ch >= cfg.n_sectors * per_sector) continue;             // unusable tracklet
        if (!std::isfinite(y[i]) || !std::isfinite(z[i])) continue;
        const int a = (st.n_ia > 1) ? ia[i] : 0;
        if (a < 0 || a >= st.n_ia) continue;                                  // no such interaction
        const int sector = ch / per_sector, layer = ch % cfg.n_layers;        // stack id unused [R12]
        const size_t c = ((size_t)(st.by_ia ? a : 0) * cfg.n_sectors + sector) * cfg.n_layers + layer;
        st.cell[c].push_back({(double)y[i], (double)z[i], (double)dydx[i], (int)i, a, chamber_dx ? chamber_dx[ch] : 0.0});
    }
    if (sort_by_y)
        for (auto& v : st.cell)
            std::sort(v.begin(), v.end(), [](const Tracklet& a, const Tracklet& b) {
                return a.y < b.y || (a.y == b.y && a.index < b.index);
            });
    st.sorted = sort_by_y;
}

struct Cand {
    int index;
    double y, z, chi2inc, dx;
};

// all tracklets of the hypothesis' sector and layer inside the road, past the inclination
// veto and the chi2 cut [R2,R3,R4,R8,R13]
void find_candidates(const Config& cfg, const Store& st, const Hyp& h, int layer, const Road& rd,
                     std::vector<Cand>& out, int* n_evals, double* margin, Counters* cnt) {
    out.clear();
    if (st.n_ia > 1 && (h.ia < 0 || h.ia >= st.n_ia)) return;                // a track of no known interaction
    const std::vector<Tracklet>& v = st.cell[((size_t)(st.by_ia ? h.ia : 0) * st.n_sectors + h.sector) * st.n_layers + layer];
    size_t lo = 0, hi = v.size();
    if (st.sorted) {
        const double wide = (rd.road_y + std::fabs(rd.tan_tilt) * rd.road_z + st.dx_max * std::fabs(rd.tanphi)) * (1.0 + kLoose);
        lo = std::lower_bound(v.begin(), v.end(), h.p[0] - wide,
                              [](const Tracklet& a, double val) { return a.y < val; }) - v.begin();
        hi = std::upper_bound(v.begin(), v.end(), h.p[0] + wide,
                              [](double val, const Tracklet& a) { return val < a.y; }) - v.begin();
    }
    const double veto = rd.veto;
    for (size_t k = lo; k < hi; ++k) {
        const Tracklet& tl = v[k];
        if (tl.ia != h.ia) continue;                                         // other interaction [R27]
        if (cnt) cnt->n_scanned++;
        const double ry = tl.y - (h.p[0] + tl.dx * rd.tanphi), rz = tl.z - (h.p[1] + tl.dx * rd.zslope);   // [R29]
        const double ryc = ry - rd.tan_tilt * rz;                            // y corrected with the extrapolated z
        const double da = std::fabs(tl.dydx - rd.tanphi);
        bool in_y = std::fabs(ryc) <= rd.road_y, in_z = std::fabs(rz) <= rd.road_z;
        bool pass = da <= veto;                                             // PAPER.md:60, 4 sigma [R8]
        const bool loose_y = std::fabs(ryc) <= rd.road_y * (1.0 + kLoose);
        const bool loose_z = std::fabs(rz) <= rd.road_z * (1.0 + kLoose);
        const bool loose_a = da <= veto * (1.0 + kLoose);
        if (loose_z && loose_a && note(margin, std::fabs(ryc), rd.road_y)) in_y = !in_y;
        if (loose_y && loose_a && note(margin, std::fabs(rz), rd.road_z)) in_z = !in_z;
        if (loose_y && loose_z && note(margin, da, veto)) pass = !pass;
        const double c2 = chi2_of(rd, ry, rz);                              // y and z only
        bool cut = c2 >= cfg.chi2_cut;                                      // per-layer cut [R4]
        if (loose_y && loose_z && loose_a && note(margin, c2, cfg.chi2_cut)) cut = !cut;
        if (!(in_y && in_z && pass)) continue;
        if (n_evals) (*n_evals)++;                                          // one "candidate evaluation"
        if (cnt) cnt->n_cand++;
        if (cnt && cnt->touched) cnt->touched[tl.index] = 1;              // distinct in-road tracklets (roofline bytes)
        if (cut) continue;
        out.push_back({tl.index, tl.y, tl.z, c2, tl.dx});
    }
}

struct Child {
    int parent;        // position of the parent in the current hypothesis list
    int tracklet;      // caller's index, or INT_MAX for the skip-child (sorts after tracklets) [R6]
    double y, z, score, chi2inc, dx;
};

struct TrackResult {
    Hyp best;
    int n_evals;
    double margin;
};

// relative gap between two neighbours of the sorted child list, (b - a) / |b| with a <= b: recorded as a margin like
// every other decision; returns true if a replay takes the two the other way round
inline bool rank_gap(double* margin, double a, double b) {
    const double m = (b - a) / std::max(std::fabs(b), 1e-300);
    if (margin && m < *margin) *margin = m;
    if (t_replay && m < t_replay->eps) {
        const int k = t_replay->n_seen++;
        if (k < t_replay->n_forced && k < kMaxDecisions) return t_replay->forced[k] != 0;
    }
    return false;
}

// one track through all layers; "only the best N_candidates
// hypotheses are propagated", Fig. 2
void match_track(const Config& cfg, const Store& st, const Hyp& seed, TrackResult& res, Counters* cnt) {
    std::vector<Hyp> hyps(1, seed), next;
    std::vector<Hyp> prop;
    std::vector<Child> children;
    std::vector<Cand> cands;
    res.n_evals = 0;
    res.margin = std::numeric_limits<double>::infinity();
    double* mg = &res.margin;
    for (int L = 0; L < cfg.n_layers; ++L) {
        children.clear();
        prop = hyps;                                        // propagated copies of the parents
        for (int ih = 0; ih < (int)hyps.size(); ++ih) {
            Hyp& h = prop[ih];
            if (h.alive) h.alive = propagate_to_layer(cfg, h, cfg.layer_x[L], mg, cnt);
            if (h.alive && has_material(cfg)) h.alive = apply_material(cfg, h, +1, mg);   // the slab in front of the plane [R32]
            if (h.alive) {
                const Road rd = make_road(cfg, h, L);
                if (cnt) cnt->n_road++;
                find_candidates(cfg, st, h, L, rd, cands, &res.n_evals, mg, cnt);
                for (const Cand& c : cands)
                    children.push_back({ih, c.index, c.y, c.z, h.score + c.chi2inc, c.chi2inc, c.dx});
            }
            children.push_back({ih, std::numeric_limits<int>::max(), 0.0, 0.0, h.score + cfg.chi2_penalty, 0.0, 0.0});
        }
        std::stable_sort(children.begin(), children.end(), [](const Child& a, const Child& b) {
            if (a.score != b.score) return a.score < b.score;
            if (a.parent != b.parent) return a.parent < b.parent;
            return a.tracklet < b.tracklet;
        });
        const int keep = std::min<int>(cfg.n_hyp, (int)children.size());
        // ranking margins: the keep boundary at every layer, the winner at the last layer; a replay may take either of
        // two children whose scores are closer than eps
        if ((int)children.size() > keep) {
            const double a = children[keep - 1].score, b = children[keep].score;
            if (rank_gap(mg, a, b)) std::swap(children[keep - 1], children[keep]);
        }
        if (L == cfg.n_layers - 1 && children.size() > 1) {
            const double a = children[0].score, b = children[1].score;
            if (rank_gap(mg, a, b)) std::swap(children[0], children[1]);
        }
        next.clear();
        for (int k = 0; k < keep; ++k) {
            const Child& c = children[k];
            Hyp h = prop[c.parent];
            h.score = c.score;
            if (c.tracklet != std::numeric_limits<int>::max()) {
                if (c.dx != 0.0) {
                    // "again propagated ... to the exact radius" before the update [R30].  A track that
                    // cannot get there keeps its state at the nominal plane, attaches nothing and only skips from now on.
                    Hyp w = h;
                    if (!propagate(cfg, w, h.x + c.dx, mg, cnt)) {
                        h.alive = false;
                        next.push_back(h);
                        continue;
                    }
                    h = w;
                }
                const double chi2inc = kalman_update(cfg, h, L, c.y, c.z);
                if (c.dx != 0.0) h.score = prop[c.parent].score + chi2inc;   // the exact chi2 replaces the linear estimate
                if (cnt) cnt->n_upd++;
                h.chi2 += chi2inc;
                h.idx[L] = c.tracklet;
                h.n_matched++;
                const bool flip = note(mg, std::fabs(h.p[2]), cfg.max_snp);
                if ((std::fabs(h.p[2]) >= cfg.max_snp) != flip) h.alive = false;     // kept, but only skips from now on
            }
            next.push_back(h);
        }
        hyps.swap(next);
    }
    // With displaced chambers the scores of the kept children were replaced by the exact ones AFTER the ranking [R30],
    // so the list is no longer ordered by them: the output is the hypothesis with the lowest final score (the first of
    // equals).  Without offsets this is hyps[0] and the gap was already recorded at the last layer.
    size_t ib = 0;
    if (st.dx_max > 0.0 && hyps.size() > 1) {
        size_t i2 = 1;
        for (size_t k = 1; k < hyps.size(); ++k) {
            if (hyps[k].score < hyps[ib].score) { i2 = ib; ib = k; }
            else if (i2 == ib || hyps[k].score < hyps[i2].score) i2 = k;
        }
        if (rank_gap(mg, hyps[ib].score, hyps[i2].score)) ib = i2;
    }
    res.best = hyps[ib];
}

inline int tri(int i, int j) { return i * (i + 1) / 2 + j; }

void load_hyp(Hyp& h, const double p[5], const double c15[15], double x, int sector) {
    std::memset(&h, 0, sizeof h);
    for (int i = 0; i < 5; ++i) h.p[i] = p[i];
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j <= i; ++j) h.C[i][j] = h.C[j][i] = c15[tri(i, j)];
    h.x = x;
    h.sector = sector;
    for (int l = 0; l < kMaxLayers; ++l) h.idx[l] = -1;
    h.alive = true;
}

void store_cov(const Hyp& h, double c15[15]) {
    for (int i = 0; i < 5; ++i)
        for (int j = 0; j <= i; ++j) c15[tri(i, j)] = h.C[i][j];
}

}  // namespace

// =========================================================================================
// C entry points for the Python wrapper (oracle/oracle.py).  Own names, own struct layout.
// =========================================================================================
extern "C" {

typedef Config orc_config;

int orc_sizeof_config(void) { return (int)sizeof(Config); }

// in-frame propagation of state + 15-element covariance; F25 (row-major 5x5) optional
int orc_propagate(const orc_config* cfg, double p[5], double c15[15], double* x, double x_new, double* F25) {
    Hyp h;
    load_hyp(h, p, c15, *x, 0);
    double out[5], F[5][5];
    if (!propagate_state(*cfg, h.p, h.x, x_new, out, F, nullptr)) return 0;
    if (F25) std::memcpy(F25, F, sizeof F);
    if (!propagate(*cfg, h, x_new, nullptr, nullptr)) return 0;
    std::memcpy(p, h.p, sizeof h.p);
    store_cov(h, c15);
    *x = h.x;
    return 1;
}

int orc_rotate(const orc_config* cfg, double p[5], double c15[15], double* x, double beta, double* J25) {
    Hyp h;
    load_hyp(h, p, c15, *x, 0);
    double out[5], J[5][5], xn;
    if (!rotate_state(*cfg, h.p, h.x, beta, out, &xn, J, nullptr)) return 0;
    if (J25) std::memcpy(J25, J, sizeof J);
    if (!rotate(*cfg, h, beta, nullptr, nullptr)) return 0;
    std::memcpy(p, h.p, sizeof h.p);
    store_cov(h, c15);
    *x = h.x;
    return 1;
}

int orc_propagate_to_layer(const orc_config* cfg, double p[5], double c15[15], double* x, int32_t* sector, double X) {
    Hyp h;
    load_hyp(h, p, c15, *x, *sector);
    if (!propagate_to_layer(*cfg, h, X, nullptr, nullptr)) return 0;
    std::memcpy(p, h.p, sizeof h.p);
    store_cov(h, c15);
    *x = h.x;
    *sector = h.sector;
    return 1;
}

// one slab of material at the current point, dir = +1 outward / -1 inward; returns 0 if the particle stops
int orc_material(const orc_config* cfg, double p[5], double c15[15], int dir) {
    Hyp h;
    load_hyp(h, p, c15, 0.0, 0);
    if (!apply_material(*cfg, h, dir, nullptr)) return 0;
    std::memcpy(p, h.p, sizeof h.p);
    store_cov(h, c15);
    return 1;
}

// Kalman update with (ym, zm); returns the chi2 increment
double orc_update(const orc_config* cfg, double p[5], double c15[15], double ym, double zm, int layer) {
    Hyp h;
    load_hyp(h, p, c15, 0.0, 0);
    const double c2 = kalman_update(*cfg, h, layer, ym, zm);
    std::memcpy(p, h.p, sizeof h.p);
    store_cov(h, c15);
    return c2;
}

// road half-widths and tan(phi) of a state: out = (road_y, road_z, tanphi, Sinv00, Sinv01, Sinv11)
void orc_road(const orc_config* cfg, const double p[5], const double c15[15], double out[6], int layer) {
    Hyp h;
    load_hyp(h, p, c15, 0.0, 0);
    const Road rd = make_road(*cfg, h, layer);
    out[0] = rd.road_y; out[1] = rd.road_z; out[2] = rd.tanphi;
    out[3] = rd.Sinv[0][0]; out[4] = rd.Sinv[0][1]; out[5] = rd.Sinv[1][1];
}

// accepted candidates of one state at one layer; returns their number (<= cap written)
int orc_candidates(const orc_config* cfg, const float* y, const float* z, const float* dydx, const int32_t* chamber,
                   int64_t n, const double p[5], const double c15[15], int sector, int layer, int brute,
                   int32_t* out_index, double* out_chi2, int cap, const double* chamber_dx) {
    Store st;
    build_store(*cfg, y, z, dydx, chamber, nullptr, 1, chamber_dx, n, !brute, st);
    Hyp h;
    load_hyp(h, p, c15, cfg->layer_x[layer], sector);
    const Road rd = make_road(*cfg, h, layer);
    std::vector<Cand> cands;
    find_candidates(*cfg, st, h, layer, rd, cands, nullptr, nullptr, nullptr);
    std::sort(cands.begin(), cands.end(), [](const Cand& a, const Cand& b) { return a.index < b.index; });
    for (int k = 0; k < (int)cands.size() && k < cap; ++k) {
        out_index[k] = cands[k].index;
        out_chi2[k] = cands[k].chi2inc;
    }
    return (int)cands.size();
}

// the whole step for n_trk tracks (float32 inputs exactly as the CUDA path receives them).
// par: 5 x n_trk, cov: 15 x n_trk (SoA, row = component).  Outputs are double / int32 SoA:
// out_idx 6 x n_trk, out_par 5 x n_trk, out_cov 15 x n_trk.  brute != 0 ignores the sorted
// index and loops over all tracklets of the (sector, layer).  counters: n_prop, n_rot,
// n_road, n_cand, n_upd, n_scanned.  seconds: index build, matching.  out_touched (optional, n_tl bytes, zeroed by the
// caller): set to 1 for every tracklet that was inside the road of some hypothesis of some track.
int orc_match(const orc_config* cfg, const float* tl_y, const float* tl_z, const float* tl_dydx,
              const int32_t* tl_chamber, int64_t n_tl, const float* par, const float* cov, const float* x,
              const int32_t* sector, int64_t n_trk, int brute, int n_threads, int32_t* out_idx, double* out_par,
              double* out_cov, double* out_x, int32_t* out_sector, double* out_chi2, int32_t* out_n_matched,
              int32_t* out_n_evals, double* out_margin, int64_t counters[6], double seconds[2],
              const int32_t* tl_ia, const int32_t* trk_ia, int32_t n_ia, const double* chamber_dx,
              unsigned char* out_touched) {
    if (cfg->n_layers > kMaxLayers || cfg->n_hyp < 1) return -1;
    if ((tl_ia == nullptr) != (trk_ia == nullptr)) return -2;
    const auto t0 = std::chrono::steady_clock::now();
    Store st;
    build_store(*cfg, tl_y, tl_z, tl_dydx, tl_chamber, tl_ia, n_ia, chamber_dx, n_tl, !brute, st);
    const auto t1 = std::chrono::steady_clock::now();
    Counters total;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel
    {
        Counters local;
        local.touched = out_touched;                  // every thread only ever stores 1: no race that matters
#pragma omp for schedule(dynamic, 256)
        for (int64_t i = 0; i < n_trk; ++i) {
            double p[5], c15[15];
            for (int k = 0; k < 5; ++k) p[k] = par[k * n_trk + i];
            for (int k = 0; k < 15; ++k) c15[k] = cov[k * n_trk + i];
            Hyp seed;
            load_hyp(seed, p, c15, x[i], sector[i]);
            seed.ia = (st.n_ia > 1) ? trk_ia[i] : 0;
            seed.alive = std::fabs(p[2]) < cfg->max_snp && sector[i] >= 0 && sector[i] < cfg->n_sectors;
            TrackResult res;
            match_track(*cfg, st, seed, res, &local);
            const Hyp& b = res.best;
            for (int l = 0; l < kMaxLayers; ++l) out_idx[l * n_trk + i] = (l < cfg->n_layers) ? b.idx[l] : -1;
            for (int k = 0; k < 5; ++k) out_par[k * n_trk + i] = b.p[k];
            store_cov(b, c15);
            for (int k = 0; k < 15; ++k) out_cov[k * n_trk + i] = c15[k];
            out_x[i] = b.x;
            out_sector[i] = b.sector;
            out_chi2[i] = b.chi2;
            out_n_matched[i] = b.n_matched;
            if (out_n_evals) out_n_evals[i] = res.n_evals;
            if (out_margin) out_margin[i] = res.margin;
        }
#pragma omp critical
        {
            total.n_prop += local.n_prop; total.n_rot += local.n_rot; total.n_road += local.n_road;
            total.n_cand += local.n_cand; total.n_upd += local.n_upd; total.n_scanned += local.n_scanned;
        }
    }
    const auto t2 = std::chrono::steady_clock::now();
    if (counters) {
        counters[0] = total.n_prop; counters[1] = total.n_rot; counters[2] = total.n_road;
        counters[3] = total.n_cand; counters[4] = total.n_upd; counters[5] = total.n_scanned;
    }
    if (seconds) {
        seconds[0] = std::chrono::duration<double>(t1 - t0).count();
        seconds[1] = std::chrono::duration<double>(t2 - t1).count();
    }
    return 0;
}

// ---- "several results are correct": is a given chain one of them? ---------------------------
// For each of the n_sel tracks sel[k] (positions in the track arrays) the target chain target_idx[l * n_sel + k] (what
// another implementation attached) is looked for among the results this algorithm reaches when decisions closer than eps
// (relative) to their threshold -- road edges, chi2 cut, inclination veto, sector edge, max_snp, a stopping particle,
// the rank gaps at the keep boundary of every layer and between the two best chains at the end -- are taken either way.
// The search replays the track with one more fragile decision flipped at a time (breadth first: the natural run, every
// single flip, every pair, ...; every set visited once), until the chain appears or max_runs replays are spent.  out_found[k] = the
// number of replays it took (1 = the natural result is the target), or minus the number spent if it never appeared.  The
// other outputs hold the result of the replay that reached the target (of the natural run if none did), n_sel columns.
namespace {

bool same_chain(const Config& cfg, const Hyp& h, const int32_t* target, int64_t stride, int64_t k) {
    for (int l = 0; l < cfg.n_layers; ++l)
        if (h.idx[l] != target[l * stride + k]) return false;
    return true;
}

bool search_alternatives(const Config& cfg, const Store& st, const Hyp& seed, const int32_t* target, int64_t stride, int64_t k,
                         double eps, int& runs, int max_runs, TrackResult& res) {
    // breadth first over the sets of flipped decisions: the natural run, then every single flip, then pairs, ...  A
    // replay with the decisions d0 < d1 < ... flipped meets the same decisions up to its last flip as its parent did,
    // so its children flip one more decision met after that one: every set is visited once.
    std::deque<Replay> queue;
    Replay root;
    root.eps = eps;
    queue.push_back(root);
    while (!queue.empty() && runs < max_runs) {
        Replay rp = queue.front();
        queue.pop_front();
        rp.n_seen = 0;
        t_replay = &rp;
        match_track(cfg, st, seed, res, nullptr);
        t_replay = nullptr;
        ++runs;
        if (same_chain(cfg, res.best, target, stride, k)) return true;
        const int n_seen = std::min(rp.n_seen, kMaxDecisions);
        for (int d = rp.n_forced; d < n_seen && (int)queue.size() < max_runs; ++d) {
            Replay child = rp;
            for (int q = rp.n_forced; q < d; ++q) child.forced[q] = 0;
            child.forced[d] = 1;
            child.n_forced = d + 1;
            queue.push_back(child);
        }
    }
    return false;
}

}  // namespace

int orc_match_alternatives(const orc_config* cfg, const float* tl_y, const float* tl_z, const float* tl_dydx,
                           const int32_t* tl_chamber, int64_t n_tl, const float* par, const float* cov, const float* x,
                           const int32_t* sector, int64_t n_trk, const int64_t* sel, int64_t n_sel, const int32_t* target_idx,
                           double eps, int max_runs, int32_t* out_found, int32_t* out_idx, double* out_par, double* out_cov,
                           double* out_x, int32_t* out_sector, double* out_chi2, int32_t* out_n_matched, int32_t* out_n_evals,
                           const int32_t* tl_ia, const int32_t* trk_ia, int32_t n_ia, const double* chamber_dx) {
    if (cfg->n_layers > kMaxLayers || cfg->n_hyp < 1) return -1;
    if ((tl_ia == nullptr) != (trk_ia == nullptr)) return -2;
    Store st;
    build_store(*cfg, tl_y, tl_z, tl_dydx, tl_chamber, tl_ia, n_ia, chamber_dx, n_tl, true, st);
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n_sel; ++k) {
        const int64_t i = sel[k];
        double p[5], c15[15];
        for (int q = 0; q < 5; ++q) p[q] = par[q * n_trk + i];
        for (int q = 0; q < 15; ++q) c15[q] = cov[q * n_trk + i];
        Hyp seed;
        load_hyp(seed, p, c15, x[i], sector[i]);
        seed.ia = (st.n_ia > 1) ? trk_ia[i] : 0;
        seed.alive = std::fabs(p[2]) < cfg->max_snp && sector[i] >= 0 && sector[i] < cfg->n_sectors;
        TrackResult res;
        int runs = 0;
        const bool found = search_alternatives(*cfg, st, seed, target_idx, n_sel, k, eps, runs, max_runs, res);
        if (!found) {                                            // report the natural result
            match_track(*cfg, st, seed, res, nullptr);
        }
        out_found[k] = found ? runs : -runs;
        const Hyp& b = res.best;
        for (int l = 0; l < kMaxLayers; ++l) out_idx[l * n_sel + k] = (l < cfg->n_layers) ? b.idx[l] : -1;
        for (int q = 0; q < 5; ++q) out_par[q * n_sel + k] = b.p[q];
        store_cov(b, c15);
        for (int q = 0; q < 15; ++q) out_cov[q * n_sel + k] = c15[q];
        out_x[k] = b.x;
        out_sector[k] = b.sector;
        out_chi2[k] = b.chi2;
        out_n_matched[k] = b.n_matched;
        out_n_evals[k] = res.n_evals;
    }
    return 0;
}

// TRD-only refit of the matched chains (calibration step 3: "refits ... ignoring the TPC clusters";
// PAPER.md:9) [R31].  For every track with at least min_tracklets attached tracklets (two): start from the
// matched final state, reset the covariance to diag(refit_var) so that nothing of the seed's (TPC) information
// enters, run the Kalman filter INWARD over the attached tracklets only (propagation to each tracklet's plane with
// the sector rule of the matcher, update with the measurement model of the matcher), then propagate to x_ref.
// in_*: the matcher's outputs (double, SoA).  out_n_used < min_tracklets marks a track that was not refitted
// (state copied through).  A tracklet whose chamber is not in the state's sector frame is skipped.
int orc_refit(const orc_config* cfg, const float* tl_y, const float* tl_z, const int32_t* tl_chamber, int64_t n_tl,
              const double* chamber_dx, const int32_t* in_idx, const double* in_par, const double* in_cov, const double* in_x,
              const int32_t* in_sector, int64_t n_trk, int min_tracklets, double* out_par, double* out_cov, double* out_x,
              int32_t* out_sector, double* out_chi2, int32_t* out_n_used) {
    const int per_sector = cfg->n_stacks * cfg->n_layers;
    for (int64_t i = 0; i < n_trk; ++i) {
        double p[5], c15[15];
        for (int k = 0; k < 5; ++k) p[k] = in_par[k * n_trk + i];
        for (int k = 0; k < 15; ++k) c15[k] = in_cov[k * n_trk + i];
        Hyp h;
        load_hyp(h, p, c15, in_x[i], in_sector[i]);
        int n_att = 0;
        for (int l = 0; l < cfg->n_layers; ++l) n_att += in_idx[l * n_trk + i] >= 0;
        int n_used = 0;
        double chi2 = 0.0;
        bool ok = n_att >= min_tracklets && std::fabs(p[2]) < cfg->max_snp;
        if (ok) {
            for (int a = 0; a < 5; ++a)
                for (int b = 0; b < 5; ++b) h.C[a][b] = (a == b) ? cfg->refit_var[a] : 0.0;
            // With material [R34] every layer plane from the outermost attached tracklet inward is a stop: the plane of
            // the attached tracklet (exact radius) or the nominal one, then the slab in front of it is crossed inward
            // (noise added, mean energy loss given back) before the next step.  Slabs outside the outermost attached
            // tracklet are not applied: the covariance is reset there anyway.
            const bool mat = has_material(*cfg);
            bool started = false;
            for (int l = cfg->n_layers - 1; l >= 0 && ok; --l) {
                const int k = in_idx[l * n_trk + i];
                const bool att = k >= 0 && k < n_tl;
                if (!att && !(mat && started)) continue;
                const int ch = att ? tl_chamber[k] : 0;
                const double X = cfg->layer_x[l] + ((att && chamber_dx) ? chamber_dx[ch] : 0.0);
                if (h.x != X) ok = propagate_to_layer(*cfg, h, X, nullptr, nullptr);
                if (!ok) break;
                if (att && ch / per_sector == h.sector) {            // attached in another frame: not used
                    chi2 += kalman_update(*cfg, h, l, (double)tl_y[k], (double)tl_z[k]);
                    ++n_used;
                    if (std::fabs(h.p[2]) >= cfg->max_snp) ok = false;
                }
                if (att) started = true;
                if (ok && mat) ok = apply_material(*cfg, h, -1, nullptr);
            }
            if (ok) ok = propagate_to_layer(*cfg, h, cfg->x_ref, nullptr, nullptr);
        }
        if (!ok) {                                                   // not refitted: the matcher's state goes through
            load_hyp(h, p, c15, in_x[i], in_sector[i]);
            n_used = 0;
            chi2 = 0.0;
        }
        for (int k = 0; k < 5; ++k) out_par[k * n_trk + i] = h.p[k];
        store_cov(h, c15);
        for (int k = 0; k < 15; ++k) out_cov[k * n_trk + i] = c15[k];
        out_x[i] = h.x;
        out_sector[i] = h.sector;
        out_chi2[i] = chi2;
        out_n_used[i] = n_used;
    }
    return 0;
}

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"
