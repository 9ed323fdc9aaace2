"""Seeded synthetic inputs for the online TRD tracking step (§3).

This module serves BOTH the oracle's tests and the CUDA path's tests / bench.  It
holds none of the method's arithmetic: no Kalman filter, no road, no chi2, no
propagation Jacobian.  All it computes is where a *true* particle crosses the TRD
planes, from the global circle through the origin (an independent derivation of
the helix, see `_truth_at_plane`), plus the smearing and noise the configs of
BASELINE.json describe.  The paper measured on ALICE Monte-Carlo and 2018 HLT data
(PAPER.md:74, 80, 94); those are not available, so these inputs stand in for them
with the paper's shapes: 18 sectors x 5 stacks x 6 layers, ~2000-5000
tracks per central event, time frames of 500-1000 collisions
(PAPER.md:86, 90), >= 450k tracks per map.

Recipe (every draw in float64, cast to float32 once at the end):
  rng      numpy.random.Generator(PCG64(seed)), seed = 317400 + config number (1..5)
  particle q = +-1, pT log-uniform [0.5, 20] GeV/c (config 4: 0.3 + Exp(0.5)),
           eta uniform (-0.8, 0.8), tan(lambda) = sinh(eta), phi0 uniform [0, 2pi),
           vertex at the origin
  seed     true state where the helix crosses local x = 247 cm in the sector whose
           |y| <= 247 tan(10 deg), smeared by N(0, diag(0.1, 0.1, 1e-3, 1e-3,
           0.01 |q/pT|)^2); covariance = that diagonal
  signal   per layer, with probability 0.9 and if |z| < 350 and |sin(phi)| < 0.95:
           y + N(0, 0.04), z -> pad-row centre (8 cm rows), dy/dx = tan(phi) + N(0, 0.02)
  noise    chamber uniform 0..539, y uniform in the chamber, z a uniform pad-row
           centre of that stack, dy/dx uniform [-0.5, 0.5]
  order    tracklets = signal ++ noise, then one seeded permutation
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, Optional

import numpy as np

# ---- geometry of the configs (BASELINE.json configs[0]) ---------------------------------
N_SECTORS = 18
N_STACKS = 5
N_LAYERS = 6
LAYER_X = (300.0, 313.0, 326.0, 338.0, 351.0, 364.0)
X_SEED = 247.0
Z_MAX = 350.0
PAD_LENGTH = 8.0
SECTOR_WIDTH = 2.0 * math.pi / N_SECTORS          # 20 degrees
TAN_HALF_SECTOR = math.tan(0.5 * SECTOR_WIDTH)    # tan(10 degrees)
KAPPA_PER_TESLA = -0.00299792458                  # curvature [1/cm] = this * Bz[T] * q/pT[c/GeV]
N_ROWS = int(round(2 * (Z_MAX + 2.0) / PAD_LENGTH))  # 88 global pad rows, centres -348..+348

SIGMA_SEED = (0.1, 0.1, 1e-3, 1e-3)               # y, z, sin(phi), tan(lambda); q/pT is relative
REL_SIGMA_QPT = 0.01
SIGMA_Y_TRACKLET = 0.04
SIGMA_DYDX_TRACKLET = 0.02
EFFICIENCY = 0.9
MAX_SNP = 0.95
NOISE_DYDX_RANGE = 0.5

# Resolution model of PAPER.md:62 / Fig. 3 (image not available: the coefficients below are this build's synthetic
# choice, R24) and pad tilt of PAPER.md:66 (R25).  sigma(s) = c0 + c2 (s - sin(Lorentz angle))^2.
SY_C0, SY_C2 = 0.03, 0.12            # cm: 0.03 at the optimum, 0.06 at |s - sL| = 0.5
SD_C0, SD_C2 = 0.015, 0.06           # dy/dx: "below 1 degree" at the optimum
LORENTZ_DEG = 8.0
TILT_DEG = 2.0

# Material of PAPER.md:64 (the ALICE material budget is not available: synthetic, R32/R33).  One slab in
# front of every layer plane; the values used by the material workloads:
PION_MASS = 0.13957                  # GeV
X_OVER_X0 = 0.04                     # radiation lengths per layer at normal incidence
ELOSS = 1.5e-3                       # GeV per layer at normal incidence and beta = 1
ELOSS_FLUCT = 0.3                    # relative width of the energy-loss fluctuation
HIGHLAND = 0.0136                    # GeV: theta0 = HIGHLAND / (beta p) sqrt(x/X0)

# Field inhomogeneity of PAPER.md:64 (the ALICE field map is not available: synthetic, R35):
# Bz(r, z) = Bz (1 + BZ_R2 r^2 + BZ_Z2 z^2), r, z in cm
BZ_R2 = -1.5e-7                      # -2 % at r = 364 cm
BZ_Z2 = -1.0e-7                      # -1.2 % at |z| = 350 cm


@dataclasses.dataclass(frozen=True)
class WorkloadSpec:
    """One of the five BASELINE.json configs (or a scaled / special variant of one)."""
    name: str
    number: int                 # 1..5; seed = 317400 + number
    n_tracks: int
    n_noise: int
    n_hyp: int
    n_sigma_road: float
    pt_spectrum: str = "loguniform"   # or "exp"
    batch: Optional[int] = None       # tracks per trd_match call (config 5: 500k)
    bz: float = 0.5
    # switches used by the oracle's pins (exact-recovery and pull tests)
    smear_seed: bool = True
    smear_tracklets: bool = True
    exact_z: bool = False             # tracklet z = true z instead of the pad-row centre
    efficiency: float = EFFICIENCY
    res_model: int = 0                # 1: sigma_y(sin phi), sigma_dydx(sin phi) polynomials and +-2 degree pad tilt
    chamber_dx_sigma: float = 0.0     # > 0: radial chamber misalignment N(0, sigma) cm, clipped at 3 sigma
    x_over_x0: float = 0.0            # > 0: a slab of that many radiation lengths in front of every layer:
    eloss: float = 0.0                # the true particle is scattered there and loses eloss * path / beta^2 GeV
    eloss_fluct: float = 0.0          # (Gaussian fluctuation of that relative width)
    bz_r2: float = 0.0                # != 0: the true particle moves in Bz (1 + bz_r2 r^2 + bz_z2 z^2), integrated numerically
    bz_z2: float = 0.0
    n_interactions: int = 0           # > 1: time-frame association: tracks i*n_ia//n_tracks form one
                                      # collision, their tracklets inherit its id, noise tracklets get a random one

    @property
    def seed(self) -> int:
        return 317400 + self.number


CONFIGS: Dict[str, WorkloadSpec] = {
    "tiny": WorkloadSpec("tiny", 1, 1_000, 2_000, 1, 3.0),
    "central": WorkloadSpec("central", 2, 5_000, 20_000, 1, 3.0),
    "central8": WorkloadSpec("central8", 3, 5_000, 20_000, 8, 5.0),
    "pileup": WorkloadSpec("pileup", 4, 25_000, 100_000, 4, 3.0, pt_spectrum="exp"),
    "timeframe": WorkloadSpec("timeframe", 5, 2_000_000, 8_000_000, 4, 3.0, batch=500_000),
}


def scaled(spec: WorkloadSpec, n_tracks: int, name: Optional[str] = None) -> WorkloadSpec:
    """Same generator, density per chamber preserved: noise scales with the track count."""
    f = n_tracks / spec.n_tracks
    return dataclasses.replace(spec, name=name or f"{spec.name}_x{n_tracks}", n_tracks=n_tracks,
                               n_noise=int(round(spec.n_noise * f)),
                               batch=None if spec.batch is None else min(spec.batch, n_tracks))


def sin_lorentz(bz: float) -> float:
    """sin of the Lorentz angle; its sign follows the field polarity ("+-8 degrees")."""
    return math.copysign(math.sin(math.radians(LORENTZ_DEG)), bz) if bz != 0.0 else 0.0


def matcher_config(spec: WorkloadSpec) -> dict:
    """The cuts and geometry of a config as a plain dict (field names of include/trdmatch.h).

    Both the oracle wrapper and the CUDA binding turn this dict into their own struct.
    """
    extra = {}
    if spec.res_model:
        extra = dict(res_model=1, sy_c0=SY_C0, sy_c2=SY_C2, sd_c0=SD_C0, sd_c2=SD_C2,
                     sin_lorentz=sin_lorentz(spec.bz), tan_tilt=math.tan(math.radians(TILT_DEG)))
    if spec.x_over_x0 > 0.0 or spec.eloss > 0.0:
        extra.update(x_over_x0=spec.x_over_x0, eloss=spec.eloss, eloss_fluct=spec.eloss_fluct, mass=PION_MASS)
    if spec.bz_r2 != 0.0 or spec.bz_z2 != 0.0:
        extra.update(bz_r2=spec.bz_r2, bz_z2=spec.bz_z2)
    return dict(extra,
        n_sectors=N_SECTORS, n_stacks=N_STACKS, n_layers=N_LAYERS,
        layer_x=list(LAYER_X), z_max=Z_MAX, pad_length=PAD_LENGTH, bz_tesla=spec.bz,
        sigma_y=SIGMA_Y_TRACKLET, sigma_z=PAD_LENGTH / math.sqrt(12.0),
        sigma_dydx=SIGMA_DYDX_TRACKLET, n_sigma_road=spec.n_sigma_road, n_sigma_angle=4.0,
        chi2_cut=15.0, chi2_penalty=15.0, max_snp=MAX_SNP, n_hyp=spec.n_hyp, ybin_width=0.0,
    )


# ---- pad rows and stacks (SURVEY.md §8(c).5 reading 12) ----------------------------------
def pad_row_centre(z):
    return PAD_LENGTH * (np.floor(np.asarray(z) / PAD_LENGTH) + 0.5)


def stack_of_z(zc):
    """Stack 0..4 of a pad-row centre: five equal 140 cm slices of [-350, 350]."""
    width = 2.0 * Z_MAX / N_STACKS
    return np.clip(np.floor((np.asarray(zc) + Z_MAX) / width), 0, N_STACKS - 1).astype(np.int64)


def _rows_by_stack():
    centres = PAD_LENGTH * (np.arange(N_ROWS) - N_ROWS // 2 + 0.5)
    st = stack_of_z(centres)
    return [centres[st == k] for k in range(N_STACKS)]


# ---- truth: the global circle through the origin ----------------------------------------
def _truth_at_plane(phi0, kappa, tanl, x_plane):
    """Where the true particle first crosses the plane local-x = x_plane of its sector.

    The particle leaves the origin with azimuth phi0; its xy projection is the circle of
    signed curvature kappa (d(azimuth)/d(path) = kappa) through the origin, centre at
    (-sin(phi0), cos(phi0))/kappa.  In a frame rotated by alpha the direction at the origin
    is phi0 - alpha and the plane x' = X is met where sin(phi') = sin(phi0 - alpha) + kappa X
    (chord of the circle), at y' = (cos(phi0 - alpha) - cos(phi'))/kappa after an arc of
    length (phi' - (phi0 - alpha))/kappa.  The sector is the one whose |y'| <= X tan(10 deg).

    Returns sector, y, z, sin(phi), ok  (ok = False where the circle does not reach).
    """
    n = phi0.shape[0]
    # azimuth of the point of the circle at distance X/cos(.) ~ X from the origin: phi0 + asin(kappa rho / 2)
    arg = np.clip(0.5 * kappa * x_plane, -1.0, 1.0)
    az = np.mod(phi0 + np.arcsin(arg), 2.0 * np.pi)
    guess = np.floor(az / SECTOR_WIDTH).astype(np.int64)
    best = dict(sec=np.zeros(n, np.int64), y=np.full(n, np.nan), z=np.full(n, np.nan),
                s=np.full(n, np.nan), ok=np.zeros(n, bool))
    edge = x_plane * TAN_HALF_SECTOR
    for d in (0, -1, 1):
        sec = np.mod(guess + d, N_SECTORS)
        alpha = (sec + 0.5) * SECTOR_WIDTH
        ploc = np.mod(phi0 - alpha + np.pi, 2.0 * np.pi) - np.pi       # direction at the origin, local
        s0 = np.sin(ploc)
        c0 = np.cos(ploc)
        s1 = s0 + kappa * x_plane
        reach = (np.abs(s1) < 1.0) & (c0 > 0.0)
        s1c = np.where(reach, s1, 0.0)
        c1 = np.sqrt(1.0 - s1c * s1c)
        straight = np.abs(kappa) < 1e-12
        ksafe = np.where(straight, 1.0, kappa)
        y = np.where(straight, x_plane * s0 / np.where(c0 > 0, c0, 1.0), (c0 - c1) / ksafe)
        arc = np.where(straight, x_plane / np.where(c0 > 0, c0, 1.0), (np.arcsin(s1c) - ploc) / ksafe)
        z = tanl * arc
        take = reach & (np.abs(y) <= edge) & ~best["ok"]
        best["sec"] = np.where(take, sec, best["sec"])
        best["y"] = np.where(take, y, best["y"])
        best["z"] = np.where(take, z, best["z"])
        best["s"] = np.where(take, s1, best["s"])
        best["ok"] |= take
    return best["sec"], best["y"], best["z"], best["s"], best["ok"]


def _truth_in_sector(phi0, kappa, tanl, x_plane, sec):
    """(y, z, sin(phi), ok) where the particle crosses the plane local-x = x_plane (array) of the GIVEN sector:
    same circle as _truth_at_plane, no sector search and no edge test (used for radially displaced chambers)."""
    alpha = (sec + 0.5) * SECTOR_WIDTH
    ploc = np.mod(phi0 - alpha + np.pi, 2.0 * np.pi) - np.pi
    s0, c0 = np.sin(ploc), np.cos(ploc)
    s1 = s0 + kappa * x_plane
    ok = (np.abs(s1) < 1.0) & (c0 > 0.0)
    s1c = np.where(ok, s1, 0.0)
    c1 = np.sqrt(1.0 - s1c * s1c)
    straight = np.abs(kappa) < 1e-12
    ksafe = np.where(straight, 1.0, kappa)
    c0s = np.where(c0 > 0, c0, 1.0)
    y = np.where(straight, x_plane * s0 / c0s, (c0 - c1) / ksafe)
    arc = np.where(straight, x_plane / c0s, (np.arcsin(s1c) - ploc) / ksafe)
    return y, tanl * arc, s1, ok


def _cross_from(gx, gy, gz, psi, kappa, tanl, x_plane, sec):
    """Crossing of the plane local-x = x_plane of sector `sec` by the helix that passes the GLOBAL point (gx, gy, gz)
    with global azimuth psi, signed curvature kappa and tan(lambda) = tanl: the chord relation of _truth_at_plane
    written from an arbitrary start point.  Returns y, z, sin(phi) (local), ok."""
    alpha = (sec + 0.5) * SECTOR_WIDTH
    ca, sa = np.cos(alpha), np.sin(alpha)
    x0 = gx * ca + gy * sa
    y0 = -gx * sa + gy * ca
    ploc = np.mod(psi - alpha + np.pi, 2.0 * np.pi) - np.pi
    s0, c0 = np.sin(ploc), np.cos(ploc)
    d = x_plane - x0
    s1 = s0 + kappa * d
    ok = (np.abs(s1) < 1.0) & (c0 > 0.0)
    s1c = np.where(ok, s1, 0.0)
    c1 = np.sqrt(1.0 - s1c * s1c)
    straight = np.abs(kappa) < 1e-12
    ksafe = np.where(straight, 1.0, kappa)
    c0s = np.where(c0 > 0, c0, 1.0)
    y = y0 + np.where(straight, d * s0 / c0s, (c0 - c1) / ksafe)
    arc = np.where(straight, d / c0s, (np.arcsin(s1c) - ploc) / ksafe)
    return y, gz + tanl * arc, s1, ok


def _cross_with_sector_search(gx, gy, gz, psi, kappa, tanl, x_plane):
    """_cross_from in the sector whose |y| <= x_plane tan(10 deg): the sector of the start point's azimuth (of the
    direction, at the origin) and its two neighbours are tried.  Returns sector, y, z, sin(phi), ok."""
    n = gx.shape[0]
    at_origin = (gx == 0.0) & (gy == 0.0)
    az = np.where(at_origin, psi + np.arcsin(np.clip(0.5 * kappa * x_plane, -1.0, 1.0)), np.arctan2(gy, gx))
    guess = np.floor(np.mod(az, 2.0 * np.pi) / SECTOR_WIDTH).astype(np.int64)
    out = dict(sec=np.zeros(n, np.int64), y=np.full(n, np.nan), z=np.full(n, np.nan), s=np.full(n, np.nan),
               ok=np.zeros(n, bool))
    edge = x_plane * TAN_HALF_SECTOR
    for d in (0, -1, 1):
        sec = np.mod(guess + d, N_SECTORS)
        y, z, s1, reach = _cross_from(gx, gy, gz, psi, kappa, tanl, x_plane, sec)
        take = reach & (np.abs(y) <= edge) & ~out["ok"]
        for k, v in (("sec", sec), ("y", y), ("z", z), ("s", s1)):
            out[k] = np.where(take, v, out[k])
        out["ok"] |= take
    return out["sec"], out["y"], out["z"], out["s"], out["ok"]


def _rk4_path(spec, kfac, gx, gy, gz, psi, qpt, tanl, path, n_sub):
    """Equations of motion in the field Bz(r, z) = Bz (1 + bz_r2 r^2 + bz_z2 z^2), independent variable the xy path
    length u:  dX/du = cos(psi), dY/du = sin(psi), dZ/du = tan(lambda), dpsi/du = kfac q/pT (1 + bz_r2 (X^2 + Y^2) +
    bz_z2 Z^2).  Classical Runge-Kutta over `path` (array, per particle) in n_sub equal steps."""
    def rhs(X, Y, Z, P):
        return np.cos(P), np.sin(P), tanl, kfac * qpt * (1.0 + spec.bz_r2 * (X * X + Y * Y) + spec.bz_z2 * Z * Z)
    h = path / n_sub
    X, Y, Z, P = gx.copy(), gy.copy(), gz.copy(), psi.copy()
    for _ in range(n_sub):
        a = rhs(X, Y, Z, P)
        b = rhs(X + 0.5 * h * a[0], Y + 0.5 * h * a[1], Z + 0.5 * h * a[2], P + 0.5 * h * a[3])
        c = rhs(X + 0.5 * h * b[0], Y + 0.5 * h * b[1], Z + 0.5 * h * b[2], P + 0.5 * h * b[3])
        d = rhs(X + h * c[0], Y + h * c[1], Z + h * c[2], P + h * c[3])
        X = X + h / 6.0 * (a[0] + 2.0 * b[0] + 2.0 * c[0] + d[0])
        Y = Y + h / 6.0 * (a[1] + 2.0 * b[1] + 2.0 * c[1] + d[1])
        Z = Z + h / 6.0 * (a[2] + 2.0 * b[2] + 2.0 * c[2] + d[2])
        P = P + h / 6.0 * (a[3] + 2.0 * b[3] + 2.0 * c[3] + d[3])
    return X, Y, Z, P


def _cross_rk4(spec, kfac, gx, gy, gz, psi, qpt, tanl, x_plane, sec, n_sub):
    """Like _cross_from, in the inhomogeneous field: the path length to the plane is found by Newton's method
    (start: the uniform-field helix), each trial integrated from the start point with _rk4_path."""
    alpha = (sec + 0.5) * SECTOR_WIDTH
    ca, sa = np.cos(alpha), np.sin(alpha)
    x0 = gx * ca + gy * sa
    ploc = np.mod(psi - alpha + np.pi, 2.0 * np.pi) - np.pi
    kappa = kfac * qpt
    s0 = np.sin(ploc)
    s1 = s0 + kappa * (x_plane - x0)
    ok = (np.abs(s1) < 1.0) & (np.cos(ploc) > 0.0)
    s1c = np.where(ok, s1, s0)
    straight = np.abs(kappa) < 1e-12
    path = np.where(straight, (x_plane - x0) / np.where(ok, np.cos(ploc), 1.0),
                    (np.arcsin(s1c) - np.arcsin(np.clip(s0, -1, 1))) / np.where(straight, 1.0, kappa))
    path = np.where(ok, path, 0.0)
    for _ in range(4):
        X, Y, Z, P = _rk4_path(spec, kfac, gx, gy, gz, psi, qpt, tanl, path, n_sub)
        cl = np.cos(P - alpha)
        ok &= cl > 0.05
        path = path + np.where(ok, (x_plane - (X * ca + Y * sa)) / np.where(ok, cl, 1.0), 0.0)
    X, Y, Z, P = _rk4_path(spec, kfac, gx, gy, gz, psi, qpt, tanl, path, n_sub)
    ok &= np.abs(X * ca + Y * sa - x_plane) < 1e-9
    return -X * sa + Y * ca, Z, np.sin(P - alpha), ok


def _cross_rk4_search(spec, kfac, gx, gy, gz, psi, qpt, tanl, x_plane, n_sub):
    """_cross_rk4 in the sector whose |y| <= x_plane tan(10 deg): the sector found with the uniform-field helix
    first, its neighbour on the side of y where that fails."""
    sec, _, _, _, okh = _cross_with_sector_search(gx, gy, gz, psi, kfac * qpt, tanl, x_plane)
    y, z, s1, ok = _cross_rk4(spec, kfac, gx, gy, gz, psi, qpt, tanl, x_plane, sec, n_sub)
    edge = x_plane * TAN_HALF_SECTOR
    with np.errstate(invalid="ignore"):
        out = okh & ok & (np.abs(y) > edge)
    if out.any():
        i = np.nonzero(out)[0]
        sec2 = np.mod(sec[i] + np.where(y[i] > 0, 1, -1), N_SECTORS)
        y2, z2, s2, ok2 = _cross_rk4(spec, kfac, gx[i], gy[i], gz[i], psi[i], qpt[i], tanl[i], x_plane, sec2, n_sub)
        sec, y, z, s1, ok = sec.copy(), y.copy(), z.copy(), s1.copy(), ok.copy()
        sec[i], y[i], z[i], s1[i] = sec2, y2, z2, s2
        ok[i] = ok2 & (np.abs(y2) <= edge)
    return sec, y, z, s1, okh & ok


def chamber_offsets(spec: "WorkloadSpec") -> np.ndarray:
    """Radial offset of every chamber from its nominal layer plane (float32 cm), own seeded stream."""
    n_ch = N_SECTORS * N_STACKS * N_LAYERS
    if spec.chamber_dx_sigma <= 0.0:
        return np.zeros(n_ch, np.float32)
    rng = np.random.Generator(np.random.PCG64(spec.seed + 1_000_003))
    sig = spec.chamber_dx_sigma
    return np.clip(rng.normal(0.0, sig, n_ch), -3.0 * sig, 3.0 * sig).astype(np.float32)


def _draw_particles(rng, spec: WorkloadSpec, n: int):
    q = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    if spec.pt_spectrum == "loguniform":
        pt = np.exp(rng.uniform(math.log(0.5), math.log(20.0), n))
    elif spec.pt_spectrum == "exp":
        pt = 0.3 + rng.exponential(0.5, n)
    else:
        raise ValueError(spec.pt_spectrum)
    eta = rng.uniform(-0.8, 0.8, n)
    phi0 = rng.uniform(0.0, 2.0 * np.pi, n)
    return q, pt, np.sinh(eta), phi0


def generate(spec: WorkloadSpec) -> dict:
    """Build the inputs of one config.  Deterministic: same spec -> identical bytes.

    Returns a dict of numpy arrays:
      tracks:    par (5, n) f32, cov (15, n) f32 lower-triangular, x (n,) f32, sector (n,) i32
      tracklets: tl_y, tl_z, tl_dydx (m,) f32, tl_chamber (m,) i32, tl_label (m,) i32 (track id, -1 noise)
      truth:     truth_par (5, n) f64 at the seed plane, truth_idx (n, 6) i32 = index of the
                 track's own tracklet per layer in the permuted tracklet arrays (-1 = none),
                 truth_last (n, 4) f64 = true (y, z, sin(phi), sector) at layer 5 (nan if not reached)
    """
    rng = np.random.Generator(np.random.PCG64(spec.seed))
    n = spec.n_tracks
    kfac = KAPPA_PER_TESLA * spec.bz

    field = spec.bz_r2 != 0.0 or spec.bz_z2 != 0.0

    def from_origin(phi0_, qpt_, tanl_, x_plane):
        if not field:
            return _truth_at_plane(phi0_, kfac * qpt_, tanl_, x_plane)
        zero = np.zeros_like(phi0_)
        return _cross_rk4_search(spec, kfac, zero, zero, zero, phi0_, qpt_, tanl_, x_plane, 64)

    # 1. particles, redrawn in blocks of n until n of them reach x = 247 and layer 0 (draw order:
    #    q, pT, eta, phi0 per block)
    keep = {k: [] for k in ("q", "pt", "tanl", "phi0")}
    have = 0
    while have < n:
        q, pt, tanl, phi0 = _draw_particles(rng, spec, max(n, 64))
        kappa = kfac * q / pt
        _, _, _, s_seed, ok_seed = from_origin(phi0, q / pt, tanl, X_SEED)
        _, _, _, s_l0, ok_l0 = from_origin(phi0, q / pt, tanl, LAYER_X[0])
        good = ok_seed & ok_l0 & (np.abs(s_seed) < MAX_SNP) & (np.abs(s_l0) < MAX_SNP)
        for k, v in (("q", q), ("pt", pt), ("tanl", tanl), ("phi0", phi0)):
            keep[k].append(v[good])
        have += int(good.sum())
    q, pt, tanl, phi0 = (np.concatenate(keep[k])[:n] for k in ("q", "pt", "tanl", "phi0"))
    qpt = q / pt
    kappa = kfac * qpt

    # 2. seed state at x = 247 (+ smearing, draw order: 5 normals per track as one (n, 5) block)
    sec, y, z, s, ok = from_origin(phi0, qpt, tanl, X_SEED)
    assert ok.all()
    truth_par = np.stack([y, z, s, tanl, qpt])
    sig = np.stack([np.full(n, SIGMA_SEED[0]), np.full(n, SIGMA_SEED[1]), np.full(n, SIGMA_SEED[2]),
                    np.full(n, SIGMA_SEED[3]), REL_SIGMA_QPT * np.abs(qpt)])
    noise = rng.standard_normal((n, 5)).T
    par = truth_par + (sig * noise if spec.smear_seed else 0.0)
    cov = np.zeros((15, n))
    for i in range(5):
        cov[i * (i + 1) // 2 + i] = sig[i] ** 2

    # 3. signal tracklets, layer by layer (draw order per layer: efficiency u, y normal, dy/dx normal)
    sig_y, sig_z, sig_d, sig_ch, sig_lab, sig_lay = [], [], [], [], [], []
    truth_last = np.full((n, 4), np.nan)
    ch_dx = chamber_offsets(spec)
    material = spec.x_over_x0 > 0.0 or spec.eloss > 0.0
    stepped = material or field
    if stepped:
        # stepped truth: global point, azimuth, tan(lambda), q/pT after the last slab crossed (the origin at first)
        gx, gy, gz = np.zeros(n), np.zeros(n), np.zeros(n)
        psi, tl_now, qpt_now, going = phi0.copy(), tanl.copy(), qpt.copy(), np.ones(n, bool)
        truth_last_par = np.full((5, n), np.nan)
    for lay, xl in enumerate(LAYER_X):
        if stepped:
            # crossing of the nominal plane, then the slab: two scattering angles and the energy loss
            # (draw order per layer: k1, k2, ke, then the draws of the plain generator; no slab draws without material)
            if field:
                secl, yl, zl, sl, okl = _cross_rk4_search(spec, kfac, gx, gy, gz, psi, qpt_now, tl_now, xl, 64 if lay == 0 else 8)
            else:
                secl, yl, zl, sl, okl = _cross_with_sector_search(gx, gy, gz, psi, kfac * qpt_now, tl_now, xl)
            okl &= going
            if material:
                k1, k2, ke = rng.standard_normal(n), rng.standard_normal(n), rng.standard_normal(n)
            else:
                k1 = k2 = ke = 0.0
            with np.errstate(invalid="ignore"):
                sc = np.where(okl, sl, 0.0)
                path = np.sqrt((1.0 + tl_now ** 2) / (1.0 - sc * sc))
                mom = np.sqrt(1.0 + tl_now ** 2) / np.abs(qpt_now)
                en = np.sqrt(mom ** 2 + PION_MASS ** 2)
                beta = mom / en
                theta0 = HIGHLAND / (beta * mom) * np.sqrt(spec.x_over_x0 * path)
                lam = np.arctan(tl_now)
                alpha_l = (secl + 0.5) * SECTOR_WIDTH
                psi_new = alpha_l + np.arcsin(sc) + theta0 * k2 / np.cos(lam)
                lam_new = lam + theta0 * k1
                en_new = en - spec.eloss * path / beta ** 2 * (1.0 + spec.eloss_fluct * ke)
                okl &= en_new > PION_MASS
                mom_new = np.sqrt(np.where(okl, en_new ** 2 - PION_MASS ** 2, 1.0))
            ca, sa = np.cos(alpha_l), np.sin(alpha_l)
            yc, zc_ = np.where(okl, yl, 0.0), np.where(okl, zl, 0.0)
            gx, gy, gz = np.where(okl, xl * ca - yc * sa, gx), np.where(okl, xl * sa + yc * ca, gy), np.where(okl, zc_, gz)
            psi = np.where(okl, psi_new, psi)
            tl_now = np.where(okl, np.tan(lam_new), tl_now)
            qpt_now = np.where(okl, q / (mom_new * np.cos(lam_new)), qpt_now)
            going = okl
            sl = np.where(okl, np.sin(psi - alpha_l), np.nan)          # the chamber sees the direction after the slab
        else:
            secl, yl, zl, sl, okl = _truth_at_plane(phi0, kappa, tanl, xl)
        u = rng.random(n)
        ny = rng.standard_normal(n)
        nd = rng.standard_normal(n)
        with np.errstate(invalid="ignore"):
            present = okl & (np.abs(zl) < Z_MAX) & (np.abs(sl) < MAX_SNP) & (u < spec.efficiency)
        if lay == N_LAYERS - 1:
            truth_last[okl] = np.stack([yl, zl, sl, secl.astype(float)], axis=1)[okl]
            if stepped:
                truth_last_par[:, okl] = np.stack([yl, zl, sl, tl_now, qpt_now])[:, okl]
        idx = np.nonzero(present)[0]
        chamber_l = secl[idx] * (N_STACKS * N_LAYERS) + stack_of_z(pad_row_centre(zl[idx])) * N_LAYERS + lay
        if spec.chamber_dx_sigma > 0.0:
            # the chamber sits at x_l + dx: the tracklet is measured where the particle crosses THAT plane
            yl, zl, sl = yl.copy(), zl.copy(), sl.copy()
            xd = xl + ch_dx[chamber_l].astype(np.float64)
            if field:
                yd, zd, sd, okd = _cross_rk4(spec, kfac, gx[idx], gy[idx], gz[idx], psi[idx], qpt_now[idx], tl_now[idx], xd, secl[idx], 2)
            elif material:
                yd, zd, sd, okd = _cross_from(gx[idx], gy[idx], gz[idx], psi[idx], kfac * qpt_now[idx], tl_now[idx], xd, secl[idx])
            else:
                yd, zd, sd, okd = _truth_in_sector(phi0[idx], kappa[idx], tanl[idx], xd, secl[idx])
            assert okd.all()
            yl[idx], zl[idx], sl[idx] = yd, zd, sd
        zc = pad_row_centre(zl[idx])
        zz = zl[idx] if spec.exact_z else zc
        tanphi = sl[idx] / np.sqrt(1.0 - sl[idx] ** 2)
        if spec.res_model:
            # precise coordinate across the tilted pad, coarse one along it: the z error (row centre instead of
            # the true z) leaks into y with tan(tilt); resolutions depend on the true sin(phi)
            ds = sl[idx] - sin_lorentz(spec.bz)
            sig_y_l, sig_d_l = SY_C0 + SY_C2 * ds * ds, SD_C0 + SD_C2 * ds * ds
            tilt = math.radians(TILT_DEG) * (1.0 if lay % 2 == 0 else -1.0)
            yy = yl[idx] + math.tan(tilt) * (zz - zl[idx]) + (math.cos(tilt) * sig_y_l * ny[idx] if spec.smear_tracklets else 0.0)
            dd = tanphi + (sig_d_l * nd[idx] if spec.smear_tracklets else 0.0)
        else:
            yy = yl[idx] + (SIGMA_Y_TRACKLET * ny[idx] if spec.smear_tracklets else 0.0)
            dd = tanphi + (SIGMA_DYDX_TRACKLET * nd[idx] if spec.smear_tracklets else 0.0)
        sig_y.append(yy); sig_z.append(zz); sig_d.append(dd)
        sig_ch.append(chamber_l)
        sig_lab.append(idx); sig_lay.append(np.full(idx.shape[0], lay))

    # 4. noise tracklets (draw order: chamber, y, row pick, dy/dx)
    m_noise = spec.n_noise
    ch = rng.integers(0, N_SECTORS * N_STACKS * N_LAYERS, m_noise)
    lay_n = ch % N_LAYERS
    st_n = (ch // N_LAYERS) % N_STACKS
    xl_n = np.asarray(LAYER_X)[lay_n]
    y_n = rng.uniform(-1.0, 1.0, m_noise) * xl_n * TAN_HALF_SECTOR
    rows = _rows_by_stack()
    pick = rng.random(m_noise)
    z_n = np.empty(m_noise)
    for k in range(N_STACKS):
        sel = st_n == k
        z_n[sel] = rows[k][np.minimum((pick[sel] * len(rows[k])).astype(np.int64), len(rows[k]) - 1)]
    d_n = rng.uniform(-NOISE_DYDX_RANGE, NOISE_DYDX_RANGE, m_noise)
    n_ia = spec.n_interactions if spec.n_interactions > 1 else 0
    if n_ia:                                               # drawn only for associated specs: other specs' bytes unchanged
        trk_ia = (np.arange(n, dtype=np.int64) * n_ia) // n
        ia_n = rng.integers(0, n_ia, m_noise)

    # 5. concatenate and permute
    tl_y = np.concatenate(sig_y + [y_n]); tl_z = np.concatenate(sig_z + [z_n])
    tl_d = np.concatenate(sig_d + [d_n]); tl_ch = np.concatenate(sig_ch + [ch])
    tl_lab = np.concatenate(sig_lab + [np.full(m_noise, -1)])
    tl_lay = np.concatenate(sig_lay + [lay_n])
    m = tl_y.shape[0]
    perm = rng.permutation(m)
    tl_y, tl_z, tl_d, tl_ch, tl_lab, tl_lay = (a[perm] for a in (tl_y, tl_z, tl_d, tl_ch, tl_lab, tl_lay))
    assoc = {}
    if n_ia:
        tl_ia = np.concatenate([trk_ia[i] for i in sig_lab] + [ia_n])[perm]
        assoc = dict(n_interactions=n_ia, interaction=trk_ia.astype(np.int32), tl_interaction=tl_ia.astype(np.int32))
    truth_idx = np.full((n, N_LAYERS), -1, np.int32)
    is_sig = tl_lab >= 0
    truth_idx[tl_lab[is_sig], tl_lay[is_sig]] = np.nonzero(is_sig)[0].astype(np.int32)

    if spec.chamber_dx_sigma > 0.0:
        assoc["chamber_dx"] = ch_dx
    if stepped:
        assoc["truth_last_par"] = truth_last_par
    return dict(
        assoc, spec=spec,
        par=np.ascontiguousarray(par, np.float32), cov=np.ascontiguousarray(cov, np.float32),
        x=np.full(n, X_SEED, np.float32), sector=sec.astype(np.int32),
        tl_y=tl_y.astype(np.float32), tl_z=tl_z.astype(np.float32), tl_dydx=tl_d.astype(np.float32),
        tl_chamber=tl_ch.astype(np.int32), tl_label=tl_lab.astype(np.int32),
        truth_par=truth_par, truth_idx=truth_idx, truth_last=truth_last,
    )


def efficiency_purity(out_idx: np.ndarray, data: dict) -> dict:
    """The paper's two quality definitions on the generator's truth labels.

    efficiency = fraction of tracks matched to >= 2 correct tracklets;
    purity     = fraction of tracks with >= 2 attached tracklets that have no fake attached.
    """
    lab = data["tl_label"]
    attached = out_idx >= 0
    lab_of = np.where(attached, lab[np.where(attached, out_idx, 0)], -2)
    own = np.arange(out_idx.shape[0])[:, None]
    correct = (lab_of == own).sum(axis=1)
    fake = (attached & (lab_of != own)).sum(axis=1)
    n_att = attached.sum(axis=1)
    ge2 = n_att >= 2
    return dict(efficiency=float((correct >= 2).mean()),
                purity=float(((fake == 0) & ge2).sum() / max(int(ge2.sum()), 1)),
                frac_ge2=float(ge2.mean()))
