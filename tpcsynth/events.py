"""Seeded synthetic TPC events (inputs only).

This module is the one thing the CPU oracle (``oracle/``) and the CUDA path
(``paper_1712_09407_b200/``) have in common: it produces *inputs* — cluster
positions grouped by (sector, pad row) — and the truth bookkeeping the tests
use.  It contains none of the tracker's arithmetic (no binning, no neighbour
criterion, no Kalman filter, no selection).

Stand-in for the paper's workload.  The paper measures on ALICE Monte-Carlo and
2010/2011 Pb-Pb data, which are not available
here.  The events below take that workload's *shape*: 2 x 18 trapezoidal
sectors and 159 pad rows, helices in a solenoidal field, a few
million clusters for a central Pb-Pb-like event.  The five configurations are
the ones ``BASELINE.json: configs`` lists; the recipe is restated in DESIGN.md
("Input recipe").

Conventions
-----------
* Global frame: z along the beam, field Bz along +z.  Sector ``j`` (0..17) has
  its central radial axis at azimuth ``(j + 0.5) * 20 deg``; sectors 0..17 hold
  z_global >= 0, sectors 18..35 hold z_global < 0.  Local frame of a sector:
  x along its axis, y across it, local z = |z_global|.
* Single-sector configurations use one sector whose local frame is the global
  frame (axis along +x); eta is folded so that all tracks have z >= 0.
* Helix: direction angle phi(s) = phi0 + kappa * s with s the path length in
  the x-y plane, kappa = -q * KB * Bz / pT  [1/cm], KB = 0.299792458e-2
  GeV/c / (T cm); x(s) = xv + (sin(phi) - sin(phi0)) / kappa,
  y(s) = yv - (cos(phi) - cos(phi0)) / kappa, z(s) = zv + tan(lambda) * s.
* A cluster is produced where the outgoing arc first crosses the regular 18-gon
  formed by the row-k lines ``x_local = row_x[k]``, rows taken in increasing k.
  The track ends when the next row is not reached within half a turn or when
  |z| exceeds z_max.
* All generator math is float64; positions are cast to float32 at the end and
  stored as (x, y, z) with x == row_x[k] exactly.

Draw order (numpy ``default_rng(seed)``, PCG64), fixed:
  per track block: pT, charge, phi, eta, vertex z, [secondaries: r, azimuth],
  kink flag; then per row k = 0..R-1 and in that order: smear_y[all tracks],
  smear_z[all tracks], drop_u[all tracks], kink_dphi[all], kink_dlam[all];
  then noise (y, z per noise cluster, in (sector, row) order); then one uniform
  shuffle key per cluster.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

KB = 0.299792458e-2          # GeV/c per (T cm)
N_ROWS = 159
SECTOR_DEG = 20.0
NOISE_ID = 0xFFFFFFFF


def row_x_table() -> np.ndarray:
    """Row radii in cm, float64: 84.85, then 62 x 0.75, 64 x 1.0, 32 x 1.5.

    BASELINE.json configs[0]: "row radii x from 84.85 cm, with 63 rows at 0.75 cm
    pitch, 64 at 1.0 cm and 32 at 1.5 cm" (rows 0..62, 63..126, 127..158).
    """
    x = np.empty(N_ROWS, dtype=np.float64)
    x[0] = 84.85
    for i in range(1, N_ROWS):
        pitch = 0.75 if i <= 62 else (1.0 if i <= 126 else 1.5)
        x[i] = x[i - 1] + pitch
    return x


@dataclass(frozen=True)
class Geometry:
    n_sectors: int = 36
    n_rows: int = N_ROWS
    tan_half_angle: float = float(np.float32(np.tan(np.deg2rad(10.0))))
    z_max: float = 250.0
    bz_tesla: float = 0.5
    row_x: np.ndarray = field(default_factory=lambda: row_x_table().astype(np.float32))


@dataclass(frozen=True)
class EventConfig:
    name: str
    n_sectors: int               # 1 or 36
    n_primaries: int
    pt_mode: str                 # "uniform" | "exp"
    pt_lo: float = 0.5           # uniform: lower edge / exp: truncation (shift)
    pt_hi: float = 5.0           # uniform: upper edge
    pt_mean: float = 0.5         # exp: mean of the exponential
    eta_max: float = 0.9
    vertex_sigma_z: float = 0.0
    n_secondaries: int = 0
    sec_rmax: float = 50.0
    sigma_yz: float = 0.1
    drop_frac: float = 0.0
    kink_frac: float = 0.0
    kink_sigma: float = 0.0
    noise_frac: float = 0.0
    default_seed: int = 0


# BASELINE.json configs[0..3]; configs[4] is a stream of config-4 events.
CONFIGS = {
    1: EventConfig("single-sector-100", 1, 100, "uniform", 0.5, 5.0, sigma_yz=0.1, default_seed=1),
    2: EventConfig("single-sector-2000", 1, 2000, "exp", 0.1, pt_mean=0.5, sigma_yz=0.1,
                   drop_frac=0.02, kink_frac=0.05, kink_sigma=2e-3, noise_frac=0.10, default_seed=2),
    3: EventConfig("pp-like", 36, 800, "exp", 0.1, pt_mean=0.5, vertex_sigma_z=5.0,
                   sigma_yz=0.1, noise_frac=0.02, default_seed=3),
    4: EventConfig("central-PbPb-like", 36, 20000, "exp", 0.1, pt_mean=0.5, vertex_sigma_z=5.0,
                   n_secondaries=3000, sec_rmax=50.0, sigma_yz=0.12, noise_frac=0.05, default_seed=4),
}
STREAM_BASE_SEED = 1000          # config 5: event e uses config 4 with seed 1000 + e


@dataclass
class Event:
    geometry: Geometry
    xyz: np.ndarray              # float32 [N, 3], sector-local cm, sorted by (sector, row)
    row_start: np.ndarray        # uint32 [n_sectors * n_rows + 1]
    truth_id: np.ndarray         # uint32 [N], track number or NOISE_ID (never given to the tracker)
    true_y: np.ndarray           # float64 [N] unsmeared local y (NaN for noise)
    true_z: np.ndarray           # float64 [N]
    true_sinphi: np.ndarray      # float64 [N] sin of local direction angle at the crossing
    tracks: dict                 # per-track truth arrays: q, pt, phi0, tanl, xv, yv, zv, kappa, kinked
    seed: int
    config: EventConfig

    @property
    def n_clusters(self) -> int:
        return int(self.xyz.shape[0])


def _cross_row(x, y, phi, kappa, X, alpha):
    """Outgoing crossing of the line x_local = X in the frame rotated by alpha.

    Returns (theta, valid): theta = kappa * ds (turning angle, sign of kappa), and
    whether a crossing with cos(phi_local) > 0 exists within half a turn.
    """
    ca, sa = np.cos(alpha), np.sin(alpha)
    xl = x * ca + y * sa
    phil = phi - alpha
    S = np.sin(phil) + kappa * (X - xl)
    valid = np.abs(S) <= 1.0
    phi1 = np.arcsin(np.clip(S, -1.0, 1.0))
    sgn = np.where(kappa >= 0.0, 1.0, -1.0)
    theta = np.mod((phi1 - phil) * sgn, 2.0 * np.pi) * sgn
    valid &= (np.abs(theta) <= np.pi) & (theta != 0.0)
    return theta, valid


def generate_event(config: EventConfig | int = 1, seed: Optional[int] = None,
                   geometry: Optional[Geometry] = None) -> Event:
    if isinstance(config, int):
        config = CONFIGS[config]
    if seed is None:
        seed = config.default_seed
    geo = geometry if geometry is not None else Geometry(n_sectors=config.n_sectors)
    if geo.n_sectors != config.n_sectors:
        geo = replace(geo, n_sectors=config.n_sectors)
    rng = np.random.default_rng(seed)
    R = geo.n_rows
    rowx = geo.row_x.astype(np.float64)
    tan_half = float(geo.tan_half_angle)
    ymax = rowx * tan_half
    single = config.n_sectors == 1
    sect = np.deg2rad(SECTOR_DEG)

    # ---- per-track draws ---------------------------------------------------
    nt = config.n_primaries + config.n_secondaries
    if config.pt_mode == "uniform":
        pt = rng.uniform(config.pt_lo, config.pt_hi, nt)
    else:
        pt = config.pt_lo + rng.exponential(config.pt_mean, nt)
    q = np.where(rng.random(nt) < 0.5, -1.0, 1.0)
    if single:
        phi0 = rng.uniform(-0.5 * sect, 0.5 * sect, nt)
    else:
        phi0 = rng.uniform(0.0, 2.0 * np.pi, nt)
    eta = rng.uniform(-config.eta_max, config.eta_max, nt)
    tanl = np.sinh(eta)
    if single:
        tanl = np.abs(tanl)
    zv = rng.normal(0.0, 1.0, nt) * config.vertex_sigma_z
    if single:
        zv = np.zeros(nt)
    xv = np.zeros(nt)
    yv = np.zeros(nt)
    if config.n_secondaries:
        rs = rng.uniform(0.0, config.sec_rmax, config.n_secondaries)
        az = rng.uniform(0.0, 2.0 * np.pi, config.n_secondaries)
        xv[config.n_primaries:] = rs * np.cos(az)
        yv[config.n_primaries:] = rs * np.sin(az)
    kinked = rng.random(nt) < config.kink_frac if config.kink_frac > 0 else np.zeros(nt, bool)
    kappa = -q * KB * geo.bz_tesla / pt

    # ---- follow the helices row by row -------------------------------------
    x, y, z, phi = xv.copy(), yv.copy(), zv.copy(), phi0.copy()
    tl = tanl.copy()
    alive = np.ones(nt, bool)
    jprev = np.zeros(nt, np.int64)
    rec_tid, rec_sec, rec_row, rec_y, rec_z, rec_ty, rec_tz, rec_sp = ([] for _ in range(8))
    for k in range(R):
        X = rowx[k]
        sm_y = rng.normal(0.0, config.sigma_yz, nt)
        sm_z = rng.normal(0.0, config.sigma_yz, nt)
        drop_u = rng.random(nt)
        kd_phi = rng.normal(0.0, 1.0, nt)
        kd_lam = rng.normal(0.0, 1.0, nt)
        if single:
            cand = np.zeros((1, nt), np.int64)
        elif k == 0:
            cand = np.repeat(np.arange(18)[:, None], nt, axis=1)
        else:
            cand = np.stack([(jprev - 1) % 18, jprev, (jprev + 1) % 18])
        best_theta = np.full(nt, np.inf)
        best_j = np.zeros(nt, np.int64)
        for c in range(cand.shape[0]):
            j = cand[c]
            alpha = np.zeros(nt) if single else (j + 0.5) * sect
            theta, valid = _cross_row(x, y, phi, kappa, X, alpha)
            better = valid & (np.abs(theta) < np.abs(best_theta))
            best_theta = np.where(better, theta, best_theta)
            best_j = np.where(better, j, best_j)
        found = alive & np.isfinite(best_theta)
        theta = np.where(found, best_theta, 0.0)
        ds = np.where(found, theta / kappa, 0.0)
        phin = phi + theta
        xn = x + (np.sin(phin) - np.sin(phi)) / kappa
        yn = y - (np.cos(phin) - np.cos(phi)) / kappa
        zn = z + tl * ds
        found &= np.abs(zn) <= geo.z_max
        alive = found
        x = np.where(found, xn, x)
        y = np.where(found, yn, y)
        z = np.where(found, zn, z)
        phi = np.where(found, phin, phi)
        jprev = np.where(found, best_j, jprev)
        alpha = np.zeros(nt) if single else (best_j + 0.5) * sect
        yl = -x * np.sin(alpha) + y * np.cos(alpha)
        inside = np.abs(yl) <= ymax[k] * (1.0 + 1e-12)
        keep = found & inside
        if config.drop_frac > 0:
            keep &= drop_u >= config.drop_frac
        idx = np.nonzero(keep)[0]
        if idx.size:
            side = (z[idx] < 0.0).astype(np.int64)
            sec = np.zeros(idx.size, np.int64) if single else best_j[idx] + 18 * side
            rec_tid.append(idx)
            rec_sec.append(sec)
            rec_row.append(np.full(idx.size, k, np.int64))
            rec_ty.append(yl[idx])
            rec_tz.append(np.abs(z[idx]))
            rec_y.append(yl[idx] + sm_y[idx])
            rec_z.append(np.abs(z[idx]) + sm_z[idx])
            rec_sp.append(np.sin(phi[idx] - alpha[idx]))
        if config.kink_frac > 0:
            kk = found & kinked
            phi = np.where(kk, phi + config.kink_sigma * kd_phi, phi)
            lam = np.arctan(tl) + np.where(kk, config.kink_sigma * kd_lam, 0.0)
            tl = np.tan(lam)

    def cat(lst, dt):
        return np.concatenate(lst).astype(dt) if lst else np.zeros(0, dt)
    tid = cat(rec_tid, np.int64)
    sec = cat(rec_sec, np.int64)
    row = cat(rec_row, np.int64)
    cy, cz = cat(rec_y, np.float64), cat(rec_z, np.float64)
    ty, tz, sp = cat(rec_ty, np.float64), cat(rec_tz, np.float64), cat(rec_sp, np.float64)

    # ---- noise --------------------------------------------------------------
    S = config.n_sectors
    sr = sec * R + row
    n_signal = np.bincount(sr, minlength=S * R)
    if config.noise_frac > 0:
        n_noise = np.floor(config.noise_frac * n_signal + 0.5).astype(np.int64)
        tot = int(n_noise.sum())
        nsr = np.repeat(np.arange(S * R), n_noise)
        ny_ = rng.uniform(-1.0, 1.0, tot) * ymax[nsr % R]
        nz_ = rng.uniform(0.0, geo.z_max, tot)
        sr = np.concatenate([sr, nsr])
        tid = np.concatenate([tid, np.full(tot, NOISE_ID, np.int64)])
        cy = np.concatenate([cy, ny_])
        cz = np.concatenate([cz, nz_])
        nan = np.full(tot, np.nan)
        ty, tz, sp = np.concatenate([ty, nan]), np.concatenate([tz, nan]), np.concatenate([sp, nan])

    # ---- shuffle inside rows, sort by (sector, row) -------------------------
    key = rng.random(sr.size)
    order = np.argsort(sr + key, kind="stable")   # (sector,row) major, shuffle key minor
    sr = sr[order]
    counts = np.bincount(sr, minlength=S * R)
    row_start = np.zeros(S * R + 1, np.uint32)
    row_start[1:] = np.cumsum(counts)
    xyz = np.empty((sr.size, 3), np.float32)
    xyz[:, 0] = geo.row_x[(sr % R)]
    xyz[:, 1] = cy[order].astype(np.float32)
    xyz[:, 2] = cz[order].astype(np.float32)
    tracks = dict(q=q, pt=pt, phi0=phi0, tanl=tanl, xv=xv, yv=yv, zv=zv, kappa=kappa, kinked=kinked)
    return Event(geo, np.ascontiguousarray(xyz), row_start, tid[order].astype(np.uint32),
                 ty[order], tz[order], sp[order], tracks, int(seed), config)


def generate_stream(n_events: int, base_seed: int = STREAM_BASE_SEED, config: int = 4):
    """Config 5: ``n_events`` events of ``config`` with seeds base_seed + e."""
    return [generate_event(config, base_seed + e) for e in range(n_events)]
