"""Synthetic pile-up-shaped events (BASELINE.json configs[0..4]); recipe in DESIGN.md / SPEC.md 2.

They STAND IN for the paper's CMS full-simulation samples (ttbar + PU200, "muon-cube";
PAPER.md:64, :99, :109), which are not available.  All arithmetic is float64 on the host with one
rounding to fp32 at the end; the PRNG is numpy's PCG64 seeded per event.

Helix (B = 3.8 T along +z, kappa = 0.3*3.8/100 GeV/cm, R = pT/kappa, q = +-1):
    psi(s) = phi0 - q s / R
    x(s) = xv - q R (sin psi - sin phi0),  y(s) = yv + q R (cos psi - cos phi0),  z(s) = zv + s cot(theta)
with s the transverse path length, restricted to the first half turn 0 < s <= pi R (no loopers).
"""
from dataclasses import dataclass, field
import numpy as np
from .geometry import (Geometry, BARREL_R, BARREL_ZMAX, TILE, N_ZTILES, DISK_Z, DISK_RMIN,
                       DISK_RMAX, N_RINGS, GAP_PS, GAP_2S)

KAPPA64 = 0.3 * 3.8 / 100.0
SIG_T_PS = 0.0100 / np.sqrt(12.0)   # 100 um pitch
SIG_L_PS = 0.15 / np.sqrt(12.0)     # 1.5 mm macro-pixel / PS strip
SIG_T_2S = 0.0090 / np.sqrt(12.0)   # 90 um pitch
SIG_L_2S = 5.0 / np.sqrt(12.0)      # 5 cm strips


@dataclass
class Event:
    # library inputs (fp32 / u32 / i8), hit order shuffled
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    key: np.ndarray          # u32: 2*module + isUpper
    pls_px: np.ndarray
    pls_py: np.ndarray
    pls_pz: np.ndarray
    pls_z0: np.ndarray
    pls_q: np.ndarray        # i8
    # truth (never seen by the oracle or the library)
    hit_particle: np.ndarray  # i32, -1 = noise
    pls_particle: np.ndarray  # i32
    particles: dict = field(default_factory=dict)

    @property
    def n_hits(self):
        return int(self.x.size)

    @property
    def n_pls(self):
        return int(self.pls_px.size)


def _circle_path(xv, yv, phi0, q, R, rho):
    """Transverse path length to the first crossing of the cylinder of radius rho within the first
    half turn; NaN where there is none.  All arrays broadcast to the particle axis."""
    cx = xv + q * R * np.sin(phi0)
    cy = yv - q * R * np.cos(phi0)
    D = np.hypot(cx, cy)
    alpha = np.arctan2(cy, cx)
    with np.errstate(invalid="ignore", divide="ignore"):
        v = (rho * rho - D * D - R * R) / (2.0 * q * R * D)
        ok = np.abs(v) <= 1.0
        a = np.arcsin(np.clip(v, -1.0, 1.0))
    best = np.full(np.shape(v), np.inf)
    for sol in (a, np.pi - a):
        psi = alpha - sol
        s = ((phi0 - psi) * q) % (2.0 * np.pi) * R
        s = np.where(s <= 0.0, np.inf, s)
        best = np.minimum(best, s)
    good = ok & (best <= np.pi * R)
    return np.where(good, best, np.nan)


def _pos(xv, yv, zv, phi0, q, R, cot, s):
    psi = phi0 - q * s / R
    x = xv - q * R * (np.sin(psi) - np.sin(phi0))
    y = yv + q * R * (np.cos(psi) - np.cos(phi0))
    z = zv + s * cot
    return x, y, z


def make_event(geo: Geometry, seed: int, *, n_particles: int = 0, per_vertex: int = 30,
               origin_muons: int = 0, n_displaced: int = 0, n_noise: int = 0,
               inefficiency: float = 0.0, smear: bool = True, eta_max: float = 2.4,
               shuffle: bool = True) -> Event:
    """Generate one event.

    origin_muons  : configs[0]-style muons from (0,0,0), pT U(1,10), |eta| < 0.8.
    n_particles   : pile-up particles, `per_vertex` per vertex with z_v ~ N(0, 5 cm), |eta| < eta_max
                    uniform, pT exponential (mean 0.6) truncated to [0.3, 50] GeV.
    n_displaced   : configs[4] particles, r_vtx U(0,50), z_vtx U(-30,30), pT U(1,20), |eta| < 2.4.
    """
    rng = np.random.Generator(np.random.PCG64(int(seed)))
    xv, yv, zv, pt, eta, phi, q, disp = [], [], [], [], [], [], [], []
    if origin_muons:
        n = origin_muons
        xv.append(np.zeros(n)); yv.append(np.zeros(n)); zv.append(np.zeros(n))
        pt.append(rng.uniform(1.0, 10.0, n)); eta.append(rng.uniform(-0.8, 0.8, n))
        phi.append(rng.uniform(0.0, 2 * np.pi, n)); q.append(rng.choice([-1.0, 1.0], n))
        disp.append(np.zeros(n, bool))
    if n_particles:
        n = n_particles
        nv = max(1, -(-n // per_vertex))
        vz = rng.normal(0.0, 5.0, nv)
        xv.append(np.zeros(n)); yv.append(np.zeros(n)); zv.append(vz[np.arange(n) // per_vertex])
        u = rng.uniform(0.0, 1.0, n)
        pt.append(0.3 - 0.6 * np.log(1.0 - u * (1.0 - np.exp(-49.7 / 0.6))))
        eta.append(rng.uniform(-eta_max, eta_max, n))
        phi.append(rng.uniform(0.0, 2 * np.pi, n)); q.append(rng.choice([-1.0, 1.0], n))
        disp.append(np.zeros(n, bool))
    if n_displaced:
        n = n_displaced
        rv = rng.uniform(0.0, 50.0, n)
        av = rng.uniform(0.0, 2 * np.pi, n)
        xv.append(rv * np.cos(av)); yv.append(rv * np.sin(av)); zv.append(rng.uniform(-30.0, 30.0, n))
        pt.append(rng.uniform(1.0, 20.0, n)); eta.append(rng.uniform(-2.4, 2.4, n))
        phi.append(rng.uniform(0.0, 2 * np.pi, n)); q.append(rng.choice([-1.0, 1.0], n))
        disp.append(np.ones(n, bool))
    cat = lambda a: np.concatenate(a) if a else np.zeros(0)
    xv, yv, zv, pt, eta, phi, q = map(cat, (xv, yv, zv, pt, eta, phi, q))
    disp = np.concatenate(disp) if disp else np.zeros(0, bool)
    P = pt.size
    R = pt / KAPPA64
    cot = np.sinh(eta)
    rvtx = np.hypot(xv, yv)

    hx, hy, hz, hkey, hpart = [], [], [], [], []
    pid = np.arange(P)

    def emit(sel, x, y, z, mod, upper):
        hx.append(x[sel]); hy.append(y[sel]); hz.append(z[sel])
        hkey.append(2 * mod[sel] + upper); hpart.append(pid[sel])

    # ---- barrel ----
    for l, r_l in enumerate(BARREL_R):
        ps = l < 3
        gap = GAP_PS if ps else GAP_2S
        sig_t, sig_l = (SIG_T_PS, SIG_L_PS) if ps else (SIG_T_2S, SIG_L_2S)
        nphi = geo.barrel_nphi[l]
        s_lo = _circle_path(xv, yv, phi, q, R, r_l)
        x0, y0, z0 = _pos(xv, yv, zv, phi, q, R, cot, s_lo)
        with np.errstate(invalid="ignore"):
            ok = np.isfinite(s_lo) & (np.abs(z0) < BARREL_ZMAX) & (rvtx < r_l)
        ph = np.where(ok, np.mod(np.arctan2(y0, x0), 2 * np.pi), 0.0)
        ip = np.minimum((ph / (2 * np.pi / nphi)).astype(np.int64), nphi - 1)
        iz = np.clip(np.floor((np.where(ok, z0, 0.0) + BARREL_ZMAX) / TILE), 0, N_ZTILES - 1).astype(np.int64)
        mod = geo.barrel_base[l] + ip * N_ZTILES + iz
        mod = np.where(ok, mod, 0)
        for upper, rho in ((0, r_l), (1, r_l + gap)):
            s = s_lo if upper == 0 else _circle_path(xv, yv, phi, q, R, rho)
            x, y, z = _pos(xv, yv, zv, phi, q, R, cot, s)
            good = ok & np.isfinite(s)
            if smear:
                pa = np.arctan2(y, x) + rng.normal(0.0, 1.0, P) * sig_t / rho
                z = z + rng.normal(0.0, 1.0, P) * sig_l
                x, y = rho * np.cos(pa), rho * np.sin(pa)
            if inefficiency > 0.0:
                good = good & (rng.uniform(0.0, 1.0, P) >= inefficiency)
            emit(good, x, y, z, mod, upper)

    # ---- endcap ----
    if geo.has_endcap:
        for s_i, sg in enumerate((-1.0, 1.0)):
            for d, zd in enumerate(DISK_Z):
                with np.errstate(divide="ignore", invalid="ignore"):
                    s_lo = (sg * zd - zv) / cot
                x0, y0, _ = _pos(xv, yv, zv, phi, q, R, cot, s_lo)
                r0 = np.hypot(x0, y0)
                with np.errstate(invalid="ignore"):
                    ok = (np.isfinite(s_lo) & (s_lo > 0) & (s_lo <= np.pi * R) & (r0 >= DISK_RMIN)
                          & (r0 < DISK_RMAX) & (np.abs(zv) < zd))
                k = np.clip(np.floor((np.where(ok, r0, DISK_RMIN) - DISK_RMIN) / TILE), 0, N_RINGS - 1).astype(np.int64)
                nphi = geo.ring_nphi[k]
                ph = np.mod(np.arctan2(y0, x0), 2 * np.pi)
                ip = np.minimum((np.where(ok, ph, 0.0) / (2 * np.pi / nphi)).astype(np.int64), nphi - 1)
                mod = np.where(ok, geo.disk_base[s_i, d, k] + ip, 0)
                ps = geo.ring_lo[k] + 0.5 * (geo.ring_hi[k] - geo.ring_lo[k]) < 60.0
                gap = np.where(ps, GAP_PS, GAP_2S)
                sig_t = np.where(ps, SIG_T_PS, SIG_T_2S)
                sig_l = np.where(ps, SIG_L_PS, SIG_L_2S)
                for upper in (0, 1):
                    zp = sg * (zd + upper * gap)
                    with np.errstate(divide="ignore", invalid="ignore"):
                        s = (zp - zv) / cot
                    x, y, _ = _pos(xv, yv, zv, phi, q, R, cot, s)
                    with np.errstate(invalid="ignore"):
                        good = ok & np.isfinite(s) & (s <= np.pi * R)
                    if smear:
                        r = np.hypot(x, y)
                        pa = np.arctan2(y, x) + rng.normal(0.0, 1.0, P) * sig_t / np.where(good, r, 1.0)
                        r = r + rng.normal(0.0, 1.0, P) * sig_l
                        x, y = r * np.cos(pa), r * np.sin(pa)
                    if inefficiency > 0.0:
                        good = good & (rng.uniform(0.0, 1.0, P) >= inefficiency)
                    emit(good, x, y, np.broadcast_to(zp, x.shape).copy(), mod, upper)

    # ---- noise: module ~ area, sensor 50/50, uniform on the surface ----
    if n_noise:
        pm = geo.area / geo.area.sum()
        mod = rng.choice(geo.n_modules, size=n_noise, p=pm)
        upper = rng.integers(0, 2, n_noise)
        ph = geo.phi_lo[mod] + rng.uniform(0.0, 1.0, n_noise) * geo.phi_w[mod]
        u = rng.uniform(0.0, 1.0, n_noise)
        barrel = geo.subdet[mod] == 0
        r = np.where(barrel, geo.pos[mod] + upper * geo.gap[mod],
                     np.sqrt(geo.a_lo[mod] ** 2 + u * (geo.a_hi[mod] ** 2 - geo.a_lo[mod] ** 2)))
        z = np.where(barrel, geo.a_lo[mod] + u * (geo.a_hi[mod] - geo.a_lo[mod]),
                     geo.pos[mod] + np.sign(geo.pos[mod]) * upper * geo.gap[mod])
        hx.append(r * np.cos(ph)); hy.append(r * np.sin(ph)); hz.append(z)
        hkey.append(2 * mod + upper); hpart.append(np.full(n_noise, -1))

    hx, hy, hz = cat(hx), cat(hy), cat(hz)
    hkey = np.concatenate(hkey).astype(np.int64) if hkey else np.zeros(0, np.int64)
    hpart = np.concatenate(hpart).astype(np.int64) if hpart else np.zeros(0, np.int64)
    if shuffle and hx.size:
        perm = rng.permutation(hx.size)
        hx, hy, hz, hkey, hpart = hx[perm], hy[perm], hz[perm], hkey[perm], hpart[perm]

    # ---- pixel seeds: every prompt particle with pT > 0.8 GeV; (pT, eta, phi) smeared 1 %, 1 mrad ----
    sel = np.flatnonzero((pt > 0.8) & ~disp)
    n = sel.size
    pts = pt[sel] * (1.0 + 0.01 * rng.normal(0.0, 1.0, n))
    etas = eta[sel] + 0.001 * rng.normal(0.0, 1.0, n)
    phis = phi[sel] + 0.001 * rng.normal(0.0, 1.0, n)
    z0s = zv[sel] + 0.01 * rng.normal(0.0, 1.0, n)
    if not smear:
        pts, etas, phis, z0s = pt[sel], eta[sel], phi[sel], zv[sel]
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return Event(
        x=f32(hx), y=f32(hy), z=f32(hz), key=np.ascontiguousarray(hkey, dtype=np.uint32),
        pls_px=f32(pts * np.cos(phis)), pls_py=f32(pts * np.sin(phis)), pls_pz=f32(pts * np.sinh(etas)),
        pls_z0=f32(z0s), pls_q=np.ascontiguousarray(q[sel], dtype=np.int8),
        hit_particle=hpart.astype(np.int32), pls_particle=sel.astype(np.int32),
        particles=dict(xv=xv, yv=yv, zv=zv, pt=pt, eta=eta, phi=phi, q=q, displaced=disp),
    )


CONFIG_SEEDS = {0: 1, 1: 2, 2: 3}


def config_event(geo: Geometry, config: int, seed: int = None, pileup: int = 200) -> Event:
    """Events of BASELINE.json configs: 0 barrel toy, 1 PU50, 2 PU200 (also configs[3]'s events with
    seeds 100-163), 4 PU`pileup` + 500 displaced (seeds 200-231)."""
    if config == 0:
        return make_event(geo, 1 if seed is None else seed, origin_muons=10)
    if config == 1:
        return make_event(geo, 2 if seed is None else seed, n_particles=1500, n_noise=2000)
    if config in (2, 3):
        return make_event(geo, 3 if seed is None else seed, n_particles=6000, n_noise=10000,
                          inefficiency=0.05)
    if config == 4:
        return make_event(geo, 200 if seed is None else seed, n_particles=30 * pileup,
                          n_noise=50 * pileup, n_displaced=500, inefficiency=0.05)
    raise ValueError(f"unknown config {config}")
