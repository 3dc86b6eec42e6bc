"""Toy outer-tracker geometry and module connectivity (BASELINE.json configs[0]/[1]).

Barrel: 6 cylinders r = 23, 36, 51, 68, 88, 108 cm, |z| < 120 cm, 10 cm x 10 cm tiles
(ceil(2 pi r / 10) phi-sectors x 24 z-tiles).  Layers 1-3 PS (gap 0.26 cm), 4-6 2S (gap 0.18 cm).
Endcap (configs[1]): 5 disks per side at |z| = 131, 156, 185, 220, 265 cm, rings
[23+10k, min(33+10k, 110)) cm, k = 0..8, ceil(2 pi r_centre / 10) phi-sectors per ring; PS where the
ring centre is below 60 cm, 2S beyond.  "Lower" sensor = smaller r (barrel) / smaller |z| (endcap).

Connectivity (the paper only says "adjacent tracker modules that fulfill some geometric
criteria"; the rule is configs[0]/[1]'s): a module links to modules of the NEXT layer
whose phi range overlaps within +-0.1 rad and whose z (barrel) / r (disk) range overlaps within
+-15 cm after projecting the source module's extent along straight lines from the origin onto
the target surface (reading B8).  Next layer: barrel l -> l+1; disk d -> d+1 on the same
side; barrel l -> disk 1 where a straight line through the module can leave the barrel before
layer l+1 (or l = 6).  The CSR is an INPUT of the library (include/lst.h), so this rule lives only
here.
"""
from dataclasses import dataclass
import numpy as np

BARREL_R = np.array([23.0, 36.0, 51.0, 68.0, 88.0, 108.0])
BARREL_ZMAX = 120.0
TILE = 10.0
N_ZTILES = 24
DISK_Z = np.array([131.0, 156.0, 185.0, 220.0, 265.0])
DISK_RMIN = 23.0
DISK_RMAX = 110.0
N_RINGS = 9
GAP_PS = 0.26
GAP_2S = 0.18
PHI_TOL = 0.1
LONG_TOL = 15.0


@dataclass
class Geometry:
    n_modules: int
    subdet: np.ndarray      # u8: 0 barrel, 1 endcap
    mtype: np.ndarray       # u8: 0 PS, 1 2S
    layer: np.ndarray       # u8: 1..6 barrel, 7..11 disks
    side: np.ndarray        # i8: 0 barrel, +-1 endcap
    conn_rowptr: np.ndarray  # i32 [n_modules+1]
    conn_col: np.ndarray     # i32 [nnz]
    # generator-only description of each module's surface
    phi_lo: np.ndarray      # f64 sector start in [0, 2pi)
    phi_w: np.ndarray       # f64 sector width
    a_lo: np.ndarray        # f64 barrel: z_lo ; endcap: r_lo
    a_hi: np.ndarray        # f64 barrel: z_hi ; endcap: r_hi
    pos: np.ndarray         # f64 barrel: r of lower sensor ; endcap: signed z of lower sensor
    gap: np.ndarray         # f64 sensor gap
    area: np.ndarray        # f64 cm^2 (noise-hit weights)
    # lookup helpers
    barrel_nphi: np.ndarray
    barrel_base: np.ndarray
    ring_nphi: np.ndarray
    ring_lo: np.ndarray
    ring_hi: np.ndarray
    disk_base: np.ndarray   # [2 sides][5 disks][9 rings] -> first module id
    has_endcap: bool


def _round_up(n, mult):
    return int(-(-int(n) // mult) * mult)


def build_geometry(endcap: bool = True, nphi_multiple: int = 1) -> Geometry:
    """Build the module table and CSR connectivity.

    `nphi_multiple` > 1 rounds every phi-sector count up to a multiple of it; 4 gives a geometry
    with an exact 90-degree symmetry (tests of rotation invariance).
    """
    subdet, mtype, layer, side = [], [], [], []
    phi_lo, phi_w, a_lo, a_hi, pos, gap, area = [], [], [], [], [], [], []
    barrel_nphi = np.array([_round_up(np.ceil(2 * np.pi * r / TILE), nphi_multiple) for r in BARREL_R])
    barrel_base = np.zeros(6, dtype=np.int64)
    n = 0
    for l, r in enumerate(BARREL_R):
        barrel_base[l] = n
        nphi = barrel_nphi[l]
        w = 2 * np.pi / nphi
        for ip in range(nphi):
            for iz in range(N_ZTILES):
                subdet.append(0); mtype.append(0 if l < 3 else 1); layer.append(l + 1); side.append(0)
                phi_lo.append(ip * w); phi_w.append(w)
                a_lo.append(-BARREL_ZMAX + TILE * iz); a_hi.append(-BARREL_ZMAX + TILE * (iz + 1))
                pos.append(r); gap.append(GAP_PS if l < 3 else GAP_2S)
                area.append(w * r * TILE)
                n += 1
    ring_lo = DISK_RMIN + TILE * np.arange(N_RINGS)
    ring_hi = np.minimum(ring_lo + TILE, DISK_RMAX)
    ring_c = 0.5 * (ring_lo + ring_hi)
    ring_nphi = np.array([_round_up(np.ceil(2 * np.pi * c / TILE), nphi_multiple) for c in ring_c])
    disk_base = np.zeros((2, 5, N_RINGS), dtype=np.int64)
    if endcap:
        for s_i, sg in enumerate((-1, 1)):
            for d, zd in enumerate(DISK_Z):
                for k in range(N_RINGS):
                    disk_base[s_i, d, k] = n
                    nphi = ring_nphi[k]
                    w = 2 * np.pi / nphi
                    ps = ring_c[k] < 60.0
                    for ip in range(nphi):
                        subdet.append(1); mtype.append(0 if ps else 1); layer.append(7 + d); side.append(sg)
                        phi_lo.append(ip * w); phi_w.append(w)
                        a_lo.append(ring_lo[k]); a_hi.append(ring_hi[k])
                        pos.append(sg * zd); gap.append(GAP_PS if ps else GAP_2S)
                        area.append(0.5 * w * (ring_hi[k] ** 2 - ring_lo[k] ** 2))
                        n += 1
    g = dict(
        n_modules=n,
        subdet=np.array(subdet, dtype=np.uint8), mtype=np.array(mtype, dtype=np.uint8),
        layer=np.array(layer, dtype=np.uint8), side=np.array(side, dtype=np.int8),
        phi_lo=np.array(phi_lo), phi_w=np.array(phi_w), a_lo=np.array(a_lo), a_hi=np.array(a_hi),
        pos=np.array(pos), gap=np.array(gap), area=np.array(area),
        barrel_nphi=barrel_nphi, barrel_base=barrel_base, ring_nphi=ring_nphi,
        ring_lo=ring_lo, ring_hi=ring_hi, disk_base=disk_base, has_endcap=bool(endcap),
    )
    rowptr, col = _connectivity(g)
    return Geometry(conn_rowptr=rowptr, conn_col=col, **g)


def _phi_overlap(src, dst, g):
    c1 = g["phi_lo"][src] + 0.5 * g["phi_w"][src]
    c2 = g["phi_lo"][dst] + 0.5 * g["phi_w"][dst]
    d = np.abs(c1[:, None] - c2[None, :])
    d = np.minimum(d, 2 * np.pi - d)
    return d <= 0.5 * (g["phi_w"][src][:, None] + g["phi_w"][dst][None, :]) + PHI_TOL


def _connectivity(g):
    n = g["n_modules"]
    layer, side = g["layer"], g["side"]
    rows = [[] for _ in range(n)]

    def link(src, dst, lo, hi):
        """src modules with projected interval [lo, hi] (already +-15 cm) vs dst [a_lo, a_hi]."""
        if len(src) == 0 or len(dst) == 0:
            return
        ok = _phi_overlap(src, dst, g)
        ok &= (lo[:, None] <= g["a_hi"][dst][None, :]) & (hi[:, None] >= g["a_lo"][dst][None, :])
        for i, s in enumerate(src):
            rows[s].extend(dst[ok[i]].tolist())

    ids = np.arange(n)
    for l in range(1, 7):
        src = ids[layer == l]
        r = BARREL_R[l - 1]
        if l < 6:
            dst = ids[layer == l + 1]
            sc = BARREL_R[l] / r
            link(src, dst, g["a_lo"][src] * sc - LONG_TOL, g["a_hi"][src] * sc + LONG_TOL)
        if g["has_endcap"]:
            for sg in (-1, 1):
                dst = ids[(layer == 7) & (side == sg)]
                ua = g["a_lo"][src] if sg > 0 else -g["a_hi"][src]
                ub = g["a_hi"][src] if sg > 0 else -g["a_lo"][src]
                reach = ub > 0
                if l < 6:
                    reach &= (ub * (BARREL_R[l] / r) + LONG_TOL > BARREL_ZMAX)
                s2 = src[reach]
                ua, ub = ua[reach], ub[reach]
                zd = DISK_Z[0]
                rlo = r * zd / ub
                with np.errstate(divide="ignore"):
                    rhi = np.where(ua > 0, r * zd / np.maximum(ua, 1e-300), np.inf)
                link(s2, dst, rlo - LONG_TOL, rhi + LONG_TOL)
    if g["has_endcap"]:
        for sg in (-1, 1):
            for d in range(4):
                src = ids[(layer == 7 + d) & (side == sg)]
                dst = ids[(layer == 8 + d) & (side == sg)]
                sc = DISK_Z[d + 1] / DISK_Z[d]
                link(src, dst, g["a_lo"][src] * sc - LONG_TOL, g["a_hi"][src] * sc + LONG_TOL)
    rowptr = np.zeros(n + 1, dtype=np.int32)
    cols = []
    for m in range(n):
        c = sorted(set(rows[m]))
        rowptr[m + 1] = rowptr[m] + len(c)
        cols.extend(c)
    return rowptr, np.array(cols, dtype=np.int32)
