"""Synthetic outer-tracker description (BASELINE.json configs).

6 barrel layers of flat 10 x 10 cm two-sensor "pT modules" (Fig. 1-2)
and, for the full detector, 5 endcap disks per side made of annular-sector modules.
Units: cm, radians.  Everything here is detector description: where the sensors are,
what kind they are, how big a box each module's lower sensor occupies.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# module categories (also the meaning of lst_geometry.category in include/lst.h)
CAT_BPS, CAT_B2S, CAT_EPS, CAT_E2S = 0, 1, 2, 3

BARREL_R = (23.0, 35.7, 50.8, 68.6, 88.6, 108.0)   # BASELINE.json config 1
BARREL_NZ = 24                                      # |z| < 120 cm in 10 cm modules
HALF_MODULE = 5.0                                   # 10 x 10 cm modules
GAP_PS, GAP_2S = 0.26, 0.18                         # sensor spacing (2.6 mm / 1.8 mm)
DISK_Z = (131.0, 155.0, 185.0, 219.0, 256.0)        # BASELINE.json config 3
N_RING = 9
RING_RLO, RING_RHI = 23.0, 110.0
D_RING = (RING_RHI - RING_RLO) / N_RING
N_PS_RINGS = 4                                      # rings 0-3 PS, 4-8 2S
GAP_OF_CAT = (GAP_PS, GAP_2S, GAP_PS, GAP_2S)

# single-hit resolutions (pitch / sqrt(12)); PS: 100 um x 1.5 mm, 2S: 90 um x 5 cm
_S12 = math.sqrt(12.0)
PITCH_T = (0.01, 0.009, 0.01, 0.009)                # precise coordinate (r-phi)
PITCH_L = (0.15, 5.0, 0.15, 5.0)                    # coarse coordinate (z barrel, r endcap)


def barrel_nphi(R: float, gap: float) -> int:
    """Smallest hermetic phi segmentation (>= 1 mm overlap at the upper sensor)."""
    n = int(math.ceil(2.0 * math.pi * R / (2.0 * HALF_MODULE)))
    while (R + gap / 2.0) * math.tan(math.pi / n) > HALF_MODULE - 0.1:
        n += 1
    return n


def ring_nphi(k: int) -> int:
    rhi = RING_RLO + (k + 1) * D_RING
    return int(math.ceil(2.0 * math.pi * rhi / (2.0 * HALF_MODULE)))


@dataclasses.dataclass
class Geometry:
    """Per-module tables (length n_modules), all numpy arrays.

    category       u8   0 bPS, 1 b2S, 2 ePS, 3 e2S
    logical_layer  u8   0-5 barrel L1-6, 6-10 disks +z, 11-15 disks -z
    rmin,rmax      f32  radial extent of the LOWER sensor (the one nearer the origin)
    phic,half_phi  f32  azimuth of the module centre and half opening angle of the lower sensor
    zmin,zmax      f32  z extent of the lower sensor (equal for endcap modules: the sensor plane)
    """
    barrel_only: bool
    category: np.ndarray
    logical_layer: np.ndarray
    rmin: np.ndarray
    rmax: np.ndarray
    phic: np.ndarray
    half_phi: np.ndarray
    zmin: np.ndarray
    zmax: np.ndarray
    # generator-internal lookup tables
    barrel_base: tuple = ()
    barrel_nphi: tuple = ()
    ring_base: tuple = ()
    ring_nphi: tuple = ()
    n_barrel: int = 0
    n_per_disk: int = 0

    @property
    def n_modules(self) -> int:
        return int(self.category.shape[0])


def build_geometry(barrel_only: bool) -> Geometry:
    cat, lay, rmin, rmax, phic, hphi, zmin, zmax = ([] for _ in range(8))
    bbase, bnphi = [], []
    for l, R in enumerate(BARREL_R):
        c = CAT_BPS if l < 3 else CAT_B2S
        gap = GAP_OF_CAT[c]
        n = barrel_nphi(R, gap)
        bbase.append(len(cat))
        bnphi.append(n)
        rl = R - gap / 2.0                      # lower sensor plane distance
        for iz in range(BARREL_NZ):
            zc = -115.0 + 10.0 * iz
            for ip in range(n):
                cat.append(c)
                lay.append(l)
                rmin.append(rl)
                rmax.append(math.hypot(rl, HALF_MODULE))
                phic.append(2.0 * math.pi * ip / n)
                hphi.append(math.atan(HALF_MODULE / rl))
                zmin.append(zc - HALF_MODULE)
                zmax.append(zc + HALF_MODULE)
    n_barrel = len(cat)
    rnphi = [ring_nphi(k) for k in range(N_RING)]
    rbase = [0]
    for n in rnphi:
        rbase.append(rbase[-1] + n)
    if not barrel_only:
        for side in (0, 1):                     # 0 = +z, 1 = -z
            sgn = 1.0 if side == 0 else -1.0
            for d, Z in enumerate(DISK_Z):
                for k in range(N_RING):
                    c = CAT_EPS if k < N_PS_RINGS else CAT_E2S
                    gap = GAP_OF_CAT[c]
                    rlo = RING_RLO + k * D_RING
                    n = rnphi[k]
                    for ip in range(n):
                        cat.append(c)
                        lay.append(6 + 5 * side + d)
                        rmin.append(rlo)
                        rmax.append(rlo + D_RING)
                        phic.append(2.0 * math.pi * (ip + 0.5) / n)
                        hphi.append(math.pi / n)
                        zl = sgn * (Z - gap / 2.0)
                        zmin.append(zl)
                        zmax.append(zl)
    f32 = lambda a: np.asarray(a, dtype=np.float32)
    return Geometry(
        barrel_only=barrel_only,
        category=np.asarray(cat, dtype=np.uint8),
        logical_layer=np.asarray(lay, dtype=np.uint8),
        rmin=f32(rmin), rmax=f32(rmax), phic=f32(phic), half_phi=f32(hphi),
        zmin=f32(zmin), zmax=f32(zmax),
        barrel_base=tuple(bbase), barrel_nphi=tuple(bnphi),
        ring_base=tuple(rbase), ring_nphi=tuple(rnphi),
        n_barrel=n_barrel, n_per_disk=rbase[-1],
    )
