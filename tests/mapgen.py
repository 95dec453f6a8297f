"""Test-side numpy statement of the module-map rule [B] (DESIGN.md section 1 [B]) on the
BASELINE geometry, vectorised per layer pair.  A TEST HELPER: the tests use it as the map INPUT of both the oracle and
the CUDA path, and pin P16 compares it with the oracle's ``lsto_build_map``.  It restates the same envelope formula, so
P16 alone pins nothing about B4; the independent pins are P15, P18 and P19 in tests/test_oracle_map.py."""
import math

import numpy as np

from paper_2207_08207_b200.synth import (B_TESLA, K_GEV_PER_T_CM, LAYER_R, MAP_PAD_PHI, MAP_PAD_Z, MAP_PT, MAP_Z0,
                                         MODULE_HALF_W, N_LAYERS, N_RINGS, RING_LEN, SENSOR_GAP, Z_MAX, Geometry, ModuleMap,
                                         _wrap)


def make_module_map(geom: Geometry) -> ModuleMap:
    r_m = MAP_PT / (K_GEV_PER_T_CM * B_TESLA)
    rows = [[] for _ in range(geom.n_modules)]
    for l in range(N_LAYERS - 1):
        r_lo = LAYER_R[l] - SENSOR_GAP[l] / 2
        r_hi = math.hypot(LAYER_R[l] + SENSOR_GAP[l] / 2, MODULE_HALF_W)
        rp_lo = LAYER_R[l + 1] - SENSOR_GAP[l + 1] / 2
        rp_hi = math.hypot(LAYER_R[l + 1] + SENSOR_GAP[l + 1] / 2, MODULE_HALF_W)
        a_out = math.asin(min(1.0, rp_hi / (2 * r_m)))
        a_in = math.asin(r_lo / (2 * r_m))
        dphi_max = a_out - a_in
        h_a = math.atan(MODULE_HALF_W / r_lo)
        h_b = math.atan(MODULE_HALF_W / rp_lo)
        phi_tol = h_a + h_b + dphi_max + MAP_PAD_PHI
        ratios = (rp_lo / r_hi, a_out / a_in)
        n_a, n_b = int(geom.n_phi[l]), int(geom.n_phi[l + 1])
        phi_a = 2 * np.pi * np.arange(n_a) / n_a
        phi_b = 2 * np.pi * np.arange(n_b) / n_b
        phi_ok = np.abs(_wrap(phi_b[None, :] - phi_a[:, None])) <= phi_tol       # [n_a, n_b]
        for j in range(N_RINGS):
            za = (-Z_MAX + RING_LEN * j - MAP_PAD_Z, -Z_MAX + RING_LEN * (j + 1) + MAP_PAD_Z)
            zs = [z0 + (z - z0) * rt for z0 in (-MAP_Z0, MAP_Z0) for z in za for rt in ratios]
            z_lo, z_hi = min(zs), max(zs)
            ring_lo = -Z_MAX + RING_LEN * np.arange(N_RINGS)
            rings_b = np.nonzero((z_hi >= ring_lo) & (z_lo <= ring_lo + RING_LEN))[0]
            for i in range(n_a):
                src = int(geom.base[l]) + j * n_a + i
                ib = np.nonzero(phi_ok[i])[0]
                t = (int(geom.base[l + 1]) + rings_b[:, None] * n_b + ib[None, :]).ravel()
                rows[src] = np.sort(t)
    counts = np.array([len(r) for r in rows], dtype=np.int64)
    row_offsets = np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)
    targets = (np.concatenate([np.asarray(r, dtype=np.int32) for r in rows if len(r)])
               if counts.sum() else np.zeros(0, np.int32))
    return ModuleMap(geom.n_modules, row_offsets, targets.astype(np.int32))
