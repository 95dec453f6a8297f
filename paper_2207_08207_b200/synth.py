"""Seeded synthetic inputs for the LST hot path: detector geometry and events.

This module produces INPUTS only (BASELINE.json ``configs[0..4]``; recipe in DESIGN.md
section "Input recipe", formulas from SURVEY.md Appendix A).  It holds none of the
method's arithmetic: no mini-doublet / segment / triplet / quintuplet selection, no
duplicate cleaning, and no module-map derivation (rule [B] is a step of the method: the
CUDA library builds the map with ``lst_build_module_map``, the oracle with ``lsto_build_map``,
and the tests keep a third, numpy statement of it in ``tests/mapgen.py``).  The CPU oracle
and the CUDA path (``csrc/``) both receive what is generated here as plain arrays, and
neither of them is imported from here.

The paper measures on CMS tt-bar + PU200 simulation, which is not
available; these events stand in for it (same gross shape: barrel pT modules, soft
pile-up-like spectrum, ~1e5 hits).

Everything is deterministic from ``seed`` (numpy PCG64, fixed draw order, see
``generate_event``).  Units: cm, GeV, tesla, radians.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# ----------------------------------------------------------------------------------------
# Detector description (BASELINE.json configs[0])
# ----------------------------------------------------------------------------------------
K_GEV_PER_T_CM = 2.99792458e-3          # pT [GeV] = K * B [T] * R [cm]
B_TESLA = 3.8
LAYER_R = (23.0, 35.7, 50.8, 68.6, 88.7, 108.0)
SENSOR_GAP = (0.26, 0.26, 0.26, 0.16, 0.16, 0.16)
SIGMA_RPHI = 0.0026                      # 26 um
SIGMA_Z = (0.043, 0.043, 0.043, 1.4, 1.4, 1.4)
MODULE_HALF_W = 4.8                      # 9.6 cm in r-phi
RING_LEN = 10.0                          # 10 cm in z
Z_MAX = 120.0
N_RINGS = 24
N_LAYERS = 6

# module-map derivation parameters (SURVEY.md 8(c) reading #6)
MAP_PT = 0.8
MAP_Z0 = 15.0
MAP_PAD_PHI = 0.01
MAP_PAD_Z = 1.0


@dataclasses.dataclass(frozen=True)
class Geometry:
    """Flat-barrel pT-module geometry. Arrays are per module unless noted."""
    n_modules: int
    n_phi: np.ndarray        # [6] modules per ring
    base: np.ndarray         # [6] first module id of each layer
    layer: np.ndarray        # int8  [n_modules] 0..5
    kind: np.ndarray         # int8  [n_modules] 0 = PS (layers 0-2), 1 = 2S (layers 3-5)
    ring: np.ndarray         # int32 [n_modules] 0..23
    iphi: np.ndarray         # int32 [n_modules]
    phi: np.ndarray          # float64 [n_modules] azimuth of the module normal
    cx: np.ndarray           # float32 module centre
    cy: np.ndarray
    cz: np.ndarray


def make_geometry() -> Geometry:
    n_phi = np.array([int(math.ceil(2.0 * math.pi * r / (2 * MODULE_HALF_W))) + 1 for r in LAYER_R],
                     dtype=np.int64)
    per_layer = n_phi * N_RINGS
    base = np.concatenate([[0], np.cumsum(per_layer)[:-1]]).astype(np.int64)
    n_modules = int(per_layer.sum())
    layer = np.empty(n_modules, np.int8)
    ring = np.empty(n_modules, np.int32)
    iphi = np.empty(n_modules, np.int32)
    phi = np.empty(n_modules, np.float64)
    for l in range(N_LAYERS):
        ids = np.arange(per_layer[l])
        sl = slice(base[l], base[l] + per_layer[l])
        layer[sl] = l
        ring[sl] = ids // n_phi[l]
        iphi[sl] = ids % n_phi[l]
        phi[sl] = 2.0 * math.pi * (ids % n_phi[l]) / n_phi[l]
    r = np.asarray(LAYER_R)[layer]
    return Geometry(
        n_modules=n_modules, n_phi=n_phi, base=base, layer=layer,
        kind=(layer >= 3).astype(np.int8), ring=ring, iphi=iphi, phi=phi,
        cx=(r * np.cos(phi)).astype(np.float32), cy=(r * np.sin(phi)).astype(np.float32),
        cz=(-Z_MAX + RING_LEN * (ring + 0.5)).astype(np.float32))


def _wrap(a):
    return (a + np.pi) % (2.0 * np.pi) - np.pi


# ----------------------------------------------------------------------------------------
# Module map container (module -> connectable modules of the next layer). CSR, rows
# sorted ascending.  The derivation itself is not here (see the module docstring).
# ----------------------------------------------------------------------------------------
@dataclasses.dataclass(frozen=True)
class ModuleMap:
    n_modules: int
    row_offsets: np.ndarray   # int32 [n_modules+1]
    targets: np.ndarray       # int32 [row_offsets[-1]]


def map_geometry(geom: Geometry) -> dict:
    """Per-module inputs of the module-map builder [B] (float64): azimuth of the normal, normal distance of the
    mid-plane, sensor gap, half width in r-phi, z range.  Input data only, none of the builder's arithmetic."""
    l = geom.layer.astype(np.int64)
    zlo = -Z_MAX + RING_LEN * geom.ring.astype(np.float64)
    return dict(layer=geom.layer.astype(np.int8), phi=geom.phi.astype(np.float64), rho=np.asarray(LAYER_R, np.float64)[l],
                gap=np.asarray(SENSOR_GAP, np.float64)[l], hw=np.full(geom.n_modules, MODULE_HALF_W, np.float64),
                zlo=zlo, zhi=zlo + RING_LEN)


# ----------------------------------------------------------------------------------------
# Events
# ----------------------------------------------------------------------------------------
@dataclasses.dataclass
class Event:
    """Hit SoA as the library receives it, plus generator truth (never seen by the method)."""
    x: np.ndarray            # float32 [n]
    y: np.ndarray
    z: np.ndarray
    module: np.ndarray       # int32 [n]
    side: np.ndarray         # uint8 [n]  0 = lower sensor (anchor), 1 = upper sensor
    truth: np.ndarray        # int32 [n]  particle index, -1 = noise
    particles: dict          # z0, q, pt, phi0, eta (float64 arrays [n_particles])

    @property
    def n(self) -> int:
        return int(self.x.shape[0])


def helix_point(pt, q, phi0, eta, z0, theta):
    """Position on the helix from (0,0,z0) at turning angle theta >= 0 (float64)."""
    R = pt / (K_GEV_PER_T_CM * B_TESLA)
    s = -q
    psi = phi0 + s * theta
    x = (R / s) * (np.sin(psi) - np.sin(phi0))
    y = -(R / s) * (np.cos(psi) - np.cos(phi0))
    z = z0 + R * theta * np.sinh(eta)
    return x, y, z


def propagate(geom: Geometry, z0, q, pt, phi0, eta, du=None, dz=None):
    """Intersections of helices with every sensor plane they cross inside an active area.

    Inputs are float64 arrays [P]. ``du``/``dz`` are optional smearing offsets of shape
    [P, 6, 2, 3] (layer, side, module candidate). Returns hit arrays in
    (particle, layer, side, candidate) order: x, y, z (float64), module, side, particle.
    """
    P = len(pt)
    R = pt / (K_GEV_PER_T_CM * B_TESLA)
    s = -q.astype(np.float64)
    out = []
    for l in range(N_LAYERS):
        n_phi = int(geom.n_phi[l])
        step = 2 * np.pi / n_phi
        reach = LAYER_R[l] < 2 * R
        phi_c = phi0 + s * np.arcsin(np.where(reach, LAYER_R[l] / (2 * R), 0.0))
        i0 = np.rint(phi_c / step).astype(np.int64)
        for side in (0, 1):
            rho = LAYER_R[l] + (side - 0.5) * SENSOR_GAP[l]
            for c in range(3):
                i = (i0 + (c - 1)) % n_phi
                Phi = step * i
                A = _wrap(phi0 - Phi)
                arg = np.sin(A) + s * rho / R
                ok = reach & (np.cos(A) > 0) & (np.abs(arg) < 1)
                theta = s * (np.arcsin(np.clip(arg, -1, 1)) - A)
                ok &= (theta > 0) & (theta < np.pi)
                x, y, z = helix_point(pt, q, phi0, eta, z0, theta)
                u = -x * np.sin(Phi) + y * np.cos(Phi)
                ok &= (np.abs(u) <= MODULE_HALF_W) & (z >= -Z_MAX) & (z < Z_MAX)
                ring = np.minimum(np.floor((z + Z_MAX) / RING_LEN).astype(np.int64), N_RINGS - 1)   # z one ulp below Z_MAX
                if du is not None:
                    u = u + du[:, l, side, c]
                    z = z + dz[:, l, side, c]
                xs = rho * np.cos(Phi) - u * np.sin(Phi)
                ys = rho * np.sin(Phi) + u * np.cos(Phi)
                mod = geom.base[l] + ring * n_phi + i
                idx = np.nonzero(ok)[0]
                key = ((idx * N_LAYERS + l) * 2 + side) * 3 + c
                out.append((key, xs[idx], ys[idx], z[idx], mod[idx],
                            np.full(len(idx), side, np.uint8), idx))
    key = np.concatenate([o[0] for o in out])
    order = np.argsort(key, kind="stable")
    cat = lambda k: np.concatenate([o[k] for o in out])[order]
    return cat(1), cat(2), cat(3), cat(4).astype(np.int32), cat(5), cat(6).astype(np.int32)


# (n_particles, pt law, |eta| max, noise fraction) per BASELINE.json config
CONFIGS = {
    0: dict(n_particles=50, pt="inv_uniform", eta_max=0.8, noise=0.0),
    1: dict(n_particles=6000, pt="exp", eta_max=1.2, noise=0.10),
    3: dict(n_particles=9000, pt="exp", eta_max=1.2, noise=0.20),
}


def generate_event(geom: Geometry, config: int = 1, seed: int = 0, *, n_particles=None,
                   noise=None, smear: bool = True, shuffle: bool = True) -> Event:
    """One event of BASELINE.json configs[0|1|3] (config 2 = config 1 with seeds 0..63).

    Draw order (fixed): z0 ~ N(0,5) [P]; charge [P]; pT variate [P]; phi0 ~ U(-pi,pi) [P];
    eta ~ U(-eta_max, eta_max) [P]; du ~ N(0,1) [P,6,2,3]; dz ~ N(0,1) [P,6,2,3];
    noise module, side, u, z-fraction [n_noise each]; final permutation of the hit order.
    """
    cfg = CONFIGS[config]
    P = cfg["n_particles"] if n_particles is None else int(n_particles)
    f_noise = cfg["noise"] if noise is None else float(noise)
    rng = np.random.Generator(np.random.PCG64(seed))
    z0 = rng.normal(0.0, 5.0, P)
    q = rng.integers(0, 2, P) * 2 - 1
    if cfg["pt"] == "inv_uniform":
        pt = 1.0 / rng.uniform(0.1, 1.0, P)
    else:
        pt = 0.6 + rng.exponential(0.7, P)
    phi0 = rng.uniform(-np.pi, np.pi, P)
    eta = rng.uniform(-cfg["eta_max"], cfg["eta_max"], P)
    du = rng.normal(0.0, 1.0, (P, N_LAYERS, 2, 3)) * SIGMA_RPHI
    dz = rng.normal(0.0, 1.0, (P, N_LAYERS, 2, 3)) * np.asarray(SIGMA_Z)[None, :, None, None]
    if not smear:
        du = np.zeros_like(du)
        dz = np.zeros_like(dz)
    x, y, z, mod, side, pid = propagate(geom, z0, q, pt, phi0, eta, du, dz)
    n_noise = int(math.floor(f_noise * len(x)))
    if n_noise:
        x, y, z, mod, side, pid = _append_noise(geom, rng, n_noise, x, y, z, mod, side, pid)
    if shuffle:
        perm = rng.permutation(len(x))
        x, y, z, mod, side, pid = (a[perm] for a in (x, y, z, mod, side, pid))
    return Event(x.astype(np.float32), y.astype(np.float32), z.astype(np.float32),
                 mod.astype(np.int32), side.astype(np.uint8), pid.astype(np.int32),
                 dict(z0=z0, q=q.astype(np.float64), pt=pt, phi0=phi0, eta=eta))


def _append_noise(geom, rng, n_noise, x, y, z, mod, side, pid):
    nm = rng.integers(0, geom.n_modules, n_noise)
    ns = rng.integers(0, 2, n_noise)
    nu = rng.uniform(-MODULE_HALF_W, MODULE_HALF_W, n_noise)
    nzf = rng.uniform(0.0, 1.0, n_noise)
    l = geom.layer[nm].astype(np.int64)
    rho = np.asarray(LAYER_R)[l] + (ns - 0.5) * np.asarray(SENSOR_GAP)[l]
    Phi = geom.phi[nm]
    nx = rho * np.cos(Phi) - nu * np.sin(Phi)
    ny = rho * np.sin(Phi) + nu * np.cos(Phi)
    nz = -Z_MAX + RING_LEN * (geom.ring[nm] + nzf)
    return (np.concatenate([x, nx]), np.concatenate([y, ny]), np.concatenate([z, nz]),
            np.concatenate([mod, nm.astype(np.int32)]), np.concatenate([side, ns.astype(np.uint8)]),
            np.concatenate([pid, np.full(n_noise, -1, np.int32)]))


def generate_occupancy_event(geom: Geometry, n_hits: int, seed: int = 0, track_fraction=0.5) -> Event:
    """BASELINE.json configs[4] (SURVEY.md reading #21): ``n_hits`` hits spread over the whole
    barrel, ``track_fraction`` of them from helices, the rest uniform noise.

    Track directions are chosen through a seed point uniform over (module, local position) so
    that large-|z| rings are populated too; pT / charge / z0 as in config 1.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    want = int(n_hits * track_fraction)
    xs, ys, zs, ms, ss, ps = [], [], [], [], [], []
    parts = dict(z0=[], q=[], pt=[], phi0=[], eta=[])
    got, base_pid = 0, 0
    while got < want:
        P = max(16, int((want - got) / 9.0) + 1)
        z0 = rng.normal(0.0, 5.0, P)
        q = rng.integers(0, 2, P) * 2 - 1
        pt = 0.6 + rng.exponential(0.7, P)
        sm = rng.integers(0, geom.n_modules, P)
        su = rng.uniform(-MODULE_HALF_W, MODULE_HALF_W, P)
        szf = rng.uniform(0.0, 1.0, P)
        l = geom.layer[sm].astype(np.int64)
        r_l = np.asarray(LAYER_R)[l]
        Phi = geom.phi[sm]
        px = r_l * np.cos(Phi) - su * np.sin(Phi)
        py = r_l * np.sin(Phi) + su * np.cos(Phi)
        pz = -Z_MAX + RING_LEN * (geom.ring[sm] + szf)
        r = np.hypot(px, py)
        R = pt / (K_GEV_PER_T_CM * B_TESLA)
        ok = r < 2 * R
        half = np.arcsin(np.where(ok, r / (2 * R), 0.0))
        s = -q.astype(np.float64)
        phi0 = np.arctan2(py, px) - s * half          # position azimuth = phi0 + s*asin(r/2R)
        arc = 2 * R * half
        eta = np.arcsinh((pz - z0) / np.where(ok, arc, 1.0))
        z0, q, pt, phi0, eta = (a[ok] for a in (z0, q, pt, phi0, eta))
        Pk = len(pt)
        du = rng.normal(0.0, 1.0, (Pk, N_LAYERS, 2, 3)) * SIGMA_RPHI
        dz = rng.normal(0.0, 1.0, (Pk, N_LAYERS, 2, 3)) * np.asarray(SIGMA_Z)[None, :, None, None]
        x, y, z, mod, side, pid = propagate(geom, z0, q, pt, phi0, eta, du, dz)
        if got + len(x) > want:                       # trim whole particles to hit the target
            keep = np.nonzero(np.cumsum(np.bincount(pid, minlength=Pk)) <= (want - got))[0]
            npart = len(keep)
            m = pid < npart
            x, y, z, mod, side, pid = (a[m] for a in (x, y, z, mod, side, pid))
            z0, q, pt, phi0, eta = (a[:npart] for a in (z0, q, pt, phi0, eta))
            want = got + len(x)                       # terminate
        xs.append(x); ys.append(y); zs.append(z); ms.append(mod); ss.append(side)
        ps.append(pid + base_pid)
        for k, v in zip(("z0", "q", "pt", "phi0", "eta"), (z0, q.astype(np.float64), pt, phi0, eta)):
            parts[k].append(v)
        got += len(x)
        base_pid += len(pt)
    x, y, z, mod, side, pid = (np.concatenate(a) if a else np.zeros(0) for a in (xs, ys, zs, ms, ss, ps))
    n_noise = max(0, n_hits - len(x))
    if n_noise:
        x, y, z, mod, side, pid = _append_noise(geom, rng, n_noise, x, y, z, mod, side, pid)
    perm = rng.permutation(len(x))
    x, y, z, mod, side, pid = (a[perm] for a in (x, y, z, mod, side, pid))
    return Event(x.astype(np.float32), y.astype(np.float32), z.astype(np.float32),
                 mod.astype(np.int32), side.astype(np.uint8), pid.astype(np.int32),
                 {k: np.concatenate(v) if v else np.zeros(0) for k, v in parts.items()})


def single_helix_event(geom: Geometry, pt, q, phi0, eta, z0, smear: bool = False, seed: int = 0) -> Event:
    """Hits of explicitly given helices (scalars or arrays); noiseless unless ``smear``."""
    pt, q, phi0, eta, z0 = (np.atleast_1d(np.asarray(a, dtype=np.float64)) for a in (pt, q, phi0, eta, z0))
    P = len(pt)
    du = dz = None
    if smear:
        rng = np.random.Generator(np.random.PCG64(seed))
        du = rng.normal(0.0, 1.0, (P, N_LAYERS, 2, 3)) * SIGMA_RPHI
        dz = rng.normal(0.0, 1.0, (P, N_LAYERS, 2, 3)) * np.asarray(SIGMA_Z)[None, :, None, None]
    x, y, z, mod, side, pid = propagate(geom, z0, q, pt, phi0, eta, du, dz)
    return Event(x.astype(np.float32), y.astype(np.float32), z.astype(np.float32),
                 mod.astype(np.int32), side.astype(np.uint8), pid.astype(np.int32),
                 dict(z0=z0, q=q, pt=pt, phi0=phi0, eta=eta))


def transform_event(ev: Event, rot: float = 0.0, mirror_z: bool = False) -> Event:
    """Rotate all hits about the beam axis by ``rot`` (module ids unchanged: only meaningful for
    cut-variable invariance checks with a map that is not re-derived) or mirror z -> -z."""
    c, s = math.cos(rot), math.sin(rot)
    x = (ev.x.astype(np.float64) * c - ev.y.astype(np.float64) * s).astype(np.float32)
    y = (ev.x.astype(np.float64) * s + ev.y.astype(np.float64) * c).astype(np.float32)
    z = -ev.z if mirror_z else ev.z.copy()
    return Event(x, y, z, ev.module.copy(), ev.side.copy(), ev.truth.copy(), ev.particles)


# ----------------------------------------------------------------------------------------
# Pixel line segments: inner-tracker seeds.  The CMS seeds are not available; this is a stand-in seed
# model: every generated particle above the seeding threshold gives, with some efficiency, the
# inner tracker's ESTIMATE of its helix -- the true parameters smeared with fixed resolutions -- plus fake seeds with
# random parameters.  Input data only: the consistency selection [P] is in the oracle and in the CUDA library.
# ----------------------------------------------------------------------------------------
SEED_PT_MIN = 0.8
SEED_EFFICIENCY = 0.9
SEED_FAKE_FRACTION = 0.2
SEED_SIGMA_KAPPA_REL = 0.01          # relative curvature (pT) resolution ...
SEED_SIGMA_KAPPA_ABS = 2.0e-5        # ... and its floor, cm^-1
SEED_SIGMA_PHI = 5.0e-4              # rad
SEED_SIGMA_Z0 = 0.01                 # cm
SEED_SIGMA_T = 1.0e-3                # cot(theta)


@dataclasses.dataclass
class Seeds:
    """Pixel line segments as the library receives them (fp32 SoA) + generator truth."""
    kappa: np.ndarray        # signed curvature, cm^-1; sign convention of the triplet curvature: -q / R
    cphi: np.ndarray         # cos / sin of the azimuth of the momentum at the beam line
    sphi: np.ndarray
    z0: np.ndarray           # z at the beam line, cm
    t: np.ndarray            # cot(theta) = sinh(eta) = dz / d(transverse arc length)
    truth: np.ndarray        # int32 particle index, -1 = fake seed

    @property
    def n(self) -> int:
        return int(self.kappa.shape[0])

    def arrays(self):
        return self.kappa, self.cphi, self.sphi, self.z0, self.t


def generate_seeds(ev: Event, seed: int = 0, *, efficiency=SEED_EFFICIENCY, fake_fraction=SEED_FAKE_FRACTION, smear: bool = True,
                   shuffle: bool = True) -> Seeds:
    """Draw order (fixed; generator PCG64(seed + 7919)): kept mask [P]; smearing of kappa, phi0, z0, t [n_true each];
    fake kappa, phi0, z0, eta [n_fake each]; final permutation."""
    rng = np.random.Generator(np.random.PCG64(seed + 7919))
    par = ev.particles
    P = len(par["pt"])
    keep = (par["pt"] >= SEED_PT_MIN) & (rng.uniform(0.0, 1.0, P) < efficiency)
    idx = np.nonzero(keep)[0]
    n = len(idx)
    R = par["pt"][idx] / (K_GEV_PER_T_CM * B_TESLA)
    kappa = -par["q"][idx] / R
    phi0, z0, t = par["phi0"][idx].copy(), par["z0"][idx].copy(), np.sinh(par["eta"][idx])
    g = rng.normal(0.0, 1.0, (4, n))
    if smear:
        kappa = kappa + g[0] * np.hypot(SEED_SIGMA_KAPPA_REL * kappa, SEED_SIGMA_KAPPA_ABS)
        phi0 = phi0 + g[1] * SEED_SIGMA_PHI
        z0 = z0 + g[2] * SEED_SIGMA_Z0
        t = t + g[3] * SEED_SIGMA_T
    n_fake = int(math.floor(fake_fraction * n))
    kmax = K_GEV_PER_T_CM * B_TESLA / SEED_PT_MIN
    fk = rng.uniform(-kmax, kmax, n_fake)
    fp = rng.uniform(-np.pi, np.pi, n_fake)
    fz = rng.normal(0.0, 5.0, n_fake)
    ft = np.sinh(rng.uniform(-1.2, 1.2, n_fake))
    kappa, phi0, z0, t = (np.concatenate(a) for a in ((kappa, fk), (phi0, fp), (z0, fz), (t, ft)))
    truth = np.concatenate([idx.astype(np.int32), np.full(n_fake, -1, np.int32)])
    if shuffle:
        perm = rng.permutation(len(kappa))
        kappa, phi0, z0, t, truth = (a[perm] for a in (kappa, phi0, z0, t, truth))
    f = lambda a: np.ascontiguousarray(a, np.float32)
    return Seeds(f(kappa), f(np.cos(phi0)), f(np.sin(phi0)), f(z0), f(t), truth.astype(np.int32))
