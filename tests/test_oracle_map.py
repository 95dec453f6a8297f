"""Pins of the oracle's module-map builder [B] (DESIGN.md section 1 [B], reading 25).  The paper verifies
its map "using simulated samples" and so does P15; the others are an independent implementation on the
BASELINE geometry, symmetries and monotonicity."""
import math

import numpy as np
import pytest

from paper_2207_08207_b200 import synth


def as_set(offs, tg):
    src = np.repeat(np.arange(len(offs) - 1), np.diff(offs))
    return set(zip(src.tolist(), tg.tolist()))


def build(o, mg, **kw):
    return o.build_map(mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"], **kw)


def test_p15_simulated_tracks_stay_inside_the_map(o64, geom):
    """PAPER.md:49 "This map was then verified using simulated samples": every pair of hits that one simulated particle
    with pT >= 0.8 GeV and |z0| <= 15 cm leaves on the lower sensors of consecutive layers sits on connected modules."""
    conn = as_set(*build(o64, synth.map_geometry(geom)))
    n_pairs = 0
    for seed in (200, 201, 202):
        ev = synth.generate_event(geom, 1, seed, n_particles=3000)
        pt, z0 = ev.particles["pt"], ev.particles["z0"]
        ok = (ev.truth >= 0) & (ev.side == 0)
        ok[ok] &= (pt[ev.truth[ok]] >= 0.8) & (np.abs(z0[ev.truth[ok]]) <= 15.0)
        mod, pid = ev.module[ok], ev.truth[ok]
        lay = geom.layer[mod]
        for p in np.unique(pid):
            m = mod[pid == p]
            l = lay[pid == p]
            for a in range(len(m)):
                for b in range(len(m)):
                    if l[b] == l[a] + 1:
                        n_pairs += 1
                        assert (int(m[a]), int(m[b])) in conn, (seed, p, m[a], m[b])
    assert n_pairs > 20000


def test_p16_equals_the_test_side_generator_on_the_baseline_geometry(o64, geom, mmap):
    offs, tg = build(o64, synth.map_geometry(geom))
    assert len(tg) == 69630
    assert np.array_equal(offs, mmap.row_offsets) and np.array_equal(tg, mmap.targets)
    assert np.all(geom.layer[tg] == geom.layer[np.repeat(np.arange(geom.n_modules), np.diff(offs))] + 1)
    for a in range(0, geom.n_modules, 97):          # rows ascending
        assert np.all(np.diff(tg[offs[a]:offs[a + 1]]) > 0)


def test_p17_symmetries_and_monotonicity(o64, geom):
    mg = synth.map_geometry(geom)
    base = as_set(*build(o64, mg))
    rot = dict(mg, phi=mg["phi"] + 0.7318)                                    # a rotation about z changes nothing
    assert as_set(*build(o64, rot)) == base
    mir = dict(mg, zlo=-mg["zhi"], zhi=-mg["zlo"])                             # z -> -z: the same map on the mirrored rings
    ring_mirror = {}
    for l in range(6):
        ids = np.nonzero(geom.layer == l)[0]
        nphi = len(ids) // 24
        for k, m in enumerate(ids):
            r, i = divmod(k, nphi)
            ring_mirror[int(m)] = int(ids[(23 - r) * nphi + i])
    assert {(ring_mirror[a], ring_mirror[b]) for a, b in base} == as_set(*build(o64, mir))
    assert as_set(*build(o64, mg, pt_min=1.0)) < base < as_set(*build(o64, mg, pt_min=0.6))      # softer tracks bend more
    assert as_set(*build(o64, mg, z0_max=5.0)) < base and as_set(*build(o64, mg, pad_phi=0.0, pad_z=0.0)) < base
    # straight-line limit: no bending allowance left, only the geometric overlap of the two modules seen from the beam line
    stiff = as_set(*build(o64, mg, pt_min=1e6, pad_phi=0.0))
    a, b = np.array(sorted(stiff)).T
    d = np.abs(np.angle(np.exp(1j * (mg["phi"][b] - mg["phi"][a]))))
    assert np.all(d <= np.arctan(4.8 / (mg["rho"][a] - mg["gap"][a] / 2)) + np.arctan(4.8 / (mg["rho"][b] - mg["gap"][b] / 2)) + 1e-12)


# ----------------------------------------------------------------------------------------
# P18: two-module special cases with textbook answers
# ----------------------------------------------------------------------------------------
def _two_modules(phi_b, zb_lo, zb_hi, za=(40.0, 50.0)):
    """A on layer 0 (rho 23.0, gap 0.26) at azimuth 0; B on layer 1 (rho 35.7, gap 0.26); half width 4.8 both."""
    return dict(layer=np.array([0, 1], np.int8), phi=np.array([0.0, phi_b]), rho=np.array([23.0, 35.7]), gap=np.array([0.26, 0.26]),
                hw=np.array([4.8, 4.8]), zlo=np.array([za[0], zb_lo]), zhi=np.array([za[1], zb_hi]))


def _connected(o64, mg, **kw):
    offs, tg = build(o64, mg, **kw)
    assert list(offs) in ([0, 0, 0], [0, 1, 1]) and list(tg) in ([], [1])
    return len(tg) == 1


@pytest.mark.parametrize("pad_z", [0.0, 1.0, 2.5])
def test_p18_z_envelope_by_similar_triangles_and_arc_lengths(o64, pad_z):
    """The z side of B4 on two modules facing each other, where the answer is elementary.  A spans z in [40, 50] (+- pad_z).
    (i) Straight tracks from the origin (pt_min -> infinity, z0_max = 0): similar triangles, z' = z_A r'/r_A, so B is
    reached iff its z range meets [(40 - pad) r'_lo / r_hi, (50 + pad) r'_hi / r_lo] -- the extreme radii being the near
    face centre (r_lo = rho - gap/2) and the far corner (r_hi = hypot(rho + gap/2, hw)) of each module.
    (ii) Straight tracks from |z0| <= 15: the line through (0, z0) and (r_A, z_A) read at r'.
    (iii) Helices at pt_min: z advances with the arc length s(r) = 2R asin(r / 2R), so the largest lever arm is
    asin(r'_hi / 2R) / asin(r_lo / 2R) at R = pt_min / (k B); the smallest stays the straight-line one."""
    r_lo, r_hi = 23.0 - 0.13, math.hypot(23.0 + 0.13, 4.8)
    rp_lo, rp_hi = 35.7 - 0.13, math.hypot(35.7 + 0.13, 4.8)
    k_min, k_straight = rp_lo / r_hi, rp_hi / r_lo
    R = 0.8 / (synth.K_GEV_PER_T_CM * synth.B_TESLA)
    k_helix = math.asin(rp_hi / (2 * R)) / math.asin(r_lo / (2 * R))
    assert k_helix > k_straight > k_min > 1.0
    cases = (dict(pt_min=1e9, z0_max=0.0, lo=(40 - pad_z) * k_min, hi=(50 + pad_z) * k_straight),
             dict(pt_min=1e9, z0_max=15.0, lo=15 + (40 - pad_z - 15) * k_min, hi=-15 + (50 + pad_z + 15) * k_straight),
             dict(pt_min=0.8, z0_max=15.0, lo=15 + (40 - pad_z - 15) * k_min, hi=-15 + (50 + pad_z + 15) * k_helix),
             dict(pt_min=0.8, z0_max=0.0, lo=(40 - pad_z) * k_min, hi=(50 + pad_z) * k_helix))
    for c in cases:
        kw = dict(pt_min=c["pt_min"], z0_max=c["z0_max"], pad_z=pad_z, pad_phi=0.0)
        for eps, want in ((-1e-6, True), (+1e-6, False)):
            # B just below the upper end of the envelope / just above it
            assert _connected(o64, _two_modules(0.0, c["hi"] * (1 + eps), c["hi"] * (1 + eps) + 10.0), **kw) == want, (c, eps)
            # B just above the lower end / just below it
            assert _connected(o64, _two_modules(0.0, c["lo"] * (1 - eps) - 10.0, c["lo"] * (1 - eps)), **kw) == want, (c, eps)
        assert _connected(o64, _two_modules(0.0, 0.5 * (c["lo"] + c["hi"]) - 5, 0.5 * (c["lo"] + c["hi"]) + 5), **kw)
    # mirrored module: the same numbers with the sign of z flipped
    c = cases[2]
    kw = dict(pt_min=0.8, z0_max=15.0, pad_z=pad_z, pad_phi=0.0)
    for eps, want in ((-1e-6, True), (+1e-6, False)):
        assert _connected(o64, _two_modules(0.0, -c["hi"] * (1 + eps) - 10.0, -c["hi"] * (1 + eps), za=(-50.0, -40.0)), **kw) == want


def test_p18_azimuth_envelope(o64):
    """The azimuth side (B3): half widths seen from the beam line + the bending of the tightest helix between the
    smallest radius of A and the largest of B (azimuth of a helix point = phi0 -+ asin(r / 2R)) + pad, across the
    +-pi cut."""
    r_lo, rp_lo, rp_hi = 23.0 - 0.13, 35.7 - 0.13, math.hypot(35.7 + 0.13, 4.8)
    for pt_min, pad in ((0.8, 0.0), (0.8, 0.01), (1e9, 0.0), (2.0, 0.05)):
        R = pt_min / (synth.K_GEV_PER_T_CM * synth.B_TESLA)
        tol = math.atan(4.8 / r_lo) + math.atan(4.8 / rp_lo) + (math.asin(rp_hi / (2 * R)) - math.asin(r_lo / (2 * R))) + pad
        for sign in (+1, -1):
            for eps, want in ((-1e-9, True), (+1e-9, False)):
                mg = _two_modules(sign * tol * (1 + eps), 60.0, 70.0)
                assert _connected(o64, mg, pt_min=pt_min, pad_phi=pad) == want, (pt_min, pad, sign, eps)
                mg["phi"] = mg["phi"] + 3.0                                      # B lands beyond +pi: wrapped difference
                assert _connected(o64, mg, pt_min=pt_min, pad_phi=pad) == want


# ----------------------------------------------------------------------------------------
# P19: helices from the edges of a module, as the paper words the derivation
# ----------------------------------------------------------------------------------------
def _edge_helices(geom, A, pad_z, pts, z0s):
    """Helices (pt, q, phi0, eta, z0) that pass through the corners, edge midpoints and face centres of both sensors of
    module A (its z range widened by pad_z), for every pT in pts, both charges, every z0 in z0s."""
    l = int(geom.layer[A])
    Phi = geom.phi[A]
    zlo = -synth.Z_MAX + synth.RING_LEN * geom.ring[A]
    out = []
    for side in (0, 1):
        rho = synth.LAYER_R[l] + (side - 0.5) * synth.SENSOR_GAP[l]
        for u in (-synth.MODULE_HALF_W, 0.0, synth.MODULE_HALF_W):
            x, y = rho * math.cos(Phi) - u * math.sin(Phi), rho * math.sin(Phi) + u * math.cos(Phi)
            r = math.hypot(x, y)
            for z in (zlo - pad_z, zlo + 0.5 * synth.RING_LEN, zlo + synth.RING_LEN + pad_z):
                for pt in pts:
                    R = pt / (synth.K_GEV_PER_T_CM * synth.B_TESLA)
                    half = math.asin(r / (2 * R))
                    for q in (-1.0, 1.0):
                        for z0 in z0s:
                            # azimuth of a helix point = phi0 + s asin(r / 2R), s = -q; z = z0 + sinh(eta) 2R asin(r / 2R)
                            out.append((pt, q, math.atan2(y, x) + q * half, math.asinh((z - z0) / (2 * R * half)), z0))
    return np.array(out).T


@pytest.mark.parametrize("pads", [(0.0, 0.0), (0.01, 1.0)])
def test_p19_helices_from_the_module_edges(o64, geom, pads):
    """"computing the possible track trajectories as helices that can start from the edges of a given module
    that are compatible with the pT threshold, and then listing all the modules in the adjacent layer that intersect
    these helices".  Done literally, by propagation (the generator's closed-form helix / plane intersections) instead of
    the envelope formula: for source modules in every layer and ring, helices through the edges of both sensors with
    pT from the threshold up, both charges, |z0| up to z0_max.  SOUNDNESS: every module of the next layer such a helix
    crosses is in the oracle's row.  TIGHTNESS: every module in the row is such a module or its neighbour (one ring,
    one azimuth step), i.e. the envelope adds no more than its stated slack."""
    pad_phi, pad_z = pads
    mg = synth.map_geometry(geom)
    offs, tg = build(o64, mg, pad_phi=pad_phi, pad_z=pad_z)
    pts = (0.8, 0.8001, 0.9, 1.2, 2.0, 5.0, 1e4)
    z0s = (-15.0, 0.0, 15.0)
    n_reached = n_rows = 0
    for l in range(5):
        nphi, nphi_b = int(geom.n_phi[l]), int(geom.n_phi[l + 1])
        for ring in range(24):
            for i in (0, nphi // 3):
                A = int(geom.base[l]) + ring * nphi + i
                pt, q, phi0, eta, z0 = _edge_helices(geom, A, pad_z, pts, z0s)
                _, _, _, mod, _, _ = synth.propagate(geom, z0, q, pt, phi0, eta)
                reached = np.unique(mod[geom.layer[mod] == l + 1])
                row = tg[offs[A]:offs[A + 1]]
                assert np.isin(reached, row).all(), (A, sorted(set(reached.tolist()) - set(row.tolist())))
                # tightness
                rr, ri = geom.ring[reached], geom.iphi[reached]
                for B in row:
                    dring = np.abs(rr - geom.ring[B])
                    di = np.abs(ri - geom.iphi[B])
                    di = np.minimum(di, nphi_b - di)
                    assert ((dring <= 1) & (di <= 1)).any(), (A, int(B))
                n_reached += len(reached)
                n_rows += len(row)
    assert n_reached > 2000 and n_rows >= n_reached
