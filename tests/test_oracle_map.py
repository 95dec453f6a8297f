"""Pins of the oracle's module-map builder [B] (DESIGN.md section 1 [B], reading 25).  The paper verifies
its map "using simulated samples" and so does P15; the others are an independent implementation on the
BASELINE geometry, symmetries and monotonicity."""
import numpy as np

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
