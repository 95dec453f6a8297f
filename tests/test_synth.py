"""Input generator: shapes, determinism and the sizes BASELINE.json / SURVEY.md 8(a) state."""
import numpy as np

from paper_2207_08207_b200 import synth


def test_geometry_counts(geom):
    # BASELINE.json configs[0]: ceil(2*pi*r/9.6)+1 modules per ring, 24 rings -> 6120 modules
    assert list(geom.n_phi) == [17, 25, 35, 46, 60, 72]
    assert geom.n_modules == 6120
    assert list(geom.base) == [0, 408, 1008, 1848, 2952, 4392]
    assert geom.layer.min() == 0 and geom.layer.max() == 5
    assert np.all(geom.kind == (geom.layer >= 3))


def test_module_map_shape(geom, mmap):
    # 69 630 entries, targets in the next layer, rows sorted ascending
    assert mmap.row_offsets[0] == 0 and mmap.row_offsets[-1] == len(mmap.targets) == 69630
    src = np.repeat(np.arange(geom.n_modules), np.diff(mmap.row_offsets))
    assert np.all(geom.layer[mmap.targets] == geom.layer[src] + 1)
    for m in (0, 407, 1500, 4391):
        row = mmap.targets[mmap.row_offsets[m]:mmap.row_offsets[m + 1]]
        assert np.all(np.diff(row) > 0)
    assert np.all(np.diff(mmap.row_offsets)[geom.layer == 5] == 0)


def test_events_deterministic_and_sized(geom):
    a = synth.generate_event(geom, 0, 0)
    b = synth.generate_event(geom, 0, 0)
    for f in ("x", "y", "z", "module", "side", "truth"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert 550 <= a.n <= 700                      # "about 600 hits"
    assert a.x.dtype == np.float32 and a.module.dtype == np.int32 and a.side.dtype == np.uint8
    c1 = synth.generate_event(geom, 1, 0)
    assert 70000 <= c1.n <= 85000                 # SURVEY.md reading #19: ~78 k
    assert abs((c1.truth < 0).mean() - 0.10 / 1.10) < 0.005
    other = synth.generate_event(geom, 1, 1)
    assert other.n != c1.n or not np.array_equal(other.x, c1.x)


def test_hits_lie_on_their_sensor_plane(geom):
    ev = synth.generate_event(geom, 1, 3, n_particles=300)
    phi = geom.phi[ev.module]
    lay = geom.layer[ev.module].astype(int)
    rho = np.asarray(synth.LAYER_R)[lay] + (ev.side.astype(float) - 0.5) * np.asarray(synth.SENSOR_GAP)[lay]
    w = ev.x * np.cos(phi) + ev.y * np.sin(phi)
    u = -ev.x * np.sin(phi) + ev.y * np.cos(phi)
    assert np.max(np.abs(w - rho)) < 2e-5 * 110
    assert np.max(np.abs(u)) < synth.MODULE_HALF_W + 6 * synth.SIGMA_RPHI


def test_occupancy_event_size(geom):
    ev = synth.generate_occupancy_event(geom, 10000, seed=1)
    assert ev.n == 10000
    frac = (ev.truth >= 0).mean()
    assert 0.45 <= frac <= 0.55
