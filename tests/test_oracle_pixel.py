"""Pins of the oracle's pixel-link selection [P] (lsto_pix_cut, lsto_pixel_link; DESIGN.md section 1 [P]; PAPER.md:39, :63
"the estimates from the pixel detector are used and the consistency of the outer hits to this hypothesis is checked").

P22  closed forms on noiseless helices: with the true parameters as the seed every x-y residual vanishes, the r-z residual is
     the remainder of the arc-length series, and the curvature difference is zero; with ONE seed parameter displaced each
     residual has a closed form (delta kappa r^2 / 2; kappa r^2 / 2 + r sin(delta - asin(kappa r / 2)); -delta z0; -delta t s).
P23  textbook reductions on generic points: e(p) is the signed distance from the seed's circle times (1 + kappa d / 2)
     (distance by numpy.hypot from the circle's centre); the arc length is (2 / kappa) asin(kappa r / 2) within the stated
     series remainder; the chi2 sums are numpy dot products with the per-layer weights.
P24  brute force + structure: Python enumeration of every (object, seed) pair == the driver; candidates = product.
P25  per-layer weight indices and per-kind thresholds: closing one entry removes exactly the links it governs.
P26  truth: links of a seed with the objects of its own particle pass (>= 99.5 %); fake seeds produce almost nothing.
"""
import math

import numpy as np
import pytest

from paper_2207_08207_b200 import synth

from test_oracle_pins import clean_helix, md_tuple, KB

SERIES = (0.16666667, 0.075, 0.04464286, 0.030381944, 0.022372158)      # as typed in the SPEC: 1/6, 3/40, 15/336, 105/3456, 945/42240 to binary32
assert all(abs(a - b) < 1e-8 for a, b in zip(SERIES, (1 / 6, 3 / 40, 15 / 336, 105 / 3456, 945 / 42240)))
VAR_XY = [(1.0e-3 * r) ** 2 + (1.0e-4 * r * r / 2) ** 2 + 0.0026 ** 2 for r in synth.LAYER_R]          # nominal seed resolutions
VAR_RZ = [sz ** 2 + 0.02 ** 2 + (2.0e-3 * r) ** 2 for r, sz in zip(synth.LAYER_R, synth.SIGMA_Z)]


def helix_seed(h):
    """The exact seed of a generated helix: (kappa, cos phi0, sin phi0, z0, t)."""
    return [-h["q"] / h["R"], math.cos(h["phi0"]), math.sin(h["phi0"]), h["z0"], math.sinh(h["eta"])]


def open_cfg(o):
    cfg = o.default_config()
    for k in range(2):
        cfg.pix_dkappa_max[k] = cfg.pix_chi2xy_max[k] = cfg.pix_chi2rz_max[k] = 1e30
    return cfg


def test_p22_closed_forms_on_helices(geom, o64):
    rng = np.random.default_rng(22)
    cfg = open_cfg(o64)
    w_xy, w_rz = np.array(o64.config_dict()["pix_inv_var_xy"]), np.array(o64.config_dict()["pix_inv_var_rz"])
    assert np.allclose(w_xy, 1 / np.array(VAR_XY), rtol=1e-6) and np.allclose(w_rz, 1 / np.array(VAR_RZ), rtol=1e-6)   # the constants table
    for _ in range(40):
        h, mds = clean_helix(geom, rng)
        t = [md_tuple(o64, l, mds[l])[0] for l in range(6)]
        seed = helix_seed(h)
        kappa, tt = seed[0], seed[4]
        for kind, n in ((0, 3), (1, 5)):
            for l in range(2):
                pts = [t[l + k][:4] for k in range(n)]
                r = np.array([p[3] for p in pts])
                s_true = (2 / kappa) * np.arcsin(kappa * r / 2)
                u2 = (kappa * r / 2) ** 2
                s_ser = r * (1 + u2 * (SERIES[0] + u2 * (SERIES[1] + u2 * (SERIES[2] + u2 * (SERIES[3] + u2 * SERIES[4])))))
                w1, w2 = w_xy[l:l + n], w_rz[l:l + n]
                ok, out, mar = o64.pix_cut(kind, l, seed, kappa, pts, cfg=cfg)
                assert ok and abs(out["dkappa"]) == 0.0
                assert out["chi2xy"] < 1e-14                                              # on the circle: e_i = 0
                assert out["chi2rz"] == pytest.approx(np.sum((tt * (s_true - s_ser)) ** 2 * w2), rel=1e-5, abs=1e-16)
                assert np.all(np.abs(s_true - s_ser) <= 0.035 * u2 ** 6 * r + 1e-8 * u2 * r + 1e-12)   # the stated remainder (+ the coefficients' rounding)
                # one parameter displaced at a time
                dk, dphi, dz, dt = 3e-5, 7e-4, 0.03, 1.5e-3
                _, o1, _ = o64.pix_cut(kind, l, [kappa + dk] + seed[1:], kappa, pts, cfg=cfg)
                assert o1["dkappa"] == pytest.approx(-dk, rel=1e-9)
                assert o1["chi2xy"] == pytest.approx(np.sum((dk * r * r / 2) ** 2 * w1), rel=1e-6)
                ph = h["phi0"] + dphi
                _, o2, _ = o64.pix_cut(kind, l, [kappa, math.cos(ph), math.sin(ph)] + seed[3:], kappa, pts, cfg=cfg)
                e = kappa * r * r / 2 + r * np.sin(dphi - np.arcsin(kappa * r / 2))
                assert o2["chi2xy"] == pytest.approx(np.sum(e * e * w1), rel=1e-6)
                _, o3, _ = o64.pix_cut(kind, l, seed[:3] + [seed[3] + dz, tt], kappa, pts, cfg=cfg)
                assert o3["chi2rz"] == pytest.approx(np.sum((tt * (s_true - s_ser) - dz) ** 2 * w2), rel=1e-6)
                _, o4, _ = o64.pix_cut(kind, l, seed[:4] + [tt + dt], kappa, pts, cfg=cfg)
                assert o4["chi2rz"] == pytest.approx(np.sum((tt * (s_true - s_ser) - dt * s_ser) ** 2 * w2), rel=1e-6)
        # P1 against the objects' own curvatures: the triplet's circumcurvature and the quintuplet's fit equal the seed's
        ok, o3_, _ = o64.t3_cut(0, t[0][:4], t[1][:4], t[2][:4])
        assert ok and o3_["kappa"] == pytest.approx(kappa, rel=1e-8)


def test_p23_distance_from_the_circle_and_arc_length(o64):
    """Generic (off-circle) points: e(p) = d (1 + kappa d / 2) with d the signed distance of p from the seed's circle, centre
    (-sin phi0, cos phi0) / kappa, radius 1 / |kappa| -- an identity, checked against numpy.hypot; chi2 sums as dot products."""
    rng = np.random.default_rng(23)
    cfg = open_cfg(o64)
    d_ = o64.config_dict()
    for _ in range(300):
        kind = int(rng.integers(0, 2)); n = 5 if kind else 3; l = int(rng.integers(0, 2))
        kappa = rng.uniform(0.0005, 0.014) * rng.choice([-1, 1]); phi0 = rng.uniform(-np.pi, np.pi)
        z0, tt = rng.normal(0, 5), rng.uniform(-1.5, 1.5)
        pts = []
        for k in range(n):
            r = synth.LAYER_R[l + k] + rng.uniform(-0.2, 0.5)
            a = phi0 + math.asin(kappa * r / 2) + rng.normal(0, 0.01)              # near the circle, not on it
            pts.append((r * math.cos(a), r * math.sin(a), rng.uniform(-100, 100), r))
        ok, out, _ = o64.pix_cut(kind, l, [kappa, math.cos(phi0), math.sin(phi0), z0, tt], 0.0, pts, cfg=cfg)
        assert ok
        xy = np.array([p[:2] for p in pts]); r = np.array([p[3] for p in pts]); z = np.array([p[2] for p in pts])
        centre = np.array([-math.sin(phi0), math.cos(phi0)]) / kappa
        dist = (np.hypot(*(xy - centre).T) - 1 / abs(kappa)) * np.sign(kappa)      # signed: positive outside for kappa > 0
        e = dist * (1 + kappa * dist / 2)
        assert out["chi2xy"] == pytest.approx(np.dot(e * e, d_["pix_inv_var_xy"][l:l + n]), rel=1e-7)
        s = (2 / kappa) * np.arcsin(kappa * r / 2)
        dz = z - z0 - tt * s
        rem = (0.035 * (kappa * r / 2) ** 12 + 1e-8 * (kappa * r / 2) ** 2) * r * abs(tt)   # what the series may be off by, per point
        lo = np.dot((np.abs(dz) - rem).clip(0) ** 2, d_["pix_inv_var_rz"][l:l + n])
        hi = np.dot((np.abs(dz) + rem) ** 2, d_["pix_inv_var_rz"][l:l + n])
        assert lo * (1 - 1e-9) <= out["chi2rz"] <= hi * (1 + 1e-9)


def test_p22b_the_returning_arc_is_excluded(geom, o64):
    """P0: a seed pointing the opposite way describes the same straight line (for a circle: its returning arc), so the x-y
    residuals of a stiff track vanish for it too; the forward requirement on the first anchor rejects it."""
    rng = np.random.default_rng(27)
    cfg = open_cfg(o64)
    n = 0
    for _ in range(20):
        h, mds = clean_helix(geom, rng, pt_lo=200.0, pt_hi=1000.0, eta_max=0.05)
        t = [md_tuple(o64, l, mds[l])[0] for l in range(6)]
        seed = helix_seed(h)
        back = [seed[0], -seed[1], -seed[2], seed[3], seed[4]]
        pts = [t[k][:4] for k in range(5)]
        ok, out, mar = o64.pix_cut(1, 0, seed, seed[0], pts, cfg=cfg)
        assert ok and out["chi2xy"] < 1e-12
        cfg2 = open_cfg(o64)
        ok_back, _, _ = o64.pix_cut(1, 0, back, seed[0], pts, cfg=cfg2)
        assert not ok_back
        e_back = [(back[0] / 2) * p[3] ** 2 + p[0] * back[2] - p[1] * back[1] for p in pts]
        assert max(abs(e) for e in e_back) < 0.6            # the residuals alone would not have rejected it (stiff track: 2 kappa r^2 / 2)
        n += 1
    assert n == 20


@pytest.fixture(scope="module")
def small(geom, o32, run_oracle):
    ev = synth.generate_event(geom, 1, 5, n_particles=1200)
    sd = synth.generate_seeds(ev, 5)
    return ev, sd, run_oracle(o32, ev, seeds=sd.arrays())


def test_p24_brute_force_and_structure(geom, o32, run_oracle):
    ev = synth.generate_event(geom, 0, 0, n_particles=16)
    sd = synth.generate_seeds(ev, 3, efficiency=1.0, fake_fraction=1.0)
    r = run_oracle(o32, ev, seeds=sd.arrays())
    lay = geom.layer[r.md_module]
    anchors = np.stack([r.md_x, r.md_y, r.md_z, r.md_r], 1)
    for kind, mds, kobj in ((0, r.t3_mds(), r.t3_kappa), (1, r.t5_mds(), r.t5_kfit)):
        want, n_cand = [], 0
        for o in range(len(mds)):
            if lay[mds[o][0]] > 1:
                continue
            for s in range(sd.n):
                n_cand += 1
                seed = [sd.kappa[s], sd.cphi[s], sd.sphi[s], sd.z0[s], sd.t[s]]
                if o32.pix_cut(kind, int(lay[mds[o][0]]), seed, kobj[o], anchors[mds[o]].tolist())[0]:
                    want.append((s, o))
        d = r.pix[kind]
        assert d["candidates"] == n_cand and list(zip(d["seed"].tolist(), d["obj"].tolist())) == sorted(want, key=lambda so: (so[1], so[0]))
        assert d["n"] > 10
        assert r.pix_tuples(kind).shape == (d["n"], 11 if kind else 7)


P25_CASES = ([("pix_inv_var_xy", l, kind) for l in range(6) for kind in (0, 1)] + [("pix_inv_var_rz", l, kind) for l in range(6) for kind in (0, 1)] +
             [(f, k, k) for f in ("pix_dkappa_max", "pix_chi2xy_max", "pix_chi2rz_max") for k in (0, 1)])


@pytest.mark.parametrize("field,idx,kind", P25_CASES)
def test_p25_weight_and_threshold_indices(geom, o32, run_oracle, small, field, idx, kind):
    """An astronomically large weight for layer l fails every link whose outer object has an anchor in layer l (its residual
    there is never exactly zero) and no other; a closed per-kind threshold removes every link of that kind and none of the other."""
    ev, sd, base = small
    cfg = o32.default_config()
    getattr(cfg, field)[idx] = 1e30 if field.startswith("pix_inv_var") else -1.0
    got = run_oracle(o32, ev, seeds=sd.arrays(), cfg=cfg)
    as_set = lambda a: set(map(tuple, a.tolist()))
    for k in (0, 1):
        before = base.pix_tuples(k)
        if field.startswith("pix_inv_var"):
            hits = before[:, 1:]
            lay = geom.layer[ev.module[hits[:, ::2]]].astype(int)
            gone = (lay == idx).any(1)
            if k == kind:
                assert 0 < gone.sum() or idx > lay.max()
        else:
            gone = np.full(len(before), k == kind)
        assert as_set(got.pix_tuples(k)) == as_set(before[~gone]), (field, idx, k)


def test_p26_truth(geom, o32, run_oracle, small):
    ev, sd, r = small
    cfg = open_cfg(o32)
    loose = run_oracle(o32, ev, seeds=sd.arrays(), cfg=cfg)
    pt = ev.particles["pt"]
    for kind in (0, 1):
        def matched(res):
            d = res.pix[kind]
            tr = ev.truth[res.pix_tuples(kind)[:, 1:]]
            same = (tr == tr[:, :1]).all(1) & (tr[:, 0] >= 0) & (tr[:, 0] == sd.truth[d["seed"]])
            same[same] = pt[tr[same, 0]] >= 0.8
            return same
        truth_links = set(map(tuple, loose.pix_tuples(kind)[matched(loose)].tolist()))
        kept = set(map(tuple, r.pix_tuples(kind).tolist()))
        assert len(truth_links) > 300 and len(truth_links & kept) / len(truth_links) >= 0.995
        m = matched(r)
        assert m.mean() > 0.5                                           # most links join a seed to its own particle's object
        fake = sd.truth[r.pix[kind]["seed"]] < 0
        assert fake.mean() < 0.05                                       # fake seeds (20 % of the input) link to almost nothing
