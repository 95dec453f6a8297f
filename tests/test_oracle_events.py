"""Event-level pins of the oracle driver (lsto_run): brute force (P3), single-helix recovery
(P4), chi2 statistics (P6), symmetries (P7), structure (P9), truth sanity (P10).
See tests/test_oracle_pins.py for the scalar cut functions (P1, P2, P5, P8)."""
import numpy as np
import pytest

from paper_2207_08207_b200 import synth


def as_set(rows):
    return set(map(tuple, np.asarray(rows).tolist()))


# ----------------------------------------------------------------------------------------
# P3: brute force
# ----------------------------------------------------------------------------------------
def test_p3_python_brute_force_all_stages(geom, mmap, o32, run_oracle):
    """Tiny event: enumerate EVERY hit pair / MD pair / segment pair / triplet pair in Python
    with the scalar cut functions; the C driver's binned, CSR-walking search must give the
    same sets of hit-index tuples (pins the driver's indexing)."""
    ev = synth.generate_event(geom, 0, 0, n_particles=12)
    r = run_oracle(o32, ev)
    n = ev.n
    layer = geom.layer
    # MDs: all ordered hit pairs, kept if same module, lower side 0, upper side 1
    mds, md_info = [], []
    for l in range(n):
        for u in range(n):
            if ev.module[l] == ev.module[u] and ev.side[l] == 0 and ev.side[u] == 1:
                ok, out, _ = o32.md_cut(int(layer[ev.module[l]]), (ev.x[l], ev.y[l], ev.z[l]), (ev.x[u], ev.y[u], ev.z[u]))
                if ok:
                    mds.append((l, u))
                    md_info.append((ev.x[l], ev.y[l], ev.z[l], out["rl"], out["ru"], out["sinA"]))
    assert as_set(mds) == as_set(r.md_hits()) and len(mds) == r.counts[0] > 20
    # segments: all ordered MD pairs whose module pair is in the map
    conn = {(a, int(b)) for a in range(geom.n_modules) for b in mmap.targets[mmap.row_offsets[a]:mmap.row_offsets[a + 1]]}
    segs = []
    for i, (li, _) in enumerate(mds):
        for o, (lo, _) in enumerate(mds):
            if (int(ev.module[li]), int(ev.module[lo])) in conn:
                if o32.seg_cut(int(layer[ev.module[li]]), md_info[i], md_info[o])[0]:
                    segs.append((i, o))
    assert as_set((*mds[i], *mds[o]) for i, o in segs) == as_set(r.seg_hits()) and len(segs) == r.counts[1] > 10
    # triplets: all ordered segment pairs sharing the middle MD
    t3s, t3k = [], []
    for a, (a_in, a_out) in enumerate(segs):
        for b, (b_in, b_out) in enumerate(segs):
            if a_out == b_in:
                ok, out, _ = o32.t3_cut(int(layer[ev.module[mds[a_in][0]]]), md_info[a_in][:4], md_info[a_out][:4], md_info[b_out][:4])
                if ok:
                    t3s.append((a_in, a_out, b_out))
                    t3k.append(out["kappa"])
    assert as_set(sum((mds[m] for m in t), ()) for t in t3s) == as_set(r.t3_hits()) and len(t3s) == r.counts[2] > 5
    # quintuplets: all ordered triplet pairs sharing the MD at the junction
    t5s = []
    for A, ta in enumerate(t3s):
        for B, tb in enumerate(t3s):
            if ta[2] == tb[0]:
                five = (*ta, tb[1], tb[2])
                ok, _, _ = o32.t5_cut(int(layer[ev.module[mds[five[0]][0]]]), t3k[A], t3k[B], [md_info[m][:4] for m in five])
                if ok:
                    t5s.append(five)
    assert as_set(sum((mds[m] for m in t), ()) for t in t5s) == as_set(r.t5_hits()) and len(t5s) == r.counts[3] > 2


def test_p3_exhaustive_equals_map_restricted(geom, o32, run_oracle):
    """(i) all adjacent-layer MD pairs filtered by map membership == module-driven loop, on a
    busy event; (ii) on the clean tiny event the search with the map IGNORED finds every
    map-restricted segment and nothing more on PS-PS layer pairs."""
    busy = synth.generate_event(geom, 1, 5, n_particles=1200)
    a = run_oracle(o32, busy, mode=0, stages=2)
    b = run_oracle(o32, busy, mode=1, stages=2)
    assert a.counts[1] == b.counts[1] > 5000 and as_set(a.seg_hits()) == as_set(b.seg_hits())
    tiny = synth.generate_event(geom, 0, 0)
    c = run_oracle(o32, tiny, mode=0, stages=2)
    d = run_oracle(o32, tiny, mode=2, stages=2)
    cs, ds = as_set(c.seg_hits()), as_set(d.seg_hits())
    assert c.counts[1] > 200 and cs <= ds
    # whatever the map excludes is a fake (hits of two particles) on a pair touching a 2S layer,
    # where the loose ZSEG lets through what the map's |z0| <= 15 cm rules out; PS-PS pairs and
    # every single-particle segment are found with or without the map
    for t in ds - cs:
        assert geom.layer[tiny.module[t[0]]] >= 2 and len(set(tiny.truth[list(t)].tolist())) > 1
    assert len(ds - cs) <= 3
    # on the busy event the unrestricted search finds strictly more: the map defines the result
    e = run_oracle(o32, busy, mode=2, stages=2)
    assert as_set(a.seg_hits()) <= as_set(e.seg_hits())


# ----------------------------------------------------------------------------------------
# P4: single-helix recovery
# ----------------------------------------------------------------------------------------
def test_p4_single_helix_recovery(geom, o32, run_oracle):
    rng = np.random.default_rng(4)
    done = 0
    while done < 40:
        pt, q = rng.uniform(1.0, 10.0), rng.choice([-1.0, 1.0])
        phi0, eta, z0 = rng.uniform(-np.pi, np.pi), rng.uniform(-0.7, 0.7), rng.normal(0, 5.0)
        ev = synth.single_helix_event(geom, pt, q, phi0, eta, z0)
        per_mod = {}
        for m, s in zip(ev.module, ev.side):
            per_mod.setdefault(int(m), set()).add(int(s))
        if ev.n != 12 or len(per_mod) != 6 or sorted(geom.layer[list(per_mod)]) != list(range(6)):
            continue                                   # crosses an overlap or leaves the barrel
        r = run_oracle(o32, ev)
        assert r.counts == [6, 5, 4, 2], (pt, q, phi0, eta, z0, r.counts)
        assert r.candidates == [6, 5, 4, 2]
        done += 1
    # smeared, with overlaps allowed: every object is made of this particle's hits and
    # the count is at least the clean one whenever all six layers have a full module
    ev = synth.single_helix_event(geom, 2.0, 1.0, 0.3, 0.2, 1.0, smear=True, seed=3)
    r = run_oracle(o32, ev)
    assert r.counts[3] >= 2


# ----------------------------------------------------------------------------------------
# P7: symmetries
# ----------------------------------------------------------------------------------------
@pytest.mark.parametrize("how", ["rot", "mirror_z", "mirror_y"])
def test_p7_symmetries(geom, o64, run_oracle, how):
    """Cuts depend only on hit coordinates (through rotation-invariant forms) and layers, so a
    rigid transformation of all hits with module ids kept leaves every set unchanged. Run in
    the fp64 build so that rounding cannot flip a decision."""
    ev = synth.generate_event(geom, 1, 2, n_particles=600)
    base = run_oracle(o64, ev)
    if how == "rot":
        tr = synth.transform_event(ev, rot=0.7)
    elif how == "mirror_z":
        tr = synth.transform_event(ev, mirror_z=True)
    else:
        tr = synth.Event(ev.x, -ev.y, ev.z, ev.module, ev.side, ev.truth, ev.particles)
    # transform_event rounds the rotated coordinates to fp32: a handful of threshold-edge flips
    # are possible for "rot"; mirrors are exact
    got = run_oracle(o64, tr)
    for name in ("md_hits", "seg_hits", "t3_hits", "t5_hits"):
        a, b = as_set(getattr(base, name)()), as_set(getattr(got, name)())
        if how == "rot":
            assert len(a ^ b) <= max(2, len(a) // 500), (name, len(a), len(a ^ b))
        else:
            assert a == b, name
    if how == "mirror_y":                            # curvature changes sign, magnitudes do not
        assert np.allclose(np.sort(base.t3_kappa), np.sort(-got.t3_kappa), rtol=1e-9, atol=1e-12)
    if how == "mirror_z":
        assert np.allclose(np.sort(base.seg_z0), np.sort(-got.seg_z0), rtol=1e-9, atol=1e-9)


# ----------------------------------------------------------------------------------------
# P9 / P10 / P6 on one PU200-like event
# ----------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def c1(geom, o32, run_oracle):
    ev = synth.generate_event(geom, 1, 0)
    return ev, run_oracle(o32, ev)


def test_p9_structure(geom, mmap, c1):
    ev, r = c1
    lay = geom.layer
    # MD: 2 hits, same module, sides (0, 1)
    assert np.all(ev.module[r.md_lower] == ev.module[r.md_upper]) and np.all(ev.module[r.md_lower] == r.md_module)
    assert np.all(ev.side[r.md_lower] == 0) and np.all(ev.side[r.md_upper] == 1)
    assert len(as_set(r.md_hits())) == r.counts[0]                  # no duplicates
    # LS: 4 distinct hits, adjacent layers, module pair in the map
    li, lo = lay[r.md_module[r.seg_in]], lay[r.md_module[r.seg_out]]
    assert np.all(lo == li + 1)
    conn = as_set(np.stack([np.repeat(np.arange(geom.n_modules), np.diff(mmap.row_offsets)), mmap.targets], 1))
    assert as_set(np.stack([r.md_module[r.seg_in], r.md_module[r.seg_out]], 1)) <= conn
    assert len(as_set(r.seg_hits())) == r.counts[1]
    # T3: segments share the middle MD; 6 distinct hits; layers l, l+1, l+2
    assert np.all(r.seg_out[r.t3_a] == r.seg_in[r.t3_b])
    t3 = r.t3_hits()
    assert t3.shape[1] == 6 and all(len(set(row)) == 6 for row in t3[:2000].tolist())
    assert np.all(np.diff(lay[r.md_module[r.t3_mds()]].astype(int), axis=1) == 1)
    # T5: triplets share the junction MD; 10 distinct hits; five consecutive layers
    a, b = r.t3_mds()[r.t5_a], r.t3_mds()[r.t5_b]
    assert np.all(a[:, 2] == b[:, 0])
    t5 = r.t5_hits()
    assert t5.shape[1] == 10 and all(len(set(row)) == 10 for row in t5[:2000].tolist())
    assert np.all(np.diff(lay[r.md_module[r.t5_mds()]].astype(int), axis=1) == 1)
    assert len(as_set(t5)) == r.counts[3]
    # sizes of SURVEY.md 8(a) (probe +-10 %; T3/T5 depend on the frozen chi2 thresholds)
    assert 31000 < r.counts[0] < 38000 and 50000 < r.counts[1] < 62000
    assert 0.9 * 738069 < r.candidates[0] < 1.1 * 738069 and 0.9 * 4747092 < r.candidates[1] < 1.1 * 4747092


def test_p10_truth_sanity_and_p6_statistics(geom, o32, run_oracle, c1):
    ev, r = c1
    pt = ev.particles["pt"]
    # fraction of output T5s matched to one particle by the 75 % rule
    tr = ev.truth[r.t5_hits()]
    matched = np.array([np.bincount(row[row >= 0]).max() >= 8 if (row >= 0).any() else False for row in tr])
    assert matched.mean() >= 0.97, matched.mean()
    # truth T5 candidates (all ten hits from one particle with pT >= 0.8 GeV, built from the
    # oracle's own T3s with the T5 cuts opened) -> at least 99.9 % pass the frozen Q1..Q5
    cfg = o32.default_config()
    cfg.t5_dkappa_max = cfg.t5_chi2xy_max = cfg.t5_kappa_max = 1e30
    cfg.t5_chi2rz_max[0] = cfg.t5_chi2rz_max[1] = 1e30
    loose = run_oracle(o32, ev, cfg=cfg)
    trl = ev.truth[loose.t5_hits()]
    one = (trl == trl[:, :1]).all(1) & (trl[:, 0] >= 0)
    one[one] = pt[trl[one, 0]] >= 0.8
    truth_cands = as_set(loose.t5_hits()[one])
    assert len(truth_cands) > 5000
    kept = len(truth_cands & as_set(r.t5_hits()))
    assert kept / len(truth_cands) >= 0.999, kept / len(truth_cands)
    # P6: for these true tracks chi2xy ~ chi2(2 dof): 5 points, 3 fitted parameters, Gaussian
    # smearing of sigma_rphi along the module (mean 2, median 1.386, p99 9.21)
    chi2xy = loose.t5_chi2xy[one]
    assert 1.6 < chi2xy.mean() < 2.4 and 1.0 < np.median(chi2xy) < 1.7     # mean 2, median 1.386
    assert np.quantile(chi2xy, 0.99) < 13.0                                # chi2(2): 9.21


def test_golden_oracle_counts():
    """tests/golden/oracle_counts.txt (written by tests/golden/make_oracle_counts.py from the oracle alone): the oracle as
    it stands reproduces the stored counts and quintuplet digests on the seeded events."""
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_oracle_counts", os.path.join(here, "make_oracle_counts.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    stored = [ln.strip() for ln in open(os.path.join(here, "oracle_counts.txt")) if ln.strip()]
    mod.CASES = tuple(c for c in mod.CASES if c[0] in ("C0", "C1small"))        # the cheap cases: a few seconds
    now = {ln.split(" |")[0]: ln for ln in mod.lines() if not ln.startswith("#")}
    assert now, "no case ran"
    for ln in stored:
        key = ln.split(" |")[0]
        if key in now:
            assert now[key] == ln, (now[key], ln)


# ----------------------------------------------------------------------------------------
# P19: per-layer threshold indices ("for different categories") and P20: the Q5 cut
# ----------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def c1small(geom, o32, run_oracle):
    ev = synth.generate_event(geom, 1, 5, n_particles=1200)
    return ev, run_oracle(o32, ev)


def _layers(geom, ev, hits):
    """[n][k] hit tuples -> [n][k/2] layer of every MD of the object."""
    return geom.layer[ev.module[np.asarray(hits)[:, ::2]]].astype(int)


INDEX_CASES = (
    [("md_dz_res", l, 1, "md", "any") for l in range(6)] +           # M3: md_dz_res[layer]
    [("md_thr", l, 1, "md", "any") for l in range(6)] +              # M2: md_cos_eps / md_sin_eps[layer]
    [("seg_z0_max", l, 2, "seg", "first") for l in range(5)] +       # S3: by inner layer
    [("md_eps", l, 2, "seg", "any") for l in range(6)] +             # S4: [inner layer] for the inner MD, [inner + 1] for the outer
    [("t3_chi2rz_max", l, 3, "t3", "first") for l in range(4)] +     # T3: by innermost layer
    [("t5_chi2rz_max", l, 4, "t5", "first") for l in range(2)])      # Q3: by innermost layer


@pytest.mark.parametrize("field,l,stages,cls,who", INDEX_CASES)
def test_p19_threshold_entry_l_removes_exactly_the_objects_of_layer_l(geom, o32, run_oracle, c1small, field, l, stages, cls, who):
    """Closing ONE entry of a per-layer threshold array removes exactly the objects that the SPEC says read that entry
    -- those whose innermost layer is l ("first"), or any of whose mini-doublets sits in layer l ("any": an MD in its own
    layer; S4 reads md_eps[inner layer] for the inner and md_eps[inner layer + 1] for the outer mini-doublet) -- and leaves
    every other object of that class in place.  An off-by-one or a constant index in the oracle fails this."""
    ev, base = c1small
    cfg = o32.default_config()
    if field == "md_thr":                         # SINTHR = t cosE + sqrt(1 - t^2) sinE < 0: nothing passes M2
        cfg.md_cos_eps[l], cfg.md_sin_eps[l] = 0.0, -1.0
    else:
        getattr(cfg, field)[l] = -1.0e30 if field == "md_dz_res" else -1.0
    got = run_oracle(o32, ev, stages=stages, cfg=cfg)
    name = {"md": "md_hits", "seg": "seg_hits", "t3": "t3_hits", "t5": "t5_hits"}[cls]
    before = getattr(base, name)()
    lay = _layers(geom, ev, before)
    hit = (lay[:, 0] == l) if who == "first" else (lay == l).any(1)
    assert 0 < hit.sum() < len(before), (field, l, hit.sum())
    assert as_set(getattr(got, name)()) == as_set(before[~hit]), (field, l)


def test_p20_q5_fitted_curvature_cut(geom, o32, run_oracle):
    """Q5 (DESIGN.md SPEC [Q] step 4): |kFit| <= t5_kappa_max.  kFit of a noiseless helix is -q/R = -q k B / pT (pin P1), so with
    the threshold moved to the curvature of a 2 GeV track (and the other quintuplet cuts left as they are: they pass
    exact helices) both quintuplets of every 1.5 GeV helix disappear and both of every 3 GeV helix stay."""
    kb = synth.K_GEV_PER_T_CM * synth.B_TESLA
    cfg = o32.default_config()
    cfg.t5_kappa_max = kb / 2.0
    rng = np.random.default_rng(20)
    done = {1.5: 0, 3.0: 0}
    while min(done.values()) < 12:
        pt = 1.5 if done[1.5] <= done[3.0] else 3.0
        q, phi0, eta, z0 = rng.choice([-1.0, 1.0]), rng.uniform(-np.pi, np.pi), rng.uniform(-0.6, 0.6), rng.normal(0, 4.0)
        ev = synth.single_helix_event(geom, pt, q, phi0, eta, z0)
        if run_oracle(o32, ev).counts != [6, 5, 4, 2]:
            continue                               # crosses an overlap or leaves the barrel: not the clean case
        r = run_oracle(o32, ev, cfg=cfg)
        assert r.counts[:3] == [6, 5, 4] and r.counts[3] == (0 if pt == 1.5 else 2), (pt, q, r.counts)
        done[pt] += 1
