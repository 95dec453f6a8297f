"""GPU parity of the optional stage LST_PIXEL (SPEC [P]): pixel line segments -> pixel triplets and pixel
quintuplets, through the C-ABI binding, against the oracle's full (outer object x seed) product on the same seeded inputs.
Link sets must be IDENTICAL -- (seed index, original hit indices of the outer object) -- the order must be the method's
(outer object, seed index), the floats within 1e-5 relative, the search-space counts equal."""
import numpy as np
import pytest

from paper_2207_08207_b200 import synth

import parity

pytestmark = pytest.mark.gpu

PIX_FLOORS = (1e-5 * 85.0, 1e-5 * 25.0, 1e-5 * parity.KAPPA_MAX)     # chi2xy, chi2rz, kappa_obj - kappa_seed


@pytest.fixture(scope="module")
def lstmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2207_08207_b200 import build as lst_build, lst
    lst_build.build()
    lst.load_library()
    return lst


@pytest.fixture(scope="module")
def ctx(lstmod, geom, mmap):
    cfg = lstmod.default_config()
    cfg.n_slots = 4
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    yield c
    c.close()


def run_pixel(ctx, lstmod, ev, seeds, slot=0, stream=None):
    ctx.load_event(slot, ev.x, ev.y, ev.z, ev.module, ev.side, stream)
    ctx.load_seeds(slot, [seeds], stream)
    ctx.run(slot, stream)
    ctx.run_stage(slot, 1, lstmod.PIXEL, stream)
    ctx.sync(slot, stream)


def compare_links(ctx, lstmod, ora, slot=0, label=""):
    """Every link of both kinds against the oracle's; returns the worst relative float difference."""
    st = ctx.stats(slot)
    worst = 0.0
    for kind in (0, 1):
        d = ora.pix[kind]
        link, f = ctx.fetch_pixel_links(slot, kind)
        assert st["pix_needed"][kind] == d["n"] == len(link), (label, kind, st["pix_needed"], d["n"])
        assert st["pix_candidates"][kind] == d["candidates"], (label, kind, st["pix_candidates"], d["candidates"])
        assert d["n"] <= st["pix_evaluated"][kind] <= d["candidates"], (label, kind, st)
        obj_hits = ctx.fetch_hit_indices(slot, lstmod.T5 if kind else lstmod.T3)
        # order: (outer object, seed index), CSR by outer object
        if len(link):
            key = link[:, 1].astype(np.int64) * (1 << 32) + link[:, 0]
            assert np.all(np.diff(key) > 0), f"{label} kind {kind}: links not ordered by (object, seed)"
        view = ctx.pixel_links(slot, kind)
        start = view["object_start"].torch().cpu().numpy()
        assert start[0] == 0 and start[-1] == len(link) and np.all(np.diff(start) >= 0)
        assert np.array_equal(np.repeat(np.arange(len(start) - 1), np.diff(start)), link[:, 1])
        assert np.array_equal(view["link"].torch().cpu().numpy(), link)
        got = np.concatenate([link[:, :1], obj_hits[link[:, 1]].reshape(len(link), obj_hits.shape[1])], 1)
        want = ora.pix_tuples(kind)
        gh, gv = parity.sort_rows(got, f)
        oh, ov = parity.sort_rows(want, np.stack([d["chi2xy"], d["chi2rz"], d["dkappa"]], 1).reshape(-1, 3))
        assert gh.shape == oh.shape and np.array_equal(gh, oh), f"{label} kind {kind}: link sets differ"
        for c in range(3):
            a, b = gv[:, c].astype(np.float64), ov[:, c].astype(np.float64)
            tol = parity.REL_TOL * np.maximum(np.abs(a), np.abs(b)) + PIX_FLOORS[c]
            assert np.all(np.abs(a - b) <= tol), f"{label} kind {kind} column {c}: worst {np.abs(a - b).max()}"
            if len(a):
                worst = max(worst, float(np.max(np.abs(a - b) / np.maximum(np.maximum(np.abs(a), np.abs(b)), PIX_FLOORS[c] / parity.REL_TOL))))
    return worst, st


@pytest.mark.parametrize("config,seed", [(0, 0), (1, 0), (1, 17), (3, 0)])
def test_pixel_parity_baseline_configs(ctx, lstmod, o32, run_oracle, geom, config, seed):
    """Full-size events of BASELINE.json configs[0], [1], [3] with the stand-in seed model: every link
    compared; the oracle evaluates the whole product (1.2e8 / 5e7 pairs on a PU200-like event)."""
    ev = synth.generate_event(geom, config, seed)
    sd = synth.generate_seeds(ev, seed)
    run_pixel(ctx, lstmod, ev, sd.arrays())
    ora = run_oracle(o32, ev, seeds=sd.arrays())
    worst, st = compare_links(ctx, lstmod, ora, label=f"C{config}/seed{seed}")
    assert st["n_seeds"] == sd.n and st["overflow"] == 0
    assert ora.pix[0]["n"] > (20 if config == 0 else 5000) and ora.pix[1]["n"] > (10 if config == 0 else 4000)
    # the objects themselves are untouched by the stage
    parity.compare(parity.gpu_tables(ctx, 0), parity.oracle_tables(ora), f"C{config}/seed{seed} objects")
    print(f"C{config} seed {seed}: {sd.n} seeds, links {st['pix_needed']}, evaluated {st['pix_evaluated']} of {st['pix_candidates']}, "
          f"rewalks {st['pix_rewalks']}, max rel err {worst:.2e}")


def test_pixel_edge_cases(ctx, lstmod, o32, run_oracle, geom):
    """No seeds; seeds that nothing can accept (NaN, infinite, zero direction); directions that are not unit vectors (scaled,
    tiny, huge: no azimuth window exists for them, they are evaluated against every object); seeds pointing along +-pi where
    the azimuth bins wrap; an event without hits."""
    ev = synth.generate_event(geom, 1, 21, n_particles=900)
    sd = synth.generate_seeds(ev, 21, efficiency=1.0, fake_fraction=0.5)
    k, c, s, z0, t = (a.copy() for a in sd.arrays())
    empty = tuple(np.zeros(0, np.float32) for _ in range(5))
    run_pixel(ctx, lstmod, ev, empty)
    ora = run_oracle(o32, ev, seeds=empty)
    compare_links(ctx, lstmod, ora, label="no seeds")
    assert ctx.stats(0)["pix_needed"] == [0, 0] and ctx.stats(0)["n_seeds"] == 0
    n = len(k)
    rng = np.random.default_rng(5)
    kind = rng.integers(0, 8, n)
    with np.errstate(over="ignore"):
        for i in range(n):
            if kind[i] == 1:
                c[i] = np.nan
            elif kind[i] == 2:
                s[i] = np.inf
            elif kind[i] == 3:
                c[i] = s[i] = 0.0
            elif kind[i] == 4:
                f = np.float32(rng.choice([0.5, 0.97, 1.02, 1.5, 1e-20, 1e15, 3e38]))
                c[i] = np.float32(c[i] * f); s[i] = np.float32(s[i] * f)
            elif kind[i] == 5:
                k[i] = np.nan if i % 2 else np.float32(0.0)
            elif kind[i] == 6:
                z0[i] = np.inf if i % 2 else z0[i]; t[i] = np.nan if i % 3 == 0 else t[i]
    seeds = (k, c, s, z0, t)
    run_pixel(ctx, lstmod, ev, seeds)
    ora = run_oracle(o32, ev, seeds=seeds)
    compare_links(ctx, lstmod, ora, label="odd seeds")
    assert ora.pix[0]["n"] > 100
    # the event rotated so that many tracks leave along phi = +-pi (bin wrap), seeds rotated with it
    for rot in (np.pi, np.pi - 1e-3, -np.pi + 2e-4):
        ev2 = synth.transform_event(ev, rot=rot)
        phi0 = np.arctan2(sd.sphi.astype(np.float64), sd.cphi.astype(np.float64)) + rot
        seeds2 = (sd.kappa, np.cos(phi0).astype(np.float32), np.sin(phi0).astype(np.float32), sd.z0, sd.t)
        run_pixel(ctx, lstmod, ev2, seeds2)
        ora2 = run_oracle(o32, ev2, seeds=seeds2)
        compare_links(ctx, lstmod, ora2, label=f"rot {rot}")
        assert ora2.pix[0]["n"] > 100
    z = np.zeros(0, np.float32)
    ctx.load_event(1, z, z, z, np.zeros(0, np.int32), np.zeros(0, np.uint8))
    ctx.load_seeds(1, [sd.arrays()])
    ctx.run(1)
    ctx.run_stage(1, 1, lstmod.PIXEL)
    ctx.sync(1)
    st = ctx.stats(1)
    assert st["pix_needed"] == [0, 0] and st["pix_candidates"] == [0, 0] and st["n_seeds"] == sd.n
    assert ctx.fetch_pixel_links(1, 0)[0].shape == (0, 2)


def test_pixel_many_links_per_object_direct_path(lstmod, geom, mmap, o32, run_oracle):
    """Every seed repeated 40 times: an object now has 40 or 80 links, a chunk of 32 objects far more than the on-chip stash
    holds, so chunks are walked twice writing directly (pix_rewalks > 0) and the links of an object, found in bin order, must
    still come out in ascending seed index.  Then the same with too small a capacity: an error, the needed size reported."""
    ev = synth.generate_event(geom, 1, 8, n_particles=400)
    sd = synth.generate_seeds(ev, 8, efficiency=1.0, fake_fraction=0.2)
    rep = 40
    perm = np.random.default_rng(3).permutation(sd.n * rep)
    seeds = tuple(np.tile(a, rep)[perm] for a in sd.arrays())
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    cfg.cap_pt3 = 256 * 1024
    cfg.cap_pt5 = 256 * 1024
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    run_pixel(c, lstmod, ev, seeds)
    ora = run_oracle(o32, ev, seeds=seeds)
    _, st = compare_links(c, lstmod, ora, label="x40")
    assert min(st["pix_rewalks"]) > 0 and ora.pix[0]["n"] > 10000
    c.close()
    for kind, field in enumerate(("cap_pt3", "cap_pt5")):
        cfg = lstmod.default_config()
        cfg.n_slots = 1
        setattr(cfg, field, ora.pix[kind]["n"] // 3)
        c = lstmod.Lst.from_synth(geom, mmap, cfg)
        c.load_event(0, ev.x, ev.y, ev.z, ev.module, ev.side)
        c.load_seeds(0, [seeds])
        c.run(0)
        c.run_stage(0, 1, lstmod.PIXEL)
        assert c.sync(0, check=False) == lstmod.ERR_OVERFLOW
        st = c.stats(0)
        assert st["overflow"] == 16 << kind and st["pix_needed"][kind] == ora.pix[kind]["n"]
        with pytest.raises(lstmod.LstError):
            c.pixel_links(0, kind)
        c.close()


def test_pixel_call_order_and_capacity_errors(lstmod, geom, mmap):
    ev = synth.generate_event(geom, 0, 0)
    sd = synth.generate_seeds(ev, 0)
    cfg = lstmod.default_config()
    cfg.n_slots = 2
    cfg.cap_seeds = 16
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    with pytest.raises(lstmod.LstError) as e:
        c.load_seeds(0, [sd.arrays()])                       # slot not loaded
    assert e.value.status == lstmod.ERR_STATE
    c.load_event(0, ev.x, ev.y, ev.z, ev.module, ev.side)
    with pytest.raises(lstmod.LstError) as e:
        c.load_seeds(0, [sd.arrays()])                       # more seeds than cap_seeds
    assert e.value.status == lstmod.ERR_OVERFLOW
    c.run(0)
    with pytest.raises(lstmod.LstError) as e:
        c.run_stage(0, 1, lstmod.PIXEL)                      # no seeds loaded
    assert e.value.status == lstmod.ERR_STATE
    few = tuple(a[:16] for a in sd.arrays())
    c.load_event(1, ev.x, ev.y, ev.z, ev.module, ev.side)
    c.load_seeds(1, [few])
    c.run_stage(1, 1, lstmod.MD)
    with pytest.raises(lstmod.LstError) as e:
        c.run_stage(1, 1, lstmod.PIXEL)                      # the quintuplets are not built yet
    assert e.value.status == lstmod.ERR_STATE
    for stage in (lstmod.SEG, lstmod.T3, lstmod.T5, lstmod.PIXEL, lstmod.CLEAN):
        c.run_stage(1, 1, stage)
    c.sync(1)
    assert c.stats(1)["n_seeds"] == 16 and c.stats(1)["n_kept"] > 0
    c.pixel_links(1, 0), c.track_candidates(1)
    c.load_event(1, ev.x, ev.y, ev.z, ev.module, ev.side)     # loading hits resets the slot, its seeds included
    c.run(1)
    with pytest.raises(lstmod.LstError):
        c.run_stage(1, 1, lstmod.PIXEL)
    c.close()
    cfg.cap_seeds = 0
    with pytest.raises(lstmod.LstError):
        lstmod.Lst.from_synth(geom, mmap, cfg)


def test_pixel_with_non_default_constants(lstmod, geom, mmap, o32):
    """Every [P] constant comes from lst_config: tightened / loosened values on both sides, including weights of zero (the
    azimuth window degrades to all bins) and thresholds so wide that the window spans half the circle."""
    ev = synth.generate_event(geom, 1, 31, n_particles=800)
    sd = synth.generate_seeds(ev, 31)
    cases = [
        dict(pix_dkappa_max=(0.0004, 0.001), pix_chi2xy_max=(40.0, 200.0), pix_chi2rz_max=(60.0, 15.0)),
        dict(pix_inv_var_xy=(0.0, 0.0, 51.984085, 16.645065, 6.149085, 2.8425808)),
        dict(pix_chi2xy_max=(1e9, 1e9), pix_dkappa_max=(1.0, 1.0), pix_chi2rz_max=(3.0, 3.0)),
        dict(pix_dkappa_max=(-1.0, float("nan"))),
    ]
    counts = []
    for ch in cases:
        cfg = lstmod.default_config()
        cfg.n_slots = 1
        cfg.cap_pt3 = cfg.cap_pt5 = 1 << 20
        ocfg = o32.default_config()
        for k, v in ch.items():
            a, b = getattr(cfg, k), getattr(ocfg, k)
            for i in range(len(v)):
                a[i] = v[i]
                b[i] = a[i]
        c = lstmod.Lst.from_synth(geom, mmap, cfg)
        run_pixel(c, lstmod, ev, sd.arrays())
        ora = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, cfg=ocfg, seeds=sd.arrays())
        compare_links(c, lstmod, ora, label=str(ch))
        counts.append((ora.pix[0]["n"], ora.pix[1]["n"]))
        c.close()
    assert counts[3] == (0, 0) and len(set(counts)) == 4 and counts[2][0] > 500, counts


def test_pixel_in_the_bench_launch_configuration(lstmod, geom, mmap, o32, run_oracle):
    """4 streams x 16-event batched launches with device-resident hits and seeds, the stage run twice over recycled slots; a
    sample of events compared in full."""
    import torch
    n_ev, n_streams = 64, 4
    per = n_ev // n_streams
    cfg = lstmod.default_config()
    cfg.n_slots = n_ev
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    evs = [synth.generate_event(geom, 1, 300 + i, n_particles=(1500 if i % 5 else 3000)) for i in range(n_ev)]
    sds = [synth.generate_seeds(evs[i], 300 + i) for i in range(n_ev)]
    dev = lambda arrs: tuple(torch.as_tensor(a).cuda() for a in arrs)
    d_ev = [dev((e.x, e.y, e.z, e.module, e.side)) for e in evs]
    d_sd = [dev(s.arrays()) for s in sds]
    streams = [torch.cuda.Stream() for _ in range(n_streams)]
    for rep in range(2):
        for k, s in enumerate(streams):
            c.load_events(k * per, d_ev[k * per:(k + 1) * per], s)
            c.load_seeds(k * per, d_sd[k * per:(k + 1) * per], s)
            c.run_batch(k * per, per, s)
            c.run_stage(k * per, per, lstmod.PIXEL, s)
        for k, s in enumerate(streams):
            c.sync_batch(k * per, per, s)
    for i in (0, 5, 15, 16, 37, 63):
        ora = run_oracle(o32, evs[i], seeds=sds[i].arrays())
        compare_links(c, lstmod, ora, slot=i, label=f"batch event {i}")
    c.close()


def test_pixel_seeds_on_the_window_edges(lstmod, geom, mmap, o32):
    """Seeds constructed to sit on the edges of the search windows of real triplets: curvature at kappa_obj +- pix_dkappa_max
    (1 -+ 1e-6) (the P1 boundary and the curvature bands) and direction such that the first anchor's P2 term is at
    +- its largest admissible value (1 -+ 1e-5) (the azimuth window).  With the x-y weights of all layers but the first
    made negligible and the r-z cut opened, pass / fail flips right there, so a window that were too tight by a few ulps would
    lose links the oracle's full product finds.  Objects starting on layer 1 then have no azimuth window at all (weight ~ 0)."""
    ev = synth.generate_event(geom, 1, 41, n_particles=600)
    base = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side)
    t3m = base.t3_mds()
    lay = geom.layer[base.md_module][t3m[:, 0]]
    pick = np.nonzero(lay == 0)[0][::3][:400]
    w0, chi_max, dk_max = 809.479, 85.0, 0.0008
    E = np.sqrt(chi_max / w0)
    K, C_, S_, Z0, T = [], [], [], [], []
    for j in pick:
        m = t3m[j, 0]
        x, y, r = float(base.md_x[m]), float(base.md_y[m]), float(base.md_r[m])
        kobj, phip = float(base.t3_kappa[j]), np.arctan2(y, x)
        for sk in (-1.0, 1.0):
            for dkr in (-1e-6, 0.0, 1e-6):
                kap = np.float32(kobj + sk * dk_max * (1.0 + dkr))
                for se in (-1.0, 1.0):
                    for der in (-1e-5, 0.0, 1e-5):
                        arg = (se * E * (1.0 + der) - 0.5 * float(kap) * r * r) / r
                        if abs(arg) >= 1.0:
                            continue
                        phi0 = phip + np.arcsin(arg)
                        K.append(kap); C_.append(np.cos(phi0)); S_.append(np.sin(phi0)); Z0.append(0.0); T.append(0.0)
    seeds = tuple(np.asarray(a, np.float32) for a in (K, C_, S_, Z0, T))
    assert 2500 < len(seeds[0]) <= 16384
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    cfg.cap_pt3 = cfg.cap_pt5 = 1 << 20
    ocfg = o32.default_config()
    for c in (cfg, ocfg):
        for l in range(1, 6):
            c.pix_inv_var_xy[l] = 1e-9
        for k in range(2):
            c.pix_chi2rz_max[k] = 1e30
            c.pix_chi2xy_max[k] = chi_max
            c.pix_dkappa_max[k] = dk_max
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    run_pixel(c, lstmod, ev, seeds)
    ora = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, cfg=ocfg, seeds=seeds)
    compare_links(c, lstmod, ora, label="edge seeds")
    # both outcomes occur at the edges, in numbers: the construction does sit on the boundary
    own = ora.pix[0]["n"]
    assert 0.2 * len(seeds[0]) < own, own
    c.close()


def test_module_ids_in_any_order(lstmod, geom, mmap, o32):
    """The library assumes nothing about how module ids are numbered: the same detector with its module ids randomly
    permuted (geometry tables, module map rows and targets, the hits' module column) gives the oracle's sets for that
    numbering -- objects and pixel links.  (With ids ordered by layer, as in the BASELINE geometry, the pixel-triplet kernel
    walks only the leading triplets; here it cannot.)"""
    rng = np.random.default_rng(11)
    n = geom.n_modules
    perm = rng.permutation(n).astype(np.int32)          # old id -> new id
    inv = np.argsort(perm)
    layer, phi = geom.layer[inv], geom.phi[inv]
    rows = [np.sort(perm[mmap.targets[mmap.row_offsets[a]:mmap.row_offsets[a + 1]]]) for a in inv]
    offs = np.zeros(n + 1, np.int32)
    offs[1:] = np.cumsum([len(r) for r in rows])
    targets = np.concatenate(rows).astype(np.int32)
    ev = synth.generate_event(geom, 1, 77, n_particles=1500)
    sd = synth.generate_seeds(ev, 77)
    module = perm[ev.module]
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    c = lstmod.Lst(layer, offs, targets, cfg, phi=phi)
    c.load_event(0, ev.x, ev.y, ev.z, module, ev.side)
    c.load_seeds(0, [sd.arrays()])
    c.run(0)
    c.run_stage(0, 1, lstmod.PIXEL)
    c.run_stage(0, 1, lstmod.CLEAN)
    c.sync(0)
    ora = o32.run(layer, offs, targets, ev.x, ev.y, ev.z, module, ev.side, seeds=sd.arrays())
    parity.compare(parity.gpu_tables(c, 0), parity.oracle_tables(ora), "permuted ids")
    compare_links(c, lstmod, ora, label="permuted ids")
    keep = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz)
    got = c.fetch_hit_indices(0, lstmod.T5)[c.fetch_kept(0)]
    assert set(map(tuple, got.tolist())) == set(map(tuple, ora.t5_hits()[keep.astype(bool)].tolist()))
    # the same objects as with the original numbering (identity is by hit index)
    ref = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side)
    assert set(map(tuple, ref.t5_hits().tolist())) == set(map(tuple, ora.t5_hits().tolist()))
    c.close()


def test_pixel_stage_in_a_cuda_graph(ctx, lstmod, o32, run_oracle, geom):
    """lst_load_seeds (device input) and LST_PIXEL only enqueue work: the whole sequence load hits -> load seeds -> a1..a4 ->
    LST_CLEAN -> LST_PIXEL is captured once over fixed device buffers and replayed with other contents."""
    import torch
    evs = [synth.generate_event(geom, 1, 190 + i, n_particles=1200) for i in range(2)]
    sds = [synth.generate_seeds(e, 190 + i) for i, e in enumerate(evs)]
    n, ns = min(e.n for e in evs), min(s.n for s in sds)
    hb = [torch.zeros(n, dtype=dt, device="cuda") for dt in (torch.float32, torch.float32, torch.float32, torch.int32, torch.uint8)]
    sb = [torch.zeros(ns, dtype=torch.float32, device="cuda") for _ in range(5)]
    st = torch.cuda.Stream()

    def fill(ev, sd):
        for b, a in zip(hb, (ev.x, ev.y, ev.z, ev.module, ev.side)):
            b.copy_(torch.from_numpy(a[:n]))
        for b, a in zip(sb, sd.arrays()):
            b.copy_(torch.from_numpy(a[:ns]))
        return (synth.Event(ev.x[:n], ev.y[:n], ev.z[:n], ev.module[:n], ev.side[:n], ev.truth[:n], {}), tuple(a[:ns] for a in sd.arrays()))

    fill(evs[0], sds[0])
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        ctx.load_events(2, [hb], stream=st)
        ctx.load_seeds(2, [sb], stream=st)
        ctx.run_batch(2, 1, st)
        ctx.run_stage(2, 1, lstmod.CLEAN, st)
        ctx.run_stage(2, 1, lstmod.PIXEL, st)
    for k in (1, 0, 1):
        cut, seeds = fill(evs[k], sds[k])
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        ctx.sync(2, st)
        ora = run_oracle(o32, cut, seeds=seeds)
        compare_links(ctx, lstmod, ora, slot=2, label=f"graph replay {k}")
        keep = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz)
        assert ctx.stats(2)["n_kept"] == int(keep.sum())


@pytest.mark.parametrize("first_layer", [1, 2, 4, 5])
def test_events_without_inner_layers(ctx, lstmod, o32, run_oracle, geom, first_layer):
    """The stage kernels walk only the owners that can have candidates (a CSR prefix when module ids are ordered by layer) and
    fill the CSR entries of the rest: events whose hits start at layer 1, 2 (no quintuplet and no pixel link can exist, but
    triplets do), 4 (segments, no triplets) and 5 (mini-doublets only) exercise the empty-prefix paths."""
    ev = synth.generate_event(geom, 1, 123, n_particles=1500)
    keep = geom.layer[ev.module] >= first_layer
    cut = synth.Event(ev.x[keep], ev.y[keep], ev.z[keep], ev.module[keep], ev.side[keep], ev.truth[keep], {})
    sd = synth.generate_seeds(ev, 123)
    run_pixel(ctx, lstmod, cut, sd.arrays(), slot=3)
    ctx.run_stage(3, 1, lstmod.CLEAN)
    ctx.sync(3)
    ora = run_oracle(o32, cut, seeds=sd.arrays())
    parity.compare(parity.gpu_tables(ctx, 3), parity.oracle_tables(ora), f"from layer {first_layer}")
    compare_links(ctx, lstmod, ora, slot=3, label=f"from layer {first_layer}")
    st = ctx.stats(3)
    assert st["needed"] == ora.counts and st["candidates"] == ora.candidates
    if first_layer >= 2:
        assert ora.counts[3] == 0 and ora.pix[0]["n"] == 0 and st["n_kept"] == 0
    if first_layer == 2:
        assert ora.counts[2] > 100
    if first_layer == 4:
        assert ora.counts[1] > 100 and ora.counts[2] == 0
    if first_layer == 5:
        assert ora.counts[0] > 100 and ora.counts[1] == 0
    # the CSR arrays are complete: every entry of the owners that were not walked equals the total
    for view, key, n_owner in ((ctx.segments(3), "md_start", st["needed"][0]), (ctx.triplets(3), "seg_start", st["needed"][1]),
                               (ctx.quintuplets(3), "t3_start", st["needed"][2])):
        start = view[key].torch().cpu().numpy()
        assert len(start) == n_owner + 1 and start[0] == 0 and start[-1] == view["n"] and np.all(np.diff(start) >= 0)
