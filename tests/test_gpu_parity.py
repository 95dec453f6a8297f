"""GPU parity: the CUDA path, called through the C-ABI binding, against the CPU oracle on the same
seeded inputs.  Object sets must be IDENTICAL (tuples of original hit indices, BASELINE.json
north_star); float payloads within 1e-5 relative (reading 20); candidate counts equal.
"""
import numpy as np
import pytest

from paper_2207_08207_b200 import synth

import parity

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lstmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2207_08207_b200 import build as lst_build, lst
    lst_build.build()           # no-op when liblst.so is up to date; compiles it (nvcc, sm_100a) on a fresh checkout
    lst.load_library()          # raises if liblst.so is missing: no fallback
    return lst


@pytest.fixture(scope="module")
def ctx(lstmod, geom, mmap):
    cfg = lstmod.default_config()
    cfg.n_slots = 8
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    yield c
    c.close()


def check_event(ctx, o32, run_oracle, ev, slot=0, label=""):
    gpu = parity.run_gpu(ctx, ev, slot)
    ora = run_oracle(o32, ev)
    worst = parity.compare(gpu, parity.oracle_tables(ora), label)
    st = ctx.stats(slot)
    assert st["needed"] == ora.counts, (label, st, ora.counts)
    assert st["candidates"] == ora.candidates, (label, st, ora.candidates)
    assert st["n_hits"] == ev.n and st["overflow"] == 0 and st["bad_hits"] == 0
    for k in range(4):      # windows only ever shrink the evaluated set, never below what passes
        assert st["needed"][k] <= st["evaluated"][k] <= st["candidates"][k], (label, st)
    return worst, st


@pytest.mark.parametrize("config,seed", [(0, 0), (0, 1), (1, 0), (1, 17), (3, 0)])
def test_parity_baseline_configs(ctx, o32, run_oracle, geom, config, seed):
    """BASELINE.json configs[0] (tiny), configs[1] (PU200-like, the bench workload's event) and
    configs[3] (PU300-like stress): full-size events, every object compared."""
    ev = synth.generate_event(geom, config, seed)
    worst, st = check_event(ctx, o32, run_oracle, ev, label=f"C{config}/seed{seed}")
    assert st["needed"][3] > (50 if config == 0 else 5000)
    print(f"C{config} seed {seed}: hits {ev.n} objects {st['needed']} candidates {st['candidates']} max rel err {worst}")


@pytest.mark.parametrize("n_particles", [1, 3, 40, 700])
def test_parity_ragged_sizes(ctx, o32, run_oracle, geom, n_particles):
    ev = synth.generate_event(geom, 1, 100 + n_particles, n_particles=n_particles)
    check_event(ctx, o32, run_oracle, ev, label=f"P{n_particles}")


def test_parity_occupancy_sweep(ctx, o32, run_oracle, geom):
    """BASELINE.json configs[4]: occupancy events at 1 k, 10 k, 100 k hits (MD + LS dominated)."""
    for n in (1000, 10000, 100000):
        ev = synth.generate_occupancy_event(geom, n, seed=4)
        check_event(ctx, o32, run_oracle, ev, label=f"occ{n}")


def test_degenerate_events(ctx, lstmod, o32, run_oracle, geom):
    # empty event
    e = synth.Event(*(np.zeros(0, t) for t in (np.float32, np.float32, np.float32, np.int32, np.uint8, np.int32)), {})
    check_event(ctx, o32, run_oracle, e, label="empty")
    # one hit; two hits on one side only; a module with lower hits only
    ev = synth.generate_event(geom, 0, 0)
    for sel in (slice(0, 1), np.nonzero(ev.side == 0)[0], np.nonzero(ev.side == 1)[0]):
        sub = synth.Event(ev.x[sel], ev.y[sel], ev.z[sel], ev.module[sel], ev.side[sel], ev.truth[sel], {})
        _, st = check_event(ctx, o32, run_oracle, sub, label="one-sided")
        assert st["needed"] == [0, 0, 0, 0]
    # all hits identical (zero-length vectors everywhere): nothing passes, nothing crashes
    n = 64
    same = synth.Event(np.full(n, 23.0, np.float32), np.zeros(n, np.float32), np.zeros(n, np.float32),
                       np.zeros(n, np.int32), (np.arange(n) % 2).astype(np.uint8), np.zeros(n, np.int32), {})
    _, st = check_event(ctx, o32, run_oracle, same, label="identical")
    assert st["candidates"][0] == 32 * 32 and st["needed"][0] == 0
    # non-finite coordinates reject (NaN never passes a '<=' cut)
    bad = synth.generate_event(geom, 0, 2)
    bad.x[::7] = np.nan
    bad.z[::11] = np.inf
    check_event(ctx, o32, run_oracle, bad, label="nonfinite")


def test_one_heavy_module(ctx, o32, run_oracle, geom):
    """Maximum-occupancy degenerate case: hundreds of hits in ONE module and its neighbours
    (several warp iterations per module, ragged tails, long CSR rows)."""
    rng = np.random.default_rng(9)
    ev = synth.generate_event(geom, 1, 9, n_particles=2500)
    phi0 = geom.phi[200]
    d = np.abs(np.angle(np.exp(1j * (ev.particles["phi0"] - phi0))))
    # keep every hit; add 400 extra noise hits on module 200 and 300 on a connected module
    extra_mod = np.concatenate([np.full(400, 200), np.full(300, 200 + 408 + 12)]).astype(np.int32)
    lay = geom.layer[extra_mod].astype(int)
    side = rng.integers(0, 2, len(extra_mod)).astype(np.uint8)
    rho = np.asarray(synth.LAYER_R)[lay] + (side - 0.5) * np.asarray(synth.SENSOR_GAP)[lay]
    u = rng.uniform(-4.8, 4.8, len(extra_mod))
    Phi = geom.phi[extra_mod]
    x = (rho * np.cos(Phi) - u * np.sin(Phi)).astype(np.float32)
    y = (rho * np.sin(Phi) + u * np.cos(Phi)).astype(np.float32)
    z = (-120 + 10 * (geom.ring[extra_mod] + rng.uniform(0, 1, len(extra_mod)))).astype(np.float32)
    big = synth.Event(np.concatenate([ev.x, x]), np.concatenate([ev.y, y]), np.concatenate([ev.z, z]),
                      np.concatenate([ev.module, extra_mod]), np.concatenate([ev.side, side]),
                      np.concatenate([ev.truth, np.full(len(x), -1, np.int32)]), ev.particles)
    assert d.size
    _, st = check_event(ctx, o32, run_oracle, big, label="heavy")
    assert st["candidates"][0] > 40000


def test_device_input_batch_and_determinism(ctx, lstmod, o32, run_oracle, geom):
    """(i) device-resident input == host input; (ii) lst_run_batch over 4 slots == 4 single runs ==
    oracle; (iii) two runs of the same event give bit-identical object arrays in the same order."""
    import torch
    evs = [synth.generate_event(geom, 1, 30 + i, n_particles=1500 + 500 * i) for i in range(4)]
    stream = torch.cuda.Stream()
    dev = []
    for s, ev in enumerate(evs):
        dev.append([torch.from_numpy(a).cuda() for a in (ev.x, ev.y, ev.z, ev.module, ev.side)])
    ctx.load_events(0, dev, stream=stream)               # one set of a0 launches for the 4 events
    ctx.run_batch(0, 4, stream)
    for s, ev in enumerate(evs):
        ctx.sync(s, stream)
        got = parity.gpu_tables(ctx, s, stream)
        ora = run_oracle(o32, ev)
        parity.compare(got, parity.oracle_tables(ora), f"batch slot {s}")
        assert ctx.stats(s)["needed"] == ora.counts
    # determinism: slot 5 single run, host input, compare raw (unsorted) arrays with slot 1
    ref = parity.gpu_tables(ctx, 1, stream)
    again = parity.run_gpu(ctx, evs[1], slot=5)
    for k in range(4):
        assert np.array_equal(ref[k][0], again[k][0]) and np.array_equal(ref[k][1], again[k][1], equal_nan=True)
    # views: CSR offsets are consistent with the object arrays
    md = ctx.mds(5); seg = ctx.segments(5); t3 = ctx.triplets(5); t5 = ctx.quintuplets(5)
    seg_md = seg["md"].torch().cpu().numpy(); start = seg["md_start"].torch().cpu().numpy()
    assert start[0] == 0 and start[-1] == seg["n"] and np.all(np.diff(start) >= 0)
    assert np.array_equal(np.repeat(np.arange(md["n"]), np.diff(start)), seg_md[:, 0])
    t3s = t3["seg_start"].torch().cpu().numpy()
    assert t3s[-1] == t3["n"] and np.array_equal(np.repeat(np.arange(seg["n"]), np.diff(t3s)), t3["seg"].torch().cpu().numpy()[:, 0])
    t5s = t5["t3_start"].torch().cpu().numpy()
    assert t5s[-1] == t5["n"] and np.array_equal(np.repeat(np.arange(t3["n"]), np.diff(t5s)), t5["t3"].torch().cpu().numpy()[:, 0])
    ms = md["module_start"].torch().cpu().numpy()
    assert np.array_equal(np.repeat(np.arange(geom.n_modules), np.diff(ms)), md["module"].torch().cpu().numpy())


def test_overflow_and_bad_input_are_reported(lstmod, geom, mmap, o32, run_oracle):
    """BASELINE.json configs[3]: candidate-buffer overflow handling — an error status, the sizes
    that were needed, never a truncated success; and invalid module ids / sides are dropped
    and reported."""
    ev = synth.generate_event(geom, 1, 3, n_particles=2000)
    ora = run_oracle(o32, ev)
    for kind, field in enumerate(("cap_md", "cap_seg", "cap_t3", "cap_t5")):
        cfg = lstmod.default_config()
        cfg.n_slots = 1
        setattr(cfg, field, max(1, ora.counts[kind] // 2))
        c = lstmod.Lst.from_synth(geom, mmap, cfg)
        c.load_event(0, ev.x, ev.y, ev.z, ev.module, ev.side)
        c.run(0)
        assert c.sync(0, check=False) == lstmod.ERR_OVERFLOW
        st = c.stats(0)
        assert st["overflow"] & (1 << kind) and st["needed"][kind] == ora.counts[kind]
        with pytest.raises(lstmod.LstError):
            c.quintuplets(0)
        c.close()
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    cfg.cap_hits = 100
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    with pytest.raises(lstmod.LstError) as e:
        c.load_event(0, ev.x, ev.y, ev.z, ev.module, ev.side)
    assert e.value.status == lstmod.ERR_OVERFLOW
    c.close()
    # bad module ids / sides: dropped, counted, status LST_ERR_ARG; the rest is processed
    c = lstmod.Lst.from_synth(geom, mmap)
    mod = ev.module.copy(); side = ev.side.copy()
    mod[:5] = geom.n_modules + 3; mod[5:8] = -1; side[8:10] = 2
    c.load_event(0, ev.x, ev.y, ev.z, mod, side)
    c.run(0)
    assert c.sync(0, check=False) == lstmod.ERR_ARG
    assert c.stats(0)["bad_hits"] == 10 and c.stats(0)["n_hits"] == ev.n - 10
    with pytest.raises(lstmod.LstError):
        c.run(1)                                     # slot never loaded -> LST_ERR_STATE
    c.close()


def test_overflow_recovery_by_regrowing(lstmod, geom, mmap, o32, run_oracle):
    """BASELINE.json configs[3] "candidate-buffer overflow handling", the recovery half: start from capacities far too small
    for the PU300-like stress event, follow lst_grown_config until the event fits (a stage that overflowed hands the next one
    a clamped input, so it can take one round per object class), and the result equals the oracle's."""
    ev = synth.generate_event(geom, 3, 0)
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    cfg.cap_hits, cfg.cap_md, cfg.cap_seg, cfg.cap_t3, cfg.cap_t5 = 160 * 1024, 8 * 1024, 8 * 1024, 8 * 1024, 1024
    rounds = 0
    while True:
        c = lstmod.Lst.from_synth(geom, mmap, cfg)
        c.load_event(0, ev.x, ev.y, ev.z, ev.module, ev.side)
        c.run(0)
        status = c.sync(0, check=False)
        if status == lstmod.OK:
            break
        assert status == lstmod.ERR_OVERFLOW and rounds < 5
        new = c.grown_config(0)
        assert any(getattr(new, f) > getattr(cfg, f) for f in ("cap_md", "cap_seg", "cap_t3", "cap_t5"))
        assert all(getattr(new, f) >= getattr(cfg, f) for f in ("cap_hits", "cap_md", "cap_seg", "cap_t3", "cap_t5"))
        c.close()
        cfg = new
        rounds += 1
    assert 1 <= rounds <= 4
    ora = run_oracle(o32, ev)
    parity.compare(parity.gpu_tables(c, 0), parity.oracle_tables(ora), "regrown")
    same = c.grown_config(0)
    assert [getattr(same, f) for f in ("cap_md", "cap_seg", "cap_t3", "cap_t5")] == [getattr(cfg, f) for f in ("cap_md", "cap_seg", "cap_t3", "cap_t5")]
    c.close()


def test_multi_stream_pipeline(ctx, o32, run_oracle, geom):
    """BASELINE.json configs[2] in miniature: 8 events on 4 streams, slots recycled, arena reused."""
    import torch
    streams = [torch.cuda.Stream() for _ in range(4)]
    evs = [synth.generate_event(geom, 1, 60 + i, n_particles=800) for i in range(8)]
    for rnd in range(2):
        for s in range(4):
            ev = evs[4 * rnd + s]
            ctx.load_event(s, ev.x, ev.y, ev.z, ev.module, ev.side, streams[s])
            ctx.run(s, streams[s])
        for s in range(4):
            ctx.sync(s, streams[s])
            got = parity.gpu_tables(ctx, s, streams[s])
            parity.compare(got, parity.oracle_tables(run_oracle(o32, evs[4 * rnd + s])), f"stream {s} round {rnd}")


@pytest.mark.parametrize("how", ["shifted", "random", "near_pi"])
def test_search_windows_never_change_the_result(lstmod, geom, mmap, o32, run_oracle, how):
    """lst_geometry.phi only orders hits for the windowed search: with a
    wrong reference azimuth per module -- shifted, random, or sitting on the +-pi cut -- windows
    degrade to full scans where an azimuth wrap is possible and the object sets stay those of the
    oracle."""
    rng = np.random.default_rng(5)
    phi = {"shifted": geom.phi + 1.0, "random": rng.uniform(-np.pi, np.pi, geom.n_modules),
           "near_pi": geom.phi + np.pi - 0.05}[how]
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    c = lstmod.Lst(geom.layer, mmap.row_offsets, mmap.targets, cfg, phi=phi)
    ev = synth.generate_event(geom, 1, 77, n_particles=1200)
    _, st = check_event(c, o32, run_oracle, ev, label=how)
    assert st["needed"][3] > 500
    c.close()


def test_fetch_batch_equals_per_slot_fetch(ctx, lstmod, geom):
    """lst_sync_batch + lst_fetch_batch (one call per batch, asynchronous copies into pinned host
    buffers) return exactly what the per-slot lst_sync + lst_fetch_* calls return, for every class."""
    import torch
    evs = [synth.generate_event(geom, 1, 80 + i, n_particles=300 + 400 * i) for i in range(3)]
    evs.append(synth.Event(*(np.zeros(0, t) for t in (np.float32, np.float32, np.float32, np.int32, np.uint8, np.int32)), {}))
    stream = torch.cuda.Stream()
    # pinned host input: the binning kernel reads it over PCIe itself (no memcpy); slot 6 gets the same event as
    # slot 3 from pageable memory (cudaMemcpyAsync path) and must produce the same arrays
    pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
    ctx.load_events(2, [tuple(pin(a) for a in (e.x, e.y, e.z, e.module, e.side)) for e in evs], stream=stream)
    ctx.run_batch(2, len(evs), stream)
    assert ctx.sync_batch(2, len(evs), stream) == 0
    pageable = parity.run_gpu(ctx, evs[1], slot=6, stream=stream)
    pinned = parity.gpu_tables(ctx, 3, stream)
    # "packed" host layout (one pinned block, arrays on 256-byte boundaries): one copy-engine transfer per event
    pk = lstmod.packed_event_buffers(evs[1].n)
    for dst, src in zip(pk[:5], (evs[1].x, evs[1].y, evs[1].z, evs[1].module, evs[1].side)):
        dst[:] = src
    ctx.load_event(7, *pk[:5], stream)
    ctx.run(7, stream)
    ctx.sync(7, stream)
    packed = parity.gpu_tables(ctx, 7, stream)
    for kind in range(4):
        assert np.array_equal(packed[kind][0], pinned[kind][0]) and np.array_equal(packed[kind][1], pinned[kind][1], equal_nan=True)
    for kind in range(4):
        assert np.array_equal(pageable[kind][0], pinned[kind][0]) and np.array_equal(pageable[kind][1], pinned[kind][1], equal_nan=True)
    for kind in range(4):
        need = [ctx.stats(2 + b)["needed"][kind] for b in range(len(evs))]
        idx = [torch.full((n + 3, parity_width(kind)[0]), -7, dtype=torch.int32).pin_memory().numpy() for n in need]
        val = [torch.full((n + 3, parity_width(kind)[1]), -7.0, dtype=torch.float32).pin_memory().numpy() for n in need]
        counts = ctx.fetch_batch(2, kind, idx, val, stream=stream, wait=False)
        stream.synchronize()
        assert counts == need
        for b, n in enumerate(need):
            assert np.array_equal(idx[b][:n], ctx.fetch_hit_indices(2 + b, kind, stream))
            assert np.array_equal(val[b][:n], ctx.fetch_values(2 + b, kind, stream), equal_nan=True)
            assert (idx[b][n:] == -7).all() and (val[b][n:] == -7.0).all()      # nothing written past the count
    # a buffer that is too small is refused before anything is copied
    small = [np.zeros((1, 10), np.int32) for _ in evs]
    with pytest.raises(Exception):
        ctx.fetch_batch(2, 3, small, None, stream=stream)


def parity_width(kind):
    return (2, 4, 6, 10)[kind], (4, 4, 2, 5)[kind]


def test_parity_in_the_bench_launch_configuration(lstmod, geom, mmap, o32, run_oracle):
    """BASELINE.json configs[2] exactly as bench.py times it: 64 PU200-like events (seeds 0..63), device-resident
    hit SoA, 64 slots, 4 CUDA streams x 16-event batched launches, two passes over the same arena.  Every event:
    object and candidate counts equal the oracle's; 8 sampled events: every object and float compared."""
    import torch
    n_ev, n_streams = 64, 4
    per = n_ev // n_streams
    evs = [synth.generate_event(geom, 1, s) for s in range(n_ev)]
    cfg = lstmod.default_config()
    cfg.n_slots = n_ev
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    d_in = [[torch.from_numpy(a).cuda() for a in (e.x, e.y, e.z, e.module, e.side)] for e in evs]
    streams = [torch.cuda.Stream() for _ in range(n_streams)]
    torch.cuda.synchronize()
    for _ in range(2):                                  # second pass: slots recycled by k_reset
        for s, st in enumerate(streams):
            c.load_events(s * per, d_in[s * per:(s + 1) * per], stream=st)
            c.run_batch(s * per, per, st)
    for s, st in enumerate(streams):
        assert c.sync_batch(s * per, per, st) == 0
    sampled = {0, 7, 15, 16, 31, 42, 48, 63}            # first / last of a batch, first / last of a stream
    for k, ev in enumerate(evs):
        ora = run_oracle(o32, ev)
        st = c.stats(k)
        assert st["needed"] == ora.counts and st["candidates"] == ora.candidates and st["n_hits"] == ev.n, (k, st)
        if k in sampled:
            parity.compare(parity.gpu_tables(c, k, streams[k // per]), parity.oracle_tables(ora), f"bench slot {k}")
    c.close()


@pytest.mark.timeout(900)
def test_occupancy_sweep_1m_hits_every_object(lstmod, geom, mmap, o32):
    """BASELINE.json configs[4] at its maximum size (1 M hits; mini-doublet and segment stages only), in the launch
    configuration `bench.py --sweep` times.  The oracle runs both stages in full (60 M mini-doublet and 1.77 G segment
    candidates, about 40 s): ALL 877 k mini-doublets and ALL 17.1 M segments are compared, sets bit-exact and floats
    within tolerance -- so every chunk that overflows the on-chip stash and is walked a second time (lst_stats.rewalks)
    is checked too, not a sample of them."""
    import torch
    ev = synth.generate_occupancy_event(geom, 1000000, seed=4)
    ora = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, stages=2)
    cfg = lstmod.default_config()
    cfg.n_slots, cfg.cap_hits, cfg.cap_md, cfg.cap_seg, cfg.cap_t3, cfg.cap_t5 = 1, ev.n, 2 * ev.n, 20 * ev.n, 1024, 1024
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    st = torch.cuda.Stream()
    d_in = [torch.from_numpy(a).cuda() for a in (ev.x, ev.y, ev.z, ev.module, ev.side)]
    c.load_events(0, [d_in], stream=st)
    c.run_stage(0, 1, lstmod.MD, st)
    c.run_stage(0, 1, lstmod.SEG, st)
    assert c.sync(0, st) == 0
    stats = c.stats(0)
    assert stats["needed"][:2] == ora.counts[:2] and stats["candidates"][:2] == ora.candidates[:2] and stats["n_hits"] == ev.n
    assert stats["needed"][1] <= stats["evaluated"][1] <= stats["candidates"][1]
    gpu = {k: (c.fetch_hit_indices(0, k, st), c.fetch_values(0, k, st)) for k in (0, 1)}
    worst = parity.compare(gpu, parity.oracle_tables(ora), "1M hits", classes=(0, 1))
    print(f"1 M hits: {stats['needed'][:2]} objects, rewalks {stats['rewalks'][:2]}, max rel err {worst}")
    # CSR offsets of the segments: ascending, every segment filed under its inner mini-doublet
    view = lstmod.SegView()
    assert c.lib.lst_get_segments(c.h, 0, view) == 0 and view.n == stats["needed"][1]
    seg_md = lstmod.DeviceArray(view.md, (view.n, 2), "<i4", c).torch()
    md_start = lstmod.DeviceArray(view.md_start, (stats["needed"][0] + 1,), "<i4", c).torch()
    assert int(md_start[0]) == 0 and int(md_start[-1]) == view.n and bool((md_start[1:] >= md_start[:-1]).all())
    assert torch.equal(torch.repeat_interleave(torch.arange(stats["needed"][0], device="cuda"), (md_start[1:] - md_start[:-1]).long()),
                       seg_md[:, 0].long())
    c.close()


@pytest.mark.timeout(600)
@pytest.mark.parametrize("config,seed,n_particles", [(0, 0, None), (0, 3, None), (1, 21, 900), (1, 0, None), (3, 0, None)])
def test_duplicate_cleaning_parity(ctx, lstmod, o32, run_oracle, geom, config, seed, n_particles):
    """Stage LST_CLEAN (DESIGN.md section 1 [D]) against the oracle's all-pairs definition: the kept set must be
    IDENTICAL (as hit tuples; the decision is taken on both sides on the same fp32 score), the kept list ascending and
    consistent with the flags; incl. the full PU200-like event (10.5 k quintuplets, 110 M pairs in the oracle) and the
    PU300-like stress event of configs[3] (17.8 k quintuplets, 317 M pairs: half a minute of oracle)."""
    import torch
    ev = synth.generate_event(geom, config, seed) if n_particles is None else synth.generate_event(geom, config, seed, n_particles=n_particles)
    st = torch.cuda.Stream()
    gpu = parity.run_gpu(ctx, ev, slot=1, stream=st)
    with pytest.raises(lstmod.LstError):
        ctx.track_candidates(1)                                   # stage not run yet -> LST_ERR_STATE
    ctx.run_stage(1, 1, lstmod.CLEAN, st)
    ctx.sync(1, st)
    ora = run_oracle(o32, ev)
    keep_o = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz, 7)
    tc = ctx.track_candidates(1)
    keep_g = tc["keep"].torch().cpu().numpy().astype(bool)
    kept_idx = ctx.fetch_kept(1, st)
    g_hits = gpu[3][0]
    assert len(keep_g) == len(g_hits) == len(keep_o) and tc["n"] == ctx.stats(1)["n_kept"] == int(keep_g.sum())
    assert np.array_equal(kept_idx, np.nonzero(keep_g)[0])
    assert np.array_equal(tc["t5"].torch().cpu().numpy(), kept_idx)
    as_set = lambda h: set(map(tuple, h.tolist()))
    assert as_set(g_hits[keep_g]) == as_set(ora.t5_hits()[keep_o])
    # scores: the same fp32 addition on both sides
    score_g = tc["score"].torch().cpu().numpy()
    gs, _ = parity.sort_rows(g_hits, score_g.reshape(-1, 1))
    order_g = np.lexsort(g_hits.T[::-1]); order_o = np.lexsort(ora.t5_hits().T[::-1])
    assert np.array_equal(score_g[order_g], (ora.t5_chi2xy + ora.t5_chi2rz).astype(np.float32)[order_o])
    assert 0 < keep_g.sum() < len(keep_g)


def test_duplicate_cleaning_batch_empty_and_ties(lstmod, geom, mmap, o32, run_oracle):
    """A batch of slots through one set of LST_CLEAN launches (incl. an empty event and an event without quintuplets),
    a second threshold (t5_dup_min_shared = 6, the smallest the library accepts), and the stage order check."""
    import torch
    cfg = lstmod.default_config()
    cfg.n_slots, cfg.t5_dup_min_shared = 4, 6
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    st = torch.cuda.Stream()
    full = synth.generate_event(geom, 1, 8, n_particles=600)
    lower_only = np.nonzero(full.side == 0)[0]
    sub = synth.Event(full.x[lower_only], full.y[lower_only], full.z[lower_only], full.module[lower_only], full.side[lower_only],
                      full.truth[lower_only], {})
    empty = synth.Event(*(np.zeros(0, t) for t in (np.float32, np.float32, np.float32, np.int32, np.uint8, np.int32)), {})
    evs = [full, empty, sub, synth.generate_event(geom, 0, 9)]
    c.load_events(0, [(e.x, e.y, e.z, e.module, e.side) for e in evs], stream=st)
    c.run_stage(0, 4, lstmod.MD, st)
    with pytest.raises(lstmod.LstError):
        c.run_stage(0, 4, lstmod.CLEAN, st)                       # needs the quintuplets first
    for stage in (lstmod.SEG, lstmod.T3, lstmod.T5, lstmod.CLEAN):
        c.run_stage(0, 4, stage, st)
    assert c.sync_batch(0, 4, st) == 0
    for k, ev in enumerate(evs):
        ora = run_oracle(o32, ev)
        keep_o = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz, 6)
        hits = c.fetch_hit_indices(k, lstmod.T5, st)
        kept = c.fetch_kept(k, st)
        assert c.stats(k)["n_kept"] == int(keep_o.sum()) == len(kept)
        assert set(map(tuple, hits[kept].tolist())) == set(map(tuple, ora.t5_hits()[keep_o].tolist()))
    assert c.stats(1)["n_kept"] == 0 and c.stats(2)["n_kept"] == 0
    # lst_fetch_batch(kind = LST_CLEAN): the kept quintuplets only, pinned (kernel writes) and pageable (copy engine) buffers
    for pinned in (True, False):
        mk = (lambda shape, dt: torch.zeros(shape, dtype=dt).pin_memory().numpy()) if pinned else (lambda shape, dt: np.zeros(shape, {torch.int32: np.int32, torch.float32: np.float32}[dt]))
        idx = [mk((c.stats(k)["n_kept"] + 2, 10), torch.int32) for k in range(4)]
        val = [mk((c.stats(k)["n_kept"] + 2, 5), torch.float32) for k in range(4)]
        counts = c.fetch_batch(0, lstmod.CLEAN, idx, val, stream=st, wait=True)
        for k in range(4):
            kept = c.fetch_kept(k, st)
            assert counts[k] == len(kept)
            assert np.array_equal(idx[k][:len(kept)], c.fetch_hit_indices(k, lstmod.T5, st)[kept])
            assert np.array_equal(val[k][:len(kept)], c.fetch_values(k, lstmod.T5, st)[kept])
    c.close()


@pytest.mark.parametrize("K", [6, 8, 10])
def test_duplicate_cleaning_with_duplicated_hits(lstmod, geom, mmap, o32, run_oracle, K):
    """Rule [D] for every threshold the library accepts, on events whose hits all exist TWICE (equal coordinates, different
    original indices): a true quintuplet becomes 2^10 quintuplets that share 0 .. 9 original hits in every pattern,
    among them pairs with five common layers and one common hit each -- 5 shared hits and no common mini-doublet, the
    case the incidence search cannot see and the reason thresholds below 6 are refused.  Kept sets equal the oracle's
    all-pairs definition; scores tie massively (identical coordinates), so the tuple order of D3 decides."""
    import torch
    cfg = lstmod.default_config()
    cfg.n_slots, cfg.t5_dup_min_shared = 2, K
    cfg.cap_t3, cfg.cap_t5 = 1 << 20, 1 << 20
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    st = torch.cuda.Stream()
    for slot, seed in enumerate((703, 709)):
        base = synth.generate_event(geom, 1, seed, n_particles=4)
        x, y, z, mod, side = (np.tile(a, 2) for a in (base.x, base.y, base.z, base.module, base.side))
        ev = synth.Event(x, y, z, mod, side, np.full(len(x), -1, np.int32), {})
        gpu = parity.run_gpu(c, ev, slot=slot, stream=st)
        c.run_stage(slot, 1, lstmod.CLEAN, st)
        c.sync(slot, st)
        ora = run_oracle(o32, ev)
        assert c.stats(slot)["needed"] == ora.counts and ora.counts[3] >= 1024
        keep_o = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz, K)
        kept = c.fetch_kept(slot, st)
        as_set = lambda h: set(map(tuple, h.tolist()))
        assert as_set(gpu[3][0][kept]) == as_set(ora.t5_hits()[keep_o]) and len(kept) == int(keep_o.sum())
        if K == 6:      # the input does hold pairs that share exactly 5 hits and no mini-doublet
            h = ora.t5_hits()[:1024]
            shared = (h[:, None, :] == h[None, :, :]).sum(2)
            mds = h.reshape(len(h), 5, 2)
            common_md = (mds[:, None, :, :] == mds[None, :, :, :]).all(3).any(2)
            assert ((shared == 5) & ~common_md).any()
    c.close()


def test_cuda_graph_capture_and_replay(ctx, o32, run_oracle, geom):
    """include/lst.h: lst_load_event(s) (device input) + lst_run_batch only enqueue work, so the sequence can be captured
    into a CUDA graph.  Capture once over fixed device buffers, then replay with two different events copied into
    those buffers: each replay must give that event's oracle result."""
    import torch
    evs = [synth.generate_event(geom, 1, 90 + i, n_particles=1000) for i in range(2)]
    n_max = max(e.n for e in evs)
    bufs = [torch.zeros(n_max, dtype=dt, device="cuda") for dt in (torch.float32, torch.float32, torch.float32, torch.int32, torch.uint8)]
    st = torch.cuda.Stream()

    def fill(ev):          # pad with hits of an invalid side? no: the graph is captured for a fixed n, so replay events are cut to it
        n = min(e.n for e in evs)
        for b, a in zip(bufs, (ev.x, ev.y, ev.z, ev.module, ev.side)):
            b[:n].copy_(torch.from_numpy(a[:n]))
        return synth.Event(ev.x[:n], ev.y[:n], ev.z[:n], ev.module[:n], ev.side[:n], ev.truth[:n], {})

    n = min(e.n for e in evs)
    view = [b[:n] for b in bufs]
    fill(evs[0])
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=st):
        ctx.load_events(3, [view], stream=st)
        ctx.run_batch(3, 1, st)
    for ev in (evs[1], evs[0]):
        cut = fill(ev)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        ctx.sync(3, st)
        parity.compare(parity.gpu_tables(ctx, 3, st), parity.oracle_tables(run_oracle(o32, cut)), "graph replay")


def test_slots_driven_from_host_threads(ctx, o32, run_oracle, geom):
    """include/lst.h: distinct slots may be driven from distinct host threads (each with its own stream)."""
    import threading
    import torch
    evs = [synth.generate_event(geom, 1, 95 + i, n_particles=700) for i in range(4)]
    pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
    out, err = {}, []

    def work(k):
        try:
            st = torch.cuda.Stream()
            e = evs[k]
            for _ in range(3):
                ctx.load_event(k, *(pin(a) for a in (e.x, e.y, e.z, e.module, e.side)), st)   # stage-in path (shared internal stream)
                ctx.run(k, st)
                ctx.sync(k, st)
            out[k] = parity.gpu_tables(ctx, k, st)
        except Exception as ex:       # noqa: BLE001
            err.append(ex)

    ts = [threading.Thread(target=work, args=(k,)) for k in range(4)]
    [t.start() for t in ts]
    [t.join() for t in ts]
    assert not err, err
    for k in range(4):
        parity.compare(out[k], parity.oracle_tables(run_oracle(o32, evs[k])), f"thread {k}")


def test_fuzz_small_events(ctx, o32, run_oracle, geom):
    """Seeded random small events of adversarial structure (noise only; all hits in a handful of modules; duplicated
    hits; coordinates scaled far off the detector; mixtures): sets, counts and floats equal the oracle's every time."""
    rng = np.random.default_rng(2024)
    n_obj = np.zeros(4, np.int64)
    for trial in range(24):
        kind = trial % 6
        base = synth.generate_event(geom, 1, 700 + trial, n_particles=12 if kind == 3 else int(rng.integers(20, 400)))
        x, y, z, mod, side = (a.copy() for a in (base.x, base.y, base.z, base.module, base.side))
        if kind == 1:       # noise only: positions scrambled among the hits of each (module, side) -- keeps them on the sensors
            p = rng.permutation(len(x)); order = np.lexsort((p, side, mod)); src = np.lexsort((np.arange(len(x)), side, mod))
            x[src], y[src], z[src] = x[order], y[order], z[order]
        elif kind == 2:     # everything folded into 12 modules of consecutive layers (heavy bins, long lists)
            keep = np.isin(mod, np.concatenate([np.arange(0, 3), 408 + np.arange(0, 3), 1008 + np.arange(0, 3), 1848 + np.arange(0, 3)]))
            if keep.sum() < 4:
                keep[:] = True
            x, y, z, mod, side = x[keep], y[keep], z[keep], mod[keep], side[keep]
        elif kind == 3:     # every hit twice (equal keys: ties by original index; a T5 becomes 2^10 of them)
            x, y, z, mod, side = (np.tile(a, 2) for a in (x, y, z, mod, side))
        elif kind == 4:     # a tenth of the hits far away / tiny / negative radius direction
            m = rng.random(len(x)) < 0.1
            x[m] *= rng.choice([1e-6, 1e4, -1.0], m.sum()).astype(np.float32)
            z[m] *= np.float32(50.0)
        elif kind == 5:     # sides swapped for a third of the modules
            m = (mod % 3) == 0
            side[m] = 1 - side[m]
        ev = synth.Event(x.astype(np.float32), y.astype(np.float32), z.astype(np.float32), mod.astype(np.int32), side.astype(np.uint8),
                         np.full(len(x), -1, np.int32), {})
        _, st = check_event(ctx, o32, run_oracle, ev, slot=trial % 8, label=f"fuzz{trial}/kind{kind}")
        n_obj += np.asarray(st["needed"])
    assert n_obj[0] > 5000 and n_obj[3] > 50, n_obj


def test_parity_with_non_default_cut_constants(lstmod, geom, mmap, o32):
    """Every threshold comes from lst_config, none is baked into a kernel: with tightened / loosened constants on BOTH
    sides (same fp32 values) the object sets and floats still agree, and differ from the default result."""
    changes = dict(z_lum=10.0, seg_cos_eps=0.999998, seg_sin_eps=0.0015, t3_kappa_max=0.012, t5_dkappa_max=0.0004,
                   t5_chi2xy_max=60.0, t5_kappa_max=0.0125)
    arrays = dict(md_dz_res=0.8, seg_z0_max=0.7, t3_chi2rz_max=0.5, t5_chi2rz_max=1.5, md_eps=0.9)
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    ocfg = o32.default_config()
    for k, v in changes.items():
        setattr(cfg, k, v)
        setattr(ocfg, k, v)
    for k, f in arrays.items():
        a, b = getattr(cfg, k), getattr(ocfg, k)
        for i in range(len(a)):
            a[i] = np.float32(a[i] * f)
            b[i] = a[i]
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    ev = synth.generate_event(geom, 1, 55, n_particles=1500)
    gpu = parity.run_gpu(c, ev)
    ora = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, cfg=ocfg)
    parity.compare(gpu, parity.oracle_tables(ora), "custom cuts")
    assert c.stats(0)["needed"] == ora.counts
    default = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side)
    assert all(a != b for a, b in zip(default.counts, ora.counts)), (default.counts, ora.counts)
    c.close()


@pytest.mark.parametrize("how", ["thinned", "fat"])
def test_parity_with_other_module_maps(lstmod, geom, mmap, o32, how):
    """The module map is an INPUT that defines the search space (reading 6): a map with 30 % of its connections
    removed, and a fat one (every module of the next layer within +-3 rings and +-3 azimuth steps: rows of up to 49
    targets, more than one warp tile per owner) must give the oracle's sets for that same map."""
    rng = np.random.default_rng(17)
    if how == "thinned":
        rows = [np.asarray(mmap.targets[mmap.row_offsets[a]:mmap.row_offsets[a + 1]]) for a in range(geom.n_modules)]
        rows = [r[rng.random(len(r)) > 0.3] for r in rows]
    else:
        nphi = {l: int((geom.layer == l).sum()) // 24 for l in range(6)}
        base = {l: int(np.nonzero(geom.layer == l)[0][0]) for l in range(6)}
        rows = []
        for a in range(geom.n_modules):
            l = int(geom.layer[a])
            if l == 5:
                rows.append(np.zeros(0, np.int64))
                continue
            ring, i = divmod(a - base[l], nphi[l])
            i2 = int(round(i * nphi[l + 1] / nphi[l]))
            t = [base[l + 1] + r * nphi[l + 1] + (i2 + d) % nphi[l + 1] for r in range(max(0, ring - 3), min(24, ring + 4)) for d in range(-3, 4)]
            rows.append(np.unique(t))
        assert max(len(r) for r in rows) > 32
    offs = np.zeros(geom.n_modules + 1, np.int32)
    offs[1:] = np.cumsum([len(r) for r in rows])
    tg = np.concatenate(rows).astype(np.int32)
    cfg = lstmod.default_config()
    cfg.n_slots = 1
    c = lstmod.Lst(geom.layer, offs, tg, cfg, phi=geom.phi)
    ev = synth.generate_event(geom, 1, 66, n_particles=1500)
    gpu = parity.run_gpu(c, ev)
    ora = o32.run(geom.layer, offs, tg, ev.x, ev.y, ev.z, ev.module, ev.side)
    parity.compare(gpu, parity.oracle_tables(ora), how)
    st = c.stats(0)
    assert st["needed"] == ora.counts and st["candidates"] == ora.candidates and ora.counts[3] > 100
    c.close()


def test_create_destroy_returns_the_arena(lstmod, geom, mmap):
    """lst_create makes ONE arena allocation (plus the small tables); lst_destroy gives everything back: 20 create / run /
    destroy cycles leave the device's free memory where it was."""
    import torch
    torch.cuda.synchronize()
    ev = synth.generate_event(geom, 0, 4)
    free0 = torch.cuda.mem_get_info()[0]
    for _ in range(20):
        cfg = lstmod.default_config()
        cfg.n_slots = 3
        c = lstmod.Lst.from_synth(geom, mmap, cfg)
        total, per_slot = c.arena_bytes()
        assert total == 3 * per_slot and torch.cuda.mem_get_info()[0] <= free0 - total
        c.load_event(2, ev.x, ev.y, ev.z, ev.module, ev.side)
        c.run(2)
        assert c.sync(2) == 0
        c.close()
    torch.cuda.synchronize()
    assert abs(torch.cuda.mem_get_info()[0] - free0) <= 64 << 20


def test_module_map_builder_parity(lstmod, geom, mmap, o64):
    """lst_build_module_map [B] against the oracle (binary64 on both sides): identical CSR (offsets and ascending
    targets) on the BASELINE geometry, with other parameters, and on a jittered geometry; the two-call size protocol;
    and the map it builds drives the path to the same result as the test-side map."""
    import ctypes as C
    mg = synth.map_geometry(geom)
    args = (mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"])
    offs, tg, ms = lstmod.build_module_map(*args)
    o_offs, o_tg = o64.build_map(*args)
    assert np.array_equal(offs, o_offs) and np.array_equal(tg, o_tg) and len(tg) == 69630
    assert np.array_equal(offs, mmap.row_offsets) and np.array_equal(tg, mmap.targets)
    print(f"map builder: count {ms[0]:.3f} ms, fill {ms[1]:.3f} ms for {geom.n_modules} modules, {len(tg)} connections")
    for kw in (dict(pt_min=0.6), dict(pt_min=1.5, z0_max=5.0), dict(pad_phi=0.0, pad_z=0.0), dict(b_tesla=2.0)):
        g_o, g_t, _ = lstmod.build_module_map(*args, **kw)
        r_o, r_t = o64.build_map(*args, **kw)
        assert np.array_equal(g_o, r_o) and np.array_equal(g_t, r_t), kw
    rng = np.random.default_rng(8)                                   # another detector: jittered radii, gaps, widths, azimuths
    jit = (mg["layer"], mg["phi"] + rng.normal(0, 0.02, geom.n_modules), mg["rho"] * rng.uniform(0.97, 1.03, geom.n_modules),
           mg["gap"] * rng.uniform(0.5, 1.5, geom.n_modules), mg["hw"] * rng.uniform(0.6, 1.2, geom.n_modules),
           mg["zlo"] + rng.normal(0, 0.5, geom.n_modules), mg["zhi"] + rng.normal(0, 0.5, geom.n_modules))
    g_o, g_t, _ = lstmod.build_module_map(*jit)
    r_o, r_t = o64.build_map(*jit)
    assert np.array_equal(g_o, r_o) and np.array_equal(g_t, r_t) and len(g_t) != 69630
    # size protocol and argument errors through the C-ABI
    lib = lstmod.load_library()
    keep = [np.ascontiguousarray(a) for a in args]
    g = lstmod.MapGeometry(geom.n_modules, *[lstmod._ptr(a) for a in keep])
    ro = np.zeros(geom.n_modules + 1, np.int32)
    small = np.zeros(10, np.int32)
    total = C.c_int64(0)
    st = lib.lst_build_module_map(C.byref(g), None, 0, lstmod._ptr(ro), lstmod._ptr(small), 10, C.byref(total), None)
    assert st == lstmod.ERR_OVERFLOW and total.value == 69630 and np.array_equal(ro, o_offs) and not small.any()
    bad = lstmod.MapGeometry(geom.n_modules, lstmod._ptr(keep[0]), 0, *[lstmod._ptr(a) for a in keep[2:]])
    assert lib.lst_build_module_map(C.byref(bad), None, 0, lstmod._ptr(ro), lstmod._ptr(small), 10, C.byref(total), None) == lstmod.ERR_ARG
    # the built map feeds lst_create
    c = lstmod.Lst(geom.layer, offs, tg, phi=geom.phi)
    ev = synth.generate_event(geom, 0, 2)
    c.load_event(0, ev.x, ev.y, ev.z, ev.module, ev.side)
    c.run(0)
    assert c.sync(0) == 0 and c.stats(0)["needed"][3] > 50
    c.close()


@pytest.mark.timeout(300)
def test_soak_mixed_sizes_repeatable(lstmod, geom, mmap, o32, run_oracle):
    """400 back-to-back steps of 16 slots on 4 streams with events of very different sizes in one batch (tiny, PU200-like,
    PU300-like, empty), the cleaning stage every third step and the pixel stage every other step: no hang of the
    ordered-output waits, identical counts at every check, and the last state still equals the oracle.  (A two-minute run of
    the round-1 loop, 77 k steps / 4.9 M events, is recorded in DESIGN.md.)"""
    import torch
    evs = [synth.generate_event(geom, 1, 300 + i, n_particles=n) for i, n in enumerate((30, 6000, 0, 900, 2500, 1, 400, 5000))]
    evs += [synth.generate_event(geom, 3, 2), synth.generate_event(geom, 0, 5)] + [synth.generate_event(geom, 1, 310 + i, n_particles=1500) for i in range(6)]
    cfg = lstmod.default_config()
    cfg.n_slots = 16
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    streams = [torch.cuda.Stream() for _ in range(4)]
    d_in = [[torch.from_numpy(a).cuda() for a in (e.x, e.y, e.z, e.module, e.side)] for e in evs]
    sds = [synth.generate_seeds(e, 300 + i) for i, e in enumerate(evs)]
    d_sd = [[torch.from_numpy(a).cuda() for a in sd.arrays()] for sd in sds]
    ref = None
    for step in range(400):
        for s, st in enumerate(streams):
            c.load_events(4 * s, d_in[4 * s:4 * s + 4], stream=st)
            if step % 2 == 1:
                c.load_seeds(4 * s, d_sd[4 * s:4 * s + 4], stream=st)
            c.run_batch(4 * s, 4, st)
            if step % 3 == 0:
                c.run_stage(4 * s, 4, lstmod.CLEAN, st)
            if step % 2 == 1:
                c.run_stage(4 * s, 4, lstmod.PIXEL, st)
        if step % 100 == 99:
            for s, st in enumerate(streams):
                assert c.sync_batch(4 * s, 4, st) == 0
            cur = [tuple(c.stats(k)["needed"]) + tuple(c.stats(k)["pix_needed"]) for k in range(16)]
            ref = ref or cur
            assert cur == ref
    for k in (1, 8, 9):
        ora = run_oracle(o32, evs[k])
        assert list(ref[k][:4]) == ora.counts
        parity.compare(parity.gpu_tables(c, k, streams[k // 4]), parity.oracle_tables(ora), f"soak slot {k}")
    ora = run_oracle(o32, evs[4], seeds=sds[4].arrays())
    assert list(ref[4][4:]) == [ora.pix[0]["n"], ora.pix[1]["n"]] and ora.pix[0]["n"] > 1000
    c.close()


@pytest.mark.parametrize("config,seed", [(0, 0), (1, 0), (3, 0)])
def test_reduced_precision_store_parity(lstmod, geom, mmap, o32, run_oracle, config, seed):
    """lst_config.store_half (DESIGN.md section 1 [H]): the output floats no selection reads are kept as
    binary16.  Relaxed parity rule (parity.compare_half): identical object sets and candidate counts; every fetched value is
    the round-to-nearest-even binary16 of the oracle's fp32 value (atan2f outputs: within one binary16 ulp); the duplicate
    cleaning, which reads chi2xy + chi2rz, still equals the fp32 oracle's kept set because its score is kept in fp32."""
    import torch
    cfg = lstmod.default_config()
    cfg.n_slots, cfg.store_half = 2, 1
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    st = torch.cuda.Stream()
    ev = synth.generate_event(geom, config, seed)
    gpu = parity.run_gpu(c, ev, slot=1, stream=st)
    ora = run_oracle(o32, ev)
    n_off = parity.compare_half(gpu, parity.oracle_tables(ora), o32, f"half C{config}")
    stt = c.stats(1)
    assert stt["needed"] == ora.counts and stt["candidates"] == ora.candidates
    # views expose the binary16 arrays; they hold what the fetch returns
    t5 = c.quintuplets(1)
    assert t5["f"].torch().dtype == torch.float16
    order = np.lexsort(gpu[3][0].T[::-1])
    assert np.array_equal(t5["f"].torch().cpu().numpy()[order].view(np.uint16), parity.sort_rows(*gpu[3])[1].view(np.uint16))
    seg = c.segments(1)
    assert np.array_equal(seg["f"].torch().cpu().numpy().view(np.uint16), gpu[1][1].view(np.uint16))
    # cleaning: same kept set as the fp32 oracle
    if config != 3:
        c.run_stage(1, 1, lstmod.CLEAN, st)
        c.sync(1, st)
        keep_o = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz, 7)
        kept = c.fetch_kept(1, st)
        as_set = lambda h: set(map(tuple, h.tolist()))
        assert as_set(gpu[3][0][kept]) == as_set(ora.t5_hits()[keep_o])
        # lst_fetch_batch of the kept quintuplets: binary16 rows of the same table, pinned and pageable buffers
        for pinned in (True, False):
            idx = np.zeros((len(kept) + 1, 10), np.int32)
            val = np.zeros((len(kept) + 1, 5), np.float16)
            if pinned:
                idx, val = torch.from_numpy(idx).pin_memory().numpy(), torch.from_numpy(val).pin_memory().numpy()
            assert c.fetch_batch(1, lstmod.CLEAN, [idx], [val], stream=st, wait=True) == [len(kept)]
            assert np.array_equal(idx[:len(kept)], gpu[3][0][kept]) and np.array_equal(val[:len(kept)].view(np.uint16), gpu[3][1][kept].view(np.uint16))
    print(f"half store C{config}: {stt['needed']} objects, {n_off} atan2f outputs one binary16 ulp off")
    c.close()


def test_launches_in_flight_hint_changes_grids_only(lstmod, geom, mmap, o32, run_oracle):
    """lst_config.launches_in_flight (include/lst.h): a sizing hint.  With it set to 4 -- single launches, batches of 3 and of
    16, the optional stages, an event that needs the direct walks -- the results still equal the oracle's; negative values are
    refused."""
    import torch
    cfg = lstmod.default_config()
    cfg.launches_in_flight = -1
    with pytest.raises(lstmod.LstError) as e:
        lstmod.Lst.from_synth(geom, mmap, cfg)
    assert e.value.status == lstmod.ERR_ARG
    cfg.launches_in_flight, cfg.n_slots = 4, 20
    c = lstmod.Lst.from_synth(geom, mmap, cfg)
    evs = [synth.generate_event(geom, 1, 900 + i, n_particles=n) for i, n in enumerate((6000, 40, 0, 2500))] + [synth.generate_event(geom, 3, 4)]
    evs += [synth.generate_event(geom, 1, 910 + i, n_particles=800 + 300 * i) for i in range(15)]
    st = torch.cuda.Stream()
    c.load_event(0, evs[0].x, evs[0].y, evs[0].z, evs[0].module, evs[0].side, st)     # one event on its own
    c.run(0, st)
    as_tuple = lambda ev: (ev.x, ev.y, ev.z, ev.module, ev.side)
    c.load_events(1, [as_tuple(ev) for ev in evs[1:4]], stream=st)                      # a batch of 3
    c.run_batch(1, 3, st)
    c.load_events(4, [as_tuple(ev) for ev in evs[4:20]], stream=st)                     # a batch of 16
    sd = synth.generate_seeds(evs[4], 4)
    c.load_seeds(4, [sd.arrays()], st)
    c.run_batch(4, 16, st)
    c.run_stage(4, 16, lstmod.CLEAN, st)
    c.run_stage(4, 1, lstmod.PIXEL, st)
    assert c.sync_batch(0, 20, st) == 0
    for k in (0, 1, 2, 3, 4, 9, 19):
        ora = run_oracle(o32, evs[k], seeds=sd.arrays() if k == 4 else None)
        parity.compare(parity.gpu_tables(c, k, st), parity.oracle_tables(ora), f"hint slot {k}")
        stt = c.stats(k)
        assert stt["needed"] == ora.counts and stt["candidates"] == ora.candidates
        if k == 4:
            keep = o32.t5_clean(ora.t5_hits(), ora.t5_chi2xy, ora.t5_chi2rz)
            t5 = c.fetch_hit_indices(4, lstmod.T5, st)
            assert set(map(tuple, t5[c.fetch_kept(4, st)].tolist())) == set(map(tuple, ora.t5_hits()[keep].tolist()))
            assert stt["pix_needed"] == [ora.pix[0]["n"], ora.pix[1]["n"]]
    c.close()
