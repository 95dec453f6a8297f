"""Randomised parity (-m gpu): events drawn with random size (1 .. 9000 particles, log-uniform), noise fraction, rotation,
z mirror and seed model go through the whole CUDA path, the duplicate cleaning [D] and the pixel stage [P] in batched
launches on two streams, and every object set is compared with the oracle's: identical tuples of original hit indices,
identical kept set, identical links, floats within 1e-5.  24 events here; the same loop run for 12 minutes on a B200
(496 events, 35.1 M objects, 1.37 M links) found no difference."""
from concurrent.futures import ThreadPoolExecutor

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
    lst_build.build()
    lst.load_library()
    return lst


def draw_event(geom, rng, i):
    """Event + seeds + a description.  Half of the events are rotated / mirrored copies (their seeds are then random
    parameters: fakes only), the others carry the stand-in seed model with a random efficiency and fake fraction."""
    conf = int(rng.choice([0, 1, 1, 1, 3]))
    top = {0: 60, 1: 7000, 3: 9000}[conf]
    n_part = int(np.exp(rng.uniform(0, np.log(top)))) if rng.random() < 0.7 else top
    noise = float(rng.choice([0.0, 0.05, 0.1, 0.3]))
    ev = synth.generate_event(geom, conf, 5000 + i, n_particles=n_part, noise=noise)
    if rng.random() < 0.5:
        ev = synth.transform_event(ev, rot=float(rng.uniform(-np.pi, np.pi)), mirror_z=bool(rng.random() < 0.5))
        n = int(rng.integers(0, 3000))
        ph = rng.uniform(-np.pi, np.pi, n)
        seeds = (rng.uniform(-0.014, 0.014, n).astype(np.float32), np.cos(ph).astype(np.float32), np.sin(ph).astype(np.float32),
                 rng.normal(0, 5, n).astype(np.float32), rng.uniform(-2.5, 2.5, n).astype(np.float32))
    else:
        seeds = synth.generate_seeds(ev, 5000 + i, efficiency=float(rng.uniform(0.3, 1.0)),
                                     fake_fraction=float(rng.uniform(0, 1.0))).arrays()
    return ev, seeds, dict(config=conf, particles=n_part, noise=noise, hits=int(ev.n), seeds=int(len(seeds[0])))


def test_random_events_whole_path_clean_and_pixel(lstmod, geom, mmap, o32):
    import torch
    cfg = lstmod.default_config()
    cfg.n_slots = 8
    ctx = lstmod.Lst.from_synth(geom, mmap, cfg)
    streams = [torch.cuda.Stream() for _ in range(2)]
    rng = np.random.default_rng(77)
    pool = ThreadPoolExecutor(8)

    def oracle_of(ev, seeds):
        r = o32.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side, seeds=seeds)
        return r, o32.t5_clean(r.t5_hits(), r.t5_chi2xy, r.t5_chi2rz)

    totals = np.zeros(7, np.int64)
    sizes = []
    for it in range(3):
        batch = [draw_event(geom, rng, 8 * it + k) for k in range(8)]
        futs = [pool.submit(oracle_of, ev, seeds) for ev, seeds, _ in batch]
        for half, st in enumerate(streams):
            sl = range(4 * half, 4 * half + 4)
            ctx.load_events(4 * half, [(batch[k][0].x, batch[k][0].y, batch[k][0].z, batch[k][0].module, batch[k][0].side) for k in sl], stream=st)
            ctx.load_seeds(4 * half, [batch[k][1] for k in sl], stream=st)
            ctx.run_batch(4 * half, 4, st)
            ctx.run_stage(4 * half, 4, lstmod.CLEAN, st)
            ctx.run_stage(4 * half, 4, lstmod.PIXEL, st)
        for half, st in enumerate(streams):
            assert ctx.sync_batch(4 * half, 4, st) == 0
        for k in range(8):
            ev, seeds, meta = batch[k]
            st = streams[k // 4]
            ora, keep = futs[k].result()
            label = f"random event {8 * it + k} {meta}"
            parity.compare(parity.gpu_tables(ctx, k, st), parity.oracle_tables(ora), label)
            s = ctx.stats(k)
            assert s["needed"] == ora.counts and s["candidates"] == ora.candidates, label
            t5 = ctx.fetch_hit_indices(k, lstmod.T5, st)
            kept = t5[ctx.fetch_kept(k, st)]
            assert set(map(tuple, kept.tolist())) == set(map(tuple, ora.t5_hits()[keep].tolist())), label + " [D]"
            links = []
            for kind, objs in ((0, ctx.fetch_hit_indices(k, lstmod.T3, st)), (1, t5)):
                link, _ = ctx.fetch_pixel_links(k, kind, st)
                got = np.concatenate([link[:, :1], objs[link[:, 1]].reshape(len(link), objs.shape[1])], 1)
                want = ora.pix_tuples(kind)
                assert got.shape == want.shape and set(map(tuple, got.tolist())) == set(map(tuple, want.tolist())), label + f" [P] kind {kind}"
                links.append(len(link))
            totals += np.array(list(ora.counts) + [int(keep.sum())] + links)
            sizes.append(meta["hits"])
    ctx.close()
    print(f"24 random events, {min(sizes)} .. {max(sizes)} hits: objects (MD, LS, T3, T5, kept, pT3, pT5) {totals.tolist()}")
    assert min(sizes) < 500 and max(sizes) > 60000 and totals[3] > 20000 and totals[5] > 5000
