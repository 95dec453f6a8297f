"""Pins of the oracle's quintuplet duplicate cleaning [D] (DESIGN.md section 1 [D], reading 24).
The paper gives no numbers for it, so the pins are: an independent restatement with Python sets
on small inputs (incl. forced ties), the properties the rule implies, order independence, the single-helix case and
truth statistics."""
import numpy as np
import pytest

from paper_2207_08207_b200 import synth

K = 7


def brute_force(hits, score, k=K):
    """Independent restatement: Python sets and tuple comparison, no sorting, no merging."""
    sets = [set(map(int, h)) for h in hits]
    key = [(float(s), tuple(map(int, h))) for s, h in zip(score, hits)]
    keep = np.ones(len(hits), bool)
    for a in range(len(hits)):
        for b in range(len(hits)):
            if a != b and len(sets[a] & sets[b]) >= k and key[b] < key[a]:
                keep[a] = False
                break
    return keep


def score32(r):
    return (r.t5_chi2xy.astype(np.float32) + r.t5_chi2rz.astype(np.float32)).astype(np.float32)


def test_p12_equals_set_based_restatement_on_tiny_event_and_random_tuples(o32, run_oracle, geom):
    ev = synth.generate_event(geom, 0, 0)
    r = run_oracle(o32, ev)
    h = r.t5_hits()
    keep = o32.t5_clean(h, r.t5_chi2xy, r.t5_chi2rz, K)
    assert np.array_equal(keep, brute_force(h, score32(r)))
    assert 0 < keep.sum() < len(h)
    # random tuples built to overlap, with many exactly equal scores (tie-break by hit tuple) and every threshold
    rng = np.random.default_rng(3)
    base = rng.permutation(400)[:200].reshape(20, 10)
    rows = []
    for t in base:
        for _ in range(6):
            v = t.copy()
            m = rng.integers(0, 5)
            v[rng.permutation(10)[:m]] = 1000 + rng.integers(0, 50, m)      # replace 0..4 hits
            if len(set(v)) == 10:
                rows.append(v)
    hits = np.asarray(rows, np.int32)
    cx = rng.integers(0, 3, len(hits)).astype(np.float32)                    # few distinct values: ties
    cz = rng.integers(0, 3, len(hits)).astype(np.float32)
    for k in (5, 6, 7, 8, 10):
        assert np.array_equal(o32.t5_clean(hits, cx, cz, k), brute_force(hits, cx + cz, k)), k
    assert o32.t5_clean(np.zeros((0, 10), np.int32), np.zeros(0, np.float32), np.zeros(0, np.float32), K).shape == (0,)


def test_p13_properties_and_order_independence(o32, run_oracle, geom):
    ev = synth.generate_event(geom, 1, 5, n_particles=1200)
    r = run_oracle(o32, ev)
    h, s = r.t5_hits(), score32(r)
    assert len(h) > 1000
    keep = o32.t5_clean(h, r.t5_chi2xy, r.t5_chi2rz, K)
    sets = [frozenset(map(int, t)) for t in h]
    key = [(float(a), tuple(map(int, t))) for a, t in zip(s, h)]
    kept = np.nonzero(keep)[0]
    by_hit = {}
    for q in range(len(h)):
        for x in sets[q]:
            by_hit.setdefault(x, []).append(q)
    near = lambda q: {b for x in sets[q] for b in by_hit[x] if b != q and len(sets[q] & sets[b]) >= K}
    for q in kept:                      # (i) no two kept quintuplets share >= K hits; nothing better overlaps a kept one
        assert all((not keep[b]) and key[b] > key[q] for b in near(q))
    for q in np.nonzero(~keep)[0]:      # (ii) every removed one has a better overlapping one
        assert any(key[b] < key[q] for b in near(q))
    assert keep[min(range(len(h)), key=lambda q: key[q])]                     # (iii) the global best is kept
    again = o32.t5_clean(h[kept], r.t5_chi2xy[kept], r.t5_chi2rz[kept], K)    # (iv) idempotent
    assert again.all()
    perm = np.random.default_rng(1).permutation(len(h))                       # (v) independent of the input order
    kp = o32.t5_clean(h[perm], r.t5_chi2xy[perm], r.t5_chi2rz[perm], K)
    assert np.array_equal(kp, keep[perm])
    # (vi) what the CUDA path's candidate search relies on: quintuplets sharing >= 7 hits share a mini-doublet
    mds = r.t5_mds()
    for q in range(0, len(h), 7):
        for b in near(q):
            assert set(mds[q]) & set(mds[b])


def test_p11_single_helix_keeps_one(o32, run_oracle, geom):
    n_two = 0
    for seed in range(30):
        ev = synth.generate_event(geom, 0, 500 + seed, n_particles=1)
        r = run_oracle(o32, ev)
        if r.counts[3] == 0:
            continue
        keep = o32.t5_clean(r.t5_hits(), r.t5_chi2xy, r.t5_chi2rz, K)
        assert keep.sum() >= 1
        if r.counts[3] == 2:            # layers 0-4 and 1-5 of one track: 8 common hits, the lower score survives
            n_two += 1
            assert keep.sum() == 1 and keep[np.argmin(score32(r))]
    assert n_two >= 5


def test_p14_truth_duplicates_removed_particles_retained(o32, run_oracle, geom):
    ev = synth.generate_event(geom, 1, 6, n_particles=2500)
    r = run_oracle(o32, ev)
    h = r.t5_hits()
    keep = o32.t5_clean(h, r.t5_chi2xy, r.t5_chi2rz, K)
    tr = ev.truth[h]
    pid = np.array([np.bincount(row[row >= 0]).argmax() if (row >= 0).any() else -1 for row in tr])
    matched = np.array([(row == p).sum() >= 8 for row, p in zip(tr, pid)])      # the 75 % rule
    def per_particle(mask):
        u, c = np.unique(pid[mask & matched], return_counts=True)
        return set(u.tolist()), float((c > 1).mean())
    before, dup_before = per_particle(np.ones(len(h), bool))
    after, dup_after = per_particle(keep)
    assert dup_before > 0.7 and dup_after < 0.05
    assert len(after) >= 0.995 * len(before)
