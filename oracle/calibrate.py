"""Calibration of the empirical chi2 / curvature-match thresholds (rule from
SURVEY.md 8(c); "chi2 cuts are derived empirically for different categories").

ORACLE-SIDE SCRIPT (test infrastructure): calls only oracle/ and the seeded input generator.

Rule: 8 config-1 events, seeds 100..107 (disjoint from every benchmark / parity seed); run the
oracle with the thresholds under calibration opened wide; take objects whose hits all come
from ONE generated particle with pT >= 0.8 GeV; per category (= innermost layer of the object)
record the maximum of each cut variable; threshold = smallest "round" value >= 1.5 x maximum.
The frozen values live in DESIGN.md and are typed by hand into oracle/lst_oracle.c and into
the CUDA library's default config; this script only prints the table that justifies them.

    python -m oracle.calibrate            # prints the table (about 10 s)
"""
from __future__ import annotations

import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from oracle import oracle  # noqa: E402
from paper_2207_08207_b200 import synth  # noqa: E402

SEEDS = tuple(range(100, 108))
HUGE = 1.0e30


def one_particle(truth_rows, pt):
    """rows of truth ids -> mask of rows whose ids are all equal, >= 0 and pT >= 0.8."""
    same = (truth_rows == truth_rows[:, :1]).all(1) & (truth_rows[:, 0] >= 0)
    ok = np.zeros(len(truth_rows), bool)
    ok[same] = pt[truth_rows[same, 0]] >= 0.8
    return ok


def main():
    o = oracle.load("f32")
    geom = synth.make_geometry()
    mg = synth.map_geometry(geom)                # the oracle's own module map [B]
    mm = synth.ModuleMap(geom.n_modules, *o.build_map(mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"]))
    cfg = o.default_config()
    for i in range(4):
        cfg.t3_chi2rz_max[i] = HUGE
    for i in range(2):
        cfg.t5_chi2rz_max[i] = HUGE
    cfg.t5_dkappa_max = HUGE
    cfg.t5_chi2xy_max = HUGE
    kappa_max = 2.0 * o.default_config().half_kappa_max
    mx = dict(t3_chi2rz=np.zeros(4), t5_dk=np.zeros(2), t5_chi2rz=np.zeros(2), t5_chi2xy=np.zeros(2))
    n = dict(t3=np.zeros(4, int), t5=np.zeros(2, int))
    for seed in SEEDS:
        ev = synth.generate_event(geom, 1, seed)
        r = o.run(geom.layer, mm.row_offsets, mm.targets, ev.x, ev.y, ev.z, ev.module, ev.side, cfg=cfg)
        pt = ev.particles["pt"]
        lay = geom.layer[r.md_module]
        t3m = r.t3_mds()
        ok3 = one_particle(ev.truth[r.t3_hits()], pt)
        for c in range(4):
            sel = ok3 & (lay[t3m[:, 0]] == c)
            n["t3"][c] += sel.sum()
            if sel.any():
                mx["t3_chi2rz"][c] = max(mx["t3_chi2rz"][c], r.t3_chi2rz[sel].max())
        t5m = r.t5_mds()
        ok5 = one_particle(ev.truth[r.t5_hits()], pt)
        dk = np.abs(r.t3_kappa[r.t5_a] - r.t3_kappa[r.t5_b])
        for c in range(2):
            sel = ok5 & (lay[t5m[:, 0]] == c)
            n["t5"][c] += sel.sum()
            if sel.any():
                mx["t5_dk"][c] = max(mx["t5_dk"][c], dk[sel].max())
                mx["t5_chi2rz"][c] = max(mx["t5_chi2rz"][c], r.t5_chi2rz[sel].max())
                mx["t5_chi2xy"][c] = max(mx["t5_chi2xy"][c], r.t5_chi2xy[sel].max())
        print(f"seed {seed}: hits {ev.n} counts {r.counts}", flush=True)
    d = o.config_dict()
    print("\ncategory = innermost layer; max over single-particle (pT >= 0.8 GeV) objects; x1.5; frozen")
    for c in range(4):
        print(f"T3 chi2rz  cat {c}: n={n['t3'][c]:7d} max={mx['t3_chi2rz'][c]:9.3f} x1.5={1.5*mx['t3_chi2rz'][c]:9.3f} frozen={d['t3_chi2rz_max'][c]}")
    for c in range(2):
        print(f"T5 chi2rz  cat {c}: n={n['t5'][c]:7d} max={mx['t5_chi2rz'][c]:9.3f} x1.5={1.5*mx['t5_chi2rz'][c]:9.3f} frozen={d['t5_chi2rz_max'][c]}")
    print(f"T5 chi2xy  all  : max={mx['t5_chi2xy'].max():9.3f} x1.5={1.5*mx['t5_chi2xy'].max():9.3f} frozen={d['t5_chi2xy_max']}")
    print(f"T5 dkappa/kappa_max all: max={mx['t5_dk'].max()/kappa_max:9.5f} x1.5={1.5*mx['t5_dk'].max()/kappa_max:9.5f} "
          f"frozen={d['t5_dkappa_max']/kappa_max:.5f}")


def main_pixel():
    """[P] pixel links (python -m oracle.calibrate pixel): with the frozen [M]..[Q] cuts and the [P] thresholds opened, the
    maximum of |kappa_obj - kappa_seed|, chi2xy and chi2rz over the links whose outer object and seed come from the same
    generated particle (pT >= 0.8 GeV); threshold = smallest multiple of 5 (chi2) / of 1e-4 cm^-1 (curvature) >= 1.5 x max."""
    o = oracle.load("f32")
    geom = synth.make_geometry()
    mg = synth.map_geometry(geom)
    mm = synth.ModuleMap(geom.n_modules, *o.build_map(mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"]))
    cfg = o.default_config()
    for k in range(2):
        cfg.pix_dkappa_max[k] = cfg.pix_chi2xy_max[k] = cfg.pix_chi2rz_max[k] = HUGE
    mx = {name: np.zeros(2) for name in ("dkappa", "chi2xy", "chi2rz")}
    n = np.zeros(2, int)
    for seed in SEEDS:
        ev = synth.generate_event(geom, 1, seed, n_particles=2000)       # the full product seeds x objects is the search space: a third of an event keeps this to a minute
        sd = synth.generate_seeds(ev, seed)
        r = o.run(geom.layer, mm.row_offsets, mm.targets, ev.x, ev.y, ev.z, ev.module, ev.side, cfg=cfg, seeds=sd.arrays())
        pt = ev.particles["pt"]
        for kind in (0, 1):
            d = r.pix[kind]
            tr = ev.truth[(r.t5_hits() if kind else r.t3_hits())[d["obj"]]]
            same = (tr == tr[:, :1]).all(1) & (tr[:, 0] >= 0) & (tr[:, 0] == sd.truth[d["seed"]])
            same[same] = pt[tr[same, 0]] >= 0.8
            n[kind] += same.sum()
            for name in mx:
                mx[name][kind] = max(mx[name][kind], np.abs(d[name][same]).max())
        print(f"seed {seed}: hits {ev.n} seeds {sd.n} counts {r.counts}", flush=True)
    d = o.config_dict()
    for kind, what in enumerate(("pixel triplets", "pixel quintuplets")):
        print(f"{what}: n={n[kind]}")
        print(f"  |dkappa| max={mx['dkappa'][kind]:.6f} x1.5={1.5 * mx['dkappa'][kind]:.6f} frozen={d['pix_dkappa_max'][kind]}")
        print(f"  chi2xy   max={mx['chi2xy'][kind]:.3f} x1.5={1.5 * mx['chi2xy'][kind]:.3f} frozen={d['pix_chi2xy_max'][kind]}")
        print(f"  chi2rz   max={mx['chi2rz'][kind]:.3f} x1.5={1.5 * mx['chi2rz'][kind]:.3f} frozen={d['pix_chi2rz_max'][kind]}")


if __name__ == "__main__":
    import sys
    main_pixel() if "pixel" in sys.argv[1:] else main()
