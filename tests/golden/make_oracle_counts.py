"""Writes tests/golden/oracle_counts.txt: object / candidate counts and a digest of the sorted quintuplet hit tuples of
the ORACLE (fp32 build) on seeded events.  Calls only oracle/ and the seeded input generators; nothing here comes from
the CUDA path.  The paper prints no worked example (PAPER.md has no numeric fixture), so these are not the paper's
values: the file is a regression fence around the oracle's arithmetic -- a change of the oracle, of the SPEC constants
or of the generators shows up here and must be justified in the commit that regenerates it.

    python tests/golden/make_oracle_counts.py
"""
import hashlib
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

from oracle import oracle                      # noqa: E402
from paper_2207_08207_b200 import synth        # noqa: E402

CASES = (("C0", 0, 0, None), ("C0", 0, 1, None), ("C1", 1, 0, None), ("C1small", 1, 5, 1200), ("C3", 3, 0, None))


def lines():
    geom = synth.make_geometry()
    o = oracle.load("f32")
    mg = synth.map_geometry(geom)                # the oracle's own module map [B] (69 630 connections on this geometry)
    mmap = synth.ModuleMap(geom.n_modules, *o.build_map(mg["layer"], mg["phi"], mg["rho"], mg["gap"], mg["hw"], mg["zlo"], mg["zhi"]))
    yield "# case config seed n_particles | hits | MD LS T3 T5 | candidates MD LS T3 T5 | kept by [D] (K = 7) | sha256(sorted T5 hit tuples)[:16]"
    for name, cfg, seed, npart in CASES:
        ev = synth.generate_event(geom, cfg, seed) if npart is None else synth.generate_event(geom, cfg, seed, n_particles=npart)
        r = o.run(geom.layer, mmap.row_offsets, mmap.targets, ev.x, ev.y, ev.z, ev.module, ev.side)
        h = r.t5_hits()
        kept = int(o.t5_clean(h, r.t5_chi2xy, r.t5_chi2rz, 7).sum())        # all pairs: half a minute on the largest event
        order = np.lexsort(h.T[::-1]) if len(h) else np.zeros(0, np.int64)
        digest = hashlib.sha256(np.ascontiguousarray(h[order], np.int32).tobytes()).hexdigest()[:16]
        yield (f"{name} {cfg} {seed} {npart} | {ev.n} | {' '.join(map(str, r.counts))} | {' '.join(map(str, r.candidates))} | "
               f"{kept} | {digest}")


if __name__ == "__main__":
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_counts.txt")
    with open(out, "w") as f:
        f.write("\n".join(lines()) + "\n")
    print(open(out).read())
