"""Helpers of the GPU parity tests: run the CUDA path through the C-ABI binding, run the oracle
on the same seeded input, compare object sets (bit-exact, as tuples of original hit indices)
and float payloads (reading 20)."""
import numpy as np

KAPPA_MAX = 0.0142401418
# (column name, absolute floor) per class, in the column order of lst_fetch_values
VALUE_SPEC = {
    0: (("md_sinA", 1e-5), ("md_dphi", 1e-5), ("md_dphichange", 1e-5), ("md_r", 1e-4)),
    1: (("seg_sinS", 1e-5), ("seg_z0", 1e-4), ("seg_dphi", 1e-5), ("seg_dphichange", 1e-5)),
    2: (("t3_kappa", 1e-5 * KAPPA_MAX), ("t3_chi2rz", 1e-5 * 25.0)),
    3: (("t5_kin", 1e-5 * KAPPA_MAX), ("t5_kout", 1e-5 * KAPPA_MAX), ("t5_kfit", 1e-5 * KAPPA_MAX),
        ("t5_chi2xy", 1e-5 * 35.0), ("t5_chi2rz", 1e-5 * 110.0)),
}
REL_TOL = 1e-5       # BASELINE.json north_star: "within 1e-5 relative in fp32"


def oracle_tables(r):
    """OracleResult -> per class (hit tuples [n][k], values [n][v]) in the oracle's order."""
    t3m = r.t3_mds()
    return {
        0: (r.md_hits(), np.stack([r.md_sinA, r.md_dphi, r.md_dphichange, r.md_r], 1).reshape(-1, 4)),
        1: (r.seg_hits(), np.stack([r.seg_sinS, r.seg_z0, r.seg_dphi, r.seg_dphichange], 1).reshape(-1, 4)),
        2: (r.t3_hits(), np.stack([r.t3_kappa, r.t3_chi2rz], 1).reshape(-1, 2)),
        3: (r.t5_hits(), np.stack([r.t3_kappa[r.t5_a], r.t3_kappa[r.t5_b], r.t5_kfit, r.t5_chi2xy, r.t5_chi2rz], 1).reshape(-1, 5)),
    }


def gpu_tables(lst, slot, stream=None):
    return {k: (lst.fetch_hit_indices(slot, k, stream), lst.fetch_values(slot, k, stream)) for k in range(4)}


def sort_rows(hits, vals):
    """Sort objects by their hit tuple (the tuple is unique per object)."""
    if len(hits) == 0:
        return hits, vals
    order = np.lexsort(hits.T[::-1])
    return hits[order], vals[order]


def compare(gpu, ora, label="", classes=range(4)):
    """Assert set equality (bit-exact) and float agreement; returns per-class max relative error."""
    worst = {}
    for k in classes:
        gh, gv = sort_rows(*gpu[k])
        oh, ov = sort_rows(*ora[k])
        assert gh.shape == oh.shape, f"{label} class {k}: gpu {gh.shape[0]} objects, oracle {oh.shape[0]}"
        assert np.array_equal(gh, oh), f"{label} class {k}: object sets differ"
        if len(gh) == 0:
            worst[k] = 0.0
            continue
        w = 0.0
        for c, (name, floor) in enumerate(VALUE_SPEC[k]):
            a, b = gv[:, c].astype(np.float64), ov[:, c].astype(np.float64)
            tol = REL_TOL * np.maximum(np.abs(a), np.abs(b)) + floor
            bad = np.abs(a - b) > tol
            assert not bad.any(), f"{label} {name}: {bad.sum()} values off, worst {np.abs(a - b).max()}"
            w = max(w, float(np.max(np.abs(a - b) / np.maximum(np.maximum(np.abs(a), np.abs(b)), floor / REL_TOL))))
        worst[k] = w
    return worst


def run_gpu(lst, ev, slot=0, stream=None):
    lst.load_event(slot, ev.x, ev.y, ev.z, ev.module, ev.side, stream)
    lst.run(slot, stream)
    lst.sync(slot, stream)
    return gpu_tables(lst, slot, stream)


# ---- reduced-precision object store [H] (DESIGN.md section 1 [H]) -----------------------------------------------
# columns of lst_fetch_values that come out of atan2f (libm and CUDA differ by an fp32 ulp or two, which can move
# the binary16 rounding by one binary16 ulp); every other column is the RNE rounding of a bit-identical fp32 value
ATAN_COLUMNS = {0: (1, 2), 1: (2, 3), 2: (), 3: ()}


def half_steps(a_bits, b_bits):
    """Distance in binary16 ulps between two arrays of bit patterns (sign-magnitude -> ordered integers)."""
    def ordered(u):
        u = u.astype(np.int32)
        return np.where(u & 0x8000, -(u & 0x7fff), u & 0x7fff)
    return np.abs(ordered(a_bits) - ordered(b_bits))


def compare_half(gpu, ora, o32, label=""):
    """Relaxed parity rule of the reduced-precision store: object sets IDENTICAL (nothing a selection reads is reduced);
    every fetched value equals the oracle's fp32 value rounded to binary16 (round to nearest even) bit for bit, except the
    atan2f outputs, which may differ by one binary16 ulp; and, against the unrounded fp32 oracle value, every value is
    within 2^-11 relative + 2^-25 absolute (half an ulp of binary16, subnormal spacing included)."""
    n_off = 0
    for k in range(4):
        gh, gv = sort_rows(*gpu[k])
        oh, ov = sort_rows(*ora[k])
        assert gv.dtype == np.float16, (label, k, gv.dtype)
        assert gh.shape == oh.shape and np.array_equal(gh, oh), f"{label} class {k}: object sets differ"
        if len(gh) == 0:
            continue
        want = o32.half_bits(ov.astype(np.float32))
        got = np.ascontiguousarray(gv).view(np.uint16)
        for c in range(gv.shape[1]):
            d = half_steps(got[:, c], want[:, c])
            if c in ATAN_COLUMNS[k]:
                assert d.max() <= 1, f"{label} class {k} column {c}: {d.max()} binary16 ulps"
                n_off += int((d > 0).sum())
            else:
                assert d.max() == 0, f"{label} class {k} column {c}: not the RNE rounding of the fp32 value ({int((d > 0).sum())} off)"
            a, b = gv[:, c].astype(np.float64), ov[:, c].astype(np.float64)
            tol = 2.0 ** -11 * np.abs(b) + 2.0 ** -25 + (2.0 ** -10 * np.abs(b) if c in ATAN_COLUMNS[k] else 0.0)
            assert np.all(np.abs(a - b) <= tol), f"{label} class {k} column {c}: beyond half an ulp of binary16"
    return n_off
