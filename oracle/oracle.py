"""ctypes wrapper around oracle/lst_oracle.c (ORACLE = test infrastructure, not the product).

Only tests/, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this.  It does not import the CUDA path and the CUDA path does not import it.

``load("f32")`` is the SPEC arithmetic (fp32, fixed operation order, no FMA contraction): the
build GPU parity is checked against.  ``load("f64")`` is the same source in double precision,
used by the CPU tests to pin the formulas against closed forms.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lst_oracle.c")
_LOCK = threading.Lock()
_LIBS: dict = {}

N_LAYERS = 6
# No -march, no -ffast-math, no FMA contraction: IEEE fp32 evaluated exactly as written.
CFLAGS = ["-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-fno-fast-math",
          "-fno-unsafe-math-optimizations", "-Wall", "-Wextra", "-Wno-unused-parameter"]

_CONFIG_FIELDS = [
    ("half_kappa_max", 1), ("z_lum", 1), ("md_cos_eps", 6), ("md_sin_eps", 6), ("md_dz_res", 6),
    ("md_eps", 6), ("seg_cos_eps", 1), ("seg_sin_eps", 1), ("seg_z0_max", 5), ("t3_kappa_max", 1),
    ("t3_chi2rz_max", 4), ("sigma_z2", 6), ("inv_sigma_z2", 6), ("t5_dkappa_max", 1),
    ("t5_chi2rz_max", 2), ("t5_chi2xy_max", 1), ("t5_sigma_xy2_scaled", 1), ("t5_kappa_max", 1),
    ("pix_dkappa_max", 2), ("pix_inv_var_xy", 6), ("pix_inv_var_rz", 6), ("pix_chi2xy_max", 2), ("pix_chi2rz_max", 2),
]


def _config_type(real):
    class Config(C.Structure):
        _fields_ = [(n, real if k == 1 else real * k) for n, k in _CONFIG_FIELDS]
    return Config


def build(precision: str = "f32", force: bool = False) -> str:
    """Compile oracle/lst_oracle.c with gcc into oracle/_build/liblsto_<precision>.so."""
    assert precision in ("f32", "f64")
    out_dir = os.path.join(_HERE, "_build")
    os.makedirs(out_dir, exist_ok=True)
    out = os.path.join(out_dir, f"liblsto_{precision}.so")
    if force or not os.path.exists(out) or os.path.getmtime(out) < os.path.getmtime(_SRC):
        tmp = out + f".tmp{os.getpid()}"
        cmd = ["gcc", *CFLAGS, f"-DLSTO_F64={1 if precision == 'f64' else 0}", _SRC, "-o", tmp, "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, out)
    return out


class OracleLib:
    def __init__(self, precision: str):
        self.precision = precision
        self.real = C.c_double if precision == "f64" else C.c_float
        self.np_real = np.float64 if precision == "f64" else np.float32
        self.Config = _config_type(self.real)
        lib = C.CDLL(build(precision))
        self.lib = lib
        assert lib.lsto_is_f64() == (1 if precision == "f64" else 0)
        assert lib.lsto_sizeof_config() == C.sizeof(self.Config)
        P = C.POINTER
        lib.lsto_default_config.argtypes = [P(self.Config)]
        lib.lsto_default_config.restype = None
        lib.lsto_run.restype = C.c_void_p
        lib.lsto_run.argtypes = [P(self.Config), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                 C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                 C.c_int, C.c_int]
        lib.lsto_free.argtypes = [C.c_void_p]
        lib.lsto_free.restype = None
        lib.lsto_count.argtypes = [C.c_void_p, C.c_int]
        lib.lsto_count.restype = C.c_int64
        lib.lsto_candidates.argtypes = [C.c_void_p, C.c_int]
        lib.lsto_candidates.restype = C.c_int64
        lib.lsto_i32.argtypes = [C.c_void_p, C.c_int]
        lib.lsto_i32.restype = P(C.c_int32)
        lib.lsto_real.argtypes = [C.c_void_p, C.c_int]
        lib.lsto_real.restype = P(self.real)
        r = self.real
        lib.lsto_md_cut.argtypes = [P(self.Config), C.c_int] + [r] * 6 + [P(r), P(r)]
        lib.lsto_seg_cut.argtypes = [P(self.Config), C.c_int] + [r] * 12 + [P(r), P(r)]
        lib.lsto_t3_cut.argtypes = [P(self.Config), C.c_int, P(r), P(r), P(r), P(r), P(r)]
        lib.lsto_t5_cut.argtypes = [P(self.Config), C.c_int, r, r, P(r), P(r), P(r)]
        for f in (lib.lsto_md_cut, lib.lsto_seg_cut, lib.lsto_t3_cut, lib.lsto_t5_cut):
            f.restype = C.c_int
        lib.lsto_t5_clean.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        lib.lsto_t5_clean.restype = C.c_int64
        lib.lsto_half_bits_array.argtypes = [C.c_int64, C.c_void_p, C.c_void_p]
        lib.lsto_half_bits_array.restype = None
        lib.lsto_pix_cut.argtypes = [P(self.Config), C.c_int, C.c_int, C.c_int, P(r), r, P(r), P(r), P(r)]
        lib.lsto_pix_cut.restype = C.c_int
        lib.lsto_pixel_link.argtypes = [P(self.Config), C.c_void_p, C.c_void_p, C.c_int, C.c_int32] + [C.c_void_p] * 5
        lib.lsto_pixel_link.restype = C.c_int64
        lib.lsto_pix_count.argtypes = lib.lsto_pix_candidates.argtypes = [C.c_void_p, C.c_int]
        lib.lsto_pix_count.restype = lib.lsto_pix_candidates.restype = C.c_int64
        lib.lsto_pix_i32.argtypes = lib.lsto_pix_real.argtypes = [C.c_void_p, C.c_int, C.c_int]
        lib.lsto_pix_i32.restype = P(C.c_int32)
        lib.lsto_pix_real.restype = P(self.real)

    # ---- configuration -------------------------------------------------------------------
    def default_config(self):
        cfg = self.Config()
        self.lib.lsto_default_config(C.byref(cfg))
        return cfg

    def config_dict(self, cfg=None) -> dict:
        cfg = cfg or self.default_config()
        return {n: (float(getattr(cfg, n)) if k == 1 else [float(v) for v in getattr(cfg, n)])
                for n, k in _CONFIG_FIELDS}

    # ---- scalar cut functions (value/threshold margins returned for near-threshold checks) --
    def _arr(self, vals):
        return (self.real * len(vals))(*[float(v) for v in vals])

    def md_cut(self, layer, lower, upper, cfg=None):
        """lower/upper = (x, y, z). Returns (passed, dict(sinA,dphi,dphichange,rl,ru), margins[4])."""
        cfg = cfg or self.default_config()
        out, mar = self._arr([np.nan] * 5), self._arr([np.nan] * 4)
        ok = self.lib.lsto_md_cut(C.byref(cfg), int(layer), *[self.real(float(v)) for v in (*lower, *upper)], out, mar)
        return bool(ok), dict(zip(("sinA", "dphi", "dphichange", "rl", "ru"), list(out))), list(mar)

    def seg_cut(self, layer_in, inner, outer, cfg=None):
        """inner/outer = (x, y, z, r, ur, sinA) of the MD anchors."""
        cfg = cfg or self.default_config()
        out, mar = self._arr([np.nan] * 4), self._arr([np.nan] * 8)
        ok = self.lib.lsto_seg_cut(C.byref(cfg), int(layer_in), *[self.real(float(v)) for v in (*inner, *outer)], out, mar)
        return bool(ok), dict(zip(("sinS", "z0", "dphi", "dphichange"), list(out))), list(mar)

    def t3_cut(self, layer1, p1, p2, p3, cfg=None):
        """p = (x, y, z, r) anchors."""
        cfg = cfg or self.default_config()
        out, mar = self._arr([np.nan] * 2), self._arr([np.nan] * 4)
        ok = self.lib.lsto_t3_cut(C.byref(cfg), int(layer1), self._arr(p1), self._arr(p2), self._arr(p3), out, mar)
        return bool(ok), dict(zip(("kappa", "chi2rz"), list(out))), list(mar)

    def t5_cut(self, layer1, kappa_a, kappa_b, pts, cfg=None):
        """pts = 5 anchors (x, y, z, r)."""
        cfg = cfg or self.default_config()
        out, mar = self._arr([np.nan] * 3), self._arr([np.nan] * 8)
        flat = [v for p in pts for v in p]
        ok = self.lib.lsto_t5_cut(C.byref(cfg), int(layer1), self.real(float(kappa_a)), self.real(float(kappa_b)),
                                  self._arr(flat), out, mar)
        return bool(ok), dict(zip(("kfit", "chi2xy", "chi2rz"), list(out))), list(mar)

    def pix_cut(self, kind, layer1, seed, kappa_obj, pts, cfg=None):
        """[P] seed = (kappa, cos phi0, sin phi0, z0, t); pts = 3 (kind 0) or 5 (kind 1) anchors (x, y, z, r).
        Returns (passed, dict(chi2xy, chi2rz, dkappa), margins[6])."""
        cfg = cfg or self.default_config()
        out, mar = self._arr([np.nan] * 3), self._arr([np.nan] * 6)
        flat = [v for p in pts for v in p]
        ok = self.lib.lsto_pix_cut(C.byref(cfg), int(kind), int(layer1), len(pts), self._arr(seed), self.real(float(kappa_obj)),
                                   self._arr(flat), out, mar)
        return bool(ok), dict(zip(("chi2xy", "chi2rz", "dkappa"), list(out))), list(mar)

    def t5_clean(self, hits, chi2xy, chi2rz, min_shared: int = 7) -> np.ndarray:
        """[D] duplicate cleaning: hits [n][10] original hit indices -> keep [n] bool (all-pairs definition)."""
        hits = np.ascontiguousarray(hits, np.int32).reshape(-1, 10)
        n = len(hits)
        cx = np.ascontiguousarray(chi2xy, self.np_real)
        cz = np.ascontiguousarray(chi2rz, self.np_real)
        assert len(cx) == n and len(cz) == n
        keep = np.zeros(max(n, 1), np.uint8)
        ptr = lambda a: a.ctypes.data_as(C.c_void_p)
        kept = self.lib.lsto_t5_clean(C.c_int64(n), ptr(hits), ptr(cx), ptr(cz), int(min_shared), ptr(keep))
        assert kept == int(keep[:n].sum())
        return keep[:n].astype(bool)

    def half_bits(self, values) -> np.ndarray:
        """[H] binary16 bit patterns (uint16) of fp32 values, round to nearest even (reduced-precision object store)."""
        v = np.ascontiguousarray(values, np.float32)
        out = np.zeros(v.shape, np.uint16)
        self.lib.lsto_half_bits_array(C.c_int64(v.size), v.ctypes.data_as(C.c_void_p), out.ctypes.data_as(C.c_void_p))
        return out

    def build_map(self, layer, phi, rho, gap, hw, zlo, zhi, pt_min=0.8, b_tesla=3.8, z0_max=15.0, pad_phi=0.01, pad_z=1.0):
        """[B] module-map builder (always double precision). Returns (row_offsets, targets)."""
        layer = np.ascontiguousarray(layer, np.int8)
        arrs = [np.ascontiguousarray(a, np.float64) for a in (phi, rho, gap, hw, zlo, zhi)]
        n = len(layer)
        ptr = lambda a: a.ctypes.data_as(C.c_void_p)
        f = self.lib.lsto_build_map
        f.restype = C.c_int64
        f.argtypes = [C.c_int32] + [C.c_void_p] * 7 + [C.c_double] * 5 + [C.c_void_p, C.c_void_p]
        offs = np.zeros(n + 1, np.int32)
        total = f(n, ptr(layer), *[ptr(a) for a in arrs], pt_min, b_tesla, z0_max, pad_phi, pad_z, ptr(offs), None)
        tg = np.zeros(max(int(total), 1), np.int32)
        f(n, ptr(layer), *[ptr(a) for a in arrs], pt_min, b_tesla, z0_max, pad_phi, pad_z, ptr(offs), ptr(tg))
        return offs, tg[:total]

    # ---- whole event -----------------------------------------------------------------------
    def run(self, layer, row_offsets, targets, x, y, z, module, side, mode=0, stages=4, cfg=None, seeds=None) -> "OracleResult":
        cfg = cfg or self.default_config()
        layer = np.ascontiguousarray(layer, np.int8)
        row_offsets = np.ascontiguousarray(row_offsets, np.int32)
        targets = np.ascontiguousarray(targets, np.int32)
        x, y, z = (np.ascontiguousarray(a, np.float32) for a in (x, y, z))
        module = np.ascontiguousarray(module, np.int32)
        side = np.ascontiguousarray(side, np.uint8)
        n_mod, n = len(layer), len(x)
        assert len(row_offsets) == n_mod + 1 and len(y) == n and len(z) == n and len(module) == n and len(side) == n
        ptr = lambda a: a.ctypes.data_as(C.c_void_p)
        h = self.lib.lsto_run(C.byref(cfg), n_mod, ptr(layer), ptr(row_offsets), ptr(targets), n,
                              ptr(x), ptr(y), ptr(z), ptr(module), ptr(side), int(mode), int(stages))
        if not h:
            raise ValueError("oracle: invalid input (module id / side / module map)")
        try:
            if seeds is not None:         # [P]: seeds = (kappa, cphi, sphi, z0, t) fp32 arrays -> pixel triplets and quintuplets
                sd = [np.ascontiguousarray(a, np.float32) for a in seeds]
                for kind in (0, 1):
                    if stages >= 3 + kind:
                        self.lib.lsto_pixel_link(C.byref(cfg), h, ptr(layer), kind, len(sd[0]), *[ptr(a) for a in sd])
            return OracleResult(self, h, pixel=seeds is not None, stages=stages)
        finally:
            self.lib.lsto_free(h)


_I32 = dict(md_lower=(0, 0), md_upper=(1, 0), md_module=(2, 0), seg_in=(3, 1), seg_out=(4, 1),
            t3_a=(5, 2), t3_b=(6, 2), t5_a=(7, 3), t5_b=(8, 3))
_REAL = dict(md_x=(0, 0), md_y=(1, 0), md_z=(2, 0), md_r=(3, 0), md_ur=(4, 0), md_sinA=(5, 0), md_dphi=(6, 0),
             md_dphichange=(7, 0), seg_sinS=(8, 1), seg_z0=(9, 1), seg_dphi=(10, 1), seg_dphichange=(11, 1),
             t3_kappa=(12, 2), t3_chi2rz=(13, 2), t5_kfit=(14, 3), t5_chi2xy=(15, 3), t5_chi2rz=(16, 3))


class OracleResult:
    """numpy copies of every output array, plus hit-index tuples per object class."""

    def __init__(self, o: OracleLib, h, pixel=False, stages=4):
        lib = o.lib
        self.pix = {}
        if pixel:
            for kind in (0, 1):
                if stages < 3 + kind:
                    continue
                n = int(lib.lsto_pix_count(h, kind))
                get_i = lambda f: np.ctypeslib.as_array(lib.lsto_pix_i32(h, kind, f), (n,)).copy() if n else np.zeros(0, np.int32)
                get_r = lambda f: np.ctypeslib.as_array(lib.lsto_pix_real(h, kind, f), (n,)).copy() if n else np.zeros(0, o.np_real)
                self.pix[kind] = dict(n=n, candidates=int(lib.lsto_pix_candidates(h, kind)), seed=get_i(0), obj=get_i(1),
                                      chi2xy=get_r(0), chi2rz=get_r(1), dkappa=get_r(2))
        self.counts = [int(lib.lsto_count(h, k)) for k in range(4)]
        self.candidates = [int(lib.lsto_candidates(h, k)) for k in range(4)]
        for name, (f, kind) in _I32.items():
            n = self.counts[kind]
            setattr(self, name, np.ctypeslib.as_array(lib.lsto_i32(h, f), (n,)).copy() if n else np.zeros(0, np.int32))
        for name, (f, kind) in _REAL.items():
            n = self.counts[kind]
            setattr(self, name, np.ctypeslib.as_array(lib.lsto_real(h, f), (n,)).copy() if n else np.zeros(0, o.np_real))

    # MD index tuples
    def seg_mds(self):
        return np.stack([self.seg_in, self.seg_out], 1).reshape(-1, 2)

    def t3_mds(self):
        return np.stack([self.seg_in[self.t3_a], self.seg_out[self.t3_a], self.seg_out[self.t3_b]], 1).reshape(-1, 3)

    def t5_mds(self):
        a, b = self.t3_mds()[self.t5_a], self.t3_mds()[self.t5_b]
        return np.concatenate([a, b[:, 1:]], 1).reshape(-1, 5)

    # original-hit-index tuples (object identity, SURVEY.md 8(c) reading #16)
    def md_hits(self):
        return np.stack([self.md_lower, self.md_upper], 1).reshape(-1, 2)

    def _hits(self, mds):
        return self.md_hits()[mds].reshape(len(mds), 2 * mds.shape[1])

    def seg_hits(self):
        return self._hits(self.seg_mds())

    def t3_hits(self):
        return self._hits(self.t3_mds())

    def t5_hits(self):
        return self._hits(self.t5_mds())

    def pix_tuples(self, kind):
        """[P] identity of a pixel link: (seed index, the 6 / 10 original hit indices of its outer object)."""
        hits = self.t5_hits() if kind else self.t3_hits()
        d = self.pix[kind]
        return np.concatenate([d["seed"].reshape(-1, 1), hits[d["obj"]].reshape(len(d["obj"]), 10 if kind else 6)], 1)


def load(precision: str = "f32") -> OracleLib:
    with _LOCK:
        if precision not in _LIBS:
            _LIBS[precision] = OracleLib(precision)
        return _LIBS[precision]
