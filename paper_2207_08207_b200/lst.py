"""Thin ctypes binding over the C-ABI library ``liblst.so`` (include/lst.h).

Argument marshalling only: every step of the path (binning, mini-doublets, segments, triplets,
quintuplets, gathers) runs in the CUDA kernels of ``csrc/``.  There is NO CPU fallback: if the
library is missing or fails to load, importing the binding's entry points raises.

PyTorch is used by callers for device memory and streams; this module itself needs only ctypes
and numpy.  Device arrays returned by the ``*_view`` calls are exposed through
``__cuda_array_interface__`` (``torch.as_tensor(view_array, device="cuda")`` is zero-copy).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "liblst.so")
N_LAYERS = 6
MD, SEG, T3, T5 = 0, 1, 2, 3
CLEAN = 4                                      # optional stage: duplicate cleaning of the quintuplets (run_stage only)
PIXEL = 5                                      # optional stage: pixel line segments -> pixel triplets / quintuplets (run_stage only)
PT3, PT5 = 0, 1                                # kinds of pixel links
KIND_NAMES = ("md", "seg", "t3", "t5")
KERNEL_NAMES = ("bin_count", "bin_scatter", "bin_order", "md", "seg", "t3", "t5",
                "clean_prepare", "clean_count", "clean_fill", "clean_mark")   # lst_stats.kernel_ms[0..10]
HITS_PER_OBJECT = (2, 4, 6, 10, 10)       # [CLEAN]: the kept quintuplets
VALUES_PER_OBJECT = (4, 4, 2, 5, 5)

OK, ERR_ARG, ERR_CUDA, ERR_OVERFLOW, ERR_STATE, ERR_NOMEM = 0, -1, -2, -3, -4, -5
ERR_LIMIT = -6
MAP_STATIC_MAX_MODULES = 32768           # LST_MAP_STATIC_MAX_MODULES


class LstError(RuntimeError):
    def __init__(self, status: int, what: str):
        super().__init__(f"{what}: {status} ({strerror(status)})")
        self.status = status


class Geometry(C.Structure):
    _fields_ = [("n_modules", C.c_int32), ("layer", C.c_void_p), ("kind", C.c_void_p), ("cx", C.c_void_p),
                ("cy", C.c_void_p), ("cz", C.c_void_p), ("phi", C.c_void_p)]


class ModuleMap(C.Structure):
    _fields_ = [("n_modules", C.c_int32), ("row_offsets", C.c_void_p), ("targets", C.c_void_p)]


class Config(C.Structure):
    _fields_ = [("half_kappa_max", C.c_float), ("z_lum", C.c_float),
                ("md_cos_eps", C.c_float * 6), ("md_sin_eps", C.c_float * 6), ("md_dz_res", C.c_float * 6),
                ("md_eps", C.c_float * 6), ("seg_cos_eps", C.c_float), ("seg_sin_eps", C.c_float),
                ("seg_z0_max", C.c_float * 5), ("t3_kappa_max", C.c_float), ("t3_chi2rz_max", C.c_float * 4),
                ("sigma_z2", C.c_float * 6), ("inv_sigma_z2", C.c_float * 6), ("t5_dkappa_max", C.c_float),
                ("t5_chi2rz_max", C.c_float * 2), ("t5_chi2xy_max", C.c_float), ("t5_sigma_xy2_scaled", C.c_float),
                ("t5_kappa_max", C.c_float),
                ("pix_dkappa_max", C.c_float * 2), ("pix_inv_var_xy", C.c_float * 6), ("pix_inv_var_rz", C.c_float * 6),
                ("pix_chi2xy_max", C.c_float * 2), ("pix_chi2rz_max", C.c_float * 2),
                ("device", C.c_int32), ("n_slots", C.c_int32), ("cap_hits", C.c_int32), ("cap_md", C.c_int32),
                ("cap_seg", C.c_int32), ("cap_t3", C.c_int32), ("cap_t5", C.c_int32), ("timing", C.c_int32),
                ("store_half", C.c_int32), ("t5_dup_min_shared", C.c_int32),
                ("cap_seeds", C.c_int32), ("cap_pt3", C.c_int32), ("cap_pt5", C.c_int32),
                ("launches_in_flight", C.c_int32)]

    CUT_FIELDS = ("half_kappa_max", "z_lum", "md_cos_eps", "md_sin_eps", "md_dz_res", "md_eps", "seg_cos_eps",
                  "seg_sin_eps", "seg_z0_max", "t3_kappa_max", "t3_chi2rz_max", "sigma_z2", "inv_sigma_z2",
                  "t5_dkappa_max", "t5_chi2rz_max", "t5_chi2xy_max", "t5_sigma_xy2_scaled", "t5_kappa_max",
                  "pix_dkappa_max", "pix_inv_var_xy", "pix_inv_var_rz", "pix_chi2xy_max", "pix_chi2rz_max")

    def cuts_dict(self) -> dict:
        out = {}
        for n in self.CUT_FIELDS:
            v = getattr(self, n)
            out[n] = float(v) if isinstance(v, float) else [float(x) for x in v]
        return out


class Hits(C.Structure):
    _fields_ = [("n", C.c_int32), ("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p),
                ("module", C.c_void_p), ("side", C.c_void_p), ("on_device", C.c_int32)]


class Seeds(C.Structure):
    _fields_ = [("n", C.c_int32), ("kappa", C.c_void_p), ("cphi", C.c_void_p), ("sphi", C.c_void_p), ("z0", C.c_void_p),
                ("t", C.c_void_p), ("on_device", C.c_int32)]


class PixView(C.Structure):
    _fields_ = [("n", C.c_int32), ("link", C.c_void_p), ("f", C.c_void_p), ("object_start", C.c_void_p)]


class MdView(C.Structure):
    _fields_ = [("n", C.c_int32), ("hits", C.c_void_p), ("module", C.c_void_p), ("anchor", C.c_void_p),
                ("ur_sina", C.c_void_p), ("dphi_dphichange", C.c_void_p), ("module_start", C.c_void_p),
                ("dphi_dphichange_h", C.c_void_p)]


class SegView(C.Structure):
    _fields_ = [("n", C.c_int32), ("md", C.c_void_p), ("f", C.c_void_p), ("md_start", C.c_void_p), ("f_h", C.c_void_p)]


class T3View(C.Structure):
    _fields_ = [("n", C.c_int32), ("md_kappa", C.c_void_p), ("seg", C.c_void_p), ("chi2rz", C.c_void_p),
                ("seg_start", C.c_void_p), ("chi2rz_h", C.c_void_p)]


class T5View(C.Structure):
    _fields_ = [("n", C.c_int32), ("md", C.c_void_p), ("t3", C.c_void_p), ("f", C.c_void_p), ("t3_start", C.c_void_p),
                ("f_h", C.c_void_p)]


class Stats(C.Structure):
    _fields_ = [("n_hits", C.c_int32), ("needed", C.c_int64 * 4), ("candidates", C.c_int64 * 4),
                ("evaluated", C.c_int64 * 4), ("overflow", C.c_int32), ("bad_hits", C.c_int32), ("stage_ms", C.c_float * 5), ("kernel_ms", C.c_float * 12),
                ("rewalks", C.c_int64 * 4), ("n_kept", C.c_int32), ("n_seeds", C.c_int32), ("pix_needed", C.c_int64 * 2),
                ("pix_candidates", C.c_int64 * 2), ("pix_evaluated", C.c_int64 * 2), ("pix_rewalks", C.c_int64 * 2),
                ("pix_ms", C.c_float * 3)]


class MapGeometry(C.Structure):
    _fields_ = [("n_modules", C.c_int32), ("layer", C.c_void_p), ("phi", C.c_void_p), ("rho", C.c_void_p), ("gap", C.c_void_p),
                ("half_width", C.c_void_p), ("z_lo", C.c_void_p), ("z_hi", C.c_void_p)]


class MapParams(C.Structure):
    _fields_ = [("pt_min", C.c_double), ("b_tesla", C.c_double), ("z0_max", C.c_double), ("pad_phi", C.c_double),
                ("pad_z", C.c_double)]


class TcView(C.Structure):
    _fields_ = [("n", C.c_int32), ("t5", C.c_void_p), ("keep", C.c_void_p), ("score", C.c_void_p)]


# every symbol include/lst.h declares: name -> (restype, argtypes)
P = C.POINTER
SYMBOLS = {
    "lst_default_config": (C.c_int, [P(Config)]),
    "lst_create": (C.c_int, [P(Geometry), P(ModuleMap), P(Config), P(C.c_void_p)]),
    "lst_destroy": (C.c_int, [C.c_void_p]),
    "lst_load_event": (C.c_int, [C.c_void_p, C.c_int, P(Hits), C.c_void_p]),
    "lst_load_events": (C.c_int, [C.c_void_p, C.c_int, C.c_int, P(Hits), C.c_void_p]),
    "lst_load_seeds": (C.c_int, [C.c_void_p, C.c_int, C.c_int, P(Seeds), C.c_void_p]),
    "lst_get_pixel_links": (C.c_int, [C.c_void_p, C.c_int, C.c_int, P(PixView)]),
    "lst_fetch_pixel_links": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]),
    "lst_run": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "lst_run_batch": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "lst_run_stage": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p]),
    "lst_sync": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p]),
    "lst_sync_batch": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p]),
    "lst_fetch_batch": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_int, P(C.c_void_p), P(C.c_void_p), P(C.c_int64),
                                  P(C.c_int32), C.c_int, C.c_void_p]),
    "lst_get_mds": (C.c_int, [C.c_void_p, C.c_int, P(MdView)]),
    "lst_get_segments": (C.c_int, [C.c_void_p, C.c_int, P(SegView)]),
    "lst_get_triplets": (C.c_int, [C.c_void_p, C.c_int, P(T3View)]),
    "lst_get_quintuplets": (C.c_int, [C.c_void_p, C.c_int, P(T5View)]),
    "lst_get_stats": (C.c_int, [C.c_void_p, C.c_int, P(Stats)]),
    "lst_get_track_candidates": (C.c_int, [C.c_void_p, C.c_int, P(TcView)]),
    "lst_fetch_kept": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int64, C.c_void_p]),
    "lst_fetch_hit_indices": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int64, C.c_void_p]),
    "lst_fetch_values": (C.c_int, [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int64, C.c_void_p]),
    "lst_default_map_params": (C.c_int, [P(MapParams)]),
    "lst_build_module_map": (C.c_int, [P(MapGeometry), P(MapParams), C.c_int, C.c_void_p, C.c_void_p, C.c_int64, P(C.c_int64),
                                       P(C.c_float)]),
    "lst_build_module_map_static": (C.c_int, [P(MapGeometry), P(MapParams), C.c_int, C.c_void_p, C.c_void_p, C.c_int64,
                                              C.c_void_p]),
    "lst_grown_config": (C.c_int, [C.c_void_p, C.c_int, P(Config)]),
    "lst_arena_bytes": (C.c_int, [C.c_void_p, P(C.c_int64), P(C.c_int64)]),
    "lst_launch_count": (C.c_int64, [C.c_void_p]),
    "lst_last_cuda_error": (C.c_int, [C.c_void_p]),
    "lst_strerror": (C.c_char_p, [C.c_int]),
    "lst_version": (C.c_char_p, []),
}

_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen liblst.so and bind every symbol; raises if the library or a symbol is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing: build it with `python -m paper_2207_08207_b200.build` "
                              "(there is no CPU fallback)")
        lib = C.CDLL(path)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(lib, name)            # AttributeError if the symbol is not exported
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def strerror(status: int) -> str:
    return load_library().lst_strerror(int(status)).decode()


def default_config() -> Config:
    cfg = Config()
    st = load_library().lst_default_config(C.byref(cfg))
    if st != OK:
        raise LstError(st, "lst_default_config")
    return cfg


class DeviceArray:
    """A borrowed device array (library-owned memory) visible to torch / cupy / numba."""

    def __init__(self, ptr: int, shape, typestr: str, owner):
        self._owner = owner
        self.shape = tuple(int(s) for s in shape)
        self.__cuda_array_interface__ = {"shape": self.shape, "typestr": typestr, "data": (int(ptr or 0), False),
                                         "version": 2, "strides": None}

    def torch(self):
        import torch
        if 0 in self.shape:
            return torch.empty(self.shape, dtype={"<i4": torch.int32, "<f4": torch.float32, "<f2": torch.float16, "|u1": torch.uint8}[self.__cuda_array_interface__["typestr"]], device="cuda")
        return torch.as_tensor(self, device="cuda")


def _ptr(a) -> int:
    """Raw address of a numpy array (host) or of anything with data_ptr() (torch tensor)."""
    if a is None:
        return 0
    if hasattr(a, "data_ptr"):
        return int(a.data_ptr())
    return int(a.ctypes.data)


def _stream(s) -> int:
    """None / int / torch.cuda.Stream -> cudaStream_t as an integer."""
    if s is None:
        return 0
    if hasattr(s, "cuda_stream"):
        return int(s.cuda_stream)
    return int(s)


def build_module_map(layer, phi, rho, gap, half_width, z_lo, z_hi, device: int = 0, **params):
    """Module-map builder [B] on the GPU (lst_build_module_map). Arrays: per module, host. Keyword parameters override
    lst_default_map_params (pt_min, b_tesla, z0_max, pad_phi, pad_z). Returns (row_offsets, targets, kernel_ms[2])."""
    lib = load_library()
    layer = np.ascontiguousarray(layer, np.int8)
    arrs = [np.ascontiguousarray(a, np.float64) for a in (phi, rho, gap, half_width, z_lo, z_hi)]
    n = len(layer)
    g = MapGeometry(n, _ptr(layer), *[_ptr(a) for a in arrs])
    p = MapParams()
    lib.lst_default_map_params(C.byref(p))
    for k, v in params.items():
        setattr(p, k, float(v))
    offs = np.zeros(n + 1, np.int32)
    total = C.c_int64(0)
    ms = (C.c_float * 2)()
    targets = np.zeros(1, np.int32)
    st = lib.lst_build_module_map(C.byref(g), C.byref(p), device, _ptr(offs), _ptr(targets), 0, C.byref(total), ms)
    if st == ERR_OVERFLOW:                       # the size is known now: second call with the buffer it asks for
        targets = np.zeros(max(int(total.value), 1), np.int32)
        st = lib.lst_build_module_map(C.byref(g), C.byref(p), device, _ptr(offs), _ptr(targets), len(targets), C.byref(total), ms)
    if st != OK:
        raise LstError(st, "lst_build_module_map")
    return offs, targets[:int(total.value)], [float(ms[0]), float(ms[1])]


def build_module_map_static(n_modules: int, layer, phi, rho, gap, half_width, z_lo, z_hi, row_offsets, targets, cap_targets: int,
                            device: int = 0, stream=None, **params):
    """lst_build_module_map_static: the module-map builder that allocates nothing. Every array argument is a DEVICE
    pointer (an int, or an object with ``data_ptr()``): int8 layer, float64 phi .. z_hi, int32 row_offsets [n_modules + 1]
    and targets [cap_targets]. Enqueues on ``stream`` and returns; raises LstError (ERR_LIMIT above
    MAP_STATIC_MAX_MODULES)."""
    lib = load_library()
    dp = lambda a: C.c_void_p(int(a.data_ptr()) if hasattr(a, "data_ptr") else int(a or 0))
    g = MapGeometry(int(n_modules), *[dp(a) for a in (layer, phi, rho, gap, half_width, z_lo, z_hi)])
    p = MapParams()
    lib.lst_default_map_params(C.byref(p))
    for k, v in params.items():
        setattr(p, k, float(v))
    st = lib.lst_build_module_map_static(C.byref(g), C.byref(p), int(device), dp(row_offsets), dp(targets), int(cap_targets),
                                         _stream(stream))
    if st != OK:
        raise LstError(st, "lst_build_module_map_static")


def packed_event_buffers(n: int):
    """Five numpy arrays (x, y, z, module, side) of length ``n`` inside ONE pinned host block in the "packed" layout of
    include/lst.h (each array on a 256-byte boundary, back to back): an event loaded from them travels as a single
    copy-engine transfer.  Fill them in place.  (torch is used for the pinned allocation only.)"""
    import torch
    a = (4 * n + 255) // 256 * 256
    block = torch.empty(4 * a + max(n, 1), dtype=torch.uint8).pin_memory()
    raw = block.numpy()
    out = (raw[0:4 * n].view(np.float32), raw[a:a + 4 * n].view(np.float32), raw[2 * a:2 * a + 4 * n].view(np.float32),
           raw[3 * a:3 * a + 4 * n].view(np.int32), raw[4 * a:4 * a + n])
    for v in out:
        v.flags.writeable = True
    return out + (block,)          # keep the last element alive as long as the views are used


class Lst:
    """One library context: geometry + module map + arena of event slots (lst_create)."""

    def __init__(self, layer, row_offsets, targets, config: Config | None = None, *, kind=None, cx=None, cy=None,
                 cz=None, phi=None):
        self.lib = load_library()
        self.cfg = config if config is not None else default_config()
        layer = np.ascontiguousarray(layer, np.int8)
        row_offsets = np.ascontiguousarray(row_offsets, np.int32)
        targets = np.ascontiguousarray(targets, np.int32)
        keep = [layer, row_offsets, targets]
        opt = []
        for a, dt in ((kind, np.int8), (cx, np.float32), (cy, np.float32), (cz, np.float32), (phi, np.float32)):
            a = None if a is None else np.ascontiguousarray(a, dt)
            opt.append(a)
            keep.append(a)
        g = Geometry(len(layer), _ptr(layer), *[_ptr(a) for a in opt])
        m = ModuleMap(len(row_offsets) - 1, _ptr(row_offsets), _ptr(targets))
        h = C.c_void_p()
        st = self.lib.lst_create(C.byref(g), C.byref(m), C.byref(self.cfg), C.byref(h))
        if st != OK:
            raise LstError(st, "lst_create")
        self.h = h
        self.n_modules = len(layer)
        self.n_slots = int(self.cfg.n_slots)
        self.store_half = bool(self.cfg.store_half)          # [H]: output floats are binary16 in views and fetches
        self._borrowed = {}

    @classmethod
    def from_synth(cls, geom, mmap, config: Config | None = None):
        return cls(geom.layer, mmap.row_offsets, mmap.targets, config, kind=geom.kind, cx=geom.cx, cy=geom.cy,
                   cz=geom.cz, phi=geom.phi)

    def close(self):
        if getattr(self, "h", None):
            self.lib.lst_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st, what, allow=()):
        if st != OK and st not in allow:
            raise LstError(st, what)
        return st

    # ---- the path ---------------------------------------------------------------------------
    def _marshal(self, x, y, z, module, side):
        on_device = hasattr(x, "data_ptr") and getattr(x, "is_cuda", False)
        n = int(x.shape[0])
        if not on_device and not hasattr(x, "data_ptr"):
            x, y, z = (np.ascontiguousarray(a, np.float32) for a in (x, y, z))
            module = np.ascontiguousarray(module, np.int32)
            side = np.ascontiguousarray(side, np.uint8)
        return (x, y, z, module, side), Hits(n, _ptr(x), _ptr(y), _ptr(z), _ptr(module), _ptr(side), 1 if on_device else 0)

    def load_event(self, slot: int, x, y, z, module, side, stream=None):
        """Arrays: all numpy (host) or all torch CUDA tensors (device); dtypes f32/f32/f32/i32/u8."""
        keep, hits = self._marshal(x, y, z, module, side)
        self._borrowed[slot] = keep                        # keep alive while the stream may read them
        return self._check(self.lib.lst_load_event(self.h, slot, C.byref(hits), _stream(stream)), "lst_load_event")

    def load_events(self, first_slot: int, events, stream=None):
        """events: sequence of (x, y, z, module, side) tuples; event b goes to slot first_slot + b."""
        arr = (Hits * len(events))()
        for b, ev in enumerate(events):
            keep, arr[b] = self._marshal(*ev)
            self._borrowed[first_slot + b] = keep
        return self._check(self.lib.lst_load_events(self.h, first_slot, len(events), arr, _stream(stream)), "lst_load_events")

    def load_seeds(self, first_slot: int, seeds, stream=None):
        """[P] seeds: sequence of (kappa, cphi, sphi, z0, t) tuples (all numpy / pinned host, or all torch CUDA tensors, f32);
        entry b goes to slot first_slot + b.  After load_event(s) of the same slots, on the same stream."""
        arr = (Seeds * len(seeds))()
        for b, sd in enumerate(seeds):
            on_device = hasattr(sd[0], "data_ptr") and getattr(sd[0], "is_cuda", False)
            if not hasattr(sd[0], "data_ptr"):
                sd = tuple(np.ascontiguousarray(a, np.float32) for a in sd)
            self._borrowed[("seeds", first_slot + b)] = sd
            arr[b] = Seeds(int(sd[0].shape[0]), *[_ptr(a) for a in sd], 1 if on_device else 0)
        return self._check(self.lib.lst_load_seeds(self.h, first_slot, len(seeds), arr, _stream(stream)), "lst_load_seeds")

    def run(self, slot: int, stream=None):
        return self._check(self.lib.lst_run(self.h, slot, _stream(stream)), "lst_run")

    def run_batch(self, first_slot: int, n_slots: int, stream=None):
        return self._check(self.lib.lst_run_batch(self.h, first_slot, n_slots, _stream(stream)), "lst_run_batch")

    def run_stage(self, first_slot: int, n_slots: int, stage: int, stream=None):
        return self._check(self.lib.lst_run_stage(self.h, first_slot, n_slots, stage, _stream(stream)), "lst_run_stage")

    def sync(self, slot: int, stream=None, check: bool = True) -> int:
        st = self.lib.lst_sync(self.h, slot, _stream(stream))
        if check:
            self._check(st, "lst_sync")
        return st

    def sync_batch(self, first_slot: int, n_slots: int, stream=None, check: bool = True) -> int:
        st = self.lib.lst_sync_batch(self.h, first_slot, n_slots, _stream(stream))
        if check:
            self._check(st, "lst_sync_batch")
        return st

    def fetch_batch(self, first_slot: int, kind: int, idx_out=None, val_out=None, stream=None, wait: bool = True):
        """One call for a batch of slots: idx_out / val_out are sequences of host arrays (numpy or pinned
        torch tensors; entries may be None), slot first_slot + b writes into entry b.  Returns the object
        counts.  wait=False only enqueues the copies: synchronise the stream before reading the buffers."""
        bufs = idx_out if idx_out is not None else val_out
        n = len(bufs)
        def table(seq):
            if seq is None:
                return None
            arr = (C.c_void_p * n)()
            for b, a in enumerate(seq):
                arr[b] = _ptr(a) or None
            return arr
        caps = (C.c_int64 * n)()
        for b in range(n):
            rows = [int(seq[b].shape[0]) for seq in (idx_out, val_out) if seq is not None and seq[b] is not None]
            caps[b] = min(rows) if rows else 0
        counts = (C.c_int32 * n)()
        self._check(self.lib.lst_fetch_batch(self.h, first_slot, n, kind, table(idx_out), table(val_out), caps, counts,
                                             1 if wait else 0, _stream(stream)), "lst_fetch_batch")
        return [int(v) for v in counts]

    # ---- results ----------------------------------------------------------------------------
    def stats(self, slot: int) -> dict:
        s = Stats()
        self._check(self.lib.lst_get_stats(self.h, slot, C.byref(s)), "lst_get_stats")
        return dict(n_hits=int(s.n_hits), needed=[int(v) for v in s.needed], candidates=[int(v) for v in s.candidates],
                    evaluated=[int(v) for v in s.evaluated], overflow=int(s.overflow), bad_hits=int(s.bad_hits), stage_ms=[float(v) for v in s.stage_ms],
                    kernel_ms=[float(v) for v in s.kernel_ms], rewalks=[int(v) for v in s.rewalks], n_kept=int(s.n_kept),
                    n_seeds=int(s.n_seeds), pix_needed=[int(v) for v in s.pix_needed], pix_candidates=[int(v) for v in s.pix_candidates],
                    pix_evaluated=[int(v) for v in s.pix_evaluated], pix_rewalks=[int(v) for v in s.pix_rewalks],
                    pix_ms=[float(v) for v in s.pix_ms])

    def _payload(self, p32, p16, shape):
        """The fp32 array of a view, or its binary16 twin when the context was created with store_half."""
        return DeviceArray(p16, shape, "<f2", self) if self.store_half else DeviceArray(p32, shape, "<f4", self)

    def mds(self, slot: int) -> dict:
        v = MdView()
        self._check(self.lib.lst_get_mds(self.h, slot, C.byref(v)), "lst_get_mds")
        n = v.n
        return dict(n=n, hits=DeviceArray(v.hits, (n, 2), "<i4", self), module=DeviceArray(v.module, (n,), "<i4", self),
                    anchor=DeviceArray(v.anchor, (n, 4), "<f4", self), ur_sina=DeviceArray(v.ur_sina, (n, 2), "<f4", self),
                    dphi_dphichange=self._payload(v.dphi_dphichange, v.dphi_dphichange_h, (n, 2)),
                    module_start=DeviceArray(v.module_start, (self.n_modules + 1,), "<i4", self))

    def segments(self, slot: int) -> dict:
        v = SegView()
        self._check(self.lib.lst_get_segments(self.h, slot, C.byref(v)), "lst_get_segments")
        n_md = self.stats(slot)["needed"][MD]
        return dict(n=v.n, md=DeviceArray(v.md, (v.n, 2), "<i4", self), f=self._payload(v.f, v.f_h, (v.n, 4)),
                    md_start=DeviceArray(v.md_start, (n_md + 1,), "<i4", self))

    def triplets(self, slot: int) -> dict:
        v = T3View()
        self._check(self.lib.lst_get_triplets(self.h, slot, C.byref(v)), "lst_get_triplets")
        n_seg = self.stats(slot)["needed"][SEG]
        return dict(n=v.n, md_kappa=DeviceArray(v.md_kappa, (v.n, 4), "<i4", self), seg=DeviceArray(v.seg, (v.n, 2), "<i4", self),
                    chi2rz=self._payload(v.chi2rz, v.chi2rz_h, (v.n,)), seg_start=DeviceArray(v.seg_start, (n_seg + 1,), "<i4", self))

    def quintuplets(self, slot: int) -> dict:
        v = T5View()
        self._check(self.lib.lst_get_quintuplets(self.h, slot, C.byref(v)), "lst_get_quintuplets")
        n_t3 = self.stats(slot)["needed"][T3]
        return dict(n=v.n, md=DeviceArray(v.md, (v.n, 5), "<i4", self), t3=DeviceArray(v.t3, (v.n, 2), "<i4", self),
                    f=self._payload(v.f, v.f_h, (v.n, 5)), t3_start=DeviceArray(v.t3_start, (n_t3 + 1,), "<i4", self))

    def track_candidates(self, slot: int) -> dict:
        """After run_stage(..., CLEAN) and sync: the kept quintuplets (device arrays)."""
        v = TcView()
        self._check(self.lib.lst_get_track_candidates(self.h, slot, C.byref(v)), "lst_get_track_candidates")
        n5 = self.stats(slot)["needed"][T5]
        return dict(n=v.n, t5=DeviceArray(v.t5, (v.n,), "<i4", self), keep=DeviceArray(v.keep, (n5,), "|u1", self),
                    score=DeviceArray(v.score, (n5,), "<f4", self))

    def pixel_links(self, slot: int, kind: int) -> dict:
        """After run_stage(..., PIXEL) and sync: links of kind PT3 / PT5 (device arrays)."""
        v = PixView()
        self._check(self.lib.lst_get_pixel_links(self.h, slot, kind, C.byref(v)), "lst_get_pixel_links")
        n_obj = self.stats(slot)["needed"][T5 if kind else T3]
        return dict(n=v.n, link=DeviceArray(v.link, (v.n, 2), "<i4", self), f=DeviceArray(v.f, (v.n, 3), "<f4", self),
                    object_start=DeviceArray(v.object_start, (n_obj + 1,), "<i4", self))

    def fetch_pixel_links(self, slot: int, kind: int, stream=None):
        """(link [n][2] = seed index, outer object index; f [n][3] = chi2xy, chi2rz, kappa_obj - kappa_seed), host numpy."""
        n = self.stats(slot)["pix_needed"][kind]
        link, f = np.empty((n, 2), np.int32), np.empty((n, 3), np.float32)
        self._check(self.lib.lst_fetch_pixel_links(self.h, slot, kind, _ptr(link), _ptr(f), n, _stream(stream)), "lst_fetch_pixel_links")
        return link, f

    def fetch_kept(self, slot: int, stream=None) -> np.ndarray:
        """Indices of the kept quintuplets (ascending), host numpy."""
        out = np.empty(max(self.stats(slot)["n_kept"], 1), np.int32)
        self._check(self.lib.lst_fetch_kept(self.h, slot, _ptr(out), out.shape[0], _stream(stream)), "lst_fetch_kept")
        return out[:self.stats(slot)["n_kept"]]

    def fetch_hit_indices(self, slot: int, kind: int, stream=None, out=None) -> np.ndarray:
        """[n][2|4|6|10] original hit indices of every object of class ``kind`` (host numpy)."""
        n = self.stats(slot)["needed"][kind]
        w = HITS_PER_OBJECT[kind]
        if out is None:
            out = np.empty((n, w), np.int32)
        self._check(self.lib.lst_fetch_hit_indices(self.h, slot, kind, _ptr(out), out.shape[0], _stream(stream)),
                    "lst_fetch_hit_indices")
        return out[:n]

    def fetch_values(self, slot: int, kind: int, stream=None, out=None) -> np.ndarray:
        n = self.stats(slot)["needed"][kind]
        w = VALUES_PER_OBJECT[kind]
        if out is None:
            out = np.empty((n, w), np.float16 if self.store_half else np.float32)
        self._check(self.lib.lst_fetch_values(self.h, slot, kind, _ptr(out), out.shape[0], _stream(stream)),
                    "lst_fetch_values")
        return out[:n]

    def grown_config(self, slot: int) -> Config:
        """After an overflow: this context's configuration with the exceeded capacities raised to what the slot needed x 1.25."""
        cfg = Config()
        self._check(self.lib.lst_grown_config(self.h, slot, C.byref(cfg)), "lst_grown_config")
        return cfg

    def arena_bytes(self):
        t, p = C.c_int64(), C.c_int64()
        self._check(self.lib.lst_arena_bytes(self.h, C.byref(t), C.byref(p)), "lst_arena_bytes")
        return int(t.value), int(p.value)

    def launch_count(self) -> int:
        return int(self.lib.lst_launch_count(self.h))

    def last_cuda_error(self) -> int:
        return int(self.lib.lst_last_cuda_error(self.h))
