"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every
symbol include/lst.h declares, its default constants equal the oracle's (typed twice from the
SPEC), and argument errors are reported without touching the GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2207_08207_b200 import build as lst_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lst_mod():
    lst_build.build()
    from paper_2207_08207_b200 import lst
    lst.load_library()
    return lst


def test_every_declared_symbol_is_exported(lst_mod):
    header = open(os.path.join(ROOT, "include", "lst.h")).read()
    declared = set(re.findall(r"^LST_API\s+[\w\s\*]+?\b(lst_\w+)\s*\(", header, flags=re.M))
    assert len(declared) >= 20
    assert declared == set(lst_mod.SYMBOLS), declared ^ set(lst_mod.SYMBOLS)
    lib = C.CDLL(lst_mod.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lst_mod.load_library().lst_version()


def test_library_holds_sm100a_code_only():
    import subprocess
    out = subprocess.run(["cuobjdump", "-lelf", lst_build.LIB], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_\w+", out))
    assert archs == {"sm_100a"}, archs


def test_default_config_equals_oracle_constants(lst_mod, o32):
    cfg = lst_mod.default_config()
    mine, theirs = cfg.cuts_dict(), o32.config_dict()
    assert set(mine) == set(theirs)
    for k in mine:
        a = np.asarray(mine[k], np.float32)
        b = np.asarray(theirs[k], np.float32)
        assert a.tobytes() == b.tobytes(), k          # bit-identical fp32 constants
    assert cfg.n_slots == 4 and cfg.cap_hits >= 130000 and cfg.timing == 0


def test_strerror_and_status_codes(lst_mod):
    for st in (0, -1, -2, -3, -4, -5):
        assert lst_mod.strerror(st)
    assert "unknown" in lst_mod.strerror(-99)


def test_create_rejects_bad_arguments_before_any_cuda_call(lst_mod, geom, mmap):
    L = lst_mod.Lst
    def status(**kw):
        args = dict(layer=geom.layer, row_offsets=mmap.row_offsets, targets=mmap.targets, phi=geom.phi)
        args.update(kw)
        try:
            L(args["layer"], args["row_offsets"], args["targets"], args.get("config"), phi=args["phi"])
        except lst_mod.LstError as e:
            return e.status
        return 0
    bad_layer = geom.layer.copy(); bad_layer[5] = 7
    assert status(layer=bad_layer) == lst_mod.ERR_ARG
    bad_t = mmap.targets.copy(); bad_t[0] = 0                      # target not in the next layer
    assert status(targets=bad_t) == lst_mod.ERR_ARG
    bad_t = mmap.targets.copy(); bad_t[0], bad_t[1] = bad_t[1], bad_t[0]   # row not ascending
    assert status(targets=bad_t) == lst_mod.ERR_ARG
    bad_r = mmap.row_offsets.copy(); bad_r[3] = bad_r[2] - 1
    assert status(row_offsets=bad_r) == lst_mod.ERR_ARG
    cfg = lst_mod.default_config(); cfg.n_slots = 0
    assert status(config=cfg) == lst_mod.ERR_ARG
    for k in (0, 5, 11):                                           # [D]: thresholds outside 6 .. 10 are refused (include/lst.h)
        cfg = lst_mod.default_config(); cfg.t5_dup_min_shared = k
        assert status(config=cfg) == lst_mod.ERR_ARG, k
    assert status(phi=None) == lst_mod.ERR_ARG                     # module azimuths are required
    bad_phi = geom.phi.copy(); bad_phi[7] = np.nan
    assert status(phi=bad_phi) == lst_mod.ERR_ARG
    # a map row longer than LST_MAX_ROW (64) is rejected
    n1 = int(geom.n_phi[1]) * 24
    big_t = np.concatenate([np.arange(int(geom.base[1]), int(geom.base[1]) + 65, dtype=np.int32), mmap.targets[mmap.row_offsets[1]:]])
    big_r = mmap.row_offsets.copy(); big_r[1:] += 65 - (mmap.row_offsets[1] - mmap.row_offsets[0])
    assert n1 > 65 and status(targets=big_t, row_offsets=big_r) == lst_mod.ERR_ARG
    if __import__("torch").cuda.is_available():
        assert status() == 0


def test_no_cpu_fallback(lst_mod, geom, mmap):
    """Without a GPU lst_create must fail with a CUDA error status: there is no host path."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(lst_mod.LstError) as e:
        lst_mod.Lst.from_synth(geom, mmap)
    assert e.value.status in (lst_mod.ERR_CUDA, lst_mod.ERR_NOMEM)


def test_product_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under the package imports, includes or opens it."""
    pkg = os.path.join(ROOT, "paper_2207_08207_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|#include\s*[\"<][^\">]*oracle|lst_oracle|liblsto|oracle[/\\]", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), (dirpath, f)
