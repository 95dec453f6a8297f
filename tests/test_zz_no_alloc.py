"""lst_build_module_map_static (include/lst.h): the module-map builder [B] for callers that cannot allocate device memory
(CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  Its only scratch is a file-scope device array of
LST_MAP_STATIC_MAX_MODULES ints; inputs and outputs are the caller's device arrays.  Checked here against the existing path
(lst_build_module_map, itself checked against the oracle in test_gpu_parity.py): integer work, so the CSR must be IDENTICAL
-- on calls in a row with different parameters (the shared scratch keeps the last call's contents), on a prefix of the
geometry, with a target buffer that is too small, and inside a captured CUDA graph.  Collected last on purpose (the name):
the suite runs with pytest -x."""
import numpy as np
import pytest

from paper_2207_08207_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def lstmod():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2207_08207_b200 import build as lst_build, lst
    lst_build.build()
    lst.load_library()
    return lst


@pytest.fixture(scope="module")
def map_inputs(geom):
    mg = synth.map_geometry(geom)
    return tuple(np.ascontiguousarray(mg[k]) for k in ("layer", "phi", "rho", "gap", "hw", "zlo", "zhi"))


def to_device(arrays):
    import torch
    return [torch.from_numpy(a).cuda() for a in arrays]


def test_static_map_builder_equals_the_allocating_path_on_calls_in_a_row(lstmod, geom, map_inputs):
    import torch
    n = geom.n_modules
    assert n <= lstmod.MAP_STATIC_MAX_MODULES
    dev = to_device(map_inputs)
    cap = 200000
    offs = torch.empty(n + 1, dtype=torch.int32, device="cuda")
    tgt = torch.empty(cap, dtype=torch.int32, device="cuda")
    stream = torch.cuda.Stream()
    # first call on the device: looks the scratch address up (may load the module); not part of the memory check below
    lstmod.build_module_map_static(n, *dev, offs, tgt, cap, 0, stream)
    stream.synchronize()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    # calls in a row on one stream, larger then smaller maps: stale row lengths of the call before would show
    for kw in (dict(), dict(pt_min=0.6), dict(pt_min=1.5, z0_max=5.0), dict(), dict(pad_phi=0.0, pad_z=0.0), dict(b_tesla=2.0)):
        offs.fill_(-7)
        tgt.fill_(-7)
        torch.cuda.synchronize()
        lstmod.build_module_map_static(n, *dev, offs, tgt, cap, 0, stream, **kw)
        stream.synchronize()
        want_o, want_t, _ = lstmod.build_module_map(*map_inputs, **kw)
        got_o = offs.cpu().numpy()
        got_t = tgt.cpu().numpy()
        assert np.array_equal(got_o, want_o), kw
        assert got_o[-1] == len(want_t) and np.array_equal(got_t[:len(want_t)], want_t), kw
        assert np.all(got_t[len(want_t):] == -7), kw                      # nothing written past the map
    assert len(lstmod.build_module_map(*map_inputs)[1]) == 69630
    # two calls back to back WITHOUT a synchronisation in between (stream order is what protects the scratch)
    offs_b = torch.empty_like(offs)
    tgt_b = torch.empty_like(tgt)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    lstmod.build_module_map_static(n, *dev, offs, tgt, cap, 0, stream, pt_min=0.6)
    lstmod.build_module_map_static(n, *dev, offs_b, tgt_b, cap, 0, stream)
    stream.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1                           # the library took no device memory
    a_o, a_t, _ = lstmod.build_module_map(*map_inputs, pt_min=0.6)
    b_o, b_t, _ = lstmod.build_module_map(*map_inputs)
    assert np.array_equal(offs.cpu().numpy(), a_o) and np.array_equal(tgt.cpu().numpy()[:len(a_t)], a_t)
    assert np.array_equal(offs_b.cpu().numpy(), b_o) and np.array_equal(tgt_b.cpu().numpy()[:len(b_t)], b_t)
    assert free1 <= free0


def test_static_map_builder_prefix_small_buffer_and_limit(lstmod, geom, map_inputs):
    """A geometry that is not a multiple of the block sizes (1 module, 1025 modules), a target buffer that is too small (only
    positions < cap_targets written, row_offsets complete), the size limit and the argument errors."""
    import ctypes as C
    import torch
    lib = lstmod.load_library()
    order = np.argsort(map_inputs[0], kind="stable")                        # keep all six layers in a prefix: interleave them
    pick = np.sort(np.concatenate([order[map_inputs[0][order] == l][:171] for l in range(6)]))[:1025]
    small_buffer_cases = 0
    for sel in (pick, pick[:1]):
        sub = tuple(np.ascontiguousarray(a[sel]) for a in map_inputs)
        dev = to_device(sub)
        m = len(sel)
        want_o, want_t, _ = lstmod.build_module_map(*sub)
        offs = torch.full((m + 1,), -7, dtype=torch.int32, device="cuda")
        tgt = torch.full((max(len(want_t), 1) + 16,), -7, dtype=torch.int32, device="cuda")
        lstmod.build_module_map_static(m, *dev, offs, tgt, len(tgt))
        torch.cuda.synchronize()
        assert np.array_equal(offs.cpu().numpy(), want_o)
        assert np.array_equal(tgt.cpu().numpy()[:len(want_t)], want_t) and np.all(tgt.cpu().numpy()[len(want_t):] == -7)
        if len(want_t) > 40:
            small_buffer_cases += 1
            small = torch.full((64,), -7, dtype=torch.int32, device="cuda")
            offs.fill_(-7)
            lstmod.build_module_map_static(m, *dev, offs, small, 40)
            torch.cuda.synchronize()
            got = small.cpu().numpy()
            assert np.array_equal(offs.cpu().numpy(), want_o) and int(offs[-1]) == len(want_t) > 40
            assert np.array_equal(got[:40], want_t[:40]) and np.all(got[40:] == -7)
            lstmod.build_module_map_static(m, *dev, offs, 0, 0)             # size query: no target buffer at all
            torch.cuda.synchronize()
            assert int(offs[-1]) == len(want_t)
    assert small_buffer_cases == 1
    # beyond the fixed maximum: rejected before anything is enqueued or any pointer is used
    dev = to_device(map_inputs)
    n = geom.n_modules
    offs = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    tgt = torch.full((16,), -7, dtype=torch.int32, device="cuda")
    with pytest.raises(lstmod.LstError) as e:
        lstmod.build_module_map_static(lstmod.MAP_STATIC_MAX_MODULES + 1, *dev, offs, tgt, 16)
    assert e.value.status == lstmod.ERR_LIMIT and "maximum" in str(e.value)
    torch.cuda.synchronize()
    assert np.all(offs.cpu().numpy() == -7) and np.all(tgt.cpu().numpy() == -7)
    for bad in (dict(n_modules=0), dict(cap_targets=-1), dict(targets=0, cap_targets=5), dict(row_offsets=0), dict(phi=0),
                dict(device=64), dict(params=dict(pt_min=0.0))):
        args = dict(n_modules=n, layer=dev[0], phi=dev[1], rho=dev[2], gap=dev[3], half_width=dev[4], z_lo=dev[5], z_hi=dev[6],
                    row_offsets=offs, targets=tgt, cap_targets=16, device=0)
        params = bad.pop("params", {})
        args.update(bad)
        with pytest.raises(lstmod.LstError) as e:
            lstmod.build_module_map_static(**args, **params)
        assert e.value.status == lstmod.ERR_ARG, bad
    g = lstmod.MapGeometry(n, *[C.c_void_p(int(t.data_ptr())) for t in dev])
    assert lib.lst_build_module_map_static(None, None, 0, C.c_void_p(int(offs.data_ptr())), C.c_void_p(int(tgt.data_ptr())), 16, None) == lstmod.ERR_ARG
    assert lib.lst_build_module_map_static(C.byref(g), None, 0, C.c_void_p(int(offs.data_ptr())), C.c_void_p(int(tgt.data_ptr())), 16, None) == lstmod.OK
    torch.cuda.synchronize()                                               # params = NULL: the defaults
    assert int(offs[-1]) == 69630


def test_static_map_builder_inside_a_captured_graph(lstmod, geom, map_inputs):
    """What the entry point is for: under stream capture cudaMalloc is not allowed; the call only enqueues three kernels, so it
    captures, and the graph replays with the inputs of the moment."""
    import torch
    n = geom.n_modules
    dev = to_device(map_inputs)
    cap = 100000
    offs = torch.full((n + 1,), -7, dtype=torch.int32, device="cuda")
    tgt = torch.full((cap,), -7, dtype=torch.int32, device="cuda")
    lstmod.build_module_map_static(n, *dev, offs, tgt, cap)                 # set-up (address look-up) outside the capture
    torch.cuda.synchronize()
    offs.fill_(-7)
    tgt.fill_(-7)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph):
        lstmod.build_module_map_static(n, *dev, offs, tgt, cap, 0, torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert int(offs[-1]) == -7                                              # captured, not run
    want_o, want_t, _ = lstmod.build_module_map(*map_inputs)
    for rep in range(2):
        graph.replay()
        torch.cuda.synchronize()
        assert np.array_equal(offs.cpu().numpy(), want_o) and np.array_equal(tgt.cpu().numpy()[:len(want_t)], want_t)
        offs.fill_(-7)
        tgt.fill_(-7)
    # the inputs of the moment: another detector in the same buffers
    rng = np.random.default_rng(8)
    phi2 = map_inputs[1] + rng.normal(0, 0.02, n)
    dev[1].copy_(torch.from_numpy(phi2))
    graph.replay()
    torch.cuda.synchronize()
    want_o, want_t, _ = lstmod.build_module_map(map_inputs[0], phi2, *map_inputs[2:])
    assert np.array_equal(offs.cpu().numpy(), want_o) and np.array_equal(tgt.cpu().numpy()[:len(want_t)], want_t)
    assert len(want_t) != 69630
