"""Pin P21 of the oracle's binary16 rounding (lsto_half_bits; DESIGN.md section 1 [H], "half precision
floats"): it must be IEEE 754 round-to-nearest-even from binary32, which is what numpy's float32 -> float16 conversion is."""
import numpy as np


def np_bits(v):
    with np.errstate(over="ignore"):
        return np.asarray(v, np.float32).astype(np.float16).view(np.uint16)


def test_p21_every_half_value_is_a_fixed_point(o32):
    h = np.arange(65536, dtype=np.uint16)
    f = h.view(np.float16).astype(np.float32)
    ok = ~np.isnan(f)
    assert np.array_equal(o32.half_bits(f)[ok], h[ok])
    assert np.all(np.isnan(o32.half_bits(f)[~ok].view(np.float16)))


def test_p21_ties_and_their_neighbours(o32):
    """Midpoints between adjacent binary16 values (exactly representable in binary32) go to the even neighbour; one
    binary32 ulp either side goes to the nearer one.  Covers subnormals, the subnormal / normal boundary, binade carries and
    the overflow threshold 65520."""
    h = np.arange(0, 0x7c00, dtype=np.uint16)                         # non-negative finite halves and their successors
    lo = h.view(np.float16).astype(np.float64)
    hi = (h + 1).astype(np.uint16).view(np.float16).astype(np.float64)
    hi[-1] = 65536.0                                                  # the value infinity stands for when rounding
    mid = ((lo + hi) / 2).astype(np.float32)
    assert np.array_equal(mid.astype(np.float64), (lo + hi) / 2)      # exact in binary32
    for sign in (1.0, -1.0):
        for v in (mid, np.nextafter(mid, np.float32(0)), np.nextafter(mid, np.float32(np.inf))):
            x = (sign * v).astype(np.float32)
            assert np.array_equal(o32.half_bits(x), np_bits(x))
    even = np.where(h % 2 == 0, h, h + 1).astype(np.uint16)
    assert np.array_equal(o32.half_bits(mid), even)


def test_p21_random_and_special_values(o32):
    rng = np.random.default_rng(21)
    x = np.concatenate([rng.normal(0, 1, 200000), rng.normal(0, 1e-4, 200000), rng.uniform(-70000, 70000, 200000),
                        10.0 ** rng.uniform(-12, 6, 200000) * rng.choice([-1, 1], 200000),
                        rng.integers(0, 2 ** 32, 400000, dtype=np.uint64).astype(np.uint32).view(np.float32).astype(np.float64)]).astype(np.float32)
    ok = ~np.isnan(x)
    assert np.array_equal(o32.half_bits(x)[ok], np_bits(x)[ok])
    sp = np.array([0.0, -0.0, np.inf, -np.inf, 65504.0, 65519.99, 65520.0, 6.1035156e-05, 5.9604645e-08, 2.9802322e-08, 2.9802326e-08, 1e-10], np.float32)
    assert np.array_equal(o32.half_bits(sp), np_bits(sp))
    assert np.isnan(o32.half_bits(np.array([np.nan], np.float32)).view(np.float16)[0])
