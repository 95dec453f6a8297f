"""Pins of the oracle (oracle/lst_oracle.c) to things other than itself.

The paper (arXiv 2207.08207) prints no worked numerical example and no formula, so nothing
here is a value quoted from it; the pins are what the paper's words and the mathematics fix
(DESIGN.md "Oracle pins"):

P1  helix closed forms: a noiseless helix through the beam line ("particle coming
    from the origin") gives sinA = -q r_u/(2R), sinS = -q r_o/(2R), kappa = kFit = -q/R, ...
P2  r-z straight-line bias of a helix in closed form ("straight line ... r-z plane")
P3  brute force: exhaustive enumeration == map-restricted search
P4  single-helix recovery: 6 MD, 5 LS, 4 T3, 2 T5 (2/4/6/10 hits)
P5  library reductions: weighted polyfit, lstsq, Heron circumradius, geometric circle fit
P6  chi2 statistics of true tracks
P7  symmetries (rotation about z, z mirror, y mirror)
P8  threshold semantics at pT = 0.8 GeV
P9  structural invariants
P10 truth sanity (PAPER.md:81, 75 % matching)
"""
import math

import numpy as np
import pytest

from paper_2207_08207_b200 import synth

KB = synth.K_GEV_PER_T_CM * synth.B_TESLA      # GeV / cm
SIG_Z = np.asarray(synth.SIGMA_Z)


# ----------------------------------------------------------------------------------------
# helpers
# ----------------------------------------------------------------------------------------
def helix_crossings(geom, pt, q, phi0, eta, z0):
    """float64 noiseless crossings of ONE helix -> dict[(layer, module)] = {side: (x, y, z)}."""
    x, y, z, mod, side, _ = synth.propagate(geom, np.array([z0]), np.array([q]), np.array([pt]),
                                            np.array([phi0]), np.array([eta]))
    out = {}
    for i in range(len(x)):
        out.setdefault((int(geom.layer[mod[i]]), int(mod[i])), {})[int(side[i])] = (x[i], y[i], z[i])
    return out


def clean_helix(geom, rng, pt_lo=0.85, pt_hi=5.0, eta_max=0.7):
    """A helix that leaves exactly one fully hit module in each of the six layers."""
    while True:
        pt = rng.uniform(pt_lo, pt_hi)
        q = rng.choice([-1.0, 1.0])
        phi0, eta, z0 = rng.uniform(-np.pi, np.pi), rng.uniform(-eta_max, eta_max), rng.normal(0, 5.0)
        cr = helix_crossings(geom, pt, q, phi0, eta, z0)
        full = [k for k, v in cr.items() if len(v) == 2]
        if len(cr) == 6 and len(full) == 6 and sorted(k[0] for k in full) == list(range(6)):
            mds = [cr[k] for k in sorted(full)]
            return dict(pt=pt, q=q, phi0=phi0, eta=eta, z0=z0, R=pt / KB), mds


def md_tuple(o, layer, md):
    """(x, y, z, r, ur, sinA) of the MD as the segment cut wants it; asserts the MD passes."""
    ok, out, _ = o.md_cut(layer, md[0], md[1])
    assert ok
    return (*md[0], out["rl"], out["ru"], out["sinA"]), out


def arc(r, R):
    return 2.0 * R * math.asin(r / (2.0 * R))


# ----------------------------------------------------------------------------------------
# P1 / P2: helix closed forms (fp64 build of the same source)
# ----------------------------------------------------------------------------------------
def test_p1_p2_helix_closed_forms(geom, o64):
    rng = np.random.default_rng(11)
    for _ in range(60):
        h, mds = clean_helix(geom, rng)
        q, R, sh, z0 = h["q"], h["R"], math.sinh(h["eta"]), h["z0"]
        t, outs = zip(*[md_tuple(o64, l, mds[l]) for l in range(6)])
        for l in range(6):
            rl, ru = t[l][3], t[l][4]
            assert rl == pytest.approx(math.hypot(mds[l][0][0], mds[l][0][1]), rel=1e-14)
            assert outs[l]["sinA"] == pytest.approx(-q * ru / (2 * R), abs=1e-10)
            assert outs[l]["dphichange"] == pytest.approx(math.asin(-q * ru / (2 * R)), abs=1e-10)
            assert outs[l]["dphi"] == pytest.approx(-q * (math.asin(ru / (2 * R)) - math.asin(rl / (2 * R))), abs=1e-10)
        for l in range(5):
            ok, s, mar = o64.seg_cut(l, t[l], t[l + 1])
            assert ok
            ri, ro = t[l][3], t[l + 1][3]
            assert s["sinS"] == pytest.approx(-q * ro / (2 * R), abs=1e-10)
            assert s["dphichange"] == pytest.approx(math.asin(-q * ro / (2 * R)), abs=1e-10)
            assert s["dphi"] == pytest.approx(-q * (math.asin(ro / (2 * R)) - math.asin(ri / (2 * R))), abs=1e-10)
            assert mar[4] < 1e-10 and mar[6] < 1e-10                      # S4 residuals vanish
            si, so = arc(ri, R), arc(ro, R)                                # P2: z0 bias
            assert s["z0"] == pytest.approx(z0 + sh * (si - ri * (so - si) / (ro - ri)), abs=1e-8)
        kap = []
        for l in range(4):
            p = [t[l + k][:4] for k in range(3)]
            ok, o3, mar = o64.t3_cut(l, *p)
            assert ok, (l, mar, h)
            assert o3["kappa"] == pytest.approx(-q / R, rel=1e-8)
            r1, r2, r3 = (pp[3] for pp in p)
            w1, w3 = (r3 - r2) / (r3 - r1), (r2 - r1) / (r3 - r1)
            delta = sh * (arc(r2, R) - w1 * arc(r1, R) - w3 * arc(r3, R))  # P2: 3-point residual
            var = SIG_Z[l + 1] ** 2 + w1 ** 2 * SIG_Z[l] ** 2 + w3 ** 2 * SIG_Z[l + 2] ** 2
            assert o3["chi2rz"] == pytest.approx(delta * delta / var, rel=1e-6, abs=1e-12)
            kap.append(o3["kappa"])
        for l in range(2):
            p = [t[l + k][:4] for k in range(5)]
            ok, o5, mar = o64.t5_cut(l, kap[l], kap[l + 2], p)
            assert mar[0] < 1e-9                                           # Q2: equal curvatures
            assert mar[4] < 1e-6                                           # Q4: exact circle -> chi2xy = 0
            if ok:
                assert o5["kfit"] == pytest.approx(-q / R, rel=1e-7)


def test_p1_fp32_build_tracks_closed_form(geom, o32):
    """The SPEC (fp32) build on fp32-rounded hits stays within input-rounding distance of P1."""
    rng = np.random.default_rng(12)
    worst = 0.0
    for _ in range(100):
        h, mds = clean_helix(geom, rng)
        for l in range(6):
            lo = tuple(np.float32(v) for v in mds[l][0])
            up = tuple(np.float32(v) for v in mds[l][1])
            ok, out, _ = o32.md_cut(l, lo, up)
            assert ok
            worst = max(worst, abs(out["sinA"] - (-h["q"] * out["ru"] / (2 * h["R"]))))
    assert worst < 2e-4          # 4 ulp of a 108 cm coordinate over a 0.16 cm lever arm


# ----------------------------------------------------------------------------------------
# P5: reductions to library routines / textbook formulas on generic (off-helix) points
# ----------------------------------------------------------------------------------------
def _rand_anchors(rng, l0, n):
    pts = []
    for k in range(n):
        r = synth.LAYER_R[l0 + k] + rng.uniform(-0.2, 0.5)
        ph = 0.3 + 0.02 * k + rng.normal(0, 0.01)
        pts.append((r * math.cos(ph), r * math.sin(ph), rng.uniform(-60, 60), r))
    return pts


def test_p5_t3_chi2_is_weighted_polyfit(o64):
    rng = np.random.default_rng(5)
    cfg = o64.default_config()
    for i in range(4):
        cfg.t3_chi2rz_max[i] = 1e30
    cfg.t3_kappa_max = 1e30
    for _ in range(200):
        l = int(rng.integers(0, 4))
        p = _rand_anchors(rng, l, 3)
        ok, out, _ = o64.t3_cut(l, *p, cfg=cfg)
        assert ok
        r = np.array([pp[3] for pp in p]); z = np.array([pp[2] for pp in p]); s = SIG_Z[l:l + 3]
        c = np.polyfit(r, z, 1, w=1.0 / s)
        chi2 = np.sum(((z - np.polyval(c, r)) / s) ** 2)
        assert out["chi2rz"] == pytest.approx(chi2, rel=1e-7, abs=1e-9)
        # circumcurvature == 4*Area/(abc) with Heron's formula, sign = orientation
        a, b, cc = (math.dist(p[i][:2], p[j][:2]) for i, j in ((0, 1), (1, 2), (0, 2)))
        sp = (a + b + cc) / 2
        area = math.sqrt(max(sp * (sp - a) * (sp - b) * (sp - cc), 0.0))
        orient = np.sign((p[1][0] - p[0][0]) * (p[2][1] - p[0][1]) - (p[1][1] - p[0][1]) * (p[2][0] - p[0][0]))
        assert out["kappa"] == pytest.approx(orient * 4 * area / (a * b * cc), rel=1e-6, abs=1e-9)


def test_p5_t5_fits_are_library_least_squares(o64):
    from scipy.optimize import least_squares
    rng = np.random.default_rng(6)
    cfg = o64.default_config()
    cfg.t5_dkappa_max = cfg.t5_chi2xy_max = cfg.t5_kappa_max = 1e30
    cfg.t5_chi2rz_max[0] = cfg.t5_chi2rz_max[1] = 1e30
    for trial in range(100):
        l = int(rng.integers(0, 2))
        R = rng.uniform(80, 2000); q = rng.choice([-1, 1])
        pts = []
        for k in range(5):                                    # circle through origin + 30 um jitter
            r = synth.LAYER_R[l + k] + rng.uniform(-0.1, 0.3)
            ph = 1.0 - q * math.asin(r / (2 * R))
            x, y = r * math.cos(ph), r * math.sin(ph)
            x += rng.normal(0, 0.003); y += rng.normal(0, 0.003)
            pts.append((x, y, rng.uniform(-50, 50), math.hypot(x, y)))
        ok, out, mar = o64.t5_cut(l, 0.0, 0.0, pts, cfg=cfg)
        assert ok
        # Q3 == weighted polyfit
        r = np.array([p[3] for p in pts]); z = np.array([p[2] for p in pts]); s = SIG_Z[l:l + 5]
        c = np.polyfit(r, z, 1, w=1.0 / s)
        assert out["chi2rz"] == pytest.approx(np.sum(((z - np.polyval(c, r)) / s) ** 2), rel=1e-7)
        # Q4 == numpy lstsq of v = A*(u^2+v^2) + B*u + C in the chord frame (any scale)
        xy = np.array([p[:2] for p in pts])
        e = (xy[4] - xy[0]) / np.linalg.norm(xy[4] - xy[0])
        d = xy - xy[2]
        u = d @ e
        v = e[0] * d[:, 1] - e[1] * d[:, 0]
        M = np.stack([u * u + v * v, u, np.ones(5)], 1)
        coef, *_ = np.linalg.lstsq(M, v, rcond=None)
        res = v - M @ coef
        assert out["chi2xy"] == pytest.approx(np.sum(res ** 2) / synth.SIGMA_RPHI ** 2, rel=1e-6, abs=1e-9)
        A, B, Cc = coef
        assert out["kfit"] == pytest.approx(2 * A / math.sqrt(1 + B * B - 4 * A * Cc), rel=1e-6, abs=1e-10)
        # ... and agrees with a geometric (orthogonal-distance) circle fit to first order
        def resid(par):
            return np.hypot(xy[:, 0] - par[0], xy[:, 1] - par[1]) - par[2]
        ph0 = 1.0 - q * math.pi / 2
        g = least_squares(resid, [R * math.cos(ph0), R * math.sin(ph0), R], xtol=1e-14, ftol=1e-14, gtol=1e-14)
        chi2_geo = np.sum(g.fun ** 2) / synth.SIGMA_RPHI ** 2
        assert out["chi2xy"] == pytest.approx(chi2_geo, rel=0.02, abs=1e-3)
        assert abs(out["kfit"]) == pytest.approx(1.0 / g.x[2], rel=2e-3)
        assert np.sign(out["kfit"]) == -q


# ----------------------------------------------------------------------------------------
# P8: threshold semantics at the pT threshold
# ----------------------------------------------------------------------------------------
def test_p8_pt_threshold_flips(geom, o64):
    cfg = o64.default_config()
    for l in range(6):
        cfg.md_cos_eps[l], cfg.md_sin_eps[l] = 1.0, 0.0
    cfg.seg_cos_eps, cfg.seg_sin_eps = 1.0, 0.0
    kmax = 2.0 * cfg.half_kappa_max
    cfg.t3_kappa_max = kmax
    pt_thr = KB / kmax                              # 0.8 GeV up to the 9-digit constant
    assert pt_thr == pytest.approx(0.8, rel=1e-7)
    rng = np.random.default_rng(8)
    n = 0
    for sign in (+1, -1):
        for _ in range(10):
            pt = pt_thr * (1 + sign * 1e-3)
            while True:
                q = rng.choice([-1.0, 1.0]); phi0 = rng.uniform(-np.pi, np.pi); eta = rng.uniform(-0.3, 0.3)
                cr = helix_crossings(geom, pt, q, phi0, eta, 0.0)
                mds = {k[0]: v for k, v in cr.items() if len(v) == 2}
                if len(cr) == len(mds) and all(l in mds for l in range(4)):
                    break
            ok_md, t = [], []
            for l in range(4):
                ok, out, mar = o64.md_cut(l, mds[l][0], mds[l][1], cfg=cfg)
                ok_md.append(ok)
                assert mar[0] / mar[1] == pytest.approx(pt_thr / pt, rel=1e-6)      # |sinA|/thr = pT_min/pT
                t.append((*mds[l][0], math.hypot(*mds[l][0][:2]), math.hypot(*mds[l][1][:2]), -q * math.hypot(*mds[l][1][:2]) * KB / (2 * pt)))
            assert all(ok_md) == (sign > 0) and any(ok_md) == (sign > 0)
            ok, _, mar = o64.seg_cut(0, t[0], t[1], cfg=cfg)
            assert ok == (sign > 0) and mar[0] / mar[1] == pytest.approx(pt_thr / pt, rel=1e-6)
            ok, _, mar = o64.t3_cut(0, t[0][:4], t[1][:4], t[2][:4], cfg=cfg)
            assert ok == (sign > 0) and mar[0] / mar[1] == pytest.approx(pt_thr / pt, rel=1e-6)
            n += 1
    assert n == 20


def test_boundary_semantics(o32):
    """Reading #14: reject on zero-length vectors, dot <= 0, dr <= 0; '<=' on thresholds."""
    assert not o32.md_cut(0, (0, 0, 0), (1, 0, 0))[0]                  # lower hit on the beam line
    assert not o32.md_cut(0, (23, 0, 0), (23, 0, 0))[0]                # identical hits
    assert not o32.md_cut(0, (23.13, 0, 0), (22.87, 0, 0))[0]          # pointing inwards: dot < 0
    assert o32.md_cut(0, (22.87, 0, 1.0), (23.13, 0, 1.0))[0]
    inner = (22.87, 0.0, 0.0, 22.87, 23.13, 0.0)
    outer = (35.57, 0.0, 0.0, 35.57, 35.83, 0.0)
    assert o32.seg_cut(0, inner, outer)[0]
    assert not o32.seg_cut(0, outer, inner)[0]                         # dr <= 0 / dot <= 0
    cfg = o32.default_config()
    ok, out, mar = o32.seg_cut(0, inner, (35.57, 0.0, 11.0, 35.57, 35.83, 0.0))
    z0 = out["z0"] if ok else mar[2]
    cfg.seg_z0_max[0] = abs(mar[2])                                    # threshold == value passes ('<=')
    assert o32.seg_cut(0, inner, (35.57, 0.0, 11.0, 35.57, 35.83, 0.0), cfg=cfg)[0]
    cfg.seg_z0_max[0] = float(np.nextafter(np.float32(abs(mar[2])), np.float32(0)))
    assert not o32.seg_cut(0, inner, (35.57, 0.0, 11.0, 35.57, 35.83, 0.0), cfg=cfg)[0]
    assert z0 == z0


# ----------------------------------------------------------------------------------------
# P18: M3 (the luminous-region term of the mini-doublet cut) in closed form + flip
# ----------------------------------------------------------------------------------------
def test_p18_m3_closed_form_and_flip(geom, o64):
    """M3 ("error terms ... take into account ... the luminous region size"; DESIGN.md SPEC [M] step 3) on
    noiseless helices, fp64 build.  A helix from (0, 0, z0) has z(r) = z0 + sinh(eta) s(r) with the arc length
    s(r) = 2R asin(r / 2R), so both sides of the inequality are known from the helix parameters and the two radii:
        lhs = |sinh(eta) (s_u - s_l) - (z0 + sinh(eta) s_l) (r_u - r_l) / r_l|,   rhs = z_lum |r_u - r_l| / r_l + 4 sqrt2 sigma_z[L].
    Flip: with md_dz_res = 0 the cut passes iff z0 lies within z_lum of a/b (a = sinh(eta) (s_u - s_l - s_l dr / r_l),
    b = dr / r_l): helices displaced to a/b +- z_lum (1 -+ 1e-3) pass, to a/b +- z_lum (1 +- 1e-3) fail."""
    rng = np.random.default_rng(18)
    z_lum = 15.0
    cfg0 = o64.default_config()
    for l in range(6):
        cfg0.md_dz_res[l] = 0.0
    n_flip = 0
    for _ in range(40):
        h, mds = clean_helix(geom, rng, eta_max=0.5)
        R, sh, z0 = h["R"], math.sinh(h["eta"]), h["z0"]
        for l in range(6):
            (xl, yl, _), (xu, yu, _) = mds[l][0], mds[l][1]
            rl, ru = math.hypot(xl, yl), math.hypot(xu, yu)
            sl, su = arc(rl, R), arc(ru, R)
            ok, _, mar = o64.md_cut(l, mds[l][0], mds[l][1])
            assert mar[2] == pytest.approx(abs(sh * (su - sl) - (z0 + sh * sl) * (ru - rl) / rl), abs=1e-9)
            assert mar[3] == pytest.approx(z_lum * abs(ru - rl) / rl + 4.0 * math.sqrt(2.0) * SIG_Z[l], rel=1e-7)   # the constant is typed as the nearest binary32
            assert ok == (mar[2] <= mar[3])
            # flip: the same trajectory in x-y displaced along the beam line
            b = (ru - rl) / rl
            centre = sh * (su - sl - sl * b) / b
            for edge in (+1.0, -1.0):
                for inside in (True, False):
                    z0n = centre + edge * z_lum * (1.0 - 1e-3 if inside else 1.0 + 1e-3)
                    lo = (xl, yl, z0n + sh * sl)
                    up = (xu, yu, z0n + sh * su)
                    ok, _, mar = o64.md_cut(l, lo, up, cfg=cfg0)
                    assert ok == inside, (l, edge, inside, mar)
                    assert mar[2] / mar[3] == pytest.approx(1.0 - 1e-3 if inside else 1.0 + 1e-3, rel=1e-6)
                    n_flip += 1
    assert n_flip == 40 * 6 * 4
