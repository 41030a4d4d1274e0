"""Value pins of the oracle's cut arithmetic (CPU only): every tolerance term, every endcap factor,
the order of the cuts and the near-threshold rule of CUTS.md section 0.

Each check builds ONE candidate by hand, with round numbers, and states the expected threshold as the
CUTS.md formula with those numbers substituted (plain float64 Python, next to the passage it comes
from); the oracle's own functions are called only as the thing under test.  Two kinds of assertion:
  * the value of the threshold the oracle reports (`vals`), to ~1e-6 relative;
  * the DECISION on a candidate placed just inside / just outside that threshold, and the NEAR flag on
    candidates placed at t*(1 +- 0.5e-5) (must be flagged) and t*(1 +- 2e-5) (must not), CUTS.md section 0.
A dropped term, a wrong operand (zA for zB, |ki| for max(|ki|,|ko|)) or a missing cut moves a threshold
by percent and flips one of these.  tests/test_oracle_mutants.py applies such one-line mistakes to a
copy of oracle/lst_oracle.c and shows that the checks below catch each of them.

The checks are plain functions of the oracle module `O` so that the mutant test can run them on a
mutated build; the pytest wrappers at the bottom run them on the real oracle.
"""
import math

import numpy as np

# CUTS.md section 1, in float64
KR = 100.0 / (0.3 * 3.8)
R_MIN = 0.8 * KR
INV_2RMIN = 1.0 / (2.0 * R_MIN)  # = 0.007125

EPS_IN = (-0.5e-5, +0.5e-5)    # inside the near window |v - t| <= 1e-5 |t|
EPS_OUT = (-2.0e-5, +2.0e-5)   # outside it


def f32(x):
    return float(np.float32(x))


def rel(a, b):
    return abs(float(a) - b) / abs(b)


def _bisect(fun, lo, hi, n=200):
    """Root of an increasing function by bisection (float64)."""
    flo = fun(lo)
    assert flo < 0.0 < fun(hi)
    for _ in range(n):
        mid = 0.5 * (lo + hi)
        if fun(mid) < 0.0:
            lo = mid
        else:
            hi = mid
    return 0.5 * (lo + hi)


def _expect(O_result, acc, near, what):
    got_acc, got_near, _ = O_result
    assert got_acc == acc, f"{what}: accept {got_acc}, expected {acc}"
    assert got_near == near, f"{what}: near {got_near}, expected {near}"


# ------------------------------------------------------------------------------------------------
# Mini-Doublets (CUTS.md section 3)
# ------------------------------------------------------------------------------------------------
def check_md_barrel_thresholds(O):
    """lim = (ra dd)(ra INV_2RMIN + MD_B_PHI_TOL), zl = Z0_MAX (rb - ra) + MD_Z_TOL ra."""
    ra, xb = 51.0, f32(51.26)
    dx = xb - 51.0

    def crs_over_lim(yb):  # a = (51, 0, .): crs = xa dy - ya dx = 51 yb
        dd = math.hypot(dx, f32(yb))
        return (51.0 * f32(yb)) / ((ra * dd) * (ra * INV_2RMIN + 0.06))

    y_thr = _bisect(lambda y: crs_over_lim(y) - 1.0, 0.01, 0.25)
    acc, near, v = O.md_test((51.0, 0.0, 0.0), (xb, y_thr * 0.5, 0.0), False)
    dd = math.hypot(dx, f32(y_thr * 0.5))
    assert rel(v["lim"], (51.0 * dd) * (51.0 * 0.007125 + 0.06)) < 2e-6
    rb = math.hypot(xb, f32(y_thr * 0.5))
    assert rel(v["zl"], 15.0 * (rb - 51.0) + 0.9 * 51.0) < 2e-6
    # first cut |crs| <= lim: decision 1e-3 inside / outside, near flag at +-0.5e-5 and not at +-2e-5
    for eps, acc_e, near_e in ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True),
                               (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
        for sgn in (+1.0, -1.0):
            y = _bisect(lambda yy: crs_over_lim(yy) - (1.0 + eps), 0.01, 0.25)
            _expect(O.md_test((51.0, 0.0, 0.0), (xb, sgn * y, 0.0), False), acc_e, near_e, f"MD barrel crs eps={eps}")
    # second cut zv = |zb ra - za rb| <= zl with za = 0, yb = 0: zv = |zb| 51, zl = 15 * 0.26 + 0.9 * 51
    zl = 15.0 * (xb - 51.0) + 0.9 * 51.0
    for eps, acc_e, near_e in ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True),
                               (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
        for sgn in (+1.0, -1.0):
            zb = sgn * zl / 51.0 * (1.0 + eps)
            _expect(O.md_test((51.0, 0.0, 0.0), (xb, 0.0, zb), False), acc_e, near_e, f"MD barrel zv eps={eps}")
    # the FIRST cut fails clearly, the second is at its threshold: not evaluated, not flagged (CUTS.md 0)
    zl3 = 15.0 * (math.hypot(xb, f32(0.3)) - 51.0) + 0.9 * 51.0   # yb = 0.3: crs = 15.3 >> lim = 8.6
    acc, near, v = O.md_test((51.0, 0.0, 0.0), (xb, 0.3, zl3 / 51.0), False)
    assert rel(v["zv"], float(v["zl"])) < 2e-6 and float(v["crs"]) > 1.5 * float(v["lim"])
    assert not acc and not near, "MD barrel: 2nd cut not evaluated after the 1st failed"
    # strict cut dot > 0 is never flagged: upper hit behind the beam line, |crs| = 0 = lim * 0
    _expect(O.md_test((51.0, 0.0, 0.0), (-xb, 0.0, 0.0), False), False, False, "MD barrel: dot <= 0")


def check_md_endcap_thresholds(O):
    """lim = rb ((((ra ra) dz) INV_2RMIN) MD_E_SLOPE / (|za| - Z0_MAX) + MD_E_TOL),
    rl = Z0_MAX |rb - ra| + MD_Z_TOL |za|.  a = (30, 0, 128), b at radius 30.125, z = 128.5."""
    ra, za, rb, zb = 30.0, 128.0, 30.125, 128.5
    lim = rb * ((((ra * ra) * 0.5) * 0.007125) * 1.15 / (128.0 - 15.0) + 0.015)   # = 1.434853...
    assert abs(lim - 1.4348531) < 1e-6
    rl = 15.0 * 0.125 + 0.9 * 128.0                                               # = 117.075
    acc, near, v = O.md_test((ra, 0.0, za), (rb, 0.0, zb), True)
    assert acc and rel(v["lim"], lim) < 2e-6 and rel(v["rl"], rl) < 2e-6
    assert rel(v["rv"], abs(rb * za - ra * zb)) < 1e-6  # |30.125 * 128 - 30 * 128.5| = 1
    # first cut: crs = xa yb - ya xb = ra rb sin(psi)
    for eps, acc_e, near_e in ((-5e-3, True, False), (+5e-3, False, False), (EPS_IN[0], True, True),
                               (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
        for sgn in (+1.0, -1.0):
            def ratio(psi):
                xb_, yb_ = f32(rb * math.cos(psi)), f32(rb * math.sin(psi))
                rb_ = math.hypot(xb_, yb_)
                return (ra * yb_) / (rb_ * ((((ra * ra) * 0.5) * 0.007125) * 1.15 / 113.0 + 0.015))
            psi = _bisect(lambda p: ratio(p) - (1.0 + eps), 1e-4, 0.1)
            b = (rb * math.cos(psi), sgn * rb * math.sin(psi), zb)
            _expect(O.md_test((ra, 0.0, za), b, True), acc_e, near_e, f"MD endcap crs eps={eps}")
    # second cut with crs = 0: b = (x, 0, 128.5), x < 30: rv = 3855 - 128 x, rl = 15 (30 - x) + 115.2
    for eps, acc_e, near_e in ((-2e-3, True, False), (+2e-3, False, False), (EPS_IN[0], True, True),
                               (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
        # 3855 - 128 x = (565.2 - 15 x)(1 + eps)
        x = (3855.0 - 565.2 * (1.0 + eps)) / (128.0 - 15.0 * (1.0 + eps))
        xr = f32(x)
        assert abs((3855.0 - 128.0 * xr) / (15.0 * (30.0 - xr) + 115.2) - (1.0 + eps)) < 2e-6
        _expect(O.md_test((ra, 0.0, za), (x, 0.0, zb), True), acc_e, near_e, f"MD endcap rv eps={eps}")
    # rv between MD_Z_TOL |za| = 115.2 and the full rl: accepted only because of the Z0_MAX |rb - ra| term
    acc, near, v = O.md_test((ra, 0.0, za), (29.15, 0.0, zb), True)
    assert acc and 115.2 < float(v["rv"]) < float(v["rl"])
    # first cut fails clearly, second at its threshold: not flagged
    x_thr = (3855.0 - 565.2) / (128.0 - 15.0)
    _expect(O.md_test((ra, 0.0, za), (x_thr * math.cos(0.3), x_thr * math.sin(0.3), zb), True), False, False,
            "MD endcap: 2nd cut not evaluated")


# ------------------------------------------------------------------------------------------------
# Line Segments (CUTS.md section 4)
# ------------------------------------------------------------------------------------------------
def _md(x, y, z, r, ux=1.0, uy=0.0):
    return np.array([x, y, z, r, ux, uy], dtype=np.float32)


def check_ls_thresholds(O):
    # --- kv = |kappa| R_MIN <= LS_KAPPA_MAX; A = (36, 0), B = 51 (cos phi, sin phi): kappa = 2 sin(phi) / c
    def kv_ratio(phi):
        xB, yB = f32(51.0 * math.cos(phi)), f32(51.0 * math.sin(phi))
        c = math.hypot(xB - 36.0, yB)
        return (2.0 * (36.0 * yB) / ((36.0 * 51.0) * c)) * R_MIN / 1.05
    for eps, near_e in ((EPS_IN[0], True), (EPS_IN[1], True), (EPS_OUT[0], False), (EPS_OUT[1], False), (3e-2, False)):
        phi = _bisect(lambda p: kv_ratio(p) - (1.0 + eps), 0.05, 0.6)
        for sgn in (+1.0, -1.0):
            B = _md(51.0 * math.cos(phi), sgn * 51.0 * math.sin(phi), 0.0, 51.0)
            acc, near, v = O.ls_test(_md(36.0, 0.0, 0.0, 36.0), True, B, True)   # endcap flags: no direction cuts
            assert near == near_e, f"LS kv eps={eps}: near {near}"
            assert acc == (eps < 0), f"LS kv eps={eps}: accept {acc}"
            assert rel(v["kv"], 1.05 * (1.0 + eps)) < 2e-6
    # --- zv = |zB - zA rho| <= Z0_MAX (rho - 1) + LS_Z_TOL, collinear with the beam line: kappa = 0, g = 1,
    #     rho = rB / rA = 51/36; zA = 10: zl = 15 (51/36 - 1) + 1.0 = 7.25
    rho = f32(51.0 / 36.0)
    zl = 15.0 * (rho - 1.0) + 1.0
    assert abs(zl - 7.25) < 1e-5
    A = _md(36.0, 0.0, 10.0, 36.0)
    for eps, acc_e, near_e in ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True),
                               (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
        for sgn in (+1.0, -1.0):
            B = _md(51.0, 0.0, 10.0 * rho + sgn * zl * (1.0 + eps), 51.0)
            acc, near, v = O.ls_test(A, False, B, False)
            assert (acc, near) == (acc_e, near_e), f"LS zv eps={eps}: {(acc, near)}"
            assert rel(v["zl"], zl) < 2e-6 and abs(float(v["rho"]) - 51.0 / 36.0) < 2e-7
    # dropping Z0_MAX (rho - 1) would leave zl = 1: a pair 5 cm off the pointing line is accepted (z0 spread)
    assert O.ls_test(A, False, _md(51.0, 0.0, 10.0 * rho + 5.0, 51.0), False)[0]
    # --- endcap: ztol = LS_Z_TOL (1 + |zB| / rB), with the OUTER MD's z and r.  A = (30, 0, 0), B = (60, 0, 16.1):
    #     rho = 2, zv = 16.1, zl = 15 + 1 + 16.1/60 = 16.26833 (with |zA|/rA = 0 it would be 16.0 < zv)
    A0, B0 = _md(30.0, 0.0, 0.0, 30.0), _md(60.0, 0.0, 16.1, 60.0)
    for eA, eB in ((True, False), (False, True), (True, True)):
        acc, near, v = O.ls_test(A0, eA, B0, eB)
        assert acc and not near and rel(v["zl"], 15.0 + 1.0 + f32(16.1) / 60.0) < 2e-6, (eA, eB)
    acc, near, v = O.ls_test(A0, False, B0, False)  # barrel pair: no endcap factor, zl = 16.0 < 16.1
    assert not acc and rel(v["zl"], 16.0) < 2e-6
    # the other way round: |zA|/rA large, |zB|/rB small must NOT widen the window
    A1, B1 = _md(30.0, 0.0, 60.0, 30.0), _md(60.0, 0.0, 120.0 + 18.5, 60.0)   # zv = 18.5, zl = 16 + 138.5/60 = 18.308
    acc, near, v = O.ls_test(A1, True, B1, True)
    assert not acc and rel(v["zl"], 16.0 + 138.5 / 60.0) < 2e-6
    # --- direction cuts, collinear pair (half = 0): dA = |uyA|, dB = |uyB| (e = (15, 0))
    for which in ("A", "B"):
        for eps, acc_e, near_e in ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True),
                                   (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
            for sgn in (+1.0, -1.0):
                u = sgn * 0.05 * (1.0 + eps)
                A = _md(36.0, 0.0, 0.0, 36.0, math.sqrt(1 - u * u) if which == "A" else 1.0, u if which == "A" else 0.0)
                B = _md(51.0, 0.0, 0.0, 51.0, math.sqrt(1 - u * u) if which == "B" else 1.0, u if which == "B" else 0.0)
                acc, near, v = O.ls_test(A, False, B, False)
                assert (acc, near) == (acc_e, near_e), f"LS d{which} eps={eps}: {(acc, near)}"
    # direction of an endcap MD is never read
    assert O.ls_test(_md(36.0, 0.0, 0.0, 36.0, 0.0, 1.0), True, _md(51.0, 0.0, 0.0, 51.0, 0.0, 1.0), True)[0]
    # --- order of the cuts: the first (kv) fails clearly, the second (zv) sits at its threshold: not flagged
    p = O.default_params(ls_kappa_max=-1.0)   # kv = 0 > -1 fails; |0 - (-1)| is far from the near window
    _expect(O.ls_test(_md(36.0, 0.0, 10.0, 36.0), False, _md(51.0, 0.0, 10.0 * rho + zl, 51.0), False, p), False, False,
            "LS: zv not evaluated after kv failed")
    # zv fails clearly, dA at its threshold: not flagged
    _expect(O.ls_test(_md(36.0, 0.0, 10.0, 36.0, math.sqrt(1 - 0.0025), 0.05), False,
                      _md(51.0, 0.0, 10.0 * rho + 9.0, 51.0), False), False, False, "LS: dA not evaluated after zv failed")
    # dA fails clearly, dB at its threshold: not flagged
    _expect(O.ls_test(_md(36.0, 0.0, 0.0, 36.0, 0.8, 0.6), False, _md(51.0, 0.0, 0.0, 51.0, math.sqrt(1 - 0.0025), 0.05),
                      False), False, False, "LS: dB not evaluated after dA failed")


def check_ls_direction_signs(O):
    """sA - half and sB + half (CUTS.md 4): on a circle through the beam line the chord makes the angle
    +-c kappa / 2 with the tangents at its two ends, with opposite signs.  Exact circle R = 100 (kappa = +0.01):
    x = R sin t, y = R (1 - cos t); tangent = (cos t, sin t)."""
    R = 100.0
    tA, tB = 2 * math.asin(36.0 / 200.0), 2 * math.asin(51.0 / 200.0)
    A = _md(R * math.sin(tA), R * (1 - math.cos(tA)), 0.0, 36.0, math.cos(tA), math.sin(tA))
    B = _md(R * math.sin(tB), R * (1 - math.cos(tB)), 0.0, 51.0, math.cos(tB), math.sin(tB))
    acc, near, v = O.ls_test(A, False, B, False)
    c = 2 * R * math.sin((tB - tA) / 2)
    assert acc and rel(v["kappa"], 0.01) < 1e-5 and rel(v["half"], c * 0.01 / 2) < 1e-5
    assert float(v["dA"]) < 1e-5 and float(v["dB"]) < 1e-5   # exact tangents: both residuals vanish
    # mirror image (kappa = -0.01)
    Am, Bm = A.copy(), B.copy()
    for m in (Am, Bm):
        m[1], m[5] = -m[1], -m[5]
    acc, near, v = O.ls_test(Am, False, Bm, False)
    assert acc and rel(v["kappa"], -0.01) < 1e-5 and float(v["dA"]) < 1e-5 and float(v["dB"]) < 1e-5


# ------------------------------------------------------------------------------------------------
# T3 (CUTS.md section 5)
# ------------------------------------------------------------------------------------------------
def _p4(x, y, z, r=None):
    return np.array([x, y, z, math.hypot(x, y) if r is None else r], dtype=np.float32)


def check_t3_thresholds(O):
    # --- kv = |k3| R_MIN <= T3_KAPPA_MAX on exact circle points through the origin (r = 23, 36, 51)
    def pts(R, sgn):
        out = []
        for r in (23.0, 36.0, 51.0):
            t = 2 * math.asin(r / (2 * R))
            out.append(_p4(R * math.sin(t), sgn * R * (1 - math.cos(t)), 0.0, r))
        return out

    def kv64(P):  # textbook: curvature = 4 K / (a b c), K = triangle area (float64 on the binary32 inputs)
        (ax, ay), (bx, by), (cx, cy) = [(float(q[0]), float(q[1])) for q in P]
        area2 = abs((bx - ax) * (cy - ay) - (by - ay) * (cx - ax))
        return 2 * area2 / (math.hypot(bx - ax, by - ay) * math.hypot(cx - bx, cy - by) * math.hypot(cx - ax, cy - ay)) * R_MIN
    for eps, near_e in ((EPS_IN[0], True), (EPS_IN[1], True), (EPS_OUT[0], False), (EPS_OUT[1], False), (-1e-2, False)):
        for sgn in (+1.0, -1.0):
            R = _bisect(lambda RR: (1.10 * (1.0 + eps)) - kv64(pts(RR, sgn)), 40.0, 90.0)
            P = pts(R, sgn)
            assert abs(kv64(P) / 1.10 - (1.0 + eps)) < 1.5e-6
            acc, near, v = O.t3_test(P[0], False, P[1], False, P[2], False)
            assert near == near_e and acc == (eps < 0), f"T3 kv eps={eps}: {(acc, near)}"
    # --- zv <= tol = T3_Z_TOL0 + T3_Z_TOL1 ratio, collinear in the transverse plane: A, B, C at x = 30, 60, 105:
    #     |AB| = 30, |BC| = 45, ratio = 1.5, zA = 0, zB = 10: zpred = 10 + 10 * 1.5 = 25, tol = 1.0 + 0.6 * 1.5 = 1.9
    A, B = _p4(30.0, 0.0, 0.0), _p4(60.0, 0.0, 10.0)
    for eps, acc_e, near_e in ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True),
                               (EPS_IN[1], False, True), (EPS_OUT[0], True, False), (EPS_OUT[1], False, False)):
        for sgn in (+1.0, -1.0):
            acc, near, v = O.t3_test(A, False, B, False, _p4(105.0, 0.0, 25.0 + sgn * 1.9 * (1.0 + eps)), False)
            assert (acc, near) == (acc_e, near_e), f"T3 zv eps={eps}: {(acc, near)}"
            assert rel(v["tol"], 1.9) < 2e-6 and rel(v["ratio"], 1.5) < 1e-6
    # zv = 1.5 is inside only because of the T3_Z_TOL1 ratio term (tol0 alone = 1.0)
    assert O.t3_test(A, False, B, False, _p4(105.0, 0.0, 26.5), False)[0]
    # --- endcap factor (1 + |zC| / rC) with the LAST MD's z and r, for each of the three flags:
    #     zC = 27.2: tol = 1.9 * (1 + 27.2 / 105) = 2.39219, zv = 2.2 (barrel tol 1.9 would reject)
    C = _p4(105.0, 0.0, 27.2)
    for e in ((True, False, False), (False, True, False), (False, False, True)):
        acc, near, v = O.t3_test(A, e[0], B, e[1], C, e[2])
        assert acc and rel(v["tol"], 1.9 * (1.0 + f32(27.2) / 105.0)) < 2e-6, e
    assert not O.t3_test(A, False, B, False, C, False)[0]
    # the factor uses |zC|: mirrored in z it is the same
    accm, _, vm = O.t3_test(_p4(30.0, 0.0, 0.0), True, _p4(60.0, 0.0, -10.0), False, _p4(105.0, 0.0, -27.2), False)
    assert accm and rel(vm["tol"], 1.9 * (1.0 + f32(27.2) / 105.0)) < 2e-6
    # --- order: kv fails clearly, zv at its threshold: not flagged
    p = O.default_params(t3_kappa_max=-1.0)
    _expect(O.t3_test(A, False, B, False, _p4(105.0, 0.0, 26.9), False, p), False, False, "T3: zv not evaluated")


# ------------------------------------------------------------------------------------------------
# T5 (CUTS.md section 6)
# ------------------------------------------------------------------------------------------------
def check_t5_thresholds(O):
    """tol = T5_TOL0 + T5_TOL1 max(|ki|, |ko|); cuts |ki - kb|, |kb - ko|, |ki - ko| <= tol in this order.
    Bridge MDs collinear (kb = 0 exactly), so the three differences are set directly by ki, ko."""
    B, C, D = _p4(36.0, 0.0, 0.0), _p4(51.0, 0.0, 0.0), _p4(68.0, 0.0, 0.0)
    six = ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True), (EPS_IN[1], False, True),
           (EPS_OUT[0], True, False), (EPS_OUT[1], False, False))
    for eps, acc_e, near_e in six:
        for sgn in (+1.0, -1.0):
            # cut 1: ko = 0, |ki| = tol (1 + eps), tol = 4e-4 + 0.05 |ki|
            k = 4e-4 * (1 + eps) / (1 - 0.05 * (1 + eps))
            acc, near, v = O.t5_test(sgn * k, 0.0, B, C, D)
            assert (acc, near) == (acc_e, near_e), f"T5 cut 1 eps={eps}: {(acc, near)}"
            assert float(v["kb"]) == 0.0 and rel(v["tol"], 4e-4 + 0.05 * k) < 2e-6
            # cut 2: ki = 0 (first cut passes with d1 = 0), |ko| = tol (1 + eps)
            acc, near, v = O.t5_test(0.0, sgn * k, B, C, D)
            assert (acc, near) == (acc_e, near_e), f"T5 cut 2 eps={eps}: {(acc, near)}"
            # cut 3 alone: ki = +a, ko = -a: d1 = d2 = a < tol, d3 = 2a = tol (1 + eps), tol = 4e-4 + 0.05 a
            a = 4e-4 * (1 + eps) / (2 - 0.05 * (1 + eps))
            acc, near, v = O.t5_test(sgn * a, -sgn * a, B, C, D)
            assert (acc, near) == (acc_e, near_e), f"T5 cut 3 eps={eps}: {(acc, near)}"
            if acc:
                assert rel(v["score"], 6 * a * a) < 1e-5   # a^2 + a^2 + (2a)^2
    # the third cut is a cut of its own: d1 = d2 = 3.5e-4 <= tol = 4.175e-4 but d3 = 7e-4
    _expect(O.t5_test(3.5e-4, -3.5e-4, B, C, D), False, False, "T5: |ki - ko| cut")
    # the SECOND cut alone fails: kb = 0.01 (circle R = 100), ki = kb - 5.5e-4, ko = kb - 1.0e-3:
    # tol = 4e-4 + 0.05 * 0.00945 = 8.7e-4; |d1| = 5.5e-4 and |d3| = 4.5e-4 pass, |d2| = 1.0e-3 does not
    Rb = 100.0
    Pb = []
    for r in (36.0, 51.0, 68.0):
        t = 2 * math.asin(r / (2 * Rb))
        Pb.append(_p4(Rb * math.sin(t), Rb * (1 - math.cos(t)), 0.0, r))
    _expect(O.t5_test(0.01 - 5.5e-4, 0.01 - 1.0e-3, *Pb), False, False, "T5: |kb - ko| cut")
    _expect(O.t5_test(0.01 - 5.5e-4, 0.01 - 3.0e-4, *Pb), True, False, "T5: all three inside")
    # max(|ki|, |ko|) with |ko| > |ki|: bridge on the circle R = 100 (kb = 0.01), ki = 0.0100, ko = 0.01092:
    # tol = 4e-4 + 0.05 * 0.01092 = 9.46e-4 >= |kb - ko| = |ki - ko| = 9.2e-4   (with |ki|: 9.0e-4 < 9.2e-4)
    R = 100.0
    Pc = []
    for r in (36.0, 51.0, 68.0):
        t = 2 * math.asin(r / (2 * R))
        Pc.append(_p4(R * math.sin(t), R * (1 - math.cos(t)), 0.0, r))
    acc, near, v = O.t5_test(0.0100, 0.01092, *Pc)
    assert rel(v["kb"], 0.01) < 1e-5 and rel(v["tol"], 4e-4 + 0.05 * 0.01092) < 2e-6
    assert acc and not near
    acc, near, v = O.t5_test(0.01092, 0.0100, *Pc)   # and with |ki| > |ko|
    assert acc and rel(v["tol"], 4e-4 + 0.05 * 0.01092) < 2e-6
    acc, near, v = O.t5_test(-0.0100, -0.01092, *[q * np.array([1, -1, 1, 1], np.float32) for q in Pc])  # fabsf
    assert acc and rel(v["tol"], 4e-4 + 0.05 * 0.01092) < 2e-6
    # order: cut 1 fails clearly (|ki| = 0.01 > tol = 9e-4), cut 2 at its threshold (|ko| = 9e-4): not flagged
    _expect(O.t5_test(0.01, 9e-4, B, C, D), False, False, "T5: cut 2 not evaluated after cut 1 failed")
    # cut 2 fails clearly, cut 3 at its threshold: ki = 5e-5, ko s.t. |ki - ko| = tol: not flagged
    _expect(O.t5_test(4e-4, -4.2e-4 / (1 - 0.05) + 4e-4, B, C, D), False, False, "T5: cut 3 not evaluated")


# ------------------------------------------------------------------------------------------------
# pT3 / pT5 (CUTS.md section 7)
# ------------------------------------------------------------------------------------------------
def _pls(pt, q, z0=1.5, z1=3.5):
    """Seed on the x axis: P0 = (3, 0, z0), P1 = (7, 0, z1): v = (4, 0), lv = 4, slope = (z1 - z0) / 4."""
    return np.array([pt, q, 3.0, 0.0, z0, 7.0, 0.0, z1], dtype=np.float32)


def check_pt_thresholds(O):
    six = ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True), (EPS_IN[1], False, True),
           (EPS_OUT[0], True, False), (EPS_OUT[1], False, False))
    # straight candidate on the seed's line: A = (23, 0), L = (51, 0): kx = 0, lq = 16 / 44, g = 1;
    # z on the seed's line: z = 3.5 + 0.5 * lq = 11.5 / 25.5
    A, L = _p4(23.0, 0.0, 11.5), _p4(51.0, 0.0, 25.5)
    # --- gate: A = 23 (cos th, sin th): gcrs = |vx wy - vy wx| = 4 |yA|, glim = (4 lw)(lw INV_2RMIN + PT_GATE_TOL)
    def gate_ratio(th):
        xA, yA = f32(23.0 * math.cos(th)), f32(23.0 * math.sin(th))
        lw = math.hypot(xA - 7.0, yA)
        return (4.0 * yA) / ((4.0 * lw) * (lw * 0.007125 + 0.05))
    for eps, acc_e, near_e in six:
        for sgn in (+1.0, -1.0):
            th = _bisect(lambda t: gate_ratio(t) - (1.0 + eps), 0.01, 0.5)
            Ag = _p4(23.0 * math.cos(th), sgn * 23.0 * math.sin(th), 11.5, 23.0)
            acc, near, v = O.pt_test(_pls(1e4, 1), Ag, False, Ag * np.float32(2.0), False, [0.0])
            assert near == near_e and bool(float(v["gcrs"]) <= float(v["glim"])) == acc_e, f"pT gate eps={eps}"
            lw = math.hypot(float(Ag[0]) - 7.0, float(Ag[1]))
            assert rel(v["glim"], (4.0 * lw) * (lw * 0.007125 + 0.05)) < 2e-6
    # strict cut gdot > 0 is never flagged; a seed pointing away is rejected whatever the rest
    _expect(O.pt_test(_pls(1e4, 1), _p4(-23.0, 0.0, 11.5), False, _p4(-51.0, 0.0, 25.5), False, [0.0]), False, False,
            "pT: gdot <= 0")
    # --- dp = kx - kp with kx = 0: |kp| = tolk (1 + eps), tolk = PT_K_TOL0 + PT_K_TOL1 |kp|  (pT ~ 20.5 GeV)
    for eps, acc_e, near_e in six:
        for q in (+1, -1):
            kp = 5e-4 * (1 + eps) / (1 - 0.1 * (1 + eps))
            pt = 1.0 / (kp * KR)
            assert 20.4 < pt < 20.6
            acc, near, v = O.pt_test(_pls(pt, q), A, False, L, False, [0.0])
            assert (acc, near) == (acc_e, near_e), f"pT dp eps={eps}: {(acc, near)}"
            assert float(v["kx"]) == 0.0 and rel(v["kp"], -q * kp) < 1e-6
    # --- dk = kx - kt with kx = 0, pT = 100 GeV (|kp| = 1.14e-4 passes dp): |kt| = tolk = 5e-4 + 0.1 |kp|
    kp = 1.0 / (f32(100.0) * KR)
    tolk = 5e-4 + 0.1 * kp
    for eps, acc_e, near_e in six:
        for sgn in (+1.0, -1.0):
            _expect(O.pt_test(_pls(100.0, 1), A, False, L, False, [sgn * tolk * (1 + eps)]), acc_e, near_e, f"pT3 dk eps={eps}")
            _expect(O.pt_test(_pls(100.0, 1), A, False, L, False, [0.0, sgn * tolk * (1 + eps)]), acc_e, near_e,
                    f"pT5 do eps={eps}")
            _expect(O.pt_test(_pls(100.0, 1), A, False, L, False, [sgn * tolk * (1 + eps), 0.0]), acc_e, near_e,
                    f"pT5 di eps={eps}")
    # --- r-z at A and at L (barrel): zq = |zQ - (z1 + slope lq)| <= PT_Z_TOL = 2
    for eps, acc_e, near_e in six:
        for sgn in (+1.0, -1.0):
            _expect(O.pt_test(_pls(100.0, 1), _p4(23.0, 0.0, 11.5 + sgn * 2.0 * (1 + eps)), False, L, False, [0.0]),
                    acc_e, near_e, f"pT rz(A) eps={eps}")
            _expect(O.pt_test(_pls(100.0, 1), A, False, _p4(51.0, 0.0, 25.5 + sgn * 2.0 * (1 + eps)), False, [0.0]),
                    acc_e, near_e, f"pT rz(L) eps={eps}")
    # --- endcap: zt = PT_Z_TOL (1 + |zQ| / rQ): zL = 25.5 + 2.9, zt = 2 (1 + 28.4 / 51) = 3.1137 (barrel: 2 < 2.9)
    Le = _p4(51.0, 0.0, 28.4)
    acc, near, v = O.pt_test(_pls(100.0, 1), A, False, Le, True, [0.0])
    assert acc and rel(v["zqL"], 2.9) < 1e-5
    assert not O.pt_test(_pls(100.0, 1), A, False, Le, False, [0.0])[0]
    Ae = _p4(23.0, 0.0, 14.0)                                    # zq = 2.5, zt = 2 (1 + 14 / 23) = 3.217
    assert O.pt_test(_pls(100.0, 1), Ae, True, L, False, [0.0])[0]
    assert not O.pt_test(_pls(100.0, 1), Ae, False, L, True, [0.0])[0]   # the flag of A, not of L, widens A's window
    for eps, acc_e, near_e in six:   # at the endcap threshold: zL - 25.5 = 2 (1 + zL / 51)(1 + eps)
        zL = (25.5 + 2.0 * (1 + eps)) / (1.0 - 2.0 * (1 + eps) / 51.0)
        _expect(O.pt_test(_pls(100.0, 1), A, False, _p4(51.0, 0.0, zL), True, [0.0]), acc_e, near_e, f"pT rz endcap eps={eps}")
    # --- tolk carries both terms.  pT = 0.9 GeV seed (|kp| = 0.012667, tolk = 5e-4 + 1.2667e-3) on hits of a
    #     0.8341 GeV helix (curvature 0.013667): |dp| = 1.0e-3 passes only through the PT_K_TOL1 |kp| term
    kx_true = 1.0 / (0.9 * KR) + 1.0e-3
    R = 1.0 / kx_true
    pts = []
    for r in (3.0, 7.0, 23.0, 51.0):
        t = 2 * math.asin(r / (2 * R))
        pts.append((R * math.sin(t), -R * (1 - math.cos(t)), 0.5 * R * t, r))     # clockwise: kappa < 0, q = +1
    seed = np.array([0.9, 1, pts[0][0], pts[0][1], pts[0][2], pts[1][0], pts[1][1], pts[1][2]], np.float32)
    Ac, Lc = _p4(*pts[2]), _p4(*pts[3])
    acc, near, v = O.pt_test(seed, Ac, False, Lc, False, [-kx_true])
    assert rel(v["kx"], -kx_true) < 1e-4 and abs(abs(float(v["kx"]) - float(v["kp"])) - 1.0e-3) < 2e-6
    assert acc and not near
    # ... and only the absolute term at high pT: pT = 100, |dp| = 5.05e-4 <= 5e-4 + 1.14e-5
    assert O.pt_test(_pls(100.0, 1), A, False, L, False, [0.0])[0]
    # --- scores: pT3 = dp^2 + dt^2; pT5 = ((dp^2 + di^2) + do^2) + score(T5)
    kp100 = -1.0 / (f32(100.0) * KR)
    acc, near, v = O.pt_test(_pls(100.0, 1), A, False, L, False, [2e-4])
    assert acc and rel(v["score"], kp100 ** 2 + 4e-8) < 1e-5
    acc, near, v = O.pt_test(_pls(100.0, 1), A, False, L, False, [2e-4, -3e-4], base_score=1e-7)
    assert acc and rel(v["score"], kp100 ** 2 + 4e-8 + 9e-8 + 1e-7) < 1e-5
    # --- order of the cuts: gate fails clearly / dp at threshold; dp fails clearly / dk at threshold; ...
    kp_thr = 5e-4 / (1 - 0.1)
    far = _p4(23.0 * math.cos(0.6), 23.0 * math.sin(0.6), 11.5, 23.0)
    _expect(O.pt_test(_pls(1.0 / (kp_thr * KR), 1), far, False, far * np.float32(2.0), False, [0.0]), False, False,
            "pT: dp not evaluated after the gate failed")
    _expect(O.pt_test(_pls(5.0, 1), A, False, L, False, [5e-4 + 0.1 / (5.0 * KR)]), False, False,
            "pT: dk not evaluated after dp failed")
    _expect(O.pt_test(_pls(100.0, 1), _p4(23.0, 0.0, 13.5), False, L, False, [0.01]), False, False,
            "pT: rz(A) not evaluated after dk failed")
    _expect(O.pt_test(_pls(100.0, 1), _p4(23.0, 0.0, 16.0), False, _p4(51.0, 0.0, 27.5), False, [0.0]), False, False,
            "pT: rz(L) not evaluated after rz(A) failed")
    _expect(O.pt_test(_pls(100.0, 1), A, False, L, False, [0.01, tolk]), False, False, "pT5: do not evaluated after di failed")


# ------------------------------------------------------------------------------------------------
# whole chain: counting of near-threshold candidates and NaN inputs (CUTS.md section 0)
# ------------------------------------------------------------------------------------------------
def check_event_near_counts(O):
    """One barrel module: lower hit (51, 0, 0); upper hits at the zv threshold * (1 +- 0.5e-5), * (1 +- 2e-5),
    well inside, well outside, and one that fails the first cut with zv at threshold: near[MD] = 2."""
    xb = f32(51.26)
    zthr = (15.0 * (xb - 51.0) + 0.9 * 51.0) / 51.0
    ups = [(xb, 0.0, zthr * (1 + e)) for e in (-0.5e-5, 0.5e-5, -2e-5, 2e-5, -0.5, 0.5)] + [(xb, 0.3, zthr)]
    x = np.array([51.0] + [u[0] for u in ups], np.float32)
    y = np.array([0.0] + [u[1] for u in ups], np.float32)
    z = np.array([0.0] + [u[2] for u in ups], np.float32)
    s = np.array([0] + [1] * len(ups), np.int32)
    r = O.run_event(np.zeros(1, np.int32), np.array([0, 0], np.int32), np.zeros(0, np.int32), x, y, z, s)
    assert r["n_tests"][0] == 7 and r["near"][0] == 2 and r["near"][1:].sum() == 0
    assert sorted(map(tuple, r["md_hits"].tolist())) == [(0, 1), (0, 3), (0, 5)]
    # NaN / Inf coordinates: every comparison with a NaN is false -> rejected, never flagged (CUTS.md 0)
    for bad in (np.nan, np.inf, -np.inf):
        x2, z2 = x.copy(), z.copy()
        x2[3] = bad   # hits 3 and 5 were accepted with finite coordinates
        z2[5] = bad
        r = O.run_event(np.zeros(1, np.int32), np.array([0, 0], np.int32), np.zeros(0, np.int32), x2, y, z2, s)
        assert sorted(map(tuple, r["md_hits"].tolist())) == [(0, 1)], bad
        assert r["near"][0] == 2 and r["n_tests"][0] == 7


# ------------------------------------------------------------------------------------------------
# duplicate removal, rule 2(b) in isolation (CUTS.md section 8)
# ------------------------------------------------------------------------------------------------
def check_dedup_rule_2b_isolated(O):
    """A pT3 whose ONLY reason to be removed is that its seed already carries a surviving pT5: its T3 shares
    no MD with anything, no other pT3 has its seed or overlaps it."""
    md_hits = np.arange(2 * 40, dtype=np.int32).reshape(40, 2)
    t5 = [[0, 1, 2, 3, 4]]
    t3 = [[10, 11, 12], [20, 21, 22]]
    pt5 = [[7, 0]]
    pt3 = [[7, 0], [8, 1]]          # pT3 0: seed 7 = seed of the pT5, T3 (10, 11, 12) disjoint from the T5
    k5, k3, kT, linked = O.dedup(md_hits, t3, t5, [0.1], pt3, [0.001, 0.001], pt5, [5.0], 10)
    assert k5.tolist() == [True]
    assert k3.tolist() == [False, True]
    assert np.nonzero(linked)[0].tolist() == [7, 8]
    # the pT5 removed (a better pT5 of ANOTHER seed overlaps it): rule 2(b) quantifies over SURVIVING pT5s only
    t5b = [[0, 1, 2, 3, 4], [0, 1, 2, 5, 6]]
    k5, k3, kT, linked = O.dedup(md_hits, t3, t5b, [0.1, 0.1], pt3, [0.001, 0.001], [[7, 0], [9, 1]], [5.0, 1.0], 10)
    assert k5.tolist() == [False, True] and k3.tolist() == [True, True]
    # rule 2(b), second clause alone: different seed, T3 shares exactly CROSS_SHARE = 2 MDs with the surviving pT5's T5
    k5, k3, kT, linked = O.dedup(md_hits, [[0, 1, 30], [0, 31, 32]], t5, [0.1], [[3, 0], [4, 1]], [0.001, 0.001],
                                 pt5, [5.0], 10)
    assert k3.tolist() == [False, True]
    # rule 3(c) threshold is CROSS_SHARE = 2, rule 3(a) threshold is T5_SHARE = 3
    k5, k3, kT, linked = O.dedup(md_hits, [[0, 1, 30]], [[0, 1, 33, 34, 35], [0, 36, 37, 38, 39]], [0.1, 0.1],
                                 [[3, 0]], [0.001], np.zeros((0, 2), np.int32), np.zeros(0, np.float32), 10)
    assert k3.tolist() == [True] and kT.tolist() == [False, True]


# ------------------------------------------------------------------------------------------------
# extensions: T4 (CUTS.md section 10) and the learned T5 selection (section 11)
# ------------------------------------------------------------------------------------------------
def check_t4_thresholds(O):
    """tol = T4_TOL0 + T4_TOL1 max(|k1|, |k2|); one cut |k1 - k2| <= tol; score = (k1 - k2)^2."""
    six = ((-1e-3, True, False), (+1e-3, False, False), (EPS_IN[0], True, True), (EPS_IN[1], False, True),
           (EPS_OUT[0], True, False), (EPS_OUT[1], False, False))
    for eps, acc_e, near_e in six:
        for sgn in (+1.0, -1.0):
            k = 4e-4 * (1 + eps) / (1 - 0.05 * (1 + eps))       # k2 = 0: |k1| = tol (1 + eps), tol = 4e-4 + 0.05 |k1|
            acc, near, v = O.t4_test(sgn * k, 0.0)
            assert (acc, near) == (acc_e, near_e), f"T4 eps={eps}: {(acc, near)}"
            assert rel(v["tol"], 4e-4 + 0.05 * k) < 2e-6 and rel(v["score"], k * k) < 1e-5
    # max(|k1|, |k2|) with |k2| > |k1|, both signs: tol = 4e-4 + 0.05 * 0.012 = 1.0e-3 >= |d| = 9.5e-4 (with |k1|: 9.5e-4 < ...)
    acc, near, v = O.t4_test(0.01105, 0.012)
    assert acc and rel(v["tol"], 4e-4 + 0.05 * 0.012) < 2e-6 and rel(v["d"], -9.5e-4) < 1e-4
    assert O.t4_test(-0.01105, -0.012)[0] and O.t4_test(0.012, 0.01105)[0]
    assert not O.t4_test(0.0110, 0.012)[0]                       # |d| = 1.0e-3 + ... just outside: 1.0e-3 vs tol 1.0e-3
    assert not O.t4_test(0.001, -0.001)[0]                       # opposite curvature: |d| = 2e-3 > 4.5e-4


def check_t5_mlp(O):
    """Section 11 with weights whose every product and partial sum is exact in binary32:
    S = 128, ki = 1/128, ko = 1/64, bridge collinear (kb = 0): f = (1, 0, 2, 1, 2, 1).
    unit 0: b1 = -20, W1 = (1..6): a = -20 + 1 + 0 + 6 + 4 + 10 + 6 = 7 -> h0 = 7
    unit 1: b1 = 1, W1 = -1: a = 1 - 7 = -6 -> h1 = 0 (rectifier);  units 2..7: 0
    s = b2 + W2.h = 0.25 + 0.5 * 7 + 100 * 0 = 3.75"""
    B, C, D = _p4(36.0, 0.0, 0.0), _p4(51.0, 0.0, 0.0), _p4(68.0, 0.0, 0.0)
    w = np.zeros(65, np.float32)
    w[0:6] = [1, 2, 3, 4, 5, 6]
    w[6:12] = -1
    w[48], w[49] = -20, 1
    w[56], w[57] = 0.5, 100
    w[64] = 0.25
    six = ((-1e-3, False, False), (+1e-3, True, False), (EPS_IN[0], False, True), (EPS_IN[1], True, True),
           (EPS_OUT[0], False, False), (EPS_OUT[1], True, False))
    for eps, acc_e, near_e in six:      # accept = s <= thr with thr = 3.75 (1 + eps)
        p = O.default_params(stage_mask=0x3f | 128, t5_mlp_scale=128.0, t5_mlp_thr=3.75 * (1 + eps), t5_mlp=w)
        acc, near, v = O.t5_test(1.0 / 128, 1.0 / 64, B, C, D, p)
        assert float(v["s"]) == 3.75 and (acc, near) == (acc_e, near_e), f"T5 MLP eps={eps}: {(acc, near, v)}"
        assert rel(v["score"], (1 / 128) ** 2 + (1 / 64) ** 2 + (1 / 128) ** 2) < 1e-6   # score as in section 6
    # |.| features: signs of the curvatures do not matter
    p = O.default_params(stage_mask=0x3f | 128, t5_mlp_scale=128.0, t5_mlp_thr=4.0, t5_mlp=w)
    assert float(O.t5_test(-1.0 / 128, -1.0 / 64, B, C, D, p)[2]["s"]) == 3.75
    # row-major W1[j][i]: a weight on feature 2 of unit 0 only
    w2 = np.zeros(65, np.float32)
    w2[2], w2[56] = 1.0, 1.0
    p = O.default_params(stage_mask=0x3f | 128, t5_mlp_scale=128.0, t5_mlp_thr=4.0, t5_mlp=w2)
    assert float(O.t5_test(1.0 / 128, 1.0 / 64, B, C, D, p)[2]["s"]) == 2.0     # = f[2] = |ko| S
    # without bit 7 the weights are ignored: the candidate fails the pairwise cuts of section 6 (|d2| = 1/64)
    assert not O.t5_test(1.0 / 128, 1.0 / 64, B, C, D, O.default_params(t5_mlp=w, t5_mlp_thr=100.0))[0]


def check_t4_dedup_and_event(O):
    """Rule 5 (CUTS.md section 10) on hand-made lists, and T4 enumeration / TC class 4 on a real event."""
    md_hits = np.arange(2 * 40, dtype=np.int32).reshape(40, 2)
    none2, none_f = np.zeros((0, 2), np.int32), np.zeros(0, np.float32)
    nk = np.zeros(0, bool)
    # (a) two T4s sharing 3 MDs: the lower score survives; sharing 2: both survive
    k4 = O.dedup_t4(md_hits, np.zeros((0, 3)), np.zeros((0, 5)), none2, none2, nk, nk, nk, [[0, 1, 2, 3], [1, 2, 3, 4]], [2.0, 1.0])
    assert k4.tolist() == [False, True]
    k4 = O.dedup_t4(md_hits, np.zeros((0, 3)), np.zeros((0, 5)), none2, none2, nk, nk, nk, [[0, 1, 2, 3], [2, 3, 4, 5]], [2.0, 1.0])
    assert k4.tolist() == [True, True]
    # (b) removed by a SURVIVING T5 / pT3 / pT5 sharing 2 MDs, not by a removed one
    t5 = [[0, 1, 10, 11, 12], [20, 21, 22, 23, 24]]
    k4 = O.dedup_t4(md_hits, np.zeros((0, 3)), t5, none2, none2, nk, nk, np.array([True, False]),
                    [[0, 1, 30, 31], [20, 21, 32, 33], [0, 34, 35, 36]], [1.0, 1.0, 1.0])
    assert k4.tolist() == [False, True, True]
    k4 = O.dedup_t4(md_hits, [[5, 6, 7]], t5, [[3, 0]], [[4, 1]], np.array([True]), np.array([True]), np.array([False, False]),
                    [[5, 6, 30, 31], [23, 24, 32, 33], [7, 34, 35, 36]], [1.0, 1.0, 1.0])
    assert k4.tolist() == [False, False, True]
    # whole event: enumeration by brute force over T3 pairs, structure, class order
    from lst_inputs import make_config_event, make_config_geometry

    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    r = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, O.default_params(stage_mask=0x7f))
    want = []
    for t1 in range(len(r["t3_ls"])):
        for t2 in np.nonzero(r["t3_ls"][:, 0] == r["t3_ls"][t1, 1])[0]:
            if O.t4_test(r["t3_k"][t1], r["t3_k"][t2])[0]:
                want.append((t1, int(t2)))
    assert sorted(want) == sorted(map(tuple, r["t4_t3"].tolist())) and len(want) > 100
    assert r["n_tests"][6] >= len(want) and r["n_tests"][6] == sum(
        int((r["t3_ls"][:, 0] == l).sum()) for l in r["t3_ls"][:, 1])
    a, b = r["t3_md"][r["t4_t3"][:, 0]], r["t3_md"][r["t4_t3"][:, 1]]
    assert np.array_equal(a[:, 1:], b[:, :2]) and np.array_equal(r["t4_md"], np.concatenate([a, b[:, 2:]], axis=1))
    tc = r["tc"]
    assert np.all(np.diff(tc[:, 0]) >= 0) and (tc[:, 0] == 4).sum() >= 1
    row = tc[tc[:, 0] == 4][0]
    t4 = np.nonzero(r["t4_t3"][:, 0] == row[3])[0]
    assert any(np.array_equal(row[4:12].reshape(4, 2), r["md_hits"][r["t4_md"][k]]) for k in t4) and np.all(row[12:] == -1)
    # the paper's four classes are untouched by the extension
    r0 = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    assert np.array_equal(tc[tc[:, 0] < 4], r0["tc"]) and len(r0["t4_md"]) == 0 and r0["n_tests"][6] == 0


CHECKS = (check_md_barrel_thresholds, check_md_endcap_thresholds, check_ls_thresholds, check_ls_direction_signs,
          check_t3_thresholds, check_t5_thresholds, check_pt_thresholds, check_event_near_counts,
          check_dedup_rule_2b_isolated, check_t4_thresholds, check_t5_mlp, check_t4_dedup_and_event)


def test_md_barrel_thresholds(oracle_mod):
    check_md_barrel_thresholds(oracle_mod)


def test_md_endcap_thresholds(oracle_mod):
    check_md_endcap_thresholds(oracle_mod)


def test_ls_thresholds(oracle_mod):
    check_ls_thresholds(oracle_mod)


def test_ls_direction_signs(oracle_mod):
    check_ls_direction_signs(oracle_mod)


def test_t3_thresholds(oracle_mod):
    check_t3_thresholds(oracle_mod)


def test_t5_thresholds(oracle_mod):
    check_t5_thresholds(oracle_mod)


def test_pt_thresholds(oracle_mod):
    check_pt_thresholds(oracle_mod)


def test_event_near_counts(oracle_mod):
    check_event_near_counts(oracle_mod)


def test_dedup_rule_2b_isolated(oracle_mod):
    check_dedup_rule_2b_isolated(oracle_mod)


def test_t4_thresholds(oracle_mod):
    check_t4_thresholds(oracle_mod)


def test_t5_mlp(oracle_mod):
    check_t5_mlp(oracle_mod)


def test_t4_dedup_and_event(oracle_mod):
    check_t4_dedup_and_event(oracle_mod)
