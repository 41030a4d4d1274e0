"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

PAPER.md prints no worked example ("parity unpinned" against the paper's numbers), so the
oracle is pinned by: closed forms of the helix geometry (float64 here, independent of the oracle's
binary32 arithmetic), the textbook circumradius, the asin series, hand-computable single tracks
(tests/golden/), brute-force all-pairs enumeration, structural invariants, and
monotonicity in the cut windows.
"""
import glob
import os

import numpy as np
import pytest

from lst_inputs import make_config_event, make_config_geometry
from lst_inputs.events import EventSpec, generate_event
from lst_inputs.helix import KR

from .util import canon, exact_helix_points

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
GAP = 0.26


# ------------------------------------------------------------------------------------------------
# constants and elementary functions
# ------------------------------------------------------------------------------------------------
def test_derived_constants_closed_form(oracle_mod):
    """north_star: R = pT/(0.3 B); pT threshold 0.8 GeV."""
    d = oracle_mod.derived()
    assert abs(float(d["KR"]) - 100.0 / (0.3 * 3.8)) < 1e-4
    assert abs(float(d["R_MIN"]) - 0.8 * 100.0 / (0.3 * 3.8)) < 1e-4
    assert abs(float(d["INV_2RMIN"]) * 2.0 * 70.1754386 - 1.0) < 1e-6
    assert abs(KR - float(d["KR"])) < 1e-4  # the generator's helices use the same radius law


def test_default_params_match_cuts_md(oracle_mod):
    """The defaults are the table of CUTS.md section 1 (parsed from the document)."""
    path = os.path.join(os.path.dirname(GOLDEN), "..", "CUTS.md")
    table = {}
    for line in open(path):
        cells = [c.strip() for c in line.split("|")]
        if len(cells) >= 4 and cells[1].startswith("`") and cells[1].endswith("`"):
            try:
                table[cells[1].strip("`").lower()] = float(cells[2])
            except ValueError:
                pass
    p = oracle_mod.default_params().as_dict()
    assert len(table) == 24   # 20 of sections 3-8 + 4 of the extensions (sections 10, 11)
    for name, val in table.items():
        assert p[name] == float(np.float32(val)), name


@pytest.mark.parametrize("u", [0.0, 1e-4, 0.01, 0.1, 0.3, 0.5])
def test_g_is_asin_series(oracle_mod, u):
    """g(u) ~ asin(sqrt u)/sqrt u (CUTS.md section 1): the truncated series is within 0.2% up to u = 0.5."""
    exact = 1.0 if u == 0 else np.arcsin(np.sqrt(u)) / np.sqrt(u)
    got = float(oracle_mod.g(u))
    assert got <= exact + 1e-6  # truncated series with positive terms undershoots
    assert abs(got - exact) / exact < (2e-3 if u > 0.3 else 2e-5 if u <= 0.1 else 3e-4)


def test_g_taylor_coefficients(oracle_mod):
    """First two series coefficients 1/6 and 3/40 (asin x = x + x^3/6 + 3x^5/40 + ...)."""
    u = 1e-2
    g = float(oracle_mod.g(u))
    assert abs((g - 1.0) / u - (1.0 / 6.0 + 0.075 * u)) < 1e-4
    u = 0.25
    g = float(oracle_mod.g(u))
    series = 1 + u / 6 + 3 * u**2 / 40 + 15 * u**3 / 336 + 105 * u**4 / 3456
    assert abs(g - series) < 1e-6


@pytest.mark.parametrize("R,ccw", [(100.0, True), (70.2, False), (1234.5, True), (30.0, False)])
def test_kappa3_is_textbook_circumradius(oracle_mod, R, ccw):
    """kappa3 = +-1/R on exact circle points; R = abc/(4K) (Heron) in float64."""
    cx, cy = 3.0, -7.0
    ang = np.array([0.1, 0.35, 0.8]) * (1 if ccw else -1)
    P = np.stack([cx + R * np.cos(ang), cy + R * np.sin(ang)], axis=1)
    k, ln = oracle_mod.kappa3(P[0], P[1], P[2])
    a, b, c = (np.linalg.norm(P[1] - P[0]), np.linalg.norm(P[2] - P[1]), np.linalg.norm(P[2] - P[0]))
    s = 0.5 * (a + b + c)
    K = np.sqrt(s * (s - a) * (s - b) * (s - c))
    assert abs(abs(float(k)) - 4 * K / (a * b * c)) < 2e-3 / R
    assert abs(float(k) * R - (1.0 if ccw else -1.0)) < 2e-3
    assert np.allclose(ln, [a, b, c], rtol=1e-5)


def test_kappa3_collinear_is_zero_and_antisymmetric(oracle_mod):
    k, _ = oracle_mod.kappa3((0, 0), (1, 2), (3, 6))
    assert float(k) == 0.0
    k1, _ = oracle_mod.kappa3((0, 0), (10, 1), (20, 5))
    k2, _ = oracle_mod.kappa3((20, 5), (10, 1), (0, 0))
    assert float(k1) > 0 and abs(float(k1) + float(k2)) < 1e-7  # reversing the path flips the sign


# ------------------------------------------------------------------------------------------------
# closed-form helix pins of every cut quantity
# ------------------------------------------------------------------------------------------------
def _md_from_points(oracle_mod, lo, hi, endcap=False):
    acc, near, v = oracle_mod.md_test(lo, hi, endcap)
    r = np.float32(np.sqrt(np.float32(lo[0]) ** 2 + np.float32(lo[1]) ** 2))
    md = np.array([lo[0], lo[1], lo[2], r, v.get("ux", 0.0), v.get("uy", 0.0)], dtype=np.float32)
    return acc, v, md


@pytest.mark.parametrize("pt,q,layer_r", [(0.8, 1, 36.0), (1.0, -1, 51.0), (2.5, 1, 108.0), (0.8, -1, 108.0)])
def test_md_barrel_tangent_chord(oracle_mod, pt, q, layer_r):
    """Helix through the beam line: sin(radial, tangent) = r/2R (CUTS.md section 3); sign = -q."""
    pts, trk = exact_helix_points(pt, q, 0.7, 0.4, 3.0, [layer_r, layer_r + GAP])
    acc, near, v = oracle_mod.md_test(pts[0], pts[1], False)
    R = pt * KR
    ra = np.hypot(pts[0][0], pts[0][1])
    sin_meas = float(v["crs"]) / (ra * float(v["dd"]))
    assert np.sign(sin_meas) == -q
    assert abs(abs(sin_meas) - ra / (2 * R)) / (ra / (2 * R)) < 0.012  # finite 2.6 mm step
    assert acc and not near
    assert abs(float(v["lim"]) / (ra * float(v["dd"])) - (ra / (2 * 70.17544) + 0.06)) < 1e-5
    assert abs(np.hypot(float(v["ux"]), float(v["uy"])) - 1.0) < 1e-6


def test_md_barrel_straight_line_pointing(oracle_mod):
    """Straight line from (0, z0): |zb ra - za rb| = |z0| (rb - ra), crs = 0 (CUTS.md section 3)."""
    z0, cot, phi = -7.5, 0.9, 2.1
    pts = [(r * np.cos(phi), r * np.sin(phi), z0 + cot * r) for r in (68.0, 68.0 + GAP)]
    acc, near, v = oracle_mod.md_test(pts[0], pts[1], False)
    assert acc
    assert abs(float(v["crs"])) < 1e-3
    assert abs(float(v["zv"]) - abs(z0) * GAP) < 5e-3
    assert abs(float(v["zl"]) - (15.0 * GAP + 0.9 * 68.0)) < 1e-3
    # a line from z0 = 300 cm (far outside the luminous region) fails the pointing cut
    pts = [(r * np.cos(phi), r * np.sin(phi), 300.0 - 2.0 * r) for r in (68.0, 68.0 + GAP)]
    assert not oracle_mod.md_test(pts[0], pts[1], False)[0]


def test_md_barrel_rejects_low_pt_and_backwards(oracle_mod):
    pts, _ = exact_helix_points(0.6, 1, 0.0, 0.0, 0.0, [51.0, 51.0 + GAP])  # r/2R = 0.485 > 0.423
    assert not oracle_mod.md_test(pts[0], pts[1], False)[0]
    pts, _ = exact_helix_points(5.0, 1, 0.0, 0.0, 0.0, [51.0, 51.0 + GAP])
    assert oracle_mod.md_test(pts[0], pts[1], False)[0]
    # upper hit on the opposite side of the beam line: dot < 0
    assert not oracle_mod.md_test((51.0, 0.0, 0.0), (-51.26, 0.0, 0.0), False)[0]


@pytest.mark.parametrize("pt,q,eta", [(0.9, 1, 1.6), (2.0, -1, 2.0), (1.2, 1, -1.8)])
def test_md_endcap_bend_and_pointing(oracle_mod, pt, q, eta):
    """Endcap MD: crs = ra rb sin(dphi) with dphi the exact helix rotation between the two planes;
    |rb za - ra zb| -> |z0| |rb - ra| for a straight line (CUTS.md section 3)."""
    from lst_inputs.helix import Tracks

    z0 = 4.0
    zd = 160.0 * np.sign(eta)
    trk = Tracks([0.0], [0.0], [z0], [1.1], [eta], [pt], [q])
    P = []
    for zz in (zd, zd + 0.4 * np.sign(eta)):
        t = trk.plane_crossing(zz)
        x, y, z = trk.pos(t)
        P.append((x[0], y[0], z[0]))
    acc, near, v = oracle_mod.md_test(P[0], P[1], True)
    ra, rb = np.hypot(*P[0][:2]), np.hypot(*P[1][:2])
    dphi = np.arctan2(P[1][1], P[1][0]) - np.arctan2(P[0][1], P[0][0])
    assert abs(float(v["crs"]) - ra * rb * np.sin(dphi)) < 2e-3
    assert np.sign(float(v["crs"])) == -q
    assert acc
    # straight line r = (z - z0) tan(theta)
    tan = 0.35
    P = [((zz - z0) * tan, 0.0, zz) for zz in (190.0, 190.4)]
    acc, near, v = oracle_mod.md_test(P[0], P[1], True)
    assert acc and abs(float(v["rv"]) - z0 * 0.4 * tan) < 5e-3 and abs(float(v["crs"])) < 1e-6


@pytest.mark.parametrize("pt,q,r1,r2", [(0.8, 1, 23.0, 36.0), (1.0, -1, 36.0, 51.0), (3.0, 1, 88.0, 108.0),
                                        (0.85, -1, 68.0, 88.0)])
def test_ls_closed_forms(oracle_mod, pt, q, r1, r2):
    """Circle through the beam line, A, B: kappa R = -q exactly; rho = arc-length ratio
    s(r) = 2R asin(r/2R); zB - zA rho = z0 (1 - rho); tangent-chord angle sin = c/2R at both ends
    with opposite signs (CUTS.md section 4)."""
    z0, eta = 5.0, 0.5
    pts, trk = exact_helix_points(pt, q, 2.3, eta, z0, [r1, r1 + GAP, r2, r2 + GAP])
    accA, _, mdA = _md_from_points(oracle_mod, pts[0], pts[1])
    accB, _, mdB = _md_from_points(oracle_mod, pts[2], pts[3])
    assert accA and accB
    acc, near, v = oracle_mod.ls_test(mdA, False, mdB, False)
    R = pt * KR
    assert abs(float(v["kappa"]) * R + q) < 2e-4
    assert abs(float(v["kv"]) - 70.17544 / R) < 2e-4
    s = lambda r: 2 * R * np.arcsin(r / (2 * R))
    assert abs(float(v["rho"]) - s(r2) / s(r1)) / (s(r2) / s(r1)) < 2.5e-3  # series truncation at low pT
    assert abs(float(v["zv"]) - abs(z0) * (float(v["rho"]) - 1.0)) < 0.15
    c = np.hypot(pts[2][0] - pts[0][0], pts[2][1] - pts[0][1])
    assert abs(float(v["half"]) - (-q) * c / (2 * R)) < 1e-4
    assert float(v["dA"]) < 4e-3 and float(v["dB"]) < 4e-3  # finite 2.6 mm step only
    assert acc
    # the direction terms really carry opposite signs: swapping the sign convention must fail
    mdB_flipped = mdB.copy()
    mdB_flipped[4:6] = -mdB[4:6]
    assert not oracle_mod.ls_test(mdA, False, mdB_flipped, False)[0]


def test_ls_rejects_low_pt_pair_and_bad_z(oracle_mod):
    pts, _ = exact_helix_points(0.6, 1, 0.3, 0.2, 0.0, [23.0, 23.0 + GAP, 36.0, 36.0 + GAP])
    mdA = np.array([*pts[0], 23.0, 1, 0], dtype=np.float32)
    mdB = np.array([*pts[2], 36.0, 1, 0], dtype=np.float32)
    acc, near, v = oracle_mod.ls_test(mdA, True, mdB, True)  # endcap flags: direction cuts skipped
    assert not acc and float(v["kv"]) > 1.05
    pts, _ = exact_helix_points(2.0, 1, 0.3, 0.2, 0.0, [23.0, 36.0])
    mdA = np.array([*pts[0], 23.0, 0, 0], dtype=np.float32)
    mdB = np.array([pts[1][0], pts[1][1], pts[1][2] + 30.0, 36.0, 0, 0], dtype=np.float32)
    assert oracle_mod.ls_test(mdA, True, np.array([*pts[1], 36.0, 0, 0], np.float32), True)[0]
    assert not oracle_mod.ls_test(mdA, True, mdB, True)[0]


@pytest.mark.parametrize("pt,q", [(0.8, 1), (1.5, -1), (10.0, 1)])
def test_t3_t5_closed_forms(oracle_mod, pt, q):
    """kappa3 R = -q on exact helix points; z is linear in arc length, so the chord-ratio prediction
    is good to a few mm; a noise-free track has T5 score ~ 0 (CUTS.md sections 5, 6)."""
    radii = [23.0, 36.0, 51.0, 68.0, 88.0]
    pts, _ = exact_helix_points(pt, q, 4.0, 0.6, -3.0, radii)
    md = [np.array([*p, r], dtype=np.float32) for p, r in zip(pts, radii)]
    R = pt * KR
    acc, near, v1 = oracle_mod.t3_test(md[0], False, md[1], False, md[2], False)
    assert acc and abs(float(v1["k3"]) * R + q) < 1e-3
    assert float(v1["zv"]) < 0.25
    acc, near, v2 = oracle_mod.t3_test(md[2], False, md[3], False, md[4], False)
    assert acc and abs(float(v2["k3"]) * R + q) < 1e-3
    acc, near, v = oracle_mod.t5_test(v1["k3"], v2["k3"], md[1], md[2], md[3])
    assert acc and abs(float(v["kb"]) * R + q) < 1e-3
    assert float(v["score"]) < 1e-9
    assert abs(float(v["tol"]) - (4e-4 + 0.05 / R)) < 2e-6
    # a T5 whose halves have opposite curvature is rejected
    assert not oracle_mod.t5_test(v1["k3"], -v2["k3"], md[1], md[2], md[3])[0] or pt > 5.0


def test_t3_rejects_kink_in_z(oracle_mod):
    radii = [23.0, 36.0, 51.0]
    pts, _ = exact_helix_points(3.0, 1, 1.0, 0.3, 0.0, radii)
    md = [np.array([*p, r], dtype=np.float32) for p, r in zip(pts, radii)]
    assert oracle_mod.t3_test(md[0], False, md[1], False, md[2], False)[0]
    md[2][2] += 5.0
    acc, near, v = oracle_mod.t3_test(md[0], False, md[1], False, md[2], False)
    assert not acc and abs(float(v["zv"]) - 5.0) < 0.3


@pytest.mark.parametrize("pt,q", [(0.9, 1), (2.0, -1), (8.0, 1)])
def test_pt_closed_forms(oracle_mod, pt, q):
    """kp = -q/(pT KR); the circle through P1 and the outer MDs has the track's curvature; z follows
    the arc length (CUTS.md section 7).  Wrong-charge seed is rejected."""
    z0, eta = 2.0, 0.7
    radii = [3.0, 7.0, 23.0, 36.0, 51.0, 68.0, 88.0]
    pts, _ = exact_helix_points(pt, q, 5.5, eta, z0, radii)
    md = [np.array([*p, r], dtype=np.float32) for p, r in zip(pts[2:], radii[2:])]
    pls = np.array([pt, q, *pts[0], *pts[1]], dtype=np.float32)
    R = pt * KR
    k3 = oracle_mod.t3_test(md[0], False, md[1], False, md[2], False)[2]["k3"]
    acc, near, v = oracle_mod.pt_test(pls, md[0], False, md[2], False, [k3])
    assert abs(float(v["kp"]) - (-q) / (pt * 87.7193)) < 1e-7
    assert abs(float(v["kx"]) * R + q) < 2e-3
    assert float(v["zqA"]) < 0.05 and float(v["zqL"]) < 0.05
    assert float(v["gdot"]) > 0 and float(v["gcrs"]) <= float(v["glim"])
    assert acc and float(v["score"]) < 1e-8
    ko = oracle_mod.t3_test(md[2], False, md[3], False, md[4], False)[2]["k3"]
    acc5, _, v5 = oracle_mod.pt_test(pls, md[0], False, md[4], False, [k3, ko], base_score=1e-3)
    assert acc5 and abs(float(v5["score"]) - 1e-3) < 1e-6
    if pt < 3:
        bad = pls.copy()
        bad[1] = -q
        assert not oracle_mod.pt_test(bad, md[0], False, md[2], False, [k3])[0]
    # seed pointing away from the T3 fails the gate
    back = pls.copy()
    back[2:5], back[5:8] = pls[5:8], pls[2:5]
    assert not oracle_mod.pt_test(back, md[0], False, md[2], False, [k3])[0]


# ------------------------------------------------------------------------------------------------
# hand-computable single tracks (tests/golden/)
# ------------------------------------------------------------------------------------------------
def _load_golden(path):
    hits, expect = [], {}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        if line.startswith("expect"):
            for tok in line.split()[1:]:
                k, v = tok.split("=")
                expect[k] = v
        else:
            x, y, z, s = line.split()
            hits.append((float(x), float(y), float(z), int(s)))
    return np.array(hits), expect


@pytest.mark.parametrize("path", sorted(glob.glob(os.path.join(GOLDEN, "*.txt"))), ids=os.path.basename)
def test_golden_single_tracks(oracle_mod, path):
    hits, exp = _load_golden(path)
    n_mod = 6 if exp["modules"] == "barrel" else 5
    subdet = np.full(n_mod, 0 if exp["modules"] == "barrel" else 1, dtype=np.int32)
    off = np.concatenate([np.arange(n_mod), [n_mod - 1]]).astype(np.int32)  # k -> k+1, last has none
    tgt = np.arange(1, n_mod, dtype=np.int32)
    r = oracle_mod.run_event(subdet, off, tgt, hits[:, 0], hits[:, 1], hits[:, 2], hits[:, 3].astype(np.int32),
                             params=oracle_mod.default_params(stage_mask=0x0f))
    assert len(r["md_hits"]) == int(exp["n_md"])
    assert len(r["ls_md"]) == int(exp["n_ls"])
    assert len(r["t3_md"]) == int(exp["n_t3"])
    assert len(r["t5_md"]) == int(exp["n_t5"])
    kappa = float(exp["kappa"])
    if len(r["ls_md"]):
        assert np.allclose(r["ls_kappa"], kappa, atol=2e-6)
        assert np.allclose(r["t3_k"], kappa, atol=2e-6)
        assert np.all(r["t5_score"] < 1e-10)
        # MD k pairs hits (2k, 2k+1) of the file, LS k links MD k -> k+1
        assert np.array_equal(r["md_hits"], np.arange(2 * n_mod).reshape(-1, 2))
        assert np.array_equal(r["ls_md"], np.stack([np.arange(n_mod - 1), np.arange(1, n_mod)], 1))
        assert np.array_equal(r["t5_md"][0], np.arange(5))


# ------------------------------------------------------------------------------------------------
# brute force on tiny events: enumeration (binning, map walk, chaining) vs all-pairs
# ------------------------------------------------------------------------------------------------
def _tiny_event(kind):
    geom, off, tgt = make_config_geometry("C1")
    if kind == "C1":
        return geom, off, tgt, make_config_event("C1")
    # 40 helices squeezed into a narrow (phi, eta) wedge so that modules hold several hits each
    spec = EventSpec(n_tracks=40, pt_dist=("loguniform", 0.8, 10.0), eta_max=0.25, noise=("count", 100),
                     seeds=True, sigma_vz=2.0, phi_range=(0.2, 0.7))
    return geom, off, tgt, generate_event(geom, spec, seed=77)


@pytest.mark.parametrize("kind", ["C1", "dense"])
def test_bruteforce_all_pairs(oracle_mod, kind):
    geom, off, tgt, ev = _tiny_event(kind)
    O = oracle_mod
    p = O.default_params()
    res = O.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, p)
    c = canon(res)
    hx = np.stack([ev.x, ev.y, ev.z], axis=1)
    n = ev.n_hits

    # candidates visited and near-threshold flags raised per stage (MD, LS, T3, T5, pT3, pT5), counted by this
    # enumeration: the oracle's n_tests / near counters (CUTS.md section 0) must equal them
    n_cand, n_near = [0] * 6, [0] * 6

    # MD: every ordered hit pair of the whole event, kept only if (lower, upper) of one module
    mds = {}
    for a in range(n):
        for b in range(n):
            sa, sb = int(ev.sensor[a]), int(ev.sensor[b])
            if sa % 2 == 0 and sb == sa + 1:
                m = sa // 2
                acc, near, v = O.md_test(hx[a], hx[b], bool(geom.subdet[m]), p)
                n_cand[0] += 1
                n_near[0] += int(near)
                if acc:
                    r = np.float32(np.sqrt(ev.x[a] * ev.x[a] + ev.y[a] * ev.y[a]))
                    ecap = bool(geom.subdet[m])
                    mds[(a, b)] = (m, np.array([*hx[a], r, 0 if ecap else v["ux"], 0 if ecap else v["uy"]], np.float32))
    assert sorted(mds) == [tuple(t) for t in c["md"]]

    conn = {m: tgt[off[m]:off[m + 1]].tolist() for m in range(geom.n_modules)}
    assert all(len(set(row)) == len(row) for row in conn.values())  # no module twice in a row of the map
    keys = sorted(mds)
    # LS: every ordered MD pair, kept only if module(B) in conn[module(A)]
    lss = {}
    for A in keys:
        mA, fA = mds[A]
        for B in keys:
            mB, fB = mds[B]
            if mB in conn[mA]:
                acc, near, v = O.ls_test(fA, bool(geom.subdet[mA]), fB, bool(geom.subdet[mB]), p)
                n_cand[1] += 1
                n_near[1] += int(near)
                if acc:
                    lss[(A, B)] = v["kappa"]
    assert sorted(a + b for a, b in lss) == [tuple(t) for t in c["ls"]]

    # T3: every ordered LS pair sharing the middle MD
    t3s = {}
    for (A, B) in lss:
        for (B2, Cc) in lss:
            if B2 == B:
                e = [bool(geom.subdet[mds[k][0]]) for k in (A, B, Cc)]
                acc, near, v = O.t3_test(mds[A][1], e[0], mds[B][1], e[1], mds[Cc][1], e[2], p)
                n_cand[2] += 1
                n_near[2] += int(near)
                if acc:
                    t3s[(A, B, Cc)] = v["k3"]
    assert sorted(a + b + d for a, b, d in t3s) == [tuple(t) for t in c["t3"]]

    # T5: every ordered T3 pair with last MD of the first = first MD of the second
    t5s = {}
    for (A, B, Cc), ki in t3s.items():
        for (C2, D, E), ko in t3s.items():
            if C2 == Cc:
                acc, near, v = O.t5_test(ki, ko, mds[B][1], mds[Cc][1], mds[D][1], p)
                n_cand[3] += 1
                n_near[3] += int(near)
                if acc:
                    t5s[(A, B, Cc, D, E)] = v["score"]
    assert sorted(sum(k, ()) for k in t5s) == [tuple(t) for t in c["t5"]]
    assert len(t5s) > 0

    # pT3 / pT5: every pLS with every T3 / T5
    if ev.n_pls:
        pt3, pt5 = [], []
        for ip in range(ev.n_pls):
            pls = [ev.pls[k][ip] for k in ("pt", "q", "x0", "y0", "z0", "x1", "y1", "z1")]
            for (A, B, Cc), k3 in t3s.items():
                t = O.pt_test(pls, mds[A][1], bool(geom.subdet[mds[A][0]]), mds[Cc][1],
                              bool(geom.subdet[mds[Cc][0]]), [k3], 0.0, p)
                n_cand[4] += 1
                n_near[4] += int(t[1])
                if t[0]:
                    pt3.append((ip,) + A + B + Cc)
            for (A, B, Cc, D, E), sc in t5s.items():
                kt = [t3s[(A, B, Cc)], t3s[(Cc, D, E)]]
                t = O.pt_test(pls, mds[A][1], bool(geom.subdet[mds[A][0]]), mds[E][1],
                              bool(geom.subdet[mds[E][0]]), kt, sc, p)
                n_cand[5] += 1
                n_near[5] += int(t[1])
                if t[0]:
                    pt5.append((ip,) + A + B + Cc + D + E)
        assert sorted(pt3) == [tuple(t) for t in c["pt3"]]
        assert sorted(pt5) == [tuple(t) for t in c["pt5"]]
        assert len(pt3) > 0 and len(pt5) > 0
    # every candidate is counted once, accepted or not, and in no other stage's counter
    assert min(n_cand[:4]) > 0 and (not ev.n_pls or min(n_cand[4:]) > 0)
    assert [int(v) for v in res["n_tests"][:6]] == n_cand, "candidates per stage"
    assert [int(v) for v in res["near"][:6]] == n_near, "near-threshold candidates per stage"
    assert int(res["n_tests"][6]) == 0 and int(res["near"][6]) == 0  # T4 is off in the default stage mask


# ------------------------------------------------------------------------------------------------
# structural invariants and physics sanity
# ------------------------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def c4_result(oracle_mod):
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    res = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls)
    return geom, off, tgt, ev, res


def test_structure_invariants(c4_result):
    geom, off, tgt, ev, r = c4_result
    md_mod = r["md_module"]
    # MD: lower hit on sensor 2m, upper on 2m+1 of the MD's module
    assert np.array_equal(ev.sensor[r["md_hits"][:, 0]], 2 * md_mod)
    assert np.array_equal(ev.sensor[r["md_hits"][:, 1]], 2 * md_mod + 1)
    # LS: (module(A), module(B)) is an edge of the connection map
    edges = {(m, int(t)) for m in range(geom.n_modules) for t in tgt[off[m]:off[m + 1]]}
    for a, b in r["ls_md"]:
        assert (int(md_mod[a]), int(md_mod[b])) in edges
    # T3: its two LSs share the middle MD; MDs = (in(ls0), out(ls0) = in(ls1), out(ls1))
    l0, l1 = r["ls_md"][r["t3_ls"][:, 0]], r["ls_md"][r["t3_ls"][:, 1]]
    assert np.array_equal(l0[:, 1], l1[:, 0])
    assert np.array_equal(r["t3_md"], np.stack([l0[:, 0], l0[:, 1], l1[:, 1]], 1))
    # T5 shares its MDs with its two T3s (north_star invariant); 5 distinct MDs
    a, b = r["t3_md"][r["t5_t3"][:, 0]], r["t3_md"][r["t5_t3"][:, 1]]
    assert np.array_equal(a[:, 2], b[:, 0])
    assert np.array_equal(r["t5_md"], np.concatenate([a, b[:, 1:]], axis=1))
    assert all(len(set(row)) == 5 for row in r["t5_md"].tolist())
    # pT3 / pT5 reference existing objects
    assert r["pt3"][:, 0].max() < ev.n_pls and r["pt3"][:, 1].max() < len(r["t3_md"])
    assert r["pt5"][:, 0].max() < ev.n_pls and r["pt5"][:, 1].max() < len(r["t5_md"])
    assert len(r["pt3"]) > 100 and len(r["pt5"]) > 100


def test_track_candidates_consistent(c4_result):
    """classes pT5, pT3, T5, unlinked pLS in this order; survivors of a class do not
    overlap (CUTS.md section 8 consequence); every pLS is either linked or output as unlinked."""
    geom, off, tgt, ev, r = c4_result
    tc = r["tc"]
    assert np.all(np.diff(tc[:, 0]) >= 0)
    assert set(np.unique(tc[:, 0])) == {0, 1, 2, 3}
    t5 = tc[tc[:, 0] == 2]
    sets = [set(map(tuple, row[4:14].reshape(5, 2).tolist())) for row in t5]
    for i in range(len(sets)):
        for j in range(i + 1, len(sets)):
            assert len(sets[i] & sets[j]) < 3
    p5 = tc[tc[:, 0] == 0]
    assert len(set(p5[:, 1].tolist())) == len(p5)  # one pT5 per seed
    sets = [set(map(tuple, row[4:14].reshape(5, 2).tolist())) for row in p5]
    for i in range(len(sets)):
        for j in range(i + 1, len(sets)):
            assert len(sets[i] & sets[j]) < 3
    linked = set(tc[tc[:, 0] <= 1][:, 1].tolist())
    unlinked = set(tc[tc[:, 0] == 3][:, 1].tolist())
    assert linked.isdisjoint(unlinked) and linked | unlinked == set(range(ev.n_pls))
    # hit_idx of a T5 candidate are the hits of the referenced T5
    row = t5[0]
    assert np.array_equal(row[4:14].reshape(5, 2), r["md_hits"][r["t5_md"][row[2]]])
    assert np.all(row[14:16] == -1)


def test_c1_no_noise_objects_are_single_track(oracle_mod):
    """C1 has no noise: every T5 is built from the hits of ONE generated helix, and a helix with MDs
    on 5+ consecutive layers yields T5s."""
    geom, off, tgt = make_config_geometry("C1")
    ev = make_config_event("C1")
    r = oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor,
                             params=oracle_mod.default_params(stage_mask=0x0f))
    assert len(r["tc"]) == 0
    t5_hits = r["md_hits"][r["t5_md"]].reshape(len(r["t5_md"]), 10)
    truth = ev.truth[t5_hits]
    assert len(t5_hits) >= 15
    assert np.all(truth == truth[:, :1])
    assert len(np.unique(truth[:, 0])) >= 10  # most of the 20 tracks are found


@pytest.mark.parametrize("field,factor", [("md_b_phi_tol", 1.5), ("ls_dir_tol", 1.5), ("ls_z_tol", 1.5),
                                          ("t3_z_tol0", 2.0), ("t5_tol0", 3.0), ("pt_k_tol0", 3.0),
                                          ("z0_max", 1.3), ("ls_kappa_max", 1.2)])
def test_monotone_in_cut_windows(oracle_mod, field, factor):
    """Widening any window can only add objects (north_star: counts monotone in the cut windows)."""
    geom, off, tgt = make_config_geometry("C4")
    ev = make_config_event("C4")
    base = oracle_mod.default_params(stage_mask=0x1f)
    wide = oracle_mod.default_params(stage_mask=0x1f)
    setattr(wide, field, getattr(base, field) * factor)
    a = canon(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, base))
    b = canon(oracle_mod.run_event(geom.subdet, off, tgt, ev.x, ev.y, ev.z, ev.sensor, ev.pls, wide))
    grew = False
    for kind in ("md", "ls", "t3", "t5", "pt3", "pt5"):
        sa, sb = set(map(tuple, a[kind].tolist())), set(map(tuple, b[kind].tolist()))
        assert sa <= sb, kind
        grew |= len(sb) > len(sa)
    assert grew


def test_invalid_input_rejected(oracle_mod):
    geom, off, tgt = make_config_geometry("C1")
    with pytest.raises(ValueError):
        oracle_mod.run_event(geom.subdet, off, tgt, [1.0], [2.0], [3.0], [2 * geom.n_modules])
    with pytest.raises(ValueError):
        oracle_mod.run_event(geom.subdet, off, tgt, [1.0], [2.0], [3.0], [-1])


def test_empty_event(oracle_mod):
    geom, off, tgt = make_config_geometry("C1")
    e = np.zeros(0, dtype=np.float32)
    r = oracle_mod.run_event(geom.subdet, off, tgt, e, e, e, np.zeros(0, dtype=np.int32))
    assert all(len(r[k]) == 0 for k in ("md_hits", "ls_md", "t3_md", "t5_md", "pt3", "pt5", "tc"))
    assert r["n_tests"].sum() == 0
