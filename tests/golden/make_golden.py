"""Writes the hand-computable single-track fixtures of tests/golden/ from closed forms.

Calls neither the oracle nor the CUDA path: the coordinates are points of a straight line or of a
circle through the origin (x = R sin t, y = R (1 - cos t), r = 2 R sin(t/2)), and the expected
values (object counts of a 6-layer / 5-disk single track, curvature 1/R) follow by hand from
PAPER.md:23, 29 and CUTS.md sections 3-6.  Cited by north_star: "hand-computed straight and curved
single tracks".  Run:  python tests/golden/make_golden.py
"""
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LAYERS = [23.0, 36.0, 51.0, 68.0, 88.0, 108.0]
GAP = 0.26
DISKS = [130.0, 160.0, 190.0, 225.0, 265.0]
DGAP = 0.4


def write(name, header, hits, expect):
    with open(os.path.join(HERE, name), "w") as f:
        for line in header:
            f.write("# " + line + "\n")
        f.write("# columns: x y z sensor   (sensor = 2*module + {0 lower, 1 upper})\n")
        for x, y, z, s in hits:
            f.write(f"{np.float32(x):.9g} {np.float32(y):.9g} {np.float32(z):.9g} {int(s)}\n")
        f.write("expect " + " ".join(f"{k}={v}" for k, v in expect.items()) + "\n")


def circle_hits(R, z0, cot):
    hits = []
    for k, rl in enumerate(LAYERS):
        for s in (0, 1):
            r = rl + s * GAP
            if r >= 2 * R:
                continue
            t = 2.0 * np.arcsin(r / (2.0 * R))
            hits.append((R * np.sin(t), R * (1.0 - np.cos(t)), z0 + cot * R * t, 2 * k + s))
    return hits


# 1. straight track along +x through the origin, z = 0.5 * r: every cut value is 0
hits = []
for k, rl in enumerate(LAYERS):
    for s in (0, 1):
        r = rl + s * GAP
        hits.append((r, 0.0, 0.5 * r, 2 * k + s))
write("straight_barrel.txt",
      ["straight track y = 0, z = 0.5 r from the origin; 6 barrel modules chained k -> k+1",
       "by hand: 6 MDs, 5 LSs, 4 T3s, 2 T5s (layers 1-5 and 2-6); all curvatures 0"],
      hits, {"n_md": 6, "n_ls": 5, "n_t3": 4, "n_t5": 2, "kappa": 0.0, "modules": "barrel"})

# 2. circle of radius 100 cm through the origin, counter-clockwise (kappa = +0.01), z0 = 2, cot = 0.5
write("circle_R100_barrel.txt",
      ["circle R = 100 cm through the origin, centre (0, 100), counter-clockwise: kappa = +1/R = +0.01",
       "x = R sin t, y = R (1 - cos t), t = 2 asin(r / 2R), z = 2 + 0.5 R t",
       "R = 100 cm > R_MIN = 0.8 * 100/(0.3*3.8) = 70.18 cm: by hand 6 MDs, 5 LSs, 4 T3s, 2 T5s"],
      circle_hits(100.0, 2.0, 0.5),
      {"n_md": 6, "n_ls": 5, "n_t3": 4, "n_t5": 2, "kappa": 0.01, "modules": "barrel"})

# 3. circle of radius 50 cm (pT = 0.57 GeV < 0.8): sin(radial, tangent) = r/2R = 0.23 at layer 1
#    exceeds the window r/(2 R_MIN) + 0.06 = 0.2239 -> no MD at all (PAPER.md:23 pT threshold)
write("circle_R50_barrel.txt",
      ["circle R = 50 cm through the origin (pT = 0.57 GeV, below the 0.8 GeV threshold, PAPER.md:23)",
       "r/2R = 0.23, 0.36, 0.51, 0.68, 0.88 exceed r/(2*70.18) + 0.06 = 0.224, 0.316, 0.423, 0.545, 0.687",
       "by hand: no MD, hence no object"],
      circle_hits(50.0, 0.0, 0.3),
      {"n_md": 0, "n_ls": 0, "n_t3": 0, "n_t5": 0, "kappa": 0.02, "modules": "barrel"})

# 4. straight track through 5 endcap disks (+z), r = 0.3 z, azimuth 0.3 rad
hits = []
for k, zd in enumerate(DISKS):
    for s in (0, 1):
        z = zd + s * DGAP
        r = 0.3 * z
        hits.append((r * np.cos(0.3), r * np.sin(0.3), z, 2 * k + s))
write("straight_endcap.txt",
      ["straight track from the origin, r = 0.3 z, azimuth 0.3 rad; 5 endcap modules chained k -> k+1",
       "by hand: 5 MDs, 4 LSs, 3 T3s, 1 T5; all curvatures 0"],
      hits, {"n_md": 5, "n_ls": 4, "n_t3": 3, "n_t5": 1, "kappa": 0.0, "modules": "endcap"})
print("golden fixtures written to", HERE)
