"""Fits the 65 weights of the learned T5 selection (CUTS.md section 11; "machine learning methods",
PAPER.md:102) on synthetic truth and writes them to lst_inputs/t5_mlp.py.

The weights are INPUTS of the method (part of the parameter record), so they are made here, next to the other
input generators, from the generator's own truth: it calls neither the oracle nor the CUDA path.
  * positives: five lower-sensor hits of ONE generated track on five consecutive barrel layers;
  * negatives: such a tuple with its last two (or first two) hits replaced by those of another track that is
    close in azimuth on the same layers -- the combinatorial background a T5 candidate (two T3s sharing
    their middle MD) is made of.
Features (CUTS.md section 11): S (|ki|, |kb|, |ko|, |ki - kb|, |kb - ko|, |ki - ko|), S = T5_MLP_SCALE = 100,
with ki, kb, ko the circumcircle curvatures of the hit triplets (A,B,C), (B,C,D), (C,D,E).
Model: 6-8-1, rectifier units; logistic loss, Adam, fixed seed.  The stored form is the spec's
"accept iff s <= T5_MLP_THR = 1": s = 1 - logit, i.e. W2 and b2 are stored negated and shifted.

Run:  python -m lst_inputs.train_t5_mlp
"""
from __future__ import annotations

import os

import numpy as np

from .configs import make_config_geometry, spec_of
from .events import generate_event

SCALE = 100.0
HERE = os.path.dirname(os.path.abspath(__file__))


def kappa3(P, Q, S):
    a, b, c = Q - P, S - Q, S - P
    crs = a[:, 0] * c[:, 1] - a[:, 1] * c[:, 0]
    return 2.0 * crs / (np.hypot(*a.T) * np.hypot(*b.T) * np.hypot(*c.T))


def features(pts):
    """pts [n, 5, 2] -> [n, 6]"""
    ki, kb, ko = kappa3(pts[:, 0], pts[:, 1], pts[:, 2]), kappa3(pts[:, 1], pts[:, 2], pts[:, 3]), kappa3(pts[:, 2], pts[:, 3], pts[:, 4])
    return SCALE * np.abs(np.stack([ki, kb, ko, ki - kb, kb - ko, ki - ko], axis=1))


def tuples_of_event(geom, ev, rng):
    m = ev.sensor // 2
    low = (ev.sensor % 2 == 0) & (geom.subdet[m] == 0) & (ev.truth >= 0)
    layer = geom.layer[m]
    xy = np.stack([ev.x, ev.y], axis=1).astype(np.float64)
    per_track = {}
    for i in np.nonzero(low)[0]:
        per_track.setdefault(int(ev.truth[i]), {}).setdefault(int(layer[i]), i)
    pos, neg = [], []
    tracks = {t: lay for t, lay in per_track.items() if len(lay) >= 5}
    tids = np.array(sorted(tracks))
    if tids.size < 2:
        return np.zeros((0, 5, 2)), np.zeros((0, 5, 2))
    phi = np.array([np.arctan2(*xy[next(iter(tracks[t].values()))][::-1]) for t in tids])
    for k, t in enumerate(tids):
        lay = tracks[t]
        for l0 in (1, 2):
            if not all(l in lay for l in range(l0, l0 + 5)):
                continue
            tup = np.array([xy[lay[l]] for l in range(l0, l0 + 5)])
            pos.append(tup)
            d = np.abs(np.angle(np.exp(1j * (phi - phi[k]))))
            near = np.nonzero((d < 0.15) & (tids != t))[0]
            for o in rng.permutation(near)[:3]:
                lo = tracks[tids[o]]
                if all(l in lo for l in (l0 + 3, l0 + 4)):
                    f = tup.copy()
                    f[3], f[4] = xy[lo[l0 + 3]], xy[lo[l0 + 4]]
                    neg.append(f)
                if all(l in lo for l in (l0, l0 + 1)):
                    f = tup.copy()
                    f[0], f[1] = xy[lo[l0]], xy[lo[l0 + 1]]
                    neg.append(f)
    return np.array(pos).reshape(-1, 5, 2), np.array(neg).reshape(-1, 5, 2)


def fit(X, y, seed=0, epochs=400, lr=0.01):
    rng = np.random.default_rng(seed)
    W1, b1 = rng.normal(0, 0.5, (8, 6)), np.zeros(8)
    W2, b2 = rng.normal(0, 0.5, 8), 0.0
    params = [W1, b1, W2, np.array([b2])]
    m = [np.zeros_like(p) for p in params]
    v = [np.zeros_like(p) for p in params]
    w_pos = (y == 0).sum() / max((y == 1).sum(), 1)
    for step in range(1, epochs + 1):
        A = X @ params[0].T + params[1]
        H = np.maximum(A, 0.0)
        z = H @ params[2] + params[3][0]
        p = 1.0 / (1.0 + np.exp(-np.clip(z, -30, 30)))
        g = (p - y) * np.where(y == 1, w_pos, 1.0) / len(y)
        gW2, gb2 = H.T @ g, g.sum()
        gH = np.outer(g, params[2]) * (A > 0)
        grads = [gH.T @ X, gH.sum(0), gW2, np.array([gb2])]
        for i in range(4):
            m[i] = 0.9 * m[i] + 0.1 * grads[i]
            v[i] = 0.999 * v[i] + 0.001 * grads[i] ** 2
            params[i] = params[i] - lr * (m[i] / (1 - 0.9 ** step)) / (np.sqrt(v[i] / (1 - 0.999 ** step)) + 1e-8)
    return params


def main():
    rng = np.random.default_rng(2407)
    geom, _, _ = make_config_geometry("C2")
    P, N = [], []
    for seed in range(40):
        ev = generate_event(geom, spec_of("C2"), 9000 + seed)
        p, n = tuples_of_event(geom, ev, rng)
        P.append(p)
        N.append(n)
    P, N = np.concatenate(P), np.concatenate(N)
    X = np.concatenate([features(P), features(N)])
    y = np.concatenate([np.ones(len(P)), np.zeros(len(N))])
    W1, b1, W2, b2 = fit(X, y)
    z = np.maximum(X @ W1.T + b1, 0.0) @ W2 + b2[0]
    acc_pos, acc_neg = float((z[y == 1] >= 0).mean()), float((z[y == 0] < 0).mean())
    # stored form: accept iff s = 1 - z <= 1
    w = np.concatenate([W1.ravel(), b1, -W2, [1.0 - b2[0]]]).astype(np.float32)
    with open(os.path.join(HERE, "t5_mlp.py"), "w") as f:
        f.write('"""Weights of the learned T5 selection (CUTS.md section 11), written by lst_inputs/train_t5_mlp.py.\n')
        f.write("Fitted on %d true and %d combinatorial five-hit tuples of 40 C2-like events (seeds 9000..9039);\n" % (len(P), len(N)))
        f.write("on that sample %.1f %% of the true tuples are accepted and %.1f %% of the combinatorial ones rejected.\n" % (100 * acc_pos, 100 * acc_neg))
        f.write('Layout: W1[8][6] row-major, b1[8], W2[8], b2; accept iff s <= T5_MLP_THR = 1 with T5_MLP_SCALE = 100."""\n')
        f.write("T5_MLP_SCALE = 100.0\nT5_MLP_THR = 1.0\nT5_MLP = (\n")
        for i in range(0, 65, 5):
            f.write("    " + " ".join("%.9g," % float(x) for x in w[i:i + 5]) + "\n")
        f.write(")\n")
    print("positives", len(P), "negatives", len(N), "accepted true %.3f rejected fake %.3f" % (acc_pos, acc_neg))


if __name__ == "__main__":
    main()
