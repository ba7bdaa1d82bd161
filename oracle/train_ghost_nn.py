"""Writes lhcb_gen/ghost_nn_weights.txt: the 339 packed values of the ghost-killing network (PAPER.md
L344-348: 8 inputs, one hidden layer of 32 nodes, output = ghost probability; reading A14b).

The paper's trained weights are not available (they were fitted on LHCb simulation), so this script fits
the same architecture on generator truth:  python -m oracle.train_ghost_nn
It calls only lhcb_gen (inputs, truth) and oracle/ (candidates and features), never the CUDA path.
Label of a candidate (seed, VELO): ghost = the seed's particle differs from the VELO track's particle.
"""
import os

import numpy as np

from lhcb_gen import config, generate, truth
from oracle.binding import Oracle

OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "lhcb_gen", "ghost_nn_weights.txt")
N_IN, N_HID = 8, 32


def pack(mu, isig, W1, b1, W2, b2, cut=0.8, margin=0.05):
    return np.concatenate([mu, isig, W1.reshape(-1), b1, W2, [b2, cut, margin]]).astype(np.float32)


def candidates(n_events=400, cfg=2):
    """All chi2- and UT-accepted candidates of the oracle (network switched off: cut = margin = +inf)."""
    ev = generate(config(cfg, n_events))
    o = Oracle(ev.geom, "f32")
    s = o.seeding(ev)
    seed_off = np.zeros(ev.n_events + 1, np.uint32)
    np.cumsum(np.bincount(s["event"], minlength=ev.n_events), out=seed_off[1:])
    open_nn = pack(np.zeros(8), np.ones(8), np.zeros((32, 8)), np.zeros(32), np.zeros(32), 0.0, np.inf, np.inf)
    nhits = (s["nx"] + s["nuv"]).astype(np.uint8)
    m = o.matching(ev.n_events, seed_off, s["state"], ev, use_ut=True, nn=open_nn, nhits=nhits)
    spid, _ = truth.seed_pids(ev, s["hits"])
    X = np.zeros((m["n"], N_IN), np.float64)
    for i, (sd, v) in enumerate(zip(m["seed"], m["velo"])):
        r = o.match_pair(s["state"][sd, :4], [ev.velo_x[v], ev.velo_y[v], ev.velo_tx[v], ev.velo_ty[v]])
        X[i] = [r["zm"], r["dx"], r["dy"], r["dtx"], r["dty"], r["chi2"], o.eta_velo(ev.velo_tx[v], ev.velo_ty[v]), nhits[sd]]
    ghost = ~((spid[m["seed"]] >= 0) & (spid[m["seed"]] == ev.velo_pid[m["velo"]]))
    return X, ghost.astype(np.float64)


def train(X, y, epochs=600, seed=0):
    rng = np.random.default_rng(seed)
    mu, sig = X.mean(0), X.std(0) + 1e-9
    U = (X - mu) / sig
    W1 = rng.normal(0, 0.3, (N_HID, N_IN)); b1 = np.zeros(N_HID); W2 = rng.normal(0, 0.3, N_HID); b2 = 0.0
    w_pos = (1 - y.mean()) / max(y.mean(), 1e-6)                 # ghosts are rare: balance the classes
    wt = np.where(y > 0.5, w_pos, 1.0); wt /= wt.sum()
    params = [W1, b1, W2, np.array([b2])]
    m = [np.zeros_like(p) for p in params]; v = [np.zeros_like(p) for p in params]
    for t in range(1, epochs + 1):
        H = np.maximum(U @ params[0].T + params[1], 0)
        p = 1 / (1 + np.exp(-(H @ params[2] + params[3][0])))
        d = (p - y) * wt                                          # d loss / d logit (weighted cross entropy)
        gW2 = H.T @ d; gb2 = np.array([d.sum()])
        dH = np.outer(d, params[2]) * (H > 0)
        grads = [dH.T @ U, dH.sum(0), gW2, gb2]
        for k in range(4):                                        # Adam
            m[k] = 0.9 * m[k] + 0.1 * grads[k]; v[k] = 0.999 * v[k] + 0.001 * grads[k] ** 2
            params[k] -= 0.02 * (m[k] / (1 - 0.9 ** t)) / (np.sqrt(v[k] / (1 - 0.999 ** t)) + 1e-8)
    return pack(mu, 1 / sig, params[0], params[1], params[2], params[3][0]), p


def main():
    X, y = candidates()
    w, p = train(X, y)
    print(f"{len(y)} candidates, {int(y.sum())} ghosts; ghost prob: mean on true {p[y < .5].mean():.3f}, on ghosts {p[y > .5].mean():.3f}; "
          f"true kept at 0.8: {(p[y < .5] < 0.8).mean():.4f}, ghosts rejected: {(p[y > .5] >= 0.8).mean():.4f}")
    with open(OUT, "w") as f:
        f.write("# ghost-killing network 8 -> 32 -> 1 (PAPER.md L344-348), packed as mu[8], isig[8], W1[32][8], b1[32], W2[32],\n"
                "# b2, cut, margin; fitted on generator truth by oracle/train_ghost_nn.py (the paper's weights are unavailable)\n")
        f.write("\n".join(repr(float(x)) for x in w) + "\n")


if __name__ == "__main__":
    main()
