"""The packed ghost-killing network (reading A14b): an input of the matching,
like the geometry.  339 float32: mu[8], isig[8], W1[32][8], b1[32], W2[32], b2, cut, margin.
`ghost_nn_weights.txt` is written by oracle/train_ghost_nn.py (fitted on generator truth)."""
import os

import numpy as np

NN_SIZE = 339
_PATH = os.path.join(os.path.dirname(os.path.abspath(__file__)), "ghost_nn_weights.txt")


def ghost_nn() -> np.ndarray:
    w = np.loadtxt(_PATH, dtype=np.float64).astype(np.float32)
    assert w.size == NN_SIZE
    return w


def unpack(w):
    w = np.asarray(w)
    return dict(mu=w[0:8], isig=w[8:16], W1=w[16:272].reshape(32, 8), b1=w[272:304], W2=w[304:336], b2=w[336],
                cut=w[337], margin=w[338])
