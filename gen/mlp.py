"""Ghost-killer MLP weights for the synthetic workload (BASELINE cfg0: 8->32->16->1, weights ~ N(0, 1/fan_in)).

Reading A-18: the second argument of N is the variance; biases are drawn the same way; matrices are
row-major [out][in]; draw order W1, b1, W2, b2, W3, b3 from numpy.random.default_rng(seed) in fp64, then fp32.
The trained weights of the paper (P:133-P:143) are not published.
"""
import numpy as np

from . import constants as C


def mlp_weights(seed: int, sizes=C.MLP_SIZES):
    rng = np.random.default_rng(seed)
    out = {}
    for li in range(len(sizes) - 1):
        fan_in, fan_out = sizes[li], sizes[li + 1]
        sd = fan_in ** -0.5
        out[f"W{li + 1}"] = rng.normal(0.0, sd, (fan_out, fan_in)).astype(np.float32)
        out[f"b{li + 1}"] = rng.normal(0.0, sd, fan_out).astype(np.float32)
    out["mu"] = np.asarray(C.MLP_MU, dtype=np.float32)
    out["inv_sigma"] = (1.0 / np.asarray(C.MLP_SIGMA, dtype=np.float64)).astype(np.float32)
    return out


# HLT1 line NNs (P:277-P:285): four networks 16 -> 32 -> 1; inputs and their normalisation: reading A-33
LINE_SIZES = (16, 32, 1)
LINE_MU = (0.0, 0.0, 0.0, 3.0, 0.0, 0.0, 0.0, 3.0, 0.0, 0.0, 1500.0, 1.0, 0.0, 0.0, 10.0, 1.0)
LINE_SIGMA = (0.2, 0.1, 0.25, 3.0, 0.2, 0.1, 0.25, 3.0, 300.0, 200.0, 500.0, 1.0, 0.2, 0.1, 10.0, 1.0)


def line_weights(seed: int):
    """Four independent weight sets {W1 [32][16], b1 [32], W3 [32], b3 [1]} ~ N(0, 1/fan_in) (A-18) plus the common
    input normalisation; the trained weights of the paper are not published."""
    rng = np.random.default_rng(seed)
    nets = []
    for _ in range(4):
        n_in, n_h, _o = LINE_SIZES
        nets.append(dict(W1=rng.normal(0.0, n_in ** -0.5, (n_h, n_in)).astype(np.float32),
                         b1=rng.normal(0.0, n_in ** -0.5, n_h).astype(np.float32),
                         W3=rng.normal(0.0, n_h ** -0.5, n_h).astype(np.float32),
                         b3=rng.normal(0.0, n_h ** -0.5, 1).astype(np.float32)))
    mu = np.asarray(LINE_MU, dtype=np.float32)
    inv_sigma = (1.0 / np.asarray(LINE_SIGMA, dtype=np.float64)).astype(np.float32)
    return dict(nets=nets, mu=mu, inv_sigma=inv_sigma)


def embed_single_hidden(w1: dict, sizes=C.MLP_SIZES) -> dict:
    """The paper's ghost killer has ONE hidden layer (8 -> 14 -> 1); the library's network is 8 -> 32 -> 16 -> 1
    (BASELINE cfg0).  A single-hidden-layer network with n_h <= 16 units runs on it unchanged: its hidden units become
    the first n_h units of layer 1 (the others get zero weights), layer 2 copies them through (ReLU of a non-negative
    number is the number itself) and W3 is padded with zeros.  w1 = {W1 [n_h][8], b1 [n_h], W3 [n_h], b3 [1], mu, inv_sigma}."""
    n_in, h1, h2, _ = sizes
    n_h = w1["W1"].shape[0]
    assert n_h <= h2 and w1["W1"].shape[1] == n_in
    out = dict(W1=np.zeros((h1, n_in), np.float32), b1=np.zeros(h1, np.float32), W2=np.zeros((h2, h1), np.float32),
               b2=np.zeros(h2, np.float32), W3=np.zeros(h2, np.float32), b3=np.asarray(w1["b3"], np.float32).reshape(1),
               mu=w1["mu"], inv_sigma=w1["inv_sigma"])
    out["W1"][:n_h] = w1["W1"]
    out["b1"][:n_h] = w1["b1"]
    out["W2"][np.arange(n_h), np.arange(n_h)] = 1.0
    out["W3"][:n_h] = np.asarray(w1["W3"]).reshape(-1)
    return out


def mlp_single_weights(seed: int = 0, n_h: int = 14) -> dict:
    """Random weights of the paper's single-hidden-layer ghost killer 8 -> 14 -> 1, drawn like mlp_weights (A-18):
    N(0, 1/fan_in), order W1, b1, W3, b3, fp64 -> fp32; the input normalisation of A-10."""
    rng = np.random.default_rng(seed + 1000)
    n_in = C.MLP_SIZES[0]
    return dict(W1=rng.normal(0.0, n_in ** -0.5, (n_h, n_in)).astype(np.float32), b1=rng.normal(0.0, n_in ** -0.5, n_h).astype(np.float32),
                W3=rng.normal(0.0, n_h ** -0.5, n_h).astype(np.float32), b3=rng.normal(0.0, n_h ** -0.5, 1).astype(np.float32),
                mu=np.asarray(C.MLP_MU, dtype=np.float32), inv_sigma=(1.0 / np.asarray(C.MLP_SIGMA, dtype=np.float64)).astype(np.float32))
