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
