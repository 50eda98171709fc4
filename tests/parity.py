"""Comparison rules between the CUDA path and the CPU oracle (BASELINE north_star; readings A-16 / A-17 in DESIGN.md).

Imports neither the CUDA package nor oracle/: it only looks at two dicts of numpy arrays.

  * integers (found, nhits, the four hit indices, keep; vertex (evt, ia, ib, flags) lists) must be identical, except
    for seeds / pairs the oracle put on its edge list (a deciding comparison within 1e-5 relative of its bound);
    those are counted and must stay below 0.01 % of the seeds / pairs;
  * floats: |gpu - oracle| <= 1e-4 * max(|oracle|, floor) with the per-quantity floors of A-17.
"""
import math

import numpy as np

REL = 1e-4
TRACK_FLOORS = dict(x=1.0, y=1.0, tx=1e-2, ty=1e-2, qop=1e-2, chi2=1.0, score=1e-3)
VTX_FLOORS = dict(x=1.0, y=1.0, z=0.0, doca=0.1, m_pipi=0.0, m_ppi=0.0)
MAX_EDGE_FRACTION = 1e-4


def close(g, o, floor):
    g, o = np.asarray(g, dtype=np.float64), np.asarray(o, dtype=np.float64)
    return np.abs(g - o) <= REL * np.maximum(np.abs(o), floor)


def compare_tracks(gpu: dict, orc: dict) -> dict:
    """gpu: host copies of the ds_tracks arrays; orc: oracle.reconstruct output.  Raises AssertionError on a mismatch
    that the edge list does not excuse.  Returns counts."""
    n = len(orc["found"])
    assert all(len(gpu[k]) == n for k in ("found", "nhits", "keep", "x"))
    hit_g = np.asarray(gpu["hit"]).reshape(n, 4)
    int_bad = ((np.asarray(gpu["found"]) != orc["found"]) | (np.asarray(gpu["nhits"]) != orc["nhits"])
               | (np.asarray(gpu["keep"]) != orc["keep"]) | (hit_g != orc["hit"]).any(axis=1))
    edge = orc["edge"].astype(bool)
    unexcused = np.nonzero(int_bad & ~edge)[0]
    assert unexcused.size == 0, f"{unexcused.size} seeds differ off the edge list, first {unexcused[:5]}"
    excused = int(np.count_nonzero(int_bad & edge))
    assert excused <= math.ceil(MAX_EDGE_FRACTION * n), f"{excused} excused mismatches of {n} seeds"
    same = ~int_bad & (orc["found"] == 1)
    for k, floor in TRACK_FLOORS.items():
        ok = close(np.asarray(gpu[k])[same], orc[k][same], floor)
        assert ok.all(), f"track {k}: {np.count_nonzero(~ok)} of {ok.size} outside 1e-4, first at {np.nonzero(same)[0][~ok][:3]}"
    # not-found slots hold zeros / -1
    nf = np.asarray(gpu["found"]) == 0
    for k in TRACK_FLOORS:
        assert not np.asarray(gpu[k])[nf].any(), k
    assert (hit_g[nf] == -1).all() and not np.asarray(gpu["keep"])[nf].any() and not np.asarray(gpu["nhits"])[nf].any()
    return dict(n=n, found=int(orc["found"].sum()), edge_list=int(edge.sum()), excused=excused)


def compare_vertices(gpu: dict, orc: dict) -> dict:
    """gpu: host copies of the ds_vertices arrays (first n entries valid) + 'n'; orc: oracle.vertex output computed on
    the SAME track arrays."""
    key_g = list(zip(np.asarray(gpu["evt"]).tolist(), np.asarray(gpu["ia"]).tolist(), np.asarray(gpu["ib"]).tolist()))
    key_o = list(zip(orc["evt"].tolist(), orc["ia"].tolist(), orc["ib"].tolist()))
    sg, so = set(key_g), set(key_o)
    assert len(sg) == len(key_g), "duplicate vertices"
    diff = sg ^ so
    unexcused = [k for k in diff if k not in orc["edge_pairs"]]
    assert not unexcused, f"{len(unexcused)} pairs differ off the edge list, first {sorted(unexcused)[:5]}"
    assert len(diff) <= math.ceil(MAX_EDGE_FRACTION * orc["n_pairs"])
    # order: (evt, ia, ib) ascending
    kk = np.asarray(gpu["evt"]).astype(np.int64) * (1 << 42) + np.asarray(gpu["ia"]).astype(np.int64) * (1 << 21) + np.asarray(gpu["ib"])
    assert (np.diff(kk) > 0).all(), "vertex list not sorted by (evt, ia, ib)"
    if not diff:
        assert key_g == key_o
        ig = io = np.arange(len(key_g))
    else:
        pos_o = {k: i for i, k in enumerate(key_o)}
        common = [(i, pos_o[k]) for i, k in enumerate(key_g) if k in pos_o]
        ig, io = np.array([c[0] for c in common], dtype=np.int64), np.array([c[1] for c in common], dtype=np.int64)
    fl_bad = np.asarray(gpu["flags"])[ig] != orc["flags"][io]
    bad_keys = [key_g[i] for i in ig[fl_bad]]
    assert all(k in orc["edge_pairs"] for k in bad_keys), "flags differ off the edge list"
    for k, floor in VTX_FLOORS.items():
        ok = close(np.asarray(gpu[k])[ig], orc[k][io], floor)
        assert ok.all(), f"vertex {k}: {np.count_nonzero(~ok)} of {ok.size} outside 1e-4"
    return dict(n=len(key_o), n_pairs=orc["n_pairs"], edge_list=len(orc["edge_pairs"]), excused=len(diff) + len(bad_keys))
