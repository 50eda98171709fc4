"""ctypes wrapper of the fp64 CPU oracle (oracle/ds_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It never imports the CUDA package.  All inputs are promoted to float64 exactly before the C code sees them, so
un-rounded fp64 generator output can be fed as well (pin P-1).
"""
from __future__ import annotations

import ctypes as ct

import numpy as np

from . import build as _build

_lib = None

c_dp = ct.POINTER(ct.c_double)
c_ip = ct.POINTER(ct.c_int32)
c_lp = ct.POINTER(ct.c_int64)


class OrcGeom(ct.Structure):
    _fields_ = [("z_layer", ct.c_double * 4), ("dxdy", ct.c_double * 4), ("z_seed", ct.c_double),
                ("z_ref", ct.c_double), ("zmag_c", ct.c_double * 4), ("kick", ct.c_double)]


class OrcParams(ct.Structure):
    _fields_ = [("w0_a", ct.c_double), ("w0_b", ct.c_double), ("w0_max", ct.c_double), ("w1_a", ct.c_double),
                ("w1_b", ct.c_double), ("y_tol", ct.c_double), ("w_mag", ct.c_double),
                ("chi2ndf_max", ct.c_double), ("miss_penalty", ct.c_double), ("min_hits", ct.c_int32),
                ("max_first_hits", ct.c_int32), ("mlp_thr", ct.c_double), ("mlp_keep_above", ct.c_int32),
                ("pad_", ct.c_int32), ("doca_max", ct.c_double), ("zv_min", ct.c_double), ("zv_max", ct.c_double),
                ("m_pi", ct.c_double), ("m_p", ct.c_double), ("m_ks", ct.c_double), ("m_lambda", ct.c_double),
                ("dm_ks", ct.c_double), ("dm_lambda", ct.c_double), ("n2_min", ct.c_double),
                ("magnet_polarity", ct.c_double), ("gamma_c0", ct.c_double), ("gamma_c1", ct.c_double),
                ("vtx_newton_iters", ct.c_int32), ("dv1", ct.c_int32), ("edge_rel", ct.c_double)]


class OrcMlp(ct.Structure):
    _fields_ = [("n_in", ct.c_int32), ("n_h1", ct.c_int32), ("n_h2", ct.c_int32), ("pad_", ct.c_int32),
                ("W1", c_dp), ("b1", c_dp), ("W2", c_dp), ("b2", c_dp), ("W3", c_dp), ("b3", c_dp),
                ("mu", c_dp), ("inv_sigma", c_dp)]


def lib():
    global _lib
    if _lib is None:
        _lib = ct.CDLL(_build.build())
        _lib.orc_vertex.restype = ct.c_int64
        _lib.orc_mlp_eval.restype = ct.c_double
        _lib.orc_inv_mass.restype = ct.c_double
        _lib.orc_inv_mass.argtypes = [ct.c_double] * 8
        _lib.orc_poca.argtypes = [ct.c_double] * 10 + [c_dp]
        _lib.orc_poca_curved.argtypes = [ct.c_double] * 12 + [ct.c_int, c_dp]
        _lib.orc_gamma.restype = ct.c_double
        _lib.orc_gamma.argtypes = [ct.c_void_p, ct.c_double]
        _lib.orc_extrapolate.argtypes = [ct.c_void_p, ct.c_void_p] + [ct.c_double] * 5 + [c_dp]
        _lib.orc_fit_line.argtypes = [ct.c_int, c_dp, c_dp, c_dp, ct.c_double, c_dp, c_dp, c_dp]
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _p(a, t=c_dp):
    return a.ctypes.data_as(t)


def make_geom(g: dict) -> OrcGeom:
    o = OrcGeom()
    o.z_layer[:] = g["z_layer"]
    o.dxdy[:] = g["dxdy"]
    o.z_seed, o.z_ref, o.kick = g["z_seed"], g["z_ref"], g["kick"]
    o.zmag_c[:] = g["zmag_c"]
    return o


def make_params(p: dict, edge_rel: float = 1e-5) -> OrcParams:
    o = OrcParams()
    for name, _ in OrcParams._fields_:
        if name in p:
            setattr(o, name, p[name])
    o.edge_rel = edge_rel
    return o


class Mlp:
    """Holds fp64 copies of the (fp32) weights and the C struct pointing at them."""

    def __init__(self, w: dict):
        self.W1, self.b1 = _d(w["W1"]), _d(w["b1"])
        self.W3, self.b3 = _d(w["W3"]).reshape(-1), _d(w["b3"]).reshape(-1)
        self.mu, self.inv_sigma = _d(w["mu"]), _d(w["inv_sigma"])
        s = OrcMlp()
        s.n_in, s.n_h1 = self.W1.shape[1], self.W1.shape[0]
        if "W2" in w and w["W2"] is not None:
            self.W2, self.b2 = _d(w["W2"]), _d(w["b2"])
            s.n_h2 = self.W2.shape[0]
            s.W2, s.b2 = _p(self.W2), _p(self.b2)
        else:
            s.n_h2 = 0
        s.W1, s.b1, s.W3, s.b3, s.mu, s.inv_sigma = (_p(self.W1), _p(self.b1), _p(self.W3), _p(self.b3),
                                                       _p(self.mu), _p(self.inv_sigma))
        self.c = s

    def eval(self, v) -> float:
        v = _d(v)
        return lib().orc_mlp_eval(ct.byref(self.c), _p(v))


# ---- unit entry points (used by the pins) ------------------------------------------------------------------------
def extrapolate(geom: dict, params: dict, xs, ys, txs, tys, qop) -> dict:
    out = np.zeros(12)
    g, p = make_geom(geom), make_params(params)
    lib().orc_extrapolate(ct.byref(g), ct.byref(p), xs, ys, txs, tys, qop, _p(out))
    return dict(z_m=out[0], x_m=out[1], y_m=out[2], y_l=out[3:7].copy(), tx_pred=out[7], xc3=out[8], w0=out[9],
                w1=out[10])


def fit_line(z, x, w, z_ref):
    z, x, w = _d(z), _d(x), _d(w)
    a, b, c2 = ct.c_double(), ct.c_double(), ct.c_double()
    lib().orc_fit_line(len(z), _p(z), _p(x), _p(w), z_ref, ct.byref(a), ct.byref(b), ct.byref(c2))
    return a.value, b.value, c2.value


def poca(xa, ya, txa, tya, xb, yb, txb, tyb, z_ref, n2_min=1e-12):
    out = np.zeros(8)
    ok = lib().orc_poca(xa, ya, txa, tya, xb, yb, txb, tyb, z_ref, n2_min, _p(out))
    return bool(ok), dict(vertex=out[0:3].copy(), doca=out[3], n2=out[4], s_a=out[5], s_b=out[6])


def poca_curved(xa, ya, txa, tya, ga, xb, yb, txb, tyb, gb, z_ref, n_iter=3, n2_min=1e-12):
    """O-S9c: Newton-Raphson closest approach of two parabolic trajectories (Eq. 4)."""
    out = np.zeros(10)
    ok = lib().orc_poca_curved(xa, ya, txa, tya, ga, xb, yb, txb, tyb, gb, z_ref, n2_min, n_iter, _p(out))
    return bool(ok), dict(vertex=out[0:3].copy(), doca=out[3], n2=out[4], u=out[5], v=out[6], last_step=out[7],
                          tx_a=out[8], tx_b=out[9])


def gamma(params: dict, qop_gev: float) -> float:
    """Eq. 3 with q/p converted from 1/GeV to 1/MeV."""
    p = make_params(params)
    return lib().orc_gamma(ct.byref(p), qop_gev)


def inv_mass(tx1, ty1, p1, m1, tx2, ty2, p2, m2) -> float:
    return lib().orc_inv_mass(tx1, ty1, p1, m1, tx2, ty2, p2, m2)


def max_threads() -> int:
    return lib().orc_max_threads()


# ---- full path -------------------------------------------------------------------------------------------------------
def reconstruct(hits: dict, hit_offsets, seeds: dict, seed_offsets, geom: dict, params: dict, mlp: Mlp,
                edge_rel: float = 1e-5, n_threads: int = 0) -> dict:
    """O-S2..O-S7 for all events.  Returns per-seed arrays (track values as fp32, as the track SoA stores them)."""
    ho, so = _i(hit_offsets), _i(seed_offsets)
    ne = len(ho) - 1
    ns = int(so[-1])
    x0, z, ymin, ymax, w = (_d(hits[k]) for k in ("x0", "z", "ymin", "ymax", "w"))
    hid = _i(hits["id"])
    sx, sy, stx, sty, sq = (_d(seeds[k]) for k in ("x", "y", "tx", "ty", "qop"))
    schi = _d(seeds["chi2"]) if seeds.get("chi2") is not None else None
    trk = np.zeros((ns, 8))
    nhits, found, keep, edge = (np.zeros(ns, dtype=np.int32) for _ in range(4))
    hit_idx = np.full((ns, 4), -1, dtype=np.int32)
    margin = np.zeros(ns)
    g, p = make_geom(geom), make_params(params, edge_rel)
    lib().orc_reconstruct(ct.byref(g), ct.byref(p), ct.byref(mlp.c), ne, _p(ho, c_ip), _p(x0), _p(z), _p(ymin),
                          _p(ymax), _p(w), _p(hid, c_ip), _p(so, c_ip), _p(sx), _p(sy), _p(stx), _p(sty), _p(sq),
                          _p(schi) if schi is not None else None, _p(trk), _p(nhits, c_ip), _p(hit_idx, c_ip),
                          _p(found, c_ip), _p(keep, c_ip), _p(edge, c_ip), _p(margin), int(n_threads))
    out = {k: trk[:, i].astype(np.float32) for i, k in enumerate(("x", "y", "tx", "ty", "qop", "chi2", "score"))}
    out.update(nhits=nhits, hit=hit_idx, found=found, keep=keep, edge=edge, margin=margin,
               score_f64=trk[:, 6].copy())
    return out


def clone_kill(tracks: dict, seed_offsets, params: dict, min_shared: int = 3) -> np.ndarray:
    """O-S6b (N3): killed[s] = 1 for found tracks that share >= min_shared UT hits with a better track."""
    so = _i(seed_offsets)
    chi2 = _d(tracks["chi2"])
    nhits, hit, found = _i(tracks["nhits"]), _i(np.asarray(tracks["hit"]).reshape(-1)), _i(tracks["found"])
    killed = np.zeros(len(chi2), dtype=np.int32)
    p = make_params(params)
    lib().orc_clone_kill.restype = ct.c_int64
    n = lib().orc_clone_kill(ct.byref(p), int(min_shared), len(so) - 1, _p(so, c_ip), _p(chi2), _p(nhits, c_ip), _p(hit, c_ip),
                             _p(found, c_ip), _p(killed, c_ip))
    assert n == int(killed.sum())
    return killed


def line_features(txa, tya, qa, c2a, txb, tyb, qb, c2b, vtx4) -> np.ndarray:
    """The 16 inputs of the HLT1 line NNs for one vertex (reading A-33)."""
    v = np.zeros(16)
    vt = _d(vtx4)
    lib().orc_line_features.argtypes = [ct.c_double] * 8 + [c_dp, c_dp]
    lib().orc_line_features(txa, tya, qa, c2a, txb, tyb, qb, c2b, _p(vt), _p(v))
    return v


def lines(line_w: dict, tracks: dict, vtx: dict, thr: float = 0.5, edge_rel: float = 1e-5) -> dict:
    """O-L (N4, P:277-P:285): the four line NNs on every vertex of `vtx` (ia, ib, x, y, z, doca) -> scores [n][4], bits, edge."""
    nets = [Mlp(dict(w, mu=line_w["mu"], inv_sigma=line_w["inv_sigma"])) for w in line_w["nets"]]
    arr = (OrcMlp * 4)(*[m.c for m in nets])
    n = len(vtx["ia"])
    ia, ib = _i(vtx["ia"]), _i(vtx["ib"])
    v4 = _d(np.stack([vtx["x"], vtx["y"], vtx["z"], vtx["doca"]], axis=1)) if n else np.zeros((0, 4))
    tx, ty, qop, chi2 = (_d(tracks[k]) for k in ("tx", "ty", "qop", "chi2"))
    scores = np.zeros((n, 4))
    bits, edge = np.zeros(n, dtype=np.int32), np.zeros(n, dtype=np.int32)
    lib().orc_lines(arr, ct.c_double(thr), ct.c_double(edge_rel), ct.c_int64(n), _p(ia, c_ip), _p(ib, c_ip), _p(v4), _p(tx),
                    _p(ty), _p(qop), _p(chi2), _p(scores), _p(bits, c_ip), _p(edge, c_ip))
    return dict(scores=scores, bits=bits, edge=edge, _keep=nets)


def vertex(tracks: dict, seed_offsets, geom: dict, params: dict, edge_rel: float = 1e-5, n_threads: int = 0,
           capacity: int | None = None) -> dict:
    """O-S8/O-S9 for all events on the given per-seed track arrays (x, y, tx, ty, qop, keep)."""
    so = _i(seed_offsets)
    ne = len(so) - 1
    x, y, tx, ty, qop = (_d(tracks[k]) for k in ("x", "y", "tx", "ty", "qop"))
    keep = _i(tracks["keep"])
    g, p = make_geom(geom), make_params(params, edge_rel)
    npe = np.zeros(ne, dtype=np.int32)
    offs = np.zeros(ne + 1, dtype=np.int64)
    n_edge, n_pairs = ct.c_int64(), ct.c_int64()
    cap = 1 << 16 if capacity is None else capacity
    ecap = 1 << 16
    while True:
        v_evt, v_ia, v_ib, v_flags = (np.zeros(cap, dtype=np.int32) for _ in range(4))
        v = np.zeros((cap, 6))
        e_evt, e_ia, e_ib = (np.zeros(ecap, dtype=np.int32) for _ in range(3))
        total = lib().orc_vertex(ct.byref(g), ct.byref(p), ne, _p(so, c_ip), _p(x), _p(y), _p(tx), _p(ty), _p(qop),
                                 _p(keep, c_ip), _p(npe, c_ip), _p(offs, c_lp), ct.c_int64(cap), _p(v_evt, c_ip),
                                 _p(v_ia, c_ip), _p(v_ib, c_ip), _p(v), _p(v_flags, c_ip), ct.c_int64(ecap),
                                 _p(e_evt, c_ip), _p(e_ia, c_ip), _p(e_ib, c_ip), ct.byref(n_edge),
                                 ct.byref(n_pairs), int(n_threads))
        if (total <= cap or capacity is not None) and n_edge.value <= ecap:
            break
        cap = max(cap, int(total))
        ecap = max(ecap, int(n_edge.value))
    n = min(int(total), cap)
    ne_ = int(n_edge.value)
    out = dict(n=int(total), n_per_event=npe, offsets=offs, evt=v_evt[:n], ia=v_ia[:n], ib=v_ib[:n],
               flags=v_flags[:n], n_pairs=int(n_pairs.value),
               edge_pairs=set(zip(e_evt[:ne_].tolist(), e_ia[:ne_].tolist(), e_ib[:ne_].tolist())))
    for i, k in enumerate(("x", "y", "z", "doca", "m_pipi", "m_ppi")):
        out[k] = v[:n, i].copy()
    return out
