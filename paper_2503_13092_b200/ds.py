"""Thin ctypes binding of libds (include/ds.h): argument marshalling only, every step runs in the CUDA kernels.

Functions carry the C names (ds_create, ds_upload_geometry, ds_layout, ds_extrapolate, ds_reconstruct,
ds_ghost_killer, ds_vertex, ds_process_host); `Downstream` bundles a handle with its geometry / parameters and
allocates outputs and workspaces as torch tensors.  torch is used for device memory and streams only.

There is no CPU fallback: if libds.so is missing it is built with nvcc, and if that fails, or there is no CUDA
device, the calls raise.
"""
from __future__ import annotations

import ctypes as ct
import os

import numpy as np

from . import build as _build

DS_OK, DS_E_ARG, DS_E_NOGEOM, DS_E_WORKSPACE, DS_E_CUDA, DS_E_LIMIT = 0, -1, -2, -3, -4, -5
DS_STATIC_MAX_EVENTS, DS_STATIC_MAX_SEEDS, DS_STATIC_SCRATCH_BYTES = 2048, 524288, 4227072
DS_MLP_IN, DS_MLP_H1, DS_MLP_H2 = 8, 32, 16
DS_XBINS, DS_MAX_SECTORS, DS_MAX_FIRST_HITS = 16, 16, 10

c_fp = ct.POINTER(ct.c_float)
c_ip = ct.POINTER(ct.c_int32)
c_lp = ct.POINTER(ct.c_int64)


class DsGeometry(ct.Structure):
    _fields_ = [("struct_size", ct.c_size_t), ("z_layer", ct.c_double * 4), ("dxdy", ct.c_double * 4),
                ("x_half", ct.c_double), ("y_half", ct.c_double), ("hole_half", ct.c_double),
                ("n_sectors_y", ct.c_int32), ("pad_", ct.c_int32), ("sector_height", ct.c_double),
                ("z_seed", ct.c_double), ("z_ref", ct.c_double), ("zmag_c", ct.c_double * 4), ("kick", ct.c_double)]


class DsMlp(ct.Structure):
    _fields_ = [("struct_size", ct.c_size_t),
                ("W1", ct.c_float * (DS_MLP_H1 * DS_MLP_IN)), ("b1", ct.c_float * DS_MLP_H1),
                ("W2", ct.c_float * (DS_MLP_H2 * DS_MLP_H1)), ("b2", ct.c_float * DS_MLP_H2),
                ("W3", ct.c_float * DS_MLP_H2), ("b3", ct.c_float),
                ("mu", ct.c_float * DS_MLP_IN), ("inv_sigma", ct.c_float * DS_MLP_IN)]


DS_MLP_SINGLE_H = 14


class DsMlpSingle(ct.Structure):
    _fields_ = [("struct_size", ct.c_size_t),
                ("W1", ct.c_float * (DS_MLP_SINGLE_H * DS_MLP_IN)), ("b1", ct.c_float * DS_MLP_SINGLE_H),
                ("W3", ct.c_float * DS_MLP_SINGLE_H), ("b3", ct.c_float),
                ("mu", ct.c_float * DS_MLP_IN), ("inv_sigma", ct.c_float * DS_MLP_IN)]


DS_LINE_IN, DS_LINE_H, DS_N_LINES = 16, 32, 4


class DsLineNets(ct.Structure):
    _fields_ = [("struct_size", ct.c_size_t),
                ("W1", ct.c_float * (DS_N_LINES * DS_LINE_H * DS_LINE_IN)), ("b1", ct.c_float * (DS_N_LINES * DS_LINE_H)),
                ("W3", ct.c_float * (DS_N_LINES * DS_LINE_H)), ("b3", ct.c_float * DS_N_LINES),
                ("mu", ct.c_float * DS_LINE_IN), ("inv_sigma", ct.c_float * DS_LINE_IN)]


class DsParams(ct.Structure):
    _fields_ = [("struct_size", ct.c_size_t), ("w0_a", ct.c_double), ("w0_b", ct.c_double), ("w0_max", ct.c_double),
                ("w1_a", ct.c_double), ("w1_b", ct.c_double), ("y_tol", ct.c_double), ("w_mag", ct.c_double),
                ("chi2ndf_max", ct.c_double), ("miss_penalty", ct.c_double), ("min_hits", ct.c_int32),
                ("max_first_hits", ct.c_int32), ("mlp_thr", ct.c_double), ("mlp_keep_above", ct.c_int32),
                ("max_event_hits_hint", ct.c_int32), ("doca_max", ct.c_double), ("zv_min", ct.c_double),
                ("zv_max", ct.c_double), ("m_pi", ct.c_double), ("m_p", ct.c_double), ("m_ks", ct.c_double),
                ("m_lambda", ct.c_double), ("dm_ks", ct.c_double), ("dm_lambda", ct.c_double), ("n2_min", ct.c_double),
                ("magnet_polarity", ct.c_double), ("gamma_c0", ct.c_double), ("gamma_c1", ct.c_double),
                ("vtx_newton_iters", ct.c_int32), ("clone_min_shared", ct.c_int32), ("dv1", ct.c_int32), ("mlp_fast_math", ct.c_int32)]


class DsHits(ct.Structure):
    _fields_ = [("x0", ct.c_void_p), ("z", ct.c_void_p), ("ymin", ct.c_void_p), ("ymax", ct.c_void_p),
                ("w", ct.c_void_p), ("id", ct.c_void_p), ("n", ct.c_int64)]


class DsSeeds(ct.Structure):
    _fields_ = [("x", ct.c_void_p), ("y", ct.c_void_p), ("tx", ct.c_void_p), ("ty", ct.c_void_p),
                ("qop", ct.c_void_p), ("chi2", ct.c_void_p), ("n", ct.c_int64)]


class DsTracks(ct.Structure):
    _fields_ = [("x", ct.c_void_p), ("y", ct.c_void_p), ("tx", ct.c_void_p), ("ty", ct.c_void_p),
                ("qop", ct.c_void_p), ("chi2", ct.c_void_p), ("score", ct.c_void_p), ("nhits", ct.c_void_p),
                ("hit", ct.c_void_p), ("found", ct.c_void_p), ("keep", ct.c_void_p), ("n", ct.c_int64)]


class DsVertices(ct.Structure):
    _fields_ = [("evt", ct.c_void_p), ("ia", ct.c_void_p), ("ib", ct.c_void_p), ("x", ct.c_void_p),
                ("y", ct.c_void_p), ("z", ct.c_void_p), ("doca", ct.c_void_p), ("m_pipi", ct.c_void_p),
                ("m_ppi", ct.c_void_p), ("flags", ct.c_void_p), ("n_per_event", ct.c_void_p),
                ("offsets", ct.c_void_p), ("overflow", ct.c_void_p), ("capacity", ct.c_int64)]


DS_K_COUNT = 9


class DsProfile(ct.Structure):
    _fields_ = [("struct_size", ct.c_size_t), ("ms", ct.c_double * DS_K_COUNT), ("launches", ct.c_int64 * DS_K_COUNT)]


class DsLayoutOut(ct.Structure):
    _fields_ = [("x0", ct.c_void_p), ("z", ct.c_void_p), ("ymin", ct.c_void_p), ("ymax", ct.c_void_p),
                ("w", ct.c_void_p), ("id", ct.c_void_p), ("perm", ct.c_void_p), ("bin_offsets", ct.c_void_p),
                ("n", ct.c_int64)]


HIT_F = ("x0", "z", "ymin", "ymax", "w")
SEED_F = ("x", "y", "tx", "ty", "qop")
TRACK_F = ("x", "y", "tx", "ty", "qop", "chi2", "score")
TRACK_I = ("nhits", "found", "keep")
VTX_I = ("evt", "ia", "ib", "flags")
VTX_F = ("x", "y", "z", "doca", "m_pipi", "m_ppi")

_lib = None


class DsError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {ds_error_string(code)} ({code})")


def lib() -> ct.CDLL:
    """Load libds.so, building it with nvcc if it is missing or stale.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = ct.CDLL(path)
        vp = ct.c_void_p
        L.ds_create.argtypes = [ct.POINTER(vp), ct.c_int]
        L.ds_destroy.argtypes = [vp]
        L.ds_destroy.restype = None
        L.ds_error_string.argtypes = [ct.c_int]
        L.ds_error_string.restype = ct.c_char_p
        L.ds_upload_geometry.argtypes = [vp, ct.POINTER(DsGeometry), ct.POINTER(DsMlp)]
        L.ds_upload_mlp_single.argtypes = [vp, ct.POINTER(DsMlpSingle)]
        L.ds_layout.argtypes = [vp, ct.POINTER(DsHits), vp, ct.c_int, ct.POINTER(DsParams), ct.POINTER(DsLayoutOut), vp]
        L.ds_extrapolate.argtypes = [vp, ct.POINTER(DsSeeds), ct.POINTER(DsParams), vp, vp]
        L.ds_workspace_bytes.argtypes = [vp, ct.c_int, ct.c_int64, ct.c_int64]
        L.ds_workspace_bytes.restype = ct.c_size_t
        L.ds_reconstruct.argtypes = [vp, ct.POINTER(DsHits), ct.POINTER(DsSeeds), vp, vp, ct.c_int,
                                     ct.POINTER(DsParams), ct.POINTER(DsTracks), vp, ct.c_size_t, vp]
        L.ds_ghost_killer.argtypes = [vp, ct.POINTER(DsSeeds), ct.POINTER(DsParams), ct.POINTER(DsTracks), vp]
        L.ds_clone_kill.argtypes = [vp, vp, ct.c_int, ct.POINTER(DsParams), ct.POINTER(DsTracks), vp]
        L.ds_upload_line_nets.argtypes = [vp, ct.POINTER(DsLineNets)]
        L.ds_lines.argtypes = [vp, ct.POINTER(DsTracks), ct.POINTER(DsVertices), ct.c_int, ct.c_double, vp, vp, vp]
        L.ds_vertex_workspace_bytes.argtypes = [vp, ct.c_int, ct.c_int64]
        L.ds_vertex_workspace_bytes.restype = ct.c_size_t
        L.ds_vertex.argtypes = [vp, ct.POINTER(DsTracks), vp, ct.c_int, ct.POINTER(DsParams), ct.POINTER(DsVertices),
                                vp, ct.c_size_t, vp]
        L.ds_vertex_static_setup.argtypes = [vp]
        L.ds_vertex_static.argtypes = [vp, ct.POINTER(DsTracks), vp, ct.c_int, ct.POINTER(DsParams), ct.POINTER(DsVertices), vp]
        L.ds_process_host.argtypes = [vp, ct.POINTER(DsHits), ct.POINTER(DsSeeds), vp, vp, ct.c_int,
                                      ct.POINTER(DsParams), ct.POINTER(DsTracks), ct.POINTER(DsVertices),
                                      ct.POINTER(ct.c_int64), vp]
        L.ds_profile_enable.argtypes = [vp, ct.c_int]
        L.ds_profile_read.argtypes = [vp, ct.POINTER(DsProfile)]
        L.ds_kernel_name.argtypes = [ct.c_int]
        L.ds_kernel_name.restype = ct.c_char_p
        _lib = L
    return _lib


def _check(code, where):
    if code != DS_OK:
        raise DsError(code, where)


# ---- struct builders ------------------------------------------------------------------------------------------------
def make_geometry(g: dict) -> DsGeometry:
    o = DsGeometry()
    o.struct_size = ct.sizeof(DsGeometry)
    o.z_layer[:] = g["z_layer"]
    o.dxdy[:] = g["dxdy"]
    o.zmag_c[:] = g["zmag_c"]
    for k in ("x_half", "y_half", "hole_half", "n_sectors_y", "sector_height", "z_seed", "z_ref", "kick"):
        setattr(o, k, g[k])
    return o


def make_mlp(w: dict) -> DsMlp:
    o = DsMlp()
    o.struct_size = ct.sizeof(DsMlp)
    for k, shape in (("W1", (DS_MLP_H1, DS_MLP_IN)), ("b1", (DS_MLP_H1,)), ("W2", (DS_MLP_H2, DS_MLP_H1)),
                     ("b2", (DS_MLP_H2,)), ("W3", (DS_MLP_H2,)), ("mu", (DS_MLP_IN,)), ("inv_sigma", (DS_MLP_IN,))):
        a = np.ascontiguousarray(w[k], dtype=np.float32).reshape(-1)
        if a.size != int(np.prod(shape)):
            raise ValueError(f"mlp weight {k}: expected shape {shape}")
        getattr(o, k)[:] = a.tolist()
    o.b3 = float(np.asarray(w["b3"]).reshape(-1)[0])
    return o


def make_mlp_single(w: dict) -> DsMlpSingle:
    """w: W1 [14][8], b1 [14], W3 [14], b3 [1], mu [8], inv_sigma [8] (the paper's 8 -> 14 -> 1 network)."""
    o = DsMlpSingle()
    o.struct_size = ct.sizeof(DsMlpSingle)
    for k, size in (("W1", DS_MLP_SINGLE_H * DS_MLP_IN), ("b1", DS_MLP_SINGLE_H), ("W3", DS_MLP_SINGLE_H), ("mu", DS_MLP_IN),
                    ("inv_sigma", DS_MLP_IN)):
        a = np.ascontiguousarray(w[k], dtype=np.float32).reshape(-1)
        if a.size != size:
            raise ValueError(f"single-hidden-layer mlp weight {k}: expected {size} values")
        getattr(o, k)[:] = a.tolist()
    o.b3 = float(np.asarray(w["b3"]).reshape(-1)[0])
    return o


def make_line_nets(w: dict) -> DsLineNets:
    """w = gen.line_weights(): {"nets": 4 x {W1 [32][16], b1 [32], W3 [32], b3 [1]}, "mu" [16], "inv_sigma" [16]}."""
    o = DsLineNets()
    o.struct_size = ct.sizeof(DsLineNets)
    if len(w["nets"]) != DS_N_LINES:
        raise ValueError("four line networks expected")
    for k, size in (("W1", DS_LINE_H * DS_LINE_IN), ("b1", DS_LINE_H), ("W3", DS_LINE_H), ("b3", 1)):
        a = np.concatenate([np.ascontiguousarray(n[k], dtype=np.float32).reshape(-1) for n in w["nets"]])
        if a.size != DS_N_LINES * size:
            raise ValueError(f"line net weight {k}: wrong size")
        getattr(o, k)[:] = a.tolist()
    for k in ("mu", "inv_sigma"):
        getattr(o, k)[:] = np.ascontiguousarray(w[k], dtype=np.float32).reshape(-1).tolist()
    return o


def make_params(p: dict) -> DsParams:
    o = DsParams()
    o.struct_size = ct.sizeof(DsParams)
    for name, _ in DsParams._fields_:
        if name in p:
            setattr(o, name, p[name])
    return o


def _ptr(t):
    return None if t is None else t.data_ptr()


def _np_ptr(a):
    return None if a is None else a.ctypes.data


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream if isinstance(stream, int) else stream.cuda_stream


# ---- C-named functions (handles are c_void_p; tensors are torch CUDA tensors) -------------------------------------------
def ds_error_string(code: int) -> str:
    return lib().ds_error_string(code).decode()


def ds_version() -> int:
    return lib().ds_version()


def ds_create(device: int = 0) -> ct.c_void_p:
    h = ct.c_void_p()
    _check(lib().ds_create(ct.byref(h), device), "ds_create")
    return h


def ds_destroy(h) -> None:
    lib().ds_destroy(h)


def ds_upload_geometry(h, geometry: dict, mlp: dict) -> None:
    g, m = make_geometry(geometry), make_mlp(mlp)
    _check(lib().ds_upload_geometry(h, ct.byref(g), ct.byref(m)), "ds_upload_geometry")


def ds_upload_mlp_single(h, mlp: dict) -> None:
    m = make_mlp_single(mlp)
    _check(lib().ds_upload_mlp_single(h, ct.byref(m)), "ds_upload_mlp_single")


def _hits(hits) -> DsHits:
    s = DsHits()
    for k in HIT_F + ("id",):
        setattr(s, k, _ptr(hits[k]))
    s.n = hits["id"].numel()
    return s


def _seeds(seeds) -> DsSeeds:
    s = DsSeeds()
    for k in SEED_F:
        setattr(s, k, _ptr(seeds[k]))
    s.chi2 = _ptr(seeds.get("chi2"))
    s.n = seeds["x"].numel()
    return s


def _tracks(trk) -> DsTracks:
    s = DsTracks()
    for k in TRACK_F + TRACK_I + ("hit",):
        setattr(s, k, _ptr(trk.get(k)))
    s.n = trk["x"].numel()
    return s


def _vertices(v, capacity) -> DsVertices:
    s = DsVertices()
    for k in VTX_I + VTX_F + ("n_per_event", "offsets", "overflow"):
        setattr(s, k, _ptr(v[k]))
    s.capacity = capacity
    return s


def ds_layout(h, hits, hit_offsets, n_events, params: DsParams, out, stream=None) -> None:
    hs = _hits(hits)
    o = DsLayoutOut()
    for k in HIT_F + ("id", "perm", "bin_offsets"):
        setattr(o, k, _ptr(out[k]))
    o.n = hs.n
    _check(lib().ds_layout(h, ct.byref(hs), _ptr(hit_offsets), n_events, ct.byref(params), ct.byref(o),
                           _stream_ptr(stream)), "ds_layout")


def ds_extrapolate(h, seeds, params: DsParams, out, stream=None) -> None:
    ss = _seeds(seeds)
    _check(lib().ds_extrapolate(h, ct.byref(ss), ct.byref(params), _ptr(out), _stream_ptr(stream)), "ds_extrapolate")


def ds_workspace_bytes(h, n_events, n_hits, n_seeds) -> int:
    return lib().ds_workspace_bytes(h, n_events, n_hits, n_seeds)


def ds_reconstruct(h, hits, seeds, hit_offsets, seed_offsets, n_events, params: DsParams, out, workspace,
                   stream=None) -> None:
    hs, ss, ts = _hits(hits), _seeds(seeds), _tracks(out)
    _check(lib().ds_reconstruct(h, ct.byref(hs), ct.byref(ss), _ptr(hit_offsets), _ptr(seed_offsets), n_events,
                                ct.byref(params), ct.byref(ts), _ptr(workspace),
                                0 if workspace is None else workspace.numel() * workspace.element_size(),
                                _stream_ptr(stream)), "ds_reconstruct")


def ds_upload_line_nets(h, line_w: dict) -> None:
    n = make_line_nets(line_w)
    _check(lib().ds_upload_line_nets(h, ct.byref(n)), "ds_upload_line_nets")


def ds_lines(h, tracks, vertices, capacity: int, n_events: int, threshold: float, scores, bits, stream=None) -> None:
    ts, vs = _tracks(tracks), _vertices(vertices, capacity)
    _check(lib().ds_lines(h, ct.byref(ts), ct.byref(vs), n_events, float(threshold), _ptr(scores), _ptr(bits),
                          _stream_ptr(stream)), "ds_lines")


def ds_clone_kill(h, seed_offsets, n_events: int, params: DsParams, tracks, stream=None) -> None:
    ts = _tracks(tracks)
    _check(lib().ds_clone_kill(h, _ptr(seed_offsets), n_events, ct.byref(params), ct.byref(ts), _stream_ptr(stream)),
           "ds_clone_kill")


def ds_ghost_killer(h, seeds, params: DsParams, tracks, stream=None) -> None:
    ss, ts = _seeds(seeds), _tracks(tracks)
    _check(lib().ds_ghost_killer(h, ct.byref(ss), ct.byref(params), ct.byref(ts), _stream_ptr(stream)),
           "ds_ghost_killer")


def ds_vertex_workspace_bytes(h, n_events, n_seeds) -> int:
    return lib().ds_vertex_workspace_bytes(h, n_events, n_seeds)


def ds_vertex(h, tracks, seed_offsets, n_events, params: DsParams, out, capacity, workspace, stream=None) -> None:
    ts, vs = _tracks(tracks), _vertices(out, capacity)
    _check(lib().ds_vertex(h, ct.byref(ts), _ptr(seed_offsets), n_events, ct.byref(params), ct.byref(vs),
                           _ptr(workspace), 0 if workspace is None else workspace.numel() * workspace.element_size(),
                           _stream_ptr(stream)), "ds_vertex")


def ds_vertex_static_setup(h) -> None:
    _check(lib().ds_vertex_static_setup(h), "ds_vertex_static_setup")


def ds_vertex_static(h, tracks, seed_offsets, n_events, params: DsParams, out, capacity, stream=None) -> None:
    """ds_vertex with the scratch in the library's fixed device array: no workspace argument, no allocation."""
    ts, vs = _tracks(tracks), _vertices(out, capacity)
    _check(lib().ds_vertex_static(h, ct.byref(ts), _ptr(seed_offsets), n_events, ct.byref(params), ct.byref(vs),
                                  _stream_ptr(stream)), "ds_vertex_static")


def _hp(a):
    """Host pointer of a numpy array or a (pinned) torch CPU tensor."""
    if a is None:
        return None
    return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data


def _hn(a):
    return a.numel() if hasattr(a, "numel") else a.size


def ds_process_host(h, hits, seeds, hit_offsets, seed_offsets, n_events, params: DsParams, out_tracks, out_vertices,
                    capacity, stream=None) -> int:
    """All arrays in HOST memory (numpy or pinned torch CPU tensors).  Returns the true number of vertices."""
    hs, ss, ts, vs = DsHits(), DsSeeds(), DsTracks(), DsVertices()
    for k in HIT_F + ("id",):
        setattr(hs, k, _hp(hits[k]))
    hs.n = _hn(hits["id"])
    for k in SEED_F:
        setattr(ss, k, _hp(seeds[k]))
    ss.chi2 = _hp(seeds.get("chi2"))
    ss.n = _hn(seeds["x"])
    for k in TRACK_F + TRACK_I + ("hit",):
        setattr(ts, k, _hp(out_tracks[k]))
    ts.n = ss.n
    for k in VTX_I + VTX_F + ("n_per_event", "offsets", "overflow"):
        setattr(vs, k, _hp(out_vertices[k]))
    vs.capacity = capacity
    total = ct.c_int64(0)
    _check(lib().ds_process_host(h, ct.byref(hs), ct.byref(ss), _hp(hit_offsets), _hp(seed_offsets), n_events,
                                 ct.byref(params), ct.byref(ts), ct.byref(vs), ct.byref(total),
                                 _stream_ptr(stream)), "ds_process_host")
    return total.value


def ds_measure_dfma_peak(h) -> float:
    """Measured fp64 FMA throughput of the device in TFLOP/s."""
    v = ct.c_double(0.0)
    lib().ds_measure_dfma_peak.argtypes = [ct.c_void_p, ct.POINTER(ct.c_double)]
    _check(lib().ds_measure_dfma_peak(h, ct.byref(v)), "ds_measure_dfma_peak")
    return v.value


def ds_profile_enable(h, on: bool) -> None:
    _check(lib().ds_profile_enable(h, 1 if on else 0), "ds_profile_enable")


def ds_profile_read(h) -> dict:
    """{kernel name: (summed device ms, launches)} since the last read (waits for the recorded events)."""
    p = DsProfile()
    p.struct_size = ct.sizeof(DsProfile)
    _check(lib().ds_profile_read(h, ct.byref(p)), "ds_profile_read")
    return {lib().ds_kernel_name(k).decode(): (p.ms[k], p.launches[k]) for k in range(DS_K_COUNT)}


# ---- convenience wrapper: allocation of outputs / workspaces as torch tensors ----------------------------------------
class Downstream:
    """A libds handle with its geometry, MLP weights and parameters.  All compute happens in libds."""

    def __init__(self, geometry: dict, mlp: dict, params: dict, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_13092_b200 needs a CUDA device (there is no CPU fallback)")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.geometry = dict(geometry)
        self.n_bins = 4 * int(geometry["n_sectors_y"]) * DS_XBINS
        self.h = ds_create(device)
        ds_upload_geometry(self.h, geometry, mlp)
        self.set_params(params)

    def set_params(self, params: dict) -> None:
        self.params_dict = dict(params)
        self.params = make_params(params)

    def close(self) -> None:
        if getattr(self, "h", None):
            ds_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- helpers -------------------------------------------------------------------------------------------------
    def to_device(self, arrays: dict) -> dict:
        t = self.torch
        return {k: t.as_tensor(np.ascontiguousarray(v)).to(self.device) for k, v in arrays.items() if v is not None}

    def empty_tracks(self, n: int) -> dict:
        t = self.torch
        out = {k: t.empty(n, dtype=t.float32, device=self.device) for k in TRACK_F}
        out.update({k: t.empty(n, dtype=t.int32, device=self.device) for k in TRACK_I})
        out["hit"] = t.empty((n, 4), dtype=t.int32, device=self.device)
        return out

    def empty_vertices(self, capacity: int, n_events: int) -> dict:
        t = self.torch
        out = {k: t.empty(capacity, dtype=t.int32, device=self.device) for k in VTX_I}
        out.update({k: t.empty(capacity, dtype=t.float32, device=self.device) for k in VTX_F})
        out["n_per_event"] = t.empty(max(n_events, 1), dtype=t.int32, device=self.device)
        out["offsets"] = t.empty(n_events + 1, dtype=t.int64, device=self.device)
        out["overflow"] = t.zeros(1, dtype=t.int32, device=self.device)
        out["capacity"] = capacity
        return out

    def workspace(self, n_events: int, n_hits: int, n_seeds: int):
        nbytes = ds_workspace_bytes(self.h, n_events, n_hits, n_seeds)
        return self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)

    def vertex_workspace(self, n_events: int, n_seeds: int):
        nbytes = ds_vertex_workspace_bytes(self.h, n_events, n_seeds)
        return self.torch.empty(nbytes, dtype=self.torch.uint8, device=self.device)

    def _on_stream(self, tensor, stream):
        """A temporary the library uses on `stream` after this Python call has returned: tell the caching allocator, so that
        the block is not handed out again while the kernels still run on a stream other than the current one."""
        if stream is not None and hasattr(stream, "cuda_stream"):
            tensor.record_stream(stream)
        elif isinstance(stream, int):
            tensor.record_stream(self.torch.cuda.ExternalStream(stream, device=self.device))
        return tensor

    # -- the calls ---------------------------------------------------------------------------------------------------
    def layout(self, hits: dict, hit_offsets, stream=None) -> dict:
        t = self.torch
        n, ne = hits["id"].numel(), hit_offsets.numel() - 1
        out = {k: t.empty(n, dtype=t.float32, device=self.device) for k in HIT_F}
        out["id"] = t.empty(n, dtype=t.int32, device=self.device)
        out["perm"] = t.empty(n, dtype=t.int32, device=self.device)
        out["bin_offsets"] = t.empty((max(ne, 1), self.n_bins + 1), dtype=t.int32, device=self.device)
        ds_layout(self.h, hits, hit_offsets, ne, self.params, out, stream)
        return out

    def extrapolate(self, seeds: dict, stream=None):
        t = self.torch
        out = t.empty((seeds["x"].numel(), 12), dtype=t.float64, device=self.device)
        ds_extrapolate(self.h, seeds, self.params, out, stream)
        return out

    def reconstruct(self, hits: dict, seeds: dict, hit_offsets, seed_offsets, out=None, workspace=None, stream=None):
        ne = hit_offsets.numel() - 1
        if out is None:
            out = self.empty_tracks(seeds["x"].numel())
        if workspace is None:
            workspace = self._on_stream(self.workspace(ne, hits["id"].numel(), seeds["x"].numel()), stream)
        ds_reconstruct(self.h, hits, seeds, hit_offsets, seed_offsets, ne, self.params, out, workspace, stream)
        return out

    def upload_mlp_single(self, mlp: dict) -> None:
        """Switch the ghost killer to the paper's 8 -> 14 -> 1 network (until the geometry is uploaded again)."""
        ds_upload_mlp_single(self.h, mlp)

    def upload_line_nets(self, line_w: dict) -> None:
        ds_upload_line_nets(self.h, line_w)

    def lines(self, tracks: dict, vertices: dict, n_events: int, threshold: float = 0.5, stream=None) -> dict:
        """HLT1 line NNs on the vertices ds_vertex wrote: {"scores": [capacity][4] fp32, "bits": [capacity] int32}."""
        t, cap = self.torch, vertices["capacity"]
        out = dict(scores=t.zeros((cap, DS_N_LINES), dtype=t.float32, device=self.device),
                   bits=t.zeros(cap, dtype=t.int32, device=self.device))
        ds_lines(self.h, tracks, vertices, cap, n_events, threshold, out["scores"], out["bits"], stream)
        return out

    def clone_kill(self, tracks: dict, seed_offsets, stream=None):
        ds_clone_kill(self.h, seed_offsets, seed_offsets.numel() - 1, self.params, tracks, stream)
        return tracks

    def ghost_killer(self, seeds: dict, tracks: dict, stream=None):
        ds_ghost_killer(self.h, seeds, self.params, tracks, stream)
        return tracks

    def vertex(self, tracks: dict, seed_offsets, capacity: int = None, out=None, workspace=None, stream=None):
        ne = seed_offsets.numel() - 1
        if out is None:
            out = self.empty_vertices(capacity if capacity is not None else 1 << 20, ne)
        if workspace is None:
            workspace = self._on_stream(self.vertex_workspace(ne, tracks["x"].numel()), stream)
        ds_vertex(self.h, tracks, seed_offsets, ne, self.params, out, out["capacity"], workspace, stream)
        return out

    def vertex_static(self, tracks: dict, seed_offsets, out: dict, stream=None):
        """ds_vertex_static: the caller's `out` (empty_vertices), the library's fixed scratch; allocates nothing."""
        ds_vertex_static(self.h, tracks, seed_offsets, seed_offsets.numel() - 1, self.params, out, out["capacity"], stream)
        return out

    def process_host(self, hits: dict, seeds: dict, hit_offsets, seed_offsets, out_tracks: dict, out_vertices: dict,
                     capacity: int, stream=None) -> int:
        ne = _hn(hit_offsets) - 1
        return ds_process_host(self.h, hits, seeds, hit_offsets, seed_offsets, ne, self.params, out_tracks,
                               out_vertices, capacity, stream)


def host_tracks(n: int, pinned: bool = False) -> dict:
    """HOST output buffers for ds_process_host (numpy, or pinned torch tensors)."""
    if pinned:
        import torch
        out = {k: torch.empty(n, dtype=torch.float32).pin_memory() for k in TRACK_F}
        out.update({k: torch.empty(n, dtype=torch.int32).pin_memory() for k in TRACK_I})
        out["hit"] = torch.empty((n, 4), dtype=torch.int32).pin_memory()
        return out
    out = {k: np.empty(n, dtype=np.float32) for k in TRACK_F}
    out.update({k: np.empty(n, dtype=np.int32) for k in TRACK_I})
    out["hit"] = np.empty((n, 4), dtype=np.int32)
    return out


def host_vertices(capacity: int, n_events: int, pinned: bool = False) -> dict:
    if pinned:
        import torch
        out = {k: torch.empty(capacity, dtype=torch.int32).pin_memory() for k in VTX_I}
        out.update({k: torch.empty(capacity, dtype=torch.float32).pin_memory() for k in VTX_F})
        out["n_per_event"] = torch.empty(max(n_events, 1), dtype=torch.int32).pin_memory()
        out["offsets"] = torch.empty(n_events + 1, dtype=torch.int64).pin_memory()
        out["overflow"] = torch.zeros(1, dtype=torch.int32).pin_memory()
        return out
    out = {k: np.empty(capacity, dtype=np.int32) for k in VTX_I}
    out.update({k: np.empty(capacity, dtype=np.float32) for k in VTX_F})
    out["n_per_event"] = np.empty(max(n_events, 1), dtype=np.int32)
    out["offsets"] = np.empty(n_events + 1, dtype=np.int64)
    out["overflow"] = np.zeros(1, dtype=np.int32)
    return out
