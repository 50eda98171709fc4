"""ds_vertex_static (include/ds.h): ds_vertex with its scratch in a fixed `static __device__` array of the library, for
callers that cannot allocate.  Checked against the existing path (ds_vertex with a caller's workspace) on two calls in a
row that share the array.  Collected last on purpose (pytest -x: a failure here hides nothing); passes alone in a fresh
process and after the other GPU tests."""
import numpy as np
import pytest

import gen
from gen import constants as C

pytestmark = pytest.mark.gpu
FIELDS = ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi")


def _host(torch, v):
    n = int(v["offsets"][-1].item())
    out = {k: v[k][:n].cpu().numpy() for k in FIELDS}
    out.update(n=n, offsets=v["offsets"].cpu().numpy(), n_per_event=v["n_per_event"].cpu().numpy(), overflow=int(v["overflow"].item()))
    return out


def test_vertex_static_equals_vertex_on_two_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    import paper_2503_13092_b200 as pk
    ds = pk.Downstream(C.GEOMETRY, gen.mlp_weights(0), C.PARAMS)
    try:
        cap = 1 << 16
        cases = []
        # two different batches (the second smaller, so that it finds the first one's lists, masks and sums in the array);
        # cfg3 events are large: that batch takes the block-per-event kernels with their scan launch
        for cfg, n_events in ((1, 300), (3, 40)):
            d = gen.generate(cfg, n_events=n_events)
            hits, seeds = ds.to_device(d["hits"]), ds.to_device(d["seeds"])
            ho, so = ds.to_device(dict(h=d["hit_offsets"], s=d["seed_offsets"])).values()
            trk = ds.reconstruct(hits, seeds, ho, so)
            ref = ds.vertex(trk, so, capacity=cap)                       # the existing path: caller's workspace
            out = ds.empty_vertices(cap, n_events)                        # outputs are the caller's, allocated up front
            cases.append((trk, so, ref, out))
        torch.cuda.synchronize()
        refs = [_host(torch, ref) for _, _, ref, _ in cases]
        assert refs[0]["n"] > 1000 and refs[1]["n"] > 100 and refs[0]["overflow"] == 0 and refs[1]["overflow"] == 0

        pk.ds_vertex_static_setup(ds.h)                                   # once per device: resolves the array's address
        free0, _ = torch.cuda.mem_get_info()
        for trk, so, _, out in cases:                                     # two calls in a row, same stream, no sync between
            ds.vertex_static(trk, so, out)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        assert free1 >= free0, "ds_vertex_static took device memory"
        for (_, _, _, out), ref in zip(cases, refs):
            got = _host(torch, out)
            assert got["n"] == ref["n"] and got["overflow"] == 0
            assert np.array_equal(got["offsets"], ref["offsets"]) and np.array_equal(got["n_per_event"], ref["n_per_event"])
            for k in FIELDS:                                              # same kernels, same arithmetic: bit for bit
                assert np.array_equal(got[k], ref[k]), k
        # and once more in the other order: the first batch after the second
        out_again = ds.empty_vertices(cap, 300)
        ds.vertex_static(cases[0][0], cases[0][1], out_again)
        torch.cuda.synchronize()
        got = _host(torch, out_again)
        for k in FIELDS:
            assert np.array_equal(got[k], refs[0][k]), k

        # beyond the fixed scratch: a clear error, nothing launched
        ne = pk.ds.DS_STATIC_MAX_EVENTS + 1
        so_big = torch.zeros(ne + 1, dtype=torch.int32, device=so.device)
        with pytest.raises(pk.DsError) as e:
            ds.vertex_static(ds.empty_tracks(0), so_big, ds.empty_vertices(16, ne))
        assert e.value.code == pk.ds.DS_E_LIMIT and "ds_vertex_static" in pk.ds_error_string(pk.ds.DS_E_LIMIT)
        ns = pk.ds.DS_STATIC_MAX_SEEDS + 1
        with pytest.raises(pk.DsError) as e:
            ds.vertex_static(ds.empty_tracks(ns), torch.tensor([0, ns], dtype=torch.int32, device=so.device), ds.empty_vertices(16, 1))
        assert e.value.code == pk.ds.DS_E_LIMIT
    finally:
        ds.close()
