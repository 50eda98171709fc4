"""Parity campaign beyond the fixed seeds of the test suite: other RNG blocks of the cfg1 / cfg3 / cfg2 generators, each with and
without per-hit jitter (z, weight, y range), alternating a tight and the default staging hint, through ds_reconstruct + ds_vertex
against the oracle under the rules of tests/parity.py (any mismatch outside the oracle's edge list raises).

    python tests/parity_campaign.py          # needs a CUDA device; about a minute on a B200
"""
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(HERE))
sys.path.insert(0, HERE)
import numpy as np, torch
import gen
from gen import constants as C
from oracle import ds_oracle as O
import paper_2503_13092_b200 as pk
import parity
w = gen.mlp_weights(0); orc = O.Mlp(w)
ds = pk.Downstream(C.GEOMETRY, w, C.PARAMS)
tot = dict(seeds=0, found=0, edge=0, exc=0, vtx=0, vexc=0)
for cfg, ne, blocks in ((1, 300, range(5, 25)), (3, 60, range(5, 15)), (2, 40, range(5, 10))):
    for b in blocks:
        for jitter in (False, True):
            d = gen.generate(cfg, n_events=ne, first_block=b)
            if jitter: d = gen.with_hit_jitter(d)
            hint = int(np.diff(d["hit_offsets"]).max()) if b % 2 else 0
            pp = dict(C.PARAMS, max_event_hits_hint=hint)
            ds.set_params(pp)
            hits, seeds = ds.to_device(d["hits"]), ds.to_device(d["seeds"])
            ho, so = ds.to_device(dict(h=d["hit_offsets"], s=d["seed_offsets"])).values()
            trk = ds.reconstruct(hits, seeds, ho, so); vtx = ds.vertex(trk, so, capacity=1 << 20)
            torch.cuda.synchronize()
            t = {k: v.cpu().numpy() for k, v in trk.items()}
            v = {k: (a.cpu().numpy() if hasattr(a, "cpu") else a) for k, a in vtx.items()}
            nv = int(v["offsets"][-1])
            for k in ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi"): v[k] = v[k][:nv]
            r = O.reconstruct(d["hits"], d["hit_offsets"], d["seeds"], d["seed_offsets"], C.GEOMETRY, pp, orc)
            st = parity.compare_tracks(t, r); sv = parity.compare_vertices(v, O.vertex(t, d["seed_offsets"], C.GEOMETRY, pp))
            tot["seeds"] += st["n"]; tot["found"] += st["found"]; tot["edge"] += st["edge_list"]; tot["exc"] += st["excused"]
            tot["vtx"] += sv["n"]; tot["vexc"] += sv["excused"]
    print("cfg", cfg, tot, flush=True)
ds.close(); print("campaign OK", tot)
