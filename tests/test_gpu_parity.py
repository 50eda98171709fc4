"""Parity of libds (CUDA, through the C ABI) against the CPU oracle on the same seeded inputs.  Needs a GPU.

Stage-wise: tracks are compared with the oracle's tracks; vertices are compared with the oracle run on
the GPU's own fp32 track arrays.  Rules in tests/parity.py.
"""
import numpy as np
import pytest

import gen
from gen import constants as C
from oracle import ds_oracle as O

import parity

pytestmark = pytest.mark.gpu
G, P = C.GEOMETRY, C.PARAMS


@pytest.fixture(scope="module")
def torch():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    return torch


@pytest.fixture(scope="module")
def ds(torch, mlp_w):
    import paper_2503_13092_b200 as pk
    d = pk.Downstream(G, mlp_w, P)
    yield d
    d.close()


def to_host(t):
    return {k: (v.cpu().numpy() if hasattr(v, "cpu") else v) for k, v in t.items()}


def gpu_run(ds, d, capacity=None, params=None):
    """ds_reconstruct + ds_vertex on device-resident copies of the generated arrays -> host dicts."""
    if params is not None:
        ds.set_params(params)
    try:
        hits, seeds = ds.to_device(d["hits"]), ds.to_device(d["seeds"])
        ho, so = ds.to_device(dict(h=d["hit_offsets"], s=d["seed_offsets"])).values()
        trk = ds.reconstruct(hits, seeds, ho, so)
        cap = capacity if capacity is not None else max(1024, 64 * len(d["seeds"]["x"]))
        vtx = ds.vertex(trk, so, capacity=cap)
        ds.torch.cuda.synchronize()
    finally:
        if params is not None:
            ds.set_params(P)
    t, v = to_host(trk), to_host(vtx)
    n = int(v["offsets"][-1])
    v["n"] = n
    for k in ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi"):
        v[k] = v[k][: min(n, cap)]
    return t, v


def oracle_run(d, orc_mlp, params=P):
    return O.reconstruct(d["hits"], d["hit_offsets"], d["seeds"], d["seed_offsets"], G, params, orc_mlp)


def check_both(ds, d, orc_mlp, params=None):
    pp = params if params is not None else P
    t, v = gpu_run(ds, d, params=params)
    r = oracle_run(d, orc_mlp, pp)
    st = parity.compare_tracks(t, r)
    ov = O.vertex(t, d["seed_offsets"], G, pp)          # oracle vertexing of the GPU's own tracks (stage-wise)
    assert v["n"] == ov["n"] or ov["edge_pairs"]
    sv = parity.compare_vertices(v, ov)
    assert (v["n_per_event"][: d["n_events"]] == ov["n_per_event"]).all() or ov["edge_pairs"]
    assert (np.diff(v["offsets"]) == v["n_per_event"][: d["n_events"]]).all() and v["overflow"][0] == 0
    return st, sv, t, v


# ---- S1 layout ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,n_events,hint,jitter", [(0, 10, 0, 0), (1, 64, 0, 0), (2, 24, 0, 0), (2, 24, 12288, 0), (1, 8, 256, 0),
                                                      (1, 64, 0, 1), (2, 12, 0, 1)])
def test_layout_equals_lexsort(ds, cfg, n_events, hint, jitter):
    d = gen.generate(cfg, n_events=n_events)
    if jitter:                                  # per-hit z, w, ymin, ymax all different: a gather from the wrong hit shows
        d = gen.with_hit_jitter(d)
    ds.set_params(dict(P, max_event_hits_hint=hint))
    try:
        hits = ds.to_device(d["hits"])
        ho = ds.to_device(dict(h=d["hit_offsets"]))["h"]
        out = to_host(ds.layout(hits, ho))
    finally:
        ds.set_params(P)
    h = d["hits"]
    ev = np.repeat(np.arange(n_events), np.diff(d["hit_offsets"]))
    layer, sector = (h["id"] >> 24) & 3, (h["id"] >> 20) & 15
    order = np.lexsort((h["id"], h["x0"], sector, layer, ev))          # last key is the primary one
    assert np.array_equal(out["perm"], order.astype(np.int32))
    for k in ("x0", "z", "ymin", "ymax", "w", "id"):
        assert np.array_equal(out[k], h[k][order]), k
    # bin table: entries of the (layer, sector) boundaries equal the counts; x0 slices are monotone and hold their x0 range
    nb = 4 * G["n_sectors_y"] * 16
    tab = out["bin_offsets"].reshape(-1, nb + 1)[:n_events]
    assert (np.diff(tab, axis=1) >= 0).all() and (tab[:, 0] == 0).all()
    assert (tab[:, nb] == np.diff(d["hit_offsets"])).all()
    coarse = (ev * 4 + layer) * G["n_sectors_y"] + sector
    cnt = np.bincount(coarse, minlength=n_events * 4 * G["n_sectors_y"]).reshape(n_events, -1)
    assert np.array_equal(np.diff(tab[:, ::16], axis=1), cnt)
    X = G["x_half"] + G["y_half"] * max(abs(v) for v in G["dxdy"])
    width = 2 * X / 16
    for e in range(min(n_events, 4)):
        xs = out["x0"][d["hit_offsets"][e]: d["hit_offsets"][e + 1]]
        b = np.searchsorted(tab[e], np.arange(len(xs)), side="right") - 1
        xb = b % 16
        lo, hi = -X + xb * width, -X + (xb + 1) * width
        assert ((xs >= lo - 1e-3) | (xb == 0)).all() and ((xs <= hi + 1e-3) | (xb == 15)).all()


def test_layout_inputs_not_16_byte_aligned(ds, torch):
    """Input arrays that start 4 bytes off a 16-byte boundary: k_layout stages them with ordinary loads instead of bulk
    copies and must give the same permutation; ds_reconstruct on the same views must equal the aligned run."""
    d = gen.generate(1, n_events=16)
    n = len(d["hits"]["id"])
    dev = ds.device
    hits_al = ds.to_device(d["hits"])
    hits_un = {}
    for k, v in d["hits"].items():
        buf = torch.empty(n + 1, dtype=hits_al[k].dtype, device=dev)
        buf[1:].copy_(hits_al[k])
        hits_un[k] = buf[1:]
        assert hits_un[k].data_ptr() % 16 == 4
    ho = ds.to_device(dict(h=d["hit_offsets"]))["h"]
    a, b = to_host(ds.layout(hits_al, ho)), to_host(ds.layout(hits_un, ho))
    for k in ("perm", "x0", "z", "ymin", "ymax", "w", "id", "bin_offsets"):
        assert np.array_equal(a[k], b[k]), k
    seeds = ds.to_device(d["seeds"])
    so = ds.to_device(dict(s=d["seed_offsets"]))["s"]
    ta, tb = to_host(ds.reconstruct(hits_al, seeds, ho, so)), to_host(ds.reconstruct(hits_un, seeds, ho, so))
    for k in ta:
        assert np.array_equal(ta[k], tb[k]), k


# ---- S2 extrapolation ----------------------------------------------------------------------------------------------
def test_extrapolate_equals_oracle(ds):
    d = gen.generate(1, n_events=4)
    s = d["seeds"]
    out = ds.extrapolate(ds.to_device(s)).cpu().numpy()
    for i in range(0, len(s["x"]), 7):
        ex = O.extrapolate(G, P, *(float(s[k][i]) for k in ("x", "y", "tx", "ty", "qop")))
        ref = np.array([ex["z_m"], ex["x_m"], ex["y_m"], *ex["y_l"], ex["tx_pred"], ex["xc3"], ex["w0"], ex["w1"], 0.0])
        assert np.allclose(out[i], ref, rtol=1e-13, atol=1e-10)


# ---- S1..S10 on the five configs ------------------------------------------------------------------------------------
def test_cfg0_noise_free(ds, orc_mlp, parity_counts):
    d = gen.generate(0)
    st, sv, t, v = check_both(ds, d, orc_mlp)
    parity_counts("cfg0", events=10, tracks=st, vertices=sv)
    assert st["found"] == 200 and (t["nhits"] == 4).all()
    sp = d["truth"]["seed_particle"]
    assert (d["truth"]["hit_particle"][t["hit"]] == sp[:, None]).all()     # P-1 on the GPU output itself


@pytest.mark.parametrize("cfg,n_events", [(1, 1000), (2, 1000), (3, 2000)])
def test_full_configs(ds, orc_mlp, parity_counts, cfg, n_events):
    d = gen.generate(cfg, n_events=n_events, workers=4)
    hint = 16384 if cfg == 2 else 0
    st, sv, t, v = check_both(ds, d, orc_mlp, params=dict(P, max_event_hits_hint=hint))
    assert st["found"] > 10 * n_events and sv["n"] > n_events
    parity_counts(f"cfg{cfg}", events=n_events, tracks=st, vertices=sv)
    print(f"cfg{cfg}: tracks {st}, vertices {sv}")


@pytest.mark.parametrize("cfg,n_events,hint,dv1,chi2ndf_max", [
    (1, 300, 0, 0, 5.0), (1, 300, 0, 0, 300.0), (1, 60, 0, 1, 300.0), (3, 30, 0, 0, 300.0),
    (2, 16, 0, 0, 300.0), (2, 16, 12288, 0, 300.0), (2, 8, 0, 1, 300.0), (2, 8, 12288, 1, 300.0)])
def test_per_hit_z_weight_and_y_range(ds, orc_mlp, parity_counts, cfg, n_events, hint, dv1, chi2ndf_max):
    """Hits whose z, weight and [ymin, ymax] differ from hit to hit (gen.with_hit_jitter): every per-hit gather of the kernels
    (the staged ymin / ymax, z and w of the first hit, of the fitted hits and of the Dv1 candidates) is now discriminated --
    fetching another hit's value of the same layer changes a window decision or the fit.  Dv0 and Dv1, staged events and
    events above the staging capacity (cfg2 with the default hint), with the default chi2 cut (most displaced candidates
    fail it) and a loose one (they pass and reach the track record)."""
    d = gen.with_hit_jitter(gen.generate(cfg, n_events=n_events))
    pp = dict(P, dv1=dv1, max_event_hits_hint=hint, chi2ndf_max=chi2ndf_max)
    st, sv, t, v = check_both(ds, d, orc_mlp, params=pp)
    assert st["found"] > n_events
    f = t["found"] == 1
    zs = d["hits"]["z"][np.maximum(t["hit"][f], 0)]
    assert len(np.unique(zs)) > 100 and len(np.unique(d["hits"]["w"])) == 3
    parity_counts(f"jitter_cfg{cfg}_hint{hint}_dv1{dv1}_chi2{chi2ndf_max:g}", events=n_events, tracks=st, vertices=sv)


def test_cfg2_oversize_path(ds, orc_mlp):
    """cfg2 events (~8000 hits) with the default 4096-hit hint: the layout takes its global-memory path."""
    d = gen.generate(2, n_events=12)
    check_both(ds, d, orc_mlp)


def test_cfg4_full(ds, orc_mlp, parity_counts):
    """BASELINE configs[4] in full: all 100 000 events, sub-batch by sub-batch (10 x 10 000 events, the launch configuration
    bench.py times, max_event_hits_hint = the sub-batch's largest event), every seed and every vertex against the oracle
    (OpenMP over events on the host cores)."""
    import os
    n_sub = C.CONFIGS[4].n_events // C.SUBBATCH_EVENTS
    bps = C.SUBBATCH_EVENTS // C.BLOCK_EVENTS
    tot_t = dict(n=0, found=0, edge_list=0, excused=0)
    tot_v = dict(n=0, n_pairs=0, edge_list=0, excused=0)
    for i in range(n_sub):
        d = gen.generate(4, n_events=C.SUBBATCH_EVENTS, first_block=i * bps, workers=min(10, os.cpu_count() or 1))
        pp = dict(P, max_event_hits_hint=int(np.diff(d["hit_offsets"]).max()))
        t, v = gpu_run(ds, d, capacity=1 << 20, params=pp)
        r = oracle_run(d, orc_mlp)
        st = parity.compare_tracks(t, r)
        ov = O.vertex(t, d["seed_offsets"], G, P)
        sv = parity.compare_vertices(v, ov)
        assert v["overflow"][0] == 0 and (np.diff(v["offsets"]) == v["n_per_event"][: d["n_events"]]).all()
        for k in tot_t:
            tot_t[k] += st[k]
        for k in tot_v:
            tot_v[k] += sv[k]
        del d, t, v, r, ov
    assert tot_t["n"] > 14e6 and tot_t["found"] > 2e6 and tot_v["n"] > 9e5
    assert tot_t["excused"] <= 1e-4 * tot_t["n"] and tot_v["excused"] <= 1e-4 * tot_v["n_pairs"]
    parity_counts("cfg4", events=C.CONFIGS[4].n_events, tracks=tot_t, vertices=tot_v)
    print(f"cfg4: tracks {tot_t}, vertices {tot_v}")


def test_cfg4_subbatch_sampled(ds, orc_mlp):
    """One 10 000-event sub-batch of cfg4 in the launch configuration bench.py times; the oracle recomputes a
    sample of events one by one (events are independent)."""
    d = gen.generate(4, n_events=C.SUBBATCH_EVENTS, workers=8)
    t, v = gpu_run(ds, d, capacity=1 << 20)
    rng = np.random.default_rng(0)
    sample = np.sort(rng.choice(C.SUBBATCH_EVENTS, 300, replace=False))
    ho, so = d["hit_offsets"], d["seed_offsets"]
    n_seeds = n_edge = n_vtx = 0
    for e in sample:
        h0, h1, s0, s1 = ho[e], ho[e + 1], so[e], so[e + 1]
        hits = {k: a[h0:h1] for k, a in d["hits"].items()}
        seeds = {k: a[s0:s1] for k, a in d["seeds"].items()}
        r = O.reconstruct(hits, [0, h1 - h0], seeds, [0, s1 - s0], G, P, orc_mlp, n_threads=1)
        r["hit"] = np.where(r["hit"] >= 0, r["hit"] + h0, -1)
        te = {k: a[s0:s1] for k, a in t.items()}
        # the 0.01 % bound is checked over the whole sample below
        bad = ((te["found"] != r["found"]) | (te["nhits"] != r["nhits"]) | (te["keep"] != r["keep"])
               | (te["hit"] != r["hit"]).any(axis=1))
        assert not (bad & (r["edge"] == 0)).any(), f"event {e}"
        n_edge += int(bad.sum())
        ok = ~bad & (r["found"] == 1)
        for k, floor in parity.TRACK_FLOORS.items():
            assert parity.close(te[k][ok], r[k][ok], floor).all(), (e, k)
        ov = O.vertex(te, [0, s1 - s0], G, P, n_threads=1)
        v0, v1 = v["offsets"][e], v["offsets"][e + 1]
        ge = {k: v[k][v0:v1] for k in ("evt", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi")}
        ge["ia"], ge["ib"] = v["ia"][v0:v1] - s0, v["ib"][v0:v1] - s0
        ge["evt"] = np.zeros_like(ge["evt"])
        assert (v["evt"][v0:v1] == e).all()
        parity.compare_vertices(ge, ov)
        n_seeds += s1 - s0
        n_vtx += ov["n"]
    assert n_edge <= 1e-4 * n_seeds + 1 and n_vtx > 300
    # properties that hold at any size, on the whole sub-batch
    assert ((t["found"] == 0) | (t["hit"][:, 3] >= 0)).all()                  # UTbX hit is mandatory
    ev_of_seed = np.repeat(np.arange(d["n_events"]), np.diff(so))
    hh = t["hit"]
    inside = (hh < 0) | ((hh >= ho[ev_of_seed][:, None]) & (hh < ho[ev_of_seed + 1][:, None]))
    assert inside.all()                                                        # hits belong to the seed's event
    lay = (d["hits"]["id"][np.maximum(hh, 0)] >> 24) & 3
    assert ((hh < 0) | (lay == np.arange(4)[None, :])).all()
    assert (t["nhits"] == (hh >= 0).sum(axis=1)).all() and ((t["found"] == 0) | (t["nhits"] >= P["min_hits"])).all()
    assert (t["chi2"][t["found"] == 1] <= P["chi2ndf_max"] * (t["nhits"][t["found"] == 1] - 1) * (1 + 1e-6)).all()
    assert (v["doca"] < P["doca_max"]).all() and (v["z"] >= P["zv_min"]).all() and (v["z"] <= P["zv_max"]).all()
    assert (t["qop"][v["ia"]] > 0).all() and (t["qop"][v["ib"]] < 0).all() and (v["flags"] > 0).all()
    assert (ev_of_seed[v["ia"]] == v["evt"]).all() and (ev_of_seed[v["ib"]] == v["evt"]).all()


# ---- variants of the parameters ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("override", [
    dict(max_first_hits=3), dict(min_hits=4), dict(mlp_keep_above=0, mlp_thr=0.5), dict(w0_b=400.0, w0_max=600.0),
    dict(chi2ndf_max=1.0, miss_penalty=0.5), dict(y_tol=60.0), dict(y_tol=130.0), dict(doca_max=0.5, dm_ks=10.0, zv_min=1000.0),
])
def test_parameter_variants(ds, orc_mlp, override):
    d = gen.generate(1, n_events=100)
    check_both(ds, d, orc_mlp, params=dict(P, **override))


def test_mirror_geometry_and_zmag_hook(ds, orc_mlp, mlp_w):
    """Another geometry on a second handle: mirrored (U/V swapped) and the z_mag polynomial (A-3) switched on."""
    import paper_2503_13092_b200 as pk
    g2 = dict(C.GEOMETRY, dxdy=tuple(-v for v in C.GEOMETRY["dxdy"]), zmag_c=(5282.0, 30.0, -20.0, 4.0))
    d = gen.generate(1, n_events=60)
    hits = dict(d["hits"], x0=-d["hits"]["x0"])
    seeds = dict(d["seeds"], x=-d["seeds"]["x"], tx=-d["seeds"]["tx"], qop=-d["seeds"]["qop"])
    d2 = dict(d, hits=hits, seeds=seeds)
    ds2 = pk.Downstream(g2, mlp_w, P)
    try:
        t, v = gpu_run(ds2, d2)
    finally:
        ds2.close()
    r = O.reconstruct(hits, d["hit_offsets"], seeds, d["seed_offsets"], g2, P, orc_mlp)
    parity.compare_tracks(t, r)
    parity.compare_vertices(v, O.vertex(t, d["seed_offsets"], g2, P))


# ---- S7 on its own ------------------------------------------------------------------------------------------------------
def test_ghost_killer_alone(ds, orc_mlp, torch):
    rng = np.random.default_rng(7)
    n = 5000
    trk = {k: (rng.normal(0, 1, n) * s + m).astype(np.float32)
           for k, m, s in zip(("x", "y", "tx", "ty", "qop", "chi2"), C.MLP_MU[:6], C.MLP_SIGMA[:6])}
    seeds = dict(x=trk["x"], y=trk["y"], tx=trk["tx"], ty=trk["ty"],
                 qop=(rng.normal(0, 0.25, n)).astype(np.float32), chi2=rng.chisquare(7, n).astype(np.float32) / 7)
    found = (rng.uniform(size=n) < 0.8).astype(np.int32)
    dev = ds.empty_tracks(n)
    for k, a in trk.items():
        dev[k].copy_(torch.as_tensor(a))
    dev["found"].copy_(torch.as_tensor(found))
    ref = np.array([orc_mlp.eval([trk["x"][i], trk["y"][i], trk["tx"][i], trk["ty"][i], trk["qop"][i], trk["chi2"][i],
                                  seeds["qop"][i], seeds["chi2"][i]]) for i in range(n)])
    med = float(np.median(ref))
    for thr, above in ((0.1, 1), (0.5, 0), (med, 1), (med, 0)):
        ds.set_params(dict(P, mlp_thr=thr, mlp_keep_above=above))
        try:
            ds.ghost_killer(ds.to_device(seeds), dev)
            torch.cuda.synchronize()
        finally:
            ds.set_params(P)
        score, keep = dev["score"].cpu().numpy(), dev["keep"].cpu().numpy()
        f = found == 1
        assert parity.close(score[f], ref[f], 1e-3).all() and not score[~f].any() and not keep[~f].any()
        want = (ref > thr) if above else (ref < thr)
        margin = np.abs(ref - thr) / thr
        assert (keep[f] == want[f])[margin[f] >= 1e-5].all()
        if thr == med:
            assert 0.4 < keep[f].mean() < 0.6


def test_paper_architecture_8_14_1(torch, mlp_w):
    """the paper's ghost killer has one hidden layer of 14 units.  Its own kernel instantiation
    (ds_upload_mlp_single -> k_mlp<14, 0>) and, as a cross-check, the exact embedding into the 8 -> 32 -> 16 -> 1 network
    (gen.embed_single_hidden) both give the scores of the oracle's single-hidden-layer evaluation; the fast-math flavour
    (__expf, __fdividef) stays within 2e-6 absolute of it, which is outside the bit-exact keep decision only for
    scores on the threshold."""
    import paper_2503_13092_b200 as pk
    rng = np.random.default_rng(14)
    w1 = dict(W1=rng.normal(0, 8 ** -0.5, (14, 8)).astype(np.float32), b1=rng.normal(0, 8 ** -0.5, 14).astype(np.float32),
              W3=rng.normal(0, 14 ** -0.5, 14).astype(np.float32), b3=rng.normal(0, 14 ** -0.5, 1).astype(np.float32),
              mu=mlp_w["mu"], inv_sigma=mlp_w["inv_sigma"])
    orc = O.Mlp(w1)                                                   # n_h2 = 0: W3 acts on the hidden layer
    assert orc.c.n_h1 == 14 and orc.c.n_h2 == 0
    n = 4000
    trk = {k: (rng.normal(0, 1, n) * s + m).astype(np.float32)
           for k, m, s in zip(("x", "y", "tx", "ty", "qop", "chi2"), C.MLP_MU[:6], C.MLP_SIGMA[:6])}
    seeds = dict(x=trk["x"], y=trk["y"], tx=trk["tx"], ty=trk["ty"], qop=rng.normal(0, 0.25, n).astype(np.float32),
                 chi2=(rng.chisquare(7, n) / 7).astype(np.float32))
    ref = np.array([orc.eval([trk["x"][i], trk["y"][i], trk["tx"][i], trk["ty"][i], trk["qop"][i], trk["chi2"][i],
                              seeds["qop"][i], seeds["chi2"][i]]) for i in range(n)])
    assert 0.05 < ref.std()

    def scores(dsx):
        dev = dsx.empty_tracks(n)
        for k, a in trk.items():
            dev[k].copy_(torch.as_tensor(a))
        dev["found"].fill_(1)
        dsx.ghost_killer(dsx.to_device(seeds), dev)
        torch.cuda.synchronize()
        return dev["score"].cpu().numpy(), dev["keep"].cpu().numpy()

    med = float(np.median(ref))
    pm = dict(P, mlp_thr=med)
    d14 = pk.Downstream(G, gen.embed_single_hidden(w1), pm)
    try:
        s_emb, k_emb = scores(d14)                                    # embedded in the 8 -> 32 -> 16 -> 1 kernel
        d14.upload_mlp_single(w1)
        s_one, k_one = scores(d14)                                    # k_mlp<14, 0, false>
        d14.set_params(dict(pm, mlp_fast_math=1))
        s_fast, k_fast = scores(d14)                                  # k_mlp<14, 0, true>
        pk.ds_upload_geometry(d14.h, G, mlp_w)                        # back to the 8 -> 32 -> 16 -> 1 network of cfg0
        d14.set_params(P)
        s_back, _ = scores(d14)
    finally:
        d14.close()
    for sc, kp in ((s_emb, k_emb), (s_one, k_one)):
        assert parity.close(sc, ref, 1e-3).all()
        margin = np.abs(ref - med) / med
        assert (kp == (ref > med))[margin >= 1e-5].all() and 0.4 < kp.mean() < 0.6
    assert np.abs(s_fast - ref).max() < 2e-6 and (k_fast != (ref > med)).sum() <= 2
    full = O.Mlp(mlp_w)
    ref_full = np.array([full.eval([trk["x"][i], trk["y"][i], trk["tx"][i], trk["ty"][i], trk["qop"][i], trk["chi2"][i],
                                    seeds["qop"][i], seeds["chi2"][i]]) for i in range(0, n, 40)])
    assert parity.close(s_back[::40], ref_full, 1e-3).all()


def test_fast_math_ghost_killer_on_tracks(ds, orc_mlp):
    """mlp_fast_math = 1 on the 8 -> 32 -> 16 -> 1 network through ds_reconstruct: same tracks, scores within 2e-6 absolute of
    the IEEE path, keep decisions equal except scores within 1e-5 of the threshold."""
    d = gen.generate(1, n_events=200)
    t0, _ = gpu_run(ds, d)
    t1, _ = gpu_run(ds, d, params=dict(P, mlp_fast_math=1))
    for k in ("x", "tx", "qop", "chi2", "found", "nhits", "hit"):
        assert np.array_equal(t0[k], t1[k]), k
    f = t0["found"] == 1
    assert f.sum() > 3000 and np.abs(t0["score"][f] - t1["score"][f]).max() < 2e-6
    diff = t0["keep"] != t1["keep"]
    assert (np.abs(t0["score"][diff] - P["mlp_thr"]) < 1e-5 * P["mlp_thr"]).all()


# ---- S8..S10 on hand-made tracks -----------------------------------------------------------------------------------------
def _tracks_from(ds, torch, arr):
    n = len(arr["x"])
    dev = ds.empty_tracks(n)
    for k in ("x", "y", "tx", "ty", "qop"):
        dev[k].copy_(torch.as_tensor(np.asarray(arr[k], dtype=np.float32)))
    dev["keep"].copy_(torch.as_tensor(np.asarray(arr["keep"], dtype=np.int32)))
    return dev


def test_vertex_closed_forms_and_overflow(ds, torch):
    """P-7 on the GPU: two lines through a common point; capacity overflow bookkeeping; cuts disabled -> n+ * n-."""
    zref = G["z_ref"]
    rng = np.random.default_rng(3)
    n_ev, per = 40, 30
    pts = np.stack([rng.normal(0, 80, n_ev), rng.normal(0, 80, n_ev), rng.uniform(700, 2300, n_ev)], 1)
    tx, ty = rng.uniform(-0.2, 0.2, (n_ev, per)), rng.uniform(-0.2, 0.2, (n_ev, per))
    arr = dict(x=(pts[:, None, 0] + tx * (zref - pts[:, None, 2])).ravel(), y=(pts[:, None, 1] + ty * (zref - pts[:, None, 2])).ravel(),
               tx=tx.ravel(), ty=ty.ravel(), qop=(rng.choice([-1.0, 1.0], n_ev * per) / rng.uniform(2, 50, n_ev * per)),
               keep=(rng.uniform(size=n_ev * per) < 0.9).astype(np.int32))
    so = np.arange(0, n_ev * per + 1, per, dtype=np.int32)
    loose = dict(P, doca_max=1e30, zv_min=-1e30, zv_max=1e30, dm_ks=1e30, dm_lambda=1e30, n2_min=0.0)
    ds.set_params(loose)
    try:
        dev = _tracks_from(ds, torch, arr)
        dso = ds.to_device(dict(s=so))["s"]
        v = to_host(ds.vertex(dev, dso, capacity=1 << 16))
        n = int(v["offsets"][-1])
        a32 = {k: np.asarray(arr[k], dtype=np.float32) for k in ("x", "y", "tx", "ty", "qop")}
        kq = (arr["keep"] == 1)
        npos = np.add.reduceat((kq & (a32["qop"] > 0)).astype(np.int64), so[:-1])
        nneg = np.add.reduceat((kq & (a32["qop"] < 0)).astype(np.int64), so[:-1])
        assert (v["n_per_event"][:n_ev] == npos * nneg).all() and n == int((npos * nneg).sum())
        assert (v["doca"][:n] < 2e-3).all()                           # fp32 storage of x, y at ~100 mm
        assert np.allclose(np.stack([v["x"][:n], v["y"][:n]], 1), pts[v["evt"][:n], :2], atol=0.05)
        assert np.allclose(v["z"][:n], pts[v["evt"][:n], 2], atol=2.0)
        ov = O.vertex(dict(a32, keep=arr["keep"]), so, G, loose)
        vv = {k: v[k][:n] for k in ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi")}
        # DOCA ~ 0 here: compare what is well-conditioned (the list, the masses)
        assert list(zip(vv["evt"], vv["ia"], vv["ib"])) == list(zip(ov["evt"], ov["ia"], ov["ib"]))
        assert parity.close(vv["m_pipi"], ov["m_pipi"], 0).all() and parity.close(vv["m_ppi"], ov["m_ppi"], 0).all()
        # overflow: capacity smaller than the list
        cap = n // 3
        v2 = to_host(ds.vertex(dev, dso, capacity=cap))
        assert int(v2["offsets"][-1]) == n and v2["overflow"][0] == n - cap
        assert np.array_equal(v2["ia"][:cap], v["ia"][:cap]) and np.array_equal(v2["doca"][:cap], v["doca"][:cap])
    finally:
        ds.set_params(P)
    # (0,0)+(t,0,1)s and (0,d)+(-t,0,1)s: DOCA = d, vertex (0, d/2, z_ref); parallel pair: no vertex (A-14)
    arr = dict(x=[0, 0, 5, 9], y=[0, 1.5, 0, 3], tx=[0.1, -0.1, 0.05, 0.05], ty=[0, 0, 0.02, 0.02], qop=[0.2, -0.25, 0.1, -0.1],
               keep=[1, 1, 1, 1])
    ds.set_params(dict(P, zv_min=-1e9, zv_max=1e9, dm_ks=1e9, dm_lambda=1e9, doca_max=1e9))
    try:
        v = to_host(ds.vertex(_tracks_from(ds, torch, arr), ds.to_device(dict(s=np.array([0, 2, 4], dtype=np.int32)))["s"], capacity=16))
    finally:
        ds.set_params(P)
    assert int(v["offsets"][-1]) == 1 and v["n_per_event"][1] == 0
    assert v["doca"][0] == pytest.approx(1.5, rel=1e-6) and v["z"][0] == pytest.approx(zref, abs=1e-3) and v["y"][0] == pytest.approx(0.75, rel=1e-6)


# ---- degenerate inputs -----------------------------------------------------------------------------------------------------
def test_empty_and_ragged_inputs(ds, orc_mlp):
    d = gen.generate(1, n_events=9)
    ho, so = d["hit_offsets"].copy(), d["seed_offsets"].copy()
    # event 2: no seeds; event 4: no hits; event 6: neither; last event: one seed
    def cut(arrs, off, e, keep_n=0):
        a, b = off[e] + keep_n, off[e + 1]
        out = {k: np.concatenate([v[:a], v[b:]]) for k, v in arrs.items()}
        off = off.copy()
        off[e + 1:] -= b - a
        return out, off
    hits, seeds = d["hits"], d["seeds"]
    seeds, so = cut(seeds, so, 2)
    hits, ho = cut(hits, ho, 4)
    seeds, so = cut(seeds, so, 6)
    hits, ho = cut(hits, ho, 6)
    seeds, so = cut(seeds, so, 8, keep_n=1)
    d2 = dict(n_events=9, hits=hits, seeds=seeds, hit_offsets=ho, seed_offsets=so)
    st, sv, t, v = check_both(ds, d2, orc_mlp)
    assert not t["found"][so[4]:so[5]].any()
    # no events at all / no seeds at all / no hits at all
    z = dict(n_events=0, hits={k: v[:0] for k, v in hits.items()}, seeds={k: v[:0] for k, v in seeds.items()},
             hit_offsets=np.zeros(1, np.int32), seed_offsets=np.zeros(1, np.int32))
    t0, v0 = gpu_run(ds, z)
    assert v0["n"] == 0 and len(t0["found"]) == 0
    z = dict(d2, seeds={k: v[:0] for k, v in seeds.items()}, seed_offsets=np.zeros(10, np.int32))
    t0, v0 = gpu_run(ds, z)
    assert v0["n"] == 0
    z = dict(d2, hits={k: v[:0] for k, v in hits.items()}, hit_offsets=np.zeros(10, np.int32))
    t0, v0 = gpu_run(ds, z)
    assert not t0["found"].any() and v0["n"] == 0
    # the "next" rows on the same ragged events: Dv1 search, clone killing, curved-track vertexing together
    check_both(ds, d2, orc_mlp, params=dict(P, dv1=1, magnet_polarity=1.0))
    t1, _ = gpu_run(ds, d2, params=dict(P, dv1=1, clone_min_shared=3))
    t2, _ = gpu_run(ds, z, params=dict(P, dv1=1, clone_min_shared=3, magnet_polarity=-1.0))
    assert not t2["found"].any() and t1["found"].sum() > 0


@pytest.mark.parametrize("cfg,n_events,mp", [(1, 300, 1.0), (1, 300, -1.0), (3, 40, 1.0)])
def test_curved_track_vertexing(ds, orc_mlp, cfg, n_events, mp):
    """parabolic trajectories upstream of the UT (Eq. 3 / Eq. 4) and Newton-Raphson closest approach
     in both vertex kernel variants (cfg1: warp per event, cfg3: block per event) against the oracle."""
    d = gen.generate(cfg, n_events=n_events)
    pc = dict(P, magnet_polarity=mp)
    st, sv, t, v = check_both(ds, d, orc_mlp, params=pc)
    t0, v0 = gpu_run(ds, d)
    assert v["n"] > 50 and v0["n"] > 50
    both = min(len(v["z"]), len(v0["z"]), 50)
    assert not np.allclose(v["z"][:both], v0["z"][:both], rtol=1e-6)      # the curvature moves the vertices
    # no curvature left: the straight-track list again
    t1, v1 = gpu_run(ds, d, params=dict(pc, gamma_c0=0.0, gamma_c1=0.0))
    assert v1["n"] == v0["n"] and np.array_equal(v1["ia"], v0["ia"]) and np.allclose(v1["z"], v0["z"], rtol=1e-6)


@pytest.mark.parametrize("cfg,n_events,hint", [(0, 10, 0), (1, 80, 0), (3, 12, 0), (2, 8, 0), (2, 8, 12288)])
def test_dv1_triplet_search(ds, orc_mlp, cfg, n_events, hint):
    """SURVEY §8f N2 (P:107-P:111, A-32): no first window, every UTbX hit of the y-compatible sectors, mandatory collinear
    UTaX hit -- staged events, events above the staging capacity (cfg2 with the default hint) and many seeds (cfg3)."""
    d = gen.generate(cfg, n_events=n_events)
    pd = dict(P, dv1=1, max_event_hits_hint=hint)
    st, sv, t, v = check_both(ds, d, orc_mlp, params=pd)
    assert st["found"] > 0 and (t["hit"][t["found"] == 1][:, [0, 3]] >= 0).all()
    t0, _ = gpu_run(ds, d, params=dict(P, max_event_hits_hint=hint))
    print(f"cfg{cfg}: Dv1 finds {int(t['found'].sum())} tracks, Dv0 {int(t0['found'].sum())}; {st}")


@pytest.mark.parametrize("cfg,n_events", [(1, 200), (3, 30)])
def test_clone_killing(ds, orc_mlp, cfg, n_events):
    """on events with doubled seeds, ds_reconstruct with clone_min_shared = 3 equals its own
    S6 output with the oracle's clone list removed, slot by slot and bit for bit; ds_clone_kill alone does the same."""
    d = gen.with_clone_seeds(gen.generate(cfg, n_events=n_events))
    t0, _ = gpu_run(ds, d)                                          # clone killing off: the S6 / S7 records
    killed = O.clone_kill(t0, d["seed_offsets"], P).astype(bool)
    assert killed.sum() > 20 and not killed[t0["found"] == 0].any()
    pk = dict(P, clone_min_shared=3)
    t1, v1 = gpu_run(ds, d, params=pk)
    exp = {k: v.copy() for k, v in t0.items()}
    for k in ("x", "y", "tx", "ty", "qop", "chi2", "score"):
        exp[k][killed] = 0.0
    for k in ("nhits", "found", "keep"):
        exp[k][killed] = 0
    exp["hit"][killed] = -1
    for k in exp:
        assert np.array_equal(t1[k], exp[k]), k
    # the vertices are those of the surviving tracks
    ov = O.vertex(t1, d["seed_offsets"], G, pk)
    assert v1["n"] == ov["n"] or ov["edge_pairs"]
    parity.compare_vertices(v1, ov)
    # standalone entry point on device-resident S6 / S7 records
    ds.set_params(pk)
    try:
        dev = ds.to_device(t0)
        so = ds.to_device(dict(s=d["seed_offsets"]))["s"]
        t2 = to_host(ds.clone_kill(dev, so))
    finally:
        ds.set_params(P)
    for k in exp:
        assert np.array_equal(t2[k], exp[k]), k


def test_line_nns(ds, orc_mlp):
    """SURVEY §8f N4 (P:277-P:285, A-33): the four line NNs on the vertices ds_vertex wrote, against the oracle fed the
    GPU's own tracks and vertices: scores within 1e-4 relative, decision bits exact except scores within 1e-5 of 0.5."""
    d = gen.generate(1, n_events=300)
    lw = gen.line_weights(3)
    ds.upload_line_nets(lw)
    hits, seeds = ds.to_device(d["hits"]), ds.to_device(d["seeds"])
    ho, so = ds.to_device(dict(h=d["hit_offsets"], s=d["seed_offsets"])).values()
    trk = ds.reconstruct(hits, seeds, ho, so)
    vtx = ds.vertex(trk, so, capacity=1 << 14)
    ln = to_host(ds.lines(trk, vtx, d["n_events"]))
    t, v = to_host(trk), to_host(vtx)
    n = int(v["offsets"][-1])
    assert 100 < n <= 1 << 14
    vv = {k: v[k][:n] for k in ("ia", "ib", "x", "y", "z", "doca")}
    o = O.lines(lw, t, vv)
    assert np.allclose(ln["scores"][:n], o["scores"], rtol=1e-4, atol=1e-6)
    diff = ln["bits"][:n] != o["bits"]
    assert not (diff & (o["edge"] == 0)).any() and diff.sum() <= max(1, n // 10000)
    assert (ln["bits"][n:] == 0).all() and 0 < (o["bits"] != 0).sum() < n
    # a capacity smaller than the vertex count: only the written vertices are scored
    small = ds.vertex(trk, so, capacity=64)
    l2 = to_host(ds.lines(trk, small, d["n_events"]))
    assert np.array_equal(l2["bits"], ln["bits"][:64]) and np.allclose(l2["scores"], ln["scores"][:64], rtol=0, atol=0)


@pytest.mark.parametrize("dv1", [0, 1])
def test_results_do_not_depend_on_the_hint(ds, dv1):
    """max_event_hits_hint only sizes the staging buffers: a hint far below the event size (global-memory paths of both
    kernels), a tight one, the default and a generous one give the same records bit for bit."""
    d = gen.generate(1, n_events=24)
    ref = None
    for hint in (64, int(np.diff(d["hit_offsets"]).max()), 0, 18000):
        t, v = gpu_run(ds, d, params=dict(P, dv1=dv1, max_event_hits_hint=hint))
        if ref is None:
            ref = (t, v)
            assert t["found"].sum() > 100 and v["n"] > 50
            continue
        for k in ref[0]:
            assert np.array_equal(ref[0][k], t[k]), (hint, k)
        for k in ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi", "offsets"):
            assert np.array_equal(ref[1][k], v[k]), (hint, k)


def test_vertexing_large_events_in_a_small_event_batch(ds, orc_mlp):
    """A few cfg3 events (~500 seeds, thousands of pairs) among many empty ones: the batch averages few seeds per event
    and takes the warp-per-event vertex kernels, whose staging capacity and pair mask these events exceed.  The same
    events alone take the block-per-event kernels; both must give the oracle's list."""
    d = gen.generate(3, n_events=5)
    pad = 40
    ho = np.concatenate([d["hit_offsets"], np.full(pad, d["hit_offsets"][-1], np.int32)])
    so = np.concatenate([d["seed_offsets"], np.full(pad, d["seed_offsets"][-1], np.int32)])
    d2 = dict(d, n_events=5 + pad, hit_offsets=ho, seed_offsets=so)
    assert len(d["seeds"]["x"]) / d2["n_events"] <= 256 < len(d["seeds"]["x"]) / d["n_events"]
    st2, sv2, t2, v2 = check_both(ds, d2, orc_mlp)
    st1, sv1, t1, v1 = check_both(ds, d, orc_mlp)
    assert v1["n"] == v2["n"] and v1["n"] > 0
    for k in ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi"):
        assert np.array_equal(v1[k], v2[k]), k
    assert np.array_equal(v1["offsets"], v2["offsets"][:6]) and (v2["offsets"][5:] == v2["offsets"][5]).all()


def test_duplicate_hits_and_ties(ds, orc_mlp):
    """Every hit duplicated with a different id: equal distances and equal scores everywhere -> id tie-breaks decide."""
    d = gen.generate(1, n_events=20)
    h = d["hits"]
    n = len(h["id"])
    ev = np.repeat(np.arange(20), np.diff(d["hit_offsets"]))
    dup = {k: np.concatenate([v, v]) for k, v in h.items()}
    dup["id"] = np.concatenate([h["id"], h["id"] + 50000])                # seq + 50000 stays below 2^20
    order = np.argsort(np.concatenate([ev, ev]), kind="stable")
    rng = np.random.default_rng(1)
    hits = {k: v[order] for k, v in dup.items()}
    ho = (2 * d["hit_offsets"]).astype(np.int32)
    for e in range(20):                                                      # shuffle inside the event
        p = rng.permutation(ho[e + 1] - ho[e]) + ho[e]
        for k in hits:
            hits[k][ho[e]:ho[e + 1]] = hits[k][p]
    assert n * 2 == ho[-1]
    d2 = dict(d, hits=hits, hit_offsets=ho)
    check_both(ds, d2, orc_mlp)
    # the same in the Dv1 triplet search: equal scores inside a fit window go through its full (hits, ids) comparison
    check_both(ds, d2, orc_mlp, params=dict(P, dv1=1))


@pytest.mark.parametrize("extra_n,x_half", [(6000, 860.0), (8000, 200.0)])
def test_dense_window_more_than_ten_first_hits(ds, orc_mlp, extra_n, x_half):
    """A crowded UTbX: > 10 (and > 32) hits inside the first window -> the 10 closest by (distance, id).  The second
    case packs the extra hits into |x| < 200 mm: first windows there hold more than 64 hits, which k_event ranks by the
    seed's own lane instead of the whole warp."""
    d = gen.generate(1, n_events=6)
    rng = np.random.default_rng(2)
    lay = np.full(extra_n, 3)
    x = rng.uniform(-x_half, x_half, extra_n)
    x[: extra_n // 2] = np.round(x[: extra_n // 2])                      # many exact ties in distance
    y = rng.uniform(-700, 700, extra_n)
    sec = np.clip(np.floor((y + 700) / 100).astype(np.int64), 0, 13)
    add = dict(x0=x.astype(np.float32), z=np.full(extra_n, G["z_layer"][3], np.float32), ymin=(-700 + 100 * sec).astype(np.float32),
               ymax=(-600 + 100 * sec).astype(np.float32), w=np.full(extra_n, C.W_HIT, np.float32),
               id=((100000 + np.arange(extra_n)) | (sec << 20) | (lay << 24)).astype(np.int32))
    e = 3
    at = d["hit_offsets"][e + 1]
    hits = {k: np.concatenate([v[:at], add[k], v[at:]]) for k, v in d["hits"].items()}
    ho = d["hit_offsets"].copy()
    ho[e + 1:] += extra_n
    st, sv, t, v = check_both(ds, dict(d, hits=hits, hit_offsets=ho), orc_mlp, params=dict(P, max_event_hits_hint=12288))
    assert st["found"] > 0


def test_hint_between_event_sizes(ds, orc_mlp):
    """A hint below the larger events of the batch: k_event takes the events that fit its staging, k_layout + k_track the
    others, inside one ds_reconstruct call; the results are those of any other hint."""
    d = gen.generate(1, n_events=60)
    sizes = np.diff(d["hit_offsets"])
    hint = int(np.median(sizes))
    assert (sizes + 3 > ((hint + 7) & ~7) + 8).any() and (sizes + 3 <= ((hint + 7) & ~7) + 8).any()
    st, sv, t, v = check_both(ds, d, orc_mlp, params=dict(P, max_event_hits_hint=hint))
    t0, v0 = gpu_run(ds, d, params=dict(P, max_event_hits_hint=0))
    for k in t:
        assert np.array_equal(t[k], t0[k]), k
    assert v["n"] == v0["n"]


# ---- host-buffer path ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pinned", [False, True])
def test_process_host_equals_device_path(ds, torch, pinned):
    import paper_2503_13092_b200 as pk
    d = gen.generate(1, n_events=50)
    t, v = gpu_run(ds, d)
    ns, ne = len(d["seeds"]["x"]), d["n_events"]
    cap = 4096
    ot, ovx = pk.host_tracks(ns, pinned), pk.host_vertices(cap, ne, pinned)
    n = ds.process_host(d["hits"], d["seeds"], d["hit_offsets"], d["seed_offsets"], ot, ovx, cap)
    ot, ovx = to_host({k: (a.numpy() if hasattr(a, "numpy") else a) for k, a in ot.items()}), \
        {k: (a.numpy() if hasattr(a, "numpy") else a) for k, a in ovx.items()}
    assert n == v["n"]
    for k in t:
        assert np.array_equal(np.asarray(ot[k]).reshape(t[k].shape), t[k]), k
    for k in ("evt", "ia", "ib", "flags", "x", "y", "z", "doca", "m_pipi", "m_ppi"):
        assert np.array_equal(ovx[k][:n], v[k]), k
    assert np.array_equal(ovx["offsets"], v["offsets"])


# ---- error codes -----------------------------------------------------------------------------------------------------------------
def test_error_codes(ds, torch, mlp_w):
    import paper_2503_13092_b200 as pk
    d = gen.generate(0)
    hits, seeds = ds.to_device(d["hits"]), ds.to_device(d["seeds"])
    ho, so = ds.to_device(dict(h=d["hit_offsets"], s=d["seed_offsets"])).values()
    trk = ds.empty_tracks(len(d["seeds"]["x"]))
    small = torch.empty(256, dtype=torch.uint8, device="cuda")
    with pytest.raises(pk.DsError) as e:
        pk.ds_reconstruct(ds.h, hits, seeds, ho, so, 10, ds.params, trk, small)
    assert e.value.code == pk.ds.DS_E_WORKSPACE
    with pytest.raises(pk.DsError) as e:
        pk.ds_reconstruct(ds.h, hits, seeds, ho, so, 10, pk.make_params(dict(P, max_first_hits=11)), trk, ds.workspace(10, 2000, 200))
    assert e.value.code == pk.ds.DS_E_ARG
    h2 = pk.ds_create(0)
    try:
        with pytest.raises(pk.DsError) as e:
            pk.ds_reconstruct(h2, hits, seeds, ho, so, 10, ds.params, trk, ds.workspace(10, 2000, 200))
        assert e.value.code == pk.ds.DS_E_NOGEOM
        with pytest.raises(pk.DsError) as e:
            pk.ds_upload_geometry(h2, dict(G, n_sectors_y=17), mlp_w)
        assert e.value.code == pk.ds.DS_E_ARG
    finally:
        pk.ds_destroy(h2)
    with pytest.raises(pk.DsError) as e:
        pk.ds_create(99)
    assert e.value.code == pk.ds.DS_E_CUDA
