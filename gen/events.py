"""Seeded synthetic Run-3-shaped events (BASELINE.json configs[0..4]; recipe in SURVEY.md §8d / DESIGN.md).

This module is the forward simulation only: particle decays, straight lines, one thin-magnet kick, detector
response.  It contains none of the reconstruction method's arithmetic and is the only code that feeds both
the CUDA library and the CPU oracle.

Determinism: `numpy.random.SeedSequence(cfg.seed).spawn(n_blocks)`; block b (events [b*B, (b+1)*B), B =
min(1000, cfg.n_events)) is generated from its own `default_rng` with a fixed draw order, so any block can be
produced independently (cfg4 sub-batches, multi-process generation, per-rank shards).
"""
from __future__ import annotations

import numpy as np

from . import constants as C

M_PI = C.PARAMS["m_pi"] / 1000.0      # GeV
M_P = C.PARAMS["m_p"] / 1000.0
M_KS = C.PARAMS["m_ks"] / 1000.0
M_L = C.PARAMS["m_lambda"] / 1000.0

HIT_FIELDS = ("x0", "z", "ymin", "ymax", "w")
SEED_FIELDS = ("x", "y", "tx", "ty", "qop", "chi2")


def _two_body_pstar(M, m1, m2):
    return np.sqrt((M * M - (m1 + m2) ** 2) * (M * M - (m1 - m2) ** 2)) / (2.0 * M)


def _offsets(ev, n_events):
    cnt = np.bincount(ev, minlength=n_events)
    off = np.zeros(n_events + 1, dtype=np.int64)
    np.cumsum(cnt, out=off[1:])
    return off


def _uniform_outside_hole(rng, n, g):
    """Uniform (x, y) on the plane, outside the square beam hole."""
    x = rng.uniform(-g["x_half"], g["x_half"], n)
    y = rng.uniform(-g["y_half"], g["y_half"], n)
    bad = (np.abs(x) < g["hole_half"]) & (np.abs(y) < g["hole_half"])
    while bad.any():
        k = int(bad.sum())
        x[bad] = rng.uniform(-g["x_half"], g["x_half"], k)
        y[bad] = rng.uniform(-g["y_half"], g["y_half"], k)
        bad = (np.abs(x) < g["hole_half"]) & (np.abs(y) < g["hole_half"])
    return x, y


def _in_ut(x, y, g):
    return ((np.abs(x) <= g["x_half"]) & (np.abs(y) <= g["y_half"])
            & ~((np.abs(x) < g["hole_half"]) & (np.abs(y) < g["hole_half"])))


def _decays(rng, cfg, ev, g):
    """Draw decays for the flat event-index array `ev`; returns per-daughter arrays (2 per decay, interleaved)."""
    n = ev.size
    is_ks = rng.uniform(size=n) < cfg.frac_ks
    zv = rng.uniform(800.0, 2200.0, n)
    sx = rng.uniform(-0.25, 0.25, n)
    sy = rng.uniform(-0.20, 0.20, n)
    P = np.exp(rng.uniform(np.log(2.0), np.log(50.0), n))          # parent momentum, GeV, log-uniform
    cth = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    anti = rng.uniform(size=n) < 0.5

    M = np.where(is_ks, M_KS, M_L)
    m1 = np.where(is_ks, M_PI, M_P)                                 # daughter 1: pi+ (K_S) or (anti)proton
    m2 = np.full(n, M_PI)
    pst = _two_body_pstar(M, m1, m2)
    sth = np.sqrt(np.maximum(0.0, 1.0 - cth * cth))
    ps = np.stack([pst * sth * np.cos(phi), pst * sth * np.sin(phi), pst * cth], axis=1)   # rest frame, daughter 1

    nrm = np.sqrt(sx * sx + sy * sy + 1.0)
    nhat = np.stack([sx / nrm, sy / nrm, 1.0 / nrm], axis=1)
    E = np.sqrt(P * P + M * M)
    gam = E / M
    bg = P / M                                                      # gamma*beta

    def boost(pvec, m):
        est = np.sqrt((pvec * pvec).sum(axis=1) + m * m)
        ppar = (pvec * nhat).sum(axis=1)
        return pvec + nhat * ((gam - 1.0) * ppar + bg * est)[:, None]

    p1 = boost(ps, m1)
    p2 = boost(-ps, m2)
    q1 = np.where(is_ks, 1.0, np.where(anti, -1.0, 1.0))
    q2 = -q1

    def il(a, b):                                                   # interleave daughters: 2k, 2k+1
        out = np.empty((2 * n,) + a.shape[1:], dtype=a.dtype)
        out[0::2] = a
        out[1::2] = b
        return out

    pvec = il(p1, p2)
    d = dict(
        ev=np.repeat(ev, 2), decay=np.repeat(np.arange(n), 2), q=il(q1, q2), mass=il(m1, m2),
        px=pvec[:, 0], py=pvec[:, 1], pz=pvec[:, 2],
        xv=np.repeat(sx * zv, 2), yv=np.repeat(sy * zv, 2), zv=np.repeat(zv, 2), is_ks=np.repeat(is_ks, 2),
    )
    pz = np.where(d["pz"] > 1e-6, d["pz"], np.nan)
    d["tx"] = d["px"] / pz
    d["ty"] = d["py"] / pz
    d["p"] = np.sqrt(d["px"] ** 2 + d["py"] ** 2 + d["pz"] ** 2)
    # UT crossings (straight from the vertex: no field upstream of the magnet kick)
    zl = np.asarray(g["z_layer"])
    d["xl"] = d["xv"][:, None] + d["tx"][:, None] * (zl[None, :] - d["zv"][:, None])
    d["yl"] = d["yv"][:, None] + d["ty"][:, None] * (zl[None, :] - d["zv"][:, None])
    ok = np.isfinite(d["tx"]) & _in_ut(d["xl"], d["yl"], g).all(axis=1)
    # thin-magnet kick and SciFi seed state
    zm = g["zmag_c"][0]
    txa = d["tx"] + d["q"] * g["kick"] / d["p"]
    d["xs"] = d["xv"] + d["tx"] * (zm - d["zv"]) + txa * (g["z_seed"] - zm)
    d["ys"] = d["yv"] + d["ty"] * (g["z_seed"] - d["zv"])
    d["txs"] = txa
    d["qop"] = d["q"] / d["p"]
    with np.errstate(invalid="ignore"):
        ok &= (np.abs(d["xs"]) < 3200.0) & (np.abs(d["ys"]) < 2500.0)          # A-26
    d["ok"] = ok
    return d


def generate_block(cfg: C.Config, block: int, n_events: int, rng_seq, dtype=np.float32):
    """Generate one block of `n_events` events.  Returns a dict of flat arrays + offsets + truth."""
    g = C.GEOMETRY
    rng = np.random.default_rng(rng_seq)
    zl = np.asarray(g["z_layer"])
    dxdy = np.asarray(g["dxdy"])

    # ---- decays -----------------------------------------------------------------------------------------
    if cfg.fixed_decays is not None:
        # cfg0: exactly `fixed_decays` accepted decays per event (both daughters reconstructible, A-23/A-26)
        over = 40 * cfg.fixed_decays
        ev = np.repeat(np.arange(n_events), over)
        d = _decays(rng, cfg, ev, g)
        both = d["ok"][0::2] & d["ok"][1::2]
        rank = np.cumsum(both.reshape(n_events, over), axis=1).reshape(-1)      # 1-based rank among accepted
        keep_dec = both & (rank <= cfg.fixed_decays)
        if not (np.bincount(ev[keep_dec], minlength=n_events) == cfg.fixed_decays).all():
            raise RuntimeError("cfg0 oversampling too small")
        dec_rank = rank - 1                                                     # 0-based accepted index
        keep = np.repeat(keep_dec, 2)
        seeded = keep & (np.repeat(dec_rank, 2) < cfg.seeded_decays)
    else:
        ndec = rng.poisson(cfg.mean_decays, n_events)
        ev = np.repeat(np.arange(n_events), ndec)
        d = _decays(rng, cfg, ev, g)
        keep = d["ok"].copy()
        seeded = keep
    part = {k: v[keep] for k, v in d.items() if k != "ok"}
    seeded = seeded[keep]
    n_part = part["ev"].size

    # ---- hits from decay daughters -------------------------------------------------------------------------
    eff_mask = rng.uniform(size=(n_part, 4)) < cfg.eff
    h_part, h_layer = np.nonzero(eff_mask)
    h_ev = part["ev"][h_part]
    h_x = part["xl"][h_part, h_layer]
    h_y = part["yl"][h_part, h_layer]
    h_truth = h_part.astype(np.int64)

    # ---- targets ------------------------------------------------------------------------------------------------
    n_hits_target = rng.poisson(cfg.n_hits, n_events) if cfg.n_hits is not None else None
    n_seed_target = rng.poisson(cfg.n_seeds, n_events) if cfg.n_seeds is not None else None

    # ---- prompt seedless tracks (cfg2, A-24) ----------------------------------------------------------------------
    if cfg.prompt_frac > 0.0:
        n_dec_hits = np.bincount(h_ev, minlength=n_events)
        want = np.maximum(0.0, cfg.prompt_frac * n_hits_target - n_dec_hits)
        n_prompt = np.round(want / (4.0 * cfg.eff * 0.93)).astype(np.int64)    # 0.93 ~ plane acceptance of a prompt line
        pev = np.repeat(np.arange(n_events), n_prompt)
        npr = pev.size
        z0 = rng.normal(0.0, 50.0, npr)
        ptx = rng.uniform(-0.30, 0.30, npr)
        pty = rng.uniform(-0.25, 0.25, npr)
        pxl = ptx[:, None] * (zl[None, :] - z0[:, None])
        pyl = pty[:, None] * (zl[None, :] - z0[:, None])
        pm = _in_ut(pxl, pyl, g) & (rng.uniform(size=(npr, 4)) < cfg.eff)
        pi_, pl_ = np.nonzero(pm)
        h_ev = np.concatenate([h_ev, pev[pi_]])
        h_layer = np.concatenate([h_layer, pl_])
        h_x = np.concatenate([h_x, pxl[pi_, pl_]])
        h_y = np.concatenate([h_y, pyl[pi_, pl_]])
        h_truth = np.concatenate([h_truth, np.full(pi_.size, -2, dtype=np.int64)])

    n_track_hits = h_ev.size
    smear = rng.normal(0.0, C.SIGMA_HIT, n_track_hits) if cfg.smear else np.zeros(n_track_hits)

    # ---- noise hits ------------------------------------------------------------------------------------------------------
    if n_hits_target is not None:
        n_noise = np.maximum(0, n_hits_target - np.bincount(h_ev, minlength=n_events))
        nev = np.repeat(np.arange(n_events), n_noise)
        nn = nev.size
        n_layer = rng.integers(0, 4, nn)
        nx, ny = _uniform_outside_hole(rng, nn, g)
        h_ev = np.concatenate([h_ev, nev])
        h_layer = np.concatenate([h_layer, n_layer])
        h_x = np.concatenate([h_x, nx])
        h_y = np.concatenate([h_y, ny])
        h_truth = np.concatenate([h_truth, np.full(nn, -1, dtype=np.int64)])
        smear = np.concatenate([smear, np.zeros(nn)])

    nh = h_ev.size
    x0 = h_x - h_y * dxdy[h_layer] + smear                                     # A-1
    sector = np.clip(np.floor((h_y + g["y_half"]) / g["sector_height"]).astype(np.int64), 0, g["n_sectors_y"] - 1)
    ymin = -g["y_half"] + g["sector_height"] * sector
    ymax = ymin + g["sector_height"]
    hoff = _offsets(h_ev, n_events)
    # seq = generation order inside the event; position = shuffled
    order0 = np.argsort(h_ev, kind="stable")
    seq = np.empty(nh, dtype=np.int64)
    seq[order0] = np.arange(nh) - hoff[h_ev[order0]]
    if (seq >= (1 << C.ID_SEQ_BITS)).any():
        raise RuntimeError("event too large for 20-bit seq")
    hid = seq | (sector << C.ID_SECTOR_SHIFT) | (h_layer.astype(np.int64) << C.ID_LAYER_SHIFT)
    perm = np.argsort(h_ev + rng.uniform(size=nh), kind="stable")              # shuffle inside each event

    hits = dict(
        x0=x0[perm].astype(dtype), z=zl[h_layer][perm].astype(dtype),
        ymin=ymin[perm].astype(dtype), ymax=ymax[perm].astype(dtype),
        w=np.full(nh, C.W_HIT).astype(dtype), id=hid[perm].astype(np.int32),
    )
    hit_truth = h_truth[perm]

    # ---- seeds -------------------------------------------------------------------------------------------------------------------
    sp = np.nonzero(seeded)[0]
    ns_true = sp.size
    s_ev = part["ev"][sp]
    sx, sy, stx, sty, sq = part["xs"][sp], part["ys"][sp], part["txs"][sp], part["ty"][sp], part["qop"][sp]
    if cfg.smear:
        sx = sx + rng.normal(0.0, 0.1, ns_true)
        sy = sy + rng.normal(0.0, 0.1, ns_true)
        stx = stx + rng.normal(0.0, 1e-4, ns_true)
        sty = sty + rng.normal(0.0, 1e-4, ns_true)
        sq = sq * (1.0 + rng.normal(0.0, 0.01, ns_true))
        schi = rng.chisquare(7, ns_true) / 7.0                                  # A-11
    else:
        schi = np.zeros(ns_true)
    s_truth = sp.astype(np.int64)
    if n_seed_target is not None:
        n_fake = np.maximum(0, n_seed_target - np.bincount(s_ev, minlength=n_events))
        fev = np.repeat(np.arange(n_events), n_fake)
        nf = fev.size
        s_ev = np.concatenate([s_ev, fev])
        sx = np.concatenate([sx, rng.uniform(-2500.0, 2500.0, nf)])
        sy = np.concatenate([sy, rng.uniform(-2000.0, 2000.0, nf)])
        stx = np.concatenate([stx, rng.uniform(-0.3, 0.3, nf)])
        sty = np.concatenate([sty, rng.uniform(-0.25, 0.25, nf)])
        sq = np.concatenate([sq, rng.uniform(-0.5, 0.5, nf)])
        schi = np.concatenate([schi, 3.0 * rng.chisquare(7, nf) / 7.0])
        s_truth = np.concatenate([s_truth, np.full(nf, -1, dtype=np.int64)])
    nsd = s_ev.size
    sperm = np.argsort(s_ev + rng.uniform(size=nsd), kind="stable")
    seeds = dict(x=sx[sperm].astype(dtype), y=sy[sperm].astype(dtype), tx=stx[sperm].astype(dtype),
                 ty=sty[sperm].astype(dtype), qop=sq[sperm].astype(dtype), chi2=schi[sperm].astype(dtype))
    soff = _offsets(s_ev, n_events)

    zref = g["z_ref"]
    truth = dict(
        hit_particle=hit_truth, seed_particle=s_truth[sperm],
        part_ev=part["ev"], part_decay=part["decay"], part_q=part["q"], part_p=part["p"],
        part_tx=part["tx"], part_ty=part["ty"], part_mass=part["mass"], part_is_ks=part["is_ks"],
        part_xref=part["xv"] + part["tx"] * (zref - part["zv"]),
        part_yref=part["yv"] + part["ty"] * (zref - part["zv"]),
        part_xv=part["xv"], part_yv=part["yv"], part_zv=part["zv"],
    )
    return dict(n_events=n_events, hits=hits, hit_offsets=hoff.astype(np.int32), seeds=seeds,
                seed_offsets=soff.astype(np.int32), truth=truth)


def block_size(cfg: C.Config) -> int:
    return min(C.BLOCK_EVENTS, cfg.n_events)


def _block_seq(cfg: C.Config, block: int):
    # identical to SeedSequence(seed).spawn(n)[block] for any n > block
    return np.random.SeedSequence(cfg.seed, spawn_key=(block,))


def concat(blocks):
    """Concatenate block dicts (offsets rebased; truth particle indices rebased)."""
    if len(blocks) == 1:
        return blocks[0]
    out = dict(n_events=sum(b["n_events"] for b in blocks))
    out["hits"] = {k: np.concatenate([b["hits"][k] for b in blocks]) for k in blocks[0]["hits"]}
    out["seeds"] = {k: np.concatenate([b["seeds"][k] for b in blocks]) for k in blocks[0]["seeds"]}
    for key, arr in (("hit_offsets", "hits"), ("seed_offsets", "seeds")):
        offs, base = [np.zeros(1, dtype=np.int64)], 0
        for b in blocks:
            offs.append(b[key][1:].astype(np.int64) + base)
            base += int(b[key][-1])
        cat = np.concatenate(offs)
        if cat[-1] >= 2 ** 31:
            raise OverflowError("int32 offsets overflow; split into sub-batches")
        out[key] = cat.astype(np.int32)
    truth, pbase, ebase = {k: [] for k in blocks[0]["truth"]}, 0, 0
    for b in blocks:
        t = b["truth"]
        for k, v in t.items():
            if k in ("hit_particle", "seed_particle"):
                v = np.where(v >= 0, v + pbase, v)
            elif k == "part_ev":
                v = v + ebase
            truth[k].append(v)
        pbase += t["part_ev"].size
        ebase += b["n_events"]
    out["truth"] = {k: np.concatenate(v) for k, v in truth.items()}
    return out


def take_events(data, n):
    """First n events of a generated dict (truth tables kept whole)."""
    if n >= data["n_events"]:
        return data
    nh, ns = int(data["hit_offsets"][n]), int(data["seed_offsets"][n])
    out = dict(n_events=n, hit_offsets=data["hit_offsets"][: n + 1].copy(), seed_offsets=data["seed_offsets"][: n + 1].copy())
    out["hits"] = {k: v[:nh].copy() for k, v in data["hits"].items()}
    out["seeds"] = {k: v[:ns].copy() for k, v in data["seeds"].items()}
    if "truth" in data:
        t = dict(data["truth"])
        t["hit_particle"] = t["hit_particle"][:nh]
        t["seed_particle"] = t["seed_particle"][:ns]
        out["truth"] = t
    return out


def _gen_one(args):
    cfg_index, block, nev, dtype_name, seed_override = args
    cfg = C.CONFIGS[cfg_index]
    if seed_override is not None:
        cfg = _with_seed(cfg, seed_override)
    return generate_block(cfg, block, nev, _block_seq(cfg, block), dtype=np.dtype(dtype_name).type)


def _with_seed(cfg, seed):
    import copy
    c = copy.copy(cfg)
    c.seed = seed
    return c


def generate(cfg_index: int, n_events: int | None = None, first_block: int = 0, dtype=np.float32,
             workers: int = 1, seed: int | None = None):
    """Generate `n_events` events of BASELINE config `cfg_index`, starting at RNG block `first_block`.

    Whole blocks are generated and the result is cut to the first `n_events` events, so a prefix of a config
    is always the same bytes whatever `n_events` is.  `seed` overrides the config's seed (per-rank shards).
    """
    cfg = C.CONFIGS[cfg_index]
    if n_events is None:
        n_events = cfg.n_events
    B = block_size(cfg)
    nb = -(-n_events // B)
    jobs = [(cfg_index, first_block + b, B, np.dtype(dtype).name, seed) for b in range(nb)]
    if workers > 1 and nb > 1:
        import multiprocessing as mp
        with mp.get_context("spawn").Pool(min(workers, nb)) as pool:
            blocks = pool.map(_gen_one, jobs, chunksize=1)
    else:
        blocks = [_gen_one(j) for j in jobs]
    return take_events(concat(blocks), n_events)


def with_clone_seeds(d: dict, every: int = 3, seed: int = 7) -> dict:
    """Every `every`-th seed of an event once more at the end of the event, slightly displaced: a second SciFi segment of
    the same particle, which finds the same UT hits -- the case clone killing exists for.  Input recipe only."""
    rng = np.random.default_rng(seed)
    so = d["seed_offsets"]
    parts, new_so = {k: [] for k in d["seeds"]}, [0]
    for e in range(d["n_events"]):
        a, b = int(so[e]), int(so[e + 1])
        dup = np.arange(a, b)[::every]
        dx = rng.normal(0, 0.05, len(dup))
        dq = rng.normal(0, 0.002, len(dup))
        for k, v in d["seeds"].items():
            c = v[dup].copy()
            if k == "x":
                c = (c + dx).astype(v.dtype)
            if k == "qop":
                c = (c * (1 + dq)).astype(v.dtype)
            parts[k] += [v[a:b], c]
        new_so.append(new_so[-1] + (b - a) + len(dup))
    return dict(d, seeds={k: np.concatenate(v) for k, v in parts.items()}, seed_offsets=np.array(new_so, dtype=np.int32))


def with_hit_jitter(d: dict, seed: int = 11, dz: float = 2.0, shrink: float = 20.0) -> dict:
    """Per-hit z, weight and y range that differ from hit to hit (ds.h allows all three): z = plane z + U(-dz, dz), w drawn
    from three values (1/0.054^2, 1/0.08^2, 1/0.03^2), [ymin, ymax] shrunk by U(0, shrink) on either side inside the sector.
    The generated configurations give every hit of a layer the same z and w and the full sector range, which leaves the
    per-hit reads of the kernels (and of the oracle) undiscriminated; this transform is the input of the tests that close
    that.  Input recipe only."""
    rng = np.random.default_rng(seed)
    h = d["hits"]
    n = len(h["id"])
    dt = h["x0"].dtype
    wvals = np.array([1.0 / 0.054 ** 2, 1.0 / 0.08 ** 2, 1.0 / 0.03 ** 2])
    hits = dict(h)
    hits["z"] = (h["z"].astype(np.float64) + rng.uniform(-dz, dz, n)).astype(dt)
    hits["w"] = wvals[rng.integers(0, 3, n)].astype(dt)
    hits["ymin"] = (h["ymin"].astype(np.float64) + rng.uniform(0.0, shrink, n)).astype(dt)
    hits["ymax"] = (h["ymax"].astype(np.float64) - rng.uniform(0.0, shrink, n)).astype(dt)
    return dict(d, hits=hits)
