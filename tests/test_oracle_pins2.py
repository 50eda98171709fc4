"""More pins of the CPU oracle (round 2): the pieces a one-line mutation of oracle/ds_oracle.c used to survive.  CPU only.

Each test names the mutant it kills (checked with a mutated copy of the oracle while writing the tests):

  M1  better(): "more hits wins" inverted                               -> test_tie_more_hits_wins
  M2  better(): id order (id3, id0, id1, id2) changed to (2, 1, 0, 3)   -> test_tie_id3_decides_first, test_tie_id1_before_id2
  M3  ndf = nhits + 1 - 2 changed to nhits + 1 - 1                      -> test_chi2_cut_sits_at_ndf_nhits_minus_one
  M4  NN inputs v[0] <-> v[1] or v[6] <-> v[7] swapped                  -> test_mlp_inputs_in_the_order_of_the_paper
  M5  upper y tolerance ymax + y_tol changed to ymax                    -> test_y_compatibility_upper_side
  M6  DOCA cut < changed to <=, z cuts <= changed to <                  -> test_vertex_cut_comparison_operators
  M7  window inclusion d <= w changed to d < w; M8 chi2 / ndf <= max changed to <
                                                                        -> test_inclusive_window_and_chi2_cut_on_exact_numbers
  M9  mass windows < changed to <=                                      -> test_mass_window_is_strict
  M13 magnet-point weight w_mag replaced by 1; M16 trajectory through the first hit with the plane z instead of the hit's z;
  M17 / M18 fit with another hit's weight / the plane z instead of the hit's own
                                                                        -> test_per_hit_z_and_weight_are_the_ones_used

The tie tests run on a toy geometry whose numbers are small integers and dyadic fractions, so that every sum of the fit is
exact in binary floating point and "equal scores" means bit-equal (A-9: ties -> more hits -> smaller (id3, id0, id1, id2)).
The proton-assignment tie of A-15 (equal momenta) has no observable: with |p_a| = |p_b| both assignments give the same
E_1 + E_2 and the same momentum sum, hence the same m_ppi; it is left unpinned on purpose.
"""
import math

import numpy as np
import pytest

from gen import constants as C
from oracle import ds_oracle as O

G, P = C.GEOMETRY, C.PARAMS

# ---- toy geometry: planes at z = -2, -1, 1, 2, magnet at 4, seed state given at 8, z_ref = 0, no stereo ------------------
TG = dict(G, z_layer=(-2.0, -1.0, 1.0, 2.0), dxdy=(0.0, 0.0, 0.0, 0.0), z_seed=8.0, z_ref=0.0, zmag_c=(4.0, 0.0, 0.0, 0.0), kick=1.0)
TP = dict(P, w0_a=4.0, w0_b=0.0, w1_a=0.5, w1_b=0.0, w_mag=1.0, miss_penalty=0.0)
SEED0 = dict(x=np.zeros(1), y=np.zeros(1), tx=np.zeros(1), ty=np.zeros(1), qop=np.zeros(1), chi2=np.zeros(1))


def toy_hits(rows):
    """rows: (layer, x, seq).  y = 0 lies in sector 7 = [0, 100]; weight 1; z = plane z."""
    lay = np.array([r[0] for r in rows])
    n = len(rows)
    return dict(x0=np.array([r[1] for r in rows], dtype=np.float64), z=np.asarray(TG["z_layer"])[lay], ymin=np.zeros(n),
                ymax=np.full(n, 100.0), w=np.ones(n), id=(np.array([r[2] for r in rows]) | (7 << 20) | (lay << 24)).astype(np.int32))


def toy_run(rows, orc_mlp, params=TP):
    return O.reconstruct(toy_hits(rows), [0, len(rows)], SEED0, [0, 1], TG, params, orc_mlp)


def line_through(x3):
    """Hits of UTaX, UTaU, UTbV exactly on the line through (x3 at z = 2) and the magnet point (0 at z = 4)."""
    return [x3 * (4.0 - z) / 2.0 for z in (-2.0, -1.0, 1.0)]


def test_tie_more_hits_wins(orc_mlp):
    """Kills M1.  With miss_penalty = 0 a perfect 4-hit candidate (first hit at x = 2: x = 4 - z through 6, 5, 3, 2 and the
    magnet point 0; S = 5, Sz = 4, Szz = 26, Sx = 16, Sxz = -10, D = 114, b = -1, a = 4, every residual exactly 0) and a perfect
    3-hit candidate have the same score 0: the one with more hits is the track, whichever is met first and whatever the ids."""
    for x3b, seq_b in ((0.0, 1), (3.0, 1), (0.0, 99), (3.0, 99)):    # the 3-hit one: closer / farther, smaller / larger ids
        xa, xb = line_through(2.0), line_through(x3b)
        rows = [(3, 2.0, 50), (0, xa[0], 51), (1, xa[1], 52), (2, xa[2], 53),
                (3, x3b, seq_b), (0, xb[0], seq_b + 1), (1, xb[1], seq_b + 2)]
        r = toy_run(rows, orc_mlp)
        assert r["found"][0] and r["chi2"][0] == 0.0 and r["nhits"][0] == 4 and r["hit"][0].tolist() == [1, 2, 3, 0]
        assert r["x"][0] == 4.0 and r["tx"][0] == -1.0
        # and with the penalty of A-9 back in place the scores differ (0 against 4): the same track
        assert toy_run(rows, orc_mlp, dict(TP, miss_penalty=4.0))["hit"][0].tolist() == [1, 2, 3, 0]


def test_tie_id3_decides_first(orc_mlp):
    """Kills M2 (first half).  Two mirror-image perfect 4-hit candidates (first hits at x = +2 and x = -2): equal score, equal
    hits.  The one whose UTbX hit has the smaller id wins although its other three ids are the larger ones."""
    for seq_p, seq_q in ((1, 2), (2, 1)):
        xp, xq = line_through(2.0), line_through(-2.0)
        rows = [(3, 2.0, seq_p), (0, xp[0], 30), (1, xp[1], 31), (2, xp[2], 32),
                (3, -2.0, seq_q), (0, xq[0], 10), (1, xq[1], 11), (2, xq[2], 12)]
        r = toy_run(rows, orc_mlp)
        want = [1, 2, 3, 0] if seq_p < seq_q else [5, 6, 7, 4]
        assert r["found"][0] and r["chi2"][0] == 0.0 and r["hit"][0].tolist() == want
        assert r["edge"][0] == 1                     # best and runner-up have the same score: the seed is on the edge list (A-16)


def test_tie_id1_before_id2(orc_mlp):
    """Kills M2 (second half).  One first hit (x = 0), one UTaX hit (x = 0), two UTaU hits at +r / -r and two UTbV hits at
    +r / -r.  The four combinations fall in two mirror classes of bit-equal chi2; inside the better class the candidates are
    (u, v) and (u', v') with id(u) < id(u') and id(v) > id(v'): (id3, id0 equal) id1 is compared before id2, so (u, v) wins."""
    r_ = 0.25
    z = np.array([-2.0, -1.0, 1.0, 2.0, 4.0])

    def chi2(s1, s2):
        x = np.array([0.0, s1 * r_, s2 * r_, 0.0, 0.0])
        A = np.stack([np.ones(5), z], axis=1)
        sol = np.linalg.lstsq(A, x, rcond=None)[0]
        return float(((x - A @ sol) ** 2).sum())
    same, opp = chi2(1, 1), chi2(1, -1)
    assert abs(same - opp) > 1e-3                    # the two classes are well separated
    s2 = 1 if same < opp else -1                     # better class: (+, s2) and (-, -s2)
    # rows: 0 UTbX, 1 UTaX, 2 u(+r), 3 u'(-r), 4 v(s2 r), 5 v'(-s2 r); id(u) = 20 < id(u') = 21, id(v) = 41 > id(v') = 40
    rows = [(3, 0.0, 1), (0, 0.0, 2), (1, r_, 20), (1, -r_, 21), (2, s2 * r_, 41), (2, -s2 * r_, 40)]
    r = toy_run(rows, orc_mlp)
    assert r["found"][0] and r["nhits"][0] == 4 and r["chi2"][0] == pytest.approx(min(same, opp), rel=1e-6)
    assert r["hit"][0].tolist() == [1, 2, 4, 0] and r["edge"][0] == 1
    # ids of the UTaU pair exchanged: now (u', v') holds the smaller id1
    rows = [(3, 0.0, 1), (0, 0.0, 2), (1, r_, 21), (1, -r_, 20), (2, s2 * r_, 41), (2, -s2 * r_, 40)]
    assert toy_run(rows, orc_mlp)["hit"][0].tolist() == [1, 3, 5, 0]


# ---- helpers on the real geometry (as in test_oracle_pins.py) -----------------------------------------------------------------
def mk_hits(rows, w=None, z=None):
    """rows: (layer, x_at_track_y, y, seq)."""
    dxdy = np.asarray(G["dxdy"])
    lay = np.array([r[0] for r in rows])
    x = np.array([r[1] for r in rows], dtype=np.float64)
    y = np.array([r[2] for r in rows], dtype=np.float64)
    seq = np.array([r[3] for r in rows])
    sec = np.clip(np.floor((y + 700.0) / 100.0).astype(int), 0, 13)
    return dict(x0=x - y * dxdy[lay], z=np.asarray(G["z_layer"])[lay] if z is None else np.asarray(z, dtype=np.float64),
                ymin=-700.0 + 100.0 * sec, ymax=-600.0 + 100.0 * sec,
                w=np.full(len(rows), C.W_HIT) if w is None else np.asarray(w, dtype=np.float64),
                id=(seq | (sec << 20) | (lay << 24)).astype(np.int32))


def one_seed(x=300.0, y=120.0, tx=0.05, ty=0.01, qop=0.1, chi2=1.0):
    return dict(x=np.array([x]), y=np.array([y]), tx=np.array([tx]), ty=np.array([ty]), qop=np.array([qop]), chi2=np.array([chi2]))


def predicted(seed):
    ex = O.extrapolate(G, P, *(float(seed[k][0]) for k in ("x", "y", "tx", "ty", "qop")))
    return ex, [ex["x_m"] + ex["tx_pred"] * (G["z_layer"][l] - ex["z_m"]) for l in range(4)]


def wls(z, x, w, z_ref):
    """Weighted straight-line fit by numpy.linalg.lstsq: a, b, chi2."""
    z, x, w = (np.asarray(v, dtype=np.float64) for v in (z, x, w))
    A = np.stack([np.ones(len(z)), z - z_ref], axis=1) * np.sqrt(w)[:, None]
    sol = np.linalg.lstsq(A, x * np.sqrt(w), rcond=None)[0]
    res = x - sol[0] - sol[1] * (z - z_ref)
    return float(sol[0]), float(sol[1]), float((w * res * res).sum())


def test_chi2_cut_sits_at_ndf_nhits_minus_one(orc_mlp):
    """Kills M3.  SURVEY O-S5: ndf = n_hits + 1 - 2 (n_hits hits + the magnet point, two fitted parameters).  A single
    candidate whose chi2 is computed here with numpy.linalg.lstsq; the cut chi2 / ndf <= chi2ndf_max is placed 1e-3 above
    and below chi2 / ndf for ndf = 3 (four hits) and ndf = 2 (three hits)."""
    seed = one_seed()
    ex, xs = predicted(seed)
    for drop in (None, 1, 2):
        offs = [0.11, -0.07, 0.05, 0.0]                        # residual pattern in mm (first hit on the prediction)
        rows = [(l, xs[l] + offs[l], ex["y_l"][l], l) for l in range(4) if l != drop]
        nh = len(rows)
        zz = [G["z_layer"][r[0]] for r in rows] + [ex["z_m"]]
        xx = [r[1] for r in rows] + [ex["x_m"]]
        ww = [C.W_HIT] * nh + [P["w_mag"]]
        _, _, c2 = wls(zz, xx, ww, G["z_ref"])
        assert c2 > 0.3
        ndf = nh - 1
        for f, ok in ((1 + 1e-3, True), (1 - 1e-3, False)):
            r = O.reconstruct(mk_hits(rows), [0, nh], seed, [0, 1], G, dict(P, chi2ndf_max=f * c2 / ndf), orc_mlp)
            assert bool(r["found"][0]) == ok, (drop, f)
            if ok:
                assert r["nhits"][0] == nh and r["chi2"][0] == pytest.approx(c2, rel=1e-5)


def test_mlp_inputs_in_the_order_of_the_paper(orc_mlp):
    """Kills M4.  P:121: the NN takes the downstream track state (x, y, tx, ty, q/p), its chi2, then the SciFi q/p and
    chi2.  A network that passes input k through unchanged (two ReLU units +f_k, -f_k recombined: t = f_k) is run through
    O.reconstruct on one hand-made track; the score must be sigmoid((v_k - mu_k) / sigma_k) with v_k worked out here from
    the hits (numpy.linalg.lstsq) and the seed, for k = 0..7."""
    seed = one_seed(x=310.0, y=-140.0, tx=0.045, ty=-0.012, qop=0.125, chi2=1.7)
    ex, xs = predicted(seed)
    # hits on a line a little steeper than predicted (so that the track q/p differs from the seed's) with small residuals
    offs = [0.30 + 0.04, 0.26 - 0.03, 0.06 + 0.05, 0.0]
    rows = [(l, xs[l] + offs[l], ex["y_l"][l], l) for l in range(4)]
    a, b, c2 = wls([G["z_layer"][l] for l in range(4)] + [ex["z_m"]], [r[1] for r in rows] + [ex["x_m"]],
                   [C.W_HIT] * 4 + [P["w_mag"]], G["z_ref"])
    ys, tys, txs = float(seed["y"][0]), float(seed["ty"][0]), float(seed["tx"][0])
    v = [a, ys + tys * (G["z_ref"] - G["z_seed"]), b, tys, (txs - b) / G["kick"], c2, float(seed["qop"][0]), float(seed["chi2"][0])]
    assert abs(v[4] - v[6]) > 1e-4 * abs(v[6]) and abs(v[5] - v[7]) > 0.1 and len({round(abs(t), 6) for t in v}) == 8
    mu, sig = np.array(C.MLP_MU), np.array(C.MLP_SIGMA)
    for k in range(8):
        w = dict(W1=np.zeros((32, 8)), b1=np.zeros(32), W2=np.zeros((16, 32)), b2=np.zeros(16), W3=np.zeros((1, 16)),
                 b3=np.zeros(1), mu=mu, inv_sigma=1.0 / sig)
        w["W1"][0, k], w["W1"][1, k] = 1.0, -1.0
        w["W2"][0, 0] = w["W2"][1, 1] = 1.0
        w["W3"][0, 0], w["W3"][0, 1] = 1.0, -1.0
        r = O.reconstruct(mk_hits(rows), [0, 4], seed, [0, 1], G, dict(P, chi2ndf_max=1e9), O.Mlp(w))
        assert r["found"][0] and r["nhits"][0] == 4
        want = 1.0 / (1.0 + math.exp(-(v[k] - mu[k]) / sig[k]))
        # the oracle feeds the track values as stored (fp32): 6e-8 relative on v_k
        assert r["score_f64"][0] == pytest.approx(want, rel=2e-6), k
    assert [r[kk][0] for kk in ("x", "y", "tx", "ty", "qop", "chi2")] == pytest.approx(v[:6], rel=1e-5)


def test_y_compatibility_upper_side(orc_mlp):
    """Kills M5.  O-S3: y-compatible iff ymin - y_tol <= y <= ymax + y_tol.  The UTbX hit lives in the sector BELOW the
    boundary yb = 200 (its ymax = 200); the track passes dy above the boundary: accepted up to y_tol = 3 mm."""
    yb = 200.0
    for dy, inside in ((2.9, True), (3.1, False)):
        s2 = one_seed(y=yb + dy - 0.01 * (G["z_layer"][3] - G["z_seed"]))          # track y at UTbX = yb + dy
        ex, xs = predicted(s2)
        assert ex["y_l"][3] == pytest.approx(yb + dy, abs=1e-9)
        tx_c = (xs[3] - ex["x_m"]) / (G["z_layer"][3] - ex["z_m"])
        rows = [(3, xs[3], yb - 10.0, 1)] + [(l, ex["x_m"] + tx_c * (G["z_layer"][l] - ex["z_m"]), ex["y_l"][l], 100 + l) for l in range(3)]
        h = mk_hits(rows)
        h["x0"][0] = xs[3]                                                          # UTbX has no stereo: x0 = x
        assert h["ymax"][0] == yb
        r = O.reconstruct(h, [0, 4], s2, [0, 1], G, P, orc_mlp)
        assert bool(r["found"][0]) == inside
    # the same in a refined window: the UTaU hit one sector below the track
    for dy, inside in ((2.9, True), (3.1, False)):
        s2 = one_seed(y=yb + dy - 0.01 * (G["z_layer"][1] - G["z_seed"]))
        ex, xs = predicted(s2)
        rows = [(l, xs[l], ex["y_l"][l], l) for l in range(4)]
        h = mk_hits(rows)
        h["ymin"][1], h["ymax"][1] = yb - 100.0, yb                               # keep x0 (computed at the track's y), move the strip
        r = O.reconstruct(h, [0, 4], s2, [0, 1], G, P, orc_mlp)
        assert r["found"][0] and (r["hit"][0, 1] >= 0) == inside and r["nhits"][0] == (4 if inside else 3)


def test_vertex_cut_comparison_operators():
    """Kills M6.  SURVEY O-S9: pass iff DOCA < doca_max and zv_min <= z_v <= zv_max.  The cut values are set to the very
    numbers the pair produces."""
    trk = dict(x=np.array([0.0, 0.0]), y=np.array([0.0, 1.25]), tx=np.array([0.125, -0.125]), ty=np.array([0.0, 0.0]),
               qop=np.array([0.2, -0.25]), keep=np.array([1, 1]))
    loose = dict(P, zv_min=-1e9, zv_max=1e9, dm_ks=1e9, dm_lambda=1e9, doca_max=1e9)
    v = O.vertex(trk, [0, 2], G, loose)
    assert v["n"] == 1
    doca, z = float(v["doca"][0]), float(v["z"][0])
    assert doca == pytest.approx(1.25, rel=1e-12) and z == pytest.approx(G["z_ref"], abs=1e-9)
    assert O.vertex(trk, [0, 2], G, dict(loose, doca_max=doca))["n"] == 0                      # DOCA < doca_max: strict
    assert O.vertex(trk, [0, 2], G, dict(loose, doca_max=np.nextafter(doca, 2 * doca)))["n"] == 1
    assert O.vertex(trk, [0, 2], G, dict(loose, zv_min=z))["n"] == 1                           # zv_min <= z: inclusive
    assert O.vertex(trk, [0, 2], G, dict(loose, zv_min=np.nextafter(z, 2 * z)))["n"] == 0
    assert O.vertex(trk, [0, 2], G, dict(loose, zv_max=z))["n"] == 1                           # z <= zv_max: inclusive
    assert O.vertex(trk, [0, 2], G, dict(loose, zv_max=np.nextafter(z, 0.0)))["n"] == 0
    # mass windows: |m - m0| < dm, strict
    m = float(v["m_pipi"][0])
    tight = dict(loose, dm_lambda=0.0, m_ks=m - 7.0)
    assert O.vertex(trk, [0, 2], G, dict(tight, dm_ks=7.0 * (1 + 1e-9)))["n"] == 1
    assert O.vertex(trk, [0, 2], G, dict(tight, dm_ks=7.0 * (1 - 1e-9)))["n"] == 0


def test_inclusive_window_and_chi2_cut_on_exact_numbers(orc_mlp):
    """O-S3 / O-S4: |x_hit - x_centre| <= w (inclusive); O-S6: chi2 / ndf <= chi2ndf_max (inclusive).  Toy geometry, exact
    arithmetic: a hit exactly w away from the window centre is inside; a candidate exactly on the cut is accepted."""
    # first window: w0 = 4, UTbX hit at x = 4 (centre 0); its partners on the line through the magnet point: 12, 10, 6
    xa = line_through(4.0)
    rows = [(3, 4.0, 1), (0, xa[0], 2), (1, xa[1], 3), (2, xa[2], 4)]
    assert toy_run(rows, orc_mlp)["found"][0]
    assert not toy_run(rows, orc_mlp, dict(TP, w0_a=np.nextafter(4.0, 0.0)))["found"][0]
    # refined window: w1 = 0.5, the UTaU hit exactly 0.5 off its prediction (10.5 instead of 10)
    rows = [(3, 4.0, 1), (0, xa[0], 2), (1, xa[1] + 0.5, 3), (2, xa[2], 4)]
    r = toy_run(rows, orc_mlp, dict(TP, chi2ndf_max=1e9))
    assert r["found"][0] and r["hit"][0, 1] == 2 and r["nhits"][0] == 4
    r = toy_run(rows, orc_mlp, dict(TP, chi2ndf_max=1e9, w1_a=np.nextafter(0.5, 0.0)))
    assert r["found"][0] and r["hit"][0, 1] == -1 and r["nhits"][0] == 3
    # chi2 cut: hits at (+r, -r, -r, +r), z = (-2, -1, 1, 2), unit weights, magnet point switched off (w_mag = 0):
    # S = 4, Sz = 0, Sx = 0, Sxz = 0 -> a = b = 0, chi2 = 4 r^2 = 0.25 exactly, ndf = 3
    q = 0.25
    rows = [(3, q, 1), (0, q, 2), (1, -q, 3), (2, -q, 4)]
    wide = dict(TP, w1_a=2.0, w_mag=0.0)
    r = toy_run(rows, orc_mlp, dict(wide, chi2ndf_max=0.25 / 3.0))
    assert r["found"][0] and r["chi2"][0] == 0.25 and r["nhits"][0] == 4 and r["x"][0] == 0.0 and r["tx"][0] == 0.0
    assert not toy_run(rows, orc_mlp, dict(wide, chi2ndf_max=np.nextafter(0.25 / 3.0, 0.0)))["found"][0]


def test_mass_window_is_strict():
    """flags bit0 = |m_pipi - m_ks| < dm_ks, bit1 = |m_ppi - m_lambda| < dm_lambda (strict, SURVEY O-S9): with m_ks = 0 the
    distance is m_pipi itself."""
    trk = dict(x=np.array([0.0, 0.0]), y=np.array([0.0, 1.25]), tx=np.array([0.125, -0.125]), ty=np.array([0.0, 0.0]),
               qop=np.array([0.2, -0.25]), keep=np.array([1, 1]))
    loose = dict(P, zv_min=-1e9, zv_max=1e9, doca_max=1e9, dm_ks=1e9, dm_lambda=1e9)
    v = O.vertex(trk, [0, 2], G, loose)
    m1, m2 = float(v["m_pipi"][0]), float(v["m_ppi"][0])
    assert v["flags"][0] == 3 and m2 > m1 > 2 * 139.57
    only1 = dict(loose, m_ks=0.0, dm_lambda=0.0)
    assert O.vertex(trk, [0, 2], G, dict(only1, dm_ks=m1))["n"] == 0
    v1 = O.vertex(trk, [0, 2], G, dict(only1, dm_ks=np.nextafter(m1, 2 * m1)))
    assert v1["n"] == 1 and v1["flags"][0] == 1
    only2 = dict(loose, m_lambda=0.0, dm_ks=0.0)
    assert O.vertex(trk, [0, 2], G, dict(only2, dm_lambda=m2))["n"] == 0
    v2 = O.vertex(trk, [0, 2], G, dict(only2, dm_lambda=np.nextafter(m2, 2 * m2)))
    assert v2["n"] == 1 and v2["flags"][0] == 2


def test_per_hit_z_and_weight_are_the_ones_used(orc_mlp):
    """A hit carries its own z and weight (BASELINE cfg0: "hits are fp32 (x at y=0, z, ymin, ymax, weight)").  O-S4: the
    trajectory through the first hit uses that hit's z; O-S5: the fit uses every hit's own z and w and the weight w_mag for
    the magnet point.  Hits displaced in z by up to 2 mm, four different weights, w_mag = 0.25: a, b, chi2 against
    numpy.linalg.lstsq on exactly those numbers; and a UTaX hit placed on the edge of the refined window that the
    first hit's own z predicts (with the plane's z instead, the centre moves by ~0.2 mm and one of the two flips)."""
    seed = one_seed(x=320.0, y=90.0, tx=0.06, ty=0.008, qop=0.15)
    ex, xs = predicted(seed)
    pp = dict(P, w_mag=0.25, chi2ndf_max=1e9)
    dz = [1.9, -1.3, 0.8, -1.7]
    ww = [1.0 / 0.054 ** 2, 1.0 / 0.08 ** 2, 1.0 / 0.03 ** 2, 1.0 / 0.1 ** 2]
    zh = [G["z_layer"][l] + dz[l] for l in range(4)]
    offs = [0.21, -0.17, 0.12, 0.0]
    rows = [(l, xs[l] + offs[l], ex["y_l"][l], l) for l in range(4)]
    r = O.reconstruct(mk_hits(rows, w=ww, z=zh), [0, 4], seed, [0, 1], G, pp, orc_mlp)
    a, b, c2 = wls(zh + [ex["z_m"]], [q[1] for q in rows] + [ex["x_m"]], ww + [pp["w_mag"]], G["z_ref"])
    assert r["found"][0] and r["nhits"][0] == 4
    assert r["x"][0] == pytest.approx(a, rel=1e-6) and r["tx"][0] == pytest.approx(b, rel=1e-6) and r["chi2"][0] == pytest.approx(c2, rel=1e-5)
    # the same hits with the plane z and a common weight give something else (the per-hit values matter here)
    a0, b0, c0 = wls(list(G["z_layer"]) + [ex["z_m"]], [q[1] for q in rows] + [ex["x_m"]], [ww[0]] * 4 + [pp["w_mag"]], G["z_ref"])
    assert abs(c0 - c2) > 0.2 * c2
    # refined-window centre from the first hit's own z
    z3 = zh[3]
    tx_c = (xs[3] - ex["x_m"]) / (z3 - ex["z_m"])
    tx_plane = (xs[3] - ex["x_m"]) / (G["z_layer"][3] - ex["z_m"])
    xp0 = ex["x_m"] + tx_c * (G["z_layer"][0] - ex["z_m"])
    assert abs(xp0 - (ex["x_m"] + tx_plane * (G["z_layer"][0] - ex["z_m"]))) > 0.05
    for sign in (+1, -1):
        for f, inside in ((1 - 1e-3, True), (1 + 1e-3, False)):
            rr = list(rows)
            rr[0] = (0, xp0 + sign * f * ex["w1"], ex["y_l"][0], 0)
            r = O.reconstruct(mk_hits(rr, w=ww, z=zh), [0, 4], seed, [0, 1], G, pp, orc_mlp)
            assert r["found"][0] and (r["hit"][0, 0] >= 0) == inside, (sign, f)
