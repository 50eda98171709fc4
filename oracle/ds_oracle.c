/*
 * ds_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU restatement of the HLT1 Downstream hot path of arXiv:2503.13092 (LHCb, "A Downstream and
 * vertexing algorithm for Long Lived Particles (LLP) selection at the first High level trigger"), written from
 * the paper text (`P:n` = /root/reference/PAPER.md line n) and the readings listed in DESIGN.md ("A-n").
 * It shares no code, header, table or constant with the CUDA library; only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.
 *
 * Every search is the plain definition: a linear scan over ALL hits of the event (no sorting, no sectors, no
 * binary search); every pair list is the double loop.  All arithmetic is IEEE double; inputs are the caller's
 * fp32/int32 values promoted exactly (the Python wrapper does astype(float64)).
 *
 * Steps (paper order):
 *   O-S2  magnet point + first-window prediction            P:93, P:95   (thin-kick model: BASELINE cfg0)
 *   O-S3  first window in UTbX, <= 10 closest hits
 *   O-S4  per first hit: line through (hit, magnet point), refined windows in UTaX/UTaU/UTbV,
 *         closest 1 / 2 / 2 hits
 *   O-S5  candidate fit + chi2                               P:115, P:121 (chi2 is a NN input), reading A-8
 *   O-S6  best candidate per SciFi seed (same-seed clone kill) P:115, reading A-9
 *   O-S7  ghost-killer FFNN: 8 inputs, ReLU hidden, sigmoid  P:121        (8->32->16->1: BASELINE cfg0)
 *   O-S8  opposite-charge pairs
 *   O-S9  closest approach of two trajectories = vertex      P:253-P:269, Eq. 4 P:266 with gamma = 0 (A-20)
 *
 * Parity unpinned (stated in DESIGN.md): the numeric VALUES of window sizes, cuts, penalty and NN normalisation
 * are free parameters the paper does not print; parity is defined with both sides given the same values.
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC -o libds_oracle.so ds_oracle.c -lm     (oracle/build.py)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    double z_layer[4];   /* plane z of UTaX, UTaU, UTbV, UTbX            */
    double dxdy[4];      /* tan(stereo angle): x_hit(y) = x0 + y*dxdy    (A-1)             */
    double z_seed;       /* z at which the SciFi seed state is given                        */
    double z_ref;        /* z0 = midpoint of the UT station           */
    double zmag_c[4];    /* z_mag = c0 + c1 ty^2 + c2 tx^2 + c3 qop^2     (A-3)       */
    double kick;         /* K [GeV]: tx_UT = tx_seed - K*qop_seed         (cfg0 kick model) */
} orc_geom;

typedef struct {
    double w0_a, w0_b, w0_max;   /* first window  w0 = min(w0_max, w0_a + w0_b |qop|)   (P:95,  A-5) */
    double w1_a, w1_b;           /* refined window w1 = w1_a + w1_b |qop|               (A-5) */
    double y_tol;
    double w_mag;                /* weight of the magnet-point pseudo-measurement       (A-8)        */
    double chi2ndf_max, miss_penalty;                                                /* (A-9)        */
    int32_t min_hits, max_first_hits;                                                /* (A-6) */
    double mlp_thr;
    int32_t mlp_keep_above;      /* 1: keep if score > thr (cfg3); 0: keep if score < thr    */
    int32_t pad_;
    double doca_max, zv_min, zv_max;
    double m_pi, m_p, m_ks, m_lambda, dm_ks, dm_lambda;
    double n2_min;               /* |d_a x d_b|^2 floor                                 (A-14)       */
    double magnet_polarity;      /* MP of Eq. 3: +1 / -1; 0 = straight tracks (gamma = 0, A-20)      */
    double gamma_c0, gamma_c1;   /* gamma = -MP (c0 + c1 q/p[1/MeV]); paper: -1.5e-8, 9.3e-3 (Eq. 3, A-27)   */
    int32_t vtx_newton_iters;    /* Newton-Raphson iterations ("three")           (A-28)              */
    int32_t dv1;                 /* 1: Dv1 triplet search (P:107-P:111); 0: Dv0         */
    double edge_rel;             /* relative margin below which a decision is "edge" (1e-5)          */
} orc_params;

typedef struct {
    int32_t n_in, n_h1, n_h2, pad_;
    const double *W1, *b1;   /* [n_h1][n_in], [n_h1] */
    const double *W2, *b2;   /* [n_h2][n_h1], [n_h2] */
    const double *W3, *b3;   /* [n_h2], [1]          */
    const double *mu, *inv_sigma; /* [n_in]          */
} orc_mlp;

#define ID_LAYER(id) (((id) >> 24) & 3)

static double relm(double lhs, double rhs)
{
    double s = fabs(rhs);
    if (s < 1e-300) s = 1e-300;
    return fabs(lhs - rhs) / s;
}

/* ------------------------------------------------------------------------------------------------------------
 * O-S2  (magnet point from the seed state at the last SciFi station by straight-line extrapolation;
 *        first search window "as a function of momentum"; BASELINE cfg0: thin kick dtx = q*K/p)
 * out[12] = { z_m, x_m, y_m, y_0, y_1, y_2, y_3, tx_pred, xc_3, w0, w1, 0 }
 * ------------------------------------------------------------------------------------------------------------ */
void orc_extrapolate(const orc_geom *g, const orc_params *p, double xs, double ys, double txs, double tys,
                     double qop, double *out)
{
    double zm = g->zmag_c[0] + g->zmag_c[1] * tys * tys + g->zmag_c[2] * txs * txs + g->zmag_c[3] * qop * qop;
    double xm = xs + txs * (zm - g->z_seed);
    double ym = ys + tys * (zm - g->z_seed);
    int l;
    out[0] = zm; out[1] = xm; out[2] = ym;
    for (l = 0; l < 4; ++l) out[3 + l] = ys + tys * (g->z_layer[l] - g->z_seed);   /* ty unchanged by the kick */
    {
        double txp = txs - g->kick * qop;
        double w0 = p->w0_a + p->w0_b * fabs(qop);
        if (w0 > p->w0_max) w0 = p->w0_max;
        out[7] = txp;
        out[8] = xm + txp * (g->z_layer[3] - zm);
        out[9] = w0;
        out[10] = p->w1_a + p->w1_b * fabs(qop);
        out[11] = 0.0;
    }
}

/* ------------------------------------------------------------------------------------------------------------
 * O-S5  weighted straight-line fit x(z) = a + b (z - z_ref) and its chi2 (textbook weighted least squares).
 * ------------------------------------------------------------------------------------------------------------ */
void orc_fit_line(int n, const double *z, const double *x, const double *w, double z_ref,
                  double *a, double *b, double *chi2)
{
    double S = 0, Sz = 0, Szz = 0, Sx = 0, Sxz = 0, D, c2 = 0;
    int i;
    for (i = 0; i < n; ++i) {
        double dz = z[i] - z_ref;
        S += w[i]; Sz += w[i] * dz; Szz += w[i] * dz * dz; Sx += w[i] * x[i]; Sxz += w[i] * x[i] * dz;
    }
    D = S * Szz - Sz * Sz;
    *b = (S * Sxz - Sz * Sx) / D;
    *a = (Szz * Sx - Sz * Sxz) / D;
    for (i = 0; i < n; ++i) {
        double r = x[i] - *a - *b * (z[i] - z_ref);
        c2 += w[i] * r * r;
    }
    *chi2 = c2;
}

/* ------------------------------------------------------------------------------------------------------------
 * O-S7  feed-forward NN, ReLU hidden layers, sigmoid output.  v = raw inputs in the order of P:121:
 *       downstream (x, y, tx, ty, q/p, chi2), SciFi (q/p, chi2).
 * ------------------------------------------------------------------------------------------------------------ */
double orc_mlp_eval(const orc_mlp *m, const double *v)
{
    double f[64], h1[256], h2[256], t;
    int i, j;
    for (i = 0; i < m->n_in; ++i) f[i] = (v[i] - m->mu[i]) * m->inv_sigma[i];
    for (j = 0; j < m->n_h1; ++j) {
        t = m->b1[j];
        for (i = 0; i < m->n_in; ++i) t += m->W1[j * m->n_in + i] * f[i];
        h1[j] = t > 0.0 ? t : 0.0;
    }
    if (m->n_h2 > 0) {
        for (j = 0; j < m->n_h2; ++j) {
            t = m->b2[j];
            for (i = 0; i < m->n_h1; ++i) t += m->W2[j * m->n_h1 + i] * h1[i];
            h2[j] = t > 0.0 ? t : 0.0;
        }
        t = m->b3[0];
        for (i = 0; i < m->n_h2; ++i) t += m->W3[i] * h2[i];
    } else {            /* single hidden layer (the paper's 8 -> 14 -> 1): W3 acts on h1 */
        t = m->b3[0];
        for (i = 0; i < m->n_h1; ++i) t += m->W3[i] * h1[i];
    }
    return 1.0 / (1.0 + exp(-t));
}

/* ------------------------------------------------------------------------------------------------------------
 * O-S9  closest approach of two straight trajectories Traj_i(s) = (x_i, y_i, z_ref) + s (tx_i, ty_i, 1)
 *       (Eq. 4, with gamma = 0).  Textbook two-line solution.
 * out[8] = { vx, vy, vz, doca, |n|^2, s_a, s_b, 0 }.  Returns 0 if |n|^2 < n2_min (no vertex), else 1.
 * ------------------------------------------------------------------------------------------------------------ */
int orc_poca(double xa, double ya, double txa, double tya, double xb, double yb, double txb, double tyb,
             double z_ref, double n2_min, double *out)
{
    double da[3] = { txa, tya, 1.0 }, db[3] = { txb, tyb, 1.0 };
    double r[3] = { xa - xb, ya - yb, 0.0 };
    double n[3] = { da[1] * db[2] - da[2] * db[1], da[2] * db[0] - da[0] * db[2], da[0] * db[1] - da[1] * db[0] };
    double n2 = n[0] * n[0] + n[1] * n[1] + n[2] * n[2];
    double A, B, Cc, Dd, Ee, den, sa, sb, qa[3], qb[3], dq[3];
    int k;
    out[4] = n2;
    if (n2 < n2_min) return 0;
    A = da[0] * da[0] + da[1] * da[1] + da[2] * da[2];
    B = da[0] * db[0] + da[1] * db[1] + da[2] * db[2];
    Cc = db[0] * db[0] + db[1] * db[1] + db[2] * db[2];
    Dd = da[0] * r[0] + da[1] * r[1] + da[2] * r[2];
    Ee = db[0] * r[0] + db[1] * r[1] + db[2] * r[2];
    den = A * Cc - B * B;
    sa = (B * Ee - Cc * Dd) / den;
    sb = (A * Ee - B * Dd) / den;
    qa[0] = xa + sa * da[0]; qa[1] = ya + sa * da[1]; qa[2] = z_ref + sa * da[2];
    qb[0] = xb + sb * db[0]; qb[1] = yb + sb * db[1]; qb[2] = z_ref + sb * db[2];
    for (k = 0; k < 3; ++k) { out[k] = 0.5 * (qa[k] + qb[k]); dq[k] = qa[k] - qb[k]; }
    out[3] = sqrt(dq[0] * dq[0] + dq[1] * dq[1] + dq[2] * dq[2]);
    out[5] = sa; out[6] = sb; out[7] = 0.0;
    return 1;
}

/* ------------------------------------------------------------------------------------------------------------
 * O-S9c  closest approach of two curved trajectories
 *     Traj_i(z) = ( x_i + tx_i (z - z0) + gamma_i (z - z0)^2,  y_i + ty_i (z - z0),  z )          (Eq. 4)
 * by Newton-Raphson on F(u, v) = |Traj_a(z0 + u) - Traj_b(z0 + v)|^2: start at the straight-line solution
 * (orc_poca), then n_iter times (u, v) -= H^-1 grad F with the exact gradient and 2x2 Hessian (A-28).
 * out[10] = { vx, vy, vz, doca, |n|^2, u, v, |last step|, tx_a at vz, tx_b at vz }.  Returns 0 if the straight
 * lines are parallel (|n|^2 < n2_min, A-14), else 1.
 * ------------------------------------------------------------------------------------------------------------ */
int orc_poca_curved(double xa, double ya, double txa, double tya, double ga, double xb, double yb, double txb,
                    double tyb, double gb, double z_ref, double n2_min, int n_iter, double *out)
{
    double po[8], u, v, step = 0.0, qa[3], qb[3], dq[3];
    int it, k;
    if (!orc_poca(xa, ya, txa, tya, xb, yb, txb, tyb, z_ref, n2_min, po)) { out[4] = po[4]; return 0; }
    u = po[5]; v = po[6];
    for (it = 0; it < n_iter; ++it) {
        /* D = Traj_a - Traj_b; dD/du = Da, dD/dv = -Db */
        double D[3] = { xa + txa * u + ga * u * u - (xb + txb * v + gb * v * v), ya + tya * u - (yb + tyb * v), u - v };
        double Da[3] = { txa + 2.0 * ga * u, tya, 1.0 }, Db[3] = { txb + 2.0 * gb * v, tyb, 1.0 };
        /* F/2: gradient and Hessian */
        double gu = D[0] * Da[0] + D[1] * Da[1] + D[2] * Da[2];
        double gv = -(D[0] * Db[0] + D[1] * Db[1] + D[2] * Db[2]);
        double Huu = Da[0] * Da[0] + Da[1] * Da[1] + Da[2] * Da[2] + D[0] * 2.0 * ga;
        double Hvv = Db[0] * Db[0] + Db[1] * Db[1] + Db[2] * Db[2] - D[0] * 2.0 * gb;
        double Huv = -(Da[0] * Db[0] + Da[1] * Db[1] + Da[2] * Db[2]);
        double det = Huu * Hvv - Huv * Huv, du, dv;
        if (det == 0.0) break;
        du = -(Hvv * gu - Huv * gv) / det;
        dv = -(Huu * gv - Huv * gu) / det;
        u += du; v += dv;
        step = sqrt(du * du + dv * dv);
    }
    qa[0] = xa + txa * u + ga * u * u; qa[1] = ya + tya * u; qa[2] = z_ref + u;
    qb[0] = xb + txb * v + gb * v * v; qb[1] = yb + tyb * v; qb[2] = z_ref + v;
    for (k = 0; k < 3; ++k) { out[k] = 0.5 * (qa[k] + qb[k]); dq[k] = qa[k] - qb[k]; }
    out[3] = sqrt(dq[0] * dq[0] + dq[1] * dq[1] + dq[2] * dq[2]);
    out[4] = po[4]; out[5] = u; out[6] = v; out[7] = step;
    /* slope dx/dz of each track at the vertex z (Eq. 2: the slope the masses are computed with) */
    out[8] = txa + 2.0 * ga * (out[2] - z_ref);
    out[9] = txb + 2.0 * gb * (out[2] - z_ref);
    return 1;
}

/* gamma of Eq. 3; q/p given in 1/GeV, the parametrisation wants 1/MeV (A-27) */
double orc_gamma(const orc_params *p, double qop_gev)
{
    return -p->magnet_polarity * (p->gamma_c0 + p->gamma_c1 * (qop_gev / 1000.0));
}

/* invariant mass of two tracks with slopes (tx, ty), momenta p [MeV] and mass hypotheses m1, m2 [MeV] */
double orc_inv_mass(double tx1, double ty1, double p1, double m1, double tx2, double ty2, double p2, double m2)
{
    double n1 = sqrt(tx1 * tx1 + ty1 * ty1 + 1.0), n2 = sqrt(tx2 * tx2 + ty2 * ty2 + 1.0);
    double px = p1 * tx1 / n1 + p2 * tx2 / n2, py = p1 * ty1 / n1 + p2 * ty2 / n2, pz = p1 / n1 + p2 / n2;
    double E = sqrt(p1 * p1 + m1 * m1) + sqrt(p2 * p2 + m2 * m2);
    double M2 = E * E - (px * px + py * py + pz * pz);
    return M2 > 0.0 ? sqrt(M2) : 0.0;
}

/* ============================================================================================================
 *  Tracking: O-S2 .. O-S7 for one seed
 * ============================================================================================================ */
typedef struct { double d; int32_t id; int32_t idx; } cand_hit;   /* idx = index into the event's hit arrays */

static int closer(const cand_hit *a, const cand_hit *b)       /* (distance, id) order: "tie -> smaller id" */
{
    if (a->d != b->d) return a->d < b->d;
    return a->id < b->id;
}

/* Definition of a search window (O-S3 / O-S4): scan ALL hits of the event; a hit of layer `layer` is accepted iff
 * it is y-compatible (ymin - y_tol <= y <= ymax + y_tol) and |x0 + dxdy*y - xc| <= w.  The accepted hits are
 * returned sorted by (distance, id), at most `keep` of them.  *edge is set if any deciding comparison
 * has a relative margin below edge_rel (see header of orc_reconstruct). */
static int window_search(const orc_geom *g, const orc_params *p, int nh, const double *x0, const double *ymin,
                         const double *ymax, const int32_t *id, int layer, double y, double xc, double w, int keep,
                         cand_hit *out, cand_hit *scratch, int *edge, double *min_margin)
{
    int n = 0, h, i, j;
    const double eps = p->edge_rel;
    for (h = 0; h < nh; ++h) {
        double ylo, yhi, my, xh, d, mx;
        int in_y, in_x;
        if (ID_LAYER(id[h]) != layer) continue;
        ylo = ymin[h] - p->y_tol; yhi = ymax[h] + p->y_tol;
        in_y = (ylo <= y) && (y <= yhi);
        my = fmin(relm(y, ylo), relm(y, yhi));
        xh = x0[h] + g->dxdy[layer] * y;
        d = fabs(xh - xc);
        in_x = d <= w;
        mx = relm(d, w);
        /* a marginal comparison matters only if the other one does not robustly reject the hit */
        if (!(!in_x && mx >= eps) && my < eps) *edge = 1;
        if (!(!in_y && my >= eps) && mx < eps) *edge = 1;
        if (in_y && in_x) {
            if (mx < *min_margin) *min_margin = mx;
            if (my < *min_margin) *min_margin = my;
            scratch[n].d = d; scratch[n].id = id[h]; scratch[n].idx = h; ++n;
        }
    }
    /* insertion sort by (distance, id) */
    for (i = 1; i < n; ++i) {
        cand_hit t = scratch[i];
        for (j = i - 1; j >= 0 && closer(&t, &scratch[j]); --j) scratch[j + 1] = scratch[j];
        scratch[j + 1] = t;
    }
    if (n > keep) {                                  /* rank cut-off: k-th vs (k+1)-th closest (A-16) */
        double m = relm(scratch[keep - 1].d, scratch[keep].d);
        if (m < eps) *edge = 1;
        if (m < *min_margin) *min_margin = m;
        n = keep;
    }
    for (i = 0; i < n; ++i) out[i] = scratch[i];
    return n;
}

typedef struct {
    int found, nhits;
    int32_t hit[4];          /* event-local hit index per layer, -1 = none */
    int32_t hid[4];          /* hit id per layer, INT32_MAX = none          */
    double a, b, chi2, score;
} best_t;

static int better(const best_t *c, const best_t *best)   /* O-S6 order: score, more hits, (id3, id0, id1, id2) */
{
    static const int ord[4] = { 3, 0, 1, 2 };
    int k;
    if (!best->found) return 1;
    if (c->score != best->score) return c->score < best->score;
    if (c->nhits != best->nhits) return c->nhits > best->nhits;
    for (k = 0; k < 4; ++k)
        if (c->hid[ord[k]] != best->hid[ord[k]]) return c->hid[ord[k]] < best->hid[ord[k]];
    return 0;
}

/* One seed.  Hit arrays are those of the seed's event (nh entries).  trk[8] = x, y, tx, ty, qop, chi2, score, 0 */
static void reconstruct_seed(const orc_geom *g, const orc_params *p, const orc_mlp *mlp, int nh, const double *x0,
                             const double *hz, const double *ymin, const double *ymax, const double *hw,
                             const int32_t *id, double xs, double ys, double txs, double tys, double qop,
                             double chi2s, cand_hit *scratch, double *trk, int32_t *nhits_out, int32_t *hit_out,
                             int32_t *found_out, int32_t *keep_out, int32_t *edge_out, double *margin_out)
{
    double ex[12], zm, xm, txp, xc3, w0, w1, yl[4];
    cand_hit F64[64], *F = F64, C0[4], C1[4], C2[4];
    int nF, f, l, edge = 0, maxF = p->max_first_hits;
    double min_margin = 1e300, second_score = 1e300;
    const double eps = p->edge_rel;
    best_t best;
    memset(&best, 0, sizeof best);
    if (maxF > 64) maxF = 64;

    /* O-S2 */
    orc_extrapolate(g, p, xs, ys, txs, tys, qop, ex);
    zm = ex[0]; xm = ex[1]; txp = ex[7]; xc3 = ex[8]; w0 = ex[9]; w1 = ex[10];
    for (l = 0; l < 4; ++l) yl[l] = ex[3 + l];
    (void)txp;

    if (!p->dv1) {
        /* O-S3: first window in UTbX (layer 3), up to 10 closest */
        nF = window_search(g, p, nh, x0, ymin, ymax, id, 3, yl[3], xc3, w0, maxF, F, scratch, &edge, &min_margin);
    } else {
        /* Dv1 (P:107-P:111; A-32): no first window that assumes a track from the origin -- every UTbX hit of the
         * y-compatible sectors starts a triplet (UTbX hit, UTaX hit, magnet point) */
        F = (cand_hit *)malloc(sizeof(cand_hit) * (size_t)(nh > 0 ? nh : 1));
        nF = window_search(g, p, nh, x0, ymin, ymax, id, 3, yl[3], 0.0, 1e300, nh > 0 ? nh : 1, F, scratch, &edge, &min_margin);
    }

    for (f = 0; f < nF; ++f) {
        /* O-S4: new trajectory from the hit position and the magnet point (Fig. 7) */
        int hf = F[f].idx, n0, n1, n2, i1, i2, o1, o2;
        double xhf = x0[hf] + g->dxdy[3] * yl[3];
        double txc = (xhf - xm) / (hz[hf] - zm);
        double xp0 = xm + txc * (g->z_layer[0] - zm);
        double xp1 = xm + txc * (g->z_layer[1] - zm);
        double xp2 = xm + txc * (g->z_layer[2] - zm);
        n0 = window_search(g, p, nh, x0, ymin, ymax, id, 0, yl[0], xp0, w1, 1, C0, scratch, &edge, &min_margin);
        if (p->dv1 && n0 == 0) continue;   /* Dv1: the triplet needs its UTaX hit collinear with UTbX hit and magnet point */
        n1 = window_search(g, p, nh, x0, ymin, ymax, id, 1, yl[1], xp1, w1, 2, C1, scratch, &edge, &min_margin);
        n2 = window_search(g, p, nh, x0, ymin, ymax, id, 2, yl[2], xp2, w1, 2, C2, scratch, &edge, &min_margin);

        /* O-S5: combinations (h0 or missing) x (each kept h1, or missing if none) x (each kept h2, or missing) */
        o1 = n1 > 0 ? n1 : 1; o2 = n2 > 0 ? n2 : 1;
        for (i1 = 0; i1 < o1; ++i1)
            for (i2 = 0; i2 < o2; ++i2) {
                double pz[5], px[5], pw[5], a, b, c2, ndf;
                int np = 0, sel[4], k;
                best_t c;
                sel[0] = n0 > 0 ? C0[0].idx : -1;
                sel[1] = n1 > 0 ? C1[i1].idx : -1;
                sel[2] = n2 > 0 ? C2[i2].idx : -1;
                sel[3] = hf;
                c.nhits = 0;
                for (k = 0; k < 4; ++k) {
                    c.hit[k] = sel[k];
                    c.hid[k] = sel[k] >= 0 ? id[sel[k]] : INT32_MAX;
                    if (sel[k] >= 0) {
                        pz[np] = hz[sel[k]];
                        px[np] = x0[sel[k]] + g->dxdy[k] * yl[k];     /* stereo hit evaluated at the track's y */
                        pw[np] = hw[sel[k]];
                        ++np; ++c.nhits;
                    }
                }
                if (c.nhits < p->min_hits) continue;
                pz[np] = zm; px[np] = xm; pw[np] = p->w_mag; ++np;   /* magnet point pseudo-measurement (A-8) */
                orc_fit_line(np, pz, px, pw, g->z_ref, &a, &b, &c2);
                ndf = (double)(c.nhits + 1 - 2);
                /* O-S6: chi2/ndf cut, score */
                {
                    double m = relm(c2 / ndf, p->chi2ndf_max);
                    if (m < eps) edge = 1;
                    if (m < min_margin) min_margin = m;
                }
                if (!(c2 / ndf <= p->chi2ndf_max)) continue;
                c.found = 1; c.a = a; c.b = b; c.chi2 = c2;
                c.score = c2 + p->miss_penalty * (double)(4 - c.nhits);
                if (better(&c, &best)) {
                    if (best.found && best.score < second_score) second_score = best.score;
                    best = c;
                } else if (c.score < second_score) second_score = c.score;
            }
    }
    if (best.found && second_score < 1e299) {           /* best vs runner-up (A-16) */
        double m = relm(best.score, second_score);
        if (m < eps) edge = 1;
        if (m < min_margin) min_margin = m;
    }

    /* outputs: state at z_ref, rounded to the fp32 storage type of the track SoA */
    for (l = 0; l < 4; ++l) hit_out[l] = -1;
    memset(trk, 0, 8 * sizeof(double));
    *nhits_out = 0; *found_out = 0; *keep_out = 0;
    if (best.found) {
        double v[8], score;
        trk[0] = (double)(float)best.a;
        trk[1] = (double)(float)(ys + tys * (g->z_ref - g->z_seed));
        trk[2] = (double)(float)best.b;
        trk[3] = (double)(float)tys;
        trk[4] = (double)(float)((txs - best.b) / g->kick);
        trk[5] = (double)(float)best.chi2;
        *nhits_out = best.nhits; *found_out = 1;
        for (l = 0; l < 4; ++l) hit_out[l] = best.hit[l];
        /* O-S7: inputs in the order of P:121 */
        v[0] = trk[0]; v[1] = trk[1]; v[2] = trk[2]; v[3] = trk[3]; v[4] = trk[4]; v[5] = trk[5];
        v[6] = qop; v[7] = chi2s;
        score = orc_mlp_eval(mlp, v);
        trk[6] = score;
        {
            double m = relm(score, p->mlp_thr);
            if (m < eps) edge = 1;
            if (m < min_margin) min_margin = m;
        }
        *keep_out = p->mlp_keep_above ? (score > p->mlp_thr) : (score < p->mlp_thr);
    }
    *edge_out = edge;
    *margin_out = min_margin;
    if (F != F64) free(F);
}

/* ------------------------------------------------------------------------------------------------------------
 * orc_reconstruct: all events.  Hit / seed arrays are flat over events with [E+1] offsets.
 *   trk_f64  [n_seeds][8]  x, y, tx, ty, qop, chi2, mlp score, 0   (values 0..5 already rounded to fp32)
 *   nhits, found, keep, edge [n_seeds]; hit_idx [n_seeds][4] GLOBAL hit index (offset + local) or -1;
 *   margin [n_seeds] smallest relative margin seen (information).
 * "edge" = some comparison that decides an index, a flag or list membership had a relative margin < edge_rel:
 *   window inclusion and y-compatibility (each only when the other does not robustly reject the hit), rank
 *   cut-offs (k-th vs (k+1)-th closest), chi2/ndf cut, best vs runner-up score, MLP threshold.
 * ------------------------------------------------------------------------------------------------------------ */
void orc_reconstruct(const orc_geom *g, const orc_params *p, const orc_mlp *mlp, int n_events,
                     const int32_t *hit_off, const double *x0, const double *hz, const double *ymin,
                     const double *ymax, const double *hw, const int32_t *id, const int32_t *seed_off,
                     const double *sx, const double *sy, const double *stx, const double *sty, const double *sqop,
                     const double *schi2, double *trk_f64, int32_t *nhits, int32_t *hit_idx, int32_t *found,
                     int32_t *keep, int32_t *edge, double *margin, int n_threads)
{
    int e;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (e = 0; e < n_events; ++e) {
        int h0 = hit_off[e], nh = hit_off[e + 1] - h0, s, k;
        cand_hit *scratch = (cand_hit *)malloc(sizeof(cand_hit) * (size_t)(nh > 0 ? nh : 1));
        for (s = seed_off[e]; s < seed_off[e + 1]; ++s) {
            reconstruct_seed(g, p, mlp, nh, x0 + h0, hz + h0, ymin + h0, ymax + h0, hw + h0, id + h0, sx[s], sy[s],
                             stx[s], sty[s], sqop[s], schi2 ? schi2[s] : 0.0, scratch, trk_f64 + 8 * (size_t)s,
                             nhits + s, hit_idx + 4 * (size_t)s, found + s, keep + s, edge + s, margin + s);
            for (k = 0; k < 4; ++k)
                if (hit_idx[4 * (size_t)s + k] >= 0) hit_idx[4 * (size_t)s + k] += h0;
        }
        free(scratch);
    }
}

/* ============================================================================================================
 *  Vertexing: O-S8 / O-S9 for one pair (i < j in seed order).  Returns 1 if the pair passes.
 *  vtx[6] = x, y, z, doca, m_pipi, m_ppi;  *ia = positive track, *ib = negative track.
 * ============================================================================================================ */
static int vertex_pair(const orc_geom *g, const orc_params *p, const double *x, const double *y, const double *tx,
                       const double *ty, const double *qop, int i, int j, int *ia, int *ib, double *vtx,
                       int *flags, int *edge)
{
    const double eps = p->edge_rel;
    double po[10], pa, pb, mpipi, mppi, m_doca, m_z1, m_z2, m_ks, m_l, m_prot, m_n2, txa, txb;
    int a, b, ok, c_doca, c_z1, c_z2, f0, f1, robust_fail, marginal;
    *edge = 0;
    if (!(qop[i] * qop[j] < 0.0)) return 0;                       /* P:279 opposite charges */
    a = qop[i] > 0.0 ? i : j; b = qop[i] > 0.0 ? j : i;
    *ia = a; *ib = b;
    txa = tx[a]; txb = tx[b];
    if (p->magnet_polarity != 0.0) {   /* curved trajectories, Newton-Raphson (N1); slopes at the vertex for the masses */
        ok = orc_poca_curved(x[a], y[a], tx[a], ty[a], orc_gamma(p, qop[a]), x[b], y[b], tx[b], ty[b],
                             orc_gamma(p, qop[b]), g->z_ref, p->n2_min, p->vtx_newton_iters, po);
        if (ok) { txa = po[8]; txb = po[9]; }
    } else {
        ok = orc_poca(x[a], y[a], tx[a], ty[a], x[b], y[b], tx[b], ty[b], g->z_ref, p->n2_min, po);
    }
    m_n2 = relm(po[4], p->n2_min);
    if (!ok) { if (m_n2 < eps) *edge = 1; return 0; }
    pa = 1000.0 / fabs(qop[a]); pb = 1000.0 / fabs(qop[b]);       /* MeV; qop in 1/GeV */
    mpipi = orc_inv_mass(txa, ty[a], pa, p->m_pi, txb, ty[b], pb, p->m_pi);
    /* proton hypothesis for the track of larger momentum, tie -> the positive one (A-15) */
    if (pa >= pb) mppi = orc_inv_mass(txa, ty[a], pa, p->m_p, txb, ty[b], pb, p->m_pi);
    else          mppi = orc_inv_mass(txa, ty[a], pa, p->m_pi, txb, ty[b], pb, p->m_p);
    m_prot = relm(pa, pb);
    vtx[0] = po[0]; vtx[1] = po[1]; vtx[2] = po[2]; vtx[3] = po[3]; vtx[4] = mpipi; vtx[5] = mppi;
    c_doca = po[3] < p->doca_max;               m_doca = relm(po[3], p->doca_max);
    c_z1 = p->zv_min <= po[2];                  m_z1 = relm(po[2], p->zv_min);
    c_z2 = po[2] <= p->zv_max;                  m_z2 = relm(po[2], p->zv_max);
    f0 = fabs(mpipi - p->m_ks) < p->dm_ks;      m_ks = relm(fabs(mpipi - p->m_ks), p->dm_ks);
    f1 = fabs(mppi - p->m_lambda) < p->dm_lambda; m_l = relm(fabs(mppi - p->m_lambda), p->dm_lambda);
    *flags = (f0 ? 1 : 0) | (f1 ? 2 : 0);
    /* edge: no cut rejects the pair robustly, and some deciding comparison is marginal */
    robust_fail = (!c_doca && m_doca >= eps) || (!c_z1 && m_z1 >= eps) || (!c_z2 && m_z2 >= eps)
                  || ((!f0 && m_ks >= eps) && (!f1 && m_l >= eps));
    marginal = m_doca < eps || m_z1 < eps || m_z2 < eps || m_ks < eps || m_l < eps || m_prot < eps || m_n2 < eps;
    if (!robust_fail && marginal) *edge = 1;
    return c_doca && c_z1 && c_z2 && (*flags != 0);
}

/* orc_vertex: all events.  Tracks are the flat per-seed arrays (fp32 values promoted); keep[] selects.
 *   pass 1 counts per event (n_per_event[E]); offsets[E+1] = exclusive scan; pass 2 writes, per event sorted by
 *   (ia, ib), up to `capacity` vertices: v_evt, v_ia, v_ib (GLOBAL track index), v_f64 [..][6], v_flags.
 *   Edge pairs (see vertex_pair) are written to e_evt/e_ia/e_ib up to edge_capacity; *n_edge = their true number.
 *   *n_pairs = number of opposite-charge pairs examined.  Returns the total number of passing vertices. */
int64_t orc_vertex(const orc_geom *g, const orc_params *p, int n_events, const int32_t *seed_off, const double *x,
                   const double *y, const double *tx, const double *ty, const double *qop, const int32_t *keep,
                   int32_t *n_per_event, int64_t *offsets, int64_t capacity, int32_t *v_evt, int32_t *v_ia,
                   int32_t *v_ib, double *v_f64, int32_t *v_flags, int64_t edge_capacity, int32_t *e_evt,
                   int32_t *e_ia, int32_t *e_ib, int64_t *n_edge, int64_t *n_pairs, int n_threads)
{
    int e, pass;
    int64_t total = 0, nedge = 0, npairs = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    for (pass = 0; pass < 2; ++pass) {
#pragma omp parallel for schedule(dynamic, 1) reduction(+ : npairs)
        for (e = 0; e < n_events; ++e) {
            int s0 = seed_off[e], s1 = seed_off[e + 1], n = 0, a, b;
            /* output order (ia, ib): loop over the positive track, then the negative one, in seed order */
            for (a = s0; a < s1; ++a) {
                if (!keep[a] || !(qop[a] > 0.0)) continue;
                for (b = s0; b < s1; ++b) {
                    int ia, ib, flags = 0, edge = 0, ok;
                    double vtx[6];
                    if (!keep[b] || !(qop[b] < 0.0)) continue;
                    ok = vertex_pair(g, p, x, y, tx, ty, qop, a < b ? a : b, a < b ? b : a, &ia, &ib, vtx, &flags, &edge);
                    if (pass == 0) {
                        ++npairs;
                        if (edge) {
                            int64_t k;
#pragma omp atomic capture
                            k = nedge++;
                            if (k < edge_capacity) { e_evt[k] = e; e_ia[k] = ia; e_ib[k] = ib; }
                        }
                    }
                    if (ok) {
                        if (pass == 1) {
                            int64_t k = offsets[e] + n;
                            if (k < capacity) {
                                v_evt[k] = e; v_ia[k] = ia; v_ib[k] = ib; v_flags[k] = flags;
                                memcpy(v_f64 + 6 * k, vtx, sizeof vtx);
                            }
                        }
                        ++n;
                    }
                }
            }
            if (pass == 0) n_per_event[e] = n;
        }
        if (pass == 0) {
            offsets[0] = 0;
            for (e = 0; e < n_events; ++e) offsets[e + 1] = offsets[e] + n_per_event[e];
            total = offsets[n_events];
        }
    }
    *n_edge = nedge; *n_pairs = npairs;
    return total;
}

/* ============================================================================================================
 *  O-S6b  clone killing across seeds: "Iterating over all possible track pairs that have
 *  more than two shared UT hits ..., the candidates with lower scores are killed."
 *  Reading A-31: two found tracks of one event share a hit when they hold the same hit index in the same layer;
 *  a pair with at least min_shared (3) shared hits is a clone pair; its worse member is killed, worse = larger
 *  chi2 + miss_penalty * (4 - nhits) (the S6 score, A-9), ties -> larger seed index.  Every pair is judged on the
 *  tracks as they came out of S6 (a killed track still kills), so the result does not depend on an iteration order.
 *  chi2 / nhits / hit / found are the per-seed track records; killed[s] = 1 for the tracks removed.  Returns their
 *  number.
 * ============================================================================================================ */
int64_t orc_clone_kill(const orc_params *p, int min_shared, int n_events, const int32_t *seed_off, const double *chi2,
                       const int32_t *nhits, const int32_t *hit, const int32_t *found, int32_t *killed)
{
    int e;
    int64_t n_killed = 0;
    for (e = 0; e < n_events; ++e) {
        int i, j, l;
        for (i = seed_off[e]; i < seed_off[e + 1]; ++i) {
            double si = chi2[i] + p->miss_penalty * (double)(4 - nhits[i]);
            killed[i] = 0;
            if (!found[i]) continue;
            for (j = seed_off[e]; j < seed_off[e + 1]; ++j) {
                double sj;
                int shared = 0;
                if (j == i || !found[j]) continue;
                for (l = 0; l < 4; ++l)
                    if (hit[4 * i + l] >= 0 && hit[4 * i + l] == hit[4 * j + l]) ++shared;
                if (shared < min_shared) continue;
                sj = chi2[j] + p->miss_penalty * (double)(4 - nhits[j]);
                if (sj < si || (sj == si && j < i)) killed[i] = 1;      /* j is the better one of the pair */
            }
            n_killed += killed[i];
        }
    }
    return n_killed;
}

/* ============================================================================================================
 *  O-L  HLT1 line NNs on the two-track vertices (P:277-P:285): "four different fast NNs with similar
 *  architectures to the one described in Sec. 2.2 ... a single hidden layer with 32 nodes and an output layer with a
 *  single node ... The NN threshold for background suppression has been set to 0.5."  The inputs "include track
 *  parameters of the two secondary tracks, vertex parameters, and parent track parameters"; the paper gives no list.
 *  Reading A-33, 16 inputs: positive track (tx, ty, q/p, chi2), negative track (tx, ty, q/p, chi2), vertex
 *  (x, y, z, DOCA), parent (tx, ty, p [GeV], pT [GeV]) with the parent momentum = sum of the two track momenta
 *  p_i = 1/|q/p_i| along (tx_i, ty_i, 1).  Parity unpinned as far as the meaning of the inputs goes.
 * ============================================================================================================ */
void orc_line_features(double txa, double tya, double qa, double c2a, double txb, double tyb, double qb, double c2b,
                       const double *vtx4, double *v)
{
    double pa = 1.0 / fabs(qa), pb = 1.0 / fabs(qb);                         /* GeV */
    double na = sqrt(txa * txa + tya * tya + 1.0), nb = sqrt(txb * txb + tyb * tyb + 1.0);
    double px = pa * txa / na + pb * txb / nb, py = pa * tya / na + pb * tyb / nb, pz = pa / na + pb / nb;
    v[0] = txa; v[1] = tya; v[2] = qa; v[3] = c2a;
    v[4] = txb; v[5] = tyb; v[6] = qb; v[7] = c2b;
    v[8] = vtx4[0]; v[9] = vtx4[1]; v[10] = vtx4[2]; v[11] = vtx4[3];
    v[12] = px / pz; v[13] = py / pz;
    v[14] = sqrt(px * px + py * py + pz * pz);
    v[15] = sqrt(px * px + py * py);
}

/* nets[4] = the four single-hidden-layer networks (n_h2 = 0); per vertex k: scores[4k + i], bits[k] = sum_i 2^i [score_i > thr].
 * ia / ib index the per-seed track arrays; vtx4 = (x, y, z, doca) per vertex.  edge[k] = 1 if some score is within
 * edge_rel of the threshold. */
void orc_lines(const orc_mlp *nets, double thr, double edge_rel, int64_t n_vtx, const int32_t *ia, const int32_t *ib,
               const double *vtx4, const double *tx, const double *ty, const double *qop, const double *chi2,
               double *scores, int32_t *bits, int32_t *edge)
{
    int64_t k;
    for (k = 0; k < n_vtx; ++k) {
        double v[16];
        int i, a = ia[k], b = ib[k];
        orc_line_features(tx[a], ty[a], qop[a], chi2[a], tx[b], ty[b], qop[b], chi2[b], vtx4 + 4 * k, v);
        bits[k] = 0; edge[k] = 0;
        for (i = 0; i < 4; ++i) {
            double sc = orc_mlp_eval(&nets[i], v);
            scores[4 * k + i] = sc;
            if (sc > thr) bits[k] |= 1 << i;
            if (relm(sc, thr) < edge_rel) edge[k] = 1;
        }
    }
}

int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
