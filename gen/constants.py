"""Workload constants for the synthetic HLT1-Downstream events (no arithmetic of the method here).

Every value is a number the workload definition fixes (BASELINE.json configs[0..4], SURVEY.md §8c
"Constants" and readings A-1..A-26).  Tests and bench.py read them from here and hand the SAME values
to the CUDA library (paper_2503_13092_b200) and to the CPU oracle (oracle/), which never import each
other.  `P:n` = /root/reference/PAPER.md line n.
"""
import math

# --- UT geometry: 4 planes UTaX, UTaU, UTbV, UTbX (Fig. 2; numeric values from BASELINE cfg0) ---
GEOMETRY = dict(
    z_layer=(2327.5, 2372.5, 2597.5, 2642.5),                    # mm
    dxdy=(0.0, math.tan(math.radians(5.0)), -math.tan(math.radians(5.0)), 0.0),  # A-1: x_hit(y) = x0 + y*dxdy
    x_half=860.0, y_half=700.0, hole_half=50.0,                  # mm
    n_sectors_y=14, sector_height=100.0,                         # A-2: 14 y-sectors of 100 mm over +-700
    z_seed=7826.0,                                               # seed state is given at this z
    z_ref=2485.0,                                                # UT midpoint
    zmag_c=(5282.0, 0.0, 0.0, 0.0),                              # A-3: z_mag = c0 + c1 ty^2 + c2 tx^2 + c3 qop^2
    kick=1.2,                                                    # GeV: dtx = q*kick/p
)

SIGMA_HIT = 0.054                                                # mm
W_HIT = 1.0 / (SIGMA_HIT * SIGMA_HIT)

# --- algorithm parameters (free parameters the paper does not print) ---
PARAMS = dict(
    w0_a=2.0, w0_b=100.0, w0_max=150.0,      # first window half-width  min(w0_max, w0_a + w0_b*|qop|)   mm (A-5)
    w1_a=1.0, w1_b=2.0,                      # refined window half-width w1_a + w1_b*|qop|               mm (A-5)
    y_tol=3.0,                               # mm
    w_mag=1.0,                               # weight of the magnet-point pseudo-measurement 1/(1 mm)^2 (A-8)
    chi2ndf_max=5.0, miss_penalty=4.0,       # A-9
    min_hits=3, max_first_hits=10,           # A-6
    mlp_thr=0.1, mlp_keep_above=1,           # A-12 (cfg3 sense)
    doca_max=2.0, zv_min=600.0, zv_max=2400.0,
    m_pi=139.57, m_p=938.27, m_ks=497.6, m_lambda=1115.68,
    dm_ks=50.0, dm_lambda=20.0,
    n2_min=1e-12,                            # A-14
    # curved-track vertexing (P:255-P:269): gamma = -MP (c0 + c1 q/p[1/MeV]) (Eq. 3); the synthetic
    # configurations have no field upstream of the UT, so MP = 0 (straight tracks, A-20) is the default
    magnet_polarity=0.0, gamma_c0=-1.5e-8, gamma_c1=9.3e-3, vtx_newton_iters=3,
    # clone killing across seeds: shared hits that make a clone pair; 0 = off (BASELINE configs)
    clone_min_shared=0,
    # Dv1 triplet search (P:107-P:111): 1 = every UTbX hit of the y-compatible sectors starts a candidate
    # and the UTaX hit is mandatory; 0 = Dv0 (first window, <= 10 closest), the BASELINE configurations
    dv1=0,
    # ghost-killer sigmoid by the paper's fast intrinsics; 0 = IEEE, the parity-tested path
    mlp_fast_math=0,
)

# A-10: fixed input normalisation (mu, sigma) for [x, y, tx, ty, qop, chi2, qop_seed, chi2_seed]
MLP_MU = (0.0, 0.0, 0.0, 0.0, 0.0, 3.0, 0.0, 1.0)
MLP_SIGMA = (500.0, 400.0, 0.2, 0.1, 0.25, 3.0, 0.25, 1.0)
MLP_SIZES = (8, 32, 16, 1)

# id encoding (A-2)
ID_SEQ_BITS = 20
ID_SECTOR_SHIFT = 20
ID_LAYER_SHIFT = 24


class Config:
    """One BASELINE.json config: generator knobs only."""

    def __init__(self, name, seed, n_events, mean_decays, frac_ks, n_seeds, n_hits, smear, eff,
                 fixed_decays=None, seeded_decays=None, prompt_frac=0.0):
        self.name = name
        self.seed = seed
        self.n_events = n_events
        self.mean_decays = mean_decays      # Poisson mean of generated decays per event
        self.frac_ks = frac_ks
        self.n_seeds = n_seeds              # Poisson mean target of seeds / event (None: true seeds only)
        self.n_hits = n_hits                # Poisson mean target of hits / event (None: track hits only)
        self.smear = smear
        self.eff = eff
        self.fixed_decays = fixed_decays    # cfg0: exactly this many accepted decays per event
        self.seeded_decays = seeded_decays  # cfg0: seeds only for daughters of the first k decays (A-23)
        self.prompt_frac = prompt_frac      # cfg2: fraction of hits that are NOT noise (A-24)


CONFIGS = [
    Config("cfg0", 0, 10, None, 1.0, None, None, smear=False, eff=1.0, fixed_decays=25, seeded_decays=10),
    Config("cfg1", 1, 1000, 15.0, 0.7, 150.0, 3000.0, smear=True, eff=0.97),
    Config("cfg2", 2, 1000, 30.0, 0.7, 300.0, 8000.0, smear=True, eff=0.97, prompt_frac=0.30),
    Config("cfg3", 3, 2000, 60.0, 0.7, 500.0, 3000.0, smear=True, eff=0.97),
    Config("cfg4", 4, 100000, 15.0, 0.7, 150.0, 3000.0, smear=True, eff=0.97),
]

BLOCK_EVENTS = 1000        # RNG granularity: one default_rng per block of events
SUBBATCH_EVENTS = 10000    # cfg4 is processed as 10 sub-batches of 10 000 events
