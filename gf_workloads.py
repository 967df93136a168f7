"""Synthetic workloads: the configurations of BASELINE.json, as data.

This module holds NONE of the method's arithmetic.  It only names the inputs
(propagator parameters, cutoff, grid box and counts, quadrature orders) and
draws the seeded parity sub-sample, so that the CUDA path
(paper_1205_0752_b200) and the CPU oracle (oracle/) can be fed the same
problem while sharing no code.  Each side builds its own grid and its own
quadrature tables from these numbers.

Shapes follow the paper's scans (square grids of a few units around the
origin, ngl >= 64, ndbl >= 49), scaled up as
BASELINE.json states; readings G3, G9, G10, G11 of DESIGN.md fix what the
configs leave open (cutoff 1e6 where omitted, endpoint-inclusive grids,
|Im x| in [1e-6, 1e-3] for the strip, line 2 carries the rational propagator).
"""
import numpy as np

PARITY_SEED = 12050752  # the arXiv number

_BUBBLE = {"kind": "massive", "m2": 1.0}
_RATIONAL = {"kind": "rational", "M2": 2.0, "a": 0.5, "b": 1.2}

CONFIGS = {
    # name: worked-example bubble, tiny (BASELINE.json configs[0])
    "cfg1_tiny": dict(
        line_k=_BUBBLE, line_pk=_BUBBLE, cutoff2=1e4,
        n_re=64, n_im=64, re=(-5.0, 1.0), im=(-2.0, 2.0), spacing="uniform", im_abs_min=0.0,
        n_rad=64, n_ang=32),
    # configs[1]
    "cfg2_mid": dict(
        line_k=_BUBBLE, line_pk=_BUBBLE, cutoff2=1e6,
        n_re=512, n_im=512, re=(-10.0, 2.0), im=(-4.0, 4.0), spacing="uniform", im_abs_min=0.0,
        n_rad=256, n_ang=128),
    # configs[2]: the production scan the headline metric is quoted on
    "cfg3_production": dict(
        line_k=_BUBBLE, line_pk=_BUBBLE, cutoff2=1e6,
        n_re=2048, n_im=2048, re=(-10.0, 2.0), im=(-4.0, 4.0), spacing="uniform", im_abs_min=0.0,
        n_rad=512, n_ang=256),
    # configs[3]: rational propagator with complex-conjugate poles on line 2
    "cfg4_rational": dict(
        line_k=_BUBBLE, line_pk=_RATIONAL, cutoff2=1e6,
        n_re=1024, n_im=1024, re=(-8.0, 2.0), im=(-4.0, 4.0), spacing="uniform", im_abs_min=0.0,
        n_rad=512, n_ang=256),
    # configs[4]: near-cut strip, log-spaced |Im x|, both signs
    "cfg5_strip": dict(
        line_k=_BUBBLE, line_pk=_BUBBLE, cutoff2=1e6,
        n_re=4096, n_im=256, re=(-10.0, -3.0), im=(-1e-3, 1e-3), spacing="log_abs_im",
        im_abs_min=1e-6, n_rad=1024, n_ang=512),
    # not a BASELINE.json config: a scan of the size the paper itself ran (its worked example, masses^2 +-i/2,
    # eq. (19); 128 x 128 points, ngl = 64 radial Gauss-Legendre and ndbl = 49 tanh-sinh nodes: PAPER.md:150,158,276),
    # kept to show what preparation and launch overheads cost on small grids (bench.py --workload paper_scan_128)
    "paper_scan_128": dict(
        line_k={"kind": "massive", "m2": 0.5j}, line_pk={"kind": "massive", "m2": -0.5j}, cutoff2=1e6,
        n_re=128, n_im=128, re=(-2.0, 2.0), im=(-2.0, 2.0), spacing="uniform", im_abs_min=0.0,
        n_rad=64, n_ang=49, ang="tanh_sinh"),
}

PREFACTOR = 2.0 / np.pi   # c0 of eq. (21): 16 pi^2 / (2 pi)^3
MAP_SCALE = 1.0           # s0 of the shifted-log radial map (reading G3)
RADIAL_RULE = "gauss_legendre"
ANGULAR_RULE = "gauss_legendre"  # what BASELINE.json's configs run (reading G5)


def n_points(cfg):
    return cfg["n_re"] * cfg["n_im"]


def n_evals(cfg):
    """Nominal integrand evaluations: points x N_r x N_a (independent of any pairing trick)."""
    return n_points(cfg) * cfg["n_rad"] * cfg["n_ang"]


def parity_sample(cfg, n_random=4096, stride=16, seed=PARITY_SEED):
    """Flat indices (row-major [n_im][n_re]) of the deterministic parity sub-sample:
    every `stride`-th index in each direction plus `n_random` seeded draws."""
    n_re, n_im = cfg["n_re"], cfg["n_im"]
    jj, ii = np.meshgrid(np.arange(0, n_im, stride), np.arange(0, n_re, stride), indexing="ij")
    lattice = (jj * n_re + ii).ravel()
    rng = np.random.default_rng(seed)
    rnd = rng.integers(0, n_re * n_im, size=n_random)
    return np.unique(np.concatenate([lattice, rnd]))


def row_partition(n_rows, world_size, rank):
    """Contiguous block of grid rows owned by `rank` (rows are independent,
    tables replicated, no collective on the data path).  Returns (first_row, n_rows_local)."""
    base, rem = divmod(n_rows, world_size)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)
