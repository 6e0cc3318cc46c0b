"""Seeded synthetic workloads (BASELINE.json configs 0-4) shared by the tests, bench.py and smoke().

A module of its own, outside both the product package (paper_1206_1779_b200/) and the oracle (oracle/): neither of
them imports it.  It holds NONE of the method's arithmetic: only shapes, parameter values, the seeded draws of
Chebyshev coefficients / boundary values, and one stored start vector (read from tests/golden/, written there by a
committed script that calls only the oracle).  Both the CUDA path and the CPU oracle receive the arrays produced here
(DESIGN.md "Input recipe").  No public dataset is involved: the paper's workloads are parameter choices (PAPER.md
Table 1 caption L364) and these configs are synthetic stand-ins of the same structure.
"""
import os

from dataclasses import dataclass, field

import numpy as np

KAPPA = 0.595353
DELTA = -9.0 / 44.0


@dataclass
class Workload:
    name: str
    n_cheb: int
    n_r: int
    n_theta: int
    eps2: float
    L2: float
    n_batch: int = 1
    x_G: float = 1e2       # subtraction points = renormalisation point mu^2 = 1e2 (reading A12)
    x_Z: float = 1e2
    alpha_mu: float = 1.0
    n_colors: float = 3.0
    delta: float = DELTA
    ir_exp_G: float = -KAPPA
    ir_exp_Z: float = 2 * KAPPA
    uv_omega: float = field(default=None)
    n_ir: int = 0          # nodes of the infrared piece int_0^{eps2} dy (eq.(26)); 0 in the BASELINE configs
    radial_split: int = 0  # 1: the paper's split at y = x with n_r nodes in each interval (eq.(26))
    angular_rule: int = 0  # 0: Gauss-Legendre in theta (BASELINE configs); 1: tanh-sinh in xi

    def __post_init__(self):
        if self.uv_omega is None:
            self.uv_omega = 11.0 * self.n_colors * self.alpha_mu / (12.0 * np.pi)

    @property
    def n_ext(self):
        return self.n_cheb + (1 if self.x_G == self.x_Z else 2)

    @property
    def points(self):
        """quadrature points per system and build: N_ext * N_r * N_theta"""
        return self.n_ext * ((2 if self.radial_split else 1) * self.n_r + self.n_ir) * self.n_theta

    @property
    def paper_equiv_evals(self):
        """(2N)^2 N_r N_theta: the paper's count of independent 2-D quadrature kernel evaluations"""
        return (2 * self.n_cheb) ** 2 * self.n_r * self.n_theta


def draw_coefficients(seed: int, n_cheb: int) -> np.ndarray:
    """c = (a_0..a_{N-1}, b_0..b_{N-1}): c_0 ~ U(-0.5, 0.5), c_j ~ N(0, (0.3/j)^2), j >= 1.

    Draw order per system: a_0, a_1..a_{N-1}, b_0, b_1..b_{N-1}."""
    rng = np.random.default_rng(seed)
    c = np.empty(2 * n_cheb)
    for h in range(2):
        c[h * n_cheb] = rng.uniform(-0.5, 0.5)
        j = np.arange(1, n_cheb)
        c[h * n_cheb + 1:(h + 1) * n_cheb] = rng.normal(0.0, 1.0, n_cheb - 1) * (0.3 / j)
    return c


CONFIGS = {
    0: Workload("cfg0-tiny", 8, 64, 16, 1e-10, 1e10),
    1: Workload("cfg1-production", 32, 256, 64, 1e-10, 1e10),
    2: Workload("cfg2-newton", 32, 256, 64, 1e-10, 1e10),
    3: Workload("cfg3-large", 64, 1024, 128, 1e-12, 1e12),
    4: Workload("cfg4-batched", 32, 256, 64, 1e-10, 1e10, n_batch=256),
}


def config_inputs(cfg: int, n_batch: int = None):
    """Returns (workload, c[n_batch, 2N], bc[n_batch, 2] = (1/G(x_G), 1/Z(x_Z)))."""
    w = CONFIGS[cfg]
    nb = w.n_batch if n_batch is None else n_batch
    if cfg in (0, 1, 3):
        c = draw_coefficients({0: 0, 1: 1, 3: 3}[cfg], w.n_cheb)[None, :].repeat(nb, 0)
        bc = np.ones((nb, 2))
    elif cfg == 2:
        c = np.zeros((nb, 2 * w.n_cheb))      # G = Z = 1  <=>  ln G = ln Z = 0
        bc = np.ones((nb, 2))
    elif cfg == 4:
        c = np.stack([draw_coefficients(1000 + b, w.n_cheb) for b in range(nb)])
        bc = np.ones((nb, 2))
        for b in range(nb):
            bc[b, 0] = np.random.default_rng(5000 + b).uniform(0.5, 1.5)   # 1/G(mu^2) per system (reading A13)
    else:
        raise KeyError(cfg)
    return w, np.ascontiguousarray(c), np.ascontiguousarray(bc)


# ---------------------------------------------------------------------------------------------------------------
# "Config 2'": the paper's own parameter set -- the convergent counterpart of
# BASELINE configs[2] (reading A17).  Inputs only: shapes, boundary values and a start guess.
def paper_scaling_workload() -> Workload:
    """eps2 = 1e-6, L2 = 5e4 GeV^2, x_G = 0 (1/G(0) = 0: scaling solution), x_Z = L2, N = 36, 96 + 32 radial nodes
    (32 of them on the infrared piece of eq.(26)), 32 angles."""
    return Workload("cfg2p-paper-scaling", 36, 96, 32, 1e-6, 5e4, x_G=0.0, x_Z=5e4, n_ir=32)


PAPER_SCALING_BC = (0.0, 1.0 / 0.256)       # (1/G(0), 1/Z(x_Z)): PAPER.md L135


def scaling_start_coefficients(w: Workload) -> np.ndarray:
    """The start vector of config 2': a scaling-shaped guess built from the paper's asymptotic forms eq.(16)-(19) (NOT the
    fit functions of ref.[16], which are not in PAPER.md).  It is INPUT DATA here: the 72 numbers are stored in
    tests/golden/scaling_start_N36.txt, written by tests/golden/make_scaling_start.py, which samples the forms at the
    mapped Chebyshev roots and projects them with the oracle's own tables (tests/scaling_setup.py -- the one place where
    that projection is written down)."""
    assert (w.n_cheb, w.eps2, w.L2, w.x_G, w.x_Z, w.n_ir) == (36, 1e-6, 5e4, 0.0, 5e4, 32), "stored for config 2' only"
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "tests", "golden", "scaling_start_N36.txt")
    c = np.array([float(line.split("#")[0]) for line in open(path) if line.split("#")[0].strip()])
    assert c.shape == (2 * w.n_cheb,)
    return c
