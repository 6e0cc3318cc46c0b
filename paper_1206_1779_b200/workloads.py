"""Seeded synthetic workloads (BASELINE.json configs 0-4) shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic: only shapes, parameter values and the seeded
draws of Chebyshev coefficients / boundary values.  Both the CUDA path and the CPU oracle receive
the arrays produced here.  No public dataset is involved: the paper's
workloads are parameter choices (Table 1 caption L364) and these configs are synthetic
stand-ins of the same structure.
"""
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
    """A scaling-shaped start guess built from the paper's asymptotic forms eq.(16)-(19) -- NOT the fit functions of
    ref.[16], which are not in PAPER.md:  ln G = -kappa ln(x/(x+1)) + delta ln(1 + omega ln(1+x)),
    ln Z = 2 kappa ln(x/(x+1)) + gamma ln(1 + omega ln(1+x)), sampled at the mapped Chebyshev roots (fn.9) and projected
    on T_j by the discrete orthogonality of the roots; a_0 is then shifted so that Z(x_Z = L2) = 0.256."""
    N = w.n_cheb
    gamma = -1.0 - 2.0 * w.delta
    i = np.arange(N)
    ang = np.pi * (i + 0.5) / N
    s = -np.cos(ang)
    x = w.eps2 * np.exp(0.5 * (s + 1.0) * np.log(w.L2 / w.eps2))
    run = np.log(1.0 + w.uv_omega * np.log(1.0 + x))
    lg = w.ir_exp_G * np.log(x / (x + 1.0)) + w.delta * run
    lz = w.ir_exp_Z * np.log(x / (x + 1.0)) + gamma * run
    j = np.arange(N)
    T = np.cos(np.outer(np.arccos(s), j))                      # T_j(s_i)
    c = np.concatenate([(2.0 / N) * (T.T @ lz), (2.0 / N) * (T.T @ lg)])
    lnZ_L2 = 0.5 * c[0] + c[1:N].sum()                         # series at s = 1 (T_j(1) = 1), c_0/2 convention
    c[0] += 2.0 * (np.log(0.256) - lnZ_L2)
    return c
