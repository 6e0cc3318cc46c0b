"""The paper's own parameter set: eps2 = 1e-6, L2 = 5e4 GeV^2, x_G = 0 with 1/G(0) = 0
(scaling solution), x_Z = L2 with Z(x_Z) = 0.256, alpha(mu^2) = 1.  The start guess is NOT the fit of ref.[16] (not in
PAPER.md): it is a scaling-shaped guess built from the paper's own asymptotic forms eq.(16)-(19)."""
import math

import numpy as np

KAPPA = 0.595353
DELTA = -9.0 / 44.0
GAMMA = -13.0 / 22.0
OMEGA = 11.0 * 3.0 / (12.0 * math.pi)
EPS2, L2 = 1e-6, 5e4
G_G, G_Z = 0.0, 1.0 / 0.256
N, N_R, N_IR, N_THETA = 36, 96, 32, 32


def start_coefficients(orc, p):
    tab = orc.tables(p)
    x = tab["x_ext"][:N]
    lg = -KAPPA * np.log(x / (x + 1)) + DELTA * np.log(1 + OMEGA * np.log(1 + x))
    lz = 2 * KAPPA * np.log(x / (x + 1)) + GAMMA * np.log(1 + OMEGA * np.log(1 + x))
    T = np.stack([orc.cheb_phi(N, s) for s in tab["s_root"]])
    T[:, 0] *= 2
    c = np.concatenate([(2.0 / N) * (T.T @ lz), (2.0 / N) * (T.T @ lg)])
    _, lnZ = orc.ln_dress(p, c, L2)
    c[0] += 2 * (math.log(0.256) - lnZ)            # Z(x_Z) = 0.256
    return c


STEP_CAP = 0.5


def damping(dmax):
    """under-relaxation: cap the update at 0.5 until the iteration is close, then rho = 1"""
    return min(1.0, STEP_CAP / dmax)
