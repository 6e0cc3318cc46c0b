"""NEXT f2 on the GPU: infrared piece of eq.(26), x_G = 0, and the paper's own scaling solution (P9) solved through
the C ABI (dse_jacobian + dse_lu_solve with under-relaxation), compared step by step with the oracle."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from test_gpu_parity import oracle_params, gpu_build, check, _torch   # noqa: E402


@pytest.mark.parametrize("kw", [
    dict(n_ir=16),                                  # infrared piece, x_G = x_Z
    dict(n_ir=12, x_G=0.0, x_Z=5e4),                # the paper's subtraction points (L135)
    dict(n_ir=0, x_G=0.0, x_Z=30.0),                # x_G = 0 without the infrared piece
    dict(n_ir=7, x_G=0.0, x_Z=5e4, angular_rule=1, n_theta=40),
    dict(radial_split=1),                           # NEXT f1: the paper's split at y = x (eq.(26)), x_G = x_Z
    dict(radial_split=1, n_ir=12, x_G=0.0, x_Z=5e4, n_r=24),        # the paper's full three-interval rule
    dict(radial_split=1, n_ir=5, x_G=3.0, x_Z=5e4, n_r=13, n_theta=21, n_cheb=12),   # ragged
])
def test_infrared_piece_and_zero_subtraction_point_parity(orc, kw):
    from workloads import Workload, draw_coefficients
    base = dict(n_cheb=16, n_r=40, n_theta=32, eps2=1e-6, L2=5e4)
    base.update(kw)
    w = Workload("f2", **base)
    c = draw_coefficients(31, w.n_cheb)[None, :]
    bc = np.array([[0.0, 1 / 0.256]])
    Fo, Jo = orc.residual_jacobian(oracle_params(w), c[0], bc[0, 0], bc[0, 1])
    for flags in (0, 1):
        J, F = gpu_build(w, c, bc, flags)
        check(J[0], F[0], Jo, Fo)


def test_paper_scaling_solution_on_gpu(orc):
    torch = _torch()
    import scaling_setup as S
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("paper-scaling", S.N, S.N_R, S.N_THETA, S.EPS2, S.L2, x_G=0.0, x_Z=S.L2, n_ir=S.N_IR)
    p = oracle_params(w)
    c_o = S.start_coefficients(orc, p)
    d = Dse(params_from_workload(w))
    c_g = torch.from_numpy(c_o[None, :].copy()).cuda()
    bc = torch.tensor([[S.G_G, S.G_Z]], dtype=torch.float64, device="cuda")
    steps = 0
    for it in range(30):
        Fo, Jo = orc.residual_jacobian(p, c_o, S.G_G, S.G_Z)
        do, so, rc = orc.lu_solve(Jo, Fo)
        J, F = d.jacobian(c_g, bc)
        x, st = d.lu_solve(J, F)
        st = st.cpu().numpy()[0]
        assert abs(st[0] - so[0]) <= 1e-7 * so[0] + 2e-11           # same |Delta| (cond(J) ~ 1e5; floor ~ cond*eps)
        c_o = c_o - S.damping(so[0]) * do
        c_g -= S.damping(float(st[0])) * x
        assert np.allclose(c_g.cpu().numpy()[0], c_o, rtol=0, atol=1e-9 * np.abs(c_o).max())   # same trajectory
        steps += 1
        if st[0] < 1e-11:
            break
    assert steps <= 15 and st[0] < 1e-11
    c = c_g.cpu().numpy()[0]
    assert np.abs(c - c_o).max() <= 1e-9 * np.abs(c_o).max()        # converged coefficients: north_star bar 1e-9

    def alpha(xv):
        g, z = orc.ln_dress(p, c, xv)                                # evaluation of the expansion only
        return math.exp(2 * g + z)

    assert abs(alpha(91.2 ** 2) - 0.118) < 1e-3
    assert abs(alpha(S.EPS2) - 2.972) < 5e-3
    # Schwinger function of the converged gluon propagator on the GPU: zero slightly below t = 5 GeV^-1 (L165)
    t = torch.linspace(0.5, 8.0, 76, dtype=torch.float64, device="cuda")
    dl = d.schwinger(c_g, t, 1 << 14, 1e-14, S.L2).cpu().numpy()[0]
    tt = t.cpu().numpy()
    zeros = [0.5 * (tt[i] + tt[i + 1]) for i in range(len(tt) - 1) if dl[i] * dl[i + 1] < 0]
    assert dl[0] > 0 and zeros and 3.0 < zeros[0] < 5.0
    d.close()
