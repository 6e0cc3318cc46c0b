"""GPU LU / Newton step against the oracle's."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from test_gpu_parity import oracle_params, _torch   # noqa: E402


def test_lu_solve_matches_oracle(orc):
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from paper_1206_1779_b200.workloads import CONFIGS
    d = Dse(params_from_workload(CONFIGS[0]))
    rng = np.random.default_rng(5)
    for n in (1, 2, 16, 64, 128, 200):
        if n > 158 and n != 16:
            continue   # large systems use the handle's own scratch (2N only)
        A = rng.normal(size=(3, n, n)) * 10.0 ** rng.uniform(-8, 8, size=(3, n, 1))
        b = rng.normal(size=(3, n)) * np.abs(A).max(axis=2)
        x, st = d.lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x = x.cpu().numpy(); st = st.cpu().numpy()
        for s in range(3):
            xo, so, rc = orc.lu_solve(A[s], b[s])
            assert rc == 0
            assert np.allclose(x[s], xo, rtol=1e-9, atol=1e-13 * np.abs(xo).max())
            assert np.allclose(st[s], so, rtol=1e-9)
    d.close()


def test_newton_trajectory_weak_coupling(orc):
    """Same start, same steps: iterates agree while cond*1e-16 allows; quadratic convergence (L226)."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from paper_1206_1779_b200.workloads import Workload
    w = Workload("newton-weak", 10, 64, 24, 1e-2, 1e2, x_G=1.0, x_Z=1.0, alpha_mu=0.05)
    d = Dse(params_from_workload(w))
    p = oracle_params(w)
    c_o = np.zeros(20)
    c_g = torch.zeros((1, 20), dtype=torch.float64, device="cuda")
    bc = torch.ones((1, 2), dtype=torch.float64, device="cuda")
    dn = []
    for it in range(8):
        c_o, so, rc = orc.newton_step(p, c_o, 1.0, 1.0, 1.0)
        st = d.newton_step(c_g, bc, 1.0).cpu().numpy()[0]
        dn.append(st[0])
        assert abs(st[0] - so[0]) <= 1e-9 * so[0] + 1e-12     # |Delta| itself carries cond(J)*eps of the iterate
        assert np.allclose(c_g.cpu().numpy()[0], c_o, rtol=0, atol=1e-9 * np.abs(c_o).max())
    assert dn[-1] < 1e-13
    d.close()
