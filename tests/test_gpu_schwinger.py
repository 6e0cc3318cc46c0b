"""NEXT f4: device-generated Gauss-Legendre rule and the Schwinger function eq.(20) against the oracle."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from test_gpu_parity import oracle_params, _torch   # noqa: E402
from test_oracle_path import _massive_propagator_coefficients   # noqa: E402


@pytest.mark.parametrize("n", [2, 3, 64, 257, 4096])
def test_device_gauss_legendre_matches_oracle(orc, n):
    _torch()
    from paper_1206_1779_b200.binding import gauss_legendre
    x, w = gauss_legendre(n)
    x = x.cpu().numpy(); w = w.cpu().numpy()
    xo, wo = orc.gauss_legendre(n)
    assert np.allclose(x, xo, rtol=0, atol=2e-15)
    assert np.allclose(w, wo, rtol=2e-11, atol=0)
    assert abs(w.sum() - 2.0) < 1e-13


def test_device_gauss_legendre_full_size_sampled(orc):
    """The paper's 2^17-node rule (fn.13): properties at full size + sampled nodes the oracle computes one by one."""
    _torch()
    from paper_1206_1779_b200.binding import gauss_legendre
    n = 1 << 17
    x, w = gauss_legendre(n)
    x = x.cpu().numpy(); w = w.cpu().numpy()
    assert np.all(np.diff(x) > 0) and np.array_equal(x, -x[::-1]) and np.array_equal(w, w[::-1])
    assert abs(w.sum() - 2.0) < 1e-12
    assert abs(np.sum(w * x ** 2) - 2.0 / 3.0) < 1e-12 and abs(np.sum(w * x ** 40) - 2.0 / 41.0) < 1e-12
    for i in (0, 1, 777, 40000, n // 2 - 1, n // 2, n - 2):
        xo, wo = orc.gl_node(n, i)
        # the recurrence at n = 2^17 carries ~n*eps of rounding in P_n': edge weights agree to ~1e-9 only (both sides)
        assert abs(x[i] - xo) < 5e-15 and abs(w[i] - wo) <= 2e-8 * wo


def test_schwinger_matches_oracle_and_closed_form(orc):
    torch = _torch()
    from paper_1206_1779_b200 import Dse
    from paper_1206_1779_b200.binding import DseParams
    N, eps2, L2 = 64, 1e-6, 1e4
    p, c = _massive_propagator_coefficients(orc, N, eps2, L2)
    prm = DseParams(N, 8, 8, 1, eps2, L2, 1.0, 3.0, 1.0, 1.0, -9.0 / 44.0, 0.0, 1.0, 0.0, 0, 0)
    d = Dse(prm)
    t = np.linspace(0.1, 8.0, 37)
    n_nodes = 3000                                           # ragged: not a multiple of the block size
    out = d.schwinger(torch.from_numpy(c[None, :]).cuda(), torch.from_numpy(t).cuda(), n_nodes, 1e-16, L2)
    torch.cuda.synchronize()
    out = out.cpu().numpy()[0]
    ref = orc.schwinger(p, c, n_nodes, 1e-16, L2, t)
    assert np.allclose(out, ref, rtol=1e-10, atol=1e-13)
    big = t >= 0.5                                          # cutoff tail ~ sin(t p_max)/(pi t p_max^2) <= 6.4e-5 there
    assert np.allclose(out[big], np.exp(-t[big]) / 2, rtol=0, atol=7e-5)      # sigma = 1/(p^2+1): exp(-t)/2
    d.close()


def test_schwinger_full_size_2p17_nodes(orc):
    """The paper's size (fn.13): 2^17 device-generated Gauss-Legendre nodes, Delta(t) against the
    oracle on the same rule (its O(n^2) node table spread over the host cores, sums serial) and, with the two cut pieces
    of the momentum window added, against the textbook exp(-t)/2 to 1e-10."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse
    from paper_1206_1779_b200.binding import DseParams
    from test_oracle_path import schwinger_cut_pieces
    N, eps2, L2 = 128, 1e-8, 1e4
    p, c = _massive_propagator_coefficients(orc, N, eps2, L2)
    prm = DseParams(N, 8, 8, 1, eps2, L2, 1.0, 3.0, 1.0, 1.0, -9.0 / 44.0, 0.0, 1.0, 0.0, 0, 0)
    d = Dse(prm)
    t = np.array([0.0, 0.1, 0.5, 1.0, 3.0, 4.7, 6.0, 8.0])
    n_nodes = 1 << 17
    out = d.schwinger(torch.from_numpy(c[None, :]).cuda(), torch.from_numpy(t).cuda(), n_nodes, 1e-20, L2)
    torch.cuda.synchronize()
    out = out.cpu().numpy()[0]
    ref = orc.schwinger_threads(p, c, n_nodes, 1e-20, L2, t)
    # node weights of the 2^17 rule carry ~n*eps of recurrence rounding on both sides (test above): 1e-9 relative
    assert np.allclose(out, ref, rtol=2e-9, atol=1e-12), np.abs(out - ref).max()
    pos = t > 0
    assert np.allclose(out[pos] + schwinger_cut_pieces(t[pos], 1e-20, L2), np.exp(-t[pos]) / 2, rtol=0, atol=2e-9)
    d.close()


def test_schwinger_batched_random_dressings(orc):
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload, draw_coefficients
    w = Workload("schw", 24, 8, 8, 1e-6, 5e4, n_batch=3)
    c = np.stack([draw_coefficients(70 + b, 24) for b in range(3)])
    d = Dse(params_from_workload(w))
    t = np.array([0.0, 0.3, 1.7, 5.0, 12.0])
    out = d.schwinger(torch.from_numpy(c).cuda(), torch.from_numpy(t).cuda(), 2048, 1e-10, 2e5)
    torch.cuda.synchronize()
    out = out.cpu().numpy()
    for b in range(3):
        ref = orc.schwinger(oracle_params(w), c[b], 2048, 1e-10, 2e5, t)
        assert np.allclose(out[b], ref, rtol=1e-10, atol=1e-12 * np.abs(ref).max())
    d.close()


def test_dressing_functions_and_coupling_parity(orc):
    """dse_dressing: ln G, ln Z (series eq.(23),(24) + continuations eq.(16)-(19)) and alpha(x) = alpha(mu^2) G^2 Z (L145)
    at momenta below eps2, inside the grid, at both matching points and above L2, for several systems."""
    import math
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload, draw_coefficients
    w = Workload("dress", 24, 16, 32, 1e-6, 5e4, x_G=1.0, x_Z=1.0, alpha_mu=0.7)
    B = 3
    p = oracle_params(w)
    c = np.stack([draw_coefficients(70 + b, w.n_cheb) for b in range(B)])
    x = np.concatenate([np.logspace(-12, -6, 9), [w.eps2, w.L2], np.logspace(-5.9, 4.6, 40), np.logspace(4.7, 5.3, 7),
                        [w.eps2 * (1 - 1e-12), w.L2 * (1 + 1e-12)]])
    d = Dse(params_from_workload(w, n_batch=B))
    lnG, lnZ, al = (t.cpu().numpy() for t in d.dressing(torch.from_numpy(c).cuda(), torch.from_numpy(x).cuda()))
    for b in range(B):
        for m, xv in enumerate(x):
            g, z = orc.ln_dress(p, c[b], float(xv))
            assert abs(lnG[b, m] - g) <= 1e-12 * max(1.0, abs(g)), (b, xv)
            assert abs(lnZ[b, m] - z) <= 1e-12 * max(1.0, abs(z)), (b, xv)
            assert abs(al[b, m] - 0.7 * math.exp(2 * g + z)) <= 1e-11 * al[b, m]
    # infrared power laws of the continuation: d ln G / d ln x = ir_exp_G, d ln Z / d ln x = ir_exp_Z below eps2
    i0, i1 = 0, 5
    dl = math.log(x[i1] / x[i0])
    assert abs((lnG[0, i1] - lnG[0, i0]) / dl - w.ir_exp_G) < 1e-10 and abs((lnZ[0, i1] - lnZ[0, i0]) / dl - w.ir_exp_Z) < 1e-10
    d.close()
