"""GPU LU / Newton step against the oracle's."""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from test_gpu_parity import oracle_params, _torch   # noqa: E402


def check_lu_stats(st, so, ties=False, ctx=None):
    """Parity bar of the one-CTA LU (2N <= 128): it fuses its updates and multiplies by a reciprocal, so it
    is NOT bit-identical to the plain C elimination.  The equilibration is the same arithmetic: max|F| scaled agrees
    exactly.  Without ties in the pivot search the pivot sequence is the oracle's, hence the smallest pivot and the growth
    factor agree to rounding: |d pmin| <= 1e-9 pmin + 1e-12 max|U| (scaled units: max|A| = 1, so max|U| = growth) and
    growth to 1e-11 relative.  With exact ties in the search (small-integer matrices) rounding may order two equal
    candidates differently on the two sides: then only sanity is asserted here and the unknowns carry the parity."""
    assert st[1] == so[1], (ctx, st, so)
    if ties:
        assert st[2] > 0.0 and st[3] >= 1.0 - 1e-12, (ctx, st, so)
        return
    assert abs(st[2] - so[2]) <= 1e-9 * so[2] + 1e-12 * so[3], (ctx, st, so)
    assert abs(st[3] - so[3]) <= 1e-11 * so[3], (ctx, st, so)


def test_lu_solve_matches_oracle(orc):
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import CONFIGS
    d = Dse(params_from_workload(CONFIGS[0]))
    rng = np.random.default_rng(5)
    for n in (1, 2, 16, 64, 128):      # n > 128 needs the handle's own scratch (n = 2N only): test_lu_cluster_* below
        A = rng.normal(size=(3, n, n)) * 10.0 ** rng.uniform(-8, 8, size=(3, n, 1))
        b = rng.normal(size=(3, n)) * np.abs(A).max(axis=2)
        x, st = d.lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x = x.cpu().numpy(); st = st.cpu().numpy()
        for s in range(3):
            xo, so, rc = orc.lu_solve(A[s], b[s])
            assert rc == 0
            assert np.allclose(x[s], xo, rtol=1e-9, atol=1e-13 * np.abs(xo).max())
            assert abs(st[s][0] - so[0]) <= 1e-9 * so[0]
            check_lu_stats(st[s], so, ctx=n)
    # frequent ties in the pivot search (small integer entries): any maximal element is a valid pivot
    for n in (24, 64, 100):
        A = rng.integers(-3, 4, size=(2, n, n)).astype(np.float64) + 7.0 * np.eye(n)
        b = rng.integers(-5, 6, size=(2, n)).astype(np.float64)
        x, st = d.lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x = x.cpu().numpy(); st = st.cpu().numpy()
        for s in range(2):
            xo, so, rc = orc.lu_solve(A[s], b[s])
            assert rc == 0
            assert np.allclose(x[s], xo, rtol=1e-9, atol=1e-13 * np.abs(xo).max())
            check_lu_stats(st[s], so, ties=True, ctx=n)
    d.close()


def test_newton_trajectory_weak_coupling(orc):
    """Same start, same steps: iterates agree while cond*1e-16 allows; quadratic convergence (L226)."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
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


def test_config2_newton_trajectory_literal(orc):
    """BASELINE configs[2] run literally (start G = Z = 1, rho = 1).  DESIGN.md reading A17: the iteration
    does not converge from this start on [1e-10, 1e10]; parity = the same trajectory as the oracle while
    cond(J)*eps allows, and the same verdict."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import config_inputs
    w, c, bc = config_inputs(2)
    d = Dse(params_from_workload(w))
    p = oracle_params(w)
    c_o = c[0].copy()
    c_g = torch.from_numpy(c).cuda()
    bt = torch.from_numpy(bc).cuda()
    # step 0: J and F themselves agree to the parity tolerance
    J, F = d.jacobian(c_g, bt)
    Fo, Jo = orc.residual_jacobian(p, c_o, 1.0, 1.0)
    assert np.linalg.norm(J.cpu().numpy()[0] - Jo) <= 1e-10 * np.linalg.norm(Jo)
    # F at G = Z = 1: the two gluon loops cancel exactly in the continuum for y >> x (fn.5 L127), so the small-x
    # rows of F are the rounding noise of sums whose terms are ~1e19: the fp64 oracle differs from its own
    # long-double build by O(1) there (tests/test_oracle_path.py::test_config2_start_is_ill_conditioned).  The
    # attainable bar is the conditioning-aware one: |dF_i| <= 1e-12 (|F_i| + ||J_i||).
    Fg = F.cpu().numpy()[0]
    assert (np.abs(Fg - Fo) / (np.abs(Fo) + np.linalg.norm(Jo, axis=1))).max() <= 1e-12
    N = w.n_cheb
    assert np.linalg.norm(Fg[N:] - Fo[N:]) <= 1e-10 * np.linalg.norm(Fo[N:])       # ghost rows: no cancellation
    c_o, so, rc = orc.newton_step(p, c_o, 1.0, 1.0, 1.0)
    st = d.newton_step(c_g, bt, 1.0).cpu().numpy()[0]
    # the first update is large (|Delta| >> 1): the literal start is far outside the convergence basin
    assert so[0] > 1.0 and st[0] > 1.0
    # both sides report the same ill-conditioning (min pivot of the row-scaled matrix)
    assert st[2] < 1e-8 and so[2] < 1e-8
    d.close()


def test_finite_difference_self_check_mode(orc):
    """NEXT f3: the paper's own Jacobian definition, eq.(38), as a GPU self-check of the analytic matrix."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import config_inputs
    w, c, bc = config_inputs(0)
    d = Dse(params_from_workload(w))
    ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()
    J, F = d.jacobian(ct, bt)
    Jfd = d.jacobian_fd(ct, bt, 1e-6)
    torch.cuda.synchronize()
    J = J.cpu().numpy()[0]; Jfd = Jfd.cpu().numpy()[0]
    assert np.linalg.norm(J - Jfd) <= 1e-8 * np.linalg.norm(J)
    assert (np.linalg.norm(J - Jfd, axis=1) / np.linalg.norm(J, axis=1)).max() < 1e-7
    # same differences as the oracle's own finite differences
    p = oracle_params(w)
    n = 2 * w.n_cheb
    Jo = np.empty((n, n))
    for j in range(n):
        h = 1e-6 * max(1.0, abs(c[0, j]))
        cp = c[0].copy(); cp[j] += h
        cm = c[0].copy(); cm[j] -= h
        Jo[:, j] = (orc.residual_jacobian(p, cp, 1, 1, jac=False) - orc.residual_jacobian(p, cm, 1, 1, jac=False)) / ((c[0, j] + h) - (c[0, j] - h))
    assert (np.linalg.norm(Jfd - Jo, axis=1) / np.linalg.norm(Jo, axis=1)).max() < 1e-6
    d.close()


def test_lu_random_sizes(orc):
    """Random sizes, scalings, tie-rich and singular matrices through the one-CTA panel LU (every padded size 32, 64, 96,
    128, ragged last panels): solution within conditioning, statistics at the bar of check_lu_stats."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import CONFIGS
    d = Dse(params_from_workload(CONFIGS[0]))
    rng = np.random.default_rng(11)
    for it in range(60):
        n = int(rng.choice([1, 2, 3, 7, 8, 9, 15, 16, 17, 31, 32, 33, 40, 63, 64, 65, 72, 100, 120, 127, 128]))
        kind = int(rng.integers(0, 4))
        if kind == 0:
            A = rng.normal(size=(2, n, n))
        elif kind == 1:
            A = rng.normal(size=(2, n, n)) * 10.0 ** rng.uniform(-8, 8, size=(2, n, 1))
        elif kind == 2:
            A = rng.integers(-2, 3, size=(2, n, n)).astype(np.float64) + 5.0 * np.eye(n)
        else:
            A = rng.normal(size=(2, n, n))
            if n > 2:
                A[:, :, n // 2] = 0.0                      # a zero column: singular, the column is skipped
        b = rng.normal(size=(2, n)) * np.abs(A).max(axis=2).clip(1e-300)
        x, st = d.lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x = x.cpu().numpy(); st = st.cpu().numpy()
        for s in range(2):
            xo, so, rc = orc.lu_solve(A[s], b[s])
            if rc == 0:
                assert np.allclose(x[s], xo, rtol=1e-7, atol=1e-10 * np.abs(xo).max()), (n, kind)
                check_lu_stats(st[s], so, ties=kind == 2, ctx=(n, kind))
            else:      # exactly singular: min |pivot| == 0 on both sides, and the library flags it with |Delta|_inf = +Inf
                assert np.array_equal(st[s][1:3], so[1:3]) and so[2] == 0.0 and np.isinf(st[s][0]), (n, kind, st[s], so)
    d.close()


def test_newton_steps_batched_systems(orc):
    """Eight systems per handle (tensor-path build + one LU CTA per system): every system follows the oracle's iterates."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("newton-weak-batch", 10, 48, 32, 1e-2, 1e2, x_G=1.0, x_Z=1.0, alpha_mu=0.05)
    B = 8
    d = Dse(params_from_workload(w, n_batch=B)); assert d.kernel_info()["variant"] == "batched-dmma"
    p = oracle_params(w)
    c0 = np.zeros((B, 20))                                   # G = Z = 1; the systems differ in their boundary values
    bcs = np.stack([[1.0 + 0.001 * b, 1.0 - 0.0005 * b] for b in range(B)])     # inside the basin of plain Newton steps
    c_g = torch.from_numpy(c0.copy()).cuda(); bc_g = torch.from_numpy(bcs).cuda()
    c_o = c0.copy()
    for it in range(8):
        st = d.newton_step(c_g, bc_g, 1.0).cpu().numpy()
        for b in range(B):
            c_o[b], so, rc = orc.newton_step(p, c_o[b], bcs[b, 0], bcs[b, 1], 1.0)
            assert rc == 0 and abs(st[b, 0] - so[0]) <= 1e-9 * so[0] + 1e-12
        assert np.allclose(c_g.cpu().numpy(), c_o, rtol=0, atol=1e-9 * np.abs(c_o).max())
    assert st[:, 0].max() < 1e-8                             # every system converges quadratically
    d.close()


@pytest.mark.parametrize("N", [65, 80, 96, 128])
def test_lu_cluster_path_exact_factorisation(orc, N):
    """128 < 2N <= 256: the register-resident LU over a cluster of 4 CTAs (distributed shared memory, split cluster
    barrier).  This kernel keeps unfused updates and correctly rounded quotients: solution within conditioning,
    factorisation bit-identical to the plain C elimination (also with ties: it tracks the textbook row positions)."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    n = 2 * N
    d = Dse(params_from_workload(Workload("lu", n_cheb=N, n_r=4, n_theta=4, eps2=1e-6, L2=1e4), n_batch=3))
    rng = np.random.default_rng(N)
    for kind in range(4):
        if kind == 0:
            A = rng.normal(size=(3, n, n))
        elif kind == 1:
            A = rng.normal(size=(3, n, n)) * 10.0 ** rng.uniform(-8, 8, size=(3, n, 1))
        elif kind == 2:
            A = rng.integers(-2, 3, size=(3, n, n)).astype(np.float64) + 5.0 * np.eye(n)
        else:
            A = rng.normal(size=(3, n, n)); A[:, :, n // 2] = 0.0
        b = rng.normal(size=(3, n)) * np.abs(A).max(axis=2)
        x, st = d.lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x = x.cpu().numpy(); st = st.cpu().numpy()
        for s in range(3):
            xo, so, rc = orc.lu_solve(A[s], b[s])
            if rc == 0:
                assert np.allclose(x[s], xo, rtol=1e-7, atol=1e-10 * np.abs(xo).max()), (n, kind)
                assert np.array_equal(st[s][1:], so[1:]), (n, kind, st[s], so)
            else:      # exactly singular: min |pivot| == 0 on both sides, and the library flags it with |Delta|_inf = +Inf
                assert np.array_equal(st[s][1:3], so[1:3]) and so[2] == 0.0 and np.isinf(st[s][0]), (n, kind, st[s], so)
    d.close()


# ----------------------------------------------------------------------------- dse_newton_solve (device-side iteration)
def test_newton_solve_graph_weak_coupling(orc):
    """The whole iteration as one CUDA graph (WHILE node) against the oracle's plain loop: same number of steps, same
    per-step record, converged coefficients to the north_star bar (1e-9); then the call-level controls."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("newton-weak", 10, 64, 24, 1e-2, 1e2, x_G=1.0, x_Z=1.0, alpha_mu=0.05)
    d = Dse(params_from_workload(w))
    p = oracle_params(w)
    bc = torch.ones((1, 2), dtype=torch.float64, device="cuda")
    c_o, hist, status = orc.newton_solve(p, np.zeros(20), 1.0, 1.0, rho=1.0, step_cap=0.0, tol=1e-12, max_iter=20)
    assert status == 1 and 3 <= len(hist) <= 8
    c_g = torch.zeros((1, 20), dtype=torch.float64, device="cuda")
    info = d.newton_solve(c_g, bc, rho=1.0, step_cap=0.0, tol=1e-12, max_iter=20).cpu().numpy()[0]
    assert info[0] == len(hist) and info[5] == 1.0
    assert abs(info[1] - hist[-1][0]) <= 1e-9 * hist[-1][0] + 1e-12 and info[4] == 1.0
    assert abs(info[3] - min(h[2] for h in hist)) <= 1e-9 * info[3]
    assert np.abs(c_g.cpu().numpy()[0] - c_o).max() <= 1e-9 * np.abs(c_o).max()
    # the same handle again, other scalars (the graph is reused): two steps only -> status 0, equal to two plain steps
    c2 = torch.zeros((1, 20), dtype=torch.float64, device="cuda")
    info2 = d.newton_solve(c2, bc, rho=1.0, step_cap=0.0, tol=1e-12, max_iter=2).cpu().numpy()[0]
    c_s = torch.zeros((1, 20), dtype=torch.float64, device="cuda")
    for _ in range(2):
        st = d.newton_step(c_s, bc, 1.0)
    assert info2[0] == 2 and info2[5] == 0.0
    assert np.abs((c2 - c_s).cpu().numpy()).max() <= 1e-15 * np.abs(c_o).max()
    assert info2[1] == st.cpu().numpy()[0, 0]
    # tol = 0: exactly max_iter steps; under-relaxation rho = 0.5 without a cap follows the oracle
    c3 = torch.zeros((1, 20), dtype=torch.float64, device="cuda")
    info3 = d.newton_solve(c3, bc, rho=0.5, step_cap=0.0, tol=0.0, max_iter=6).cpu().numpy()[0]
    c_o3, hist3, status3 = orc.newton_solve(p, np.zeros(20), 1.0, 1.0, rho=0.5, step_cap=0.0, tol=0.0, max_iter=6)
    assert info3[0] == 6 and info3[5] == 0.0 and status3 == 0 and info3[4] == 0.5
    assert np.abs(c3.cpu().numpy()[0] - c_o3).max() <= 1e-9 * np.abs(c_o3).max()
    # argument checks
    import ctypes
    from paper_1206_1779_b200.binding import _dev_ptr, _stream_ptr
    for bad in [(0.0, 0.0, 1e-12, 5), (1.5, 0.0, 1e-12, 5), (1.0, 0.0, -1.0, 5), (1.0, 0.0, 1e-12, 0), (float("nan"), 0.0, 1e-12, 5)]:
        rc = d.lib.dse_newton_solve(d._h, _dev_ptr(c3), _dev_ptr(bc), ctypes.c_double(bad[0]), ctypes.c_double(bad[1]),
                                    ctypes.c_double(bad[2]), bad[3], None, _stream_ptr())
        assert rc == -1, bad
    d.close()


def test_newton_solve_graph_batched_systems(orc):
    """Eight systems in one graph: each stops on its own criterion (frozen once converged), the loop ends with the
    last one; every system matches its own oracle solve."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("newton-weak-batch", 10, 48, 32, 1e-2, 1e2, x_G=1.0, x_Z=1.0, alpha_mu=0.05)
    B = 8
    d = Dse(params_from_workload(w, n_batch=B))
    p = oracle_params(w)
    bcs = np.stack([[1.0 + 0.001 * b, 1.0 - 0.0005 * b] for b in range(B)])     # inside the basin of plain Newton steps
    c0 = np.zeros((B, 20))                                   # G = Z = 1 ...
    c0[3] = orc.newton_solve(p, c0[3], bcs[3, 0], bcs[3, 1], tol=1e-13, max_iter=25)[0]   # ... but system 3 starts converged
    c_g = torch.from_numpy(c0.copy()).cuda()
    info = d.newton_solve(c_g, torch.from_numpy(bcs).cuda(), rho=1.0, step_cap=0.5, tol=1e-10, max_iter=25).cpu().numpy()
    c = c_g.cpu().numpy()
    steps = []
    for b in range(B):
        c_o, hist, status = orc.newton_solve(p, c0[b], bcs[b, 0], bcs[b, 1], rho=1.0, step_cap=0.5, tol=1e-10, max_iter=25)
        assert status == 1 and info[b, 5] == 1.0
        assert info[b, 0] == len(hist), (b, info[b], len(hist))
        assert np.abs(c[b] - c_o).max() <= 1e-9 * np.abs(c_o).max()
        steps.append(len(hist))
    assert steps[3] == 1 and len(set(steps)) >= 3            # the systems really stop at different steps
    d.close()


def test_newton_solve_graph_paper_scaling_solution(orc):
    """The paper's own parameter set (L135, L364) solved by ONE call: same step count and converged coefficients as
    the oracle's loop with the same relaxation rule (reading A26), and the paper's printed alpha(M_Z^2), alpha(0)."""
    torch = _torch()
    import math
    import scaling_setup as S
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("paper-scaling", S.N, S.N_R, S.N_THETA, S.EPS2, S.L2, x_G=0.0, x_Z=S.L2, n_ir=S.N_IR)
    p = oracle_params(w)
    c0 = S.start_coefficients(orc, p)
    c_o, hist, status = orc.newton_solve(p, c0, S.G_G, S.G_Z, rho=1.0, step_cap=S.STEP_CAP, tol=1e-11, max_iter=30)
    assert status == 1
    d = Dse(params_from_workload(w, flags=1))
    c_g = torch.from_numpy(c0[None, :].copy()).cuda()
    bc = torch.tensor([[S.G_G, S.G_Z]], dtype=torch.float64, device="cuda")
    info = d.newton_solve(c_g, bc, rho=1.0, step_cap=S.STEP_CAP, tol=1e-11, max_iter=30).cpu().numpy()[0]
    assert info[5] == 1.0 and info[0] == len(hist)
    c = c_g.cpu().numpy()[0]
    assert np.abs(c - c_o).max() <= 1e-9 * np.abs(c_o).max()

    # the coupling at M_Z^2 and its infrared fixed point, evaluated on the device (dse_dressing)
    xs = torch.tensor([91.2 ** 2, S.EPS2, 1e-9, 1e-8], dtype=torch.float64, device="cuda")
    lnG, lnZ, al = (t.cpu().numpy()[0] for t in d.dressing(c_g, xs))
    assert abs(al[0] - 0.118) < 1e-3 and abs(al[1] - 2.972) < 5e-3
    g, z = orc.ln_dress(p, c, 91.2 ** 2)
    assert abs(al[0] - math.exp(2 * g + z)) < 1e-12
    kap = -(lnG[3] - lnG[2]) / math.log(10.0)               # G ~ x^-kappa below eps2 (eq.(17))
    assert abs(kap - S.KAPPA) < 1e-9
    d.close()


def test_newton_solve_graph_paper_solution_family(orc):
    """PAPER.md L139-151 (Fig. 3, 4): the scaling solution and the two decoupling solutions G(x_G = 0)^-1 = 0, 0.01, 0.1 of the
    paper's parameter set as ONE dse_newton_solve call with three systems.  Three systems are below the batch size of the
    tensor-path kernel (n_batch >= 8), so this runs the per-system one-kernel builds and one LU CTA per system inside
    the graph (the test says which variant ran); the members stop after different numbers of steps (per-system freeze).
    Same step counts and converged coefficients as the oracle's loops; the printed facts are pinned on the oracle side
    by tests/test_oracle_path.py::test_paper_decoupling_solutions_P13 and re-read here from the device."""
    torch = _torch()
    import scaling_setup as S
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("paper-family", S.N, S.N_R, S.N_THETA, S.EPS2, S.L2, x_G=0.0, x_Z=S.L2, n_ir=S.N_IR)
    p = oracle_params(w)
    c0 = S.start_coefficients(orc, p)
    gGs = [0.0, 0.01, 0.1]
    ref = [orc.newton_solve(p, c0.copy(), gG, S.G_Z, rho=1.0, step_cap=S.STEP_CAP, tol=1e-11, max_iter=40) for gG in gGs]
    assert all(r[2] == 1 for r in ref)
    d = Dse(params_from_workload(w, n_batch=3, flags=1))
    assert d.kernel_info()["variant"] == "pipelined"
    c_g = torch.from_numpy(np.stack([c0, c0, c0])).cuda()
    bc = torch.tensor([[gG, S.G_Z] for gG in gGs], dtype=torch.float64, device="cuda")
    info = d.newton_solve(c_g, bc, rho=1.0, step_cap=S.STEP_CAP, tol=1e-11, max_iter=40).cpu().numpy()
    c = c_g.cpu().numpy()
    steps = []
    for b, (c_o, hist, status) in enumerate(ref):
        assert info[b, 5] == 1.0 and info[b, 0] == len(hist), (b, info[b], len(hist))
        assert np.abs(c[b] - c_o).max() <= 1e-9 * np.abs(c_o).max(), b
        steps.append(int(info[b, 0]))
    assert len(set(steps)) == 3                                       # 9, 11 and 15 steps: every member froze on its own
    xs = torch.tensor([91.2 ** 2, S.EPS2, 1e-5], dtype=torch.float64, device="cuda")
    lnG, lnZ, al = (t.cpu().numpy() for t in d.dressing(c_g, xs))
    assert np.all(np.abs(al[:, 0] - 0.118) < 1e-3)                    # alpha(M_Z^2), fn.7: all three members
    assert abs(al[0, 1] - 2.972) < 5e-3                               # scaling: infrared fixed point (L151)
    assert al[1, 1] < 0.02 and al[2, 1] < 1e-3 and np.all(al[1:, 1] < al[1:, 2])    # decoupling: alpha vanishes in the infrared
    assert 0.98 / 0.01 < math.exp(lnG[1, 1]) <= 1 / 0.01 and 0.98 / 0.1 < math.exp(lnG[2, 1]) <= 1 / 0.1      # finite G(0) = 1/g_G
    d.close()


def test_newton_solve_graph_large_system_cluster_lu(orc):
    """2N = 144: inside the solve graph the Newton update runs on the cluster LU (4 CTAs, distributed shared memory);
    same steps and coefficients as the oracle's loop."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload
    w = Workload("newton-weak-72", 72, 96, 32, 1e-2, 1e2, x_G=1.0, x_Z=1.0, alpha_mu=0.05)
    d = Dse(params_from_workload(w))
    p = oracle_params(w)
    c_o, hist, status = orc.newton_solve(p, np.zeros(144), 1.0, 1.0, rho=1.0, step_cap=0.0, tol=1e-10, max_iter=12)
    assert status == 1
    c_g = torch.zeros((1, 144), dtype=torch.float64, device="cuda")
    bc = torch.ones((1, 2), dtype=torch.float64, device="cuda")
    info = d.newton_solve(c_g, bc, tol=1e-10, max_iter=12).cpu().numpy()[0]
    assert info[5] == 1.0 and info[0] == len(hist)
    assert np.abs(c_g.cpu().numpy()[0] - c_o).max() <= 1e-9 * np.abs(c_o).max()
    d.close()


def test_lu_extreme_exponents(orc):
    """Entries far outside 2^+-500 after equilibration (columns scaled by 1e-200 / 1e-180, a 1e150 row): the reciprocal of
    the pivot stays in range (normal pivots down to 2^-1022) and the factorisation stays at the bar of check_lu_stats
    (the smallest pivot, ~1e-200, to 1e-9 RELATIVE)."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import CONFIGS
    d = Dse(params_from_workload(CONFIGS[0]))
    rng = np.random.default_rng(77)
    for n in (8, 40, 64, 128):
        A = rng.normal(size=(2, n, n))
        A[:, :, 1] *= 1e-200                                     # tiny column: quotients of tiny numbers
        A[:, :, n // 2] *= 1e-180
        A[:, n // 3, :] *= 1e150                                 # a huge row (removed by the equilibration)
        b = rng.normal(size=(2, n))
        x, st = d.lu_solve(torch.from_numpy(A).cuda(), torch.from_numpy(b).cuda())
        x = x.cpu().numpy(); st = st.cpu().numpy()
        for s in range(2):
            xo, so, rc = orc.lu_solve(A[s], b[s])
            assert st[s][1] == so[1] and abs(st[s][2] - so[2]) <= 1e-9 * so[2] and abs(st[s][3] - so[3]) <= 1e-11 * so[3], (n, st[s], so)
            assert np.allclose(x[s], xo, rtol=1e-6, atol=0), n
    d.close()
