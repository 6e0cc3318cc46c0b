"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element on the same
seeded inputs.  Tolerance: BASELINE.json north_star -- <= 1e-10 normwise relative error on J and F;
we additionally bound the worst row-wise relative error (one row dominates the normwise number,
row norms span ~19 decades) at 1e-9."""
import ctypes

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_NORM = 1e-10
TOL_ROW = 1e-9


def _torch():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


def oracle_params(w):
    from oracle.oracle import make_params
    return make_params(w.n_cheb, w.n_r, w.n_theta, w.eps2, w.L2, w.x_G, w.x_Z, w.alpha_mu, w.n_colors, w.delta,
                       w.ir_exp_G, w.ir_exp_Z, w.uv_omega, getattr(w, "angular_rule", 0), getattr(w, "n_ir", 0), getattr(w, "radial_split", 0))


def gpu_build(w, c, bc, flags=0, jac=True):
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    d = Dse(params_from_workload(w, n_batch=c.shape[0], flags=flags))
    ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()
    if jac:
        J, F = d.jacobian(ct, bt)
        torch.cuda.synchronize()
        out = J.cpu().numpy(), F.cpu().numpy()
    else:
        F = d.residual(ct, bt)
        torch.cuda.synchronize()
        out = None, F.cpu().numpy()
    d.close()
    return out


def check(J, F, Jo, Fo, label=None):
    assert np.all(np.isfinite(J)) and np.all(np.isfinite(F))
    en = np.linalg.norm(J - Jo) / np.linalg.norm(Jo)
    ef = np.linalg.norm(F - Fo) / np.linalg.norm(Fo)
    er = (np.linalg.norm(J - Jo, axis=1) / np.linalg.norm(Jo, axis=1)).max()
    # row-wise F: F_i is a difference of sums that are up to 1e19 times larger than itself, so its attainable accuracy is
    # set by the size of what was summed -- |F_i| + |J_i| measures that (conditioning-aware metric, asserted); the plain
    # |dF_i|/|F_i| maximum is printed beside it for the reader (pytest -s / -rP shows it)
    efr = (np.abs(F - Fo) / (np.abs(Fo) + np.linalg.norm(Jo, axis=1))).max()
    efp = (np.abs(F - Fo) / np.maximum(np.abs(Fo), 1e-300)).max()
    if label is not None:
        print(f"parity {label}: |dJ|/|J| = {en:.2e}, |dF|/|F| = {ef:.2e}, worst J row = {er:.2e}, "
              f"worst F row: plain |dF_i|/|F_i| = {efp:.2e}, conditioning-aware = {efr:.2e}")
    assert en <= TOL_NORM and ef <= TOL_NORM, (en, ef)
    assert er <= TOL_ROW and efr <= TOL_ROW, (er, efr)
    return en, ef, er


@pytest.mark.parametrize("flags", [0, 1])
@pytest.mark.parametrize("cfg", [0, 1])
def test_configs_0_1_full_parity(orc, cfg, flags):
    from workloads import config_inputs
    w, c, bc = config_inputs(cfg)
    Fo, Jo = orc.residual_jacobian(oracle_params(w), c[0], bc[0, 0], bc[0, 1])
    J, F = gpu_build(w, c, bc, flags)
    check(J[0], F[0], Jo, Fo, label=f"cfg {cfg} flags {flags}")
    # residual-only entry point gives the same F
    _, F2 = gpu_build(w, c, bc, flags, jac=False)
    assert np.allclose(F2, F, rtol=1e-12, atol=0)      # different template instance: same math, other rounding


def test_tables_match_oracle(orc):
    _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import CONFIGS
    for cfg in (0, 3):
        w = CONFIGS[cfg]
        d = Dse(params_from_workload(w))
        t = d.tables(); d.close()
        o = orc.tables(oracle_params(w))
        # x = eps2 exp((s+1) Lg/2): the double-precision oracle carries ~Lg*eps of relative error
        assert np.allclose(t["x_ext"], o["x_ext"], rtol=1e-13)
        assert np.allclose(t["y"], o["y"], rtol=1e-13)
        assert np.allclose(t["Wy"], o["Wy"], rtol=1e-11)
        assert np.allclose(t["theta"], o["theta"], rtol=1e-14)
        assert np.allclose(t["Omega"], o["Omega"], rtol=1e-11)


@pytest.mark.parametrize("shape", [
    dict(n_cheb=5, n_r=7, n_theta=3),          # ragged everything: N not a multiple of 8, odd rows, g = 4 with padding
    dict(n_cheb=12, n_r=33, n_theta=21),       # NCH = 2, g = 32 with 11 padded lanes
    dict(n_cheb=36, n_r=20, n_theta=40),       # paper's N = 36: NCH = 5 (non power of two), two angular batches
    dict(n_cheb=2, n_r=2, n_theta=2),          # minimum sizes
    dict(n_cheb=16, n_r=40, n_theta=32, x_G=3.0, x_Z=5e3),   # distinct subtraction points (N_ext = N + 2)
    dict(n_cheb=128, n_r=6, n_theta=8),        # maximum N
    dict(n_cheb=20, n_r=12, n_theta=32),       # NCH = 3: pipelined kernel with idle phase-2 lanes (30 of 32)
    dict(n_cheb=48, n_r=10, n_theta=64),       # NCH = 6
    dict(n_cheb=52, n_r=9, n_theta=32),        # NCH = 7
    dict(n_cheb=96, n_r=5, n_theta=32),        # the paper's N = 96: NCH = 12, 24 of 32 lanes
    dict(n_cheb=128, n_r=4, n_theta=32),       # maximum N with full-warp angular batches: fewer warps per CTA (shared memory)
])
def test_ragged_and_edge_shapes(orc, shape):
    from workloads import Workload, draw_coefficients
    kw = dict(eps2=1e-6, L2=5e4)
    kw.update(shape)
    w = Workload("edge", **kw)
    c = draw_coefficients(17, w.n_cheb)[None, :]
    bc = np.array([[0.8, 1.7]])
    Fo, Jo = orc.residual_jacobian(oracle_params(w), c[0], 0.8, 1.7)
    for flags in (0, 1):
        J, F = gpu_build(w, c, bc, flags)
        check(J[0], F[0], Jo, Fo)


def test_batched_systems(orc):
    """config 4 at reduced batch: every system against the oracle."""
    from workloads import config_inputs
    w, c, bc = config_inputs(4, n_batch=5)
    J, F = gpu_build(w, c, bc)
    for b in range(5):
        Fo, Jo = orc.residual_jacobian(oracle_params(w), c[b], bc[b, 0], bc[b, 1])
        check(J[b], F[b], Jo, Fo)


@pytest.mark.parametrize("shape,B", [
    (dict(n_cheb=32, n_r=24, n_theta=64), 16),                              # two angular batches per row
    (dict(n_cheb=27, n_r=9, n_theta=40, x_G=3.0, x_Z=5e3), 16),             # padded j and theta, N_ext = N + 2
    (dict(n_cheb=30, n_r=8, n_theta=32, n_ir=6, radial_split=1, x_G=0.0), 16),   # per-point rules, infrared piece, x_G = 0
    (dict(n_cheb=12, n_r=10, n_theta=32), 13),                              # 16-index tiles; batch padded 13 -> 16
    (dict(n_cheb=36, n_r=8, n_theta=64), 8),                                # the paper's N = 36: 48-index tiles, N_pad = 40
    (dict(n_cheb=60, n_r=6, n_theta=32), 14),                               # the paper's N = 60: 64-index tiles, 14 -> 16
])
def test_batched_tensor_path_every_system(orc, shape, B, monkeypatch):
    """n_batch >= 8 and N <= 64: eight systems per warp on the fp64 tensor path (mma.sync m8n8k4).
    Every system against the oracle, both geometry modes, and against the per-system kernel of the same library."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload, draw_coefficients
    kw = dict(eps2=1e-6, L2=5e4); kw.update(shape)
    w = Workload("batched", **kw)
    c = np.stack([draw_coefficients(100 + b, w.n_cheb) for b in range(B)])
    bc = np.stack([[0.5 + 0.05 * b, 1.2 + 0.03 * b] for b in range(B)])
    d = Dse(params_from_workload(w, n_batch=B)); assert d.kernel_info()["variant"] == "batched-dmma"; d.close()
    Js = []
    for flags in (0, 1):
        J, F = gpu_build(w, c, bc, flags)
        Js.append(J)
        for b in range(B):
            Fo, Jo = orc.residual_jacobian(oracle_params(w), c[b], bc[b, 0], bc[b, 1])
            check(J[b], F[b], Jo, Fo)
        _, F2 = gpu_build(w, c, bc, flags, jac=False)          # dse_residual: the residual-only variant of the kernel
        assert np.allclose(F2, F, rtol=1e-12, atol=0)
    # DSE_FLAG_PER_SYSTEM_KERNELS (a dse_params flag, not an environment switch): the same batch through the single-system kernels
    from paper_1206_1779_b200 import DSE_FLAG_PER_SYSTEM_KERNELS
    d = Dse(params_from_workload(w, n_batch=B, flags=DSE_FLAG_PER_SYSTEM_KERNELS))
    assert d.kernel_info()["variant"] != "batched-dmma"; d.close()
    J1, F1 = gpu_build(w, c, bc, DSE_FLAG_PER_SYSTEM_KERNELS)
    assert np.linalg.norm(J1 - Js[0]) <= 1e-12 * np.linalg.norm(J1)


def test_deterministic_bitwise():
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import config_inputs
    w, c, bc = config_inputs(1)
    d = Dse(params_from_workload(w))
    ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()
    J0, F0 = d.jacobian(ct, bt)
    J0 = J0.clone(); F0 = F0.clone()
    for _ in range(5):
        J, F = d.jacobian(ct, bt)
        assert torch.equal(J, J0) and torch.equal(F, F0)
    assert d.launch_count() == 6 * 1      # cfg 1: ONE kernel per build (H1 in its prologue, H7 + H8 in its tail)
    assert d.kernel_info()["kernels_per_build"] == 1
    d.close()


def test_constant_slot_is_explicit_and_order_independent(orc):
    """DSE_FLAG_CONST_COEF (include/dse.h): the constant-bank coefficient slot is taken only on request; a second
    request while it is held fails with DSE_EBUSY; handles without the flag run the same kernel variant whatever the
    creation order.  All of them match the oracle and each other."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, DseError, params_from_workload, DSE_FLAG_CONST_COEF
    from paper_1206_1779_b200.binding import DSE_EBUSY
    from workloads import config_inputs
    w, c, bc = config_inputs(1)
    Fo, Jo = orc.residual_jacobian(oracle_params(w), c[0], bc[0, 0], bc[0, 1])
    ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()

    def run(d, stream=None):
        if stream is None:
            J, F = d.jacobian(ct, bt)
        else:
            with torch.cuda.stream(stream):
                J, F = d.jacobian(ct * 1.0, bt)
        torch.cuda.synchronize()
        J = J.cpu().numpy()[0]; F = F.cpu().numpy()[0]
        check(J, F, Jo, Fo)
        return J

    for order in (0, 1):                                   # plain handle before / after the slot owner
        if order == 0:
            p1 = Dse(params_from_workload(w)); own = Dse(params_from_workload(w, flags=DSE_FLAG_CONST_COEF))
        else:
            own = Dse(params_from_workload(w, flags=DSE_FLAG_CONST_COEF)); p1 = Dse(params_from_workload(w))
        p2 = Dse(params_from_workload(w))
        i1, i2, io = p1.kernel_info(), p2.kernel_info(), own.kernel_info()
        assert i1 == i2, (i1, i2)                         # equal variants, registers, shared memory: no "first handle wins"
        assert io["variant"] == "pipelined"
        with pytest.raises(DseError) as ei:
            Dse(params_from_workload(w, flags=DSE_FLAG_CONST_COEF))
        assert ei.value.code == DSE_EBUSY
        s2 = torch.cuda.Stream()
        Jo_ = run(own); J1 = run(p1, s2); J2 = run(p2)
        assert np.array_equal(J1, J2)
        assert np.allclose(Jo_, J1, rtol=1e-11, atol=0)
        own.close()
        own = Dse(params_from_workload(w, flags=DSE_FLAG_CONST_COEF))      # released by dse_destroy
        run(own)
        own.close(); p1.close(); p2.close()
    # shapes that cannot use the slot are refused, not silently downgraded
    from workloads import Workload
    with pytest.raises(DseError) as ei:
        Dse(params_from_workload(Workload("odd", 36, 16, 32, 1e-6, 5e4), flags=DSE_FLAG_CONST_COEF))
    assert ei.value.code == -1


def test_alternating_coefficient_sets_back_to_back(orc):
    """Several hundred builds back to back on one handle, alternating two coefficient sets (with and without the
    constant-bank slot): every result must be the one of ITS coefficients -- nothing stale from the build before (the
    constant bank is refreshed by an in-stream copy, the tail's counters are cleared by the build itself)."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload, DSE_FLAG_CONST_COEF, DSE_FLAG_GEOMETRY_CACHE
    from workloads import config_inputs, draw_coefficients
    w, c, bc = config_inputs(1)
    cA = torch.from_numpy(c).cuda(); cB = torch.from_numpy(draw_coefficients(77, w.n_cheb)[None, :]).cuda()
    bt = torch.from_numpy(bc).cuda()
    n2 = 2 * w.n_cheb
    for flags in (DSE_FLAG_CONST_COEF, 0, DSE_FLAG_CONST_COEF | DSE_FLAG_GEOMETRY_CACHE):
        d = Dse(params_from_workload(w, flags=flags))
        JA, FA = d.jacobian(cA, bt); JA = JA.clone(); FA = FA.clone()
        JB, FB = d.jacobian(cB, bt); JB = JB.clone(); FB = FB.clone()
        assert not torch.equal(JA, JB)
        outs = [(torch.empty((1, n2, n2), dtype=torch.float64, device="cuda"), torch.empty((1, n2), dtype=torch.float64, device="cuda"))
                for _ in range(300)]
        for i, (J, F) in enumerate(outs):
            d.jacobian(cA if i % 2 == 0 else cB, bt, J, F)
        torch.cuda.synchronize()
        for i, (J, F) in enumerate(outs):
            assert torch.equal(J, JA if i % 2 == 0 else JB) and torch.equal(F, FA if i % 2 == 0 else FB), (flags, i)
        d.close()
    Fo, Jo = orc.residual_jacobian(oracle_params(w), cB.cpu().numpy()[0], bc[0, 0], bc[0, 1])
    check(JB.cpu().numpy()[0], FB.cpu().numpy()[0], Jo, Fo)


@pytest.mark.parametrize("cfg,split", [(0, 0), (1, 0), (3, 0), (1, 1)])
def test_user_tables_isolate_kernel_error(orc, cfg, split):
    """DSE_FLAG_USER_TABLES (SURVEY 8(b) flags.bit0; PAPER.md L62 never gives the radial node map, so the two table
    builders are independent pieces of code): with the ORACLE's nodes and weights injected, what is left of the J/F
    difference is kernel arithmetic alone (summation order, FMA contraction, exp/log) -- printed beside the error with
    the library's own tables."""
    _torch()
    import dataclasses
    from paper_1206_1779_b200 import Dse, params_from_workload, DSE_FLAG_USER_TABLES
    from workloads import config_inputs
    import torch
    w, c, bc = config_inputs(cfg)
    if split:
        w = dataclasses.replace(w, radial_split=1, n_r=96, name="cfg1-split")
    p = oracle_params(w)
    Fo, Jo = orc.residual_jacobian(p, c[0], bc[0, 0], bc[0, 1])
    ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()
    ot = orc.tables(p)
    if split:      # the oracle's rule of every external point
        ys, Ws = zip(*[orc.radial_rule_split(p, x) for x in ot["x_ext"]])
        ot = dict(ot, y=np.stack(ys), Wy=np.stack(Ws))
    errs = {}
    for name, tabs, fl in (("own tables", None, 0), ("oracle tables", ot, DSE_FLAG_USER_TABLES)):
        d = Dse(params_from_workload(w, flags=fl), tables=tabs)
        if tabs is not None:
            t = d.tables()
            for k in ("x_ext", "y", "Wy", "theta", "Omega"):
                assert np.array_equal(t[k], np.asarray(tabs[k]).reshape(t[k].shape)), k      # taken as they are
        J, F = d.jacobian(ct, bt)
        torch.cuda.synchronize()
        errs[name] = check(J.cpu().numpy()[0], F.cpu().numpy()[0], Jo, Fo)
        d.close()
    print(f"cfg {cfg} split {split}: (|dJ|/|J|, |dF|/|F|, worst J row) with own tables {errs['own tables']}, "
          f"with the oracle's tables {errs['oracle tables']}")
    assert errs["oracle tables"][0] <= 1e-12      # kernel arithmetic alone


def test_config3_full_size_parity(orc):
    """BASELINE configs[3] at full size, in the launch configuration bench.py times (both geometry modes)."""
    from workloads import config_inputs
    w, c, bc = config_inputs(3)
    Fo, Jo = orc.residual_jacobian(oracle_params(w), c[0], bc[0, 0], bc[0, 1])
    for flags in (0, 1):
        J, F = gpu_build(w, c, bc, flags)
        check(J[0], F[0], Jo, Fo, label=f"cfg 3 flags {flags}")


def test_config4_full_batch_every_system(orc):
    """BASELINE configs[4]: all 256 systems built in one launch sequence (the configuration bench.py times), EVERY system
    against the oracle (0.09 s each, spread over the host cores), plus the property that the boundary value only
    shifts F."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    from workloads import config_inputs
    w, c, bc = config_inputs(4)
    assert c.shape[0] == 256
    p = oracle_params(w)
    with ThreadPoolExecutor(max_workers=min(os.cpu_count() or 1, 32)) as pool:      # ctypes releases the GIL
        ref = list(pool.map(lambda b: orc.residual_jacobian(p, c[b], bc[b, 0], bc[b, 1]), range(256)))
    for flags in (0, 1):
        J, F = gpu_build(w, c, bc, flags)
        worst = 0.0
        for b in range(256):
            Fo, Jo = ref[b]
            en, ef, er = check(J[b], F[b], Jo, Fo)
            worst = max(worst, en, ef)
        print(f"parity cfg 4 flags {flags}: worst normwise error over all 256 systems = {worst:.2e}")
    # same coefficients, different boundary value: J identical, ghost rows of F shifted by the difference
    c2 = c.copy(); c2[1] = c2[0]
    J2, F2 = gpu_build(w, c2[:2], bc[:2])
    N = w.n_cheb
    assert np.array_equal(J2[0], J2[1])
    assert np.allclose(F2[1, N:] - F2[0, N:], -(bc[1, 0] - bc[0, 0]), rtol=0, atol=1e-12)
    assert np.array_equal(F2[1, :N], F2[0, :N])


@pytest.mark.parametrize("n_theta", [16, 64, 40, 2, 3])      # 2: both nodes in the tails, next to theta = 0 and pi
def test_tanh_sinh_angular_rule_parity(orc, n_theta):
    """NEXT f3: tanh-sinh rule in xi = cos(theta); only the tables change."""
    _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload, draw_coefficients
    w = Workload("tanh-sinh", 16, 48, n_theta, 1e-6, 5e4, angular_rule=1)
    c = draw_coefficients(23, w.n_cheb)[None, :]
    bc = np.array([[1.1, 0.9]])
    Fo, Jo = orc.residual_jacobian(oracle_params(w), c[0], 1.1, 0.9)
    for flags in (0, 1):
        J, F = gpu_build(w, c, bc, flags)
        check(J[0], F[0], Jo, Fo)
    d = Dse(params_from_workload(w))
    t = d.tables(); d.close()
    o = orc.tables(oracle_params(w))
    assert np.allclose(t["theta"], o["theta"], rtol=1e-13) and np.allclose(t["Omega"], o["Omega"], rtol=1e-12)


def test_random_shapes_against_oracle(orc):
    """Seeded random shapes, batch sizes, rules and flags (every kernel variant gets picked): J, F and the residual-only
    entry point against the oracle.  This sweep found the N = 128 / n_theta >= 32 shared-memory limit and reading A25."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload, draw_coefficients
    rng = np.random.default_rng(2024)
    seen = set()
    for it in range(60):
        N = int(rng.choice([2, 3, 5, 8, 9, 16, 17, 24, 31, 32, 33, 40, 47, 48, 56, 63, 64, 65, 72, 96, 120, 128]))
        nr = int(rng.integers(2, 24)); nt = int(rng.choice([2, 3, 7, 8, 16, 31, 32, 33, 40, 64, 65, 96]))
        B = int(rng.choice([1, 1, 2, 3, 8, 9, 13, 16]))
        if N > 64 and B > 2:
            B = 2
        kw = dict(n_cheb=N, n_r=nr, n_theta=nt, eps2=10.0 ** rng.integers(-12, -3), L2=10.0 ** rng.integers(2, 12))
        if rng.random() < 0.3: kw.update(x_G=3.0, x_Z=5e1)
        if rng.random() < 0.2: kw.update(radial_split=1)
        if rng.random() < 0.2: kw.update(n_ir=int(rng.integers(1, 6)))
        if rng.random() < 0.15: kw.update(x_G=0.0)
        if rng.random() < 0.2: kw.update(angular_rule=1)
        w = Workload("fuzz", **kw)
        flags = int(rng.integers(0, 2))
        c = np.stack([draw_coefficients(1000 * it + b, N) for b in range(B)])
        bc = np.stack([[0.7 + 0.1 * b, 1.3 - 0.05 * b] for b in range(B)])
        d = Dse(params_from_workload(w, n_batch=B, flags=flags)); seen.add(d.kernel_info()["variant"])
        ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()
        J, F = d.jacobian(ct, bt); F2 = d.residual(ct, bt); torch.cuda.synchronize()
        J = J.cpu().numpy(); F = F.cpu().numpy(); F2 = F2.cpu().numpy(); d.close()
        for b in range(min(B, 3)):
            Fo, Jo = orc.residual_jacobian(oracle_params(w), c[b], bc[b, 0], bc[b, 1])
            # normwise only: with few radial nodes single rows are differences of terms 1e15 times their size
            assert np.all(np.isfinite(J[b])) and np.all(np.isfinite(F[b]))
            en = np.linalg.norm(J[b] - Jo) / np.linalg.norm(Jo); ef = np.linalg.norm(F[b] - Fo) / np.linalg.norm(Fo)
            assert en <= TOL_NORM and ef <= TOL_NORM, (kw, B, flags, en, ef)
            assert np.allclose(F2[b], F[b], rtol=1e-11, atol=1e-13 * np.abs(F[b]).max()), kw
    assert seen == {"generic", "pipelined", "batched-dmma"}


def test_host_buffer_entry_point_and_back_to_back_builds(orc):
    """dse_jacobian_host (the end-to-end path of bench.py: one staged H2D copy, results written by the assemble kernel into a
    mapped host buffer when small, copied back when large) returns exactly what dse_jacobian computes; and builds issued
    back to back on one handle with alternating coefficient sets (programmatic dependent launches, constant-bank
    coefficient slot rewritten by every prep_kernel) are bitwise reproducible."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload
    from workloads import Workload, draw_coefficients
    w = Workload("host", 16, 40, 32, 1e-6, 5e4, x_G=1.0, x_Z=30.0)
    p = oracle_params(w)
    for B in (1, 3, 130):                                    # 130 x (32*32 + 32) x 8 B > 1 MiB: the copy-back path
        c = np.stack([draw_coefficients(200 + b, w.n_cheb) for b in range(B)])
        bc = np.stack([[1.0 + 0.01 * b, 0.9 + 0.003 * b] for b in range(B)])
        d = Dse(params_from_workload(w, n_batch=B))
        J, F = d.jacobian(torch.from_numpy(c).cuda(), torch.from_numpy(bc).cuda())
        J = J.cpu().numpy(); F = F.cpu().numpy()
        Jh = np.full_like(J, np.nan); Fh = np.full_like(F, np.nan)
        d.jacobian_host(c, bc, Jh, Fh)
        assert np.array_equal(Jh, J) and np.array_equal(Fh, F)
        Fr = np.full_like(F, np.nan)
        d.jacobian_host(c, bc, None, Fr)                     # residual only
        assert np.abs(Fr - F).max() <= 1e-12 * np.abs(F).max()
        for b in (0, B - 1):
            Fo, Jo = orc.residual_jacobian(p, c[b], bc[b, 0], bc[b, 1])
            check(Jh[b], Fh[b], Jo, Fo)
        d.close()
    # alternating inputs, no synchronisation in between
    d = Dse(params_from_workload(w))
    cs = [torch.from_numpy(draw_coefficients(300 + i, w.n_cheb)[None, :]).cuda() for i in range(2)]
    bt = torch.tensor([[1.0, 0.9]], dtype=torch.float64, device="cuda")
    outs = [d.jacobian(cs[i % 2], bt) for i in range(8)]
    torch.cuda.synchronize()
    for i in range(2, 8):
        assert torch.equal(outs[i][0], outs[i % 2][0]) and torch.equal(outs[i][1], outs[i % 2][1])
    assert not torch.equal(outs[0][0], outs[1][0])
    d.close()


def test_fused_tail_fallback_path(orc):
    """dse_tail.cuh: the owner of a collocation point normally writes its rows of J and F itself once the rows of x_Z, x_G
    are published; with zero polls (include/dse_diag.h) every owner gives up at once and the CTA that completes the
    system's counter writes all rows.  Same arithmetic on both paths: bitwise equal results, and the counters are left
    clean for the next build (checked by alternating the two settings)."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload, DSE_FLAG_GEOMETRY_CACHE
    from workloads import config_inputs
    for cfg, flags in ((1, DSE_FLAG_GEOMETRY_CACHE), (0, 0)):
        w, c, bc = config_inputs(cfg)
        d = Dse(params_from_workload(w, flags=flags))
        ct = torch.from_numpy(c).cuda(); bt = torch.from_numpy(bc).cuda()
        J0, F0 = d.jacobian(ct, bt)
        J0 = J0.clone(); F0 = F0.clone()
        for polls in (0, 4096, 0, 0, 4096):
            d.set_tail_polls(polls)
            J, F = d.jacobian(ct, bt)
            assert torch.equal(J, J0) and torch.equal(F, F0), (cfg, polls)
        p = oracle_params(w)
        Fo, Jo = orc.residual_jacobian(p, c[0], bc[0, 0], bc[0, 1])
        assert np.linalg.norm(J0.cpu().numpy()[0] - Jo) <= 1e-10 * np.linalg.norm(Jo)
        d.close()


@pytest.mark.parametrize("kw,B", [(dict(n_cheb=12, n_r=40, n_theta=32, x_G=0.0, x_Z=5e4, n_ir=6, eps2=1e-6, L2=5e4), 1),
                                   (dict(n_cheb=20, n_r=64, n_theta=64, x_G=3.0, x_Z=70.0, eps2=1e-8, L2=1e8), 3),
                                   (dict(n_cheb=8, n_r=48, n_theta=16, eps2=1e-10, L2=1e10), 2)])
def test_fused_tail_stress(orc, kw, B):
    """The hand-shakes of the fused tail (arrival counters, published subtraction points, per-system counter, pending mask)
    over 1500 back-to-back builds per shape: two subtraction points (x_G != x_Z, also x_G = 0), several systems per
    handle on the per-system kernels, the generic kernel (n_theta = 16), alternating coefficient sets and poll budgets.
    Every build must reproduce, bit for bit, the first build of its coefficient set; one of them is checked against the
    oracle."""
    torch = _torch()
    from paper_1206_1779_b200 import Dse, params_from_workload, DSE_FLAG_GEOMETRY_CACHE
    from workloads import Workload, draw_coefficients
    w = Workload("tail-stress", **kw)
    d = Dse(params_from_workload(w, n_batch=B, flags=DSE_FLAG_GEOMETRY_CACHE))
    assert d.kernel_info()["variant"] != "batched-dmma"
    cs = [torch.from_numpy(np.stack([draw_coefficients(900 + 10 * v + b, w.n_cheb) for b in range(B)])).cuda() for v in range(2)]
    bt = torch.from_numpy(np.stack([[0.05 * b, 1.0 + 0.1 * b] for b in range(B)])).cuda()
    n2 = 2 * w.n_cheb
    ref = []
    for v in range(2):
        J, F = d.jacobian(cs[v], bt)
        ref.append((J.clone(), F.clone()))
    J = torch.empty((B, n2, n2), dtype=torch.float64, device="cuda"); F = torch.empty((B, n2), dtype=torch.float64, device="cuda")
    bad = torch.zeros(1, dtype=torch.int64, device="cuda")
    for i in range(1500):
        if i % 250 == 0:
            d.set_tail_polls(0 if (i // 250) % 3 == 1 else (3 if (i // 250) % 3 == 2 else 4096))
        v = (i * 7 + i // 5) % 2
        d.jacobian(cs[v], bt, J, F)
        bad += ((J != ref[v][0]).any() | (F != ref[v][1]).any()).to(torch.int64)      # checked on the device: the builds stay back to back
    assert int(bad.item()) == 0
    p = oracle_params(w)
    c0 = cs[0].cpu().numpy(); b0 = bt.cpu().numpy()
    for b in range(B):
        Fo, Jo = orc.residual_jacobian(p, c0[b], b0[b, 0], b0[b, 1])
        check(ref[0][0].cpu().numpy()[b], ref[0][1].cpu().numpy()[b], Jo, Fo)
    d.close()
