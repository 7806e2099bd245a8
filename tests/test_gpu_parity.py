"""GPU parity: the CUDA path (through the C-ABI binding) vs the CPU oracle, element by element, on the same
seeded inputs.  Tolerances (BASELINE.json north_star): 1e-9 relative on log-determinants and f, 1e-6 per
gradient component gated as in DESIGN.md reading R16; intermediates (factor, solve, selected inverse)
1e-9 of the block scale."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import bta_oracle as O
from workloads import draw_obs, make_config, make_model, make_w0, uniform_design
from workloads.generate import draw_theta

TOL_F, TOL_G = 1e-9, 1e-6


def _model(model, obs):
    from paper_2605_06392_b200 import BtaModel
    return BtaModel.from_workload(model, obs, device=0)


def grad_ok(g, ref):
    gate = np.maximum(np.abs(ref), 1e-3 * np.max(np.abs(ref)))     # R16
    return np.all(np.abs(g - ref) <= TOL_G * gate)


CASES = {
    "w0": lambda: make_w0(),
    "cfg0": lambda: make_config(0),
    "b25_ragged": lambda: (lambda m: (m, draw_obs(m, 300, 31), draw_theta(m, 31)))(make_model(5, 1, 7, 3)),
    "b81_two_tiles": lambda: (lambda m: (m, draw_obs(m, 900, 32), draw_theta(m, 32)))(make_model(9, 1, 5, 4)),
    "b144_h07": lambda: (lambda m: (m, draw_obs(m, 2000, 33), draw_theta(m, 33)))(make_model(12, 1, 4, 2, h=0.7)),
    "nt1": lambda: (lambda m: (m, draw_obs(m, 100, 34), draw_theta(m, 34)))(make_model(6, 1, 1, 2)),
    "nt2": lambda: (lambda m: (m, draw_obs(m, 100, 35), draw_theta(m, 35)))(make_model(6, 1, 2, 1)),
    "mv_k3_tiny": lambda: (lambda m: (m, draw_obs(m, 40, 5), draw_theta(m, 5)))(make_model(3, 3, 4, 6)),
    "mv_k2_b162": lambda: (lambda m: (m, draw_obs(m, 500, 6), draw_theta(m, 6)))(make_model(9, 2, 5, 4)),
    "mv_k3_b300": lambda: (lambda m: (m, draw_obs(m, 700, 7), draw_theta(m, 7)))(make_model(10, 3, 6, 6)),
    "a8": lambda: (lambda m: (m, draw_obs(m, 800, 36), draw_theta(m, 36)))(make_model(8, 1, 6, 8)),
    "no_obs": lambda: (lambda m: (m, draw_obs(m, 0, 37), draw_theta(m, 37)))(make_model(5, 1, 4, 2)),
    "uniform_design": lambda: (lambda m: (m, uniform_design(m, 2), draw_theta(m, 38)))(make_model(6, 1, 5, 2)),
    "nt3_twist_min": lambda: (lambda m: (m, draw_obs(m, 200, 41), draw_theta(m, 41)))(make_model(7, 1, 3, 2)),
    "nt4_twist": lambda: (lambda m: (m, draw_obs(m, 200, 42), draw_theta(m, 42)))(make_model(6, 1, 4, 3)),
    "mv_k4": lambda: (lambda m: (m, draw_obs(m, 60, 43), draw_theta(m, 43)))(make_model(3, 4, 5, 8)),
    "mv_k2_a8": lambda: (lambda m: (m, draw_obs(m, 300, 44), draw_theta(m, 44)))(make_model(8, 2, 7, 8)),
    "cfg1": lambda: make_config(1),
}


@pytest.mark.parametrize("name", list(CASES))
def test_value_and_grad_parity(name):
    model, obs, th = CASES[name]()
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    f, g, st = M.inla_value_and_grad(th, stages=True)
    im = M.last_intermediates()
    n0 = M.kernel_launches()
    f2, g2 = M.inla_value_and_grad(th)                                     # deterministic: bitwise repeatable
    assert f2 == f and np.array_equal(g, g2)
    assert M.kernel_launches() > n0 > 0
    M.close()
    assert abs(im["ld_p"] - ref["ld_p"]) <= TOL_F * abs(ref["ld_p"])
    assert abs(im["ld_c"] - ref["ld_c"]) <= TOL_F * abs(ref["ld_c"])
    assert abs(f - ref["f"]) <= TOL_F * abs(ref["f"])
    assert grad_ok(g, ref["grad"]), (g, ref["grad"])
    scale = max(np.max(np.abs(ref["x"])), 1e-30)
    assert np.max(np.abs(im["x"] - ref["x"])) <= 1e-9 * scale
    for key in ("phaseA", "phaseB", "phaseC"):
        s = max(np.max(np.abs(ref[key])), 1e-30)
        assert np.max(np.abs(im[key] - ref[key])) <= 1e-9 * s, key
    assert np.allclose(im["rss"], ref["rss"], rtol=1e-10, atol=1e-12)
    assert abs(im["quad_p"] - ref["quad_p"]) <= 1e-9 * max(abs(ref["quad_p"]), 1e-30)
    assert st["total"] > 0


@pytest.mark.parametrize("name", ["w0", "b81_two_tiles", "b144_h07", "nt1", "nt2", "nt3_twist_min", "nt4_twist",
                                  "mv_k2_b162", "mv_k3_b300", "cfg1"])
def test_carry_mode_matches_oracle_and_factor_mode(name):
    """Storage policy a7: carry-based reconstruction gives the same f, grad with about half the
    block storage."""
    model, obs, th = CASES[name]()
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    ws_factor = M.workspace_bytes()
    f0, g0 = M.inla_value_and_grad(th)
    M.bta_set_store_mode(1)
    assert M.bta_get_store_mode() == 1
    ws_carry = M.workspace_bytes()
    f1, g1 = M.inla_value_and_grad(th)
    f2, g2 = M.inla_value_and_grad(th)          # second call: CUDA-graph replay of the carry-mode sweep
    im = M.last_intermediates()
    M.close()
    assert f1 == f2 and np.array_equal(g1, g2)
    assert abs(f1 - ref["f"]) <= TOL_F * abs(ref["f"]) and grad_ok(g1, ref["grad"])
    assert abs(f1 - f0) <= 1e-12 * abs(f0) and np.max(np.abs(g1 - g0)) <= 1e-10 * np.max(np.abs(g0))
    assert abs(im["ld_c"] - ref["ld_c"]) <= TOL_F * abs(ref["ld_c"])
    if model.nt >= 8:
        assert ws_carry < 0.62 * ws_factor       # nt carries + 6 scratch blocks vs 2 nt + 3


def test_w0_printed_digits(golden):
    g = golden("w0.txt")
    model, obs, th = make_w0()
    M = _model(model, obs)
    f, grad = M.inla_value_and_grad(th)
    im = M.last_intermediates()
    M.close()
    assert abs(f - g["f"][0]) <= TOL_F * abs(g["f"][0])
    assert np.all(np.abs(grad - np.array(g["grad"])) <= TOL_G * np.abs(g["grad"]))
    assert abs(im["ld_c"] - g["ld_c"][0]) <= TOL_F * g["ld_c"][0]
    assert abs(im["ld_p"] - g["ld_p"][0]) <= TOL_F * g["ld_p"][0]


OP_CASES = ["cfg0", "b81_two_tiles", "mv_k3_tiny", "mv_k2_b162", "b144_h07"]


def _stack(lst):
    return np.stack(lst) if len(lst) else np.zeros((0,) + (1, 1))


@pytest.mark.parametrize("name", OP_CASES)
@pytest.mark.parametrize("which", [0, 1])
def test_assemble_factor_solve_selinv_parity(name, which):
    import torch
    model, obs, th = CASES[name]()
    agg = O.aggregates(model, obs)
    ref = O.assemble(model, agg, th, "cond" if which else "prior")
    b, nt, a, N = model.b, model.nt, model.a, model.N
    M = _model(model, obs)
    blk = M.alloc_blocks()
    M.bta_assemble(th, which, blk)
    D = blk.D.cpu().numpy()
    for t in range(nt):
        assert np.max(np.abs(D[t] - np.tril(ref.D[t]))) <= 1e-13 * np.max(np.abs(ref.D[t]))   # strict upper zero
    if nt > 1:
        assert np.max(np.abs(blk.B.cpu().numpy() - np.stack(ref.B))) <= 1e-13 * np.max(np.abs(np.stack(ref.B)))
    assert np.allclose(blk.C.cpu().numpy(), np.stack(ref.C), rtol=1e-13, atol=1e-15)
    assert np.allclose(blk.T.cpu().numpy(), ref.T, rtol=1e-13, atol=1e-15)
    if which:
        assert np.allclose(blk.rhs.cpu().numpy(), ref.r, rtol=1e-13, atol=1e-15)
    # ---- factor + logdet (Algorithm 1); factor kept as X = L_D^-1, L_B, L_C, L_T
    F = O.factor_forward(O.Blocks(ref.D, ref.B, ref.C, ref.T, None))
    diagL = torch.empty(N, dtype=torch.float64, device=blk.D.device)
    ld = M.bta_factor_logdet(blk, which, diagL=diagL)
    assert abs(ld - F.logdet) <= TOL_F * abs(F.logdet)
    X = blk.D.cpu().numpy()
    dl = diagL.cpu().numpy()
    for t in range(nt):
        Xref = np.linalg.inv(F.LD[t])
        assert np.max(np.abs(X[t] - Xref)) <= 1e-9 * np.max(np.abs(Xref))
        assert np.allclose(dl[t * b:(t + 1) * b], np.diag(F.LD[t]), rtol=1e-11)
    assert np.allclose(dl[nt * b:], np.diag(F.LT), rtol=1e-11)
    LB = blk.B.cpu().numpy()
    for t in range(nt - 1):
        assert np.max(np.abs(LB[t] - F.LB[t])) <= 1e-9 * max(np.max(np.abs(F.LB[t])), 1e-30)
    if which:
        assert np.max(np.abs(blk.C.cpu().numpy() - np.stack(F.LC))) <= 1e-9 * np.max(np.abs(np.stack(F.LC)))
    assert np.max(np.abs(blk.T.cpu().numpy() - F.LT)) <= 1e-9 * np.max(np.abs(F.LT))
    # ---- solve with 1, 3 and 11 right-hand sides (two chunks)
    for nrhs in (1, 3, 11):
        rhs = np.cos(0.37 * np.arange(nrhs * N)).reshape(nrhs, N) + 0.1
        xr = np.stack([O.solve(ref, rhs[r]) for r in range(nrhs)])
        rd = torch.tensor(rhs, device=blk.D.device)
        M.bta_solve(blk, which, rd)
        assert np.max(np.abs(rd.cpu().numpy() - xr)) <= 1e-9 * np.max(np.abs(xr))
    # ---- selected inversion in place
    Z = O.selinv(F)
    M.bta_selinv(blk, which)
    ZD = blk.D.cpu().numpy()
    sc = max(np.max(np.abs(z)) for z in Z.ZD)
    for t in range(nt):
        assert np.max(np.abs(ZD[t] - Z.ZD[t])) <= 1e-9 * sc
    ZB = blk.B.cpu().numpy()
    for t in range(nt - 1):
        assert np.max(np.abs(ZB[t] - Z.ZB[t])) <= 1e-9 * sc
    if which:
        assert np.max(np.abs(blk.C.cpu().numpy() - np.stack(Z.ZC))) <= 1e-9 * sc
    assert np.max(np.abs(blk.T.cpu().numpy() - Z.ZT)) <= 1e-9 * np.max(np.abs(Z.ZT))
    M.close()


def test_not_spd_is_reported():
    import torch
    from paper_2605_06392_b200 import BtaError
    model, obs, th = make_config(0)
    M = _model(model, obs)
    blk = M.alloc_blocks()
    M.bta_assemble(th, 1, blk)
    blk.D[2, 5, 5] = -1.0                       # global row 2*16 + 5 + 1 = 38 (1-based)
    with pytest.raises(BtaError) as ei:
        M.bta_factor_logdet(blk, 1)
    assert ei.value.code == 4 and M.last_pivot() == 38
    M.close()


def test_gemm_kernel_modes():
    import torch
    from paper_2605_06392_b200 import gemm
    rng = np.random.default_rng(0)
    for (Mm, Nn, Kk) in [(64, 64, 64), (100, 52, 37), (129, 257, 75), (27, 27, 27), (400, 400, 400)]:
        for mode in (0, 1, 2):
            A = rng.standard_normal((Mm, Kk) if mode != 2 else (Kk, Mm))
            B = rng.standard_normal((Kk, Nn) if mode != 1 else (Nn, Kk))
            C0 = rng.standard_normal((Mm, Nn))
            ref = -1.5 * (A if mode != 2 else A.T) @ (B if mode != 1 else B.T) + 0.5 * C0
            Cd = torch.tensor(C0, device="cuda")
            gemm(mode, torch.tensor(A, device="cuda"), torch.tensor(B, device="cuda"), Cd, alpha=-1.5, beta=0.5)
            assert np.max(np.abs(Cd.cpu().numpy() - ref)) <= 1e-12 * Kk
    n = 320
    L = np.tril(rng.standard_normal((n, n)))
    Bm = rng.standard_normal((n, n))
    t = lambda x: torch.tensor(x, device="cuda")
    z = lambda: torch.zeros(n, n, dtype=torch.float64, device="cuda")
    assert np.max(np.abs(gemm(1, t(Bm), t(L), z(), khi=1).cpu().numpy() - Bm @ L.T)) < 1e-11
    assert np.max(np.abs(gemm(0, t(Bm), t(L), z(), klo=1).cpu().numpy() - Bm @ L)) < 1e-11
    assert np.max(np.abs(gemm(0, t(L), t(Bm), z(), khi=2).cpu().numpy() - L @ Bm)) < 1e-11
    assert np.max(np.abs(gemm(2, t(L), t(L), z(), klo=2, out=2).cpu().numpy() - L.T @ L)) < 1e-11
    assert np.max(np.abs(gemm(1, t(Bm), t(Bm), z(), out=1).cpu().numpy() - np.tril(Bm @ Bm.T))) < 1e-11


def test_gemm_tile_classes_and_ragged_edges():
    """The three tile classes of launch_gemm (32x32 / 64x64 / 128x128), ragged tails in M, N and K,
    and the triangular k-ranges / lower-only outputs at sizes that reach the 64x64 and 128x128 tiles."""
    import torch
    from paper_2605_06392_b200 import gemm
    rng = np.random.default_rng(1)
    t = lambda x: torch.tensor(x, device="cuda")
    for (Mm, Nn, Kk) in [(1000, 900, 520),      # 16 x 15 small tiles -> 64x64 class
                         (1990, 2000, 301),     # 16 x 16 big tiles -> 128x128 class, ragged in M and K
                         (2304, 2304, 130)]:    # 324 big tiles = 2.19 waves -> 64x64 class by the wave rule
        for mode in (0, 1, 2):
            A = rng.standard_normal((Mm, Kk) if mode != 2 else (Kk, Mm))
            B = rng.standard_normal((Kk, Nn) if mode != 1 else (Nn, Kk))
            C0 = rng.standard_normal((Mm, Nn))
            ref = 0.75 * (A if mode != 2 else A.T) @ (B if mode != 1 else B.T) - 2.0 * C0
            Cd = t(C0)
            gemm(mode, t(A), t(B), Cd, alpha=0.75, beta=-2.0)
            assert np.max(np.abs(Cd.cpu().numpy() - ref)) <= 1e-12 * Kk, (Mm, Nn, Kk, mode)
    for n in (1100, 1930):                      # 64x64 class; 128x128 class with a ragged last tile
        L = np.tril(rng.standard_normal((n, n)))
        Bm = rng.standard_normal((n, n))
        z = lambda: torch.zeros(n, n, dtype=torch.float64, device="cuda")
        tol = 1e-12 * n
        assert np.max(np.abs(gemm(1, t(Bm), t(L), z(), khi=1).cpu().numpy() - Bm @ L.T)) < tol
        assert np.max(np.abs(gemm(0, t(Bm), t(L), z(), klo=1).cpu().numpy() - Bm @ L)) < tol
        assert np.max(np.abs(gemm(0, t(L), t(Bm), z(), khi=2).cpu().numpy() - L @ Bm)) < tol
        assert np.max(np.abs(gemm(2, t(L), t(L), z(), klo=2, out=2).cpu().numpy() - L.T @ L)) < tol
        assert np.max(np.abs(gemm(1, t(Bm), t(Bm), z(), out=1).cpu().numpy() - np.tril(Bm @ Bm.T))) < tol


def test_cta_trace_twins_are_bit_identical_and_count_ctas():
    """The TRACE instantiations of the GEMM kernel (bta_debug_cta_trace; diagnostics only) are separate code: they must
    return the same bits as the production kernels, record one entry per working CTA, and switch off again."""
    import torch
    from paper_2605_06392_b200 import gemm
    from paper_2605_06392_b200.binding import cta_trace_count, cta_trace_start
    rng = np.random.default_rng(2)
    t = lambda x: torch.tensor(x, device="cuda")
    cases = [(200, 200, 96, 32), (1000, 900, 130, 64), (2000, 1990, 70, 128)]   # 32x32, 64x64, 128x128 tile classes
    for (Mm, Nn, Kk, tile) in cases:
        A, B = rng.standard_normal((Mm, Kk)), rng.standard_normal((Kk, Nn))
        plain = gemm(0, t(A), t(B), torch.zeros(Mm, Nn, dtype=torch.float64, device="cuda")).cpu().numpy()
        buf = torch.zeros(4096, 4, dtype=torch.int64, device="cuda")
        cta_trace_start(buf)
        try:
            traced = gemm(0, t(A), t(B), torch.zeros(Mm, Nn, dtype=torch.float64, device="cuda")).cpu().numpy()
            n = cta_trace_count()
        finally:
            cta_trace_start(None)
        assert np.array_equal(plain, traced)
        assert n == -(-Mm // tile) * -(-Nn // tile), (n, Mm, Nn, tile)
        r = buf[:n].cpu().numpy()
        assert np.all(r[:, 1] >= r[:, 0]) and np.all((r[:, 2] >> 16) & 0xFFF == tile) and np.all((r[:, 2] & 0xFFFF) < 148)
        # switched off again (which also resets the counter, include/bta.h): a further launch records nothing
        gemm(0, t(A), t(B), torch.zeros(Mm, Nn, dtype=torch.float64, device="cuda"))
        assert cta_trace_count() == 0


@pytest.mark.parametrize("name", ["w0", "b81_two_tiles", "mv_k3_tiny", "mv_k2_b162"])
def test_value_fd_gradient_and_hessian(name):
    """value-only pass, the finite-difference baseline (Eq. 2) and the Hessian by
    differences of exact gradients (Eq. 13), against the same quantities formed from the oracle."""
    model, obs, th = CASES[name]()
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    assert abs(M.inla_value(th) - ref["f"]) <= TOL_F * abs(ref["f"])
    h = 1e-3
    f0, gfd = M.inla_fd_grad(th, h)
    assert abs(f0 - ref["f"]) <= TOL_F * abs(ref["f"])
    gfd_ref = np.zeros(model.d)
    for j in range(model.d):
        e = np.zeros(model.d)
        e[j] = h
        gfd_ref[j] = (O.dense_objective(model, obs, th + e)["f"] - O.dense_objective(model, obs, th - e)["f"]) / (2 * h)
    scale = np.max(np.abs(ref["grad"]))
    assert np.max(np.abs(gfd - gfd_ref)) <= 1e-6 * scale             # same differences, f to 1e-9 relative
    assert np.max(np.abs(gfd - ref["grad"])) <= 2e-4 * scale          # O(h^2) truncation
    hh = 5e-3
    f1, g1, H = M.inla_hessian(th, hh)
    M.close()
    assert abs(f1 - ref["f"]) <= TOL_F * abs(ref["f"]) and grad_ok(g1, ref["grad"])
    Href = np.zeros((model.d, model.d))
    for j in range(model.d):
        e = np.zeros(model.d)
        e[j] = hh
        Href[:, j] = (O.value_and_grad(model, obs, th + e)["grad"] - O.value_and_grad(model, obs, th - e)["grad"]) / (2 * hh)
    assert np.max(np.abs(H - Href)) <= 1e-6 * np.max(np.abs(Href))
    assert np.max(np.abs(H - H.T)) <= 1e-3 * np.max(np.abs(H))       # symmetric up to O(h^2)


@pytest.mark.parametrize("name", ["w0", "mv_k3_tiny"])
def test_mode_search_matches_scipy_on_the_oracle(name):
    """L-BFGS over theta with exact GPU gradients reaches the optimum that scipy's
    L-BFGS-B finds on the oracle's objective."""
    from scipy.optimize import minimize
    model, obs, th0 = CASES[name]()
    M = _model(model, obs)
    th, f, g, iters, evals = M.inla_optimize(th0, max_iter=200, gtol=1e-7)
    M.close()
    assert np.max(np.abs(g)) <= 1e-5 and iters > 0 and evals >= iters
    fun = lambda t: tuple(-np.asarray(v) for v in (lambda r: (r["f"], r["grad"]))(O.value_and_grad(model, obs, t)))
    ref = minimize(fun, th0, jac=True, method="L-BFGS-B", options=dict(maxiter=500, ftol=1e-15, gtol=1e-9))
    assert abs(f - (-ref.fun)) <= 1e-8 * abs(ref.fun)
    assert np.max(np.abs(th - ref.x)) <= 1e-4
    r = O.value_and_grad(model, obs, th)            # the oracle agrees at the GPU optimum
    assert abs(r["f"] - f) <= TOL_F * abs(f) and np.max(np.abs(r["grad"])) <= 1e-4


def test_workspace_canaries():
    """compute-sanitizer is closed on this pool (profiles/r02_sanitizer_refusal.md), so out-of-bounds writes are
    looked for directly: guard words on both sides of the caller-provided workspace must survive a gradient in either
    store mode (ragged block size, twisted path, arrow width 3)."""
    import torch
    model, obs, th = CASES["b25_ragged"]()
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    for mode in (0, 1):
        M.bta_set_store_mode(mode)
        need = M.workspace_bytes()
        guard = 1 << 16
        buf = torch.full((need + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
        M._ws = buf[guard: guard + need]                       # the binding hands this view's pointer to the library
        f, g = M.inla_value_and_grad(th)
        assert abs(f - ref["f"]) <= TOL_F * abs(ref["f"]) and grad_ok(g, ref["grad"])
        assert bool((buf[:guard] == 0xA5).all()) and bool((buf[guard + need:] == 0xA5).all())
    M.close()


def test_many_observations_on_one_site():
    """Model setup sorts each site's observation list (fixed summation order): 20,000 rows on ONE latent site plus a
    uniform remainder -- the O(n log n) per-site sort of assemble.cu, against the oracle's aggregates."""
    model = make_model(6, 1, 4, 2)
    obs = draw_obs(model, 25000, 51)
    obs.node[:20000] = 7
    obs.time[:20000] = 2
    th = draw_theta(model, 51)
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    f, g = M.inla_value_and_grad(th)
    M.close()
    assert abs(f - ref["f"]) <= TOL_F * abs(ref["f"]) and grad_ok(g, ref["grad"])


def test_second_device_ordinal():
    """cudaFuncSetAttribute is per device: a context on ordinal 1 must work after ordinal 0, and the caller's
    current device is left alone (round-1 advisor finding)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    from paper_2605_06392_b200 import BtaModel
    model, obs, th = CASES["b144_h07"]()
    ref = O.value_and_grad(model, obs, th)
    for dev in (0, 1):
        torch.cuda.set_device(0)
        M = BtaModel.from_workload(model, obs, device=dev)
        with torch.cuda.device(dev):
            f, g = M.inla_value_and_grad(th)
        assert torch.cuda.current_device() == 0
        M.close()
        assert abs(f - ref["f"]) <= TOL_F * abs(ref["f"]) and grad_ok(g, ref["grad"])


@pytest.mark.parametrize("name", ["nt3_twist_min", "nt4_twist", "b81_two_tiles", "mv_k2_a8", "mv_k3_b300", "cfg1"])
def test_host_staged_carries(name):
    """SURVEY.md §8(f) NEXT-4 / PAPER.md:185 (§III-C c): the carries are written to pinned host memory in the forward
    sweep and streamed back in the backward sweep; the device keeps a ring of 4 diagonal-block slots per sub-chain.
    Same f, grad as carry mode; device workspace independent of nt."""
    model, obs, th = CASES[name]()
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    M.bta_set_store_mode(1)
    ws_carry = M.workspace_bytes()
    f1, g1 = M.inla_value_and_grad(th)
    M.bta_set_store_mode(2)
    assert M.bta_get_store_mode() == 2
    assert M.bta_host_bytes() == 2 * (model.nt - 1) * model.b * model.b * 8
    ws_host = M.workspace_bytes()
    f2, g2 = M.inla_value_and_grad(th)
    f3, g3 = M.inla_value_and_grad(th)          # again (graph replay for small b; ring events reused)
    im = M.last_intermediates()
    M.close()
    assert f2 == f3 and np.array_equal(g2, g3)
    assert abs(f2 - f1) <= 1e-12 * abs(f1) and np.max(np.abs(g2 - g1)) <= 1e-12 * np.max(np.abs(g1))
    assert abs(f2 - ref["f"]) <= TOL_F * abs(ref["f"]) and grad_ok(g2, ref["grad"])
    assert np.max(np.abs(im["x"] - ref["x"])) <= 1e-9 * np.max(np.abs(ref["x"]))
    if model.nt >= 12:
        assert ws_host < ws_carry


def test_host_staged_workspace_is_independent_of_nt():
    """Device workspace O(b^2): growing nt from 8 to 64 adds less than two b x b blocks (the O(nt a b)
    row stacks) in host mode, against 2 x 56 blocks in carry mode."""
    from paper_2605_06392_b200 import BtaModel
    ws = {}
    for nt in (8, 64):
        model = make_model(20, 1, nt, 2)
        M = BtaModel.from_workload(model, draw_obs(model, 10, 1), device=0)
        for mode in (1, 2):
            M.bta_set_store_mode(mode)
            ws[mode, nt] = M.workspace_bytes()
        M.close()
    block = 400 * 400 * 8
    assert ws[2, 64] - ws[2, 8] < 2 * block, ws
    assert ws[1, 64] - ws[1, 8] > 100 * block, ws


PART_CASES = {
    "nt3": lambda: CASES["nt3_twist_min"](),
    "nt5_b25": lambda: (lambda m: (m, draw_obs(m, 300, 61), draw_theta(m, 61)))(make_model(5, 1, 5, 3)),
    "nt7_b36": lambda: (lambda m: (m, draw_obs(m, 400, 62), draw_theta(m, 62)))(make_model(6, 1, 7, 2)),
    "nt12_mv_b162": lambda: (lambda m: (m, draw_obs(m, 900, 63), draw_theta(m, 63)))(make_model(9, 2, 12, 4)),
    "nt9_b144_a8": lambda: (lambda m: (m, draw_obs(m, 700, 64), draw_theta(m, 64)))(make_model(12, 1, 9, 8)),
    "cfg1": lambda: make_config(1),
}


@pytest.mark.parametrize("P", [2, 3, 4])
@pytest.mark.parametrize("name", list(PART_CASES))
def test_time_domain_partitioning(name, P):
    """SURVEY.md §8(f) NEXT-3 / PAPER.md:177-183: P partitions inside one GPU -- interior chains with fill to the top
    boundary, a reduced system of 2P-1 boundary blocks, reversed order in the backward pass -- against the oracle,
    component by component, and against the two-way elimination."""
    model, obs, th = PART_CASES[name]()
    ref = O.value_and_grad(model, obs, th)
    M = _model(model, obs)
    f0, g0 = M.inla_value_and_grad(th)
    M.bta_set_partitions(P)
    plan = M.bta_partition_plan(P)
    assert plan[0][0] == 0 and plan[-1][1] == model.nt - 1
    assert all(plan[i][0] == plan[i - 1][1] + 1 and plan[i][1] > plan[i][0] for i in range(1, len(plan)))
    assert len(plan) == min(P, (model.nt + 1) // 2) or model.nt < 2 * P - 1
    f, g = M.inla_value_and_grad(th)
    im = M.last_intermediates()
    f2, g2 = M.inla_value_and_grad(th)          # graph replay for small b; bitwise repeatable
    v = M.inla_value(th)
    M.close()
    assert f2 == f and np.array_equal(g, g2)
    assert abs(v - ref["f"]) <= TOL_F * abs(ref["f"])
    assert abs(im["ld_p"] - ref["ld_p"]) <= TOL_F * abs(ref["ld_p"])
    assert abs(im["ld_c"] - ref["ld_c"]) <= TOL_F * abs(ref["ld_c"])
    assert abs(f - ref["f"]) <= TOL_F * abs(ref["f"])
    assert np.max(np.abs(im["x"] - ref["x"])) <= 1e-9 * np.max(np.abs(ref["x"]))
    for key in ("phaseA", "phaseB", "phaseC"):
        s = max(np.max(np.abs(ref[key])), 1e-30)
        assert np.max(np.abs(im[key] - ref[key])) <= 1e-9 * s, (key, im[key], ref[key])
    assert grad_ok(g, ref["grad"]), (g, ref["grad"])
    assert abs(f - f0) <= 1e-11 * abs(f0) and np.max(np.abs(g - g0)) <= 1e-9 * np.max(np.abs(g0))


@pytest.mark.parametrize("name,P", [("nt3", 2), ("nt5_b25", 2), ("nt7_b36", 3), ("nt12_mv_b162", 4), ("nt9_b144_a8", 3),
                                    ("cfg1", 4), ("cfg1", 8)])
def test_partitioning_across_ranks_emulated(name, P):
    """The multi-rank form (include/bta.h: inla_part_*) with the ranks emulated one after the other
    in this process: P contexts, each eliminating ONE partition; slabs concatenated in rank order (= all-gather);
    partial sums added (= all-reduce); every rank must return the oracle's f and gradient."""
    import torch
    model, obs, th = PART_CASES[name]()
    ref = O.value_and_grad(model, obs, th)
    ranks = [_model(model, obs) for _ in range(P)]
    for M in ranks:
        M.bta_set_partitions(P)
    assert len(ranks[0].bta_partition_plan(P)) == P
    slabs = [M.inla_part_phase1(th, r, P) for r, M in enumerate(ranks)]
    gathered = torch.cat(slabs)
    parts = [M.inla_part_phase2(r, P, gathered) for r, M in enumerate(ranks)]
    total = torch.stack(parts).sum(0)
    out = [M.inla_part_finish(total.clone()) for M in ranks]
    ims = [M.last_intermediates(want_x=False) for M in ranks]
    for M in ranks:
        M.close()
    for (f, g), im in zip(out, ims):
        assert f == out[0][0] and np.array_equal(g, out[0][1])          # identical on every rank
        assert abs(f - ref["f"]) <= TOL_F * abs(ref["f"])
        assert grad_ok(g, ref["grad"]), (g, ref["grad"])
        assert abs(im["ld_p"] - ref["ld_p"]) <= TOL_F * abs(ref["ld_p"])
        assert abs(im["ld_c"] - ref["ld_c"]) <= TOL_F * abs(ref["ld_c"])
        for key in ("phaseA", "phaseB", "phaseC"):
            s = max(np.max(np.abs(ref[key])), 1e-30)
            assert np.max(np.abs(im[key] - ref[key])) <= 1e-9 * s, key


def test_partitioning_across_ranks_two_processes():
    """Two real processes (torch.distributed, gloo, both on cuda:0 -- the collectives are host-side, no kernel of one
    rank waits for the other) run paper_2605_06392_b200.partitioned.value_and_grad on config 1's shapes."""
    import json
    import os
    import socket
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", str(port),
                          os.path.join(root, "tests", "dist_partition_worker.py")],
                         capture_output=True, text=True, cwd=root, timeout=600)
    assert out.returncode == 0, out.stdout[-2000:] + out.stderr[-2000:]
    # the two ranks share one stdout: their lines can arrive glued together, so scan for objects, not for lines
    lines, dec, pos = [], json.JSONDecoder(), 0
    while True:
        pos = out.stdout.find('{"rank"', pos)
        if pos < 0:
            break
        obj, pos = dec.raw_decode(out.stdout, pos)
        lines.append(obj)
    assert sorted(l["rank"] for l in lines) == [0, 1]
    assert lines[0]["f"] == lines[1]["f"] and lines[0]["grad"] == lines[1]["grad"]
    assert all(l["ok"] for l in lines), lines
