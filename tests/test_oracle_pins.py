"""Pins for the CPU oracle.  Each pin checks the oracle against
something other than itself: a library routine on the dense matrix, an invariant, a closed form,
extended-precision differences, or digits stored under tests/golden/ (with citation)."""
import numpy as np
import pytest

from oracle import bta_oracle as O
from workloads import draw_obs, make_config, make_model, make_w0, uniform_design
from workloads.generate import draw_theta

from closed_form import closed_form


def rel(a, b):
    a, b = np.asarray(a, dtype=float), np.asarray(b, dtype=float)
    return np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-300))


@pytest.fixture(scope="module")
def cfg0():
    model, obs, th = make_config(0)
    return model, obs, th, O.value_and_grad(model, obs, th, keep=True)


@pytest.fixture(scope="module")
def mv():
    model = make_model(g=3, k=3, nt=4, a=6)
    obs = draw_obs(model, 40, seed=5)
    th = draw_theta(model, 5)
    return model, obs, th, O.value_and_grad(model, obs, th, keep=True)


# ---- P1: assembly -------------------------------------------------------------------------
@pytest.mark.parametrize("which", ["cfg0", "mv"])
def test_p1_assembly_matches_literal_kronecker(which, request):
    model, obs, th, r = request.getfixturevalue(which)
    d = O.dense_objective(model, obs, th)
    Qp = O.dense_from_blocks(r["Qp"])
    Qc = O.dense_from_blocks(r["Qc"])
    assert np.max(np.abs(Qp - d["Qp"])) < 1e-13
    assert np.max(np.abs(Qc - d["Qc"])) < 1e-12
    assert np.array_equal(Qc, Qc.T)
    w = O.unpack_theta(model, th)[2][obs.var]
    assert np.allclose(r["Qc"].r, d["A"].T @ (w * obs.y), rtol=1e-13, atol=1e-13)


def test_p1_row_sums_of_Qst():
    # K2 1 = 0 and G 1 = 0, so Q_st (1 (x) 1) = e^{th3} (M2 1) (x) (C 1): 1 at the end blocks, 0 inside
    model, obs, th = make_config(0)
    agg = O.aggregates(model, obs)
    Q = O.dense_from_blocks(O.assemble(model, agg, th, "prior"))[: model.nt * model.b, : model.nt * model.b]
    rs = Q @ np.ones(model.nt * model.b)
    expect = np.zeros((model.nt, model.b))
    expect[0] = expect[-1] = np.exp(th[2]) * model.h ** 2
    assert np.allclose(rs, expect.ravel(), atol=1e-12)


def test_p1_base_matrix_stencils():
    K2, G, C = O.spatial_matrices(4, 1.0)
    assert G[0, 0] == 2 and G[1, 1] == 3 and G[5, 5] == 4 and G[5, 6] == -1 and G[5, 9] == -1  # R21
    assert np.count_nonzero(K2[5 * 1 + 5 - 0]) <= 13
    M0, M1, M2 = O.temporal_matrices(6)
    assert list(np.diag(M1)) == [1, 2, 2, 2, 2, 1] and list(np.diag(M2)) == [2] * 6     # R4
    assert M1[1, 0] == -1 and M2[1, 0] == -1 and M1[2, 0] == 0


# ---- P2/P3: factor, logdet, solve ----------------------------------------------------------
@pytest.mark.parametrize("which", ["cfg0", "mv"])
def test_p2_logdet_and_factor_vs_dense_library(which, request):
    model, obs, th, r = request.getfixturevalue(which)
    for bl, F, ld in ((r["Qc"], r["Fc"], r["ld_c"]), (r["Qp"], r["Fp"], r["ld_p"])):
        Q = O.dense_from_blocks(bl)
        sign, ref = np.linalg.slogdet(Q)
        assert sign > 0 and abs(ld - ref) <= 1e-12 * abs(ref)
        L = np.linalg.cholesky(Q)
        b = model.b
        for t in range(model.nt):
            assert np.allclose(F.LD[t], L[t * b:(t + 1) * b, t * b:(t + 1) * b], atol=1e-12)
            assert np.allclose(F.LC[t], L[model.nt * b:, t * b:(t + 1) * b], atol=1e-12)
        for t in range(model.nt - 1):
            assert np.allclose(F.LB[t], L[(t + 1) * b:(t + 2) * b, t * b:(t + 1) * b], atol=1e-12)
        assert np.allclose(F.LT, L[model.nt * b:, model.nt * b:], atol=1e-12)


@pytest.mark.parametrize("which", ["cfg0", "mv"])
def test_p3_solve_vs_dense(which, request):
    model, obs, th, r = request.getfixturevalue(which)
    Q = O.dense_from_blocks(r["Qc"])
    assert np.allclose(r["x"], np.linalg.solve(Q, r["Qc"].r), rtol=1e-11, atol=1e-13)
    assert np.max(np.abs(Q @ r["x"] - r["Qc"].r)) < 1e-11
    rhs = np.cos(np.arange(model.N) * 0.37)
    assert np.allclose(O.solve(r["Qc"], rhs), np.linalg.solve(Q, rhs), rtol=1e-10, atol=1e-12)


# ---- P4: selected inversion ----------------------------------------------------------------
@pytest.mark.parametrize("which", ["cfg0", "mv"])
def test_p4_selinv_vs_dense_inverse_and_invariant(which, request):
    model, obs, th, r = request.getfixturevalue(which)
    b, nt, a = model.b, model.nt, model.a
    for bl, Z in ((r["Qc"], r["Zc"]), (r["Qp"], r["Zp"])):
        S = np.linalg.inv(O.dense_from_blocks(bl))
        scale = np.max(np.abs(S))
        for t in range(nt):
            assert np.max(np.abs(Z.ZD[t] - S[t * b:(t + 1) * b, t * b:(t + 1) * b])) < 1e-12 * scale
            assert np.max(np.abs(Z.ZC[t] - S[nt * b:, t * b:(t + 1) * b])) < 1e-12 * scale
        for t in range(nt - 1):
            assert np.max(np.abs(Z.ZB[t] - S[(t + 1) * b:(t + 2) * b, t * b:(t + 1) * b])) < 1e-12 * scale
        assert np.max(np.abs(Z.ZT - S[nt * b:, nt * b:])) < 1e-12 * scale
        # invariant Sigma Q = I from pattern blocks only
        for t in range(nt):
            acc = Z.ZD[t] @ bl.D[t] + Z.ZC[t].T @ bl.C[t]
            if t > 0:
                acc += Z.ZB[t - 1] @ bl.B[t - 1].T
            if t < nt - 1:
                acc += Z.ZB[t].T @ bl.B[t]
            assert np.max(np.abs(acc - np.eye(b))) < 1e-10
        tip = Z.ZT @ bl.T + sum(Z.ZC[t] @ bl.C[t].T for t in range(nt))
        assert np.max(np.abs(tip - np.eye(a))) < 1e-10


# ---- block route vs dense definition ----------------------------------------------------------
@pytest.mark.parametrize("which", ["cfg0", "mv"])
def test_block_route_equals_dense_definition(which, request):
    model, obs, th, r = request.getfixturevalue(which)
    d = O.dense_value_and_grad(model, obs, th)
    assert abs(r["f"] - d["f"]) <= 1e-12 * abs(d["f"])
    assert rel(r["grad"], d["grad"]) < 1e-10
    assert np.allclose(r["x"], d["x"], rtol=1e-10, atol=1e-13)


def test_h_half_exercises_Cinv():
    model = make_model(g=4, k=1, nt=6, a=2, h=0.5)
    obs = draw_obs(model, 200, seed=11)
    th = np.array([0.1, -0.2, 0.3, 0.2])
    r = O.value_and_grad(model, obs, th)
    d = O.dense_value_and_grad(model, obs, th)
    assert abs(r["f"] - d["f"]) <= 1e-12 * abs(d["f"]) and rel(r["grad"], d["grad"]) < 1e-10


# ---- P6, P7, P8, P10, P11 ---------------------------------------------------------------------
def test_p6_value_identity(cfg0):
    model, obs, th, r = cfg0
    tau = np.exp(th[3])
    lhs = -0.5 * r["quad_p"] - 0.5 * tau * r["rss"][0]
    rhs = 0.5 * r["Qc"].r @ r["x"] - 0.5 * tau * obs.y @ obs.y
    assert abs(lhs - rhs) < 1e-11 * abs(rhs)


@pytest.mark.parametrize("which", ["cfg0", "mv"])
def test_p7_p8_sum_rules(which, request):
    model, obs, th, r = request.getfixturevalue(which)
    k = model.k
    # Q_c is linear-homogeneous in the e^theta's (given Lam) plus the fixed tip: per-variable + noise comps
    idx = list(range(3 * k)) + list(range(model.d - k, model.d))
    assert abs(np.sum(r["phaseA"][idx]) + model.fixed_prec * np.trace(r["Zc"].ZT) - model.N) < 1e-9 * model.N
    assert abs(np.sum(r["phaseC"][: 3 * k]) - model.nt * model.b) < 1e-9 * model.N


def test_p10_multivariate(mv):
    model, obs, th, r = mv
    E, Lam, tau = O.unpack_theta(model, th)
    ld = 0.0
    Ks, Ms = O.spatial_matrices(model.g, model.h), O.temporal_matrices(model.nt)
    for m in range(model.k):
        Qm = sum(E[m, c] * np.kron(Ms[c], Ks[c]) for c in range(3))
        ld += np.linalg.slogdet(Qm)[1]
    assert abs(r["ld_p"] - (ld + model.a * np.log(model.fixed_prec))) < 1e-11 * abs(ld)   # det Lam = 1
    lam_idx = slice(3 * model.k, 3 * model.k + 3)
    assert np.max(np.abs(r["phaseC"][lam_idx])) < 1e-10                                    # d ld_p / d lam = 0


def test_p11_no_observations():
    model = make_model(g=3, k=1, nt=4, a=2)
    obs = draw_obs(model, 0, seed=1)
    th = np.array([0.2, -0.1, 0.05, 0.3])
    r = O.value_and_grad(model, obs, th)
    assert abs(r["f"] + 0.5 * th @ th) < 1e-12
    assert np.allclose(r["grad"], -th, atol=1e-12)
    assert np.max(np.abs(r["x"])) == 0.0
