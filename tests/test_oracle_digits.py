"""Oracle pins P5, P9, P12, P13, P14: extended-precision differences, the DCT closed
form, and digits stored under tests/golden/."""
import mpmath as mp
import numpy as np
import pytest

from oracle import bta_oracle as O
from workloads import draw_obs, make_config, make_model, make_w0, uniform_design
from workloads.generate import draw_theta

from closed_form import closed_form


def rel(a, b):
    a, b = np.asarray(a, dtype=float), np.asarray(b, dtype=float)
    return np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-6 * np.max(np.abs(b))))


# ---- P14: worked example W0, printed digits -----------------------------------------------------
def test_p14_w0_digits(golden):
    g = golden("w0.txt")
    model, obs, th = make_w0()
    r = O.value_and_grad(model, obs, th)
    tol = 1e-12   # cos/sin may differ by an ulp across libms
    assert abs(r["ld_p"] - g["ld_p"][0]) <= tol * abs(g["ld_p"][0])
    assert abs(r["ld_c"] - g["ld_c"][0]) <= tol * abs(g["ld_c"][0])
    assert abs(r["f"] - g["f"][0]) <= tol * abs(g["f"][0])
    assert rel(r["grad"], g["grad"]) < 1e-11
    assert rel(r["phaseA"], g["phaseA"]) < 1e-11
    assert rel(r["phaseB"][:3], g["phaseB"]) < 1e-11
    assert rel(r["rss"], g["rss"]) < tol and abs(r["quad_p"] - g["quad_p"][0]) < 1e-11 * g["quad_p"][0]
    assert rel(r["x"][-2:], g["xT"]) < 1e-10
    d = O.dense_value_and_grad(model, obs, th)     # the dense definition hits the same digits
    assert abs(d["f"] - g["f"][0]) <= tol * abs(g["f"][0]) and rel(d["grad"], g["grad"]) < 1e-11


# ---- P13 / P9 / P12: closed form and stored digits -----------------------------------------------
def test_p13_digits_and_closed_form(golden):
    g = golden("p13.txt")
    th = np.array([0.1, -0.2, 0.3, 0.0])
    for h, kld, ktr in ((1.0, "ld_Qst_h1", "traces_h1"), (0.5, "ld_Qst_h05", "traces_h05")):
        model = make_model(g=4, k=1, nt=6, a=2, h=h)
        obs = draw_obs(model, 50, seed=3)
        r = O.value_and_grad(model, obs, th)
        ld_st = r["ld_p"] - model.a * np.log(model.fixed_prec)
        assert abs(ld_st - g[kld][0]) < 1e-12 * g[kld][0]
        assert rel(r["phaseC"][:3], g[ktr]) < 1e-11
        ld_cf, tr_cf = closed_form(4, 6, h, th)
        assert abs(ld_cf - g[kld][0]) < 1e-12 * g[kld][0] and rel(tr_cf, g[ktr]) < 1e-11
    assert abs(g["ld_Qp_h1"][0] - (g["ld_Qst_h1"][0] + 2 * np.log(1e-3))) < 1e-12


@pytest.mark.parametrize("g_,nt,h", [(7, 9, 1.0), (10, 5, 0.7), (5, 1, 1.0), (6, 2, 1.0)])
def test_p9_closed_form_other_sizes(g_, nt, h):
    model = make_model(g=g_, k=1, nt=nt, a=3, h=h)
    obs = draw_obs(model, 300, seed=g_)
    th = draw_theta(model, g_ + 100)
    r = O.value_and_grad(model, obs, th)
    ld_cf, tr_cf = closed_form(g_, nt, h, th)
    ld_st = r["ld_p"] - model.a * np.log(model.fixed_prec)
    assert abs(ld_st - ld_cf) < 1e-11 * abs(ld_cf)
    assert rel(r["phaseC"][:3], tr_cf) < 1e-9


def test_p12_uniform_design(golden):
    g = golden("p13.txt")
    model = make_model(g=4, k=1, nt=6, a=2)
    obs = uniform_design(model, c=1)
    th = np.array([0.1, -0.2, 0.3, 0.0])       # tau = 1, c = 1: latent part of Q_c = Q_st + I
    r = O.value_and_grad(model, obs, th, keep=True)
    # zero covariates: the arrow decouples, ld_c = ld(Q_st + I) + log det(1e-3 I_a)
    ld = r["ld_c"] - model.a * np.log(model.fixed_prec)
    assert abs(ld - g["ld_uniform"][0]) < 1e-12 * g["ld_uniform"][0]
    assert rel(r["phaseA"][:3], g["traces_uniform"]) < 1e-11
    ld_cf, tr_cf = closed_form(4, 6, 1.0, th, shift=1.0)
    assert abs(ld - ld_cf) < 1e-12 * ld_cf and rel(r["phaseA"][:3], tr_cf) < 1e-11


# ---- P5: the whole gradient vs 40-digit central differences of the TOTAL f ----------------------
def _mp_objective(consts, theta):
    """Eq. 1 at 40 digits from constant float64 matrices (exact integers for h=1) scaled in mpmath:
    Q_p = sum_c e^{th_c} P_c + 1e-3 I_a, Q_c = Q_p + e^{th_4} A^T A, x* re-solved at this theta."""
    P, AtA, Aty, yy, m, N, a = consts
    e = [mp.e ** t for t in theta]
    Qp = e[0] * P[0] + e[1] * P[1] + e[2] * P[2]
    for i in range(N - a, N):
        Qp[i, i] += mp.mpf("0.001")
    Qc = Qp + e[3] * AtA
    Lp, Lc = mp.cholesky(Qp), mp.cholesky(Qc)
    ld_p = 2 * sum(mp.log(Lp[i, i]) for i in range(N))
    ld_c = 2 * sum(mp.log(Lc[i, i]) for i in range(N))
    x = mp.cholesky_solve(Qc, e[3] * Aty)
    rss = yy - 2 * (Aty.T * x)[0] + (x.T * AtA * x)[0]
    quad = (x.T * Qp * x)[0]
    th2 = sum(t * t for t in theta)
    return -th2 / 2 + ld_p / 2 - ld_c / 2 - quad / 2 + m * theta[3] / 2 - e[3] * rss / 2


def test_p5_gradient_vs_mpmath_central_differences():
    mp.mp.dps = 40
    model = make_model(g=3, k=1, nt=4, a=2)          # N = 38: 9 evaluations at 40 digits stay fast
    obs = draw_obs(model, 60, seed=21)
    th = np.array([0.1, -0.2, 0.3, 0.15])
    r = O.value_and_grad(model, obs, th)
    Ks, Ms = O.spatial_matrices(model.g, model.h), O.temporal_matrices(model.nt)
    N, a = model.N, model.a
    P = []
    for c in range(3):
        M = np.zeros((N, N))
        M[: N - a, : N - a] = np.kron(Ms[c], Ks[c])
        P.append(mp.matrix(M.tolist()))
    A = O.dense_A(model, obs)
    A_mp = mp.matrix(A.tolist())
    y_mp = mp.matrix(obs.y.tolist())
    consts = (P, A_mp.T * A_mp, A_mp.T * y_mp, (y_mp.T * y_mp)[0], obs.m, N, a)
    theta = [mp.mpf(float(t)) for t in th]
    f0 = _mp_objective(consts, theta)
    assert abs(float(f0) - r["f"]) < 1e-12 * abs(r["f"])
    hstep = mp.mpf(10) ** -10
    for j in range(4):
        tp, tm = list(theta), list(theta)
        tp[j] += hstep
        tm[j] -= hstep
        fd = (_mp_objective(consts, tp) - _mp_objective(consts, tm)) / (2 * hstep)
        assert abs(float(fd) - r["grad"][j]) < 1e-11 * abs(float(fd)), (j, float(fd), r["grad"][j])


def test_p5_multivariate_gradient_vs_fourth_order_differences():
    model = make_model(g=3, k=3, nt=4, a=6)
    obs = draw_obs(model, 40, seed=5)
    th = draw_theta(model, 5)
    r = O.value_and_grad(model, obs, th)
    h = 2e-3
    f = lambda t: O.dense_objective(model, obs, t)["f"]   # literal (Lam (x) I)^T blockdiag (Lam (x) I)
    for j in range(model.d):
        e = np.zeros(model.d)
        e[j] = h
        fd = (-f(th + 2 * e) + 8 * f(th + e) - 8 * f(th - e) + f(th - 2 * e)) / (12 * h)
        assert abs(fd - r["grad"][j]) < 2e-8 * max(abs(fd), 1e-3 * np.max(np.abs(r["grad"]))), (j, fd, r["grad"][j])
