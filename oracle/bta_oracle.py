"""Plain, slow, obviously-correct CPU implementation (numpy, float64) of the exact INLA
objective f(theta) and its gradient over a block-tridiagonal-arrowhead (BTA) precision
matrix -- ADELIA, arxiv/paper_2605_06392.  TEST INFRASTRUCTURE: see oracle/__init__.py.

Two independent routes are provided:

* the DENSE DEFINITION (`dense_value_and_grad`): Eq. 1 through a dense N x N Cholesky and
  Eq. 6 through the dense inverse, tr(Q^-1 dQ/dtheta_k), with Q and dQ built by literal
  Kronecker products and a literal projection matrix A;
* the BLOCK-SEQUENTIAL ALGORITHM (`value_and_grad`): Algorithm 1 (as
  repaired in SURVEY.md App. A.1 / DESIGN.md reading R8), Eqs. 3-5,
  BTA selected inversion (recurrences of DESIGN.md reading R10), the
  per-block traces of Eq. 7 and quadratic forms of Eq. 9
   with explicit dense block Jacobians (Eqs. 10-12).

Library primitives used as steps: numpy.linalg.cholesky, scipy.linalg.solve_triangular,
matmul.  No blocking, fusion or reordering beyond what the paper states.  1-based block
index i of the paper = 0-based index i-1 here.

Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): dense Cholesky log-determinant
and dense inverse on tiny inputs, Sigma Q = I on pattern blocks, 40-digit central
differences of f (mpmath), the printed digits of worked example W0 and of pin P13
(tests/golden/), the DCT closed form at any size, the sum rules P7/P8, special cases
m=0 and the uniform design.  No function here is "parity unpinned".
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np
from scipy.linalg import solve_triangular


# --------------------------------------------------------------------------------------
# Base matrices (BASELINE.json configs[0]; readings R3, R4, R21)
# --------------------------------------------------------------------------------------
def spatial_matrices(g: int, h: float):
    """[K_0, K_1, K_2] paired with temporal terms c = 0,1,2:
    c=0: M0 (x) K2 with K2 = G C^-1 G;  c=1: M1 (x) K1 with K1 = G;  c=2: M2 (x) K0, K0 = C.
    C = h^2 I (lumped mass); G = 5-point graph Laplacian, degree - adjacency (R21)."""
    ns = g * g
    G = np.zeros((ns, ns))
    for iy in range(g):
        for ix in range(g):
            s = iy * g + ix
            for dy, dx in ((0, 1), (0, -1), (1, 0), (-1, 0)):
                jy, jx = iy + dy, ix + dx
                if 0 <= jy < g and 0 <= jx < g:
                    G[s, s] += 1.0
                    G[s, jy * g + jx] -= 1.0
    C = (h * h) * np.eye(ns)
    Cinv = np.eye(ns) / (h * h)
    K2 = G @ Cinv @ G
    return [K2, G, C]


def temporal_matrices(nt: int):
    """[M0, M1, M2] as dense nt x nt: M0 = I; M1 = D^T D, D the (nt-1) x nt first
    difference; M2 = tridiag(-1, 2, -1) with every diagonal entry 2 (reading R4)."""
    M0 = np.eye(nt)
    Dm = np.zeros((max(nt - 1, 0), nt))
    for i in range(nt - 1):
        Dm[i, i] = -1.0
        Dm[i, i + 1] = 1.0
    M1 = Dm.T @ Dm
    M2 = 2.0 * np.eye(nt)
    for i in range(nt - 1):
        M2[i, i + 1] = -1.0
        M2[i + 1, i] = -1.0
    return [M0, M1, M2]


# --------------------------------------------------------------------------------------
# Hyperparameters (reading R13) and coregional weights (Eq. 10, reading R12)
# --------------------------------------------------------------------------------------
def unpack_theta(model, theta):
    """theta = [theta_{1,1..3}, ..., theta_{k,1..3}, lambda_21, lambda_31, lambda_32, ...,
    log tau_1..k]  ->  (E[k,3] = exp(theta_{m,c}), Lam[k,k] unit lower, tau[k])."""
    k = model.k
    theta = np.asarray(theta, dtype=np.float64)
    E = np.exp(theta[: 3 * k]).reshape(k, 3)
    Lam = np.eye(k)
    p = 3 * k
    for a in range(k):
        for bb in range(a):
            Lam[a, bb] = theta[p]
            p += 1
    tau = np.exp(theta[p : p + k])
    return E, Lam, tau


def lambda_index(model):
    """[(a, b)] of the coupling parameters in theta order: (1,0), (2,0), (2,1), ..."""
    return [(a, bb) for a in range(model.k) for bb in range(a)]


def weights(model, theta):
    """W_c[i][j] = sum_m e^{theta_{m,c}} Lam[m,i] Lam[m,j]  (Eq. 10 with reading R12)."""
    E, Lam, _ = unpack_theta(model, theta)
    return [sum(E[m, c] * np.outer(Lam[m], Lam[m]) for m in range(model.k)) for c in range(3)]


def weight_jacobian(model, theta, j):
    """d W_c / d theta_j for a prior hyperparameter j < 3k + k(k-1)/2 (Eqs. 11, 12).
    Returns [dW_0, dW_1, dW_2] (k x k each)."""
    k = model.k
    E, Lam, _ = unpack_theta(model, theta)
    out = [np.zeros((k, k)) for _ in range(3)]
    if j < 3 * k:  # per-variable parameter theta_{m,c}: only its own term moves (Eq. 11)
        m, c = divmod(j, 3)
        out[c] = E[m, c] * np.outer(Lam[m], Lam[m])
    else:  # coupling parameter Lam[a,b]: the weights move, the Q_m do not (Eq. 12)
        a, bb = lambda_index(model)[j - 3 * k]
        dLam = np.zeros(k)
        dLam[bb] = 1.0
        for c in range(3):
            out[c] = E[a, c] * (np.outer(dLam, Lam[a]) + np.outer(Lam[a], dLam))
    return out


# --------------------------------------------------------------------------------------
# Observation aggregates (theta-independent)
# --------------------------------------------------------------------------------------
@dataclass
class Aggregates:
    cnt: np.ndarray    # [nt, b]     number of observations of latent (t, v, s)
    zsum: np.ndarray   # [nt, a, b]  sum of covariate rows hitting latent (t, v, s), arrow columns
    ZZ: np.ndarray     # [k, a, a]   sum_i z_i z_i^T over rows of variable v
    ysum: np.ndarray   # [nt, b]
    zy: np.ndarray     # [k, a]
    yy: np.ndarray     # [k]
    mv: np.ndarray     # [k]         observations per variable


def covariate_rows(model, obs):
    """Full-width covariate rows Z[m, a]: obs.cov placed in the columns of its variable (R14)."""
    Z = np.zeros((obs.m, model.a))
    apr = model.a_per_row
    for p in range(apr):
        Z[np.arange(obs.m), obs.var * apr + p] = obs.cov[:, p]
    return Z


def aggregates(model, obs) -> Aggregates:
    nt, b, a, k, ns = model.nt, model.b, model.a, model.k, model.ns
    col = obs.var.astype(np.int64) * ns + obs.node
    Z = covariate_rows(model, obs)
    cnt = np.zeros((nt, b))
    ysum = np.zeros((nt, b))
    zsum = np.zeros((nt, a, b))
    np.add.at(cnt, (obs.time, col), 1.0)
    np.add.at(ysum, (obs.time, col), obs.y)
    for p in range(a):
        np.add.at(zsum[:, p, :], (obs.time, col), Z[:, p])
    ZZ = np.zeros((k, a, a))
    zy = np.zeros((k, a))
    yy = np.zeros(k)
    mv = np.zeros(k)
    for v in range(k):
        sel = obs.var == v
        ZZ[v] = Z[sel].T @ Z[sel]
        zy[v] = Z[sel].T @ obs.y[sel]
        yy[v] = obs.y[sel] @ obs.y[sel]
        mv[v] = sel.sum()
    return Aggregates(cnt, zsum, ZZ, ysum, zy, yy, mv)


# --------------------------------------------------------------------------------------
# Block assembly (Eq. 10) -- dense blocks, literal Kronecker products
# --------------------------------------------------------------------------------------
@dataclass
class Blocks:
    """BTA matrix in the paper's notation: D_i (b x b), B_i = block
    (i+1, i), C_i = block (T, i) (a x b), tip T (a x a); rhs r = (r_1..r_n, r_T)."""
    D: list
    B: list
    C: list
    T: np.ndarray
    r: np.ndarray | None = None


def prior_block(model, Wc, Ks, Mrow):
    """sum_c Mrow[c] * (W_c (x) K_c): one b x b block of Q_st (Eq. 10)."""
    out = np.zeros((model.b, model.b))
    for c in range(3):
        if Mrow[c] != 0.0:
            out += Mrow[c] * np.kron(Wc[c], Ks[c])
    return out


def assemble(model, agg: Aggregates, theta, which: str) -> Blocks:
    """which = 'prior': Q_p = blockdiag(Q_st, fixed_prec I_a) (R5), BT (C_i = 0).
    which = 'cond' : Q_c = Q_p + sum_v tau_v A_v^T A_v and r = sum_v tau_v A_v^T y_v."""
    nt, b, a, k, ns = model.nt, model.b, model.a, model.k, model.ns
    Ks = spatial_matrices(model.g, model.h)
    Ms = temporal_matrices(nt)
    Wc = weights(model, theta)
    _, _, tau = unpack_theta(model, theta)
    tau_col = np.repeat(tau, ns)  # tau of the variable owning each latent column
    D = [prior_block(model, Wc, Ks, [Ms[c][t, t] for c in range(3)]) for t in range(nt)]
    B = [prior_block(model, Wc, Ks, [Ms[c][t + 1, t] for c in range(3)]) for t in range(nt - 1)]
    C = [np.zeros((a, b)) for _ in range(nt)]
    T = model.fixed_prec * np.eye(a)
    r = None
    if which == "cond":
        r = np.zeros(model.N)
        for t in range(nt):
            D[t] = D[t] + np.diag(tau_col * agg.cnt[t])
            C[t] = agg.zsum[t] * tau_col[None, :]
            r[t * b : (t + 1) * b] = tau_col * agg.ysum[t]
        for v in range(k):
            T = T + tau[v] * agg.ZZ[v]
            r[nt * b :] += tau[v] * agg.zy[v]
    elif which != "prior":
        raise ValueError(which)
    return Blocks(D, B, C, T, r)


def dense_from_blocks(bl: Blocks) -> np.ndarray:
    nt, b, a = len(bl.D), bl.D[0].shape[0], bl.T.shape[0]
    N = nt * b + a
    Q = np.zeros((N, N))
    for t in range(nt):
        Q[t * b : (t + 1) * b, t * b : (t + 1) * b] = bl.D[t]
        Q[N - a :, t * b : (t + 1) * b] = bl.C[t]
        Q[t * b : (t + 1) * b, N - a :] = bl.C[t].T
    for t in range(nt - 1):
        Q[(t + 1) * b : (t + 2) * b, t * b : (t + 1) * b] = bl.B[t]
        Q[t * b : (t + 1) * b, (t + 1) * b : (t + 2) * b] = bl.B[t].T
    Q[N - a :, N - a :] = bl.T
    return Q


# --------------------------------------------------------------------------------------
# Algorithm 1: fused BTA Cholesky + lower solve (reading R8)
# --------------------------------------------------------------------------------------
@dataclass
class Factor:
    LD: list
    LB: list
    LC: list
    LT: np.ndarray
    z: list | None
    zT: np.ndarray | None
    S: list            # Schur carries S_1..S_{n-1} (the paper's stored intermediates)
    logdet: float


def _right_solve_LT(M, L):
    """M L^-T  (rows of M solved against lower-triangular L)."""
    return solve_triangular(L, M.T, lower=True).T


def _right_solve_L(M, L):
    """M L^-1."""
    return solve_triangular(L, M.T, lower=True, trans="T").T


def factor_forward(bl: Blocks) -> Factor:
    n, b, a = len(bl.D), bl.D[0].shape[0], bl.T.shape[0]
    have_rhs = bl.r is not None
    S_prev = np.zeros((b, b))                         # line 1: S_0 <- 0
    Tt = bl.T.copy()                                  #         T~_0 <- T
    LC_prev = np.zeros((a, b))                        #         C^L_0 <- 0
    LB_prev = np.zeros((b, b))                        #         L_B0 <- 0
    z_prev = np.zeros(b)                              #         z_0 <- 0
    vT = np.zeros(a)                                  #         v_T <- 0
    LD, LB, LC, z, S = [], [], [], [], []
    logdet = 0.0
    for i in range(n):                                # line 2
        LDi = np.linalg.cholesky(bl.D[i] - S_prev)    # line 3
        LCi = _right_solve_LT(bl.C[i] - LC_prev @ LB_prev.T, LDi)          # line 4
        if have_rhs:                                  # line 5
            zi = solve_triangular(LDi, bl.r[i * b : (i + 1) * b] - LB_prev @ z_prev, lower=True)
            vT = vT + LCi @ zi
            z.append(zi)
            z_prev = zi
        if i < n - 1:                                 # line 6 (guard "if i < n", R8)
            LBi = _right_solve_LT(bl.B[i], LDi)
            Si = LBi @ LBi.T
            LB.append(LBi)
            S.append(Si)
            S_prev, LB_prev = Si, LBi
        Tt = Tt - LCi @ LCi.T                         # line 9
        LC_prev = LCi
        LD.append(LDi)
        LC.append(LCi)
        logdet += 2.0 * np.sum(np.log(np.diag(LDi)))
    LT = np.linalg.cholesky(Tt)                       # line 11
    zT = solve_triangular(LT, bl.r[n * b :] - vT, lower=True) if have_rhs else None
    logdet += 2.0 * np.sum(np.log(np.diag(LT)))
    return Factor(LD, LB, LC, LT, z if have_rhs else None, zT, S, float(logdet))


def solve_upper(F: Factor) -> np.ndarray:
    """Eqs. 3-5: L^T x* = z, sweeping i = n..1."""
    n, b = len(F.LD), F.LD[0].shape[0]
    a = F.LT.shape[0]
    x = np.zeros(n * b + a)
    xT = solve_triangular(F.LT, F.zT, lower=True, trans="T")                 # Eq. 3
    x[n * b :] = xT
    x_next = None
    for i in range(n - 1, -1, -1):
        rhs = F.z[i] - F.LC[i].T @ xT                                        # Eq. 4
        if i < n - 1:
            rhs = rhs - F.LB[i].T @ x_next                                   # Eq. 5
        x_next = solve_triangular(F.LD[i], rhs, lower=True, trans="T")
        x[i * b : (i + 1) * b] = x_next
    return x


def solve(bl: Blocks, rhs: np.ndarray) -> np.ndarray:
    """Q x = rhs through Algorithm 1 + Eqs. 3-5 (what `bta_solve` computes)."""
    F = factor_forward(Blocks(bl.D, bl.B, bl.C, bl.T, rhs))
    return solve_upper(F)


# --------------------------------------------------------------------------------------
# BTA selected inversion (recurrences from Sigma L = L^-T, reading R10)
# --------------------------------------------------------------------------------------
@dataclass
class SelInv:
    ZD: list   # Z_Di = [Q^-1]_{ii}
    ZB: list   # Z_Bi = [Q^-1]_{i+1,i}
    ZC: list   # Z_Ci = [Q^-1]_{T,i}
    ZT: np.ndarray


def selinv(F: Factor) -> SelInv:
    n, b = len(F.LD), F.LD[0].shape[0]
    a = F.LT.shape[0]
    LTinv = solve_triangular(F.LT, np.eye(a), lower=True)
    ZT = LTinv.T @ LTinv                                                     # Z_T = L_T^-T L_T^-1
    ZD = [None] * n
    ZB = [None] * (n - 1)
    ZC = [None] * n
    for i in range(n - 1, -1, -1):
        LD, LC = F.LD[i], F.LC[i]
        LDinvT = solve_triangular(LD, np.eye(b), lower=True, trans="T")      # L_Di^-T
        if i == n - 1:
            ZC[i] = -_right_solve_L(ZT @ LC, LD)
            ZD[i] = _right_solve_L(LDinvT - ZC[i].T @ LC, LD)
        else:
            LB = F.LB[i]
            ZC[i] = -_right_solve_L(ZC[i + 1] @ LB + ZT @ LC, LD)
            ZB[i] = -_right_solve_L(ZD[i + 1] @ LB + ZC[i + 1].T @ LC, LD)
            ZD[i] = _right_solve_L(LDinvT - ZB[i].T @ LB - ZC[i].T @ LC, LD)
    return SelInv(ZD, ZB, ZC, ZT)


# --------------------------------------------------------------------------------------
# Block Jacobians dD_i/dtheta_j, dB_i/dtheta_j, dC_i, dT (Eqs. 10-12)
# --------------------------------------------------------------------------------------
class Jacobians:
    """Explicit dense block Jacobians of Q_p and Q_c, built from the closed-form block
    construction.  Prior hyperparameters move Q_p and Q_c identically on the latent part;
    the noise precisions move only Q_c (tau_v A_v^T A_v)."""

    def __init__(self, model, agg: Aggregates, theta):
        self.model, self.agg, self.theta = model, agg, np.asarray(theta, dtype=np.float64)
        self.Ks = spatial_matrices(model.g, model.h)
        self.Ms = temporal_matrices(model.nt)
        self.n_prior = 3 * model.k + model.k * (model.k - 1) // 2
        self._cache = {}

    def _prior(self, j, Mrow):
        key = (j, tuple(Mrow))
        if key not in self._cache:
            dW = weight_jacobian(self.model, self.theta, j)
            self._cache[key] = prior_block(self.model, dW, self.Ks, Mrow)
        return self._cache[key]

    def dD_prior(self, j, t):
        return self._prior(j, [self.Ms[c][t, t] for c in range(3)])

    def dB_prior(self, j, t):
        return self._prior(j, [self.Ms[c][t + 1, t] for c in range(3)])

    def noise(self, v):
        """(dD diag [nt,b], dC [nt,a,b], dT [a,a]) of Q_c w.r.t. log tau_v."""
        mo = self.model
        _, _, tau = unpack_theta(mo, self.theta)
        mask = np.zeros(mo.b)
        mask[v * mo.ns : (v + 1) * mo.ns] = 1.0
        return (tau[v] * self.agg.cnt * mask[None, :],
                tau[v] * self.agg.zsum * mask[None, None, :],
                tau[v] * self.agg.ZZ[v])


def residual_sq(model, obs, x):
    """||y_v - A_v x||^2 per variable v, row by row of the literal A."""
    nt, b, ns, apr = model.nt, model.b, model.ns, model.a_per_row
    lat = obs.time.astype(np.int64) * b + obs.var.astype(np.int64) * ns + obs.node
    pred = x[lat]
    xT = x[nt * b :]
    for p in range(apr):
        pred = pred + obs.cov[:, p] * xT[obs.var * apr + p]
    res = obs.y - pred
    return np.array([np.sum(res[obs.var == v] ** 2) for v in range(model.k)])


def quad_blocks(D, B, x, b):
    """Eq. 8: x^T Q x over the BT pattern = sum x_i^T D_i x_i + 2 sum x_{i+1}^T B_i x_i (R7)."""
    n = len(D)
    q = 0.0
    for i in range(n):
        xi = x[i * b : (i + 1) * b]
        q += xi @ D[i] @ xi
    for i in range(n - 1):
        q += 2.0 * x[(i + 1) * b : (i + 2) * b] @ B[i] @ x[i * b : (i + 1) * b]
    return q


def value_and_grad(model, obs, theta, keep=False):
    """Block-sequential f (Eq. 1; readings R1, R2, R20) and grad f (Eq. 6).  Returns a dict
    with every intermediate a GPU stage can be checked against."""
    theta = np.asarray(theta, dtype=np.float64)
    nt, b, a, k = model.nt, model.b, model.a, model.k
    agg = aggregates(model, obs)
    _, _, tau = unpack_theta(model, theta)
    Qp = assemble(model, agg, theta, "prior")
    Qc = assemble(model, agg, theta, "cond")
    Fc = factor_forward(Qc)
    x = solve_upper(Fc)
    Zc = selinv(Fc)
    Fp = factor_forward(Qp)
    Zp = selinv(Fp)
    xT = x[nt * b :]
    quad_p = quad_blocks(Qp.D, Qp.B, x, b) + model.fixed_prec * (xT @ xT)
    rss = residual_sq(model, obs, x)
    nprior = 3 * k + k * (k - 1) // 2
    th_tau = theta[nprior:]
    f = (-0.5 * theta @ theta + 0.5 * Fp.logdet - 0.5 * Fc.logdet - 0.5 * quad_p
         + np.sum(0.5 * agg.mv * th_tau - 0.5 * tau * rss))
    J = Jacobians(model, agg, theta)
    grad = np.zeros(model.d)
    phaseA = np.zeros(model.d)
    phaseB = np.zeros(model.d)
    phaseC = np.zeros(model.d)
    for j in range(nprior):
        for t in range(nt):
            dD = J.dD_prior(j, t)
            xt = x[t * b : (t + 1) * b]
            phaseA[j] += np.sum(Zc.ZD[t] * dD)                          # Eq. 7, first sum
            phaseC[j] += np.sum(Zp.ZD[t] * dD)
            phaseB[j] += xt @ dD @ xt                                   # Eq. 9, first sum
        for t in range(nt - 1):
            dB = J.dB_prior(j, t)
            phaseA[j] += 2.0 * np.sum(Zc.ZB[t] * dB)                    # Eq. 7, second sum
            phaseC[j] += 2.0 * np.sum(Zp.ZB[t] * dB)
            phaseB[j] += 2.0 * x[(t + 1) * b : (t + 2) * b] @ dB @ x[t * b : (t + 1) * b]
        grad[j] = -0.5 * phaseA[j] - 0.5 * phaseB[j] + 0.5 * phaseC[j] - theta[j]
    for v in range(k):
        j = nprior + v
        dDdiag, dC, dT = J.noise(v)
        for t in range(nt):
            phaseA[j] += np.sum(np.diag(Zc.ZD[t]) * dDdiag[t])          # Eq. 7 on tau A^T A
            phaseA[j] += 2.0 * np.sum(Zc.ZC[t] * dC[t])
        phaseA[j] += np.sum(Zc.ZT * dT)
        grad[j] = -0.5 * phaseA[j] + 0.5 * agg.mv[v] - 0.5 * tau[v] * rss[v] - theta[j]
    out = dict(f=float(f), grad=grad, ld_p=Fp.logdet, ld_c=Fc.logdet, x=x, quad_p=float(quad_p),
               rss=rss, phaseA=phaseA, phaseB=phaseB, phaseC=phaseC)
    if keep:
        out.update(Qp=Qp, Qc=Qc, Fc=Fc, Fp=Fp, Zc=Zc, Zp=Zp, agg=agg)
    return out


# --------------------------------------------------------------------------------------
# The dense definition (PAPER.md:44-48 Eq. 1; :121-122 Eq. 6) -- O(N^3), tiny inputs only
# --------------------------------------------------------------------------------------
def interleave_perm(model):
    """Index map from variable-major (v, t, s) to the interleaved latent order (t, v, s) (R6)."""
    k, nt, ns = model.k, model.nt, model.ns
    perm = np.zeros(k * nt * ns, dtype=np.int64)
    for v in range(k):
        for t in range(nt):
            for s in range(ns):
                perm[(v * nt + t) * ns + s] = (t * k + v) * ns + s
    return perm


def dense_prior_literal(model, E, Lam):
    """Q_p by its definition: (Lam (x) I)^T blockdiag(Q_1..Q_k) (Lam (x) I) in variable-major
    order, Q_m = sum_c E[m,c] M_c (x) K_c, then interleaved per time step; plus the
    fixed-effect prior fixed_prec I_a (BASELINE.json configs[0], configs[3])."""
    k, nt, ns, a = model.k, model.nt, model.ns, model.a
    Ks = spatial_matrices(model.g, model.h)
    Ms = temporal_matrices(nt)
    n1 = nt * ns
    blk = np.zeros((k * n1, k * n1))
    for m in range(k):
        blk[m * n1 : (m + 1) * n1, m * n1 : (m + 1) * n1] = sum(E[m, c] * np.kron(Ms[c], Ks[c]) for c in range(3))
    LI = np.kron(Lam, np.eye(n1))
    Qvm = LI.T @ blk @ LI
    perm = interleave_perm(model)
    N = model.N
    Q = np.zeros((N, N))
    Q[np.ix_(perm, perm)] = Qvm
    Q[N - a :, N - a :] = model.fixed_prec * np.eye(a)
    return Q


def dense_A(model, obs):
    """The literal projection matrix A [m, N] and per-row variable labels."""
    A = np.zeros((obs.m, model.N))
    lat = obs.time.astype(np.int64) * model.b + obs.var.astype(np.int64) * model.ns + obs.node
    A[np.arange(obs.m), lat] = 1.0
    A[:, model.nt * model.b :] = covariate_rows(model, obs)
    return A


def dense_objective(model, obs, theta):
    """Eq. 1 from dense matrices only: returns f and the pieces."""
    theta = np.asarray(theta, dtype=np.float64)
    E, Lam, tau = unpack_theta(model, theta)
    Qp = dense_prior_literal(model, E, Lam)
    A = dense_A(model, obs)
    w = tau[obs.var]
    Qc = Qp + A.T @ (w[:, None] * A)
    r = A.T @ (w * obs.y)
    Lp = np.linalg.cholesky(Qp)
    Lc = np.linalg.cholesky(Qc)
    ld_p = 2.0 * np.sum(np.log(np.diag(Lp)))
    ld_c = 2.0 * np.sum(np.log(np.diag(Lc)))
    x = solve_triangular(Lc, solve_triangular(Lc, r, lower=True), lower=True, trans="T")
    res = obs.y - A @ x
    nprior = model.d - model.k
    loglik = sum(0.5 * np.sum(obs.var == v) * theta[nprior + v] - 0.5 * tau[v] * np.sum(res[obs.var == v] ** 2)
                 for v in range(model.k))
    f = -0.5 * theta @ theta + 0.5 * ld_p - 0.5 * ld_c - 0.5 * x @ Qp @ x + loglik
    return dict(f=float(f), ld_p=float(ld_p), ld_c=float(ld_c), x=x, Qp=Qp, Qc=Qc, A=A, res=res)


def dense_value_and_grad(model, obs, theta):
    """Eq. 6 with dense inverses: dQ/dtheta_j built by differentiating the literal
    definition term by term (product rule on (Lam (x) I)^T blockdiag (Lam (x) I))."""
    theta = np.asarray(theta, dtype=np.float64)
    k = model.k
    o = dense_objective(model, obs, theta)
    E, Lam, tau = unpack_theta(model, theta)
    Sc = np.linalg.inv(o["Qc"])
    Sp = np.linalg.inv(o["Qp"])
    x, A = o["x"], o["A"]
    grad = np.zeros(model.d)
    nprior = model.d - k
    for j in range(nprior):
        if j < 3 * k:
            m, c = divmod(j, 3)
            Ej = np.zeros_like(E)
            Ej[m, c] = E[m, c]
            dQ = dense_prior_literal(model, Ej, Lam)
        else:
            a_, b_ = lambda_index(model)[j - 3 * k]
            dLam = np.zeros_like(Lam)
            dLam[a_, b_] = 1.0
            # d/dlam of Lam^T X Lam = dLam^T X Lam + Lam^T X dLam: by polarisation of the literal builder
            dQ = 0.5 * (dense_prior_literal(model, E, Lam + dLam) - dense_prior_literal(model, E, Lam - dLam))
        dQ[model.nt * model.b :, model.nt * model.b :] = 0.0   # the fixed-effect prior does not move
        grad[j] = -0.5 * np.sum(Sc * dQ) - 0.5 * x @ dQ @ x + 0.5 * np.sum(Sp * dQ) - theta[j]
    for v in range(k):
        sel = obs.var == v
        dQ = tau[v] * A[sel].T @ A[sel]
        grad[nprior + v] = (-0.5 * np.sum(Sc * dQ) + 0.5 * np.sum(sel)
                            - 0.5 * tau[v] * np.sum(o["res"][sel] ** 2) - theta[nprior + v])
    o["grad"] = grad
    o["Sc"], o["Sp"] = Sc, Sp
    return o
