"""Regenerates tests/golden/w0.txt and p13.txt from the DENSE DEFINITION at 40 digits (mpmath), independently of
oracle/ and of the CUDA path: Eq. 1 through a dense Cholesky of the literal N x N matrices, Eq. 6
 through the dense inverse, tr(Q^-1 dQ/dtheta_j).  The stored digits were first computed by the survey
(SURVEY.md §8(c), App. B); this script makes them reproducible.

    python tests/golden/make_golden.py            # print both files' key = value lines
    python tests/golden/make_golden.py --check    # compare with the stored files (relative 1e-13), exit 1 on mismatch

Inputs only from `workloads` (the RNG-free worked example W0); base matrices are rebuilt here from their
definitions (readings R3, R4, R21 of DESIGN.md): C = h^2 I, G = degree - adjacency on the g x g grid, K2 = G C^-1 G,
M0 = I, M1 = D^T D, M2 = tridiag(-1, 2, -1).
"""
import os
import sys

import mpmath as mp

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
mp.mp.dps = 40


def kron(A, B):
    out = mp.zeros(A.rows * B.rows, A.cols * B.cols)
    for i in range(A.rows):
        for j in range(A.cols):
            if A[i, j] != 0:
                for p in range(B.rows):
                    for q in range(B.cols):
                        out[i * B.rows + p, j * B.cols + q] = A[i, j] * B[p, q]
    return out


def base_matrices(g, nt, h):
    ns = g * g
    G = mp.zeros(ns, ns)
    for iy in range(g):
        for ix in range(g):
            s = iy * g + ix
            for dy, dx in ((0, 1), (0, -1), (1, 0), (-1, 0)):
                jy, jx = iy + dy, ix + dx
                if 0 <= jy < g and 0 <= jx < g:
                    G[s, s] += 1
                    G[s, jy * g + jx] -= 1
    h2 = mp.mpf(h) ** 2
    K = [G * G / h2, G, mp.eye(ns) * h2]                      # paired with M0, M1, M2
    M0, M1, M2 = mp.eye(nt), mp.zeros(nt, nt), mp.eye(nt) * 2
    for i in range(nt - 1):
        M1[i, i] += 1
        M1[i + 1, i + 1] += 1
        M1[i, i + 1] -= 1
        M1[i + 1, i] -= 1
        M2[i, i + 1] = M2[i + 1, i] = -1
    return [kron(M, Kc) for M, Kc in zip((M0, M1, M2), K)]   # P_c = M_c (x) K_c, latent part


def logdet(Q):
    L = mp.cholesky(Q)
    return 2 * sum(mp.log(L[i, i]) for i in range(Q.rows))


def frob(A, B):
    return sum(A[i, j] * B[i, j] for i in range(A.rows) for j in range(A.cols))


def embed(P, N):
    out = mp.zeros(N, N)
    for i in range(P.rows):
        for j in range(P.cols):
            out[i, j] = P[i, j]
    return out


def w0_values():
    from workloads import make_w0
    model, obs, th = make_w0()
    N, a, n = model.N, model.a, model.nt * model.b
    theta = [mp.mpf(float(t)) for t in th]
    e = [mp.e ** t for t in theta]
    P = [embed(Pc, N) for Pc in base_matrices(model.g, model.nt, model.h)]
    Qp = e[0] * P[0] + e[1] * P[1] + e[2] * P[2]
    for i in range(n, N):
        Qp[i, i] += mp.mpf("0.001")
    A = mp.zeros(obs.m, N)
    for i in range(obs.m):
        A[i, int(obs.time[i]) * model.b + int(obs.node[i])] = 1
        for p in range(a):
            A[i, n + p] = mp.mpf(float(obs.cov[i, p]))
    y = mp.matrix([mp.mpf(float(v)) for v in obs.y])
    AtA = A.T * A
    Qc = Qp + e[3] * AtA
    x = mp.cholesky_solve(Qc, e[3] * (A.T * y))
    res = y - A * x
    rss = (res.T * res)[0]
    quad = (x.T * Qp * x)[0]
    ld_p, ld_c = logdet(Qp), logdet(Qc)
    f = -sum(t * t for t in theta) / 2 + ld_p / 2 - ld_c / 2 - quad / 2 + obs.m * theta[3] / 2 - e[3] * rss / 2
    Sc, Sp = Qc ** -1, Qp ** -1
    phaseA = [e[j] * frob(Sc, P[j]) for j in range(3)] + [e[3] * frob(Sc, AtA)]
    phaseB = [e[j] * (x.T * P[j] * x)[0] for j in range(3)]
    phaseC = [e[j] * frob(Sp, P[j]) for j in range(3)]
    grad = [-phaseA[j] / 2 - phaseB[j] / 2 + phaseC[j] / 2 - theta[j] for j in range(3)]
    grad.append(-phaseA[3] / 2 + mp.mpf(obs.m) / 2 - e[3] * rss / 2 - theta[3])
    return {"ld_p": [ld_p], "ld_c": [ld_c], "f": [f], "grad": grad, "phaseA": phaseA, "phaseB": phaseB,
            "rss": [rss], "quad_p": [quad], "xT": [x[n], x[n + 1]]}


def p13_values():
    out = {}
    th = [mp.mpf("0.1"), mp.mpf("-0.2"), mp.mpf("0.3")]
    e = [mp.e ** t for t in th]
    for h, tag in ((1.0, "h1"), (0.5, "h05")):
        P = base_matrices(4, 6, h)
        Q = e[0] * P[0] + e[1] * P[1] + e[2] * P[2]
        S = Q ** -1
        out["ld_Qst_" + tag] = [logdet(Q)]
        out["traces_" + tag] = [e[j] * frob(S, P[j]) for j in range(3)]
        if tag == "h1":
            out["ld_Qp_h1"] = [logdet(Q) + 2 * mp.log(mp.mpf("0.001"))]
            Qu = Q + mp.eye(Q.rows)                                  # uniform design c = 1, tau = 1 (pin P12)
            Su = Qu ** -1
            out["ld_uniform"] = [logdet(Qu)]
            out["traces_uniform"] = [e[j] * frob(Su, P[j]) for j in range(3)]
    return out


def read_stored(name):
    out = {}
    with open(os.path.join(ROOT, "tests", "golden", name)) as fh:
        for line in fh:
            line = line.split("#", 1)[0].strip()
            if line:
                k, v = line.split("=", 1)
                out[k.strip()] = [mp.mpf(t) for t in v.split()]
    return out


def main():
    check = "--check" in sys.argv
    bad = 0
    for name, vals in (("w0.txt", w0_values()), ("p13.txt", p13_values())):
        stored = read_stored(name) if check else {}
        print(f"# {name}")
        for k, v in vals.items():
            print(f"{k} = " + " ".join(mp.nstr(t, 17) for t in v))
            if check:
                for got, want in zip(v, stored[k]):
                    if abs(got - want) > mp.mpf("1e-13") * abs(want):
                        print(f"  MISMATCH {k}: stored {want}")
                        bad += 1
    return 1 if bad else 0


if __name__ == "__main__":
    sys.exit(main())
