"""Pin P9: spatial-DCT closed form for log det Q_st and the Phase-C traces,
independent of every block routine.  G (free-boundary 5-point graph Laplacian on a g x g grid)
has eigenvalues lam_pq = (2 - 2cos(pi p/g)) + (2 - 2cos(pi q/g)); in that basis
Q_st = e^{th1} M0 (x) G C^-1 G + e^{th2} M1 (x) G + e^{th3} M2 (x) C decouples into ns scalar
nt x nt tridiagonals T_lam = e^{th1} lam^2/h^2 I + e^{th2} lam M1 + e^{th3} h^2 M2 (+ shift I).
TEST-ONLY: the hot path treats blocks as dense and never uses this separability.
"""
import numpy as np


def _tridiag(nt, d_end, d_mid, off):
    T = np.zeros((nt, nt))
    for i in range(nt):
        T[i, i] = d_end if i in (0, nt - 1) else d_mid
    for i in range(nt - 1):
        T[i, i + 1] = off
        T[i + 1, i] = off
    return T


def closed_form(g, nt, h, th, shift=0.0):
    """-> (ld, traces[3]): ld = log det(Q_st + shift I); traces[j] = e^{th_j} <(Q_st+shift I)^-1, P_j>."""
    e1, e2, e3 = np.exp(th[0]), np.exp(th[1]), np.exp(th[2])
    M1 = _tridiag(nt, 1.0, 2.0, -1.0) if nt > 1 else np.zeros((1, 1))
    M2 = _tridiag(nt, 2.0, 2.0, -1.0)
    I = np.eye(nt)
    ld = 0.0
    tr = np.zeros(3)
    for p in range(g):
        for q in range(g):
            lam = (2.0 - 2.0 * np.cos(np.pi * p / g)) + (2.0 - 2.0 * np.cos(np.pi * q / g))
            X = [e1 * lam * lam / (h * h) * I, e2 * lam * M1, e3 * h * h * M2]
            T = X[0] + X[1] + X[2] + shift * I
            sign, l = np.linalg.slogdet(T)
            assert sign > 0
            ld += l
            Ti = np.linalg.inv(T)
            for j in range(3):
                tr[j] += np.sum(Ti * X[j])
    return ld, tr
