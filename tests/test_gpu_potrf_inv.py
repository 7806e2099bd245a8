"""Kernel-level check of the block factorisation of the forward sweeps (Algorithm 1 line 3, in the
inverse-diagonal form of DESIGN.md §5): the one-CTA POTRF + TRTRI leaf (n <= 128) and the blocked recursion over
leaves and DMMA GEMMs (n > 128), through include/bta_diag.h: bta_diag_potrf_inv, against numpy's dense Cholesky and
triangular inverse in FP64 on ragged sizes.  (The whole-gradient parity tests run through the same code; this test
isolates it and covers sizes and scalings the models do not produce.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from workloads import make_w0

SIZES = [1, 15, 16, 17, 100, 128, 129, 144, 250, 256, 300, 400, 417, 511, 512, 640]


def _spd(n, seed):
    rng = np.random.default_rng(seed)
    M = rng.standard_normal((n, n))
    A = M @ M.T / n + np.eye(n) * (0.5 + rng.random())
    s = np.exp(rng.uniform(-2.0, 2.0, n))             # rows / columns of very different magnitude
    return A * s[:, None] * s[None, :]


@pytest.fixture(scope="module")
def ctx():
    from paper_2605_06392_b200 import BtaModel
    model, obs, _ = make_w0()
    M = BtaModel.from_workload(model, obs, device=0)
    yield M
    M.close()


@pytest.mark.parametrize("n", SIZES)
def test_potrf_inv_matches_numpy(ctx, n):
    import torch
    A = _spd(n, 100 + n)
    L = np.linalg.cholesky(A)
    X = np.linalg.inv(L)
    ld = n + 3                                           # a leading dimension that is not the size
    runs = []
    for _ in range(2):                                   # fresh input twice: bitwise repeatable
        buf = torch.full((n, ld), 7.0, dtype=torch.float64, device="cuda")
        buf[:, :n] = torch.from_numpy(np.tril(A)).cuda()   # lower triangle authoritative, strict upper zero
        dl = torch.zeros(n, dtype=torch.float64, device="cuda")
        ctx.diag_potrf_inv(buf[:, :n], diagL=dl)
        runs.append((buf.cpu().numpy(), dl.cpu().numpy()))
    assert np.array_equal(runs[0][0], runs[1][0]) and np.array_equal(runs[0][1], runs[1][1])
    full, dl = runs[0]
    assert np.all(full[:, n:] == 7.0)                    # nothing written beyond the block's columns
    got = full[:, :n]
    assert np.all(np.triu(got, 1) == 0.0)
    assert np.max(np.abs(got @ L - np.eye(n))) <= 1e-13 * np.linalg.cond(L) + 1e-12
    assert np.max(np.abs(got - X)) <= 1e-10 * np.max(np.abs(X))
    assert np.allclose(dl, np.diag(L), rtol=1e-12, atol=0.0)


@pytest.mark.parametrize("n,badrow", [(100, 37), (300, 201)])
def test_potrf_inv_reports_first_bad_pivot(ctx, n, badrow):
    import torch
    from paper_2605_06392_b200 import binding as B
    A = _spd(n, 5)
    A[badrow - 1, badrow - 1] = -1.0                     # leading minor of order badrow-1 SPD, pivot badrow not
    buf = torch.from_numpy(np.tril(A)).cuda()
    with pytest.raises(B.BtaError) as ei:
        ctx.diag_potrf_inv(buf)
    assert ei.value.code == 4                            # BTA_ERR_NOTSPD
    assert ctx.last_pivot() == badrow
