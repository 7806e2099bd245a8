"""Kernel-level check of the bandwidth-bound rows-times-block products of the sweeps (csrc/skinny.cu): the forward
sweeps' transposed form  out = alpha R M^T + beta in  (Algorithm 1 lines 4-5 and 9) and the backward
sweeps' form  out = alpha R M + beta in  (Eqs. 3-5), full and triangular, against the same products
formed with numpy in FP64, on ragged sizes, in place, and bitwise repeatable."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

SHAPES = [(1, 16, 16), (2, 25, 25), (4, 81, 81), (9, 400, 400), (9, 417, 417), (5, 1000, 700), (16, 300, 300),
          (9, 2304, 2304)]


@pytest.mark.parametrize("P,J,K", SHAPES)
@pytest.mark.parametrize("tri", [0, 1])
def test_rows_times_block_t(P, J, K, tri):
    import torch
    from paper_2605_06392_b200 import binding as B
    if tri and J != K:
        pytest.skip("triangular operand is square")
    rng = np.random.default_rng(1000 * P + J + tri)
    R = rng.standard_normal((P, K))
    M = rng.standard_normal((J, K))
    inp = rng.standard_normal((P, J))
    Mref = np.tril(M) if tri else M
    ref = -0.75 * R @ Mref.T + 1.25 * inp
    Rd, Md = torch.from_numpy(R).cuda(), torch.from_numpy(M).cuda()      # garbage above the diagonal must not be read
    out = torch.from_numpy(inp).cuda()                                   # in place: in == out
    B.rows_times_block_t(Rd, Md, out, alpha=-0.75, beta=1.25, inp=out, tri=tri)
    got = out.cpu().numpy()
    scale = np.max(np.abs(ref))
    assert np.max(np.abs(got - ref)) <= 1e-13 * scale * np.sqrt(K)
    out2 = torch.from_numpy(inp).cuda()
    B.rows_times_block_t(Rd, Md, out2, alpha=-0.75, beta=1.25, inp=out2, tri=tri)
    assert torch.equal(out, out2)
    out3 = torch.full((P, J), 3.0, dtype=torch.float64, device="cuda")  # beta = 0: `in` is never read
    B.rows_times_block_t(Rd, Md, out3, alpha=2.0, beta=0.0, inp=None, tri=tri)
    assert np.max(np.abs(out3.cpu().numpy() - 2.0 * R @ Mref.T)) <= 1e-13 * 2.0 * scale * np.sqrt(K) + 1e-12


@pytest.mark.parametrize("P,K,J", [(1, 400, 400), (9, 417, 417), (4, 1000, 700), (9, 2304, 2304)])
@pytest.mark.parametrize("tri", [0, 1])
def test_rows_times_block(P, K, J, tri):
    import torch
    from paper_2605_06392_b200 import binding as B
    if tri and J != K:
        pytest.skip("triangular operand is square")
    rng = np.random.default_rng(77 * P + J + tri)
    R = rng.standard_normal((P, K))
    M = rng.standard_normal((K, J))
    inp = rng.standard_normal((P, J))
    Mref = np.tril(M) if tri else M
    ref = 0.5 * R @ Mref - inp
    Rd, Md = torch.from_numpy(R).cuda(), torch.from_numpy(M).cuda()
    out = torch.from_numpy(inp).cuda()
    part = torch.empty(((K + 127) // 128) * P * J, dtype=torch.float64, device="cuda")
    B.rows_times_block(Rd, Md, out, part, alpha=0.5, beta=-1.0, inp=out, tri=tri)
    assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-13 * np.max(np.abs(ref)) * np.sqrt(K)
