import numpy as np

from workloads import CONFIGS, draw_obs, make_config, make_w0
from workloads.generate import normals, uniforms


def test_streams_deterministic_and_elementwise():
    u = uniforms(1000, 0, 1000)
    assert np.array_equal(u, uniforms(1000, 0, 1000))
    assert np.array_equal(u[:10], uniforms(1000, 0, 10))       # counter-based: prefix-stable
    assert not np.array_equal(u, uniforms(1000, 1, 1000))
    assert 0.0 <= u.min() and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.03
    z = normals(1001, 1, 200000)
    assert abs(z.mean()) < 0.01 and abs(z.std() - 1.0) < 0.01


def test_config_shapes():
    for idx, (b, nt, a, m, d) in {0: (16, 6, 2, 200, 4), 1: (400, 50, 4, 20000, 4)}.items():
        model, obs, th = make_config(idx)
        assert (model.b, model.nt, model.a, obs.m, model.d) == (b, nt, a, m, d)
        assert th.shape == (d,)
        assert obs.cov.shape == (m, model.a_per_row)
        assert obs.node.max() < model.ns and obs.time.max() < model.nt
    mo = CONFIGS[3][0]
    assert (mo.b, mo.d, mo.a_per_row, mo.N) == (3072, 15, 2, 64 * 3072 + 6)
    mo = CONFIGS[4][0]
    assert (mo.b, mo.nt, mo.N) == (4096, 128, 524296)
    assert np.allclose(make_config(0)[2], [0.1, -0.2, 0.3, 0.0])


def test_multivariate_rows():
    mo = CONFIGS[3][0]
    obs = draw_obs(mo, 100, 3)
    assert obs.m == 300
    assert np.array_equal(np.bincount(obs.var), [100, 100, 100])


def test_w0_recipe():
    model, obs, th = make_w0()
    assert obs.m == 200
    pick = obs.time * 16 + obs.node
    assert pick[0] == 11 and pick[1] == 48
    cnt = np.bincount(pick, minlength=96)
    assert cnt.min() >= 1 and cnt.max() == 3          # every site hit, max count 3
    assert abs(obs.y[0] - np.sin(1.3)) < 1e-15
