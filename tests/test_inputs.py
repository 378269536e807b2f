"""The seeded input generators: determinism, shapes and sizes of the BASELINE.json configs, and
that the angle-addition table fill equals the direct cosine sum it documents."""
import numpy as np

from paper_1802_06922_b200 import inputs


def test_config_sizes_match_baseline():
    # BASELINE.json: ~1.8 GB, ~8.6 GB, ~21 GB fp32 tables; fp64 Ainv 4 GB total at 'large'
    assert abs(inputs.CONFIGS["mid"].table_bytes() / 1e9 - 1.81) < 0.01
    assert abs(inputs.CONFIGS["large"].table_bytes() / 1e9 - 8.59) < 0.01
    assert abs(inputs.CONFIGS["xlarge"].table_bytes() / 1e9 - 21.47) < 0.01
    c = inputs.CONFIGS["large"]
    assert c.nw * c.norb * c.norb * 8 == 4 * 2 ** 30


def test_tiny_is_deterministic_and_in_range():
    a, b = inputs.make_inputs("tiny"), inputs.make_inputs("tiny")
    assert np.array_equal(a.coefs_numpy(), b.coefs_numpy())
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.delta, b.delta)
    assert a.coefs.shape == (16, 16, 16, 8) and a.pos.shape == (4, 8, 3)
    assert a.delta.shape == (1, 8, 4, 3) and a.unif.shape == (1, 8, 4)
    assert float(a.coefs.abs().max()) <= 1.0
    assert 0.0 <= a.unif.min() and a.unif.max() < 1.0
    assert abs(a.delta.std() - 0.05) < 0.01


def test_planewave_table_equals_direct_sum():
    cfg = inputs.custom_config("pw", (6, 5, 7), 9, (2.0, 2.5, 3.0), nw=2, kmax=(2, 2, 3))
    x = inputs.make_inputs(cfg)
    n, a, th = x.pw["n"], x.pw["a"], x.pw["theta"]
    I = np.stack(np.meshgrid(np.arange(6) / 6, np.arange(5) / 5, np.arange(7) / 7, indexing="ij"), -1)
    ref = np.zeros((6, 5, 7, 9))
    for j in range(9):
        for m in range(cfg.nterms):
            ref[..., j] += a[j, m] * np.cos(2 * np.pi * (I @ n[j, m]) + th[j, m])
    got = x.coefs_numpy()
    assert got.dtype == np.float32
    assert np.max(np.abs(got - ref)) < 2e-7
    assert np.max(np.abs(got)) <= 1.0
    # chunked fill gives the same bits
    y = inputs.planewave_table(cfg.grid, n, a, th, xchunk=1)
    assert np.array_equal(y.numpy(), got)


def test_positions_inside_cell_and_overrides():
    x = inputs.make_inputs("small", nw=3, nsweeps=1, with_table=False)
    assert x.coefs is None and x.pos.shape == (3, 128, 3) and x.delta.shape == (1, 128, 3, 3)
    u = x.pos @ np.linalg.inv(x.lattice)
    assert u.min() >= 0 and u.max() < 1
    assert abs(x.delta.std() - 0.16) < 0.01
