"""The seeded generator: shapes, determinism, in-bounds scans, recipe facts."""
import numpy as np
import pytest

from paper_2505_07814_b200 import synth


@pytest.mark.parametrize("c", [1, 2, 3, 4, 5])
def test_scan_geometry_in_bounds(c):
    cfg = synth.get_config(c)
    assert cfg.origin == {1: 3, 2: 3, 3: 3, 4: 35, 5: 37}[c]
    for pos in (synth.true_positions(cfg), synth.raster(cfg)):
        r = np.floor(pos.astype(np.float64) + 0.5)
        assert pos.shape == (cfg.n_positions, 2)
        assert r.min() >= 0 and r.max() + cfg.N <= cfg.H
    rng = np.random.default_rng(1000 * c + 4)          # evaluation point A perturbation bound
    assert cfg.origin - cfg.jitter - 0.6 > 0.5


def test_config1_arrays_and_determinism():
    cfg = synth.get_config(1)
    t1, t2 = synth.truth(cfg), synth.truth(cfg)
    for k in t1:
        assert np.array_equal(t1[k], t2[k])
    assert t1["object"].shape == (1, 160, 160) and t1["object"].dtype == np.complex64
    assert t1["probe"].shape == (1, 64, 64) and t1["probe"].dtype == np.complex64
    assert t1["positions"].dtype == np.float32
    assert np.isclose(np.abs(np.angle(t1["object"])).max(), 0.5, rtol=1e-5)
    assert np.isclose((np.abs(t1["probe"]) ** 2).sum(), 1e4, rtol=1e-5)
    a, b = synth.eval_point(cfg, "A"), synth.eval_point(cfg, "B")
    assert not np.array_equal(a["object"], t1["object"])
    assert np.allclose(np.abs(b["object"]), 1.0) and np.array_equal(b["positions"], synth.raster(cfg).astype(np.float32))


def test_probe_modes_orthogonal_with_stated_powers():
    cfg = synth.get_config(2)
    P = synth.make_probe(cfg).astype(np.complex128).reshape(cfg.M, -1)
    G = P.conj() @ P.T
    pw = np.real(np.diag(G))
    assert np.allclose(pw / pw.sum(), cfg.powers, atol=1e-6)
    assert np.abs(G - np.diag(np.diag(G))).max() < 1e-6 * pw.max()


def test_minibatches_partition_the_scan_and_poisson_is_per_position():
    cfg = synth.get_config(1)
    idx = np.concatenate([synth.minibatch(cfg, j) for j in range(cfg.n_positions // cfg.B)])
    assert sorted(idx.tolist()) == list(range(cfg.n_positions))
    assert synth.compact_minibatch(cfg, 1).tolist() == list(range(32, 64))
    I = np.full((3, 4, 4), 5.0)
    a = synth.poisson_amplitudes(cfg, I, [7, 3, 9])
    b = synth.poisson_amplitudes(cfg, I[:2], [3, 7])
    assert a.dtype == np.float32 and np.array_equal(a[0], b[1]) and np.array_equal(a[1], b[0])
    assert np.allclose(a ** 2, np.round(a ** 2))
