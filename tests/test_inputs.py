"""Input generator (dfjk_inputs): determinism, distribution, recipe structure. No DF-JK arithmetic."""
import numpy as np

import dfjk_inputs as gi


def test_counter_rng_is_pure_and_uniform():
    a = gi.uniform(3, 5, 20000)
    b = gi.uniform(3, 5, 20000)
    assert np.array_equal(a, b)
    assert not np.array_equal(a, gi.uniform(4, 5, 20000))
    assert not np.array_equal(a, gi.uniform(3, 6, 20000))
    assert 0.0 < a.min() and a.max() < 1.0
    assert abs(a.mean() - 0.5) < 0.01 and abs(a.var() - 1 / 12) < 0.005
    z = gi.normals(3, 2, 40000)
    assert abs(z.mean()) < 0.02 and abs(z.std() - 1.0) < 0.02
    assert len(np.unique(gi.raw_bits(0, 0, 5000))) == 5000


def test_rows_are_independent_of_slab_choice():
    cfg = gi.CONFIGS[1]
    full = gi.fill_B_host(cfg)
    assert full.shape == (cfg.naux, cfg.npair)
    part = gi.fill_B_host(cfg, P0=37, nrows=11)
    assert np.array_equal(full[37:48], part)


def test_recipe_structure():
    cfg = gi.CONFIGS[1]
    x, a = gi.centers(cfg), gi.aux_scales(cfg)
    assert np.all(np.diff(x) >= 0) and 0 <= x.min() and x.max() <= 10
    P = np.arange(cfg.naux)
    u = a / np.exp(-P / cfg.naux)
    assert u.min() >= 0.05 and u.max() <= 1.0
    B = gi.fill_B_host(cfg)
    il = np.tril_indices(cfg.nao)
    g = np.exp(-0.25 * (x[il[0]] - x[il[1]]) ** 2)
    z = (B / (a[:, None] * g[None, :]) - 1.0) / 0.1
    assert abs(z.mean()) < 0.02 and abs(z.std() - 1.0) < 0.02


def test_orbitals_orthonormal_and_schedules():
    for cid in (1, 2):
        cfg = gi.CONFIGS[cid]
        C0 = gi.orbitals(cfg, 0)[0]
        assert C0.shape == (cfg.nao, cfg.nocc[0]) and C0.flags.c_contiguous
        assert np.allclose(C0.T @ C0, np.eye(cfg.nocc[0]), atol=1e-12)
    cfg = gi.CONFIGS[2]
    assert not np.allclose(gi.orbitals(cfg, 0)[0], gi.orbitals(cfg, 1)[0])
    rot = gi.custom_config(40, 10, (4, 3), seed=9, calls=3, schedule="rotate")
    Ca0, Cb0 = gi.orbitals(rot, 0)
    Ca1, _ = gi.orbitals(rot, 1)
    assert Ca0.shape == (40, 4) and Cb0.shape == (40, 3)
    assert np.allclose(Ca1.T @ Ca1, np.eye(4), atol=1e-12)
    # a small rotation: subspaces close but not equal
    s = np.linalg.svd(Ca0.T @ Ca1, compute_uv=False)
    assert s.min() > 0.9 and s.min() < 1.0 - 1e-6
