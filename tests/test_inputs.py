"""The seeded input generators (lqcd_inputs): reproducible, order-independent, right distributions.
P1 of SURVEY.md §8(c4): generated links are unitary with det = 1."""
import numpy as np
import torch

import lqcd_inputs as gen


def c(a):
    return np.ascontiguousarray(a).view(np.complex128)[..., 0]


def test_links_are_su3():
    U = c(gen.random_su3_links((4, 4, 4, 2)).numpy())
    eye = np.eye(3)
    assert np.abs(U @ np.conj(np.swapaxes(U, -1, -2)) - eye).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
    # not something trivial: mean |Re tr U| of Haar-ish matrices is well below 3
    assert np.abs(np.trace(U, axis1=-2, axis2=-1)).mean() < 1.5


def test_generation_is_counter_based():
    L = (4, 2, 4, 2)
    a = gen.random_su3_links(L, chunk=1 << 20)
    b = gen.random_su3_links(L, chunk=37)
    assert torch.equal(a, b)
    f1 = gen.gaussian_field(L, chunk=1 << 20)
    f2 = gen.gaussian_field(L, chunk=101)
    assert torch.equal(f1, f2)
    assert not torch.equal(gen.gaussian_field(L, seed=1), gen.gaussian_field(L, seed=2))
    assert not torch.equal(gen.random_su3_links(L, seed=1), gen.random_su3_links(L, seed=2))
    # the field and the link streams are unrelated even with equal seeds
    assert abs(float(torch.corrcoef(torch.stack((
        gen.gaussian_field(L, seed=5).flatten()[:384], gen.random_su3_links(L, seed=5).flatten()[:384]
    )))[0, 1])) < 0.2


def test_gaussian_moments():
    f = gen.gaussian_field((8, 8, 8, 8)).numpy().ravel()
    n = f.size
    assert abs(f.mean()) < 5 / np.sqrt(n)
    assert abs(f.var() - 1) < 5 * np.sqrt(2 / n)
    assert abs((f ** 4).mean() - 3) < 0.15
    re, im = f[0::2], f[1::2]
    assert abs(np.corrcoef(re, im)[0, 1]) < 5 / np.sqrt(n / 2)


def test_uniform_is_open_interval_and_flat():
    ctr = torch.arange(0, 200000, dtype=torch.int64)
    u = gen.uniform01(3, 4, ctr).numpy()
    assert u.min() > 0 and u.max() < 1
    hist, _ = np.histogram(u, bins=20, range=(0, 1))
    assert np.abs(hist - 10000).max() < 500


def test_configs_and_shifts():
    s = gen.CONFIGS["config2_16^4"]["shifts"]
    assert len(s) == 8 and abs(s[0] - 1e-4) < 1e-18 and abs(s[-1] - 1e-4 * 10 ** 3.5) < 1e-12
    s = gen.CONFIGS["config4_48^4"]["shifts"]
    assert len(s) == 16 and abs(s[0] - 1e-5) < 1e-18 and abs(s[-1] - 1.0) < 1e-12
    assert gen.CONFIGS["config5_64^4"]["mass"] == 0.005
    U = gen.unit_links((2, 2, 2, 2))
    assert U.shape == (4, 16, 3, 3, 2) and float(U.sum()) == 4 * 16 * 3
