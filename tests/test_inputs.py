"""The seeded generator (paper_2502_07060_b200/inputs.py): on-shell, momentum
conserving, transverse -- the checks PAPER.md:182 lists for its phase-space
generator (tests/test_phase_space.py there) -- plus determinism and slicing."""
import numpy as np
import pytest

from paper_2502_07060_b200 import inputs

P = inputs.P31


def _dot_fp(x, y):
    x = x.astype(object)
    y = y.astype(object)
    t = x * y
    return (t[..., 0] - t[..., 1:].sum(-1)) % P


@pytest.mark.parametrize("n,d", [(4, 4), (8, 6), (10, 8), (12, 6)])
def test_fp_points_are_physical(n, d):
    mom, pol, info = inputs.make_fp_inputs(n, d, 64, seed=0)
    assert mom.dtype == np.uint32 and mom.shape == (64, n, d)
    assert mom.max() < P and pol.max() < P
    assert not (mom.astype(object).sum(axis=1) % P).any()            # conservation
    assert not _dot_fp(mom, mom).any()                               # on shell
    assert not _dot_fp(pol, mom).any()                               # transverse
    m = n - 1
    for i in range(m):
        for j in range(i + 1, m):
            if i == 0 and j == m - 1:
                continue
            Pij = mom[:, i:j + 1].astype(object).sum(axis=1) % P
            assert _dot_fp(Pij, Pij).all()                           # proper invariants != 0
    assert info["redraws"] >= 0


@pytest.mark.parametrize("n,d,hel", [(6, 4, (-1, -1, 1, 1, 1, 1)), (12, 6, None), (5, 5, None)])
def test_complex_points_are_physical(n, d, hel):
    mom, pol, _ = inputs.make_complex_inputs(n, d, 64, seed=0, helicities=hel)

    def dot(x, y):
        return x[..., 0] * y[..., 0] - (x[..., 1:] * y[..., 1:]).sum(-1)

    assert np.abs(mom.sum(axis=1)).max() < 1e-9
    assert np.abs(dot(mom, mom)).max() < 1e-9
    assert np.abs(dot(pol, mom)).max() < 1e-7


def test_determinism_and_slicing():
    a = inputs.make_fp_inputs(6, 4, 100, seed=7)
    b = inputs.make_fp_inputs(6, 4, 100, seed=7)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
    c = inputs.make_fp_inputs(6, 4, 40, seed=7, start=60)
    assert np.array_equal(a[0][60:], c[0]) and np.array_equal(a[1][60:], c[1])
    d_ = inputs.make_fp_inputs(6, 4, 100, seed=8)
    assert not np.array_equal(a[0], d_[0])
    x = inputs.make_complex_inputs(6, 4, 50, seed=7)
    y = inputs.make_complex_inputs(6, 4, 20, seed=7, start=30)
    assert np.array_equal(x[0][30:], y[0]) and np.array_equal(x[1][30:], y[1])


def test_value_distribution():
    mom, pol, _ = inputs.make_fp_inputs(8, 6, 2048, seed=0)
    # residues fill the field: mean ~ p/2
    assert abs(mom.astype(np.float64).mean() / P - 0.5) < 0.02
    assert abs(pol.astype(np.float64).mean() / P - 0.5) < 0.02
    momc, _, _ = inputs.make_complex_inputs(8, 6, 2048, seed=0)
    free = momc[:, :6, 2:]          # transverse components of the free legs are the raw draws
    assert free.real.min() >= -1 and free.real.max() < 1
    assert abs(free.real.mean()) < 0.05 and abs(free.imag.mean()) < 0.05


def test_configs_table():
    assert set(inputs.CONFIGS) == {"cfg0", "cfg1", "cfg2", "cfg3", "cfg4a", "cfg4b"}
    mom, pol, _ = inputs.make_config("cfg1", batch=8)
    assert mom.shape == (8, 6, 4) and mom.dtype == np.complex128
    mom, pol, _ = inputs.make_config("cfg3", batch=8)
    assert mom.shape == (8, 10, 8) and mom.dtype == np.uint32
