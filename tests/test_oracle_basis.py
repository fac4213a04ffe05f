"""Pins for the oracle's sizes and radial basis (C2; Eqs. 17-18; Table II)."""
import os

import numpy as np

from oracle import nep_oracle as O
from paper_2606_19557_b200.workloads import ModelSpec
from tests._ref_np import np_fk

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [l.split() for l in f if l.strip() and not l.startswith("#")]


def test_table2_parameter_counts():
    # the paper's printed integers pin inclusive index ranges, D, (D+2)H per species,
    # one shared b1 and T^2 independent coefficient sets
    for r in _rows("table2_param_counts.txt"):
        T, nR, nA, bR, bA, l3, l4, l5, H, npar = map(int, r)
        m = ModelSpec(T, 6.0, 5.0, nR, nA, bR, bA, l3, l4, l5, H)
        assert O.num_params(m) == npar
        assert m.n_par == npar            # the generator module's bookkeeping agrees
        assert O.num_descriptors(m) == (nR + 1) + (nA + 1) * 6


def test_descriptor_count_3body_only():
    m = ModelSpec(1, 5.0, 4.0, 4, 4, 8, 8, 4, 0, 0, 30)
    assert O.num_descriptors(m) == 25 and O.num_params(m) == 901


def test_basis_vanishes_with_derivative_at_cutoff():
    # "Both f_k(r) and its first derivative vanish continuously at r = r_c"
    for rc in (3.7, 6.0):
        f, df = O.radial_basis(rc, rc, 12)
        assert np.abs(f).max() < 1e-15 and np.abs(df).max() < 1e-14
        f, df = O.radial_basis(rc * (1 - 1e-6), rc, 12)
        assert np.abs(f).max() < 1e-10 and np.abs(df).max() < 1e-4


def test_basis_limits():
    f, _ = O.radial_basis(1e-12, 5.0, 8)
    assert np.allclose(f, 1.0, atol=1e-10)          # T_k(1) = 1, fc(0) = 1
    for r in (0.3, 2.2, 4.9):
        f, _ = O.radial_basis(r, 5.0, 8)
        assert abs(f[0] - 0.5 * (np.cos(np.pi * r / 5.0) + 1)) < 1e-15   # f_0 = f_c (Eq. 18)


def test_basis_against_numpy_chebyshev():
    rng = np.random.default_rng(0)
    for rc, bs in ((5.0, 8), (4.2, 10), (6.0, 12)):
        for r in rng.uniform(0.05, rc, size=20):
            f, _ = O.radial_basis(r, rc, bs)
            assert np.allclose(f, np_fk(r, rc, bs), rtol=0, atol=2e-13)


def test_basis_derivative_against_finite_difference():
    rng = np.random.default_rng(1)
    h = 1e-6
    for r in rng.uniform(0.2, 4.9, size=10):
        _, df = O.radial_basis(r, 5.0, 10)
        fp, _ = O.radial_basis(r + h, 5.0, 10)
        fm, _ = O.radial_basis(r - h, 5.0, 10)
        assert np.allclose(df, (fp - fm) / (2 * h), atol=1e-7)
