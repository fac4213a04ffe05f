"""Pins of oracle/pair_correction.py (the short-range pair correction of P:105, fixed form with the caller's constants: DESIGN G29)
against what physics and mathematics fix, not against its own formula:
Coulomb's law in the unscreened limit (also pins "one phi per undirected pair"), the slope of a one-term screening function, the
switch at its mid-point / quarter-point / outer radius, forces and virial as finite differences of the energy (periodic, multi-image,
multi-species), Newton's third law, and independence of the model's parameters."""
import dataclasses

import numpy as np
import pytest

from oracle import nep_oracle as O
from oracle import pair_correction as PC
from paper_2606_19557_b200 import workloads as wl

KC = 14.4          # any positive number serves: the constant is the caller's
MODEL = wl.ModelSpec(2, 4.0, 3.0, 1, 1, 2, 2, 4, 0, 0, 3)


def _dimer(r, box=40.0, types=(0, 1)):
    pos = np.array([[1.0, 2.0, 3.0], [1.0 + r * 0.6, 2.0, 3.0 + r * 0.8]])      # |d| = r, oblique
    st = wl.StructureSet(np.array([2], np.int32), pos, (np.eye(3) * box).reshape(1, 9), np.array(types, np.int32), ["dimer"])
    return O.OracleData(MODEL, st)


def test_unscreened_limit_is_coulombs_law_once_per_pair():
    Z = np.array([3.0, 5.0])
    for r in (0.4, 1.1, 2.5):
        E, F, W = PC.pair_correction(_dimer(r), Z, 3.0, 3.5, [0.25, 0.75], [0.0, 0.0], 0.7, 0.3, KC)
        assert E[0] == pytest.approx(KC * 15.0 / r, rel=1e-13)                    # k q1 q2 / r: not half of it, not twice
        f = KC * 15.0 / r ** 2                                                    # repulsion of magnitude k q1 q2 / r^2 along the axis
        assert np.allclose(F[0], -f * np.array([0.6, 0.0, 0.8]), rtol=1e-12) and np.allclose(F[1], -F[0], rtol=1e-12)


def test_one_term_screening_has_the_slope_expo_over_a():
    Z = np.array([4.0, 9.0])
    a = 0.9 / (4.0 ** 0.23 + 9.0 ** 0.23)
    r = np.array([0.5, 0.8, 1.3])
    ratio = []
    for x in r:
        E, _, _ = PC.pair_correction(_dimer(x), Z, 3.0, 3.5, [1.0], [1.7], 0.9, 0.23, KC)
        ratio.append(E[0] / (KC * 36.0 / x))
    slope = np.diff(np.log(ratio)) / np.diff(r)
    assert np.allclose(slope, -1.7 / a, rtol=1e-12)
    # same species on both sides: a = a_prefac / (2 Z^p)
    E, _, _ = PC.pair_correction(_dimer(0.8, types=(1, 1)), Z, 3.0, 3.5, [1.0], [1.7], 0.9, 0.23, KC)
    assert np.log(E[0] / (KC * 81.0 / 0.8)) == pytest.approx(-1.7 * 0.8 * 2 * 9.0 ** 0.23 / 0.9, rel=1e-12)


def test_switch_midpoint_quarter_and_outer_radius():
    Z = np.array([2.0, 7.0])
    args = ([0.6, 0.4], [0.9, 2.2], 0.8, 0.25, KC)
    ri, ro = 1.0, 2.0
    for r, want in ((1.5, 0.5), (1.25, 0.5 * (1 + np.cos(np.pi / 4))), (0.9, 1.0), (1.0, 1.0)):
        E, _, _ = PC.pair_correction(_dimer(r), Z, ri, ro, *args)
        E0, _, _ = PC.pair_correction(_dimer(r), Z, 2.9, 3.0, *args)             # the same pair well inside the inner radius: sw = 1
        assert E[0] / E0[0] == pytest.approx(want, rel=1e-13)
    # value and first derivative vanish at r_outer: E ~ delta^2 just inside, exactly 0 at and beyond
    e = [PC.pair_correction(_dimer(ro - d), Z, ri, ro, *args)[0][0] for d in (1e-3, 5e-4)]
    assert e[0] > 0 and e[0] / e[1] == pytest.approx(4.0, rel=5e-3)
    for r in (ro, ro + 0.3):
        E, F, W = PC.pair_correction(_dimer(r), Z, ri, ro, *args)
        assert abs(E[0]) < 1e-25 and np.abs(F).max() < 1e-12 and np.abs(W).max() < 1e-12    # |d| = r_outer up to one rounding


def _periodic_problem():
    w = wl.tiny_workload(21, n_species=2, sizes=(7, 3), box=(3.3, 2.6))          # thin boxes: several images, self-images
    w = dataclasses.replace(w, model=MODEL)
    return w


PARAMS = dict(Z=np.array([6.0, 11.0]), r_inner=1.2, r_outer=3.4, coef=[0.3, 0.5, 0.2], expo=[0.4, 1.1, 2.9], a_prefac=0.85, a_pow=0.23,
              coulomb_k=KC)


def _energy(st):
    return PC.pair_correction(O.OracleData(MODEL, st), **PARAMS)[0]


def test_forces_are_minus_the_gradient_and_sum_to_zero():
    st = _periodic_problem().structures
    E, F, W = PC.pair_correction(O.OracleData(MODEL, st), **PARAMS)
    assert E.min() > 0
    off = st.atom_off
    for s in range(st.n_struct):
        assert np.abs(F[off[s]:off[s + 1]].sum(axis=0)).max() < 1e-10 * np.abs(F).max()
    h = 1e-5
    rng = np.random.default_rng(0)
    for i in rng.choice(len(st.pos), size=5, replace=False):
        for k in range(3):
            p = st.pos.copy(); p[i, k] += h
            m = st.pos.copy(); m[i, k] -= h
            fd = -(_energy(dataclasses.replace(st, pos=p)).sum() - _energy(dataclasses.replace(st, pos=m)).sum()) / (2 * h)
            assert F[i, k] == pytest.approx(fd, rel=1e-6, abs=1e-7)


def test_virial_is_minus_the_strain_derivative():
    st = _periodic_problem().structures
    E, F, W = PC.pair_correction(O.OracleData(MODEL, st), **PARAMS)
    h = 1e-6
    off = st.atom_off
    for a in range(3):
        for b in range(3):
            def strained(sign):
                eps = np.eye(3); eps[a, b] += sign * h
                box = (st.box.reshape(-1, 3, 3) @ eps.T).reshape(-1, 9)          # x -> (1 + eps) x for cell vectors and positions
                return _energy(dataclasses.replace(st, pos=st.pos @ eps.T, box=box))
            dE = (strained(+1) - strained(-1)) / (2 * h)
            # W_ab = -sum d_a dE/dd_b = -dE/d eps_ab
            assert np.allclose(W[:, 3 * a + b], -dE, rtol=1e-6, atol=1e-6)
    assert np.allclose(W.reshape(-1, 3, 3), W.reshape(-1, 3, 3).transpose(0, 2, 1), atol=1e-12)      # central forces: symmetric


def test_correction_takes_no_model_parameter_and_vanishes_without_close_pairs():
    """The term has no theta in it (the function is not even given one), and a set whose shortest distance is beyond r_outer gets nothing."""
    import inspect
    assert "theta" not in inspect.signature(PC.pair_correction).parameters
    st = _periodic_problem().structures
    data = O.OracleData(MODEL, st)
    Ec, Fc, Wc = PC.pair_correction(data, **dict(PARAMS, r_inner=0.2, r_outer=0.9))     # the generator keeps atoms >= 1 A apart
    assert Ec.shape == (2,) and Fc.shape == (10, 3) and Wc.shape == (2, 9)
    assert not Ec.any() and not Fc.any() and not Wc.any()
