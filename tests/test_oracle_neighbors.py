"""Pins for C1 (neighbour lists): textbook shell counts, brute force with a wide fixed image range,
pair symmetry, canonical order, thin boxes with multi- and self-images."""
import os

import numpy as np

from oracle import nep_oracle as O
from paper_2606_19557_b200 import workloads as wl
from tests._ref_np import np_neighbors

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _one(pos, cell, types=None):
    pos = np.asarray(pos, float)
    return wl.StructureSet(np.array([len(pos)], np.int32), wl._wrap(pos, cell), np.asarray(cell, float).reshape(1, 9),
                           np.zeros(len(pos), np.int32) if types is None else types, ["x"])


def test_ideal_lattice_shell_counts():
    with open(os.path.join(GOLD, "lattice_shell_counts.txt")) as f:
        rows = [l.split() for l in f if l.strip() and not l.startswith("#")]
    for lat, a, rc, cnt in rows:
        pos, cell = wl._lattice(lat, float(a), (4, 4, 4))
        off, j, sh = O.build_neighbors(_one(pos, cell), float(rc))
        assert (np.diff(off) == int(cnt)).all(), (lat, a, rc)


def test_primitive_cell_single_atom_self_images():
    # one atom in an fcc primitive cell: all 42 neighbours within 5.0 are images of the atom itself
    pos, cell = wl._lattice("fcc_prim", 3.6, (1, 1, 1))
    off, j, sh = O.build_neighbors(_one(pos, cell), 5.0)
    assert off[-1] == 42 and (j == 0).all() and not (sh == 0).all(axis=1).any()


def test_against_wide_brute_force_and_order():
    w = wl.tiny_workload(3, sizes=(6, 4), box=(3.1, 5.0))
    st = w.structures
    for rc in (w.model.rc_R, w.model.rc_A):
        off, j, sh = O.build_neighbors(st, rc)
        ao = st.atom_off
        for s in range(st.n_struct):
            ref = np_neighbors(st.pos[ao[s]:ao[s + 1]], st.box[s], rc, wide=5)
            ref_set = sorted((i, jj, sft) for i, jj, sft, _ in ref)
            got = []
            for i in range(ao[s], ao[s + 1]):
                lst = [(int(j[p]), tuple(int(v) for v in sh[p])) for p in range(off[i], off[i + 1])]
                assert lst == sorted(lst)                      # canonical (j, na, nb, nc) order
                assert len(set(lst)) == len(lst)
                got += [(i - ao[s], jj, sft) for jj, sft in lst]
            assert sorted(got) == ref_set
            gs = set(got)
            for i, jj, sft in got:                             # (i->j, n) present <=> (j->i, -n) present
                assert (jj, i, tuple(-v for v in sft)) in gs


def test_angular_list_is_subset_of_radial():
    w = wl.tiny_workload(4)
    d = O.OracleData(w.model, w.structures)
    for i in range(d.n_atoms_total):
        R = {(int(d.jR[p]), tuple(d.shR[p])) for p in range(d.offR[i], d.offR[i + 1])}
        A = {(int(d.jA[p]), tuple(d.shA[p])) for p in range(d.offA[i], d.offA[i + 1])}
        assert A <= R


def test_image_range_covers_cutoff():
    rng = np.random.default_rng(5)
    for _ in range(20):
        cell = np.eye(3) * rng.uniform(2.0, 9.0, size=3) + rng.normal(scale=0.5, size=(3, 3))
        if np.linalg.det(cell) < 0:
            cell[0] *= -1
        m = O.image_range(cell, 6.0)
        V = abs(np.linalg.det(cell))
        for k in range(3):
            h = V / np.linalg.norm(np.cross(cell[(k + 1) % 3], cell[(k + 2) % 3]))
            assert m[k] >= np.ceil(6.0 / h)


def test_empty_structure_set_and_isolated_atom():
    pos = np.array([[1.0, 1.0, 1.0]])
    off, j, sh = O.build_neighbors(_one(pos, np.eye(3) * 20.0), 5.0)
    assert off[-1] == 0 and len(j) == 0
