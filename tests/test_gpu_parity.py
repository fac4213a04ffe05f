"""GPU parity: libnep_b200 (through the C ABI binding) against the fp64 oracle, element by element, on the same
seeded inputs.  Tolerances are BASELINE.json's: neighbour lists bit-exact; E <= 1e-5 eV/atom; F, W <= 1e-4 relative in
norm; gradient <= 1e-3 relative in norm.  Sizes: several 32-atom slices plus ragged tails, multi-image boxes."""
import numpy as np
import pytest

from oracle import nep_oracle as O
from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H

pytestmark = pytest.mark.gpu


def _cases():
    m5 = wl.config5_sweep()
    return {
        "tiny_T2": lambda: wl.tiny_workload(0),
        "tiny_T1": lambda: wl.tiny_workload(1, n_species=1, sizes=(3, 9, 1), box=(3.0, 4.0, 2.9)),
        "tiny_T3_ragged": lambda: wl.tiny_workload(2, n_species=3, sizes=(33, 2, 40), box=(7.5, 3.1, 8.0)),
        "tiny_thin_boxes": lambda: wl.tiny_workload(7, n_species=2, sizes=(1, 2, 3), box=(1.6, 2.2, 2.0)),   # images up to +-2
        "tiny_3body_only": lambda: wl.tiny_workload(3, model=wl.ModelSpec(2, 3.2, 2.6, 2, 0, 3, 1, 4, 0, 0, 5)),
        "tiny_4body_only": lambda: wl.tiny_workload(4, model=wl.ModelSpec(2, 3.2, 3.2, 0, 2, 1, 3, 4, 2, 0, 3)),
        "tiny_5body_only": lambda: wl.tiny_workload(5, model=wl.ModelSpec(2, 3.0, 2.0, 1, 1, 2, 2, 4, 0, 1, 9)),
        # other three-body orders: l_max_3b = 1, 2, 3 with and without the 4-/5-body terms
        "tiny_l3_1_5body": lambda: wl.tiny_workload(8, model=wl.ModelSpec(2, 3.2, 2.6, 2, 2, 3, 3, 1, 0, 1, 5)),
        "tiny_l3_2_4body": lambda: wl.tiny_workload(9, model=wl.ModelSpec(2, 3.2, 2.8, 1, 3, 2, 4, 2, 2, 0, 6)),
        "tiny_l3_3_full": lambda: wl.tiny_workload(10, n_species=3, sizes=(33, 2, 40), box=(7.5, 3.1, 8.0),
                                                   model=wl.ModelSpec(3, 3.2, 2.6, 2, 5, 3, 4, 3, 2, 1, 7)),
        # the largest basis (17 functions: the K = 17 instantiations) with 6 angular channels (two chunks of 3), one and two species
        "tiny_K17_T1": lambda: wl.tiny_workload(11, n_species=1, sizes=(35, 6), box=(7.2, 4.1),
                                                model=wl.ModelSpec(1, 3.3, 2.9, 3, 5, 16, 16, 4, 2, 1, 6)),
        "tiny_K17_T2": lambda: wl.tiny_workload(12, n_species=2, sizes=(12, 38), box=(4.4, 7.4),
                                                model=wl.ModelSpec(2, 3.3, 2.9, 2, 5, 12, 16, 4, 2, 1, 5)),
        "cfg1a": lambda: wl.make_config(1),
        "cfg1b": lambda: wl.make_config(1, n_struct=2, variant="1b"),
        "cfg2": lambda: wl.make_config(2, n_struct=6),
        "cfg3": lambda: wl.make_config(3, n_struct=8),
        "cfg4": lambda: wl.make_config(4, n_struct=12),
        "cfg5_small_model": lambda: wl.make_config(5, n_struct=8),
        "cfg5_large_model": lambda: wl.make_config(5, n_struct=8, model=m5[-1]),      # n_max 8, basis 12, 100 neurons
        "cfg5_mixed_model": lambda: wl.make_config(5, n_struct=6, model=m5[5]),       # n_max 8, basis 8, 100 neurons
        # the other five models of config 5's sweep (index = 4 [n_max 8] + 2 [basis 12] + 1 [100 neurons]); models 4 and 6 have D = 63:
        # eight K steps per tcgen05 product, accumulator width 112 / 128
        "cfg5_model1": lambda: wl.make_config(5, n_struct=6, model=m5[1]),
        "cfg5_model2": lambda: wl.make_config(5, n_struct=6, model=m5[2]),
        "cfg5_model3": lambda: wl.make_config(5, n_struct=6, model=m5[3]),
        "cfg5_model4": lambda: wl.make_config(5, n_struct=6, model=m5[4]),
        "cfg5_model6": lambda: wl.make_config(5, n_struct=6, model=m5[6]),
        # the widest network tiles that fit the tensor-core kernels, on ragged slices: D = 63 with three species; D = 125 (n_max 10 / 18:
        # 19 angular channels) with 24 neurons; 128 neurons with D = 21; 100 neurons with two species (see TC_CASES below)
        "tiny_D63_H40_T3": lambda: wl.tiny_workload(13, n_species=3, sizes=(33, 2, 40), box=(7.5, 3.1, 8.0),
                                                    model=wl.ModelSpec(3, 3.2, 2.6, 8, 8, 4, 4, 4, 2, 1, 40)),
        "tiny_D125_H24_T2": lambda: wl.tiny_workload(14, n_species=2, sizes=(35, 44), box=(7.2, 7.6),
                                                     model=wl.ModelSpec(2, 3.3, 2.9, 10, 18, 4, 4, 4, 2, 1, 24)),
        "tiny_D21_H128_T1": lambda: wl.tiny_workload(15, n_species=1, sizes=(37, 5), box=(7.3, 3.6),
                                                     model=wl.ModelSpec(1, 3.2, 2.6, 2, 2, 4, 4, 4, 2, 1, 128)),
        "tiny_D35_H100_T2": lambda: wl.tiny_workload(16, n_species=2, sizes=(6, 41), box=(3.9, 7.5),
                                                     model=wl.ModelSpec(2, 3.2, 2.6, 4, 4, 8, 8, 4, 2, 1, 100)),
        "wide_T16": lambda: wl.tiny_workload(6, n_species=16, sizes=(40, 37), box=(7.0, 6.5),
                                             model=wl.ModelSpec(16, 3.2, 2.6, 3, 3, 4, 4, 4, 2, 1, 12)),
    }


CASES = _cases()
_cache = {}
# cases whose network products must run on the tensor cores (nep_network_on_tensor_cores): a parity case that silently fell back
# to the FFMA tiles would say nothing about the tcgen05 kernels
TC_CASES = ["cfg2", "cfg3", "cfg4", "cfg5_small_model", "cfg5_model2", "cfg5_model4", "cfg5_model6", "tiny_D63_H40_T3", "tiny_D125_H24_T2",
            "tiny_D21_H128_T1", "tiny_D35_H100_T2", "tiny_K17_T1"]


def _prob(name):
    if name not in _cache:
        _cache[name] = H.make_problem(CASES[name]())
    return _cache[name]


@pytest.mark.parametrize("name", list(CASES))
def test_neighbor_lists_bit_exact(name):
    prob = _prob(name)
    with H.make_gpu(prob, labels=False, scaler=None) as nep:
        H.check_neighbors(nep, prob.data)
        s = nep.get_sizes()
        assert s["P_R"] == len(prob.data.jR) and s["P_A"] == len(prob.data.jA) and s["N"] == prob.data.n_atoms_total


@pytest.mark.parametrize("name", TC_CASES)
def test_case_runs_on_the_tensor_core_network_kernels(name):
    from paper_2606_19557_b200.binding import Nep
    with Nep.from_model(CASES[name]().model) as nep:
        assert nep.network_on_tensor_cores(), name


@pytest.mark.parametrize("name", list(CASES))
def test_descriptors(name):
    prob = _prob(name)
    q_o = O.descriptors(prob.data, prob.theta)
    with H.make_gpu(prob) as nep:
        nep.forward(want=())
        q = nep.get_descriptors()
    # compare in scaled units (q~ = s q is what the network sees): absolute error per component of O(1) ranges
    err = np.max(np.abs((q - q_o) * prob.scaler))
    assert err < 2e-5, err


@pytest.mark.parametrize("name", list(CASES))
def test_forward_energy_force_virial(name):
    prob = _prob(name)
    with H.make_gpu(prob) as nep:
        H.check_forward(nep, prob)
        # running it twice gives the same answer up to the order of atomic additions (state is reset every call)
        E1, F1, W1 = nep.forward()
        E2, F2, W2 = nep.forward()
        assert np.allclose(E1, E2, rtol=0, atol=1e-5 * prob.workload.structures.n_atoms.max())
        assert H.relnorm(F1, F2) < 1e-5 and H.relnorm(W1, W2) < 1e-5


@pytest.mark.parametrize("name", list(CASES))
def test_loss_and_gradient(name):
    prob = _prob(name)
    with H.make_gpu(prob) as nep:
        eg, errs, g, go = H.check_grad(nep, prob, prob.workload.lambdas, per_block_tol=2e-3)


@pytest.mark.parametrize("lam", [(1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0)])
@pytest.mark.parametrize("name", ["tiny_T2", "cfg3"])
def test_gradient_single_terms(name, lam):
    prob = _prob(name)
    with H.make_gpu(prob) as nep:
        H.check_grad(nep, prob, lam, per_block_tol=2e-3)


@pytest.mark.parametrize("name", ["tiny_T3_ragged", "cfg3", "cfg4"])
def test_mini_batches(name):
    """A batch is a list of structure ids in any order; outputs come back in batch order."""
    prob = _prob(name)
    S = prob.workload.structures.n_struct
    rng = np.random.default_rng(7)
    with H.make_gpu(prob) as nep:
        for ids in (rng.permutation(S)[: max(1, S // 2)], [S - 1], rng.permutation(S)):
            nep.set_batch(ids)
            H.check_forward(nep, prob, batch=ids)
            H.check_grad(nep, prob, (1.0, 1.0, 1.0), batch=ids)
        nep.set_batch(None)
        H.check_forward(nep, prob)


def test_same_batch_selected_again():
    """nep_set_batch with the ids of the current batch re-uploads the tables but keeps the derived device tables: results, the reset of
    the whole-batch normalisers and the step graph behave as after any nep_set_batch."""
    prob = _prob("cfg3")
    S = prob.workload.structures.n_struct
    ids = np.random.default_rng(3).permutation(S)[: S - 2]
    lam = (1.0, 2.0, 3.0)
    l4o, go = O.loss_grad(prob.data, prob.theta, prob.scaler, lam, batch=list(ids))
    with H.make_gpu(prob) as nep:
        nep.set_batch(ids)
        nep.set_batch(ids)                                   # fast path
        H.check_forward(nep, prob, batch=ids)
        H.check_grad(nep, prob, lam, batch=ids)
        nat = prob.workload.structures.n_atoms
        nep.set_batch_normalisers(2 * len(ids), 2 * int(nat[ids].sum()), 2 * len(ids))
        nep.forward(want=())
        half = nep.loss_grad(*lam)
        assert np.allclose(half, 0.5 * l4o, rtol=2e-4)       # counts of a batch twice as large: every mean halves
        nep.set_batch(ids)                                   # the local counts again
        nep.forward(want=())
        assert np.allclose(nep.loss_grad(*lam), l4o, rtol=2e-4)
        nep.set_batch(ids[::-1].copy())                      # another order is another batch
        H.check_forward(nep, prob, batch=ids[::-1])
        th0 = nep.get_params()
        for _ in range(3):                                   # stepping through the graph with the batch re-selected every step
            nep.set_batch(ids)
            nep.train_step(*lam, 1e-3, use_graph=True)
        th_a = nep.get_params()
        nep.set_params(th0); nep.set_adam_state(np.zeros_like(th0), np.zeros_like(th0), np.zeros_like(th0), 0)
        nep.set_batch(ids)
        for _ in range(3):
            nep.train_step(*lam, 1e-3, use_graph=False)
        th_b = nep.get_params()
        assert np.linalg.norm(th_a - th_b) <= 1e-3 * np.linalg.norm(th_a - th0)     # same trajectory up to the order of atomic sums


def _two_species_equal_shape_problem():
    """Four 128-atom bcc cells (config 2's recipe) with two species: structures 0, 1 hold 100 + 28 atoms of species 0 / 1, structures
    2, 3 hold 28 + 100.  The batches [0, 1] and [2, 3] agree in every count the launch shapes depend on (structures, atoms, slices,
    network tiles) and differ only in where the tiles of species 1 start."""
    w = wl.make_config(2, n_struct=4, model=wl.ModelSpec(2, 6.0, 4.0, 4, 4, 8, 8, 4, 2, 1, 30))
    ty = w.structures.type.reshape(4, 128)
    ty[:2, 100:] = 1
    ty[2:, 28:] = 1
    return H.make_problem(w)


def test_step_graph_over_equal_shape_batches_of_different_composition():
    """A captured step graph carries the first network tile of every species by value.  Two mini-batches of the same shape with other
    atoms per species must not replay each other's graph: the graph path lands on the parameters of the three-call path."""
    prob = _two_species_equal_shape_problem()
    lam = (1.0, 1.0, 1.0)
    A, B = np.array([0, 1], np.int32), np.array([2, 3], np.int32)
    th = {}
    for use_graph in (True, False):
        with H.make_gpu(prob) as nep:
            th0 = nep.get_params()
            for ids in (A, A, A, B, B, B, A, B):        # the third step on a batch replays the graph captured at the second
                nep.set_batch(ids)
                nep.train_step(*lam, 1e-3, use_graph=use_graph)
            th[use_graph] = nep.get_params()
    assert np.linalg.norm(th[True] - th[False]) <= 1e-3 * np.linalg.norm(th[False] - th0)


def test_step_graph_after_a_second_neighbour_build():
    """nep_build_neighbors releases and re-allocates the lists, the pair cache and the slot tables: a step graph captured before it
    points at freed buffers and has to be captured again (include/nep.h, nep_train_step)."""
    prob = _prob("tiny_T3_ragged")
    lam = (1.0, 2.0, 3.0)
    th = {}
    for use_graph in (True, False):
        with H.make_gpu(prob) as nep:
            th0 = nep.get_params()
            for _ in range(3):
                nep.train_step(*lam, 1e-3, use_graph=use_graph)
            junk = [nep._torch.empty(1 << 20, dtype=nep._torch.uint8, device="cuda") for _ in range(8)]   # noqa: F841  other addresses next time
            nep.build_neighbors()
            for _ in range(3):
                nep.train_step(*lam, 1e-3, use_graph=use_graph)
            th[use_graph] = nep.get_params()
    assert np.linalg.norm(th[True] - th[False]) <= 1e-3 * np.linalg.norm(th[False] - th0)


def test_empty_batch_and_state_errors():
    from paper_2606_19557_b200.binding import NepError, NEP_ESTATE, NEP_EINVAL
    prob = _prob("tiny_T2")
    with H.make_gpu(prob) as nep:
        nep.set_batch([])
        E, F, W = nep.forward()
        assert E.shape == (0,) and F.shape == (0, 3) and W.shape == (0, 9)
        l4 = nep.loss_grad(1.0, 1.0, 1.0)
        assert np.all(l4 == 0.0) and np.all(nep.get_grad() == 0.0)
        nep.set_batch(None)
        with pytest.raises(NepError) as e:
            nep.loss_grad(1.0, 1.0, 1.0)           # forward must come first
        assert e.value.code == NEP_ESTATE
        with pytest.raises(NepError) as e:
            nep.set_batch([0, 0])
        assert e.value.code == NEP_EINVAL
        with pytest.raises(NepError) as e:
            nep.set_batch([5])
        assert e.value.code == NEP_EINVAL
        nep.forward(want=())
        nep.loss_grad(1.0, 1.0, 1.0)
        nep.adam_step(1e-3)
        with pytest.raises(NepError) as e:
            nep.adam_step(1e-3)                    # gradient consumed
        assert e.value.code == NEP_ESTATE


def test_load_rejects_bad_input():
    from paper_2606_19557_b200.binding import Nep, NepError, NEP_EINVAL
    w = wl.tiny_workload(0)
    st = w.structures
    with Nep.from_model(w.model) as nep:
        bad = st.pos.copy(); bad[0, 0] = np.nan
        with pytest.raises(NepError) as e:
            nep.load_structures(st.n_atoms, bad, st.box, st.type)
        assert e.value.code == NEP_EINVAL
        bad = st.pos.copy(); bad[0] += st.box[0].reshape(3, 3)[0] * 1.5      # outside the cell
        with pytest.raises(NepError):
            nep.load_structures(st.n_atoms, bad, st.box, st.type)
        badt = st.type.copy(); badt[1] = w.model.n_species
        with pytest.raises(NepError):
            nep.load_structures(st.n_atoms, st.pos, st.box, badt)
        badb = st.box.copy(); badb[0, :3] *= -1
        with pytest.raises(NepError):
            nep.load_structures(st.n_atoms, st.pos, badb, st.type)
        nep.load_structures(st.n_atoms, st.pos, st.box, st.type)           # still usable afterwards
        nep.build_neighbors()


def test_rejected_labels_leave_the_old_ones_in_place():
    """nep_set_labels validates before it releases anything: after a rejected call (NaN label) the previous labels still
    serve nep_loss_grad, with the values they had."""
    from paper_2606_19557_b200.binding import NepError, NEP_EINVAL
    prob = _prob("tiny_T2")
    with H.make_gpu(prob) as nep:
        nep.forward(want=())
        l4 = nep.loss_grad(1.0, 2.0, 3.0)
        for which in range(3):
            E, F, W = prob.E.copy(), prob.F.copy(), prob.W.copy()
            (E, F, W)[which].flat[0] = np.nan if which != 1 else np.inf
            with pytest.raises(NepError) as e:
                nep.set_labels(E, F, W)
            assert e.value.code == NEP_EINVAL
        nep.forward(want=())
        assert np.array_equal(nep.loss_grad(1.0, 2.0, 3.0), l4)


def test_null_allocator_is_refused():
    """include/nep.h: the library never calls cudaMalloc; a context without allocator callbacks is NEP_EINVAL."""
    import ctypes
    from paper_2606_19557_b200 import binding
    L = binding.load_library()
    h = ctypes.c_void_p(None)
    rc = L.nep_create(ctypes.byref(h), 1, 5.0, 4.0, 4, 4, 8, 8, 4, 2, 1, 30, ctypes.cast(None, binding.ALLOC_FN),
                      ctypes.cast(None, binding.FREE_FN), None, None)
    assert rc == binding.NEP_EINVAL and b"alloc" in L.nep_last_error(None) and not h.value


def test_virial_mask():
    prob = _prob("tiny_T3_ragged")
    hv = np.array([1, 0, 1], np.uint8)
    prob.data.set_labels(prob.E, prob.F, prob.W, has_virial=hv)
    try:
        with H.make_gpu(prob) as nep:
            nep.set_labels(prob.E, prob.F, prob.W, hv)
            H.check_grad(nep, prob, (1.0, 2.0, 3.0), per_block_tol=2e-3)
            nep.set_labels(prob.E, prob.F, prob.W, np.zeros(3, np.uint8))      # no virial labels at all: dV = 0
            prob.data.set_labels(prob.E, prob.F, prob.W, has_virial=np.zeros(3, np.uint8))
            _, _, g, go = H.check_grad(nep, prob, (1.0, 2.0, 3.0))
    finally:
        prob.data.set_labels(prob.E, prob.F, prob.W)


@pytest.mark.parametrize("name", ["tiny_T2", "cfg1a", "cfg4"])
def test_compute_scaler_matches_definition(name):
    """Eq. 2: s = 1 / (max - min) over every loaded atom; the oracle's scaler is that definition in fp64."""
    prob = _prob(name)
    with H.make_gpu(prob, scaler="compute") as nep:
        s = nep.get_scaler()
    assert np.allclose(s, prob.scaler, rtol=2e-5), np.max(np.abs(s / prob.scaler - 1))


def test_compute_scaler_small_descriptors():
    """Eq. 2 on components that are small but well resolved: with the angular coefficients scaled by 0.05 the 4-/5-body invariants
    have ranges of 1e-6 ... 2e-8 (below 64 eps_fp32, where an absolute threshold would return 1) and the oracle's 1 / range holds."""
    prob = _prob("tiny_T3_ragged")
    th = prob.theta.copy()
    th[prob.workload.model.block_slices()["cA"]] *= 0.05
    th = th.astype(np.float32).astype(np.float64)
    q = O.descriptors(prob.data, th)
    rng = q.max(axis=0) - q.min(axis=0)
    assert rng.min() > 1e-8 and np.sum(rng < 64 * 1.2e-7) >= 4
    with H.make_gpu(prob, labels=False, scaler=None) as nep:
        nep.set_params(th.astype(np.float32))
        nep.compute_scaler()
        s = nep.get_scaler()
    assert np.allclose(s, O.scaler(q), rtol=1e-4), np.max(np.abs(s / O.scaler(q) - 1))


def test_scaler_of_a_perfect_lattice():
    """Reading G10: a component that is the same for every atom has no range and gets s = 1.  On a perfect lattice every
    component is constant; in fp32 its "range" is summation noise (~1e-7 |q|), which must not be inverted into s ~ 1e7."""
    pos, cell = wl._lattice("bcc", 3.16, (4, 4, 4))
    st = wl.StructureSet(np.array([len(pos)], np.int32), wl._wrap(pos, cell), cell.reshape(1, 9), np.zeros(len(pos), np.int32), ["bcc"])
    w = wl.make_config(2, n_struct=1)
    import dataclasses
    w = dataclasses.replace(w, structures=st)
    from paper_2606_19557_b200.binding import Nep
    th = wl.ParamDraw(w.model, w.seeds["student"]).coefficients()
    q = O.descriptors(O.OracleData(w.model, st), th)
    assert np.array_equal(O.scaler(q), np.ones(w.model.D))               # the oracle: every range is below 1e-12 max(1, |q|)
    with Nep.from_model(w.model) as nep:
        nep.load_structure_set(st)
        nep.build_neighbors()
        nep.set_params(th.astype(np.float32))
        nep.compute_scaler()
        assert np.array_equal(nep.get_scaler(), np.ones(w.model.D))
        lo, hi = nep.compute_descriptor_range()
        assert np.all(hi - lo <= 1e-5 * np.maximum(1.0, np.abs(hi)))     # fp32 noise only
        assert np.allclose(0.5 * (lo + hi), q.mean(0), rtol=1e-5, atol=1e-6)


def test_descriptor_range_of_two_contexts_gives_the_scaler_of_the_union():
    """Eq. 2 is over every atom of the set.  Two contexts hold different structures: their ranges, reduced element-wise
    (the MIN / MAX all-reduce of dataparallel.DataParallelNep.compute_scaler), give each of them the scaler that one context
    holding everything computes, which is the oracle's."""
    from paper_2606_19557_b200 import dataparallel as dp
    from paper_2606_19557_b200.binding import Nep
    prob = _prob("cfg3")
    w = prob.workload; st = w.structures
    s_union = O.scaler(O.descriptors(prob.data, prob.theta))
    los, his, ctxs = [], [], []
    try:
        for rank in range(2):
            ids = dp.Shard.make(st.n_atoms, rank, 2).global_ids
            nep = Nep.from_model(w.model)
            ctxs.append(nep)
            nep.load_structure_set(st.subset(ids))
            nep.build_neighbors()
            nep.set_params(prob.theta.astype(np.float32))
            lo, hi = nep.compute_descriptor_range()
            los.append(lo); his.append(hi)
        assert not np.allclose(los[0], los[1]) and not np.allclose(his[0], his[1])
        lo, hi = np.minimum(*los), np.maximum(*his)
        for nep in ctxs:
            nep.set_scaler_from_range(lo, hi)
        s0, s1 = ctxs[0].get_scaler(), ctxs[1].get_scaler()
        assert np.array_equal(s0, s1)
        assert np.allclose(s0, s_union, rtol=2e-5), np.max(np.abs(s0 / s_union - 1))
        with H.make_gpu(prob, labels=False, scaler="compute") as whole:
            assert np.allclose(s0, whole.get_scaler(), rtol=1e-6)
        # an empty context reports the neutral elements and takes the reduced range like every other
        with Nep.from_model(w.model) as empty:
            empty.load_structure_set(st.subset([]))
            empty.build_neighbors()
            empty.set_params(prob.theta.astype(np.float32))
            elo, ehi = empty.compute_descriptor_range()
            assert np.all(np.isposinf(elo)) and np.all(np.isneginf(ehi))
            empty.set_scaler_from_range(lo, hi)
            assert np.array_equal(empty.get_scaler(), s0)
    finally:
        for nep in ctxs:
            nep.destroy()


@pytest.mark.parametrize("variant", [0, 1])
def test_adam_same_gradient_both_sides(variant):
    """Eqs. 9-13: three steps with the SAME gradients fed to both sides; theta within fp32 rounding."""
    prob = _prob("cfg1a")
    rng = np.random.default_rng(3)
    n = prob.workload.model.n_par
    th = prob.theta.copy(); m = np.zeros(n); v = np.zeros(n); vm = np.zeros(n); t = 0
    with H.make_gpu(prob) as nep:
        for _ in range(3):
            g = (rng.normal(size=n) * 10.0 ** rng.uniform(-4, 1, size=n)).astype(np.float32)
            t = O.adam_step(th, g.astype(np.float64), m, v, vm, t, 1e-2, 0.9, 0.999, 1e-8, variant)
            nep.set_grad(g)
            nep.adam_step(1e-2, 0.9, 0.999, 1e-8, variant)
        gth = nep.get_params()
        gm, gv, gvm, gt = nep.get_adam_state()
    assert gt == t == 3
    assert np.max(np.abs(gth - th)) <= 1e-6 * max(1.0, np.max(np.abs(th)))
    assert np.allclose(gm, m, rtol=1e-5, atol=1e-12) and np.allclose(gv, v, rtol=1e-5, atol=1e-20)
    assert np.allclose(gvm, vm, rtol=1e-5, atol=1e-20)


def test_full_training_steps_track_the_oracle():
    """Five full steps (forward, loss+grad, Adam) on both sides from the same start: loss trajectories agree."""
    prob = _prob("cfg1a")
    n = prob.workload.model.n_par
    lam = (1.0, 1.0, 1.0)
    th = prob.theta.copy(); m = np.zeros(n); v = np.zeros(n); vm = np.zeros(n); t = 0
    Lo, Lg = [], []
    with H.make_gpu(prob) as nep:
        for _ in range(5):
            l4o, go = O.loss_grad(prob.data, th, prob.scaler, lam)
            t = O.adam_step(th, go, m, v, vm, t, 1e-3)
            Lo.append(l4o[0])
            nep.forward(want=())
            Lg.append(nep.loss_grad(*lam)[0])
            nep.adam_step(1e-3)
        thg = nep.get_params()
    assert np.allclose(Lg, Lo, rtol=1e-3), (Lg, Lo)
    assert Lo[-1] < Lo[0]
    assert H.relnorm(thg, th) < 1e-4


@pytest.mark.parametrize("name", ["cfg1a", "cfg3"])
def test_train_step_graph_matches_the_three_calls(name):
    """nep_train_step (one CUDA graph launch per step, loss weights / learning rate / bias corrections re-written into its nodes)
    against nep_forward + nep_loss_grad + nep_adam_step: same parameters and loss terms, across a change of the loss weights
    and of the learning rate, a new batch (graph captured again) and both Adam variants; the first step also against the oracle."""
    prob = _prob(name)
    S = prob.workload.structures.n_struct
    sched = [((1.0, 1.0, 1.0), 1e-3, 0), ((1.0, 1.0, 1.0), 1e-3, 0), ((2.0, 0.5, 3.0), 5e-4, 0), ((2.0, 0.5, 3.0), 2e-4, 0)]
    with H.make_gpu(prob) as ref, H.make_gpu(prob) as gr, H.make_gpu(prob) as st:
        def run(batch, sched, check_oracle=False):
            for nep in (ref, gr, st):
                nep.set_batch(batch)
            for i, (lam, lr, variant) in enumerate(sched):
                ref.forward_device(); ref.loss_grad(*lam, fetch_loss=False); ref.adam_step(lr, variant=variant)
                gr.train_step(*lam, lr, variant=variant, use_graph=True)
                st.train_step(*lam, lr, variant=variant, use_graph=False)
                l_ref, l_gr, l_st = ref.get_loss(), gr.get_loss(), st.get_loss()
                assert np.allclose(l_gr, l_ref, rtol=1e-5, atol=1e-14) and np.allclose(l_st, l_ref, rtol=1e-5, atol=1e-14)
                th_ref, th_gr, th_st = ref.get_params(), gr.get_params(), st.get_params()
                scale = max(1.0, float(np.max(np.abs(th_ref))))
                assert np.max(np.abs(th_gr - th_ref)) <= 2e-6 * scale and np.max(np.abs(th_st - th_ref)) <= 2e-6 * scale
                if check_oracle and i == 0:
                    l4o, go = O.loss_grad(prob.data, prob.theta, prob.scaler, lam, batch=None if batch is None else list(batch))
                    th = prob.theta.copy(); n = th.size
                    O.adam_step(th, go, np.zeros(n), np.zeros(n), np.zeros(n), 0, lr)
                    assert np.allclose(l_gr, l4o, rtol=2e-4) and np.max(np.abs(th_gr - th)) < 1e-5
        run(None, sched, check_oracle=True)
        sub = np.arange(S, dtype=np.int32)[::2]
        run(sub, sched[:2])                                   # new batch: the step is captured again
        run(sub, [((1.0, 1.0, 1.0), 1e-3, 1)] * 2)            # other Adam variant: other kernel, captured again
        assert gr.get_adam_state()[3] == ref.get_adam_state()[3] == st.get_adam_state()[3]
        assert gr.launch_count() == ref.launch_count()        # a replayed graph counts the kernels it launches
