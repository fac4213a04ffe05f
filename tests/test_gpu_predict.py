"""a trained model written to a file, read back into a new context, and prediction-only evaluation of
structures the model has never seen, against the oracle's forward pass with the same parameters and scaler."""
import numpy as np
import pytest

from oracle import nep_oracle as O
from paper_2606_19557_b200 import workloads as wl
from paper_2606_19557_b200.binding import Nep, NepError, NEP_EINVAL, NEP_ESTATE
from tests import _gpu_harness as H

pytestmark = pytest.mark.gpu

MODELS = {
    "nep4_T2": wl.ModelSpec(2, 3.4, 2.8, 3, 2, 4, 3, 4, 2, 1, 8),
    "l3_2_T3": wl.ModelSpec(3, 3.2, 2.6, 2, 2, 3, 3, 2, 2, 0, 6),
}


@pytest.mark.parametrize("name", list(MODELS))
def test_model_file_round_trip_and_prediction(name, tmp_path):
    model = MODELS[name]
    T = model.n_species
    train = H.make_problem(wl.tiny_workload(21, n_species=T, sizes=(20, 9, 33), box=(6.1, 4.4, 7.3), model=model))
    fresh = H.make_problem(wl.tiny_workload(22, n_species=T, sizes=(7, 41), box=(4.0, 7.9), model=model))   # other structures
    path = str(tmp_path / "model.txt")
    with H.make_gpu(train) as nep:
        for _ in range(3):                               # a few steps so that the file holds trained values, not the draw
            nep.train_step(1.0, 1.0, 1.0, 1e-2, use_graph=False)
        theta, scaler = nep.get_params(), nep.get_scaler()
        nep.save_model(path)
        hyper = nep.get_model()
    head = open(path).read().split("\n")[:7]
    assert head[0] == "nep_b200_model 1" and head[1] == f"n_species {T}" and head[5] == f"l_max {model.l_max_3b} {model.l_max_4b} {model.l_max_5b}"
    with Nep.from_model_file(path) as pred:
        assert pred.get_model() == hyper
        assert hyper["n_max_R"] == model.n_max_R and hyper["basis_A"] == model.basis_A and hyper["neurons"] == model.neurons
        assert pred.D == model.D and pred.n_par == model.n_par
        assert np.array_equal(pred.get_params(), theta)                     # fp32 values round-trip through 9 digits
        assert np.array_equal(pred.get_scaler().astype(np.float32), scaler.astype(np.float32))
        E, F, W = pred.predict(fresh.workload.structures)                    # no labels anywhere
        Eo, Fo, Wo = O.forward(fresh.data, theta.astype(np.float64), scaler.astype(np.float32).astype(np.float64))
        n = fresh.workload.structures.n_atoms.astype(np.float64)
        assert np.max(np.abs(E - Eo) / n) <= H.TOL_E_PER_ATOM
        assert H.relnorm(F, Fo) <= H.TOL_FW_REL and H.relnorm(W, Wo) <= H.TOL_FW_REL
        with pytest.raises(NepError) as e:                                   # a prediction context has no labels
            pred.loss_grad(1.0, 1.0, 1.0)
        assert e.value.code == NEP_ESTATE


def test_model_file_errors(tmp_path):
    bad = tmp_path / "bad.txt"
    bad.write_text("something else 1\n")
    with pytest.raises(NepError) as e:
        Nep.from_model_file(str(bad))
    assert e.value.code == NEP_EINVAL
    with pytest.raises(NepError):
        Nep.from_model_file(str(tmp_path / "missing.txt"))
    trunc = tmp_path / "trunc.txt"
    trunc.write_text("nep_b200_model 1\nn_species 1\ncutoff 3 2\nn_max 1 1\nbasis_size 2 2\nl_max 4 0 0\nneuron 2\nscaler 10\n1 1 1\n")
    with pytest.raises(NepError) as e:
        Nep.from_model_file(str(trunc))
    assert e.value.code == NEP_EINVAL
    with Nep.from_model(wl.ModelSpec(1, 3.0, 2.0, 1, 1, 2, 2, 4, 0, 0, 2)) as nep:     # nothing to save yet
        with pytest.raises(NepError) as e:
            nep.save_model(str(tmp_path / "x.txt"))
        assert e.value.code == NEP_ESTATE
