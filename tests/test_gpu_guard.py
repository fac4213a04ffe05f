"""Out-of-bounds writes: every device buffer the library gets is surrounded by guard bands (binding.Nep(guard_bytes=...));
after set-up, full steps (three calls and the graph), a mini-batch, a scaler computation and a label change the bands must be
untouched.  Stands in for `compute-sanitizer --tool memcheck`, which is closed on the GPU pool this repo is developed on."""
import numpy as np
import pytest

from paper_2606_19557_b200 import workloads as wl
from tests import _gpu_harness as H

pytestmark = pytest.mark.gpu

CASES = {
    "cfg1a": lambda: wl.make_config(1),
    "T5_ragged": lambda: wl.tiny_workload(21, n_species=5, sizes=(40, 37, 9, 1), box=(7.0, 6.5, 4.2, 2.9),
                                          model=wl.ModelSpec(5, 3.2, 2.6, 4, 4, 8, 8, 4, 2, 1, 30)),
    "cfg3": lambda: wl.make_config(3, n_struct=8),
    "cfg5_large_model": lambda: wl.make_config(5, n_struct=6, model=wl.config5_sweep()[-1]),     # FFMA network tiles
    "wide_T16": lambda: wl.tiny_workload(6, n_species=16, sizes=(40, 37), box=(7.0, 6.5), model=wl.ModelSpec(16, 3.2, 2.6, 3, 3, 4, 4, 4, 2, 1, 12)),
}


@pytest.mark.parametrize("name", list(CASES))
def test_no_write_outside_the_buffers(name):
    from paper_2606_19557_b200.binding import Nep
    prob = H.make_problem(CASES[name]())
    st = prob.workload.structures
    with Nep.from_model(prob.workload.model, guard_bytes=1024) as nep:
        nep.load_structure_set(st, prob.E, prob.F, prob.W)
        nep.build_neighbors()
        nep.set_params(prob.theta.astype(np.float32))
        nep.compute_scaler()
        nep.set_scaler(prob.scaler)
        H.check_forward(nep, prob)
        H.check_grad(nep, prob, (1.0, 2.0, 3.0))
        nep.adam_step(1e-3)
        for _ in range(3):
            nep.train_step(1.0, 1.0, 1.0, 1e-3, use_graph=True)
        if st.n_struct > 1:
            nep.set_batch(np.arange(st.n_struct, dtype=np.int32)[::-1][: st.n_struct - 1])
            nep.train_step(1.0, 1.0, 1.0, 1e-3, use_graph=False)
            nep.set_batch([])
            nep.train_step(1.0, 1.0, 1.0, 1e-3, use_graph=True)
        nep.set_labels(prob.E, prob.F, prob.W, np.zeros(st.n_struct, np.uint8))
        nep.set_batch(None)
        nep.forward(); nep.loss_grad(1.0, 1.0, 1.0)
        assert nep.check_guards() > 20
