"""Shared set-up of the GPU parity tests: one oracle Problem -> one libnep_b200 context fed the same inputs."""
import numpy as np

from oracle import nep_oracle as O
from oracle.problem import make_problem  # noqa: F401  (re-exported)

# tolerances of BASELINE.json's north_star
TOL_E_PER_ATOM = 1e-5    # eV/atom, absolute
TOL_FW_REL = 1e-4        # forces, virials: relative in norm
TOL_G_REL = 1e-3         # parameter gradient: relative in norm (fp32)


def make_gpu(prob, labels=True, scaler="oracle"):
    from paper_2606_19557_b200.binding import Nep
    st = prob.workload.structures
    nep = Nep.from_model(prob.workload.model)
    if labels:
        nep.load_structure_set(st, prob.E, prob.F, prob.W)
    else:
        nep.load_structure_set(st)
    nep.build_neighbors()
    nep.set_params(prob.theta.astype(np.float32))
    if scaler == "oracle":
        nep.set_scaler(prob.scaler)
    elif scaler == "compute":
        nep.compute_scaler()
    return nep


def relnorm(a, b):
    a = np.asarray(a, np.float64).ravel(); b = np.asarray(b, np.float64).ravel()
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a - b)


def check_neighbors(nep, data):
    for which, (off, j, sh) in enumerate(((data.offR, data.jR, data.shR), (data.offA, data.jA, data.shA))):
        goff, gj, gsh = nep.get_neighbors(which)
        assert np.array_equal(goff, off), f"list {which}: offsets differ"
        assert np.array_equal(gj, j), f"list {which}: neighbour indices differ"
        assert np.array_equal(gsh, sh), f"list {which}: image shifts differ"


def check_forward(nep, prob, batch=None):
    """E per atom abs, F and W relative norm over the batch.  Returns the errors."""
    st = prob.workload.structures
    ids = np.arange(st.n_struct) if batch is None else np.asarray(batch)
    Eo, Fo, Wo = O.forward(prob.data, prob.theta, prob.scaler, batch=None if batch is None else list(batch))
    E, F, W = nep.forward()
    n = st.n_atoms[ids].astype(np.float64)
    eE = np.max(np.abs(E - Eo) / n) if len(ids) else 0.0
    eF, eW = relnorm(F, Fo), relnorm(W, Wo)
    assert eE <= TOL_E_PER_ATOM, f"energy error {eE:.3e} eV/atom"
    assert eF <= TOL_FW_REL, f"force error {eF:.3e}"
    assert eW <= TOL_FW_REL, f"virial error {eW:.3e}"
    return eE, eF, eW


def check_grad(nep, prob, lambdas, batch=None, per_block_tol=None):
    l4o, go = O.loss_grad(prob.data, prob.theta, prob.scaler, lambdas, batch=None if batch is None else list(batch))
    nep.forward(want=())
    l4 = nep.loss_grad(*lambdas)
    g = nep.get_grad()
    assert np.allclose(l4, l4o, rtol=2e-4, atol=1e-12), f"loss {l4} vs {l4o}"
    eg = relnorm(g, go)
    assert eg <= TOL_G_REL, f"gradient error {eg:.3e}"
    sl = prob.workload.model.block_slices()
    blocks = {"b1": [sl["b1"]], "cR": [sl["cR"]], "cA": [sl["cA"]], "w0": sl["w0"], "b0": sl["b0"], "w1": sl["w1"]}
    errs = {}
    gn = np.linalg.norm(go)
    for name, ss in blocks.items():
        a = np.concatenate([g[s] for s in ss]); b = np.concatenate([go[s] for s in ss])
        # relative to the block's own norm, floored by a fraction of the total norm (a block that is ~0 is compared absolutely)
        errs[name] = np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-3 * gn, 1e-300)
        if per_block_tol is not None:
            assert errs[name] <= per_block_tol, f"gradient block {name}: {errs[name]:.3e}"
    return eg, errs, g, go
