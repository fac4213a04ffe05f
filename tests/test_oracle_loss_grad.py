"""Pins for C9-C13 (loss Eqs. 4-7, gradient Eq. 8, Adam/AMSGrad Eqs. 9-13)."""
import numpy as np
import pytest
import torch

from oracle import nep_oracle as O
from oracle.problem import make_problem
from paper_2606_19557_b200 import workloads as wl


@pytest.fixture(scope="module")
def prob():
    return make_problem(wl.tiny_workload(0))


def test_loss_hand_evaluated(prob):
    lam = (1.3, 0.7, 2.1)
    loss4, _ = O.loss_grad(prob.data, prob.theta, prob.scaler, lam, want_grad=False)
    E, F, W = O.forward(prob.data, prob.theta, prob.scaler)
    st = prob.workload.structures
    n = st.n_atoms.astype(float)
    dE = np.mean(((E - prob.E) / n) ** 2)                                       # Eq. 5
    dF = np.sum((F - prob.F) ** 2) / (3 * len(F))                               # Eq. 6
    dV = np.sum(((W - prob.W) / n[:, None]) ** 2) / (9 * st.n_struct)           # Eq. 7
    assert np.allclose(loss4[1:], [dE, dF, dV], rtol=1e-13)
    assert abs(loss4[0] - (lam[0] * dE + lam[1] * dF + lam[2] * dV)) < 1e-13     # Eq. 4


def test_loss_batch_normalisers_and_virial_mask(prob):
    lam = (1.0, 1.0, 1.0)
    E, F, W = O.forward(prob.data, prob.theta, prob.scaler, batch=[1])
    l4, _ = O.loss_grad(prob.data, prob.theta, prob.scaler, lam, batch=[1], want_grad=False)
    n1 = float(prob.workload.structures.n_atoms[1])
    ao = prob.workload.structures.atom_off
    assert abs(l4[1] - ((E[0] - prob.E[1]) / n1) ** 2) < 1e-14
    assert abs(l4[2] - np.sum((F - prob.F[ao[1]:ao[2]]) ** 2) / (3 * n1)) < 1e-14
    prob.data.set_labels(prob.E, prob.F, prob.W, has_virial=[0, 1])
    try:
        l4m, gm = O.loss_grad(prob.data, prob.theta, prob.scaler, lam)
        assert abs(l4m[3] - np.sum(((O.forward(prob.data, prob.theta, prob.scaler)[2][1] - prob.W[1]) / n1) ** 2) / 9) < 1e-14
    finally:
        prob.data.set_labels(prob.E, prob.F, prob.W)


@pytest.mark.parametrize("lam", [(1.0, 2.0, 3.0), (1.0, 0.0, 0.0), (0.0, 1.0, 0.0), (0.0, 0.0, 1.0)])
def test_gradient_matches_central_fd_per_block(prob, lam):
    th = prob.theta
    _, g = O.loss_grad(prob.data, th, prob.scaler, lam)
    h = 1e-5
    gfd = np.zeros_like(g)
    for p in range(len(g)):
        t = th.copy(); t[p] += h
        Lp = O.loss_grad(prob.data, t, prob.scaler, lam, want_grad=False)[0][0]
        t[p] -= 2 * h
        Lm = O.loss_grad(prob.data, t, prob.scaler, lam, want_grad=False)[0][0]
        gfd[p] = (Lp - Lm) / (2 * h)
    assert np.linalg.norm(g - gfd) / np.linalg.norm(gfd) < 1e-7
    sl = prob.workload.model.block_slices()
    blocks = [sl["b1"], sl["cR"], sl["cA"]] + sl["w0"] + sl["b0"] + sl["w1"]
    for s in blocks:
        nrm = np.linalg.norm(gfd[s])
        if nrm > 1e-9:
            assert np.linalg.norm(g[s] - gfd[s]) / nrm < 1e-6


def test_gradient_3body_only_model_and_single_species():
    model = wl.ModelSpec(1, 3.2, 2.6, 1, 2, 3, 2, 4, 0, 0, 3)
    pr = make_problem(wl.tiny_workload(2, n_species=1, model=model))
    lam = (0.5, 1.5, 2.5)
    _, g = O.loss_grad(pr.data, pr.theta, pr.scaler, lam)
    h = 1e-5
    gfd = np.zeros_like(g)
    for p in range(len(g)):
        t = pr.theta.copy(); t[p] += h
        Lp = O.loss_grad(pr.data, t, pr.scaler, lam, want_grad=False)[0][0]
        t[p] -= 2 * h
        Lm = O.loss_grad(pr.data, t, pr.scaler, lam, want_grad=False)[0][0]
        gfd[p] = (Lp - Lm) / (2 * h)
    assert np.linalg.norm(g - gfd) / np.linalg.norm(gfd) < 1e-7


def test_teacher_equals_student_gives_zero_loss_and_gradient(prob):
    l4, g = O.loss_grad(prob.data, prob.theta_teacher, prob.scaler_teacher, (1.0, 1.0, 1.0))
    assert l4[0] == 0.0 and np.abs(g).max() == 0.0


def test_adam_first_step_closed_form_and_constant_gradient():
    rng = np.random.default_rng(0)
    n = 50
    g = rng.normal(size=n); th0 = rng.normal(size=n)
    th = th0.copy(); m = np.zeros(n); v = np.zeros(n); vm = np.zeros(n)
    t = O.adam_step(th, g, m, v, vm, 0, 1e-2)
    assert t == 1
    # first step from zero state: m^ = g, v^ = g^2  ->  dtheta = -lr g / sqrt(g^2 + eps)   (Eqs. 9-13)
    assert np.allclose(th - th0, -1e-2 * g / np.sqrt(g * g + 1e-8), rtol=1e-12)
    for k in range(2, 6):                               # constant g: m^ = g, v^ = g^2 at every step
        t = O.adam_step(th, g, m, v, vm, t, 1e-2)
        assert np.allclose(th - th0, -k * 1e-2 * g / np.sqrt(g * g + 1e-8), rtol=1e-10)


def test_adam_amsgrad_keeps_running_max_of_bias_corrected_v():
    n = 4
    th = np.zeros(n); m = np.zeros(n); v = np.zeros(n); vm = np.zeros(n)
    g1 = np.full(n, 2.0); g2 = np.full(n, 0.01)
    t = O.adam_step(th, g1, m, v, vm, 0, 1e-3)
    assert np.allclose(vm, 4.0)
    t = O.adam_step(th, g2, m, v, vm, t, 1e-3)
    vhat2 = (0.999 * 0.001 * 4.0 + 0.001 * 1e-4) / (1 - 0.999 ** 2)
    assert vhat2 < 4.0 and np.allclose(vm, 4.0)          # Eq. 12: max(v^max_{t-1}, v^_t)
    assert np.allclose(v, 0.999 * 0.004 + 0.001 * 1e-4)


def test_adam_variant1_matches_torch_amsgrad():
    rng = np.random.default_rng(3)
    n = 64
    th0 = rng.normal(size=n)
    p = torch.nn.Parameter(torch.tensor(th0, dtype=torch.float64))
    opt = torch.optim.Adam([p], lr=3e-3, betas=(0.9, 0.999), eps=1e-8, amsgrad=True)
    th = th0.copy(); m = np.zeros(n); v = np.zeros(n); vm = np.zeros(n); t = 0
    for k in range(7):
        g = rng.normal(size=n) * (1.0 if k % 3 else 5.0)
        p.grad = torch.tensor(g, dtype=torch.float64)
        opt.step()
        t = O.adam_step(th, g, m, v, vm, t, 3e-3, variant=1)
        assert np.allclose(th, p.detach().numpy(), rtol=1e-12, atol=1e-14)
