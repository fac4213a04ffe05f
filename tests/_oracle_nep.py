"""An oracle-backed stand-in for `binding.Nep` with the same method names, for CPU tests of the host logic that drives a
context (dataparallel.DataParallelNep, trainer.Trainer) where no GPU exists.  Test infrastructure only: it lives under tests/
and calls oracle/; the product never imports it."""
import numpy as np
import torch

from oracle import nep_oracle as O


class OracleNep:
    def __init__(self, model):
        self.model = model
        self.D, self.n_par = model.D, model.n_par
        self.stream = None
        self.theta = np.zeros(model.n_par)
        self.m = np.zeros(model.n_par); self.v = np.zeros(model.n_par); self.vmax = np.zeros(model.n_par); self.t = 0
        self.scaler = None
        self._g = torch.zeros(model.n_par, dtype=torch.float32)
        self._l4 = torch.zeros(4, dtype=torch.float64)
        self.whole = None

    @classmethod
    def from_model(cls, model, **kw):
        return cls(model)

    # ---- data ----
    def load_structure_set(self, st, E=None, F=None, W=None, has_virial=None):
        self.st = st
        self.n_struct = st.n_struct
        self.labels = None if E is None else (np.asarray(E, float), np.asarray(F, float), np.asarray(W, float), has_virial)

    def set_labels(self, E, F, W, has_virial=None):
        self.labels = (np.asarray(E, float), np.asarray(F, float), np.asarray(W, float), has_virial)
        if getattr(self, "data", None) is not None and self.st.n_struct:
            self.data.set_labels(*self.labels)

    def build_neighbors(self):
        self.data = O.OracleData(self.model, self.st) if self.st.n_struct else None
        if self.data is not None and self.labels is not None:
            self.data.set_labels(*self.labels)
        self.batch = list(range(self.st.n_struct))

    def set_params(self, theta):
        self.theta = np.asarray(theta, np.float32).astype(np.float64)

    def get_params(self):
        return self.theta.astype(np.float32)

    # ---- Eq. 2 ----
    def compute_descriptor_range(self):
        if self.data is None:
            return np.full(self.D, np.inf), np.full(self.D, -np.inf)
        q = O.descriptors(self.data, self.theta)
        return q.min(0), q.max(0)

    def set_scaler_from_range(self, qmin, qmax):
        self.scaler = O.scaler(np.stack([np.asarray(qmin, float), np.asarray(qmax, float)]))   # 1/(max-min), degenerate -> 1

    def set_scaler(self, s):
        self.scaler = np.asarray(s, float)

    def get_scaler(self):
        return self.scaler.copy()

    # ---- step ----
    def set_batch(self, ids=None):
        self.batch = list(range(self.st.n_struct)) if ids is None else [int(i) for i in ids]
        self.whole = None

    def batch_shape(self):
        return len(self.batch), int(self.st.n_atoms[self.batch].sum()) if self.batch else 0

    def batch_counts(self):
        Sb, Nb = self.batch_shape()
        hv = None if self.labels is None else self.labels[3]
        return Sb, Nb, Sb if hv is None else int(np.asarray(hv)[self.batch].sum()) if self.batch else 0

    def set_batch_normalisers(self, S, N, Sv):
        self.whole = (S, N, Sv)

    def forward_device(self):
        pass

    def loss_grad(self, lE, lF, lV, fetch_loss=True):
        g = np.zeros(self.n_par); l4 = np.zeros(4)
        if self.batch:
            hv = self.labels[3]
            Sr, Nr = self.batch_shape()
            Svr = Sr if hv is None else int(np.asarray(hv)[self.batch].sum())
            whole = self.whole or (Sr, Nr, Svr)
            # the oracle divides by the counts of the batch it is given: re-weight every term to the whole batch's counts
            for k, (cr, cw, lam) in enumerate(((Sr, whole[0], lE), (Nr, whole[1], lF), (Svr, whole[2], lV))):
                if cr == 0 or lam == 0.0:
                    continue
                one = [0.0, 0.0, 0.0]; one[k] = lam
                l4k, gk = O.loss_grad(self.data, self.theta, self.scaler, tuple(one), batch=self.batch)
                g += gk * (cr / cw); l4[0] += l4k[0] * (cr / cw); l4[1 + k] += l4k[1 + k] * (cr / cw)
        self._g.copy_(torch.from_numpy(g.astype(np.float32))); self._l4.copy_(torch.from_numpy(l4))
        return l4 if fetch_loss else None

    def grad_loss_tensors(self):
        return self._g, self._l4

    def get_loss(self):
        return self._l4.numpy().copy()

    def adam_step(self, lr, beta1=0.9, beta2=0.999, eps=1e-8, variant=0):
        self.t = O.adam_step(self.theta, self._g.numpy().astype(np.float64), self.m, self.v, self.vmax, self.t, lr, beta1, beta2, eps, variant)
