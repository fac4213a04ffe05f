"""ctypes front end of the CPU fp64 oracle (oracle/nep_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It imports nothing from the CUDA package except the plain-data
`ModelSpec` / `StructureSet` containers of the shared, arithmetic-free workload module
(duck-typed: any object with the same attributes works).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "nep_oracle.c")
_LIB = os.path.join(_HERE, "libnep_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off (no FMA contraction: neighbour predicate is bit-reproducible)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-Wall", "-shared", "-fPIC",
                               "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Cfg(C.Structure):
    _fields_ = [("T", C.c_int), ("rcR", C.c_double), ("rcA", C.c_double), ("nmaxR", C.c_int), ("nmaxA", C.c_int),
                ("basR", C.c_int), ("basA", C.c_int), ("l3", C.c_int), ("l4", C.c_int), ("l5", C.c_int), ("H", C.c_int)]


class _Data(C.Structure):
    _fields_ = [("S", C.c_int), ("atom_off", C.c_void_p), ("pos", C.c_void_p), ("box", C.c_void_p), ("type", C.c_void_p),
                ("offR", C.c_void_p), ("jR", C.c_void_p), ("shR", C.c_void_p),
                ("offA", C.c_void_p), ("jA", C.c_void_p), ("shA", C.c_void_p),
                ("E", C.c_void_p), ("F", C.c_void_p), ("W", C.c_void_p), ("has_virial", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.nepo_num_descriptors.restype = C.c_int
        L.nepo_num_params.restype = C.c_int64
        L.nepo_max_threads.restype = C.c_int
        L.nepo_num_harmonics.restype = C.c_int
        L.nepo_build_neighbors.restype = C.c_int64
        L.nepo_adam_step.restype = C.c_int64
        L.nepo_radial_basis.argtypes = [C.c_double, C.c_double, C.c_int, C.c_void_p, C.c_void_p]
        L.nepo_build_neighbors.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                           C.c_void_p, C.c_void_p, C.c_void_p]
        L.nepo_loss_grad.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                     C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.nepo_forward.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p,
                                   C.c_void_p, C.c_void_p, C.c_void_p]
        L.nepo_adam_step.argtypes = [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                     C.c_int64, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int]
        L.nepo_scaler.argtypes = [C.c_int, C.c_int64, C.c_void_p, C.c_void_p]
        L.nepo_descriptors.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.nepo_angular_functions.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_void_p, C.c_void_p]
        L.nepo_harmonic_weights.argtypes = [C.c_int, C.c_void_p]
        L.nepo_image_range.argtypes = [C.c_void_p, C.c_double, C.c_void_p]
        _lib = L
    return _lib


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _cfg(model) -> _Cfg:
    return _Cfg(model.n_species, model.rc_R, model.rc_A, model.n_max_R, model.n_max_A, model.basis_R, model.basis_A,
                model.l_max_3b, model.l_max_4b, model.l_max_5b, model.neurons)


def max_threads() -> int:
    return lib().nepo_max_threads()


def set_num_threads(n: int) -> None:
    lib().nepo_set_num_threads(int(n))


def num_descriptors(model) -> int:
    c = _cfg(model)
    return lib().nepo_num_descriptors(C.byref(c))


def num_params(model) -> int:
    c = _cfg(model)
    return int(lib().nepo_num_params(C.byref(c)))


def radial_basis(r: float, rc: float, basis_size: int):
    """C2 / Eqs. 17-18: returns (f[K], df/dr[K]) with K = basis_size + 1."""
    f = np.zeros(basis_size + 1); df = np.zeros(basis_size + 1)
    lib().nepo_radial_basis(float(r), float(rc), int(basis_size), _p(f), _p(df))
    return f, df


def harmonic_weights(l3: int) -> np.ndarray:
    w = np.zeros(l3 * (l3 + 2))
    lib().nepo_harmonic_weights(int(l3), _p(w))
    return w


def angular_functions(d: Sequence[float], l3: int = 4, has4: bool = True, has5: bool = True):
    """C4: (phi[NA], dphi[NA,3]) for a bond vector d; NA = l3(l3+2) + 9*has4 + 3*has5."""
    d = np.ascontiguousarray(d, np.float64)
    NA = l3 * (l3 + 2) + (9 if has4 else 0) + (3 if has5 else 0)
    phi = np.zeros(NA); dphi = np.zeros((NA, 3))
    lib().nepo_angular_functions(_p(d), int(l3), int(has4), int(has5), _p(phi), _p(dphi))
    return phi, dphi


def image_range(box: np.ndarray, rc: float) -> np.ndarray:
    b = np.ascontiguousarray(box, np.float64).reshape(9)
    m = np.zeros(3, np.int32)
    lib().nepo_image_range(_p(b), float(rc), _p(m))
    return m


def build_neighbors(structs, rc: float):
    """C1: brute-force periodic neighbour lists.  Returns (pair_off int64 [N+1], j int32 [P] (local to the
    structure), shift int8 [P,3]) in ascending (j, na, nb, nc) order per atom."""
    ao = np.ascontiguousarray(structs.atom_off, np.int64)
    pos = np.ascontiguousarray(structs.pos, np.float64)
    box = np.ascontiguousarray(structs.box, np.float64)
    N = int(ao[-1])
    off = np.zeros(N + 1, np.int64)
    P = lib().nepo_build_neighbors(structs.n_struct, _p(ao), _p(pos), _p(box), float(rc), _p(off), None, None)
    j = np.zeros(max(P, 1), np.int32); sh = np.zeros((max(P, 1), 3), np.int8)
    P2 = lib().nepo_build_neighbors(structs.n_struct, _p(ao), _p(pos), _p(box), float(rc), _p(off), _p(j), _p(sh))
    assert P2 == P
    return off, j[:P], sh[:P]


class OracleData:
    """A structure set with its neighbour lists (built once: P:143) and optional labels."""

    def __init__(self, model, structs, E=None, F=None, W=None, has_virial=None):
        self.model = model
        self.structs = structs
        self.atom_off = np.ascontiguousarray(structs.atom_off, np.int64)
        self.pos = np.ascontiguousarray(structs.pos, np.float64)
        self.box = np.ascontiguousarray(structs.box, np.float64).reshape(-1, 9)
        self.type = np.ascontiguousarray(structs.type, np.int32)
        self.offR, self.jR, self.shR = build_neighbors(structs, model.rc_R)
        self.offA, self.jA, self.shA = build_neighbors(structs, model.rc_A)
        self.set_labels(E, F, W, has_virial)

    def set_labels(self, E=None, F=None, W=None, has_virial=None):
        self.E = None if E is None else np.ascontiguousarray(E, np.float64)
        self.F = None if F is None else np.ascontiguousarray(F, np.float64).reshape(-1, 3)
        self.W = None if W is None else np.ascontiguousarray(W, np.float64).reshape(-1, 9)
        self.has_virial = None if has_virial is None else np.ascontiguousarray(has_virial, np.uint8)

    @property
    def n_struct(self):
        return len(self.atom_off) - 1

    @property
    def n_atoms_total(self):
        return int(self.atom_off[-1])

    def _c(self) -> _Data:
        # contiguous non-empty views (ctypes needs a valid pointer even for P = 0)
        def nz(a, dt):
            return a if a.size else np.zeros(1, dt)
        self._keep = [nz(self.jR, np.int32), nz(self.shR, np.int8), nz(self.jA, np.int32), nz(self.shA, np.int8)]
        return _Data(self.n_struct, _p(self.atom_off), _p(self.pos), _p(self.box), _p(self.type),
                     _p(self.offR), _p(self._keep[0]), _p(self._keep[1]),
                     _p(self.offA), _p(self._keep[2]), _p(self._keep[3]),
                     _p(self.E), _p(self.F), _p(self.W), _p(self.has_virial))


def descriptors(data: OracleData, theta: np.ndarray) -> np.ndarray:
    """C3-C5: q[N, D] for every atom of the set (unscaled)."""
    c = _cfg(data.model); X = data._c()
    th = np.ascontiguousarray(theta, np.float64)
    assert th.size == num_params(data.model)
    q = np.zeros((data.n_atoms_total, num_descriptors(data.model)))
    lib().nepo_descriptors(C.byref(c), C.byref(X), _p(th), _p(q))
    return q


def scaler(q: np.ndarray) -> np.ndarray:
    """C6 / Eq. 2: s = 1/(max - min) per descriptor component over all atoms."""
    q = np.ascontiguousarray(q, np.float64)
    s = np.zeros(q.shape[1])
    lib().nepo_scaler(q.shape[1], q.shape[0], _p(q), _p(s))
    return s


def _batch(data, batch):
    if batch is None:
        return data.n_struct, None, np.arange(data.n_struct)
    b = np.ascontiguousarray(batch, np.int32)
    return len(b), b, b


def forward(data: OracleData, theta, scal, batch=None):
    """C7-C8: (E[nb], F[batch atoms, 3], W[nb, 9]) for the structures of `batch` (default all), batch order."""
    c = _cfg(data.model); X = data._c()
    th = np.ascontiguousarray(theta, np.float64); sc = np.ascontiguousarray(scal, np.float64)
    assert th.size == num_params(data.model) and sc.size == num_descriptors(data.model)
    nb, b, ids = _batch(data, batch)
    na = int(sum(data.atom_off[s + 1] - data.atom_off[s] for s in ids))
    E = np.zeros(nb); F = np.zeros((max(na, 1), 3)); W = np.zeros((max(nb, 1), 9))
    lib().nepo_forward(C.byref(c), C.byref(X), _p(th), _p(sc), nb, _p(b), _p(E), _p(F), _p(W))
    return E, F[:na], W[:nb]


def loss_grad(data: OracleData, theta, scal, lambdas, batch=None, want_grad=True):
    """C9-C12 / Eqs. 4-8: (loss4 = [L, dE, dF, dV], grad[N_par] or None)."""
    c = _cfg(data.model); X = data._c()
    th = np.ascontiguousarray(theta, np.float64); sc = np.ascontiguousarray(scal, np.float64)
    assert th.size == num_params(data.model) and sc.size == num_descriptors(data.model)
    assert data.E is not None and data.F is not None and data.W is not None
    nb, b, _ = _batch(data, batch)
    loss4 = np.zeros(4)
    g = np.zeros(th.size) if want_grad else None
    lib().nepo_loss_grad(C.byref(c), C.byref(X), _p(th), _p(sc), nb, _p(b),
                         float(lambdas[0]), float(lambdas[1]), float(lambdas[2]), _p(loss4), _p(g))
    return loss4, g


def adam_step(theta, g, m, v, vmax, t, lr, beta1=0.9, beta2=0.999, eps=1e-8, variant=0) -> int:
    """C13 / Eqs. 9-13, in place on float64 arrays; returns the new step count."""
    for a in (theta, g, m, v, vmax):
        assert a.dtype == np.float64 and a.flags.c_contiguous
    return int(lib().nepo_adam_step(theta.size, _p(theta), _p(g), _p(m), _p(v), _p(vmax), int(t),
                                    float(lr), float(beta1), float(beta2), float(eps), int(variant)))
