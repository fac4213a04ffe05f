"""Thin ctypes binding of libnep_b200 (include/nep.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch supplies device memory (the allocator
callback below hands out `torch.empty(nbytes, dtype=uint8, device='cuda')` tensors and keeps them alive) and
the CUDA stream.  There is no CPU fallback: a missing shared library or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libnep_b200.so")

NEP_OK, NEP_EINVAL, NEP_ESTATE, NEP_ECUDA, NEP_ENOMEM, NEP_ECAPACITY = 0, -1, -2, -3, -4, -5
_CODE_NAMES = {NEP_EINVAL: "NEP_EINVAL", NEP_ESTATE: "NEP_ESTATE", NEP_ECUDA: "NEP_ECUDA", NEP_ENOMEM: "NEP_ENOMEM",
               NEP_ECAPACITY: "NEP_ECAPACITY"}

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_void_p, C.c_size_t)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)

# every symbol include/nep.h declares: name -> (restype, argtypes)
_P = C.c_void_p
SIGNATURES = {
    "nep_version": (C.c_char_p, []),
    "nep_create": (C.c_int, [C.POINTER(_P), C.c_int, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                             C.c_int, C.c_int, C.c_int, ALLOC_FN, FREE_FN, _P, _P]),
    "nep_save_model": (C.c_int, [_P, C.c_char_p]),
    "nep_create_from_model_file": (C.c_int, [C.POINTER(_P), C.c_char_p, ALLOC_FN, FREE_FN, _P, _P]),
    "nep_get_model": (C.c_int, [_P, C.POINTER(C.c_int), _P, _P, _P, _P, C.POINTER(C.c_int)]),
    "nep_destroy": (C.c_int, [_P]),
    "nep_last_error": (C.c_char_p, [_P]),
    "nep_num_descriptors": (C.c_int, [_P]),
    "nep_num_params": (C.c_int64, [_P]),
    "nep_load_structures": (C.c_int, [_P, C.c_int, _P, _P, _P, _P, _P, _P, _P, _P]),
    "nep_set_labels": (C.c_int, [_P, _P, _P, _P, _P]),
    "nep_build_neighbors": (C.c_int, [_P]),
    "nep_get_neighbors": (C.c_int, [_P, C.c_int, C.POINTER(C.c_int64), _P, _P, _P]),
    "nep_set_params": (C.c_int, [_P, _P]),
    "nep_get_params": (C.c_int, [_P, _P]),
    "nep_get_grad": (C.c_int, [_P, _P]),
    "nep_set_grad": (C.c_int, [_P, _P]),
    "nep_set_adam_state": (C.c_int, [_P, _P, _P, _P, C.c_int64]),
    "nep_get_adam_state": (C.c_int, [_P, _P, _P, _P, C.POINTER(C.c_int64)]),
    "nep_compute_scaler": (C.c_int, [_P]),
    "nep_set_scaler": (C.c_int, [_P, _P]),
    "nep_get_scaler": (C.c_int, [_P, _P]),
    "nep_compute_descriptor_range": (C.c_int, [_P, _P, _P]),
    "nep_set_scaler_from_range": (C.c_int, [_P, _P, _P]),
    "nep_scaler_static": (C.c_int, [_P, C.c_int64, C.c_int, _P, _P]),
    "nep_set_batch": (C.c_int, [_P, C.c_int, _P]),
    "nep_forward": (C.c_int, [_P, _P, _P, _P, C.c_int]),
    "nep_set_pair_correction": (C.c_int, [_P, _P, C.c_double, C.c_double, C.c_int, _P, _P, C.c_double, C.c_double, C.c_double]),
    "nep_get_descriptors": (C.c_int, [_P, _P]),
    "nep_loss_grad": (C.c_int, [_P, C.c_double, C.c_double, C.c_double, _P]),
    "nep_get_loss": (C.c_int, [_P, _P]),
    "nep_set_batch_normalisers": (C.c_int, [_P, C.c_int64, C.c_int64, C.c_int64]),
    "nep_grad_device_ptr": (C.c_int, [_P, C.POINTER(_P), C.POINTER(_P)]),
    "nep_adam_step": (C.c_int, [_P, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int]),
    "nep_train_step": (C.c_int, [_P, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int]),
    "nep_synchronize": (C.c_int, [_P]),
    "nep_launch_count": (C.c_int, [_P, C.POINTER(C.c_int64)]),
    "nep_profile_enable": (C.c_int, [_P, C.c_int]),
    "nep_profile_pause": (C.c_int, [_P, C.c_int]),
    "nep_profile_read": (C.c_int, [_P, C.c_int, _P, _P, _P, C.POINTER(C.c_int)]),
    "nep_network_on_tensor_cores": (C.c_int, [_P]),
    "nep_measure_fp32_peak": (C.c_int, [_P, C.POINTER(C.c_double)]),
    "nep_get_sizes": (C.c_int, [_P, _P]),
}

_lib = None


class NepError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"{_CODE_NAMES.get(code, code)}: {msg}")
        self.code = code


def load_library() -> C.CDLL:
    """dlopen libnep_b200.so and declare the prototypes.  Raises if the library was not built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_19557_b200.build` "
                              "(there is no CPU or PyTorch fallback for the NEP step)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(L, name)          # AttributeError if the symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _np(a, dtype, shape=None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=dtype)
    if shape is not None:
        a = a.reshape(shape)
    return a


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


NEP_STATIC_MAX_DESCRIPTORS = 128


def scaler_static(q, s, stream=None) -> None:
    """nep_scaler_static (include/nep.h): Eq. 2's scaler s [D] from the descriptor matrix q [N][D], both float32 CUDA tensors that
    the CALLER owns, on the current device.  For callers that cannot give the library an allocator (a context needs one) and
    cannot call cudaMalloc themselves: the call allocates nothing, its working memory is a fixed array inside the library, so
    D <= NEP_STATIC_MAX_DESCRIPTORS (NepError NEP_ECAPACITY beyond) and calls that could overlap on one GPU must be serialised.
    Enqueues on `stream` (default: torch's current stream) and returns without synchronising."""
    import torch
    L = load_library()
    if not (q.is_cuda and s.is_cuda and q.dtype == torch.float32 and s.dtype == torch.float32 and q.is_contiguous() and s.is_contiguous()):
        raise ValueError("q and s must be contiguous float32 CUDA tensors")
    if q.dim() != 2 or s.numel() != q.shape[1]:
        raise ValueError("q must be [N][D] and s [D]")
    if stream is None:
        stream = torch.cuda.current_stream()
    rc = L.nep_scaler_static(C.c_void_p(q.data_ptr()), int(q.shape[0]), int(q.shape[1]), C.c_void_p(s.data_ptr()), C.c_void_p(stream.cuda_stream))
    if rc != NEP_OK:
        raise NepError(rc, (L.nep_last_error(None) or b"").decode())


def measure_fp32_peak(stream=None) -> float:
    """nep_measure_fp32_peak: TFLOP/s of a register-resident FP32 FMA loop on the current device (measurement aid for bench.py)."""
    import torch
    L = load_library()
    if stream is None:
        stream = torch.cuda.current_stream()
    v = C.c_double(0.0)
    rc = L.nep_measure_fp32_peak(C.c_void_p(stream.cuda_stream), C.byref(v))
    if rc != NEP_OK:
        raise NepError(rc, (L.nep_last_error(None) or b"").decode())
    return v.value


class Nep:
    """One context = one CUDA device + one stream (include/nep.h).  Method names are the C calls without `nep_`."""

    def __init__(self, n_species: int = 0, rc_R: float = 0.0, rc_A: float = 0.0, n_max_R: int = 0, n_max_A: int = 0, basis_R: int = 0,
                 basis_A: int = 0, l_max_3b: int = 4, l_max_4b: int = 2, l_max_5b: int = 1, neurons: int = 30, stream=None,
                 guard_bytes: int = 0, model_file: Optional[str] = None):
        import torch
        self._L = load_library()
        self._h = C.c_void_p(None)
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the NEP step has no CPU fallback")
        self._torch = torch
        self._bufs = {}
        self.bytes_allocated = 0
        # debugging aid (compute-sanitizer is not available everywhere): every device buffer handed to the library gets a guard
        # band of `guard_bytes` (a multiple of 256) filled with 0xA5 on both sides; check_guards() verifies they are untouched
        self._guard = int(guard_bytes)
        if self._guard % 256:
            raise ValueError("guard_bytes must be a multiple of 256")
        if stream is None:
            stream = torch.cuda.current_stream()
        self.stream = stream

        def _alloc(_user, nbytes):
            try:
                # allocate on the stream the library launches on: the caching allocator then reuses a freed block only
                # in that stream's order, whatever torch's current stream is when the callback runs
                with torch.cuda.stream(self.stream):
                    t = torch.empty(int(nbytes) + 2 * self._guard, dtype=torch.uint8, device="cuda")
                    if self._guard:
                        t[:self._guard].fill_(0xA5); t[self._guard + int(nbytes):].fill_(0xA5)
            except Exception:      # noqa: BLE001  (OOM -> NULL -> NEP_ENOMEM)
                return None
            p = t.data_ptr() + self._guard
            self._bufs[p] = t[self._guard:self._guard + int(nbytes)] if self._guard else t
            if self._guard:
                self._guarded = getattr(self, "_guarded", {})
                self._guarded[p] = (t, int(nbytes))
            self.bytes_allocated += int(nbytes)
            return p

        def _free(_user, p):
            t = self._bufs.pop(p, None)
            if t is not None:
                self.bytes_allocated -= t.numel()
            if self._guard and p in getattr(self, "_guarded", {}):
                self._freed_ok = getattr(self, "_freed_ok", True) and self._bands_intact(*self._guarded.pop(p))

        self._alloc_cb = ALLOC_FN(_alloc)
        self._free_cb = FREE_FN(_free)
        h = C.c_void_p(None)
        if model_file is not None:
            rc = self._L.nep_create_from_model_file(C.byref(h), os.fsencode(model_file), self._alloc_cb, self._free_cb, None,
                                                    C.c_void_p(stream.cuda_stream))
        else:
            rc = self._L.nep_create(C.byref(h), n_species, rc_R, rc_A, n_max_R, n_max_A, basis_R, basis_A, l_max_3b, l_max_4b,
                                    l_max_5b, neurons, self._alloc_cb, self._free_cb, None, C.c_void_p(stream.cuda_stream))
        if rc != NEP_OK:
            raise NepError(rc, (self._L.nep_last_error(None) or b"").decode())
        self._h = h
        self.D = self._L.nep_num_descriptors(h)
        self.n_par = int(self._L.nep_num_params(h))
        self.n_struct = 0
        self.n_atoms_total = 0

    def _bands_intact(self, t, nbytes) -> bool:
        g = self._guard
        return bool((t[:g] == 0xA5).all().item()) and bool((t[g + nbytes:] == 0xA5).all().item())

    def check_guards(self) -> int:
        """Number of live buffers whose guard bands were verified; raises if a band was written (also for buffers already freed)."""
        self._torch.cuda.synchronize()
        if not self._guard:
            raise RuntimeError("context was created without guard_bytes")
        if not getattr(self, "_freed_ok", True):
            raise RuntimeError("a guard band of a buffer that has since been released was overwritten")
        bad = [hex(p) for p, (t, n) in getattr(self, "_guarded", {}).items() if not self._bands_intact(t, n)]
        if bad:
            raise RuntimeError(f"guard bands overwritten next to {len(bad)} device buffers: {bad[:4]}")
        return len(getattr(self, "_guarded", {}))

    @classmethod
    def from_model_file(cls, path: str, **kw) -> "Nep":
        """nep_create_from_model_file: hyper-parameters, scaler and parameters from a file written by save_model."""
        return cls(model_file=path, **kw)

    def save_model(self, path: str):
        self._ck(self._L.nep_save_model(self._h, os.fsencode(path)))

    def get_model(self) -> dict:
        """Hyper-parameters of the context in the vocabulary of Table I."""
        T, H = C.c_int(0), C.c_int(0)
        rc = np.zeros(2, np.float64); nm = np.zeros(2, np.int32); bs = np.zeros(2, np.int32); lm = np.zeros(3, np.int32)
        self._ck(self._L.nep_get_model(self._h, C.byref(T), _ptr(rc), _ptr(nm), _ptr(bs), _ptr(lm), C.byref(H)))
        return dict(n_species=T.value, rc_R=float(rc[0]), rc_A=float(rc[1]), n_max_R=int(nm[0]), n_max_A=int(nm[1]), basis_R=int(bs[0]),
                    basis_A=int(bs[1]), l_max_3b=int(lm[0]), l_max_4b=int(lm[1]), l_max_5b=int(lm[2]), neurons=H.value)

    def predict(self, st):
        """Prediction-only path: structures without labels in, (E [S], F [N,3], W [S,9]) out.  The calls are
        nep_load_structures (labels NULL) + nep_build_neighbors + nep_forward; parameters and scaler stay as they are."""
        self.load_structure_set(st)
        self.build_neighbors()
        return self.forward()

    @classmethod
    def from_model(cls, model, **kw) -> "Nep":
        return cls(model.n_species, model.rc_R, model.rc_A, model.n_max_R, model.n_max_A, model.basis_R, model.basis_A,
                   model.l_max_3b, model.l_max_4b, model.l_max_5b, model.neurons, **kw)

    # ---- plumbing ----
    def _ck(self, rc: int):
        if rc != NEP_OK:
            raise NepError(rc, (self._L.nep_last_error(self._h) or b"").decode())

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h:
            self._L.nep_destroy(self._h)
            self._h = C.c_void_p(None)
            self._bufs.clear()

    def __del__(self):
        try:
            self.destroy()
        except Exception:   # noqa: BLE001
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    @staticmethod
    def version() -> str:
        return load_library().nep_version().decode()

    # ---- data ----
    def load_structures(self, n_atoms, pos, box, type_, E=None, F=None, W=None, has_virial=None):
        n_atoms = _np(n_atoms, np.int32)
        S = len(n_atoms); N = int(n_atoms.sum())
        pos = _np(pos, np.float64, (N, 3)); box = _np(box, np.float64, (S, 9)); type_ = _np(type_, np.int32, (N,))
        E = None if E is None else _np(E, np.float64, (S,))
        F = None if F is None else _np(F, np.float64, (N, 3))
        W = None if W is None else _np(W, np.float64, (S, 9))
        hv = None if has_virial is None else _np(has_virial, np.uint8, (S,))
        self._ck(self._L.nep_load_structures(self._h, S, _ptr(n_atoms), _ptr(pos), _ptr(box), _ptr(type_), _ptr(E), _ptr(F),
                                             _ptr(W), _ptr(hv)))
        self.n_struct, self.n_atoms_total = S, N
        self._n_atoms = n_atoms.copy()
        self._has_virial = np.ones(S, np.uint8) if hv is None else hv.copy()     # the mask the context normalises Eq. 7 with

    def load_structure_set(self, st, E=None, F=None, W=None, has_virial=None):
        self.load_structures(st.n_atoms, st.pos, st.box, st.type, E, F, W, has_virial)

    def set_labels(self, E, F, W, has_virial=None):
        S, N = self.n_struct, self.n_atoms_total
        E = _np(E, np.float64, (S,)); F = _np(F, np.float64, (N, 3)); W = _np(W, np.float64, (S, 9))
        hv = None if has_virial is None else _np(has_virial, np.uint8, (S,))
        self._ck(self._L.nep_set_labels(self._h, _ptr(E), _ptr(F), _ptr(W), _ptr(hv)))
        self._has_virial = np.ones(S, np.uint8) if hv is None else hv.copy()

    def build_neighbors(self):
        self._ck(self._L.nep_build_neighbors(self._h))
        self._batch_ids = np.arange(self.n_struct, dtype=np.int32)

    def get_neighbors(self, which: int):
        """(offsets int64 [N+1], j int32 [P], shift int8 [P,3]) of the radial (0) or angular (1) list."""
        P = C.c_int64(0)
        off = np.zeros(self.n_atoms_total + 1, np.int64)
        self._ck(self._L.nep_get_neighbors(self._h, which, C.byref(P), _ptr(off), None, None))
        j = np.zeros(max(P.value, 1), np.int32); sh = np.zeros((max(P.value, 1), 3), np.int8)
        self._ck(self._L.nep_get_neighbors(self._h, which, C.byref(P), None, _ptr(j), _ptr(sh)))
        return off, j[:P.value], sh[:P.value]

    # ---- parameters ----
    def set_params(self, theta):
        th = _np(theta, np.float32, (self.n_par,))
        self._ck(self._L.nep_set_params(self._h, _ptr(th)))

    def get_params(self) -> np.ndarray:
        th = np.zeros(self.n_par, np.float32)
        self._ck(self._L.nep_get_params(self._h, _ptr(th)))
        return th

    def get_grad(self) -> np.ndarray:
        g = np.zeros(self.n_par, np.float32)
        self._ck(self._L.nep_get_grad(self._h, _ptr(g)))
        return g

    def set_grad(self, g):
        g = _np(g, np.float32, (self.n_par,))
        self._ck(self._L.nep_set_grad(self._h, _ptr(g)))

    def set_adam_state(self, m, v, vmax, t: int):
        m = _np(m, np.float32, (self.n_par,)); v = _np(v, np.float32, (self.n_par,)); vmax = _np(vmax, np.float32, (self.n_par,))
        self._ck(self._L.nep_set_adam_state(self._h, _ptr(m), _ptr(v), _ptr(vmax), int(t)))

    def get_adam_state(self):
        m = np.zeros(self.n_par, np.float32); v = np.zeros_like(m); vmax = np.zeros_like(m)
        t = C.c_int64(0)
        self._ck(self._L.nep_get_adam_state(self._h, _ptr(m), _ptr(v), _ptr(vmax), C.byref(t)))
        return m, v, vmax, t.value

    def compute_scaler(self):
        self._ck(self._L.nep_compute_scaler(self._h))
        self._batch_ids = np.arange(self.n_struct, dtype=np.int32)

    def set_scaler(self, s):
        s = _np(s, np.float64, (self.D,))
        self._ck(self._L.nep_set_scaler(self._h, _ptr(s)))

    def get_scaler(self) -> np.ndarray:
        s = np.zeros(self.D, np.float64)
        self._ck(self._L.nep_get_scaler(self._h, _ptr(s)))
        return s

    def compute_descriptor_range(self):
        """(qmin, qmax), float64 [D] each: range of every descriptor component over this context's atoms."""
        lo = np.zeros(self.D, np.float64); hi = np.zeros(self.D, np.float64)
        self._ck(self._L.nep_compute_descriptor_range(self._h, _ptr(lo), _ptr(hi)))
        self._batch_ids = np.arange(self.n_struct, dtype=np.int32)
        return lo, hi

    def set_scaler_from_range(self, qmin, qmax):
        lo = _np(qmin, np.float64, (self.D,)); hi = _np(qmax, np.float64, (self.D,))
        self._ck(self._L.nep_set_scaler_from_range(self._h, _ptr(lo), _ptr(hi)))

    # ---- step ----
    def set_batch(self, ids: Optional[Sequence[int]] = None):
        if ids is None:
            self._ck(self._L.nep_set_batch(self._h, 0, None))
            self._batch_ids = np.arange(self.n_struct, dtype=np.int32)
        else:
            ids = _np(ids, np.int32)
            # a zero-length numpy array still has a valid (non-NULL) data pointer: ids != NULL, n = 0 -> empty batch
            self._ck(self._L.nep_set_batch(self._h, len(ids), _ptr(ids) if len(ids) else _ptr(np.zeros(1, np.int32))))
            self._batch_ids = ids.copy()

    def batch_shape(self):
        """(S_b, N_b) of the current batch."""
        ids = self._batch_ids
        return len(ids), int(self._n_atoms[ids].sum()) if len(ids) else 0

    def batch_counts(self):
        """(S_b, N_b, S_v) of the current batch: the counts Eqs. 5-7 divide by (S_v = structures whose virial label counts, from the
        mask given with the labels)."""
        ids = self._batch_ids
        Sb, Nb = self.batch_shape()
        return Sb, Nb, int(self._has_virial[ids].sum()) if len(ids) else 0

    def forward(self, want=("E", "F", "W")):
        """S1-S5.  Returns host float32 arrays (E [S_b], F [N_b,3], W [S_b,9]) (None for those not wanted)."""
        Sb, Nb = self.batch_shape()
        E = np.zeros(Sb, np.float32) if "E" in want else None
        F = np.zeros((Nb, 3), np.float32) if "F" in want else None
        W = np.zeros((Sb, 9), np.float32) if "W" in want else None
        self._ck(self._L.nep_forward(self._h, _ptr(E), _ptr(F), _ptr(W), 1))
        return E, F, W

    def forward_device(self, E=None, F=None, W=None):
        """S1-S5 without synchronising.  E, F, W: optional float32 CUDA tensors receiving the outputs."""
        dp = lambda t: None if t is None else C.c_void_p(t.data_ptr())   # noqa: E731
        self._ck(self._L.nep_forward(self._h, dp(E), dp(F), dp(W), 0))

    def set_pair_correction(self, Z=None, r_inner=0.0, r_outer=0.0, coef=(), expo=(), a_prefac=1.0, a_pow=1.0, coulomb_k=1.0):
        """nep_set_pair_correction: the short-range pair term of P:105 with the caller's constants; Z=None switches it off."""
        if Z is None:
            self._ck(self._L.nep_set_pair_correction(self._h, None, 0.0, 0.0, 0, None, None, 1.0, 1.0, 1.0))
            return
        Z = _np(Z, np.float64, (self.get_model()["n_species"],)); coef = _np(coef, np.float64); expo = _np(expo, np.float64, (len(coef),))
        self._ck(self._L.nep_set_pair_correction(self._h, _ptr(Z), float(r_inner), float(r_outer), len(coef), _ptr(coef), _ptr(expo),
                                                 float(a_prefac), float(a_pow), float(coulomb_k)))

    def get_descriptors(self) -> np.ndarray:
        Sb, Nb = self.batch_shape()
        q = np.zeros((Nb, self.D), np.float32)
        self._ck(self._L.nep_get_descriptors(self._h, _ptr(q)))
        return q

    def loss_grad(self, lambda_E: float, lambda_F: float, lambda_V: float, fetch_loss: bool = True):
        """S6-S9.  Returns loss4 = [L, dE, dF, dV] (float64, host) or None when fetch_loss is False (no sync)."""
        l4 = np.zeros(4, np.float64) if fetch_loss else None
        self._ck(self._L.nep_loss_grad(self._h, lambda_E, lambda_F, lambda_V, _ptr(l4)))
        return l4

    def get_loss(self) -> np.ndarray:
        l4 = np.zeros(4, np.float64)
        self._ck(self._L.nep_get_loss(self._h, _ptr(l4)))
        return l4

    # ---- data-parallel training (include/nep.h: nep_set_batch_normalisers) ----
    def set_batch_normalisers(self, n_struct_whole: int, n_atoms_whole: int, n_virial_whole: int):
        self._ck(self._L.nep_set_batch_normalisers(self._h, int(n_struct_whole), int(n_atoms_whole), int(n_virial_whole)))

    def grad_loss_tensors(self):
        """(g, loss4): torch views (float32 [N_par], float64 [4]) of the context's gradient and loss terms on the device,
        for in-place collectives.  Needs the torch allocator (the views alias the tensors it handed to the library)."""
        g, l = C.c_void_p(None), C.c_void_p(None)
        self._ck(self._L.nep_grad_device_ptr(self._h, C.byref(g), C.byref(l)))
        torch = self._torch

        def view(ptr, dtype, count):
            isz = torch.empty(0, dtype=dtype).element_size()
            for base, t in self._bufs.items():
                if base <= ptr < base + t.numel():
                    off = ptr - base
                    return t[off:off + count * isz].view(dtype)
            raise RuntimeError("device pointer is not inside an allocation of this context")
        return view(g.value, torch.float32, self.n_par), view(l.value, torch.float64, 4)

    def adam_step(self, lr: float, beta1: float = 0.9, beta2: float = 0.999, eps: float = 1e-8, variant: int = 0):
        self._ck(self._L.nep_adam_step(self._h, lr, beta1, beta2, eps, variant))

    def train_step(self, lambda_E: float, lambda_F: float, lambda_V: float, lr: float, beta1: float = 0.9, beta2: float = 0.999,
                   eps: float = 1e-8, variant: int = 0, use_graph: bool = True):
        """forward + loss_grad + adam_step on the current batch as one call (one CUDA graph launch with use_graph)."""
        self._ck(self._L.nep_train_step(self._h, lambda_E, lambda_F, lambda_V, lr, beta1, beta2, eps, variant, int(use_graph)))

    def synchronize(self):
        self._ck(self._L.nep_synchronize(self._h))

    # ---- measurement aids ----
    def launch_count(self) -> int:
        n = C.c_int64(0)
        self._ck(self._L.nep_launch_count(self._h, C.byref(n)))
        return n.value

    def profile_enable(self, on: bool = True):
        self._ck(self._L.nep_profile_enable(self._h, int(on)))

    def profile_pause(self, paused: bool = True):
        self._ck(self._L.nep_profile_pause(self._h, int(paused)))

    def profile_read(self, cap: int = 64):
        """{kernel name: (total ms, launches)} since the last read."""
        names = (C.c_char_p * cap)(); ms = (C.c_double * cap)(); ln = (C.c_int64 * cap)(); n = C.c_int(0)
        self._ck(self._L.nep_profile_read(self._h, cap, C.cast(names, C.c_void_p), C.cast(ms, C.c_void_p), C.cast(ln, C.c_void_p),
                                          C.byref(n)))
        return {names[i].decode(): (ms[i], ln[i]) for i in range(n.value)}

    def network_on_tensor_cores(self) -> bool:
        return bool(self._L.nep_network_on_tensor_cores(self._h))

    def get_sizes(self) -> dict:
        s = np.zeros(8, np.int64)
        self._ck(self._L.nep_get_sizes(self._h, _ptr(s)))
        return dict(zip(("S", "N", "P_R", "P_A", "S_b", "N_b", "P_R_b", "P_A_b"), (int(x) for x in s)))
