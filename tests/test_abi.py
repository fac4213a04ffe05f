"""The C-ABI library loads and exports every symbol include/nep.h declares (no compute calls: no GPU needed)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "nep.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(nep_[a-z0-9_]+)\s*\(", src)) - {"nep_alloc_fn", "nep_free_fn"})


@pytest.fixture(scope="module")
def built():
    from paper_2606_19557_b200 import build
    return build.build()


def test_header_declares_the_calls_of_the_north_star():
    names = _declared()
    for need in ("nep_create", "nep_load_structures", "nep_build_neighbors", "nep_forward", "nep_loss_grad", "nep_adam_step"):
        assert need in names


def test_library_exports_every_declared_symbol(built):
    L = ctypes.CDLL(built)
    for name in _declared():
        assert hasattr(L, name), name


def test_binding_covers_every_declared_symbol(built):
    from paper_2606_19557_b200 import binding
    assert sorted(binding.SIGNATURES) == _declared()
    L = binding.load_library()
    assert b"sm_100a" in L.nep_version()


def test_create_without_gpu_fails_loudly_or_validates(built):
    """No CPU fallback: without a device nep_create returns NEP_ECUDA; bad arguments are NEP_EINVAL before that."""
    from paper_2606_19557_b200 import binding
    L = binding.load_library()
    h = ctypes.c_void_p(None)
    null_a, null_f = ctypes.cast(None, binding.ALLOC_FN), ctypes.cast(None, binding.FREE_FN)
    rc = L.nep_create(ctypes.byref(h), 0, 5.0, 4.0, 4, 4, 8, 8, 4, 2, 1, 30, null_a, null_f, None, None)
    assert rc == binding.NEP_EINVAL and b"n_species" in L.nep_last_error(None)
    rc = L.nep_create(ctypes.byref(h), 1, 4.0, 5.0, 4, 4, 8, 8, 4, 2, 1, 30, null_a, null_f, None, None)
    assert rc == binding.NEP_EINVAL
    for l3, l4, l5 in ((0, 2, 1), (5, 2, 1), (4, 1, 1), (4, 2, 2)):          # l_max_3b in 1..4, l_max_4b in {0,2}, l_max_5b in {0,1}
        rc = L.nep_create(ctypes.byref(h), 1, 5.0, 4.0, 4, 4, 8, 8, l3, l4, l5, 30, null_a, null_f, None, None)
        assert rc == binding.NEP_EINVAL and b"l_max" in L.nep_last_error(None)
    rc = L.nep_create_from_model_file(ctypes.byref(h), b"/nonexistent/model.txt", null_a, null_f, None, None)
    assert rc == binding.NEP_EINVAL and b"cannot open" in L.nep_last_error(None)
    import os
    import tempfile
    import torch
    with tempfile.TemporaryDirectory() as td:               # the model-file reader runs on the host: header checks need no device
        bad = os.path.join(td, "bad.txt")
        open(bad, "w").write("nep_b200_model 2\nn_species 1\n")
        rc = L.nep_create_from_model_file(ctypes.byref(h), bad.encode(), null_a, null_f, None, None)
        assert rc == binding.NEP_EINVAL and b"not a nep_b200 model file" in L.nep_last_error(None)
        good = os.path.join(td, "good.txt")
        open(good, "w").write("nep_b200_model 1\nn_species 1\ncutoff 3 2\nn_max 0 0\nbasis_size 1 1\nl_max 4 0 0\nneuron 1\n"
                              "scaler 5\n1\n1\n1\n1\n1\ntheta 12\n" + "0.5\n" * 12)
        rc = L.nep_create_from_model_file(ctypes.byref(h), good.encode(), null_a, null_f, None, None)
        # a well-formed header reaches nep_create: without a device that is NEP_ECUDA, with one the NULL allocator is refused
        assert rc == (binding.NEP_EINVAL if torch.cuda.is_available() else binding.NEP_ECUDA)
        assert b"not a nep_b200 model file" not in L.nep_last_error(None)
    if not torch.cuda.is_available():
        rc = L.nep_create(ctypes.byref(h), 1, 5.0, 4.0, 4, 4, 8, 8, 4, 2, 1, 30, null_a, null_f, None, None)
        assert rc == binding.NEP_ECUDA and b"no CPU fallback" in L.nep_last_error(None)
        with pytest.raises(RuntimeError):
            binding.Nep(1, 5.0, 4.0, 4, 4, 8, 8)
