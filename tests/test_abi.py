"""`-m "not gpu"`: the C-ABI library builds for sm_100a, loads, and exports every symbol include/gwlnl.h
declares; argument validation that needs no device; the product path fails loudly without a GPU."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
COVERED_HEADERS = ("gwlnl.h", "gwlnl_tuning.h", "gwpop.h", "gwprobe.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1904_02863_b200.csrc import build as csrc_build
    csrc_build.build()
    from paper_1904_02863_b200 import binding
    return binding.load_library()


def _declared_functions(header="gwlnl.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(gw_[a-z0-9_]+)\s*\(", text)))


def test_header_symbols_are_exported(lib):
    from paper_1904_02863_b200 import binding
    names = _declared_functions()
    assert {"gw_ctx_create", "gw_waveform_batch", "gw_lnl_batch", "gw_ctx_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in gwlnl.h but not exported"
    assert sorted(binding.EXPORTS) == names
    tuning = _declared_functions("gwlnl_tuning.h")
    assert sorted(binding.TUNING_EXPORTS) == tuning and tuning
    for n in tuning:
        assert hasattr(lib, n), f"{n} declared in gwlnl_tuning.h but not exported"
    from paper_1904_02863_b200 import population
    pop = _declared_functions("gwpop.h")
    assert sorted(population.EXPORTS) == pop and {"gw_pop_ctx_create", "gw_pop_lnl_batch", "gw_pop_ctx_destroy"} <= set(pop)
    for n in pop:
        assert hasattr(lib, n), f"{n} declared in gwpop.h but not exported"
    # the probes (fp64 rate, HBM bandwidth) live in their own library, not in the product library
    assert not any(hasattr(lib, n) for n in _declared_functions("gwprobe.h"))


def test_probe_library_exports_its_header():
    from paper_1904_02863_b200.csrc import build as csrc_build
    csrc_build.build_probe()
    from paper_1904_02863_b200 import probes
    plib = probes.load_library()
    names = _declared_functions("gwprobe.h")
    assert sorted(probes.EXPORTS) == names and names
    for n in names:
        assert hasattr(plib, n), f"{n} declared in gwprobe.h but not exported"


def test_every_header_is_covered():
    """Each header under include/ is checked against the library that implements it."""
    assert sorted(os.listdir(os.path.join(ROOT, "include"))) == sorted(COVERED_HEADERS)


def test_no_compute_calls(lib):
    assert lib.gw_abi_version() == 5
    assert lib.gw_strerror(0) == b"ok" and b"invalid" in lib.gw_strerror(-1)
    assert lib.gw_ctx_destroy(None) == 0
    assert lib.gw_ctx_info(None, None, None, None, None) == -1
    assert lib.gw_ctx_n_param(None) == -1
    assert lib.gw_lnl_batch(None, 1, None, None, None, None) == -1
    assert lib.gw_waveform_batch(None, 1, None, None, None) == -1
    assert lib.gw_ctx_reserve(None, 8) == -1
    assert lib.gw_last_cuda_error(None) == 0 and lib.gw_ctx_launch_count(None) == 0
    from paper_1904_02863_b200 import population
    population._lib()
    assert lib.gw_pop_ctx_destroy(None) == 0 and lib.gw_pop_ctx_launch_count(None) == 0
    assert lib.gw_pop_ctx_info(None, None, None, None, None) == -1
    assert lib.gw_pop_lnl_batch(None, 1, None, None, None) == -1
    h = ctypes.c_void_p()
    x = np.zeros(12)
    assert lib.gw_pop_ctx_create(ctypes.byref(h), 0, 2, x.ctypes.data, x.ctypes.data, 1, None) == -1 and not h
    assert lib.gw_pop_ctx_create(ctypes.byref(h), 1, 2, None, x.ctypes.data, 1, None) == -1 and not h


def test_create_rejects_bad_arguments_before_touching_cuda(lib):
    from paper_1904_02863_b200 import binding
    h = ctypes.c_void_p()
    f = np.arange(20.0, 30.0, 0.25)
    d = np.zeros((1, f.size, 2))
    S = np.ones((1, f.size))
    det = binding.detector_structs(np.array([[1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 0, 0.0]]))
    fp, dp, sp = f.ctypes.data, d.ctypes.data, S.ctypes.data
    assert lib.gw_ctx_create(None, f.size, fp, 1, dp, sp, det, 0.0, None, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_ctx_create(ctypes.byref(h), 1, fp, 1, dp, sp, det, 0.0, None, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_ctx_create(ctypes.byref(h), f.size, None, 1, dp, sp, det, 0.0, None, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_ctx_create(ctypes.byref(h), f.size, fp, 0, dp, sp, det, 0.0, None, None) == binding.GW_ERR_INVALID_ARG
    assert lib.gw_ctx_create(ctypes.byref(h), f.size, fp, 9, dp, sp, det, 0.0, None, None) == binding.GW_ERR_INVALID_ARG
    opt = binding.gw_options(1, 2, 16, 0, 0)      # isco_cut must be 0 or 1
    assert lib.gw_ctx_create(ctypes.byref(h), f.size, fp, 1, dp, sp, det, 0.0, ctypes.byref(opt), None) == binding.GW_ERR_INVALID_ARG
    assert not h


def test_product_path_fails_loudly_without_gpu(lib):
    """No CPU fallback: on a box without a CUDA device the context cannot be created (and nothing under
    paper_1904_02863_b200 imports the oracle)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1904_02863_b200 import binding
    h = ctypes.c_void_p()
    f = np.arange(20.0, 30.0, 0.25)
    d = np.zeros((1, f.size, 2))
    S = np.ones((1, f.size))
    det = binding.detector_structs(np.array([[1, 0, 0, 0, 0, 0, 0, 0, 0, 0, 1, 0, 0.0]]))
    rc = lib.gw_ctx_create(ctypes.byref(h), f.size, f.ctypes.data, 1, d.ctypes.data, S.ctypes.data, det, 0.0, None, None)
    assert rc in (binding.GW_ERR_CUDA, binding.GW_ERR_ARCH) and not h


def test_binding_rejects_bad_output_buffers():
    """Caller-supplied outputs are validated before their raw pointers reach the library (no GPU needed: the checks
    are static methods of the binding)."""
    from paper_1904_02863_b200.binding import GwContext, GwError
    for bad in (np.empty(7), np.empty(8, dtype=np.float32), np.empty((8, 2))[:, 0], [0.0] * 8):
        with pytest.raises(GwError):
            GwContext._out_host(bad, 8, "out")
    ro = np.empty(8)
    ro.flags.writeable = False
    with pytest.raises(GwError):
        GwContext._out_host(ro, 8, "out")
    assert GwContext._out_host(np.empty(8), 8, "out") is not None
    import torch
    like = torch.empty(1)
    for bad in (torch.empty(8), np.empty(8)):          # CPU tensor / not a tensor
        with pytest.raises(GwError):
            GwContext._out_dev(bad, 8, like, "out")


def test_package_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1904_02863_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), fn
                assert "gw_oracle" not in text, fn
