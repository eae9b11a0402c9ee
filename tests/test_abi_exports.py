"""C ABI (include/manta.h) without a GPU: the library loads, exports every function the header declares, the Python
binding names the same set, argument checks that need no device work, and there is no CPU fallback."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "manta.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^(?:int|void|uint64_t|const char \*)\s*\**\s*(manta_\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_2007_03614_b200 import binding, build
    build.build_all()
    return binding.load_library()


def test_header_declares_the_four_calls_of_the_boundary():
    names = declared_functions()
    for n in ("manta_create", "manta_load_trips", "manta_step", "manta_readback", "manta_destroy", "manta_last_error"):
        assert n in names
    assert len(names) >= 12


def test_library_exports_every_declared_symbol(lib):
    from paper_2007_03614_b200 import binding
    names = declared_functions()
    missing = [n for n in names if not hasattr(lib, n)]
    assert not missing, missing
    assert set(binding.EXPORTS) == set(names)        # the binding names exactly the header's functions


def test_null_handle_is_rejected_without_touching_the_device(lib):
    from paper_2007_03614_b200 import binding
    lib.manta_step.restype = C.c_int
    lib.manta_step.argtypes = [C.c_void_p, C.c_uint32]
    assert lib.manta_step(None, 1) == binding.ERR_INVALID_ARG
    lib.manta_sync.restype = C.c_int
    lib.manta_sync.argtypes = [C.c_void_p]
    assert lib.manta_sync(None) == binding.ERR_INVALID_ARG
    lib.manta_last_error.restype = C.c_char_p
    lib.manta_last_error.argtypes = [C.c_void_p]
    assert b"null" in lib.manta_last_error(None)


def test_no_cpu_fallback():
    """Without a CUDA device the product path fails loudly (MANTA_ERR_CUDA / an exception), it never computes."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2007_03614_b200 import binding, workloads as wl
    net = wl.straight_road(n_edges=2, length_m=50.0)
    with pytest.raises(Exception):
        binding.Sim(net)
    # and nothing of the package imports the oracle
    import paper_2007_03614_b200
    pkg = os.path.dirname(paper_2007_03614_b200.__file__)
    for f in os.listdir(pkg):
        if f.endswith(".py"):
            txt = open(os.path.join(pkg, f)).read()
            assert not re.search(r"^\s*(from|import)\s+oracle|manta_oracle|libmanta_oracle", txt, flags=re.M), f
