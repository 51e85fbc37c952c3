"""CPU-side checks of the C-ABI boundary (include/hpmc.h): the library loads without a GPU, exports every
symbol the header declares, the Python binding marshals the same structs, and -- with no CUDA device -- the
product path fails loudly instead of falling back to anything (no compute call is made here)."""
import ctypes as C
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "hpmc.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)
    return sorted(set(re.findall(r"\b(hpmc_[a-z_0-9]+)\s*\(", src)))


@pytest.fixture(scope="module")
def lib():
    from paper_1508_07077_b200 import build as cuda_build
    cuda_build.build()
    import paper_1508_07077_b200 as hp
    return hp.load_library()


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for n in ("hpmc_init", "hpmc_build_cells", "hpmc_sweep", "hpmc_counters"):
        assert n in names


def test_library_exports_every_declared_symbol(lib):
    from paper_1508_07077_b200 import binding
    names = _declared_functions()
    assert len(names) >= 17
    for n in names:
        assert hasattr(lib, n), "libhpmc_b200.so does not export %s" % n
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS and include/hpmc.h disagree"


def test_struct_layouts_match_header():
    from paper_1508_07077_b200 import binding
    # hpmc_params: int32 + 6 floats; hpmc_counters_t: 13 x uint64, in header order
    assert C.sizeof(binding.Params) == 28
    assert C.sizeof(binding.Counters) == 13 * 8
    src = open(HEADER).read()
    body = src[src.index("typedef struct {\n  uint64_t trials_trans"):src.index("} hpmc_counters_t;")]
    body = re.sub(r"/\*.*?\*/", " ", body, flags=re.S)
    fields = re.findall(r"\b([a-z_]+)\s*[,;]", body)
    assert tuple(fields) == binding.COUNTER_NAMES


def test_signatures_have_no_torch_types():
    src = open(HEADER).read()
    code = re.sub(r"/\*.*?\*/", " ", src, flags=re.S)          # comments may name torch (where a stream comes from)
    assert "torch" not in code.lower()
    assert "at::" not in src and "c10::" not in src and "#include <torch" not in src
    assert 'extern "C"' in src


def test_library_is_sm100a_only():
    so = os.path.join(ROOT, "paper_1508_07077_b200", "libhpmc_b200.so")
    out = subprocess.run(["/usr/local/cuda/bin/cuobjdump", "-lelf", so], capture_output=True, text=True).stdout
    archs = set(re.findall(r"sm_(\d+a?)", out))
    assert archs == {"100a"}, archs


def test_no_gpu_means_loud_failure_not_fallback(lib):
    """Without a CUDA device hpmc_init must return HPMC_E_CUDA with a message; bad arguments are rejected before
    any device work."""
    import torch
    from paper_1508_07077_b200 import binding
    ctx = C.c_void_p()
    p = binding.Params(0, 1.0, 0.0, 0.0, 0.1, 20.0, 0.05)
    assert lib.hpmc_init(C.byref(ctx), None, 10, None, None, None) == -1          # HPMC_E_BADARG
    assert lib.hpmc_init(C.byref(ctx), C.byref(p), 0, None, None, None) == -1
    small = binding.Params(0, 1.0, 0.0, 0.0, 0.1, 4.0, 0.05)
    assert lib.hpmc_init(C.byref(ctx), C.byref(small), 10, None, None, None) == -2  # HPMC_E_GEOMETRY
    flat = binding.Params(3, 1.0, 0.5, 0.1, 0.1, 20.0, 0.05)                        # ellipsoid, aspect ratio 5 > 4
    assert lib.hpmc_init(C.byref(ctx), C.byref(flat), 10, None, None, None) == -1
    assert b"aspect" in lib.hpmc_last_error(None)
    if torch.cuda.is_available():
        pytest.skip("a GPU is present: the no-device branch cannot be exercised")
    rc = lib.hpmc_init(C.byref(ctx), C.byref(p), 10, None, None, None)
    assert rc == -5 and not ctx.value                                             # HPMC_E_CUDA
    assert b"CUDA" in lib.hpmc_last_error(None)
    with pytest.raises(binding.HPMCError):
        import paper_1508_07077_b200 as hp
        hp.HPMC("sphere", 1.0, 0.1, 20.0, 0.05, None, None, N=10)


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1508_07077_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in text.lower(), "%s mentions the oracle" % f
    osrc = open(os.path.join(ROOT, "oracle", "hpmc_oracle.cpp")).read()
    assert "#include \"" not in osrc.replace('#include "omp.h"', ""), "oracle includes a project header"
