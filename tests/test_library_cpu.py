"""CPU-side checks of the boundary (-m "not gpu"): the C-ABI library builds, loads, and exports every
symbol include/sdm.h declares; host-only entry points behave; the product path fails loudly (no CPU
fallback) when there is no CUDA device.  No compute call is made here."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2103_17238_b200 import _build, binding
    _build.build()
    return binding.load_library()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sdm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sdm_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_all_exported(lib):
    from paper_2103_17238_b200 import binding
    names = _declared_symbols()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/sdm.h but not exported"
    assert sorted(binding.EXPORTS) == names


def test_workspace_bytes_host_only(lib):
    from paper_2103_17238_b200 import workspace_bytes, host_staging_bytes
    a = workspace_bytes(8192, 1)
    b = workspace_bytes(2 ** 23, 2 ** 16)
    assert 0 < a < b
    # two 8-byte ping-pong buffers and the two 8-byte resident copies of a HYBRID run dominate: between 32 and 40 bytes
    # per super-droplet at scale
    assert 32 * 2 ** 23 <= b <= 40 * 2 ** 23
    assert workspace_bytes(-1, 1) == 0
    assert workspace_bytes(2 ** 30, 1) == 0
    assert workspace_bytes(10, 0) == 0
    assert host_staging_bytes(1000) >= 20 * 1000
    assert host_staging_bytes(-5) == 0


def test_strerror_and_null_handling(lib):
    assert lib.sdm_strerror(0) == b"ok"
    assert b"invalid" in lib.sdm_strerror(-1)
    assert lib.sdm_launch_count(None) == 0
    assert lib.sdm_last_path(None) == 0
    assert lib.sdm_set_path(None, 0) == -1
    assert lib.sdm_poll_error(None) == -1
    out = C.c_void_p()
    assert lib.sdm_init(C.byref(out), 0, 100, 1, None, 0, None) == -1          # null workspace
    assert lib.sdm_init(None, 0, 100, 1, None, 0, None) == -1


def test_no_cpu_fallback_without_cuda(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2103_17238_b200 as sdm
    with pytest.raises(sdm.SDMError):
        sdm.SDMContext(1024, 1)
    # straight through the C ABI: a plausible workspace pointer but no device -> SDM_ERR_CUDA
    out = C.c_void_p()
    fake = C.c_void_p(1 << 20)
    assert lib.sdm_init(C.byref(out), 0, 100, 1, fake, 1 << 30, None) == -3
    assert not out.value


def test_static_entry_point_host_side_checks(lib):
    """sdm_remove_zero_multiplicity_static validates on the host before it touches CUDA: the size limit of its fixed
    scratch array, negative sizes and null pointers are refused with their own codes (no device needed, nothing is
    dereferenced)."""
    limit = lib.sdm_static_max_n_sd()
    assert limit == 2 ** 26
    fake = C.c_void_p(1 << 20)
    f = lib.sdm_remove_zero_multiplicity_static
    assert f(fake, fake, fake, limit + 1, fake, None) == -5            # SDM_ERR_STATIC_LIMIT
    assert f(fake, fake, fake, -1, fake, None) == -1                   # SDM_ERR_INVALID_ARG
    assert f(fake, fake, fake, 10, None, None) == -1                   # no place for the result
    assert f(None, fake, fake, 10, fake, None) == -1
    assert b"2^26" in lib.sdm_strerror(-5)


def test_product_package_does_not_import_oracle():
    """The product path must not route through the oracle (nor the oracle through the product)."""
    for sub in ("paper_2103_17238_b200", "sdm_workloads"):
        for dirpath, _, files in os.walk(os.path.join(ROOT, sub)):
            for f in files:
                if f.endswith((".py", ".cu", ".cuh", ".h")):
                    src = open(os.path.join(dirpath, f)).read()
                    assert not re.search(r"^\s*(import|from)\s+oracle\b", src, flags=re.M), (dirpath, f)
                    assert "oracle/" not in src.replace("oracle/:", "") or f.endswith((".cu", ".cuh", ".h", ".py")) and \
                        not re.search(r"#include\s+\"[^\"]*oracle", src), (dirpath, f)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+(paper_2103_17238_b200|sdm_workloads)\b", src, flags=re.M)
            assert "csrc" not in src or f.endswith(".cpp")
