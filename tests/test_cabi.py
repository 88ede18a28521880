"""CPU-side checks of the boundary: the C-ABI library builds, loads, exports every symbol that
include/nolsm.h declares, and the binding's structs match the header. No compute calls (no GPU here)."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2205_12182_b200 import build, load_library
    build.build()
    return load_library()


def _declared_functions():
    text = open(os.path.join(ROOT, "include", "nolsm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(nolsm_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared_functions()
    assert {"nolsm_create", "nolsm_assemble", "nolsm_density_matrix", "nolsm_energy", "nolsm_destroy"} <= set(names)
    for n in names:
        assert hasattr(lib, n), f"{n} declared in nolsm.h but not exported"


def test_option_and_stats_structs_match_header():
    from paper_2205_12182_b200 import NolsmOptions, NolsmStats
    text = open(os.path.join(ROOT, "include", "nolsm.h")).read()
    opt = re.search(r"typedef struct \{(.*?)\} nolsm_options;", text, flags=re.S).group(1)
    opt = re.sub(r"/\*.*?\*/", "", opt, flags=re.S)
    fields = [m.group(1) for m in re.finditer(r"\b([a-z_0-9]+)(?:\[\d+\])?\s*;", opt)]
    assert fields == [f for f, _ in NolsmOptions._fields_]
    st = re.search(r"typedef struct \{((?:(?!typedef).)*?)\} nolsm_stats;", text, flags=re.S).group(1)
    st = re.sub(r"/\*.*?\*/", "", st, flags=re.S)
    names = []
    for decl in st.split(";"):
        decl = decl.strip()
        if decl:
            names += [x.strip() for x in decl.split(None, 1)[1].split(",")]
    assert names == [f for f, _ in NolsmStats._fields_]


def test_abi_version_and_struct_sizes_are_checked_at_load(lib):
    """The library reports its ABI version and its own sizeof of both structs; the binding compares them at load time and
    refuses a mismatch (a stale libnolsm.so would otherwise misread the options silently)."""
    from paper_2205_12182_b200 import NolsmOptions, NolsmStats, binding
    text = open(os.path.join(ROOT, "include", "nolsm.h")).read()
    assert int(re.search(r"#define NOLSM_ABI_VERSION (\d+)", text).group(1)) == binding.ABI_VERSION == lib.nolsm_abi_version()
    assert lib.nolsm_sizeof_options() == ctypes.sizeof(NolsmOptions)
    assert lib.nolsm_sizeof_stats() == ctypes.sizeof(NolsmStats)

    class Stale:
        def __init__(self, version, so, ss):
            self.nolsm_abi_version = ctypes.CFUNCTYPE(ctypes.c_int)(lambda: version)
            self.nolsm_sizeof_options = ctypes.CFUNCTYPE(ctypes.c_size_t)(lambda: so)
            self.nolsm_sizeof_stats = ctypes.CFUNCTYPE(ctypes.c_size_t)(lambda: ss)

    so, ss = ctypes.sizeof(NolsmOptions), ctypes.sizeof(NolsmStats)
    binding._check_abi(Stale(binding.ABI_VERSION, so, ss), "x.so")
    for bad in (Stale(binding.ABI_VERSION - 1, so, ss), Stale(binding.ABI_VERSION, so - 4, ss), Stale(binding.ABI_VERSION, so, ss + 8)):
        with pytest.raises(ImportError, match="stale"):
            binding._check_abi(bad, "x.so")
    with pytest.raises(ImportError, match="predates"):
        binding._check_abi(object(), "x.so")


def test_create_fails_loudly_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2205_12182_b200 import Nolsm, NolsmError
    with pytest.raises(NolsmError):
        Nolsm(0)


def test_null_arguments_are_rejected(lib):
    assert lib.nolsm_create(None, 0, None) == 1
    assert lib.nolsm_destroy(None) == 1
    e = ctypes.c_double()
    assert lib.nolsm_energy(None, ctypes.byref(e)) == 1
    assert lib.nolsm_last_error(None) == b"null context"


def test_product_path_does_not_touch_the_oracle():
    """The package must not import, link or execute anything under oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_2205_12182_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read().lower(), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            assert "paper_2205_12182_b200" not in open(os.path.join(ROOT, "oracle", f)).read().replace(
                "(paper_2205_12182_b200/)", "")
