"""No-GPU checks of the boundary: the library loads, exports every symbol include/zfac.h
declares, and its host-only entry points behave.  No compute call is made here."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def binding():
    from paper_2404_19163_b200 import build, binding as b
    build.build()                      # cross-compiles for sm_100a; no GPU needed
    return b


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "zfac.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(zfac_[a-z_0-9]+)\s*\(", src)))


def test_header_symbols_are_exported(binding):
    names = _declared_functions()
    assert len(names) >= 10
    L = binding.lib()
    for n in names:
        assert hasattr(L, n), f"libzfac.so does not export {n}"
    assert sorted(binding.EXPORTS) == names       # the Python layer carries the same names


def test_host_only_entry_points(binding):
    b = binding
    assert b.zfac_padded_n(4617, b.ZFAC_MODE_SPLIT16) == 4864       # tile 256 (tcgen05 modes)
    assert b.zfac_padded_n(4617, b.ZFAC_MODE_F64) == 4736           # tile 128 (DMMA mode)
    assert b.zfac_padded_n(256, b.ZFAC_MODE_TF32) == 256
    assert b.zfac_workspace_bytes(0, b.ZFAC_MODE_F64) == 0
    assert b.zfac_workspace_bytes(100, 9) == 0
    for mode, elt in ((b.ZFAC_MODE_F64, 8), (b.ZFAC_MODE_TF32, 4), (b.ZFAC_MODE_SPLIT16, 4)):
        n = 1000
        npad = b.zfac_padded_n(n, mode)
        ws = b.zfac_workspace_bytes(n, mode)
        assert ws > 7 * npad * npad * elt                # S, W, T, R, Q, Z x2 (+ pairs in SPLIT16)
        assert ws < 12 * npad * npad * elt + (1 << 22)
    assert "WORKSPACE" in b.zfac_status_string(b.ZFAC_E_WORKSPACE)
    assert "no fallback" in b.zfac_status_string(b.ZFAC_E_UNSUPPORTED)


def test_create_rejects_bad_arguments_before_touching_a_device(binding):
    b = binding
    with pytest.raises(b.ZfacError) as e:
        b.zfac_create(0, b.ZFAC_MODE_F64, 0, 0)
    assert e.value.status == b.ZFAC_E_INVALID
    with pytest.raises(b.ZfacError) as e:
        b.zfac_create(64, b.ZFAC_MODE_F64, 0, 1 << 30)          # null workspace
    assert e.value.status == b.ZFAC_E_WORKSPACE


def test_product_path_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing in the package may import it."""
    pkg = os.path.join(ROOT, "paper_2404_19163_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in txt.replace("no oracle", "").replace("No oracle", "").lower() or f == "workloads.py", f
    txt = open(os.path.join(ROOT, "oracle", "zfac_oracle.py")).read()
    assert "paper_2404_19163_b200" not in txt.split('"""')[2]


def test_no_gpu_means_loud_failure(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        binding.Zfac(64, "f64")


def test_header_is_c99_and_a_plain_c_consumer_links(binding, tmp_path):
    """include/zfac.h is a C header (no C++ in it) and a C99 program that calls the ABI links against libzfac.so
    (tests/abi_consumer.c; the GPU suite runs it)."""
    import subprocess
    res = subprocess.run(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-fsyntax-only", "-x", "c",
                          os.path.join(ROOT, "include", "zfac.h")], capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    from abi_build import compile_consumer
    assert os.path.exists(compile_consumer(str(tmp_path / "abi_consumer")))


def test_library_reads_no_environment_variable():
    """Behaviour is set through zfac_set_option only (include/zfac.h): no hidden process-global state."""
    csrc = os.path.join(ROOT, "paper_2404_19163_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f
