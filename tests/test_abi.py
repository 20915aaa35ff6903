"""CPU-side checks of the boundary: libteuk.so loads, exports every symbol include/teuk.h declares,
fails loudly without a GPU, and the product never touches oracle/."""
import ctypes
import os
import re
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PKG = os.path.join(ROOT, "paper_1206_0270_b200")


@pytest.fixture(scope="module")
def lib_path():
    from paper_1206_0270_b200 import build
    return build.build()


def _declared():
    text = open(os.path.join(ROOT, "include", "teuk.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(teuk_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported(lib_path):
    names = _declared()
    assert {"teuk_create", "teuk_set_initial", "teuk_set_source", "teuk_step", "teuk_extract"} <= set(names)
    lib = ctypes.CDLL(lib_path)
    for n in names:
        assert hasattr(lib, n), n
    from paper_1206_0270_b200 import teuk
    assert sorted(teuk.SYMBOLS) == names


def test_library_is_sm100a_and_has_the_kernels(lib_path):
    out = subprocess.run(["cuobjdump", "-lelf", lib_path], capture_output=True, text=True)
    if out.returncode != 0:
        pytest.skip("cuobjdump unavailable")
    assert "sm_100a" in out.stdout


def test_create_fails_loudly_without_gpu(lib_path):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_1206_0270_b200 import teuk
    with pytest.raises(teuk.TeukError) as e:
        teuk.Solver(0.0, 1.0, [2], -50.0, 150.0, 64, 32, 0.01)
    assert e.value.code == teuk.TEUK_ECUDA and "no CPU fallback" in str(e.value)


def test_every_option_and_stat_key_is_documented_in_the_header():
    """include/teuk.h is the contract: each key teuk_set_option / teuk_get_stat accepts must be described there."""
    src = open(os.path.join(PKG, "csrc", "teuk_api.cu")).read()
    header = open(os.path.join(ROOT, "include", "teuk.h")).read()
    opt = src[src.index("int teuk_set_option("):src.index("int teuk_get_stat(")]
    stat = src[src.index("int teuk_get_stat("):]
    keys = set(re.findall(r'strcmp\(key, "([a-z_0-9]+)"\)', opt)) | set(re.findall(r'strcmp\(key, "([a-z_0-9]+)"\)', stat))
    assert {"outer_bc", "kernel", "slab_rows", "pdl", "resident_cache", "steps", "launches"} <= keys
    for k in sorted(keys):
        assert '"%s"' % k in header, "option / counter %r is not documented in include/teuk.h" % k


def test_product_never_references_the_oracle():
    for dirpath, _, files in os.walk(PKG):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle", text, flags=re.M), f
                assert "liboracle" not in text and "orc_" not in text, f
                assert "oracle" not in text.lower(), "%s mentions the oracle: the product has no path shaped around it" % f
                assert "TEUK_LIB" not in text, "%s: no library override in the product" % f
    code = "import sys; import paper_1206_0270_b200; assert not any(m.startswith('oracle') for m in sys.modules)"
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
    oracle_src = open(os.path.join(ROOT, "oracle", "teuk_oracle.cpp")).read()
    assert "paper_1206_0270_b200" not in oracle_src.replace("paper_1206_0270_b200/csrc and neither", "")
    assert "import paper_1206_0270_b200" not in open(os.path.join(ROOT, "oracle", "oracle.py")).read()
