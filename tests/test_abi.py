"""The C-ABI library: builds, loads, exports every symbol include/lbm.h declares, and fails loudly without a
GPU.  No compute calls.  CPU only."""
import ctypes
import os
import re

import pytest

import paper_2506_21804_b200 as P
from paper_2506_21804_b200 import binding, build as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return P.load_library()


def _declared():
    text = open(os.path.join(ROOT, "include", "lbm.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(lbm_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree():
    assert _declared() == sorted(binding.EXPORTS)


def test_library_exports_every_declared_symbol(lib):
    for name in _declared():
        assert hasattr(lib, name), name


def test_every_accepted_option_key_is_documented_in_the_header():
    """lbm_set_option: the keys the library compares against (lbm_api.cu) are exactly the keys include/lbm.h lists"""
    api = open(os.path.join(ROOT, "paper_2506_21804_b200", "csrc", "lbm_api.cu")).read()
    body = api[api.index("int lbm_set_option("):]
    accepted = sorted(set(re.findall(r'std::strcmp\(key, "([a-z_]+)"\)', body)))
    header = open(os.path.join(ROOT, "include", "lbm.h")).read()
    doc = header[header.index("/* Tuning knobs"):header.index("int lbm_set_option(")]
    documented = sorted(set(re.findall(r'^ \*   "([a-z_]+)"', doc, flags=re.M)))
    assert accepted == documented and len(accepted) >= 7, (accepted, documented)


def test_params_struct_layout_matches_header(tmp_path):
    """the ctypes mirror against the C compiler's view of include/lbm.h (offsetof / sizeof printed by a gcc-built probe)"""
    import subprocess
    S = P.LbmParams
    names = [f for f, _ in S._fields_]
    assert names == ["tau0", "cs_smago", "use_hlbm", "u_in", "wm_enable", "wm_kappa", "wm_E", "collision", "sigma", "u_wall", "rho_out", "fringe_len", "fringe_factor"]
    src = tmp_path / "probe.c"
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "lbm.h"\nint main(void){printf("%zu", sizeof(lbm_params));'
                   + "".join('printf(" %%zu", offsetof(lbm_params, %s));' % n for n in names) + "return 0;}\n")
    exe = tmp_path / "probe"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = [int(t) for t in subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout.split()]
    assert ctypes.sizeof(S) == out[0] == 136
    assert [getattr(S, f).offset for f in names] == out[1:] == [0, 8, 16, 24, 48, 56, 64, 72, 80, 88, 112, 120, 128]


def test_bad_arguments_are_rejected_without_touching_the_gpu(lib):
    for args in [(18, 8, 8, 8, 4), (19, 8, 8, 8, 2), (19, 0, 8, 8, 4), (19, 2048, 2048, 2048, 4)]:
        with pytest.raises(P.LbmError):
            P.lbm_create(*args)
        assert "lbm_create" in P.lbm_last_error(None)
    assert lib.lbm_query(None, 0) == -1
    assert lib.lbm_step(None, 1, None) == binding.LBM_EINVAL
    lib.lbm_destroy(None)


def test_no_cpu_fallback_when_no_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(P.LbmError) as e:
        P.lbm_create(19, 8, 8, 8, 4)
    assert "no usable CUDA device" in str(e.value)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2506_21804_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in text.replace("oracle/", "").replace("the oracle", "").lower() or \
                    not re.search(r"^\s*(from|import)\s+oracle|#include\s+\".*oracle", text, flags=re.M), fn
    otext = open(os.path.join(ROOT, "oracle", "oracle.py")).read() + open(os.path.join(ROOT, "oracle", "lbm_oracle.cpp")).read()
    assert not re.search(r"^\s*(from|import)\s+paper_2506_21804_b200|#include\s+\".*(lbm\.h|lbm_kernels)", otext, flags=re.M)
