"""CPU-only checks of the boundary: the C-ABI library loads without a GPU and exports every symbol
include/optflow.h declares; the binding declares exactly those; argument errors are reported."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "optflow.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(of_[a-z0-9_]+)\s*\(", text)))


@pytest.fixture(scope="module")
def binding():
    from paper_1306_2461_b200 import build, binding as b
    build.build()
    return b


def test_header_symbols_are_exported_and_bound(binding):
    syms = declared_symbols()
    assert "of_create" in syms and "of_compute" in syms and "of_destroy" in syms
    L = binding.lib()
    for s in syms:
        assert hasattr(L, s), "liboptflow.so does not export %s" % s
    assert sorted(binding.SIGNATURES) == syms


def test_no_torch_types_and_extern_c():
    text = open(os.path.join(ROOT, "include", "optflow.h")).read()
    assert 'extern "C"' in text and "torch" not in text.lower() and "at::" not in text


def test_argument_errors_without_gpu(binding):
    L = binding.lib()
    assert not L.of_create(0, 10, 1, 1, 1, 0)
    assert "bad image size" in binding.last_error()
    assert not L.of_create(64, 64, 3, 8, 1, 0)          # coarsest level 16x16 < 17
    assert "coarsest" in binding.last_error()
    assert not L.of_create(64, 64, 1, 40, 1, 0)
    assert L.of_compute(None, None, None, None, None, None) < 0
    assert L.of_stream_submit(None) < 0
    L.of_destroy(None)


def test_product_path_has_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.OptflowError):
        binding.OpticalFlow(64, 64, 1, 4, 1, 0)
    # of_create itself fails loudly without a device
    assert not binding.lib().of_create(64, 64, 1, 4, 1, 0)
    assert binding.last_error() != ""


def test_package_does_not_import_oracle():
    import subprocess, sys
    code = ("import sys; sys.path.insert(0, %r); import paper_1306_2461_b200.binding, "
            "paper_1306_2461_b200.synthetic, paper_1306_2461_b200.build; "
            "assert not any(m.startswith('oracle') for m in sys.modules), 'product imports oracle'") % ROOT
    subprocess.check_call([sys.executable, "-c", code])
    for f in ("binding.py", "synthetic.py", "build.py", "csrc/optflow.cu", "csrc/of_kernels.cuh"):
        src = open(os.path.join(ROOT, "paper_1306_2461_b200", f)).read()
        assert "import oracle" not in src and "from oracle" not in src and "optflow_oracle" not in src
