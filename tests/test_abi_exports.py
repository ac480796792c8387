"""CPU-only: the C-ABI library builds/loads and exports every symbol include/pic.h declares
(no compute calls without a GPU); struct layouts of the binding match the header's sizes."""
import ctypes as C
import os
import re

from paper_1111_5295_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "pic.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pic_[a-z_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported():
    names = _declared()
    assert "pic_init" in names and "pic_move_accumulate" in names and "pic_residual" in names
    L = B.load()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(B.EXPORTS) == names


def test_struct_sizes():
    assert C.sizeof(B.PicGrid) == 16
    assert C.sizeof(B.PicSpecies) == 24
    assert C.sizeof(B.PicParams) == 48
    assert C.sizeof(B.PicStats) == 80
    assert C.sizeof(B.PicJfnkOpts) == 48
    assert C.sizeof(B.PicJfnkInfo) == 40


def test_no_cpu_fallback():
    """Without a CUDA device pic_init must fail loudly (PIC_ERR_CUDA), never compute."""
    import numpy as np
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(B.PicError) as ei:
        B.Pic(4, 4.0, [dict(q_over_m=-1.0, w_q=-1.0, x=np.array([0.5]), v=np.array([1.0]))])
    assert ei.value.code == -2


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1111_5295_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "pic_oracle" not in txt, f
