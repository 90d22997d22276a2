"""The C-ABI library loads on a machine without a GPU and exports every symbol that
include/bytescale_attn.h declares; argument validation works without launching anything."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "bytescale_attn.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(bs_[a-z_0-9]+)\s*\(", text)))


def test_exports_every_declared_symbol():
    from paper_2502_21231_b200 import binding
    syms = declared_symbols()
    assert len(syms) >= 20
    for s in syms:
        assert hasattr(binding.lib, s), s
    assert sorted(binding.EXPORTS) == syms
    assert binding.lib.bs_version() == 100


def test_validation_without_gpu():
    from paper_2502_21231_b200 import binding as b
    sh = b.make_shape(4, 4, 96, 16, 16)  # head_dim 96 unsupported
    with pytest.raises(b.BsError) as e:
        b.attn_workspace_bytes(sh, 1, False)
    assert e.value.code == -2 and "head_dim" in str(e.value)
    sh = b.make_shape(6, 4, 64, 16, 16)  # Hq % Hkv != 0
    with pytest.raises(b.BsError) as e:
        b.attn_workspace_bytes(sh, 1, False)
    assert e.value.code == -1
    sh = b.make_shape(4, 2, 128, 1000, 1000)
    assert b.attn_workspace_bytes(sh, 3, False) >= 256
    assert b.attn_workspace_bytes(sh, 3, True) >= 256
    # null pointers are rejected before any launch
    rc = b.lib.bs_attn_fwd(ctypes.byref(sh), None, None, None, None, 0, 0, 10, None, None, None, 0,
                           None, None)
    assert rc == -1
    rc = b.lib.bs_lse_merge(0, None, None, ctypes.byref(sh), 0, 1, None, None, None)
    assert rc == -1
