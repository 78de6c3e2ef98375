"""CPU-only: the C-ABI library loads without a GPU and exports every symbol include/ibp.h declares."""
import ctypes
import re
from pathlib import Path

import pytest

from paper_2605_30728_b200 import _build
from paper_2605_30728_b200 import binding as ibp

ROOT = Path(__file__).resolve().parent.parent


def _declared():
    text = (ROOT / "include" / "ibp.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ibp_[a-z0-9_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported_and_bound():
    names = _declared()
    assert "ibp_build" in names and "ibp_gather_decompress" in names and "ibp_decompress_resident" in names \
        and "ibp_upload_metadata" in names
    L = ctypes.CDLL(str(_build.build_library()))
    for n in names:
        assert hasattr(L, n), f"{n} declared in ibp.h but not exported by libibp.so"
    assert sorted(ibp.SIGNATURES) == names, "binding.SIGNATURES and ibp.h disagree"


def test_struct_sizes_match_header():
    # the C side checks struct_size at run time: a mismatch makes ibp_build fail, so a successful build proves it
    import numpy as np
    h = ibp.ibp_build(np.zeros((4, 8), np.uint8), 8, 0, 2, flags=ibp.IBP_FLAG_PAGEABLE_STORE)
    assert h.info().n_groups == 2 and h.info().row_bytes == 8 and h.info().device == -1
    h.destroy()
    assert "sm_100a" in ibp.ibp_version()


def test_hot_path_fails_loudly_without_gpu():
    import numpy as np
    try:
        import torch
        if torch.cuda.is_available():
            pytest.skip("GPU present")
    except ImportError:
        pass
    h = ibp.ibp_build(np.zeros((4, 8), np.uint8), 8, 0, 2)
    with pytest.raises(ibp.IbpError) as e:
        h.upload_metadata(0)
    assert e.value.status == 3                                   # IBP_ERR_CUDA: there is no CPU fallback
    h.destroy()
