"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every symbol include/sc_ivr.h declares.
No compute calls here (no GPU on the CPU box)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "sc_ivr.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sc_ivr_[a-z0-9_]+)\s*\(", src)))


def test_library_builds_loads_and_exports_the_header():
    from paper_1312_4698_b200 import binding, build
    path = build.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    names = _declared()
    assert "sc_ivr_create" in names and "sc_ivr_run" in names and "sc_ivr_propagate" in names
    for n in names:
        assert hasattr(L, n), f"{n} is declared in include/sc_ivr.h but not exported"
    assert sorted(binding.EXPORTS) == names
    binding.lib()


def test_create_fails_loudly_without_a_device_or_with_bad_arguments():
    """No CPU fallback: without a CUDA device create returns SC_IVR_ECUDA; bad arguments are EINVAL either way."""
    import numpy as np
    import pytest
    from paper_1312_4698_b200 import binding
    with pytest.raises(binding.ScIvrError) as e:
        binding.ScIvr(1, binding.PES_MORSE1D, [0.17, 1.0, 1.4], [18.0], 10.0, 100)  # 3 coefficients instead of 4
    assert e.value.status == binding.EINVAL
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(binding.ScIvrError) as e:
            binding.ScIvr(1, binding.PES_MORSE1D, np.array([0.17, 1.0, 1.4, 918.0]), [18.0], 10.0, 100)
        assert e.value.status == binding.ECUDA and "no CPU fallback" in str(e.value)
