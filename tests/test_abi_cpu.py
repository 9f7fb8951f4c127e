"""CPU-side checks of the boundary: the library loads and exports every symbol best.h declares,
and entry points fail loudly (no CPU fallback) when there is no device."""
import os
import re

import numpy as np
import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "best.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(best_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import __graft_entry__ as entry
    entry.build()
    from paper_2606_04895_b200 import binding
    L = binding.lib()
    names = _declared_functions()
    assert len(names) >= 18
    for n in names:
        assert hasattr(L, n), f"libbest.so does not export {n}"
    assert sorted(binding.EXPORTS) == names
    assert "sm_100a" in binding.version()


def test_argument_errors_need_no_gpu():
    from paper_2606_04895_b200 import binding, workloads as WL
    w = WL.tiny()
    w.d = 40                                   # out of range ⇒ BEST_ERR_ARG before any CUDA call
    with pytest.raises(binding.BestError) as e:
        binding.Context(w)
    assert e.value.code == binding.BEST_ERR_ARG
    w = WL.tiny()
    w.Sigma_inv = -np.eye(w.d)                 # not SPD
    with pytest.raises(binding.BestError) as e:
        binding.Context(w)
    assert e.value.code == binding.BEST_ERR_NOT_SPD
    w = WL.tiny()
    w.L = np.zeros((w.d, w.d))
    with pytest.raises(binding.BestError) as e:
        binding.Context(w)
    assert e.value.code == binding.BEST_ERR_NOT_SPD


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful without a GPU")
def test_no_cpu_fallback():
    from paper_2606_04895_b200 import binding, workloads as WL
    with pytest.raises(binding.BestError) as e:
        binding.Context(WL.tiny())
    assert e.value.code == binding.BEST_ERR_CUDA
    assert "no CPU fallback" in str(e.value)


def test_probe_argument_errors_need_no_gpu():
    from paper_2606_04895_b200 import binding
    for bad in ((1 << 19, 10), (200 << 20, 10), (16 << 20, 0)):
        with pytest.raises(binding.BestError) as e:
            binding.probe_l2_read(*bad)
        assert e.value.code == binding.BEST_ERR_ARG
