"""The C-ABI library builds for sm_100a, loads without a GPU and exports every symbol include/*.h declares."""
import ctypes
import os
import re

from paper_2501_05993_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    syms = set()
    inc = os.path.join(ROOT, "include")
    for name in sorted(os.listdir(inc)):
        text = open(os.path.join(inc, name)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        syms |= set(re.findall(r"\b(pcal_[a-z0-9_]+)\s*\(", text))
    return sorted(syms)


def test_probes_are_not_in_the_product_header():
    text = open(os.path.join(ROOT, "include", "pcal.h")).read()
    for name in ("pcal_read_probe", "pcal_pipe_probe", "pcal_set_profiling", "pcal_get_profile"):
        assert name not in text


def test_library_builds_loads_and_exports_every_declared_symbol():
    path = binding.build()
    assert os.path.exists(path)
    L = ctypes.CDLL(path)
    syms = declared_symbols()
    assert len(syms) >= 16, syms
    for s in syms:
        assert hasattr(L, s), f"{s} declared in include/ but not exported"
    # the binding wires exactly the declared entry points
    binding.lib()
    L.pcal_strerror.restype = ctypes.c_char_p
    assert L.pcal_strerror(0) == b"ok"
    assert b"aligned" in L.pcal_strerror(-2)


def test_library_is_sm100a_native():
    out = os.popen(f"cuobjdump -lelf {binding.build()} 2>/dev/null").read()
    assert "sm_100a" in out, out


def test_no_fallback_without_gpu():
    """Without a CUDA device pcal_create must fail loudly (PCAL_ERR_DEVICE), never compute on the CPU."""
    import torch
    if torch.cuda.is_available():
        return
    import pytest
    with pytest.raises(binding.PcalError) as e:
        binding.Pcal(32e6, 1e6, 0.0, 32, binding.ENC_IEEE_FLOAT, 1)
    assert e.value.code == -5
