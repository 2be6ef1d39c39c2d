"""The C-ABI boundary without a GPU: libsoap_b200.so loads, exports every function include/soap_b200.h declares,
the binding knows them all, and the product path fails loudly (no CPU fallback) when there is no CUDA device."""
from __future__ import annotations

import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "soap_b200.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(soap_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_function():
    import paper_2301_04259_b200 as soap
    lib = soap.binding.load_library()
    names = _declared()
    assert len(names) >= 15 and "soap_disk_geometry" in names and "soap_integrate_quiet" in names and "soap_active_timeseries" in names
    for n in names:
        assert hasattr(lib, n), f"{n} is declared in include/soap_b200.h but not exported"
    assert set(names) == set(soap.binding.EXPORTED_SYMBOLS), set(names) ^ set(soap.binding.EXPORTED_SYMBOLS)
    assert lib.soap_version() >= 100


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    import paper_2301_04259_b200 as soap
    lib = soap.binding.load_library()
    h = ctypes.c_void_p()
    rc = lib.soap_create(ctypes.byref(h), 0)
    assert rc == soap.binding.SOAP_ERR_CUDA and not h.value
    assert b"no CPU fallback" in lib.soap_last_error(None)
    with pytest.raises(soap.SoapError):
        soap.soap_create(0)


def test_product_package_does_not_import_the_oracle():
    import subprocess
    import sys
    code = "import sys; import paper_2301_04259_b200; import workloads; print(int(any(m == 'oracle' or m.startswith('oracle.') for m in sys.modules)))"
    out = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, cwd=ROOT)
    assert out.returncode == 0 and out.stdout.strip() == "0", out.stderr[-500:]
