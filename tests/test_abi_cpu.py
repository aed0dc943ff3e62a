"""CPU-side checks of the C-ABI boundary: the shared library builds/loads, exports every symbol that
include/dns.h declares, and validates arguments before touching CUDA (no compute calls without a GPU)."""
import ctypes
import os
import re

import pytest

from paper_2306_12739_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def declared_functions():
    """Every function include/*.h declares: the product ABI (dns.h) and the test / measurement hooks (dns_debug.h)."""
    names = set()
    for h in ("dns.h", "dns_debug.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(dns_[a-z0-9_]+)\s*\(", src))
    names.discard("dns_exchange_fn")
    return sorted(names)


def test_debug_hooks_are_not_in_the_product_header():
    src = open(os.path.join(ROOT, "include", "dns.h")).read()
    assert "dns_debug_" not in re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    for f in os.listdir(os.path.join(ROOT, "paper_2306_12739_b200", "csrc")):
        assert "getenv" not in open(os.path.join(ROOT, "paper_2306_12739_b200", "csrc", f)).read(), f


def test_header_and_binding_agree(lib):
    decl = declared_functions()
    assert "dns_plan_create" in decl and "dns_step" in decl and "dns_diagnostics" in decl
    assert sorted(binding.EXPORTS) == decl
    for name in decl:
        assert hasattr(lib, name), name               # dlsym succeeds
        assert callable(getattr(binding, name)), name  # same name in the Python binding


def test_strerror(lib):
    assert binding.dns_strerror(0) == "ok"
    assert "invalid" in binding.dns_strerror(binding.DNS_EINVAL)
    assert "CUDA" in binding.dns_strerror(binding.DNS_ECUDA)
    assert binding.dns_strerror(12345) == "unknown status"


@pytest.mark.parametrize("args", [
    (15, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 0),     # odd Nx
    (16, 33, 14, 2, 400.0, 5.0, 3.0, 0.02, 0),     # Mz = 21 is not 2^a 3^b
    (8, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 0),      # Mx = 12 < 16
    (96, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 0),     # Mx = 144 > 128
    (16, 4, 16, 2, 400.0, 5.0, 3.0, 0.02, 0),      # Ny < 5
    (16, 33, 16, 0, 400.0, 5.0, 3.0, 0.02, 0),     # E < 1
    (16, 33, 16, 2, -1.0, 5.0, 3.0, 0.02, 0),      # Re <= 0
    (16, 33, 16, 2, 400.0, 0.0, 3.0, 0.02, 0),     # Lx <= 0
    (16, 33, 16, 2, 400.0, 5.0, 3.0, float("nan"), 0),
    (16, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 7),     # unknown flow
])
def test_plan_create_rejects_bad_arguments(lib, args):
    st, h = binding.dns_plan_create(*args)
    assert st == binding.DNS_EINVAL and not h.value


def test_null_handles_are_rejected(lib):
    assert lib.dns_plan_create(None, 16, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 0) == binding.DNS_EINVAL
    null = ctypes.c_void_p()
    assert binding.dns_plan_workspace_bytes(null) == 0
    assert binding.dns_step(null, 1) == binding.DNS_EINVAL
    assert binding.dns_plan_bind(null, 0, 0) == binding.DNS_EINVAL
    assert binding.dns_launches_per_step(null) == 0
    assert binding.dns_plan_destroy(null) == binding.DNS_OK


def test_no_cpu_fallback_without_a_device(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    st, h = binding.dns_plan_create(16, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 0)
    assert st == binding.DNS_ECUDA and not h.value
    with pytest.raises(binding.DnsError):
        binding.Plan(16, 33, 16, 2, 400.0, 5.0, 3.0, 0.02, 0)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2306_12739_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    txt = open(os.path.join(ROOT, "oracle", "dns_oracle.py")).read()
    assert "import paper_2306" not in txt and "from paper_2306" not in txt
