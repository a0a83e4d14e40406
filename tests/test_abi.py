"""CPU-side checks of the C-ABI boundary (no GPU): the library builds for sm_100a, exports
every symbol include/hhrr.h declares, sizes its workspace, and fails loudly -- never falls
back -- when there is no CUDA device."""
import ctypes as C
import re
import subprocess
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def built():
    from paper_2510_13726_b200 import build
    return build.build()


def _declared():
    text = (ROOT / "include" / "hhrr.h").read_text()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(hhrr_[a-z_0-9]+)\s*\(", text)))


def test_header_and_binding_agree():
    from paper_2510_13726_b200 import binding
    assert _declared() == sorted(binding.SYMBOLS)


def _libraries(built):
    from paper_2510_13726_b200 import build
    assert build.LIBS[27] == built
    return list(build.LIBS.items())     # D3Q27 (libhhrr.so) and D3Q19 (libhhrr_q19.so): same ABI, same sources


def test_library_exports_every_declared_symbol(built):
    for q, path in _libraries(built):
        out = subprocess.run(["nm", "-D", "--defined-only", str(path)], capture_output=True, text=True, check=True).stdout
        exported = set(re.findall(r"\bT (hhrr_[a-z_0-9]+)$", out, flags=re.M))
        assert set(_declared()) <= exported, (q, set(_declared()) - exported)


def test_library_is_sm100a_with_lineinfo(built):
    for q, path in _libraries(built):
        out = subprocess.run(["cuobjdump", "-lelf", str(path)], capture_output=True, text=True).stdout
        assert "sm_100a" in out, q


def test_velocity_set_of_each_build(built):
    from paper_2510_13726_b200 import binding as B
    assert B.lib(27).hhrr_velocity_set() == 27 and B.lib(19).hhrr_velocity_set() == 19
    assert b"D3Q27" in B.lib(27).hhrr_version() and b"D3Q19" in B.lib(19).hhrr_version()
    p = B.make_params(128, 64, 64)
    assert B.workspace_bytes(p, q=19) < B.workspace_bytes(p, q=27)    # 19 instead of 27 planes per buffer


def test_workspace_bytes_and_argument_errors(built):
    from paper_2510_13726_b200 import binding as B
    p = B.make_params(768, 384, 364)
    n = 768 * 384 * 364
    nb = B.workspace_bytes(p)
    assert nb > 2 * 27 * 4 * n            # A/B population buffers
    assert nb < 60e9                      # fits a 180 GB B200 several times over
    nb_r = B.workspace_bytes(p, rotor_shape=(497, 497, 161))
    assert nb_r - nb >= 5 * 497 * 497 * 161
    bad = B.make_params(0, 4, 4)
    assert B.lib().hhrr_workspace_bytes(C.byref(bad), None) == 0
    bad = B.make_params(8, 8, 8, tau0=0.5)
    assert B.lib().hhrr_workspace_bytes(C.byref(bad), None) == 0


def test_no_cpu_fallback(built):
    """Without a device (this box) create fails with a message; with one, a host pointer is refused."""
    from paper_2510_13726_b200 import binding as B
    p = B.make_params(8, 8, 8)
    h = C.c_void_p()
    buf = (C.c_char * 1024)()
    rc = B.lib().hhrr_create(C.byref(p), C.cast(buf, C.c_void_p), 1024, None, C.byref(h))
    assert rc in (-1, -3) and not h.value
    assert B.lib().hhrr_last_error()
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(RuntimeError):
            B.Lattice(p)


def test_product_does_not_import_oracle():
    pkg = ROOT / "paper_2510_13726_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + list(pkg.rglob("*.h")):
        t = f.read_text()
        assert "import oracle" not in t and "from oracle" not in t and "hhrr_oracle" not in t, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c"):
            assert "paper_2510_13726_b200 import" not in f.read_text(), f
