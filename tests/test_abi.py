"""Host-side checks that need no GPU: the C-ABI library loads, exports every symbol include/kpz.h declares,
validates arguments, and fails loudly (KPZ_ECUDA, never a CPU fallback) when there is no device."""
import ctypes
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def pkg():
    import __graft_entry__ as g
    g.build()
    import paper_1110_6745_b200 as pkg
    return pkg


def test_header_symbols_all_exported(pkg):
    header = (ROOT / "include" / "kpz.h").read_text()
    declared = set(re.findall(r"\b(kpz_[a-z0-9_]+)\s*\(", header))
    declared.discard("kpz_ctx")
    assert declared == set(pkg.exported_symbols)
    lib = pkg.load_library()
    for name in declared:
        assert getattr(lib, name) is not None


def test_workspace_bytes_and_argument_validation(pkg):
    lat, scr = pkg.workspace_bytes(256, 16, 1)
    assert lat == 256 * 256 // 4                      # 2 bits per site
    assert pkg.workspace_bytes(1 << 17, 64, 1)[0] == 1 << 32     # 4 GB at 2^17
    assert pkg.workspace_bytes(128, 16, 1024)[0] == 1024 * 128 * 128 // 4
    assert scr > 0
    for (L, T) in ((256, 5), (256, 128), (100, 16), (48, 16), (0, 16), (64, 64)):
        with pytest.raises(pkg.KpzError) as e:
            pkg.workspace_bytes(L, T, 1)
        assert e.value.code == pkg.KPZ_EINVAL
    with pytest.raises(pkg.KpzError):
        pkg.workspace_bytes(256, 16, 0)


def test_create_validates_and_never_falls_back_to_cpu(pkg):
    import torch
    lib = pkg.load_library()
    h = ctypes.c_void_p()
    assert lib.kpz_create(ctypes.addressof(h), 256, 1.5, 0.0, 16, 1) == pkg.KPZ_EINVAL
    assert lib.kpz_create(ctypes.addressof(h), 256, 1.0, -0.1, 16, 1) == pkg.KPZ_EINVAL
    assert lib.kpz_create(ctypes.addressof(h), 250, 1.0, 0.0, 16, 1) == pkg.KPZ_EINVAL
    assert lib.kpz_create(None, 256, 1.0, 0.0, 16, 1) == pkg.KPZ_EINVAL
    rc = lib.kpz_create(ctypes.addressof(h), 256, 1.0, 0.0, 16, 1)
    if torch.cuda.is_available():
        assert rc == pkg.KPZ_OK
        assert lib.kpz_run(h, 1) == pkg.KPZ_ESTATE          # not bound yet
        assert b"kpz_bind" in lib.kpz_last_error(h)
        assert lib.kpz_destroy(h) == pkg.KPZ_OK
    else:
        assert rc == pkg.KPZ_ECUDA and not h.value          # no device -> loud failure, no CPU path
    assert lib.kpz_destroy(None) == pkg.KPZ_OK


def test_product_never_touches_the_oracle():
    """Plain grep: no file of the product (package, header, C ABI) names the oracle package, its library or its
    symbols; no file of the oracle names the product package.  bench.py and __graft_entry__.py may (cpu_baseline,
    --impl reference, smoke)."""
    needles = ("import oracle", "from oracle", "libkpz_oracle", "kpzo_", "oracle/", "oracle.")
    files = [f for f in (ROOT / "paper_1110_6745_b200").rglob("*") if f.suffix in (".py", ".cu", ".cuh", ".h")]
    files += list((ROOT / "include").glob("*.h"))
    assert files
    for f in files:
        txt = f.read_text()
        for n in needles:
            assert n not in txt, (f, n)
    for f in (ROOT / "oracle").rglob("*"):
        if f.suffix in (".py", ".cpp", ".h"):
            txt = f.read_text()
            assert "import paper_1110_6745_b200" not in txt and "from paper_1110_6745_b200" not in txt, f
            assert "libkpz_b200" not in txt and "kpz.h" not in txt and "kpz_device" not in txt, f
