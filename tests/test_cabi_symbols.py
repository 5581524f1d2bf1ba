"""The C-ABI library builds, loads and exports every symbol include/*.h declares (no GPU needed)."""
import os
import re

from paper_1206_3229_b200 import binding as vb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header="vlasov.h", prefix="vlasov_"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(%s[a-z_]+)\s*\(" % prefix, text)))


def test_header_and_binding_agree():
    assert declared_symbols() == sorted(vb.EXPORTS)
    assert declared_symbols("hmf_md.h", "hmf_md_") == sorted(vb.MD_EXPORTS)
    assert declared_symbols("hmf_noalloc.h", "hmf_noalloc_") == sorted(vb.NOALLOC_EXPORTS)


def test_library_builds_loads_and_exports_every_symbol():
    lib = vb.load()
    for name in declared_symbols() + declared_symbols("hmf_md.h", "hmf_md_") + declared_symbols("hmf_noalloc.h", "hmf_noalloc_"):
        assert hasattr(lib, name), name


def test_md_calls_fail_loudly_without_init_or_device():
    lib = vb.load()
    lib.hmf_md_free()
    assert lib.hmf_md_step(1) == vb.ENOTINIT
    import torch

    if not torch.cuda.is_available():
        assert lib.hmf_md_init(100, 0.1) == vb.ECUDA


def test_calls_fail_loudly_without_init_or_device():
    vb.load().vlasov_free()
    try:
        vb.vlasov_step(1)
        raise AssertionError("vlasov_step must fail before vlasov_init")
    except vb.VlasovError as e:
        assert e.code == vb.ENOTINIT
    import torch

    if not torch.cuda.is_available():  # on the CPU box: init must refuse, not fall back
        try:
            vb.vlasov_init(1, (8, 8), (-1, 1, -1, 1), 0.1)
            raise AssertionError("vlasov_init must fail without a CUDA device")
        except vb.VlasovError as e:
            assert e.code == vb.ECUDA
        try:
            vb.Vlasov(1, (8, 8), (-1, 1, -1, 1), 0.1)
            raise AssertionError("Vlasov() must fail without a CUDA device")
        except vb.VlasovError as e:
            assert e.code == vb.ECUDA


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1206_3229_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in src and "from oracle" not in src and "oracle/" not in src, fn
