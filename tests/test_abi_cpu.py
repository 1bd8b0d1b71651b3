"""CPU-side checks of the boundary: the C-ABI library builds, loads and exports every symbol that
include/sparda.h declares; argument validation that needs no GPU; binding struct layout."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpath():
    from paper_2606_04511_b200 import build
    return build.build()


def _declared_symbols():
    text = open(os.path.join(ROOT, "include", "sparda.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sparda_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(libpath):
    from paper_2606_04511_b200 import binding
    L = ctypes.CDLL(libpath)
    decl = _declared_symbols()
    assert len(decl) >= 12
    for sym in decl:
        assert hasattr(L, sym), f"{sym} declared in sparda.h but not exported"
    assert sorted(binding.EXPORTS) == decl, "binding.EXPORTS out of sync with include/sparda.h"


def test_strerror_and_version_without_gpu(libpath):
    L = ctypes.CDLL(libpath)
    L.sparda_strerror.restype = ctypes.c_char_p
    L.sparda_version.restype = ctypes.c_char_p
    assert L.sparda_strerror(0) == b"ok"
    assert b"invalid" in L.sparda_strerror(-1)
    assert b"sm_100" in L.sparda_strerror(-2)
    assert b"sm_100a" in L.sparda_version()


def test_create_rejects_bad_config_and_missing_gpu(libpath):
    import torch
    from paper_2606_04511_b200 import binding
    L = binding.lib()
    h = ctypes.c_void_p()
    assert L.sparda_create(None, ctypes.byref(h)) == -1
    bad = binding.SpardaConfig(1, 4, 1, 96, 64, 64, 8, 0, 0, 0, 0)         # head_dim 96
    assert L.sparda_create(ctypes.byref(bad), ctypes.byref(h)) == -1
    bad = binding.SpardaConfig(1, 4, 1, 64, 32, 64, 8, 0, 0, 0, 0)         # block_size != 64
    assert L.sparda_create(ctypes.byref(bad), ctypes.byref(h)) == -1
    if not torch.cuda.is_available():
        ok = binding.SpardaConfig(1, 4, 1, 64, 64, 64, 8, 0, 0, 0, 0)
        assert L.sparda_create(ctypes.byref(ok), ctypes.byref(h)) == -2     # no sm_100 device: unsupported, no fallback
        with pytest.raises(binding.SpardaError):
            binding.Sparda(1, 4, 1, 64, 64, 8)


def test_binding_struct_layout_matches_header():
    from paper_2606_04511_b200 import binding
    text = open(os.path.join(ROOT, "include", "sparda.h")).read()
    cfg_body = re.search(r"typedef struct \{(.*?)\} sparda_config;", text, flags=re.S).group(1)
    cfg_body = re.sub(r"/\*.*?\*/", "", cfg_body, flags=re.S)
    fields = re.findall(r"int\s+([a-z_]+);", cfg_body)
    assert fields == [f[0] for f in binding.SpardaConfig._fields_]
    lay_body = re.search(r"typedef struct \{(.*?)\} sparda_layer;", text, flags=re.S).group(1)
    lay_body = re.sub(r"/\*.*?\*/", "", lay_body, flags=re.S)
    lfields = re.findall(r"\*\s*([A-Za-z_]+);", lay_body)
    assert lfields == [f[0] for f in binding.SpardaLayer._fields_]
    assert ctypes.sizeof(binding.SpardaLayer) == len(lfields) * ctypes.sizeof(ctypes.c_void_p) == 9 * ctypes.sizeof(ctypes.c_void_p)


def test_product_does_not_import_oracle():
    """The product path shares nothing with the oracle (and has no CPU fallback to route through)."""
    pkg = os.path.join(ROOT, "paper_2606_04511_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"import oracle|from oracle|sparda_oracle|oracle/", src), f"{f} reaches into oracle/"
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_04511_b200" not in src and "from paper_2606_04511_b200" not in src
            assert "csrc" not in src.replace("paper_2606_04511_b200/csrc/", "")
