"""The C-ABI library builds for sm_100a, loads, and exports every symbol include/mori.h declares
(no compute calls: this runs without a GPU)."""
import ctypes
import os
import re

from paper_2606_00866_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "mori.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(mori_[a-z_]+)\s*\(", text)))


def test_header_symbols_are_exported_and_bound():
    build.build()
    lib = ctypes.CDLL(binding.LIB_PATH)
    names = _declared()
    assert "mori_rank_partition" in names and "mori_demote" in names and "mori_sync" in names
    for name in names:
        assert hasattr(lib, name), f"{name} declared in mori.h but not exported"
    assert sorted(binding.EXPORTS) == names
    for name in names:
        if name not in ("mori_create", "mori_destroy", "mori_last_error"):
            assert hasattr(binding.Mori, name), f"binding lacks {name}"


def test_config_struct_matches_header_field_order():
    text = open(os.path.join(ROOT, "include", "mori.h")).read()
    body = re.search(r"typedef struct \{(.*?)\} mori_config;", text, flags=re.S).group(1)
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    fields = []
    for decl in body.split(";"):
        decl = decl.strip()
        if not decl:
            continue
        typ, names = re.match(r"(int32_t|int64_t|void\*)\s+(.*)", decl, flags=re.S).groups()
        fields += [n.strip() for n in names.split(",")]
    assert fields == [f[0] for f in binding.MoriConfig._fields_]


def test_create_rejects_bad_config_without_a_gpu_call():
    lib = binding.load()
    h = ctypes.c_void_p()
    cfg = binding.MoriConfig()          # all zero
    assert lib.mori_create(ctypes.byref(cfg), ctypes.byref(h)) == binding.ERR_INVALID_ARG
    assert h.value is None and lib.mori_last_error(None)
    assert lib.mori_create(None, ctypes.byref(h)) == binding.ERR_INVALID_ARG
    assert lib.mori_sync(None, 3) == binding.ERR_INVALID_ARG
    assert lib.mori_destroy(None) == binding.OK
