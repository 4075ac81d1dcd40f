"""The C-ABI library loads (no GPU needed) and exports every symbol include/smoothagent.h declares;
the Python binding declares a prototype for each of them."""
import ctypes
import os
import re

from paper_2607_00151_b200 import binding
from paper_2607_00151_b200.build import build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "smoothagent.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\bSA_API\s+[\w\s\*]*?\b(sa_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = _declared()
    assert "sa_kv_pool_create" in names and "sa_rope_kv_append" in names
    assert "sa_mixed_attention" in names and "sa_latency_table" in names
    lib = ctypes.CDLL(build())
    for n in names:
        assert hasattr(lib, n), "libsmoothagent.so does not export %s" % n


def test_binding_covers_every_declared_symbol():
    names = _declared()
    assert sorted(binding.PROTOTYPES) == names
    for n in names:
        assert callable(getattr(binding, n)), "binding lacks %s" % n


def test_status_strings():
    build()
    assert binding.sa_status_string(0) == "SA_OK"
    assert binding.sa_status_string(-2) == "SA_ERR_OUT_OF_PAGES"
    assert binding.sa_status_string(-5) == "SA_ERR_WORKSPACE_TOO_SMALL"


def test_unsupported_shapes_rejected():
    build()
    good = dict(num_q_heads=8, num_kv_heads=2, head_dim=64, page_size=16, num_pages=8, max_sessions=2,
                max_session_tokens=64, rope_base=1e4)
    assert binding.sa_kv_pool_storage_bytes(binding.PoolConfig(**good)) > 0
    for bad in (dict(head_dim=96), dict(page_size=32), dict(num_q_heads=6, num_kv_heads=4), dict(num_q_heads=6, num_kv_heads=2)):
        try:
            binding.sa_kv_pool_storage_bytes(binding.PoolConfig(**{**good, **bad}))
        except binding.SAError as e:
            assert e.status == binding.SA_ERR_UNSUPPORTED
        else:
            raise AssertionError("accepted %r" % bad)


def test_no_oracle_in_product():
    """The product path must not import, call, link or open anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_2607_00151_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|libsa_oracle|sa_oracle_|oracle/|oracle\.py|\boracle\.", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                text = open(os.path.join(dirpath, f)).read()
                assert not pat.search(text), "%s reaches into the oracle" % f
