"""The C-ABI library builds, loads and exports every symbol include/murmur.h declares; calls that
need no device (sizing, strings, NULL-argument rejection) behave as the header says.  No GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2606_01483_b200 import binding

    return binding.lib()


def _declared():
    text = open(os.path.join(ROOT, "include", "murmur.h")).read()
    return sorted(set(re.findall(r"MURMUR_API[^;(]*?\b(murmur_[a-z_0-9]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(L):
    from paper_2606_01483_b200 import binding

    names = _declared()
    assert len(names) >= 20
    for n in names:
        assert hasattr(L, n), f"{n} declared in murmur.h but not exported"
    assert sorted(binding.EXPORTED_SYMBOLS) == names


def test_no_stray_exports():
    import subprocess

    from paper_2606_01483_b200 import build

    out = subprocess.run(["nm", "-D", "--defined-only", build.LIB], capture_output=True, text=True, check=True).stdout
    syms = [ln.split()[-1] for ln in out.splitlines() if ln.strip()]
    assert syms and all(s.startswith("murmur_") for s in syms), syms


def test_sizing_calls(L):
    from paper_2606_01483_b200.binding import CacheDesc

    d = CacheDesc(28, 28, 4, 128, 64, 12, 61, 740, None, None, None, 0)
    assert L.murmur_pool_bytes(C.byref(d)) == 28 * 740 * 4 * 64 * 128 * 2
    ws = L.murmur_workspace_bytes(C.byref(d))
    assert ws > 0 and ws % 256 == 0
    for bad in (dict(head_dim=64), dict(page_size=48), dict(page_size=128), dict(n_q_heads=36), dict(n_pages=0)):
        kw = dict(n_layers=28, n_q_heads=28, n_kv_heads=4, head_dim=128, page_size=64, max_seqs=12,
                  max_blocks_per_seq=61, n_pages=740)
        kw.update(bad)
        d2 = CacheDesc(kw["n_layers"], kw["n_q_heads"], kw["n_kv_heads"], kw["head_dim"], kw["page_size"],
                       kw["max_seqs"], kw["max_blocks_per_seq"], kw["n_pages"], None, None, None, 0)
        assert L.murmur_workspace_bytes(C.byref(d2)) == 0
        assert L.murmur_pool_bytes(C.byref(d2)) == 0
    assert L.murmur_pool_bytes(None) == 0


def test_strings_and_null_handles(L):
    assert L.murmur_status_str(0) == b"MURMUR_OK"
    assert L.murmur_status_str(3) == b"MURMUR_ERR_OOM_PAGES"
    assert b"sm_100a" in L.murmur_version()
    # NULL handle / NULL out-pointer are rejected before any CUDA call
    assert L.murmur_kv_evict(None, None, 0, None) == 1
    assert L.murmur_kv_append(None, None, None, 0, None, None, 0, 1, None) == 1
    assert L.murmur_decode_attn(None, None, 0, None, None, None, 0, 1, C.c_float(1.0), None) == 1
    assert L.murmur_cache_create(None, None, None) == 1
    assert L.murmur_cache_destroy(None) == 0


def test_product_does_not_import_oracle():
    """The product package must not reach into oracle/ (parity would be void)."""
    pkg = os.path.join(ROOT, "paper_2606_01483_b200")
    for dirpath, _d, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, re.M), f
                assert "oracle/" not in text.replace("NOT shared with oracle/", ""), f
