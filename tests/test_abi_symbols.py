"""-m "not gpu": the C-ABI library builds for sm_100a without a GPU, loads, and exports every function that
include/sangam.h declares; argument validation that needs no device behaves as the header says."""
import ctypes
import os
import re

import paper_2607_04206_b200 as sg
from paper_2607_04206_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_in_header():
    text = open(os.path.join(ROOT, "include", "sangam.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(sangam_[a-z_]+)\s*\(", text)))


def test_header_and_binding_agree():
    assert _declared_in_header() == sorted(sg.DECLARED_SYMBOLS)


def test_library_builds_and_exports_every_symbol():
    from paper_2607_04206_b200.build import build
    path = build()                     # nvcc cross-compiles sm_100a without a GPU
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for name in _declared_in_header():
        assert hasattr(lib, name), f"libsangam.so does not export {name}"
    assert set(sg.exported_symbols()) >= set(sg.DECLARED_SYMBOLS)
    lib.sangam_version.restype = ctypes.c_char_p
    assert b"sm_100a" in lib.sangam_version()


def test_create_rejects_bad_geometry_without_touching_a_device():
    lib = binding.load_library()
    out = ctypes.c_void_p()

    def create(**kw):
        cfg = dict(num_q_heads=8, num_kv_heads=8, head_dim=128, page_size=16, num_pages=64, max_batch=4,
                   max_total_q=128, max_pages_per_req=16, device=0)
        cfg.update(kw)
        return lib.sangam_create(ctypes.byref(binding._Config(**cfg)), ctypes.byref(out))

    assert create(page_size=32) == -2            # SANGAM_ERR_UNSUPPORTED: pages are 16 tokens
    assert create(head_dim=96) == -2
    assert create(num_q_heads=7, num_kv_heads=2) == -1   # SANGAM_ERR_INVALID_ARG: Hq % Hkv != 0
    assert create(num_pages=0) == -1
    assert create(num_q_heads=256, num_kv_heads=1) == -2  # G > 128
    assert lib.sangam_create(None, ctypes.byref(out)) == -1
    assert lib.sangam_launch_count(None) == 0
