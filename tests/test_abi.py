"""GPU-less: the C-ABI library loads and exports every symbol include/ckf.h declares; host-side argument checks."""
import ctypes as C
import os
import re

from paper_2505_22822_b200 import binding as B
from paper_2505_22822_b200 import _build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    _build.build()
    lib = B.load_library()
    hdr = open(os.path.join(ROOT, "include", "ckf.h")).read()
    declared = set(re.findall(r"\b(ckf_[a-z_]+)\s*\(", hdr))
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert lib.ckf_abi_version() == 11


def test_struct_layouts_match_header_field_order():
    hdr = open(os.path.join(ROOT, "include", "ckf.h")).read()
    for struct in (B.ckf_geometry, B.ckf_field, B.ckf_config, B.ckf_measurements, B.ckf_seeds, B.ckf_tracks,
                   B.ckf_counters, B.ckf_timing, B.ckf_fits, B.ckf_resolution, B.ckf_seeding, B.ckf_seed_out):
        body = re.search(r"typedef struct \{([^{}]*)\} %s;" % struct.__name__, hdr, re.S).group(1)
        body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
        names = re.findall(r"[\s\*]([a-z_0-9]+)(?:\[\d+\])?\s*;", body)
        assert names == [n for n, _ in struct._fields_], struct.__name__


def test_create_rejects_bad_arguments_without_a_gpu():
    import synth
    lib = B.load_library()
    det, fld, cfg = synth.config_bundle(0)
    keep = []
    g, f = B.make_geometry(det, keep), B.make_field(fld, keep)
    c = B.make_config(cfg.ckf, 16, 10, 10, 10, 10)      # precision 16 is not supported
    h = C.c_void_p()
    assert lib.ckf_create(C.byref(g), C.byref(f), C.byref(c), C.byref(h)) == -1
    assert b"precision" in lib.ckf_last_error(None)
    c = B.make_config(cfg.ckf, 64, 10, 10, 10, 10)
    c.max_branches_per_surface = 99
    assert lib.ckf_create(C.byref(g), C.byref(f), C.byref(c), C.byref(h)) == -1
    assert lib.ckf_create(None, C.byref(f), C.byref(c), C.byref(h)) == -1


def test_no_cpu_fallback_in_binding():
    import torch
    if torch.cuda.is_available():
        return
    import pytest
    import synth
    det, fld, cfg = synth.config_bundle(0)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.CKF(det, fld, cfg.ckf, 64, 10, 10)
