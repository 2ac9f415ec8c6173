"""No-GPU check of the boundary: libffpp.so builds for sm_100a, loads, and exports every symbol include/ffpp.h declares."""
import ctypes
import os
import re
import subprocess

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols(header="ffpp.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ffpp_[a-z_0-9]+)\s*\(", text)))


def test_library_builds_loads_and_exports_the_header():
    import paper_2512_07009_b200 as m
    path = m.build()
    lib = ctypes.CDLL(path)
    syms = declared_symbols()
    assert set(syms) == set(m.EXPORTS), (syms, m.EXPORTS)
    dbg = declared_symbols("ffpp_debug.h")
    assert set(dbg) == set(m.DEBUG_EXPORTS), (dbg, m.DEBUG_EXPORTS)
    assert not [s for s in syms if "debug" in s], "include/ffpp.h is the contract only"
    nxt = declared_symbols("ffpp_next.h")
    assert set(nxt) == set(m.NEXT_EXPORTS), (nxt, m.NEXT_EXPORTS)
    noa = declared_symbols("ffpp_noalloc.h")
    assert set(noa) == set(m.NOALLOC_EXPORTS), (noa, m.NOALLOC_EXPORTS)
    for s in syms + dbg + nxt + noa:
        assert hasattr(lib, s), f"libffpp.so does not export {s}"
    # null-handle calls that need no device
    lib.ffpp_destroy.argtypes = [ctypes.c_void_p]
    assert lib.ffpp_destroy(None) == 0
    lib.ffpp_last_error.restype = ctypes.c_char_p
    lib.ffpp_last_error.argtypes = [ctypes.c_void_p]
    assert isinstance(lib.ffpp_last_error(None), bytes)


def test_binary_is_sm100a_and_uses_the_bulk_copy_engine():
    import paper_2512_07009_b200 as m
    path = m.build()
    elf = subprocess.run(["cuobjdump", "-lelf", path], capture_output=True, text=True).stdout
    assert "sm_100a" in elf, elf
    syms = subprocess.run(["cuobjdump", "-elf", path], capture_output=True, text=True).stdout
    k1 = sorted(set(re.findall(r"(_ZN4ffpp20k1_threshold_compactILb1EjEE\w+)", syms)))
    assert k1, "k1_threshold_compact<true, uint32_t> not found in the fatbin"
    sass = subprocess.run(["cuobjdump", "-sass", "-fun", k1[0], path], capture_output=True, text=True).stdout
    assert "UBLKCP" in sass          # cp.async.bulk (TMA engine) in the HBM-bound streaming kernel


def test_no_cpu_fallback_without_a_device():
    import pytest
    import torch
    import paper_2512_07009_b200 as m
    if torch.cuda.is_available():
        pytest.skip("device present")
    with pytest.raises(RuntimeError):
        m.FFPP(dict(dtype="fp16", conf_thresh=0.25, iou_thresh=0.45, top_k=10, sigma_cells=2.0),
               max_frames=1, max_total_candidates=8400, max_frame_w=640, max_frame_h=640)
