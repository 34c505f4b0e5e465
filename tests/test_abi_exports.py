"""The C-ABI library builds for sm_100a without a GPU, loads, and exports every function include/af.h declares.
No compute call is made here (this runs on CPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    names = []
    for hdr in ("af.h", "af_debug.h"):          # the C ABI proper + the test / bench helpers of the same library
        src = open(os.path.join(ROOT, "include", hdr)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names += re.findall(r"\b(af_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_debug_helpers_live_in_their_own_header():
    src = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "include", "af.h")).read(), flags=re.S)
    assert "af_debug_" not in src


def test_header_declares_the_north_star_calls():
    names = _declared_functions()
    for must in ("af_ring_create", "af_ring_reset_slot", "af_packed_forward", "af_logits_rows", "af_ring_destroy"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2512_20276_b200 import build, binding
    path = build.build()
    assert os.path.exists(path)
    lib = ctypes.CDLL(path)
    for n in _declared_functions():
        assert hasattr(lib, n), f"{n} is declared in include/af.h but not exported"
    assert sorted(binding.EXPORTS) == _declared_functions(), "binding.EXPORTS must list exactly the header's functions"


def test_binding_fails_loudly_without_the_library(monkeypatch, tmp_path):
    from paper_2512_20276_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", str(tmp_path / "missing.so"))
    try:
        binding.load_library()
    except RuntimeError as e:
        assert "no CPU fallback" in str(e)
    else:
        raise AssertionError("load_library() must raise when the CUDA library is missing")


def test_host_helpers_need_no_gpu():
    """af_ring_bytes / af_workspace_bytes are pure host arithmetic."""
    from paper_2512_20276_b200 import binding, inputs as I
    L = binding.load_library()
    c = binding._cfg_struct(I.CFG_7B)
    r = binding.af_ring_cfg(8, 512)
    assert L.af_ring_bytes(ctypes.byref(c), ctypes.byref(r)) == 2 * 32 * 8 * 32 * 512 * 128 * 2
    assert L.af_workspace_bytes(ctypes.byref(c), 288, 8) > 288 * (4096 * 6 + 3 * 11008) * 2
    assert L.af_gate_up_rows(11008) == 172 * 128 and L.af_gate_up_rows(688) == 11 * 128 and L.af_gate_up_rows(0) == 0
