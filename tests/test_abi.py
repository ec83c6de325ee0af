"""CPU-only checks of the boundary: libfcg.so loads, exports every symbol include/fcg.h declares, the
ctypes binding covers the same set, and the host-only entry points behave.  No compute calls."""
import ctypes
import os
import re

import pytest
import torch

from paper_2606_13097_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "fcg.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return set(re.findall(r"\b(fcg_[a-z0-9_]+)\s*\(", text))


def test_library_is_built_and_exports_every_declared_symbol():
    assert os.path.exists(binding.LIB_PATH), "run `python -m paper_2606_13097_b200.build` (or __graft_entry__.build())"
    lib = ctypes.CDLL(binding.LIB_PATH)
    declared = _declared()
    assert len(declared) >= 17
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in fcg.h but not exported"
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)


def test_version_and_error_string():
    assert "sm_100a" in binding.fcg_version()
    assert isinstance(binding.fcg_last_error(), str)


def test_arena_bytes_required_is_host_arithmetic():
    cfg = binding.make_config(n_layers=32, n_q_heads=32, n_kv_heads=8, head_dim=128, page_size=16, max_segments=64,
                              max_tasks=4, max_task_tokens=8192, n_pages=512, workspace_bytes=64 << 20)
    pool = 32 * 512 * 8 * 16 * 128 * 2
    tables = 4 * 512 * 4
    base = binding.fcg_arena_bytes_required(cfg, 0)
    assert base >= 2 * pool + tables + (64 << 20)
    per_tok = 32 * 8 * 128 * 2 * 2
    assert binding.fcg_arena_bytes_required(cfg, 1000) - base == 1000 * per_tok
    bad = binding.make_config(n_layers=1, n_q_heads=3, n_kv_heads=2, head_dim=128)
    assert binding.fcg_arena_bytes_required(bad, 0) == 0
    for hd in (72, 8, 0, 272, 100):                       # R27: multiples of 16 in [16, 256] only
        bad = binding.make_config(n_layers=1, n_q_heads=2, n_kv_heads=2, head_dim=hd)
        assert binding.fcg_arena_bytes_required(bad, 0) == 0, hd
    for hd in (16, 80, 96, 192, 256):
        ok = binding.make_config(n_layers=1, n_q_heads=2, n_kv_heads=2, head_dim=hd)
        assert binding.fcg_arena_bytes_required(ok, 0) > 0, hd


def test_create_rejects_bad_config_and_needs_a_device():
    cfg = binding.make_config(n_layers=1, n_q_heads=2, n_kv_heads=2, head_dim=64, arena=0, arena_bytes=0)
    with pytest.raises(binding.FcgError) as e:
        binding.fcg_library_create(cfg)
    assert e.value.status == binding.FCG_ERR_INVALID_ARG            # NULL arena
    cfg = binding.make_config(n_layers=1, n_q_heads=2, n_kv_heads=2, head_dim=64, arena=256, arena_bytes=1024)
    with pytest.raises(binding.FcgError) as e:
        binding.fcg_library_create(cfg)
    assert e.value.status == binding.FCG_ERR_OUT_OF_ARENA
    if not torch.cuda.is_available():
        # no CPU fallback: with no device the product path fails loudly
        cfg = binding.make_config(n_layers=1, n_q_heads=2, n_kv_heads=2, head_dim=64, arena=256, arena_bytes=1 << 40)
        with pytest.raises(binding.FcgError) as e:
            binding.fcg_library_create(cfg)
        assert e.value.status == binding.FCG_ERR_CUDA


def test_null_handles_are_rejected():
    lib = binding.load()
    assert lib.fcg_library_destroy(None) == binding.FCG_ERR_INVALID_ARG
    assert lib.fcg_task_release(None, 0) == binding.FCG_ERR_INVALID_ARG
    assert "NULL" in binding.fcg_last_error()


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2606_13097_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "oracle" not in src.replace("the oracle", "").replace("CPU oracle", "").replace("fp64 oracle", "") \
                    or f == "synth.py", f"{f} mentions the oracle package"
    for f in ("fcg_oracle.py",):
        src = open(os.path.join(ROOT, "oracle", f)).read()
        assert "import paper_2606_13097_b200" not in src and "from paper_2606_13097_b200" not in src


def test_header_is_plain_c():
    """include/fcg.h compiles as C99 on its own (no C++, no CUDA, no torch types in the boundary)."""
    import shutil
    import subprocess
    gcc = shutil.which("gcc")
    if gcc is None:
        pytest.skip("no gcc")
    r = subprocess.run([gcc, "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-x", "c", os.path.join(ROOT, "include", "fcg.h")],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
