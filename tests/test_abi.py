"""CPU-side checks of the boundary: libdovetail_draft.so builds for sm_100a, loads, and
exports every symbol include/dovetail.h declares; the ctypes structs match the header's
layout; without a usable device the entry points fail loudly (no fallback)."""
import ctypes as C
import os
import re

import pytest
import torch

from paper_2412_18934_b200 import binding, build
from paper_2412_18934_b200.configs import CONFIGS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.load()


def _declared(header):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)  # prototypes only, not the prose
    return sorted(set(re.findall(r"\b(dovetail_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared("dovetail.h")
    assert set(names) == set(binding.EXPORTS)
    hooks = _declared("dovetail_hooks.h")
    assert set(hooks) == set(binding.HOOK_EXPORTS)
    for n in names + hooks:
        assert getattr(lib, n) is not None


def test_no_environment_variables_in_the_library():
    """no env vars, no global state in the product."""
    csrc = os.path.join(ROOT, "paper_2412_18934_b200", "csrc")
    for f in os.listdir(csrc):
        assert "getenv" not in open(os.path.join(csrc, f)).read(), f


def test_struct_layouts_match_header():
    # sizes implied by include/dovetail.h (LP64): 7 int32 + 2 float + 8 int32; 9 pointers; ...
    assert C.sizeof(binding.ConfigT) == 18 * 4
    assert C.sizeof(binding.LayerWeightsT) == 16 * 8
    assert C.sizeof(binding.WeightsT) == 12 * 8
    assert C.sizeof(binding.KVCacheT) == 24
    assert C.sizeof(binding.TreeSpecT) == 4 * (1 + 16 + 16 + 1)
    assert C.sizeof(binding.DraftOutT) == 5 * 8
    assert C.sizeof(binding.HooksT) == 11 * 8


def test_null_arguments_are_rejected(lib):
    assert lib.dovetail_draft_init(None, None, None) == binding.EINVAL
    assert lib.dovetail_draft_step(None, None, None, 1, None, None, None, None) == binding.EINVAL
    assert lib.dovetail_kv_commit(None, None, None, 0, 0, None, None) == binding.EINVAL
    assert lib.dovetail_last_launch_count(None) == 0
    assert lib.dovetail_draft_status(None, None) == binding.EINVAL
    assert lib.dovetail_hooks_set(None, None) == binding.EINVAL
    assert lib.dovetail_forward_bytes(None, 0) == 0
    assert b"null" in lib.dovetail_last_error(None)
    lib.dovetail_draft_destroy(None)


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-device behaviour")
def test_no_device_means_error_not_fallback(lib):
    """With no sm_100 device dovetail_draft_init returns DOVETAIL_ECUDA: nothing computes on the CPU."""
    cfg = CONFIGS["c1"]
    c = binding.config_t(cfg)
    dummy = C.c_void_p(16)  # never dereferenced: the device check comes first
    layers = (binding.LayerWeightsT * cfg.n_layers)(*[binding.LayerWeightsT(*[16] * 16) for _ in range(cfg.n_layers)])
    w = binding.WeightsT(16, 16, 16, 16, 16, layers, None, 16, None, None, None, None)
    out = C.c_void_p()
    rc = lib.dovetail_draft_init(C.byref(w), C.byref(c), C.byref(out))
    assert rc == binding.ECUDA and not out.value
    assert lib.dovetail_last_error(None)


def test_binding_refuses_missing_library(monkeypatch):
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "LIB_PATH", "/nonexistent/libdovetail_draft.so")
    with pytest.raises(FileNotFoundError):
        binding.load()


def test_headers_compile_as_plain_c_and_a_c_program_links(tmp_path):
    """The boundary is a C ABI: both headers are valid C99 and C++17 on their own (-Wall -Wextra -pedantic -Werror),
    and a C program with no Python, torch or CUDA headers links against the library and gets error codes, not
    aborts, from NULL arguments."""
    import subprocess
    inc = os.path.join(ROOT, "include")
    libdir = os.path.join(ROOT, "paper_2412_18934_b200")
    binding.load()  # builds the library if it is missing
    for hdr in ("dovetail.h", "dovetail_hooks.h"):
        for comp, std, lang in (("gcc", "-std=c99", "c"), ("g++", "-std=c++17", "c++")):
            subprocess.run([comp, std, "-Wall", "-Wextra", "-pedantic", "-Werror", "-fsyntax-only", "-x", lang, "-I", inc,
                            os.path.join(inc, hdr)], check=True)
    src = tmp_path / "main.c"
    src.write_text('#include <stdio.h>\n#include <string.h>\n#include "dovetail.h"\n'
                   "int main(void) {\n"
                   "  if (dovetail_draft_init(NULL, NULL, NULL) != DOVETAIL_EINVAL) return 1;\n"
                   "  if (dovetail_tree_replay_static(NULL, NULL, NULL, 0, 0, NULL, NULL) != DOVETAIL_EINVAL) return 2;\n"
                   '  if (strstr(dovetail_last_error(NULL), "null") == NULL) return 3;\n'
                   "  if (dovetail_forward_bytes(NULL, 0) != 0) return 4;\n"
                   "  dovetail_draft_destroy(NULL);\n"
                   '  puts("ok");\n  return 0;\n}\n')
    exe = tmp_path / "main"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", inc, str(src), "-o", str(exe), "-L", libdir,
                    "-ldovetail_draft", f"-Wl,-rpath,{libdir}"], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True)
    assert out.stdout.strip() == "ok"
