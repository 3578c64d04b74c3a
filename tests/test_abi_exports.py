"""The C-ABI library loads without a GPU and exports every function include/aframe.h declares."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "aframe.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(aframe_[a-z_0-9]+)\s*\(", src)))


def test_header_declares_the_four_named_calls():
    names = _declared()
    for n in ("aframe_psd_welch", "aframe_whiten", "aframe_forward", "aframe_stream_step"):
        assert n in names


def test_library_builds_loads_and_exports_every_symbol():
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    lib = ctypes.CDLL(af.LIB_PATH)
    for n in _declared():
        assert hasattr(lib, n), f"{n} declared in aframe.h but not exported"
    assert sorted(af.EXPORTS) == _declared()


def test_host_side_validation_needs_no_gpu():
    import paper_2403_18661_b200 as af
    lib = af.load_library()
    cfg = af.default_config()
    assert cfg.size == ctypes.sizeof(af.aframe_config) and cfg.welch_nfft == 4096 and cfg.psd_len == 131072
    h = ctypes.c_void_p()
    bad = af.default_config(welch_nfft=3000)
    assert lib.aframe_create(ctypes.byref(bad), None, ctypes.byref(h)) == af.EINVAL
    bad = af.default_config(psd_update=1000)
    assert lib.aframe_create(ctypes.byref(bad), None, ctypes.byref(h)) == af.ESHAPE
    assert lib.aframe_create(None, None, ctypes.byref(h)) == af.EINVAL
    assert lib.aframe_last_error(None) == b"no context"
    import torch
    if not torch.cuda.is_available():
        # no device: creation must fail loudly, never fall back
        assert lib.aframe_create(ctypes.byref(cfg), None, ctypes.byref(h)) == af.EUNSUPPORTED
        with pytest.raises((af.AframeError, RuntimeError, AssertionError)):
            af.Context()


def test_header_is_plain_c_and_a_c_program_links_against_the_library(tmp_path):
    """include/aframe.h compiles as C11 with gcc (no C++ or CUDA types leak into the boundary) and a C program that takes
    the address of every declared entry point links against the shared library; it runs the host-side validation."""
    import shutil
    import subprocess
    import __graft_entry__ as ge
    ge.build()
    import paper_2403_18661_b200 as af
    if shutil.which("gcc") is None:
        pytest.skip("no gcc")
    names = _declared()
    src = ['#include "aframe.h"', "#include <stdio.h>", "int main(void) {",
           "  aframe_config cfg; aframe_ctx* ctx = 0;",
           "  if (aframe_config_default(&cfg) != AFRAME_OK || cfg.size != sizeof(cfg)) return 2;",
           "  cfg.welch_nfft = 3000;",
           "  if (aframe_create(&cfg, 0, &ctx) != AFRAME_EINVAL || ctx != 0) return 3;",
           "  void* fns[] = {" + ", ".join(f"(void*){n}" for n in names) + "};",
           '  printf("%d entry points\\n", (int)(sizeof(fns) / sizeof(fns[0])));', "  return 0;", "}"]
    c = tmp_path / "abi.c"
    c.write_text("\n".join(src))
    exe = tmp_path / "abi"
    libdir = os.path.dirname(af.LIB_PATH)
    libname = os.path.basename(af.LIB_PATH)
    cmd = ["gcc", "-std=c11", "-Wall", "-Werror", "-pedantic", "-Wno-pedantic", "-I", os.path.join(ROOT, "include"), str(c),
           "-o", str(exe), "-L", libdir, f"-l:{libname}", f"-Wl,-rpath,{libdir}"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    assert r.returncode == 0, r.stderr
    r = subprocess.run([str(exe)], capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip() == f"{len(names)} entry points", (r.returncode, r.stdout, r.stderr)
