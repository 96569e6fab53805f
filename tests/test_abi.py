"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol that
include/ch.h declares, and refuses to run without a CUDA device (no CPU fallback).
No compute call is made here."""
import ctypes
import os
import re

import pytest

from paper_1911_03386_b200 import binding, build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build.build()
    return binding.lib()


def declared_functions():
    text = open(os.path.join(ROOT, "include", "ch.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ch_[a-z_]+)\s*\(", text)))


def test_every_declared_symbol_is_exported(lib):
    names = declared_functions()
    assert len(names) >= 19
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/ch.h but not exported by libch.so"
    assert sorted(binding.EXPORTS) == names, "binding.EXPORTS out of sync with include/ch.h"


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "ch.h"\nint main(void){ch_ctx *c = 0; (void)c; return CH_OK;}\n')
    rc = os.system(f"gcc -std=c99 -Wall -Werror -pedantic -I{ROOT}/include -c {src} -o {tmp_path}/t.o")
    assert rc == 0


def test_workspace_bytes_and_argument_errors(lib):
    assert lib.ch_workspace_bytes(0, 64, 2) == 0
    assert lib.ch_workspace_bytes(1, 4, 2) == 0
    assert lib.ch_workspace_bytes(1, 64, 4) == 0
    b = lib.ch_workspace_bytes(128, 512, 2)
    assert b >= 2 * 128 * 512 * 512 * 8 and b < 2.01 * 128 * 512 * 512 * 8
    ctx = ctypes.c_void_p()
    assert lib.ch_create(ctypes.byref(ctx), 1, 4, 2, 1.0, 0.01) == binding.CH_EINVAL
    assert lib.ch_create(ctypes.byref(ctx), 1, 64, 2, -1.0, 0.01) == binding.CH_EINVAL
    assert lib.ch_create(None, 1, 64, 2, 1.0, 0.01) == binding.CH_EINVAL
    assert b"ch_create" in lib.ch_last_error(None)
    assert lib.ch_destroy(None) == binding.CH_EINVAL
    assert lib.ch_step(None, 1) == binding.CH_EINVAL
    assert lib.ch_kernel_kinds() == 12
    assert [lib.ch_kernel_kind_name(k) for k in range(12)] == [b"rhs", b"rhs_diag", b"finish", b"sweep_x", b"sweep_y", b"sweep_z",
                                                                b"rhs_sweep_y", b"rhs_sweep_y_diag", b"sweep_x_update", b"sweep_xy",
                                                                b"step_local", b"step_resident"]
    d = ctypes.c_void_p()
    assert lib.ch_droplet_create(ctypes.byref(d), 0, 128, 1e-3) == binding.CH_EINVAL
    assert lib.ch_droplet_create(ctypes.byref(d), 4, 128, -1.0) == binding.CH_EINVAL
    assert lib.ch_droplet_create(None, 4, 128, 1e-3) == binding.CH_EINVAL
    assert b"ch_droplet_create" in lib.ch_droplet_last_error(None)
    assert lib.ch_droplet_destroy(None) == binding.CH_EINVAL


def test_no_cpu_fallback_without_a_gpu(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(binding.ChError) as e:
        binding.ch_create(1, 64, 2, 1.0, 0.01)
    assert e.value.code == binding.CH_ECUDA and "no CPU fallback" in str(e.value)


def test_product_never_touches_the_oracle():
    """The package may not import, link or execute anything under oracle/."""
    pkg = os.path.join(ROOT, "paper_1911_03386_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "ch_oracle" not in text and "oracle/" not in text and "import oracle" not in text, f
    for line in open(os.path.join(ROOT, "oracle", "ch_oracle.py")):
        if line.lstrip().startswith(("import ", "from ")):
            assert "paper_1911_03386_b200" not in line and "binding" not in line, line
    for line in open(os.path.join(ROOT, "oracle", "ch_oracle.c")):
        if line.lstrip().startswith("#include"):
            assert "csrc" not in line and "ch.h" not in line and "ch_factor" not in line, line
