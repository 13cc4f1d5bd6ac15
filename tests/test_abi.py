"""C-ABI boundary: the library builds for sm_100a, loads, and exports every symbol include/dmrg_b200.h
declares; argument errors that need no GPU are reported through status codes (no compute here)."""
import ctypes as C
import os
import re
import subprocess
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dmrg_b200.h")


@pytest.fixture(scope="module")
def lib():
    from paper_1309_5571_b200 import build, binding
    build.build()
    return binding.load_library()


def declared_symbols():
    txt = open(HEADER).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(dmrg_[a-zA-Z0-9_]+)\s*\(", txt)))


def test_header_symbols_are_exported(lib):
    from paper_1309_5571_b200 import binding
    syms = declared_symbols()
    assert "dmrg_apply_H" in syms and "dmrg_davidson_step" in syms and "dmrg_lowest_eigenpair" in syms
    for s in syms:
        assert hasattr(lib, s), f"{s} declared in the header but not exported"
    assert sorted(binding.EXPORTS) == syms
    out = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    exported = sorted(set(re.findall(r" T (dmrg_[A-Za-z0-9_]+)", out)))
    assert exported == syms, "exported dmrg_* symbols differ from the header"


def test_header_compiles_as_plain_c(tmp_path):
    src = tmp_path / "t.c"
    src.write_text('#include "dmrg_b200.h"\nint main(void){ dmrg_problem p; dmrg_options o; dmrg_stats s; (void)p;(void)o;(void)s; return 0; }\n')
    r = subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-c", str(src), "-o", str(tmp_path / "t.o")],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_struct_layout_matches_header(tmp_path, lib):
    """sizeof of the ctypes mirrors equals sizeof in C (catches a field added on one side only)."""
    from paper_1309_5571_b200 import binding
    src = tmp_path / "s.c"
    src.write_text('#include <stdio.h>\n#include "dmrg_b200.h"\nint main(void){printf("%zu %zu %zu %zu %zu\\n", sizeof(dmrg_sectors), '
                   'sizeof(dmrg_block_op), sizeof(dmrg_problem), sizeof(dmrg_options), sizeof(dmrg_stats));return 0;}\n')
    exe = tmp_path / "s"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    sizes = [int(v) for v in subprocess.run([str(exe)], capture_output=True, text=True).stdout.split()]
    mine = [C.sizeof(binding._Sectors), C.sizeof(binding._BlockOp), C.sizeof(binding._Problem),
            C.sizeof(binding._Options), C.sizeof(binding.Stats)]
    assert sizes == mine


def test_argument_errors_without_gpu(lib):
    from paper_1309_5571_b200 import binding
    assert lib.dmrg_version() >= 100
    h = C.c_void_p()
    assert lib.dmrg_plan_create(None, None, C.byref(h)) == binding.DMRG_E_INVALID_ARG
    assert b"NULL" in lib.dmrg_last_error(None)
    assert lib.dmrg_plan_create(None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_apply_H(None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_plan_destroy(None) == binding.DMRG_E_INVALID_ARG
    # every entry point that takes a handle rejects a NULL one before touching the device
    k = C.c_int32(1)
    assert lib.dmrg_davidson_init(None, None, 0, None, None, 0, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_davidson_step(None, None, None, 0, C.byref(k), None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_davidson_step_host(None, None, None, 0, C.byref(k), None, None, None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_davidson_poll(None, None, None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_lowest_eigenpair(None, None, 0, None, None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_ritz_vector(None, None, 0, 1, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_get_small(None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_set_small(None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_gemv_trans(None, None, 0, 1, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_gemv_sub(None, None, 0, 1, None, None, None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_get_stats(None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_get_unit_trace(None, None, 0, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_set_timing(None, 1) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_get_timing(None, None) == binding.DMRG_E_INVALID_ARG
    assert lib.dmrg_probe_fp64_peak(5, 1, None, None) == binding.DMRG_E_INVALID_ARG
    pr = binding._Problem()
    pr.model = 7
    assert lib.dmrg_plan_create(C.byref(pr), None, C.byref(h)) == binding.DMRG_E_INVALID_ARG


def test_product_fails_loudly_without_cuda():
    """No CPU fallback: on a box without a GPU the binding raises instead of computing."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    import paper_1309_5571_b200 as lib
    from oracle import blocks
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        lib.Plan(blocks.heisenberg_exact(2, 2))


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_1309_5571_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cpp")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1309_5571_b200" not in txt.replace("``paper_1309_5571_b200/``", ""), f
