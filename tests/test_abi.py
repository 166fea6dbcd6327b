"""CPU-side checks of the boundary: the C-ABI library builds/loads without a GPU and exports every
symbol include/lqx.h declares; the Python binding declares a signature for each; the product path
refuses to run without a CUDA device (no CPU fallback); nothing in the package touches oracle/."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "lqx.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lqx_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_the_boundary_calls():
    names = _declared()
    # geometry, field store, catalogue, reductions, smear-step
    for want in ["lqx_init", "lqx_finalize", "lqx_neighbor_table", "lqx_field_alloc", "lqx_field_attach",
                 "lqx_field_free", "lqx_field_push", "lqx_field_pop", "lqx_copy", "lqx_shift",
                 "lqx_mm_plus_madj", "lqx_trace_mm", "lqx_ax_minus_shift", "lqx_mat_vec", "lqx_hop", "lqx_axpy",
                 "lqx_scale", "lqx_sum", "lqx_norm2", "lqx_trace", "lqx_plaquette", "lqx_smear_step",
                 "lqx_smear_iterate", "lqx_strerror", "lqx_last_error"]:
        assert want in names


def test_library_loads_and_exports_every_declared_symbol():
    import paper_1105_2279_b200 as lqx

    lib = ctypes.CDLL(lqx.library_path())
    for name in _declared():
        assert hasattr(lib, name), f"{name} declared in include/lqx.h but not exported"
        assert name in lqx.SIGNATURES, f"{name} has no ctypes signature in the binding"
    assert lqx.version().startswith("lqx")


def test_no_compute_without_gpu_and_no_fallback():
    import torch

    import paper_1105_2279_b200 as lqx

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        lqx.Lattice((4, 4, 4, 4))
    # the C entry itself refuses too (no device): negative status, no crash
    lib = ctypes.CDLL(lqx.library_path())
    lib.lqx_init.restype = ctypes.c_int
    out = ctypes.c_void_p()
    rc = lib.lqx_init((ctypes.c_int * 4)(4, 4, 4, 4), 0, None, ctypes.byref(out))
    assert rc < 0 and not out.value


def test_strerror_and_null_handles_are_safe():
    import paper_1105_2279_b200 as lqx

    lib = lqx._lib
    assert lib.lqx_strerror(0) == b"ok"
    assert lib.lqx_strerror(-4) == b"destination aliases a shifted operand"
    assert lib.lqx_finalize(None) == -1
    assert lib.lqx_copy(None, None) == -1
    assert lib.lqx_volume(None) < 0
    assert lib.lqx_field_data(None) is None


def test_product_path_does_not_reference_the_oracle():
    pkg = os.path.join(ROOT, "paper_1105_2279_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "import oracle" not in text and "from oracle" not in text, fn
                assert "lattice_oracle" not in text, fn
    # and the oracle does not reference the product
    for fn in os.listdir(os.path.join(ROOT, "oracle")):
        if fn.endswith((".py", ".cpp")):
            text = open(os.path.join(ROOT, "oracle", fn)).read()
            assert "paper_1105_2279_b200" not in text.replace("paper_1105_2279_b200/csrc", ""), fn
            assert "lqx_internal" not in text, fn


def test_bench_looks_up_ncu_captures_by_kernel_and_precision():
    """bench.py attaches the DRAM traffic of a committed ncu capture to its roofline block only if that capture is of
    the kernel (and precision) that ran: the lookup must find the round-2 captures by name and refuse unknown kernels."""
    import bench

    cap, src = bench._ncu_capture("k_smear_rowlit", "f32")
    assert cap is not None and src.startswith("profiles/r02") and "rowlit" in src
    traffic = cap["dram__bytes_read.sum"] + cap["dram__bytes_write.sum"]
    assert 6.1e9 < traffic < 9e9  # configs[3]: 6.115 GB algorithmic per launch
    assert 0 < cap["l1tex__data_pipe_lsu_wavefronts.avg.pct_of_peak_sustained_elapsed"] < 100
    c32, s32 = bench._ncu_capture("k_smear_rolled", "f32")
    c64, s64 = bench._ncu_capture("k_smear_rolled", "f64")
    assert c32 is not None and c64 is not None and s32 != s64
    none, why = bench._ncu_capture("k_no_such_kernel", "f32")
    assert none is None and "k_no_such_kernel" in why


def test_no_odd_descriptor_registers_in_the_library():
    """ptxas 12.9 was seen to put the descriptor of a cache-hinted cp.async in an ODD uniform register pair
    (`LDGSTS ... desc[UR1]`) in one instantiation of the smear kernel; the hardware rejects that as an illegal instruction
    at run time (DESIGN.md sec.6.1 item 16).  Wide uniform operands must be even-aligned: scan the built library's SASS."""
    import re
    import shutil
    import subprocess

    import paper_1105_2279_b200 as lqx

    cuobjdump = shutil.which("cuobjdump") or "/usr/local/cuda/bin/cuobjdump"
    if not os.path.exists(cuobjdump):
        pytest.skip("cuobjdump not available")
    sass = subprocess.run([cuobjdump, "-sass", lqx.library_path()], capture_output=True, text=True, check=True).stdout
    regs = {int(m) for m in re.findall(r"desc\[UR(\d+)\]", sass)}
    assert regs, "no descriptor-based memory instructions found: is this the right library?"
    assert not [r for r in regs if r % 2], sorted(regs)
    # the same rule for 64-bit address operands held in register pairs
    assert not [r for r in set(re.findall(r"\bU?R(\d+)\.64", sass)) if int(r) % 2]
