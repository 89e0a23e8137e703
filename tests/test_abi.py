"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/dmpt.h
declares, its structs have the layout the ctypes binding assumes, and the host-only entry points
behave.  No compute call is made here (there is no GPU on this box and no CPU fallback)."""
import ctypes as C
import os
import re
import subprocess
import sys
import tempfile

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "dmpt.h")


def _declared_functions():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(dmpt_[a-z0-9_]+)\s*\(", text)))


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2203_09621_b200 import EXPORTED_SYMBOLS, lib
    from paper_2203_09621_b200.build import build_library

    build_library()                       # no-op when up to date
    L = lib()
    declared = _declared_functions()
    assert len(declared) >= 12
    for name in declared:
        assert hasattr(L, name), f"libdmpt.so lacks {name} declared in include/dmpt.h"
    assert sorted(EXPORTED_SYMBOLS) == declared, "binding.EXPORTED_SYMBOLS and include/dmpt.h disagree"


def test_struct_layout_matches_the_header():
    """Compile a C program against include/dmpt.h and compare sizeof/offsetof with ctypes."""
    from paper_2203_09621_b200.binding import DmptOptions, _CResult

    src = r'''
#include <stdio.h>
#include <stddef.h>
#include "dmpt.h"
int main(void) {
    printf("%zu %zu %zu %zu %zu\n", sizeof(dmpt_options), offsetof(dmpt_options, bounds),
           offsetof(dmpt_options, eps_min), offsetof(dmpt_options, num_fields), offsetof(dmpt_options, reserved));
    printf("%zu %zu %zu %zu %zu %zu %zu\n", sizeof(dmpt_result), offsetof(dmpt_result, launches),
           offsetof(dmpt_result, eps_min), offsetof(dmpt_result, ms_loop), offsetof(dmpt_result, ms_split),
           offsetof(dmpt_result, sigma), offsetof(dmpt_result, fro_err3));
    return 0;
}
'''
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "layout.c")
        exe = os.path.join(d, "layout")
        open(c, "w").write(src)
        subprocess.run(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), c, "-o", exe], check=True)
        out = subprocess.run([exe], check=True, capture_output=True, text=True).stdout.split("\n")
    o = [int(x) for x in out[0].split()]
    r = [int(x) for x in out[1].split()]
    assert o == [C.sizeof(DmptOptions), DmptOptions.bounds.offset, DmptOptions.eps_min.offset,
                 DmptOptions.num_fields.offset, DmptOptions.reserved.offset]
    assert r == [C.sizeof(_CResult), _CResult.launches.offset, _CResult.eps_min.offset, _CResult.ms_loop.offset,
                 _CResult.ms_split.offset, _CResult.sigma.offset, _CResult.fro_err3.offset]


def test_host_only_entry_points():
    import paper_2203_09621_b200 as p

    o = p.dmpt_default_options()
    assert (o.max_layers, o.order, o.s0_shift, o.s1_autoscale, o.bounds, o.wave_sync, o.num_fields) == \
        (200, 1, -1, 1, 0, 1, 1)
    assert list(o.reserved) == [0] * 1 and o.order0_narrow == 0 and o.loop_graph == 0 and o.epilogue_direct == 0 and o.lanczos_steps == 0 and o.no_pdl == 0
    assert p.dmpt_strerror(0) == "ok"
    for code in range(-7, 0):
        assert p.dmpt_strerror(code) not in ("ok", "unknown error code")
    assert p.dmpt_strerror(-99) == "unknown error code"
    # workspace: 3 fp32 + 8 fp16 padded matrices + 2 fp32 staging matrices + scalars
    assert p.dmpt_workspace_bytes(0) == 0 and p.dmpt_workspace_bytes(-5) == 0 and p.dmpt_workspace_bytes(64, 4) == 0
    for n in (1, 100, 256, 2048, 16384):
        npad = (n + 255) // 256 * 256            # CTA-pair tiles: 256 rows
        need = 3 * npad * npad * 4 + 8 * npad * npad * 2 + 2 * n * n * 4
        got = p.dmpt_workspace_bytes(n, 1)
        assert need <= got <= need + (4 << 20), (n, need, got)
        assert p.dmpt_workspace_bytes(n, 0) == got and p.dmpt_workspace_bytes_fields(n, 1) == got
        # each further field: 2 fp32 + 4 fp16 padded matrices + one n x n staging matrix (dmpt_run_fields_host)
        per_field = 2 * npad * npad * 4 + 4 * npad * npad * 2 + (n * n * 4 + 255) // 256 * 256
        assert p.dmpt_workspace_bytes_fields(n, 3) - got == 2 * per_field
    assert p.dmpt_workspace_bytes(2048, 3) > p.dmpt_workspace_bytes(2048, 2) > p.dmpt_workspace_bytes(2048, 1)
    # order-parallel pair: each side has the workspace of a context of its own order
    from paper_2203_09621_b200 import binding as B
    assert B.dmpt_pair_workspace_bytes(2048, 0) == p.dmpt_workspace_bytes(2048, 0)
    assert B.dmpt_pair_workspace_bytes(2048, 1) == p.dmpt_workspace_bytes(2048, 1)
    assert B.dmpt_pair_workspace_bytes(2048, 2) == 0 and B.dmpt_pair_workspace_bytes(0, 0) == 0
    assert p.dmpt_workspace_bytes_fields(64, 0) == 0 and p.dmpt_workspace_bytes_fields(64, 4) == 0


def test_invalid_arguments_are_rejected_before_any_cuda_call():
    import paper_2203_09621_b200 as p

    L = p.lib()
    h = C.c_void_p()
    assert L.dmpt_create(None, 256, None, None, 0, None) == p.binding.DMPT_EINVAL
    assert L.dmpt_create(C.byref(h), 0, None, C.c_void_p(256), 1 << 30, None) == p.binding.DMPT_EINVAL
    assert L.dmpt_create(C.byref(h), 256, None, None, 1 << 30, None) == p.binding.DMPT_EINVAL
    # too small / misaligned workspace
    assert L.dmpt_create(C.byref(h), 256, None, C.c_void_p(256), 1024, None) == p.binding.DMPT_EWORKSPACE
    assert L.dmpt_create(C.byref(h), 256, None, C.c_void_p(257), 1 << 30, None) == p.binding.DMPT_EWORKSPACE
    assert h.value is None
    assert L.dmpt_destroy(None) == p.binding.DMPT_EINVAL
    assert L.dmpt_run(None, None, None, None, 0, None) == p.binding.DMPT_EINVAL
    assert L.dmpt_set_hamiltonian(None, None, None, 0, 0) == p.binding.DMPT_EINVAL
    assert L.dmpt_run_orders(None, None, 0, None) == p.binding.DMPT_EINVAL
    assert L.dmpt_pair_create(None, 256, None, 0, None, 0, 0, None, 0) == p.binding.DMPT_EINVAL
    assert L.dmpt_pair_create(C.byref(h), 256, None, 0, None, 0, 0, None, 0) == p.binding.DMPT_EINVAL
    assert L.dmpt_pair_run(None, None, None, 0, None) == p.binding.DMPT_EINVAL
    assert L.dmpt_pair_set_hamiltonian(None, None, None, 0, 0) == p.binding.DMPT_EINVAL
    assert L.dmpt_pair_destroy(None) == p.binding.DMPT_EINVAL


def test_product_never_imports_the_oracle():
    """The CUDA path and the oracle share no code: nothing under the package or include/ names it."""
    pkg = os.path.join(ROOT, "paper_2203_09621_b200")
    for base, _dirs, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(base, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", text, flags=re.M), f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2203_09621_b200" not in text.replace("`paper_2203_09621_b200/`", ""), f


def test_no_cpu_fallback_without_cuda():
    import torch

    import paper_2203_09621_b200 as p

    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(p.DmptError):
        p.Dmpt(64, device="cpu")
