"""CPU-side checks of the boundary: libawr.so builds and loads, exports every symbol that
include/awr.h declares, the ctypes mirror has the C layout, and the host-side argument checks
return the documented status codes (no compute without a GPU)."""
import ctypes as C
import os
import re
import subprocess
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "awr.h")

from paper_2606_05597_b200 import _abi  # noqa: E402


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"AWR_API\s+[\w\s\*]+?\b(awr_\w+)\s*\(", text)))


def test_header_symbols_match_binding_table():
    assert declared_symbols() == sorted(_abi.SYMBOLS)


def test_library_exports_every_declared_symbol():
    lib = _abi.load()
    for name in declared_symbols():
        assert hasattr(lib, name), name
    out = subprocess.check_output(["nm", "-D", "--defined-only", _abi.lib_path()]).decode()
    exported = set(re.findall(r"\bT (awr_\w+)", out))
    assert exported == set(declared_symbols()), exported ^ set(declared_symbols())
    assert lib.awr_version() == 200


def test_struct_layout_matches_c(tmp_path):
    """sizeof / offsetof from a C compile of include/awr.h against the ctypes mirror."""
    structs = {"awr_batch": _abi.awr_batch, "awr_params": _abi.awr_params,
               "awr_outputs": _abi.awr_outputs, "awr_head_batch": _abi.awr_head_batch,
               "awr_head_outputs": _abi.awr_head_outputs}
    lines = ['#include <stdio.h>', '#include <stddef.h>', '#include "awr.h"', 'int main(void){']
    for name, st in structs.items():
        lines.append('printf("%s %%zu\\n", sizeof(%s));' % (name, name))
        for f, _ in st._fields_:
            lines.append('printf("%s.%s %%zu\\n", offsetof(%s, %s));' % (name, f, name, f))
    lines.append("return 0;}")
    src = tmp_path / "layout.c"
    src.write_text("\n".join(lines))
    exe = tmp_path / "layout"
    subprocess.check_call(["gcc", "-std=c99", "-I", os.path.join(ROOT, "include"), str(src),
                           "-o", str(exe)])
    got = dict(l.split() for l in subprocess.check_output([str(exe)]).decode().splitlines())
    for name, st in structs.items():
        assert int(got[name]) == C.sizeof(st), name
        for f, _ in st._fields_:
            assert int(got["%s.%s" % (name, f)]) == getattr(st, f).offset, (name, f)


def test_header_is_plain_c_without_torch_types():
    text = open(HEADER).read()
    assert "torch" not in text and "at::" not in text and "#include <cuda" not in text


def test_host_side_status_codes():
    lib = _abi.load()
    P = _abi.awr_params(10.0, 0.2, 0.0, 1.0, 0.0, 0, 0, 0)
    B = _abi.awr_batch()
    Oo = _abi.awr_outputs()
    f = lib.awr_loss_fwd_bwd
    assert f(None, C.byref(P), C.byref(Oo), None, 0, None) == _abi.AWR_ERR_NULL
    B.n_tok, B.V, B.ld = 4, 16, 8
    assert f(C.byref(B), C.byref(P), C.byref(Oo), None, 0, None) == _abi.AWR_ERR_SHAPE
    B.ld = 16
    B.logits_dtype = 7
    assert f(C.byref(B), C.byref(P), C.byref(Oo), None, 0, None) == _abi.AWR_ERR_DTYPE
    B.logits_dtype = 0
    for bad in (dict(k_norm=0.0), dict(clip_eps=1.0), dict(clip_eps=-0.1), dict(normalizer=3),
                dict(flags=16), dict(dual_clip_c=float("nan")), dict(kernel=13),
                dict(stale_cap=float("nan"))):
        Q = _abi.awr_params(10.0, 0.2, 0.0, 1.0, 0.0, 0, 0, 0)
        for k, v in bad.items():
            setattr(Q, k, v)
        assert f(C.byref(B), C.byref(Q), C.byref(Oo), None, 0, None) == _abi.AWR_ERR_PARAM, bad
    assert f(C.byref(B), C.byref(P), C.byref(Oo), None, 0, None) == _abi.AWR_ERR_NULL
    assert lib.awr_status_string(_abi.AWR_ERR_ARCH).decode().startswith("device is not sm_100")
    assert lib.awr_workspace_bytes(1000, 151936, 10, 8, 2) % 256 == 0
    assert lib.awr_workspace_bytes(-1, 1, 1, 1, 1) == 0
    assert lib.awr_select_kernel(151936, 151936, 0) == _abi.KERNEL_CLUSTER_RFS
    assert lib.awr_select_kernel(151936, 151936, 1) == _abi.KERNEL_GENERIC
    assert lib.awr_select_kernel(1024, 1024, 0) == _abi.KERNEL_GENERIC


def test_binding_refuses_cpu_tensors():
    """No CPU path: device entry points reject host tensors instead of falling back."""
    import paper_2606_05597_b200 as A
    z = torch.zeros(4, 16, dtype=torch.bfloat16)
    i = torch.zeros(4, dtype=torch.int32)
    x = torch.zeros(4)
    off = torch.tensor([0, 4], dtype=torch.int32)
    one = torch.tensor([0, 1], dtype=torch.int32)
    with pytest.raises(TypeError):
        A.awr_loss_fwd_bwd(z, i, x, x, off, one, one, torch.zeros(1))


def test_product_never_imports_oracle():
    """The product path shares nothing with oracle/ (and gen/ holds no method arithmetic)."""
    pkg = os.path.join(ROOT, "paper_2606_05597_b200")
    for dirpath, _, files in os.walk(pkg):
        for fn in files:
            if fn.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, fn)).read()
                assert "oracle" not in text.replace("not the oracle", ""), fn
    code = ("import sys; import paper_2606_05597_b200; "
            "assert not any(m.startswith('oracle') for m in sys.modules)")
    subprocess.check_call([sys.executable, "-c", code], cwd=ROOT)
