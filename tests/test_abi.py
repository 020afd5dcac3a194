"""CPU-side checks of the C-ABI boundary: the library builds for sm_100a, loads, exports every symbol that
include/lrp.h declares, and its host-only entry points behave (no compute calls: there is no GPU here)."""
import ctypes as C
import os
import re

import pytest

from paper_2607_06021_b200 import build as B
from paper_2607_06021_b200 import lrp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    B.build()
    return lrp.load_library()


def _declared():
    src = open(os.path.join(ROOT, "include", "lrp.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(lrp_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(lib):
    names = _declared()
    assert set(["lrp_dst1_batched", "lrp_sample_fibers", "lrp_leverage_select", "lrp_scross",
                "lrp_cross_deim_solve"]) <= set(names)
    for nme in names:
        assert hasattr(lib, nme), nme
    assert sorted(lrp.EXPORTS) == names


def test_struct_sizes_match_header(lib):
    # a C probe compiled against the header prints sizeof/offsetof; the ctypes mirrors must agree
    import subprocess, tempfile
    code = r'''
#include <stdio.h>
#include <stddef.h>
#include "lrp.h"
int main(void){ printf("%zu %zu %zu %zu %zu %zu %zu\n", sizeof(lrp_solve_opts), sizeof(lrp_solve_info),
  offsetof(lrp_solve_opts, replay_final_rank), offsetof(lrp_solve_info, ms_dst_fwd),
  offsetof(lrp_solve_info, launches), offsetof(lrp_solve_opts, h_replay_keepI), offsetof(lrp_solve_opts, flags)); return 0; }
'''
    with tempfile.TemporaryDirectory() as d:
        p = os.path.join(d, "probe.c")
        open(p, "w").write(code)
        exe = os.path.join(d, "probe")
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), p, "-o", exe])
        vals = [int(v) for v in subprocess.check_output([exe]).split()]
    assert vals[0] == C.sizeof(lrp.SolveOpts) and vals[1] == C.sizeof(lrp.SolveInfo)
    assert vals[2] == lrp.SolveOpts.replay_final_rank.offset
    assert vals[3] == lrp.SolveInfo.ms_dst_fwd.offset
    assert vals[4] == lrp.SolveInfo.launches.offset
    assert vals[5] == lrp.SolveOpts.h_replay_keepI.offset
    assert vals[6] == lrp.SolveOpts.flags.offset


def test_host_only_entry_points(lib):
    assert lib.lrp_strerror(0) == b"ok"
    assert b"out of range" in lib.lrp_strerror(lrp.LRP_ERR_UNSUPPORTED_N)
    # one-pass regime needs no workspace, the four-step regime does
    assert lib.lrp_dst1_workspace_bytes(4095, 8) == 0
    assert lib.lrp_dst1_workspace_bytes(16383, 8) == 0
    assert lib.lrp_dst1_workspace_bytes((1 << 20) - 1, 4) >= 4 * (1 << 20) * 8      # W: 8 N bytes per column
    assert lib.lrp_dst1_workspace_bytes(1000, 4) >= 2048 * 16   # general n: Bluestein needs the transformed chirp (P = 2048)
    assert lib.lrp_dst1_workspace_bytes((1 << 23) + 5, 4) == 0  # out of range -> 0
    # solve workspace grows with n and with the rank cap
    a = lib.lrp_workspace_bytes(255, 4, 16, 8)
    b = lib.lrp_workspace_bytes(4095, 4, 16, 8)
    c = lib.lrp_workspace_bytes(4095, 4, 64, 8)
    assert 0 < a < b < c
    assert c >= 6 * 4095 * 2 * (64 + 8) * 8
    assert lib.lrp_workspace_bytes(4094, 4, 16, 8) > b            # general n is supported
    assert lib.lrp_workspace_bytes((1 << 23) + 5, 4, 16, 8) == 0


def test_no_device_fails_loudly(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    h = C.c_void_p()
    assert lib.lrp_create(C.byref(h), 0, None) == lrp.LRP_ERR_CUDA
    with pytest.raises(RuntimeError):
        lrp.Context(0)
