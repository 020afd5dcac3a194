"""lrp_cross_deim_solve_host: a batch of independent low-rank Poisson solves (section 3.2; Alg. 4,
PAPER.md:129-192) whose factors live in HOST memory, with the copies of the neighbouring problems overlapping the
solve.  Checked against the device-pointer call on the same inputs (same kernels, same order: identical results) and,
for one problem, against the CPU oracle."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2607_06021_b200 import build, lrp
    build.build()
    c = lrp.Context(0)
    yield c
    c.close()


def _host_problem(w, pinned):
    import torch
    UF = torch.from_numpy(np.ascontiguousarray(w.UF.T)); VF = torch.from_numpy(np.ascontiguousarray(w.VF.T))
    SF = torch.from_numpy(np.ascontiguousarray(w.SF))
    return tuple(t.pin_memory() if pinned else t for t in (UF, SF, VF))


def _host_output(w, pinned):
    import torch
    UW = torch.full((w.max_rank, w.n), np.nan, dtype=torch.float64); VW = torch.full_like(UW, np.nan)
    SW = torch.full((w.max_rank,), np.nan, dtype=torch.float64)
    return tuple(t.pin_memory() if pinned else t for t in (UW, SW, VW))


@pytest.mark.parametrize("pinned,lanes", [(True, 2), (True, 1), (False, 2)])
def test_host_batch_matches_device_call(ctx, pinned, lanes):
    """Seven problems (different seeds) through the staging slots of one or two lanes: every slot is reused at least
    once; results equal the device-pointer call's, problem by problem, whatever the number of lanes."""
    import torch
    from paper_2607_06021_b200 import lrp
    ws = [W.make("C2", seed) for seed in range(7)]
    w0 = ws[0]
    kw = dict(tol=w0.tol, max_rank=w0.max_rank, oversample=w0.oversample, max_sweeps=w0.max_sweeps, safeguard=w0.safeguard)
    probs = [_host_problem(w, pinned) for w in ws]
    outs = [_host_output(w, pinned) for w in ws]
    res = ctx.cross_deim_solve_host(probs, outs, lanes=lanes, **kw)
    assert len(res) == 7
    for w, r, (UW, SW, VW) in zip(ws, res, outs):
        dev = ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF), **kw)
        k = r["rank"]
        assert (k, r["sweeps"], r["converged"]) == (dev["rank"], dev["sweeps"], dev["converged"])
        assert torch.equal(SW[:k], dev["SW"].cpu())
        assert torch.equal(UW[:k], dev["UW"].cpu()) and torch.equal(VW[:k], dev["VW"].cpu())
        assert torch.isnan(UW[k:]).all() and torch.isnan(SW[k:]).all()          # nothing written beyond the rank


def test_host_batch_output_pool_and_oracle(ctx):
    """Outputs drawn from a pool of two buffers, problem p in buffer p mod 2 (the documented reuse: same lane, ordered
    downloads): the last two problems' results survive; one of them is compared with the CPU oracle entry by entry at the
    parity bar of the converged C2 runs (1e-10)."""
    from paper_2607_06021_b200 import lrp
    ws = [W.make("C2", seed) for seed in (3, 4, 5, 6)]
    w0 = ws[0]
    kw = dict(tol=w0.tol, max_rank=w0.max_rank, oversample=w0.oversample, max_sweeps=w0.max_sweeps, safeguard=w0.safeguard)
    pool = [_host_output(w0, True), _host_output(w0, True)]
    res = ctx.cross_deim_solve_host([_host_problem(w, True) for w in ws], [pool[p & 1] for p in range(4)], **kw)
    w = ws[3]
    UW, SW, VW = pool[1]
    k = res[3]["rank"]
    opts = w.opts(); opts["safeguard"] = w0.safeguard
    ref = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **opts)
    assert res[3]["converged"] and ref.converged and k == ref.rank
    rows, cols = W.sample_pairs(w.n, 4096, seed=5)
    got = np.einsum("kt,k,kt->t", UW[:k].numpy()[:, rows], SW[:k].numpy(), VW[:k].numpy()[:, cols])
    exp = O.lowrank_entries(ref.UW, ref.SW, ref.VW, rows, cols)
    assert np.abs(got - exp).max() <= 1e-10 * np.abs(exp).max()


def test_device_batch_matches_single_calls(ctx):
    """lrp_cross_deim_solve_batch (device factors, two lanes): problem by problem the same results as lrp_cross_deim_solve."""
    import torch
    from paper_2607_06021_b200 import lrp
    ws = [W.make("C2", seed) for seed in range(5)]
    w0 = ws[0]
    kw = dict(tol=w0.tol, max_rank=w0.max_rank, oversample=w0.oversample, max_sweeps=w0.max_sweeps, safeguard=w0.safeguard)
    probs = [(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF)) for w in ws]
    for lanes in (2, 1):
        res = ctx.cross_deim_solve_batch(probs, lanes=lanes, **kw)
        for (UF, SF, VF), r in zip(probs, res):
            dev = ctx.cross_deim_solve(UF, SF, VF, **kw)
            assert (r["rank"], r["sweeps"], r["converged"]) == (dev["rank"], dev["sweeps"], dev["converged"])
            assert torch.equal(r["SW"], dev["SW"]) and torch.equal(r["UW"], dev["UW"]) and torch.equal(r["VW"], dev["VW"])


def test_host_batch_padded_leading_dimensions(ctx):
    """Host factors and results with ld > n (the pitched copies of the call): same results as the device-pointer call."""
    import ctypes as C
    import torch
    from paper_2607_06021_b200 import lrp
    ws = [W.make("C2", seed) for seed in (7, 8, 9)]
    w0 = ws[0]
    n, rF, R = w0.n, w0.UF.shape[1], w0.max_rank
    ldi, ldo = n + 3, n + 5
    kw = dict(tol=w0.tol, max_rank=R, oversample=w0.oversample, max_sweeps=w0.max_sweeps, safeguard=w0.safeguard)
    ins, outs = [], []
    for w in ws:
        UF = torch.zeros((rF, ldi), dtype=torch.float64).pin_memory(); VF = torch.zeros((rF, ldi), dtype=torch.float64).pin_memory()
        UF[:, :n] = torch.from_numpy(np.ascontiguousarray(w.UF.T)); VF[:, :n] = torch.from_numpy(np.ascontiguousarray(w.VF.T))
        ins.append((UF, torch.from_numpy(np.ascontiguousarray(w.SF)).pin_memory(), VF))
        outs.append((torch.full((R, ldo), np.nan, dtype=torch.float64).pin_memory(), torch.full((R,), np.nan, dtype=torch.float64).pin_memory(),
                     torch.full((R, ldo), np.nan, dtype=torch.float64).pin_memory()))
    ctx.ensure_workspace(ctx.lib.lrp_solve_host_workspace_bytes(n, rF, R, w0.oversample, 2), exact=True)
    o = lrp.SolveOpts(); o.tol, o.max_rank, o.oversample, o.max_sweeps = w0.tol, R, w0.oversample, w0.max_sweeps
    sg = np.ascontiguousarray(w0.safeguard, dtype=np.int32); o.h_safeguard, o.n_safeguard = sg.ctypes.data, sg.size
    arr = lambda ts: (C.c_void_p * len(ts))(*[t.data_ptr() for t in ts])
    info = (lrp.SolveInfo * len(ws))()
    rc = ctx.lib.lrp_cross_deim_solve_host(ctx.h, n, rF, len(ws), arr([p[0] for p in ins]), ldi, arr([p[1] for p in ins]), arr([p[2] for p in ins]), ldi,
                                           C.byref(o), arr([q[0] for q in outs]), ldo, arr([q[1] for q in outs]), arr([q[2] for q in outs]), ldo, info)
    assert rc >= 0
    for w, (UW, SW, VW), inf in zip(ws, outs, info):
        dev = ctx.cross_deim_solve(lrp.tall_from_numpy(w.UF), torch.from_numpy(w.SF).cuda(), lrp.tall_from_numpy(w.VF), **kw)
        k = inf.rank
        assert k == dev["rank"] and inf.sweeps == dev["sweeps"]
        assert torch.equal(UW[:k, :n], dev["UW"].cpu()) and torch.equal(VW[:k, :n], dev["VW"].cpu()) and torch.equal(SW[:k], dev["SW"].cpu())
        assert torch.isnan(UW[:, n:]).all() and torch.isnan(VW[k:]).all()                 # padding and unused columns untouched


def test_host_batch_argument_errors(ctx):
    """Too small a workspace and null entries are reported, not dereferenced."""
    import ctypes as C
    import torch
    from paper_2607_06021_b200 import lrp
    w = W.make("C1", 0)
    need = ctx.lib.lrp_solve_host_workspace_bytes(w.n, w.UF.shape[1], w.max_rank, w.oversample, 1)
    base = ctx.lib.lrp_workspace_bytes(w.n, w.UF.shape[1], w.max_rank, w.oversample)
    assert need > base > 0
    assert ctx.lib.lrp_solve_host_workspace_bytes(w.n, w.UF.shape[1], w.max_rank, w.oversample, 2) == 2 * need
    assert ctx.lib.lrp_solve_host_workspace_bytes(w.n, w.UF.shape[1], w.max_rank, w.oversample, 3) == 0     # at most two lanes
    assert ctx.lib.lrp_solve_host_workspace_bytes(w.n, w.UF.shape[1], 1, 0, 1) == 0      # K_cap = 2 < rF + 1: the first selection would not fit
    small = torch.empty(base, dtype=torch.uint8, device="cuda")
    ctx.lib.lrp_set_workspace(ctx.h, C.c_void_p(small.data_ptr()), small.numel())
    ctx._ws = small
    o = lrp.SolveOpts(); o.tol, o.max_rank, o.oversample, o.max_sweeps = w.tol, w.max_rank, w.oversample, w.max_sweeps
    prob = _host_problem(w, False); out = _host_output(w, False)
    one = lambda t: (C.c_void_p * 1)(t.data_ptr())
    info = (lrp.SolveInfo * 1)()
    args = (ctx.h, w.n, w.UF.shape[1], 1, one(prob[0]), w.n, one(prob[1]), one(prob[2]), w.n, C.byref(o),
            one(out[0]), w.n, one(out[1]), one(out[2]), w.n, info)
    assert ctx.lib.lrp_cross_deim_solve_host(*args) == -3                                  # LRP_ERR_WORKSPACE
    ctx.ensure_workspace(need)
    bad = list(args); bad[4] = (C.c_void_p * 1)(None)
    assert ctx.lib.lrp_cross_deim_solve_host(*bad) == -1                                   # LRP_ERR_BADARG
    assert ctx.lib.lrp_cross_deim_solve_host(*args) >= 0
    assert info[0].rank == 4 and not torch.isnan(out[0][:4]).any()
