"""Pins for the option paths of the oracle's solve loop that no closed form reaches through the default call: the
safeguard fallback when the pre-drawn list is exhausted (Alg. 4 lines 7-12, reading Q9), the K_cap
tail truncation (reading Q10), the U0 / V0 override (Alg. 4 inputs, reading Q7), the absolute
tolerance mode (PAPER.md:182, 189 as printed, reading Q15) and the r* > r_max flag (reading Q20).
Each expected value is built by hand or follows from an invariance of the method, not from re-running the formula."""
import numpy as np
import pytest

from oracle import lrp_oracle as O
from paper_2607_06021_b200 import workloads as W


# ---------------------------------------------------------------------------------------------- safeguard fallback
def test_safeguard_takes_first_unused_entry_of_the_list():
    cur = np.array([3, 5], dtype=np.int32)
    scores = np.array([0.1, 0.9, 0.5, 0.8, 0.2, 0.7])
    out = O._safeguard(cur, [5, 3, 4, 1], scores)             # 5 and 3 are present: 4 is the first usable entry
    assert out.tolist() == [3, 5, 4]


def test_safeguard_fallback_when_list_is_exhausted_or_missing():
    scores = np.array([0.1, 0.9, 0.5, 0.8, 0.2, 0.7])
    cur = np.array([3, 5], dtype=np.int32)
    # every list entry already present -> the best-scoring index outside the set: 1 (0.9)
    assert O._safeguard(cur, [3, 5, 5, 3], scores).tolist() == [3, 5, 1]
    assert O._safeguard(cur, None, scores).tolist() == [3, 5, 1]
    assert O._safeguard(cur, [], scores).tolist() == [3, 5, 1]
    # the best ones taken: next in (score desc, index asc) order is 2 (0.5)
    assert O._safeguard(np.array([1, 3, 5], dtype=np.int32), None, scores).tolist() == [1, 3, 5, 2]
    # ties are broken by the lower index
    tied = np.array([0.5, 0.5, 0.5, 0.9])
    assert O._safeguard(np.array([3], dtype=np.int32), None, tied).tolist() == [3, 0]
    # nothing left: unchanged
    assert O._safeguard(np.arange(4, dtype=np.int32), None, tied).tolist() == [0, 1, 2, 3]


def test_solve_without_safeguard_list_appends_the_best_unselected_index():
    """k = 0 always appends a safeguard index (reading Q9); with no list it is the best-leverage index outside I*: the
    (num_select + 1)-th entry of the full ranking -- checked against a full sort done here."""
    w = W.make("C2", 0, 255)
    r = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, tol=w.tol, max_rank=w.max_rank, oversample=w.oversample, max_sweeps=1,
                           safeguard=None)
    t = r.trace[0]
    for star, sc, cur in ((t.Istar, t.scoresU, t.I), (t.Jstar, t.scoresV, t.J)):
        ranking = sorted(range(w.n), key=lambda i: (-sc[i], i))
        assert cur[:-1].tolist() == star.tolist() == ranking[:len(star)]
        assert int(cur[-1]) == ranking[len(star)]


# ---------------------------------------------------------------------------------------------- K_cap truncation
def test_kcap_truncation_keeps_the_head_of_the_union_list():
    """Reading Q10: I_k is cut to K_cap = 2 (r_max + p_os) entries from the tail.  max_rank only enters through K_cap and
    the final rank, so a run with a large cap has the same history up to the first cut, and the cut list must be the
    first K_cap entries of the uncut one."""
    w = W.make("C2", 0, 511)
    full = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, tol=w.tol, max_rank=64, oversample=8, max_sweeps=4, safeguard=w.safeguard)
    sizes = [len(t.I) for t in full.trace]
    kcap = 2 * (4 + 8)
    first_cut = next(s for s, m in enumerate(sizes) if m > kcap)
    cut = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, tol=w.tol, max_rank=4, oversample=8, max_sweeps=first_cut + 1,
                             safeguard=w.safeguard)
    for s in range(first_cut):
        assert cut.trace[s].I.tolist() == full.trace[s].I.tolist() and cut.trace[s].J.tolist() == full.trace[s].J.tolist()
    assert len(cut.trace[first_cut].I) == kcap and len(cut.trace[first_cut].J) == kcap
    assert cut.trace[first_cut].I.tolist() == full.trace[first_cut].I.tolist()[:kcap]
    assert cut.trace[first_cut].J.tolist() == full.trace[first_cut].J.tolist()[:kcap]
    assert cut.rank <= 4 and cut.rank_capped and not full.rank_capped


# ---------------------------------------------------------------------------------------------- U0 / V0
def test_initial_guess_override_drives_the_first_selection_only():
    w = W.make("C2", 1, 511)
    base = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    # (a) the default initial guess is the spectral RHS factors (reading Q7): passing them explicitly changes nothing
    same = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, U0=base.UhF, V0=base.VhF, **w.opts())
    assert [t.I.tolist() for t in same.trace] == [t.I.tolist() for t in base.trace]
    assert np.array_equal(same.SW, base.SW)
    # (b) leverage scores depend on the column space only: another basis of the same space selects the same sets
    rng = np.random.default_rng(0)
    M = rng.standard_normal((w.rF, w.rF)) + 3 * np.eye(w.rF)
    mixed = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, U0=base.UhF @ M, V0=base.VhF @ M.T, **w.opts())
    assert mixed.trace[0].I.tolist() == base.trace[0].I.tolist() and mixed.trace[0].J.tolist() == base.trace[0].J.tolist()
    # (c) unit-vector columns have leverage 1 on their rows and 0 elsewhere: the first selection is exactly those rows
    # (ordered by index among equal scores), then the remaining p_os picks are score-0 rows in index order
    rowsU, rowsV = [7, 100, 33], [2, 250, 9]
    U0 = np.zeros((w.n, 3)); V0 = np.zeros((w.n, 3))
    U0[rowsU, np.arange(3)] = 1.0; V0[rowsV, np.arange(3)] = 1.0
    forced = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, U0=U0, V0=V0, tol=w.tol, max_rank=w.max_rank, oversample=2,
                                max_sweeps=1, safeguard=[400])
    assert forced.trace[0].I.tolist() == sorted(rowsU) + [0, 1] + [400]
    assert forced.trace[0].J.tolist() == sorted(rowsV) + [0, 1] + [400]
    # the fibers still come from G: the iterate is exact on the selected cross
    t = forced.trace[0]
    got = O.lowrank_entries(forced.Uhat, forced.Shat, forced.Vhat, np.repeat(t.I, len(t.J)), np.tile(t.J, len(t.I)))
    ref = O.G_entries(forced.UhF, w.SF, forced.VhF, forced.d, np.repeat(t.I, len(t.J)), np.tile(t.J, len(t.I)))
    assert np.abs(got - ref).max() < 1e-9 * np.abs(ref).max()


# ---------------------------------------------------------------------------------------------- absolute tolerance mode
def test_final_rank_absolute_versus_relative_threshold():
    S = np.array([10.0, 1.0, 0.1])
    # absolute (as printed): tails 0.01 < 0.25, 1.01 > 0.25 -> r* = 2
    assert O.final_rank(S, 0.5, 16, tol_mode=1) == 2
    # relative to sum S^2 = 101.01: threshold 25.25; tails 0.01, 1.01 < 25.25, 101.01 > 25.25 -> r* = 1
    assert O.final_rank(S, 0.5, 16, tol_mode=0) == 1
    assert O.final_rank(S, 1e-9, 2, tol_mode=1) == 2 and O.final_rank(S, 1e-9, 16, tol_mode=1) == 3      # r_max cap
    assert O.final_rank(S, 1e3, 16, tol_mode=1) == 1                                                     # never below 1


def test_absolute_mode_is_homogeneous_and_relative_mode_is_scale_free():
    """F -> c F scales W, rho, the indicator and S by c (the method is linear in F; index selection is scale-free).
    Relative mode (reading Q15) must not notice; absolute mode (the paper's literal '< eps') with eps -> c eps must
    reproduce the unscaled absolute run decision for decision."""
    w = W.make("C2", 2, 255)
    c = 2.0 ** 20                                              # a power of two: every fp64 operation scales exactly
    o = dict(max_rank=w.max_rank, oversample=w.oversample, max_sweeps=w.max_sweeps, safeguard=w.safeguard)
    rel = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, tol=1e-9, tol_mode=0, **o)
    rel_c = O.cross_deim_solve(w.n, w.UF, c * w.SF, w.VF, tol=1e-9, tol_mode=0, **o)
    assert rel_c.sweeps == rel.sweeps and rel_c.rank == rel.rank and np.array_equal(rel_c.SW, c * rel.SW)
    snorm = rel.trace[-1].snorm
    ab = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, tol=1e-9 * snorm, tol_mode=1, **o)
    ab_c = O.cross_deim_solve(w.n, w.UF, c * w.SF, w.VF, tol=c * 1e-9 * snorm, tol_mode=1, **o)
    assert ab_c.sweeps == ab.sweeps and ab_c.rank == ab.rank and ab_c.converged == ab.converged
    assert np.array_equal(ab_c.SW, c * ab.SW)
    # with eps = 1e-9 ||S|| the absolute test is the relative one up to the drift of ||S_k|| between sweeps
    assert abs(ab.sweeps - rel.sweeps) <= 1 and abs(ab.rank - rel.rank) <= 1
    # and the unscaled tolerance applied to the scaled problem is 2^20 times stricter: it cannot stop earlier
    strict = O.cross_deim_solve(w.n, w.UF, c * w.SF, w.VF, tol=1e-9 * snorm, tol_mode=1, **o)
    assert strict.sweeps >= ab_c.sweeps and strict.rank >= ab_c.rank


# ---------------------------------------------------------------------------------------------- r* > r_max
def test_rank_cap_is_reported():
    w = W.make("C2", 0, 255)
    free = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **w.opts())
    assert not free.rank_capped and free.rank > 3
    o = w.opts(); o["max_rank"] = 3
    capped = O.cross_deim_solve(w.n, w.UF, w.SF, w.VF, **o)
    assert capped.rank == 3 and capped.rank_capped
    # the kept singular values are the leading ones of a converged iterate
    assert np.abs(capped.SW - free.SW[:3]).max() < 1e-6 * free.SW[0]


# ---------------------------------------------------------------------------------------------- Alg. 3 lines 4-5 (Bernoulli)
def test_counter_uniforms_are_uniform_and_keyed():
    """The generator is a pure function of (seed, sweep, side, i): reproducible, different for different keys, and
    statistically uniform on [0, 1) (moments, a Kolmogorov-Smirnov distance, lag-1 correlation, bit balance)."""
    n = 200000
    u = O.counter_uniforms(5, 3, 1, n)
    assert np.array_equal(u, O.counter_uniforms(5, 3, 1, n))
    assert np.array_equal(u[:1000], O.counter_uniforms(5, 3, 1, 1000))          # entry i does not depend on n
    for other in (O.counter_uniforms(6, 3, 1, n), O.counter_uniforms(5, 4, 1, n), O.counter_uniforms(5, 3, 0, n)):
        assert np.mean(other == u) < 1e-3
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 4 / np.sqrt(12 * n) and abs(u.var() - 1 / 12) < 1e-3
    ks = np.abs(np.sort(u) - (np.arange(n) + 0.5) / n).max()
    assert ks < 2.0 / np.sqrt(n)
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 4 / np.sqrt(n)
    bits = (u * 2.0 ** 53).astype(np.uint64)
    for b in (0, 1, 17, 40, 52):
        assert abs(np.mean((bits >> np.uint64(b)) & np.uint64(1)) - 0.5) < 4 / np.sqrt(4 * n)


def test_bernoulli_select_by_hand():
    scores = np.array([0.5, 0.0, 1.0, 0.25, 0.25])             # cols = 2: pi = scores / 2
    # c = 2: p = min(1, scores) = [0.5, 0, 1, 0.25, 0.25]
    u = np.array([0.49, 0.0, 0.999, 0.25, 0.2499])
    # kept iff u < p: index 0 (0.49 < 0.5), not 1 (0 < 0 false), 2 (p = 1), not 3 (0.25 < 0.25 false), 4
    # order: score desc, index asc -> 2 (1.0), 0 (0.5), 4 (0.25)
    assert O.bernoulli_select(scores, 2, 2.0, u, 10).tolist() == [2, 0, 4]
    assert O.bernoulli_select(scores, 2, 2.0, u, 2).tolist() == [2, 0]                      # cap keeps the best
    # c large: every index with a positive score has p = 1 and is kept whatever u is
    assert O.bernoulli_select(scores, 2, 1e9, np.full(5, 0.999999), 10).tolist() == [2, 0, 3, 4]
    # c = 0: nothing
    assert O.bernoulli_select(scores, 2, 0.0, np.zeros(5), 10).size == 0


def test_bernoulli_expected_sample_size():
    """E #kept = sum_i min(1, c pi_i) (Alg. 3 line 5): averaged over 400 independent keys."""
    rng = np.random.default_rng(0)
    n, cols = 5000, 6
    Q, _ = np.linalg.qr(rng.standard_normal((n, cols)) * np.exp(-np.arange(n) / 300.0)[:, None])
    sc = O.leverage_scores(Q)
    c = 14.0
    expect = np.minimum(1.0, c * sc / cols).sum()
    counts = [O.bernoulli_select(sc, cols, c, O.counter_uniforms(s, 0, 0, n), n).size for s in range(400)]
    assert abs(np.mean(counts) - expect) < 4 * np.sqrt(expect / 400) + 0.05
    assert expect <= c + 1e-9


def test_bernoulli_selection_escapes_the_deterministic_stall():
    """with LS 'its probabilistic nature makes it exceedingly unlikely that exactly the same index set is
    selected twice in a row'.  The deterministic top-k form re-selects the same indices on the Hilbert matrix (n = 1024,
    this initial guess) and never passes the stop test; the printed Bernoulli form converges to the same matrix."""
    n = 1024
    U0, V0, sg = W.matrix_initial_guess(n, 4, 1)
    kw = dict(tol=1e-9, max_rank=64, oversample=8, max_sweeps=12, safeguard=sg)
    det = O.cross_deim(n, O.matrix_fibers("hilbert", n), U0, V0, **kw)
    assert not det.converged and [len(t.I) for t in det.trace][-4:] == [len(t.I) for t in det.trace][-6:-2]      # period-2 stall
    rnd = O.cross_deim(n, O.matrix_fibers("hilbert", n), U0, V0, selection="bernoulli", ls_seed=7, **kw)
    assert rnd.converged and rnd.sweeps <= 8
    i = np.arange(n)
    G = O.hilbert_entries(i[:, None], i[None, :])
    A = (rnd.U[:, :rnd.rank] * rnd.S[:rnd.rank]) @ rnd.V[:, :rnd.rank].T
    assert np.linalg.norm(A - G) <= 5e-9 * np.linalg.norm(G)
    # every sweep's selection is exactly the Bernoulli draw of that sweep's key, in (score desc, index asc) order
    t = rnd.trace[1]
    expect = O.bernoulli_select(t.scoresU, rnd.trace[0].rank, float(rnd.trace[0].rank + 8), O.counter_uniforms(7, 1, 0, n), 2 * 2 * (64 + 8))
    assert t.Istar.tolist() == expect.tolist()
