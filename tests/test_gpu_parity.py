"""GPU parity: the CUDA path through the C ABI (include/hk.h) against the fp64 CPU
oracle on the same seeded inputs.  Tolerance (BASELINE.json north_star): relative
error <= 1e-4 per bin where oracle >= 1e-8 max(k), absolute <= 1e-8 max(k) elsewhere;
integer extents and centre bins exact."""
import math
import os
import re

import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import hk_oracle as O
from workload import linelists as W

from parity_util import check_parity, check_parity_plinth, check_parity_subtracted, sample_windows

_HK_NODES = int(re.search(r"#define HK_NODES (\d+)", open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "..", "include", "hk.h")).read()).group(1))
B_SEP_MIN = {8: 4.0, 10: 2.5, 12: 2.0}[_HK_NODES] - 0.25     # smallest node separation hk_set_node_separation accepts

pytestmark = pytest.mark.gpu

import os
N_FUZZ = int(os.environ.get("HK_FUZZ_SEEDS", "40"))     # cases per randomised differential test (more: HK_FUZZ_SEEDS=400)


@pytest.fixture(scope="module")
def B():
    """The binding, with one invariant checked on EVERY hk_get_stats of this module: the node kernel finds the entries of
    its lines from the geometry, so the (line, tile) pairs it evaluated must be exactly the pairs node_range_kernel
    counted -- a missed or doubled entry would show here before it shows in k(nu)."""
    from paper_2101_02005_b200 import binding
    if not getattr(binding.Opacity, "_stats_checked", False):
        plain = binding.Opacity.stats

        def stats(self):
            st = plain(self)
            assert st["n_pairs_node_eval"] == st["n_pairs_node"], (st["n_pairs_node_eval"], st["n_pairs_node"])
            return st

        binding.Opacity.stats = stats
        binding.Opacity._stats_checked = True
    return binding


def _to_cuda(lines_np):
    return {k: torch.as_tensor(np.ascontiguousarray(v), dtype=torch.float64).cuda() for k, v in lines_np.items()}


def _gpu_k(B, lines_np, cond, grid, cut, debug_mode=0, tile_bins=0):
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_debug_mode(debug_mode)
    op.set_tile_bins(tile_bins)
    dl = _to_cuda(lines_np)
    k = op.compute(dl, cut)
    torch.cuda.synchronize()
    st = op.stats()
    ext = tuple(t.cpu().numpy() for t in op.extents(dl))
    op.close()
    return k.cpu().numpy(), st, ext


def _check_extents(ext, lines_np, cond, grid, cut):
    numin, numax, dnu = grid
    N = O.grid_size(*grid)
    _, _, _, valid = O.line_params(lines_np, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    ilo, ihi, jc = O.extents(lines_np["nu0"], valid, numin, dnu, N, cut)
    empty = ilo > ihi
    ilo = np.where(empty, 0, ilo)
    ihi = np.where(empty, -1, ihi)
    g_ilo, g_ihi, g_jc = ext
    assert np.array_equal(g_ilo.astype(np.int64), ilo)
    assert np.array_equal(g_ihi.astype(np.int64), ihi)
    in32 = (jc > -(1 << 31)) & (jc < (1 << 31) - 1)
    assert np.array_equal(g_jc.astype(np.int64)[in32], jc[in32])
    return int((ihi - ilo + 1).sum())


def _mini(cfg, n):
    lines = W.to_numpy(W.make_lines(cfg, n=n, seed=0))
    c = W.CONFIGS[cfg]
    return lines, W.conditions(cfg), c["grid"], c["cut"]


# ---- full-grid parity on configs the oracle finishes in seconds -----------------------

@pytest.mark.parametrize("cfg,n", [(1, None), (2, 20_000), (3, 200_000), (4, 6_000)])
def test_full_grid_parity(B, cfg, n):
    """Config 1 at full size; mini twins (same generator, fewer lines, full grid) of 2-4."""
    lines, cond, grid, cut = _mini(cfg, n)
    k_gpu, st, ext = _gpu_k(B, lines, cond, grid, cut)
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    n_ev = _check_extents(ext, lines, cond, grid, cut)
    assert st["n_evals"] == evals == n_ev
    assert st["n_evals_far"] + st["n_evals_mid"] + st["n_evals_core"] == st["n_evals"]
    rel, ab, frac = check_parity(k_gpu, k_ref, what=f"config {cfg}")
    print(f"config {cfg}: n={len(lines['nu0'])} rel={rel:.2e} abs={ab:.2e} frac_rel={frac:.3f} evals={evals}")


def test_uncut_atom_like_sampled_bins(B):
    """Config 5 mini twin (2000 lines, all 5e6 bins on the GPU); the oracle sums every
    line on 4096 sampled bins + windows around the strongest lines."""
    lines, cond, grid, cut = _mini(5, 2000)
    k_gpu, st, ext = _gpu_k(B, lines, cond, grid, cut)
    N = O.grid_size(*grid)
    assert st["n_evals"] == 2000 * N
    rng = np.random.default_rng(5)
    bins = set(rng.integers(0, N, 3000).tolist()) | {0, 1, N - 2, N - 1}
    S, _, _, _ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    for l in np.argsort(S)[-8:]:
        jc = int((lines["nu0"][l] - grid[0]) / grid[2])
        bins |= set(range(max(0, jc - 40), min(N, jc + 40)))
    jmax = int(k_gpu.argmax())
    bins |= set(range(max(0, jmax - 8), min(N, jmax + 8)))
    bins = np.array(sorted(bins), dtype=np.int64)
    k_ref, _ = O.opacity_bins(lines, cond, grid, cut, bins)
    kmax = float(k_ref.max())                    # the oracle's maximum; the GPU's argmax bin is among the sampled ones
    assert k_gpu.max() <= kmax * (1 + 1e-4)
    check_parity(k_gpu[bins], k_ref, kmax=kmax, what="config 5 mini")
    _check_extents(ext, lines, cond, grid, cut)


def test_cross_path_nodes_vs_direct(B):
    """SURVEY 8(d) cross-path check on ALL bins: the default path (separated tiles at Chebyshev nodes, mode 0)
    against direct evaluation of every pair (mode 3), against everything through the masked near kernel (mode 1)
    and against far pairs through the mid kernel (mode 2)."""
    for cfg, n, tb in [(2, 20_000, 0), (4, 6_000, 0), (4, 6_000, 2), (3, 100_000, 2), (5, 300, 0)]:
        lines, cond, grid, cut = _mini(cfg, n)
        k0, st0, _ = _gpu_k(B, lines, cond, grid, cut, debug_mode=0, tile_bins=tb)
        assert st0["n_levels"] >= 1 and st0["n_pairs_node"] > 0 and st0["n_pairs_centre"] > 0
        k3, st3, _ = _gpu_k(B, lines, cond, grid, cut, debug_mode=3, tile_bins=tb)
        assert st3["n_levels"] == 0 and st3["n_pairs_node"] == 0 and st3["n_pairs_far"] > 0 and st3["n_pairs_mid"] > 0
        # every (line, bin) pair of the definition is covered exactly once by one of the four paths
        for st in (st0, st3):
            cover = st["n_pairs_far"] + st["n_pairs_mid"] + st["n_bins_node"]
            edge_node_bins = st["n_pairs_edge_node"] * 32 * st["bins_per_lane"]
            assert cover <= st["n_evals"] <= cover + st["n_pairs_near"] + st["n_pairs_edge"] + st["n_pairs_centre"] + edge_node_bins
        big = k3 >= 1e-8 * k3.max()
        assert np.abs(k0[big] / k3[big] - 1.0).max() <= 3e-5
        if cfg == 5:
            continue
        for mode in (1, 2):
            k1, st1, _ = _gpu_k(B, lines, cond, grid, cut, debug_mode=mode, tile_bins=tb)
            assert st1["n_pairs_far"] == 0 and st1["n_pairs_node"] == 0
            assert np.abs(k1[big] / k3[big] - 1.0).max() <= 4e-5


@pytest.mark.parametrize("cfg,n", [(2, 20_000), (3, 200_000), (4, 6_000), (1, None)])
def test_edge_nodes_on_vs_off(B, cfg, n):
    """Extent ends through the per-bin node accumulators (default) against the masked direct edge kernel, all bins,
    and both against the oracle."""
    lines, cond, grid, cut = _mini(cfg, n)
    dl = _to_cuda(lines)
    ks = []
    for on in (True, False):
        op = B.Opacity(*grid)
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        op.set_edge_nodes(on)
        k = op.compute(dl, cut)
        torch.cuda.synchronize()
        st = op.stats()
        if on:
            assert st["n_pairs_edge_node"] > 0
            n_on_edge = st["n_pairs_edge"]
        else:
            assert st["n_pairs_edge_node"] == 0 and st["n_pairs_edge"] > n_on_edge
        ks.append(k.cpu().numpy())
        op.close()
    k_ref, _ = O.opacity_grid(lines, cond, grid, cut)
    for k in ks:
        check_parity(k, k_ref, what=f"config {cfg} edge nodes")
    big = k_ref >= 1e-8 * k_ref.max()
    assert np.abs(ks[0][big] / ks[1][big] - 1.0).max() <= 3e-5


def test_counting_sort_unsorted_input(B):
    """Step a2 on its own path: an UNSORTED list with compact keys goes through the counting sort by centre bin (bucket
    array in the sort scratch), most of its lines off the grid (sentinel keys: the last bucket); all bins against the oracle."""
    lines, cond, _, cut = _mini(2, 300_000)
    grid = (3500.0, 4000.0, 0.01)
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    dl = _to_cuda(lines)
    k = op.compute(dl, cut).cpu().numpy()
    torch.cuda.synchronize()
    st = op.stats()
    assert st["sort_bits"] == 0 and st["n_unsorted"] > 0 and st["n_off_grid"] > 100_000
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    assert st["n_evals"] == evals
    rel, ab, frac = check_parity(k, k_ref, what="counting sort, unsorted input")
    _check_extents(tuple(t.cpu().numpy() for t in op.extents(dl)), lines, cond, grid, cut)
    print(f"counting sort: rel={rel:.2e} abs={ab:.2e} off grid {st['n_off_grid']}")
    op.close()


def _stat_ints(st):
    """the integer work counts that must not depend on how the records were written"""
    keys = ("n_lines", "n_skipped", "n_off_grid", "n_evals", "n_evals_far", "n_evals_mid", "n_evals_core", "n_evals_gh6",
            "n_evals_trap", "n_evals_gh10", "n_pairs_far", "n_pairs_mid", "n_pairs_near", "n_pairs_edge", "n_pairs_centre",
            "n_pairs_node", "n_bins_node", "n_pairs_edge_node", "n_pairs_node_far", "bins_per_lane", "n_levels")
    return {k: st[k] for k in keys}


@pytest.mark.parametrize("cfg,n", [(3, 200_000), (4, 6_000), (2, 20_000), (1, None)])
def test_single_pass_preprocess(B, cfg, n):
    """Steps a1 + a2 in one kernel (line_sorted_kernel): the SECOND compute on a workspace, when the first found the list
    sorted with every line on the grid, writes its sorted records in one pass.  Checked: which path ran (hk_stats.single_pass;
    never on a first call, never for an unsorted list), the result of the single pass against the oracle on all bins, the
    extents from its records, every integer work count equal to the two-pass path's, and the two results equal to the
    rounding of the fp32 partial sums."""
    lines, cond, grid, cut = _mini(cfg, n)
    sorted_in = bool((np.diff(lines["nu0"]) >= 0).all())
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    dl = _to_cuda(lines)
    k1 = op.compute(dl, cut).cpu().numpy()
    st1 = op.stats()
    assert st1["single_pass"] == 0
    k2 = op.compute(dl, cut).cpu().numpy()
    st2 = op.stats()
    ext2 = tuple(t.cpu().numpy() for t in op.extents(None, n=len(lines["nu0"])))
    # (sort_bits == 0: the counting sort ran, which is the path that learns whether the list arrived in order; a few
    #  thousand lines on millions of bins go through the radix sort and never take the single pass)
    expect = sorted_in and st1["sort_bits"] == 0 and st1["n_off_grid"] == 0 and st1["n_skipped"] == 0
    assert st2["single_pass"] == (1 if expect else 0), (sorted_in, st1)
    assert expect or cfg != 3
    assert _stat_ints(st1) == _stat_ints(st2) and st1["scale_exp"] == st2["scale_exp"]
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    assert st2["n_evals"] == evals == _check_extents(ext2, lines, cond, grid, cut)
    rel, ab, _ = check_parity(k2, k_ref, what=f"config {cfg}, second compute")
    # (the order of the lines inside one centre bin differs between the paths, and fp32 partial sums follow it)
    same = np.abs(k2 - k1).max() / k_ref.max()
    assert same <= 2e-6, same
    # switched off: two passes again, same counts
    op.set_single_pass(False)
    k3 = op.compute(dl, cut).cpu().numpy()
    st3 = op.stats()
    assert st3["single_pass"] == 0 and _stat_ints(st3) == _stat_ints(st1)
    assert np.abs(k3 - k1).max() / k_ref.max() <= 2e-6
    print(f"config {cfg}: sorted {sorted_in}, single pass {st2['single_pass']}, rel={rel:.2e} abs={ab:.2e}, 1st vs 2nd {same:.1e}")
    op.close()


def test_single_pass_falls_back(B):
    """The hint is checked on the device every time.  After a sorted list has set it: (a) the same workspace gets an
    UNSORTED list, (b) a sorted list with one invalid and one off-grid line, (c) conditions that move the launch scale by
    more than the window (T 1500 -> 200 K, Q x 1e6), (d) conditions that move it by less -- (a)-(c) must run the two passes,
    (d) the single pass with the HINTED scale; all four against the oracle."""
    lines, cond, grid, cut = _mini(3, 200_000)
    n = len(lines["nu0"])
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])

    def run(ln, cd, expect, what):
        op.set_conditions(cd["T"], cd["P_atm"], cd["mass_amu"], cd["Q"])
        k = op.compute(_to_cuda(ln), cut).cpu().numpy()
        st = op.stats()
        k_ref, evals = O.opacity_grid(ln, cd, grid, cut)
        assert st["n_evals"] == evals
        rel, ab, _ = check_parity(k, k_ref, what=what)
        assert st["single_pass"] == expect, (what, st["single_pass"])
        print(f"{what}: single pass {st['single_pass']}, scale 2^{st['scale_exp']}, rel={rel:.2e}")
        return st

    s0 = run(lines, cond, 0, "first call")
    run(lines, cond, 1, "second call")
    rng = np.random.default_rng(5)
    perm = rng.permutation(n)
    shuffled = {k: v[perm] for k, v in lines.items()}
    run(shuffled, cond, 0, "(a) unsorted list after a sorted one")
    run(shuffled, cond, 0, "(a) unsorted list again")
    run(lines, cond, 0, "sorted list after an unsorted one (two passes: the hint said unsorted)")
    run(lines, cond, 1, "sorted list, hint restored")
    bad = {k: v.copy() for k, v in lines.items()}
    bad["A"][n // 3] = np.nan
    bad["nu0"][-1] = grid[1] + 10 * cut
    sb = run(bad, cond, 0, "(b) sorted list with an invalid and an off-grid line")
    assert sb["n_skipped"] == 1 and sb["n_off_grid"] == 1
    run(bad, cond, 0, "(b) again")
    run(lines, cond, 0, "clean list after (b)")
    run(lines, cond, 1, "clean list, hint restored")
    cold = dict(cond, T=200.0, Q=cond["Q"] * 1.0e6)
    sc = run(lines, cold, 0, "(c) T 1500 -> 200 K, Q x 1e6")
    assert abs(sc["scale_exp"] - s0["scale_exp"]) > 8, (sc["scale_exp"], s0["scale_exp"])
    run(lines, cold, 1, "(c) again")
    near = dict(cold, T=230.0, P_atm=cond["P_atm"] * 3.0, Q=cold["Q"] * 7.0)
    sd = run(lines, near, 1, "(d) T 200 -> 230 K, 3 x P, Q x 7")
    assert sd["scale_exp"] == sc["scale_exp"]          # the hinted scale was used, not this call's own
    se = run(lines, near, 1, "(d) again")
    assert se["scale_exp"] != sd["scale_exp"]          # ... and the hint was re-centred on this call's maxima
    op.close()


@pytest.mark.parametrize("cfg,n", [(2, 20_000), (3, 200_000), (4, 6_000), (5, 300)])
def test_node_kernels_agree(B, cfg, n):
    """The line-stationary node kernel against the entry-stationary one it replaced (hk_set_node_kernel): the same
    (line, tile) pairs -- counted, and evaluated, exactly once by both -- with the same arithmetic per pair, so the two
    spectra differ by summation order only; and the sorted-input count of the counting sort."""
    lines, cond, grid, cut = _mini(cfg, n)
    ks, sts = [], []
    for entry_stationary in (False, True):
        op = B.Opacity(*grid)
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        op.set_node_kernel(entry_stationary)
        op.set_core_nodes(False)             # (the core at nodes exists in the line-stationary kernel only)
        ks.append(op.compute(_to_cuda(lines), cut).cpu().numpy())
        torch.cuda.synchronize()
        sts.append(op.stats() if not entry_stationary else None)       # (only the line-stationary kernel counts its pairs)
        op.close()
    assert sts[0]["n_pairs_node"] > 0 and sts[0]["n_pairs_node_eval"] == sts[0]["n_pairs_node"]
    nu0 = lines["nu0"]
    if sts[0]["sort_bits"] == 0:             # counting sort by centre bin (compact keys, bucket array fits the scratch)
        assert (sts[0]["n_unsorted"] == 0) == bool((nu0[1:] >= nu0[:-1]).all())
    big = ks[1] >= 1e-8 * ks[1].max()
    assert np.abs(ks[0][big] / ks[1][big] - 1.0).max() <= 1e-6


@pytest.mark.parametrize("cfg,n", [(2, 20_000), (3, 200_000), (4, 6_000), (1, None)])
def test_core_at_nodes_on_vs_off(B, cfg, n):
    """hk_set_core_nodes: separated tiles of the core (|z|^2 >= 49 on all of them) through the node hierarchy, their node
    values from the 4-point Gauss-Hermite form, against direct evaluation of every core bin by the centre kernels.  Both
    against the oracle on all bins; the pairs that moved are counted; the two spectra differ by the interpolation error
    (tests/test_nodes.py: <= 1.3e-5) plus the node record's quantisation."""
    lines, cond, grid, cut = _mini(cfg, n)
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    ks, sts = [], []
    for on in (True, False):
        op = B.Opacity(*grid)
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        op.set_core_nodes(on)
        ks.append(op.compute(_to_cuda(lines), cut).cpu().numpy())
        st = op.stats()
        sts.append(st)
        assert st["n_evals"] == evals
        rel, ab, _ = check_parity(ks[-1], k_ref, what=f"config {cfg}, core at nodes {on}")
        print(f"config {cfg} core at nodes {on}: rel={rel:.2e} abs={ab:.2e} node pairs {st['n_pairs_node']} (core {st['n_pairs_node_core']}) "
              f"centre slots {st['n_pairs_centre']}")
        op.close()
    assert sts[1]["n_pairs_node_core"] == 0
    if cfg in (2, 4):                        # 0.01 cm^-1 grids: the core spans several level-0 tiles
        assert sts[0]["n_pairs_node_core"] > 0
    assert sts[1]["n_evals_core_nodes"] == 0
    if sts[0]["n_pairs_node_core"] > 0:
        assert sts[0]["n_pairs_centre"] < sts[1]["n_pairs_centre"] and sts[0]["n_pairs_node"] > sts[1]["n_pairs_node"]
        # the core bins now covered by interpolation lie in the (line, tile) slots that left the centre kernels
        moved = sts[1]["n_pairs_centre"] - sts[0]["n_pairs_centre"]
        assert 0 < sts[0]["n_evals_core_nodes"] <= moved
        assert sts[0]["n_evals_core_nodes"] <= sts[0]["n_evals_core"] - sts[0]["n_evals_gh6"] - sts[0]["n_evals_trap"]
    else:                                    # (cores narrower than the separation distance: nothing to move)
        assert sts[0]["n_pairs_centre"] == sts[1]["n_pairs_centre"] and sts[0]["n_pairs_node"] == sts[1]["n_pairs_node"]
    big = k_ref >= 1e-8 * k_ref.max()
    assert np.abs(ks[0][big] / ks[1][big] - 1.0).max() <= 4e-5


@pytest.mark.parametrize("aD_bins", [0.7, 3.0, 9.0, 25.0, 80.0])
@pytest.mark.parametrize("y", [1e-3, 0.2, 1.2, 6.0])
def test_core_at_nodes_across_widths(B, aD_bins, y):
    """The core at nodes over the whole range of geometries: Doppler widths from under a bin to more than a level-0 tile
    (so that the separated tiles of the core are found at level 0, or only at higher levels), damping from next to none
    to Lorentz-dominated; isolated lines and a dense clump, all bins against the oracle."""
    rng = np.random.default_rng(int(aD_bins * 10) + int(y * 1000))
    dnu, nbins = 0.005, 60_000
    grid = (20000.0, 20000.0 + nbins * dnu, dnu)
    cut = 60.0                                                    # 12000 bins: several levels of the hierarchy
    T, mass = 1000.0, 30.0
    beta = math.sqrt(2 * 1.380649e-16 * T / (mass / 6.02214076e23)) / 2.99792458e10
    # the mass that gives alpha_D = aD_bins * dnu at 20150 cm^-1
    mass = mass * (beta * 20150.0 / (aD_bins * dnu)) ** 2
    n = 300
    nu0 = np.sort(np.concatenate([rng.uniform(grid[0] - 5.0, grid[1] + 5.0, n - 60), rng.normal(20150.0, 0.3, 60)]))
    aD = aD_bins * dnu
    lines = _simple_lines(nu0, A=10 ** rng.uniform(-1, 2, n), gamma_ref=np.full(n, y * aD), n_exp=np.zeros(n))
    cond = dict(T=T, P_atm=1.0, mass_amu=mass, Q=50.0)
    _, gL, aDs, _ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    assert abs(np.median(aDs) / dnu / aD_bins - 1.0) < 0.02 and abs(np.median(gL / aDs) / y - 1.0) < 0.05
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    k = op.compute(_to_cuda(lines), cut).cpu().numpy()
    st = op.stats()
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    assert st["n_evals"] == evals
    rel, ab, _ = check_parity(k, k_ref, what=f"core at nodes, alpha_D {aD_bins} bins, y {y}")
    if aD_bins >= 3.0:                       # the core (25 alpha_D) reaches beyond the two tiles next to the line
        assert st["n_pairs_node_core"] > 0 and st["n_evals_core_nodes"] > 0
    print(f"alpha_D {aD_bins} bins, y {y}: rel={rel:.2e} abs={ab:.2e} core pairs {st['n_pairs_node_core']} "
          f"core bins at nodes {st['n_evals_core_nodes']} of {st['n_evals_core']}")
    op.close()


@pytest.mark.parametrize("sep", [B_SEP_MIN, 2.0, 3.0, 4.0, 6.0])
def test_node_separation_sweep(B, sep):
    """The node hierarchy at other separations (fewer / more pairs at nodes) against the oracle, down to the smallest
    the library accepts (its default minus a quarter of a tile half-width: interpolation error 4.5e-5 worst case, tests/test_nodes.py)."""
    if sep < B_SEP_MIN:
        pytest.skip("below the smallest separation of this build")
    lines, cond, grid, cut = _mini(2, 20_000)
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_node_separation(sep)
    k = op.compute(_to_cuda(lines), cut)
    torch.cuda.synchronize()
    st = op.stats()
    assert st["n_levels"] >= 1 and st["n_pairs_node"] > 0
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    assert st["n_evals"] == evals
    check_parity(k.cpu().numpy(), k_ref, what=f"node separation {sep}")
    with pytest.raises(B.HKError):
        op.set_node_separation(B_SEP_MIN - 0.125)  # closer than that the interpolant is outside the error budget
    op.close()


@pytest.mark.parametrize("tile_bins", [2, 4, 8])
@pytest.mark.parametrize("cfg,n", [(1, None), (2, 20_000), (3, 200_000)])
def test_every_tile_geometry(B, cfg, n, tile_bins):
    """Each tile geometry (bins per lane 2/4/8) on each workload shape against the oracle."""
    lines, cond, grid, cut = _mini(cfg, n)
    k_gpu, st, _ = _gpu_k(B, lines, cond, grid, cut, tile_bins=tile_bins)
    assert st["bins_per_lane"] == tile_bins
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    assert st["n_evals"] == evals
    check_parity(k_gpu, k_ref, what=f"config {cfg} tile_bins {tile_bins}")


def test_host_pipeline_and_accumulate(B):
    """hk_compute_host (blocks copied host->device while the previous block computes) and
    hk_accumulate (block-wise sum) against the one-shot device result and the oracle."""
    lines, cond, grid, cut = _mini(2, 30_000)
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    hl = {k: torch.as_tensor(v).pin_memory() for k, v in lines.items()}
    for block in (0, 7_000, 30_000, 100_000):
        k_host = op.compute_host(hl, cut, block_lines=block)
        st = op.stats()
        assert st["n_evals"] == evals and st["n_lines"] == 30_000
        check_parity(k_host.numpy(), k_ref, what=f"host pipeline block {block}")
    k_page = op.compute_host({k: torch.as_tensor(v) for k, v in lines.items()}, cut,
                             out=torch.empty(op.N, dtype=torch.float64), block_lines=9_000)   # pageable memory
    check_parity(k_page.numpy(), k_ref, what="host pipeline, pageable")
    dl = _to_cuda(lines)
    k = torch.zeros(op.N, dtype=torch.float64, device="cuda")
    for a, b in ((0, 11_000), (11_000, 11_000), (11_000, 30_000)):          # includes an empty block
        op.compute({f: v[a:b].contiguous() for f, v in dl.items()}, cut, out=k, accumulate=True)
    torch.cuda.synchronize()
    check_parity(k.cpu().numpy(), k_ref, what="hk_accumulate")
    op.close()


def test_batched_conditions(B):
    """hk_compute_batch (the paper's many pressure points per run, L361, L733): every row of the
    batch is the definition at that (T, P, Q) -- checked against the oracle per condition -- and equals the one-shot
    hk_compute at that condition bit for bit (the shared sort changes no arithmetic)."""
    lines, cond, grid, cut = _mini(2, 20_000)
    T = [300.0, 1500.0, 1500.0, 2900.0]
    P = [1e-3, cond["P_atm"], 25.0, 0.3]
    Q = [170.0, cond["Q"], cond["Q"], 9000.0]
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    dl = _to_cuda(lines)
    kb = op.compute_batch(dl, cut, T, P, Q)
    torch.cuda.synchronize()
    assert kb.shape == (4, op.N)
    st = op.stats()
    for c in range(4):
        cnd = dict(T=T[c], P_atm=P[c], mass_amu=cond["mass_amu"], Q=Q[c])
        k_ref, evals = O.opacity_grid(lines, cnd, grid, cut)
        assert st["n_evals"] == evals
        check_parity(kb[c].cpu().numpy(), k_ref, what=f"batch condition {c}")
        op1 = B.Opacity(*grid)
        op1.set_conditions(T[c], P[c], cond["mass_amu"], Q[c])
        op1.set_core_nodes(False)            # (a batch keeps the core out of the node hierarchy: its ranges serve several conditions)
        k1 = op1.compute(dl, cut)
        torch.cuda.synchronize()
        big = k_ref >= 1e-8 * k_ref.max()
        assert np.abs(kb[c].cpu().numpy()[big] / k1.cpu().numpy()[big] - 1.0).max() <= 1e-6   # atomics order only
        op1.close()
    # the handle's own conditions are untouched; an empty batch and a bad condition
    k_after = op.compute(dl, cut)
    k_ref, _ = O.opacity_grid(lines, cond, grid, cut)
    check_parity(k_after.cpu().numpy(), k_ref, what="after batch")
    assert op.compute_batch(dl, cut, [], [], []).shape == (0, op.N)
    with pytest.raises(B.HKError) as e:
        op.compute_batch(dl, cut, [300.0, -1.0], [1.0, 1.0], [10.0, 10.0])
    assert e.value.status == B.HK_EINVAL
    op.close()


@pytest.mark.parametrize("cfg,n", [(2, 20_000), (4, 6_000), (5, 300)])
def test_batch_pressure_sweep(B, cfg, n):
    """The paper's use of a batch: many PRESSURES at one temperature (L361, L733).  From the second point on only the
    Lorentz widths are recomputed (rewidth_kernel: same order, ranges and node lists); every point against the oracle,
    P = 0 (natural widths only) included."""
    lines, cond, grid, cut = _mini(cfg, n)
    P = [1e-3, 0.0, 1.0, 30.0, 0.2]
    T, Q = [cond["T"]] * len(P), [cond["Q"]] * len(P)
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    dl = _to_cuda(lines)
    kb = op.compute_batch(dl, cut, T, P, Q).cpu().numpy()
    torch.cuda.synchronize()
    st = op.stats()
    for c in range(len(P)):
        cnd = dict(T=T[c], P_atm=P[c], mass_amu=cond["mass_amu"], Q=Q[c])
        k_ref, evals = O.opacity_grid(lines, cnd, grid, cut)
        assert st["n_evals"] == evals
        rel, ab, frac = check_parity(kb[c], k_ref, what=f"config {cfg} pressure point {c} (P = {P[c]} atm)")
        print(f"pressure sweep config {cfg} P={P[c]:g}: rel={rel:.2e} abs={ab:.2e}")
    op.close()


def _oracle_illcond(lines, cond, grid, cut, slack=1.0):
    """Oracle-side count of the lines (with an extent) whose value at the fixed cutting length exceeds 1/512 of their
    peak value (HK_PLINTH_RATIO: the accuracy contract of hk_set_plinth); slack scales the threshold."""
    S_, gL_, aD_, valid_ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    ilo_, ihi_, _ = O.extents(lines["nu0"], valid_, grid[0], grid[2], O.grid_size(*grid), cut)
    live = (valid_ > 0) & (ihi_ >= ilo_)
    y = gL_[live] / aD_[live]
    ratio = O.voigt_K(cut / aD_[live], y) / O.voigt_K(np.zeros_like(y), y)
    return int((ratio * 512.0 * slack > 1.0).sum())


def _check_plinth(op, k, k_ref, k_raw, what):
    """The accuracy contract of hk_set_plinth (include/hk.h): while every line's value at its cutting length is below 1/512
    of its peak (hk_stats.n_plinth_illcond == 0) the SUBTRACTED opacity meets the north_star pair, up to the rounding of
    the two fp32 terms (2^-22 of the opacity before removal: seen only in the last bins before the extent end of an
    isolated line, found by the randomised test at 300 seeds); otherwise the opacity before removal is the reference
    magnitude (R27)."""
    in_core = op.stats()["n_plinth_illcond"]
    if in_core == 0:
        return check_parity_subtracted(k, k_ref, k_raw, what=what + " (subtracted reference)"), in_core
    return check_parity_plinth(k, k_ref, k_raw, what=what + f" ({in_core} ill-conditioned lines)"), in_core


@pytest.mark.parametrize("case", ["config2", "config3", "config4", "resolved", "tiny_cut", "edge_off"])
def test_plinth_removal(B, case):
    """hk_set_plinth (section 2.1.1): every line's value at the cutting length removed from
    its bins, against the oracle's plinth option: the north_star pair with the opacity before removal as the reference
    magnitude (R27), and -- wherever the cut lies outside the line cores -- against the subtracted value too."""
    if case in ("config2", "edge_off"):
        lines, cond, grid, cut = _mini(2, 20_000)
    elif case == "config3":
        lines, cond, grid, cut = _mini(3, 200_000)
    elif case == "config4":
        lines, cond, grid, cut = _mini(4, 6_000)
    else:
        rng = np.random.default_rng(21)
        n = 1500
        lines = _simple_lines(np.sort(rng.uniform(995.0, 1025.0, n)), A=10 ** rng.uniform(-3, 2, n),
                              E_low=rng.uniform(0, 4000, n), gamma_ref=rng.uniform(0.01, 0.2, n))
        cond, grid = COND, (1000.0, 1020.5, 0.001)
        cut = 3.0 if case == "resolved" else 0.004            # tiny: the cut falls inside the line cores
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_plinth(True)
    op.set_edge_nodes(case != "edge_off")
    k = op.compute(_to_cuda(lines), cut)
    torch.cuda.synchronize()
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut, plinth=True)
    k_raw, _ = O.opacity_grid(lines, cond, grid, cut)
    assert op.stats()["n_evals"] == evals
    assert (k_ref < k_raw).any()
    # the library's count of lines with V(cut) > V(0)/512, against the oracle's profile (threshold +- 1 %)
    n_in = op.stats()["n_plinth_illcond"]
    assert _oracle_illcond(lines, cond, grid, cut, 0.99) <= n_in <= _oracle_illcond(lines, cond, grid, cut, 1.01)
    assert (n_in > 0) == (case == "tiny_cut")
    # every other case: the SUBTRACTED opacity at the plain north_star tolerance; tiny_cut: the cut lies inside the cores,
    # the opacity before removal is the reference magnitude (hk.h, R27; PAPER.md L57-59 with L367)
    rel, n_in = _check_plinth(op, k.cpu().numpy(), k_ref, k_raw, f"plinth {case}")
    print(f"plinth {case}: rel={rel:.2e} ill-conditioned lines {n_in} removed fraction of the integral {1 - k_ref.sum() / k_raw.sum():.3f}")
    # uncut: no plinth
    if case == "config2":
        ku = op.compute(_to_cuda(lines), 0.0)
        op.set_plinth(False)
        ku0 = op.compute(_to_cuda(lines), 0.0)
        torch.cuda.synchronize()
        assert torch.equal(ku, ku0) or float((ku / ku0 - 1).abs().max()) <= 1e-6
    op.close()


@pytest.mark.parametrize("profile", ["lorentz", "doppler", "binned_gaussian"])
@pytest.mark.parametrize("case", ["config2", "config3", "resolved", "uncut"])
def test_lorentz_and_doppler_profiles(B, profile, case):
    """hk_set_profile (section 2.1) against the oracle's profile options, with and
    without plinth removal."""
    if case == "config2":
        lines, cond, grid, cut = _mini(2, 20_000)
    elif case == "config3":
        lines, cond, grid, cut = _mini(3, 200_000)
    elif case == "uncut":
        lines, cond, grid, cut = _mini(5, 300)
        grid = (grid[0], 5000.0, grid[2])
    else:
        rng = np.random.default_rng(22)
        n = 1500
        lines = _simple_lines(np.sort(rng.uniform(995.0, 1025.0, n)), A=10 ** rng.uniform(-3, 2, n),
                              E_low=rng.uniform(0, 4000, n), gamma_ref=rng.uniform(0.01, 0.2, n))
        cond, grid, cut = COND, (1000.0, 1020.5, 0.001), 3.0
    dl = _to_cuda(lines)
    for plinth in (False, True):
        op = B.Opacity(*grid)
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        op.set_profile(profile)
        op.set_plinth(plinth)
        k = op.compute(dl, cut)
        torch.cuda.synchronize()
        k_ref, evals = O.opacity_grid(lines, cond, grid, cut, plinth=plinth, profile=profile)
        assert op.stats()["n_evals"] == evals
        rel, ab, frac = check_parity(k.cpu().numpy(), k_ref, what=f"{profile} {case} plinth={plinth}")
        print(f"{profile} {case} plinth={plinth}: rel={rel:.2e} abs={ab:.2e} frac_rel={frac:.3f}")
        op.close()
    with pytest.raises(B.HKError):
        B.Opacity(*grid).set_profile(7)


def test_hitran_style_inputs(B):
    """hk_compute_hitran: Eq. 4 air/self broadening, pressure shift, isotopologue table, against
    the oracle's HITRAN path -- per-line parameters to 1e-12, integer extents of the SHIFTED centres exactly, k(nu) at
    the north_star tolerance -- plus the reduction to the ExoMol entry point."""
    n = 20_000
    hl = W.make_lines_hitran(n, seed=0)
    lines = {k: v.numpy() for k, v in hl.items()}
    lines["iso"][17] = 9                                       # outside the table: skipped
    cond, grid, cut = dict(W.HITRAN_COND), W.CONFIGS[2]["grid"], W.CONFIGS[2]["cut"]
    dl = {k: torch.as_tensor(v).cuda() for k, v in lines.items()}
    op = B.Opacity(*grid)
    with pytest.raises(B.HKError) as e:
        op.compute_hitran(dl, cut)
    assert e.value.status == B.HK_ESTATE
    op.set_conditions_hitran(cond["T"], cond["P_atm"], cond["P_self_atm"], cond["isos"])
    k = op.compute_hitran(dl, cut)
    torch.cuda.synchronize()
    st = op.stats()
    S0, gL0, aD0, ctr, valid = O.line_params_hitran(lines, cond)
    assert st["n_skipped"] == 1 and valid.sum() == n - 1
    # hk_get_extents returns what that compute wrote (shifted centres), without the lines
    r_ilo, r_ihi, r_jc = (t.cpu().numpy() for t in op.extents(None, n=n))
    S, gL, aD, ilo, ihi, jc = (t.cpu().numpy() for t in op.line_params_hitran(dl, cut))
    v = valid > 0
    assert np.array_equal(r_ilo, ilo) and np.array_equal(r_ihi, ihi) and np.array_equal(r_jc[v], jc[v])
    assert np.abs(S[v] / S0[v] - 1).max() <= 1e-12 and np.abs(gL[v] / gL0[v] - 1).max() <= 1e-12
    assert np.abs(aD[v] / aD0[v] - 1).max() <= 1e-13
    N = O.grid_size(*grid)
    ilo0, ihi0, jc0 = O.extents(ctr, valid, grid[0], grid[2], N, cut)
    empty = ilo0 > ihi0
    assert np.array_equal(ilo.astype(np.int64), np.where(empty, 0, ilo0))
    assert np.array_equal(ihi.astype(np.int64), np.where(empty, -1, ihi0))
    assert np.array_equal(jc.astype(np.int64)[v], jc0[v])
    assert (jc0[v] != np.floor((lines["nu0"][v] - grid[0]) / grid[2])).mean() > 0.5      # the shift really moves bins
    k_ref, evals = O.opacity_grid_hitran(lines, cond, grid, cut)
    assert st["n_evals"] == evals
    rel, ab, frac = check_parity(k.cpu().numpy(), k_ref, what="hitran")
    print(f"hitran: rel={rel:.2e} abs={ab:.2e} frac_rel={frac:.3f}")
    with pytest.raises(B.HKError):
        op.set_conditions_hitran(1000.0, 1.0, 2.0, cond["isos"])           # P_self > P
    # one isotopologue, air = self, no shift: the ExoMol entry point on the same handle
    ex = W.to_numpy(W.make_lines(2, n=5000, seed=0))
    h1 = {k2: ex[k2] for k2 in ("nu0", "A", "g_up", "E_low", "n_exp")}
    h1.update(gamma_air=ex["gamma_ref"], gamma_self=ex["gamma_ref"], delta=np.zeros(5000), iso=np.zeros(5000, dtype=np.int32))
    op.set_conditions_hitran(1500.0, 0.9, 0.2, [(18.0, 2000.0, 1.0)])
    ka = op.compute_hitran({k2: torch.as_tensor(v2).cuda() for k2, v2 in h1.items()}, cut).clone()
    kb = op.compute(_to_cuda(ex), cut)
    torch.cuda.synchronize()
    big = kb >= 1e-8 * kb.max()
    assert float((ka[big] / kb[big] - 1).abs().max()) <= 1e-6
    op.close()


@pytest.mark.parametrize("seed", range(6))
def test_pressure_shift_moves_wide_cores(B, seed):
    """Tile classification under pressure shift (R23): the profile is centred at nu0 + delta P while alpha_D uses
    the tabulated nu0.  Lines at 1-20 cm^-1 shifted DOWN by up to half their wavenumber, a light species and a fine grid:
    the true core is up to twice as wide as beta x (shifted centre) and dozens of tiles across.  The library bounds
    alpha_D with the largest |delta P| of the list (apply_shift_bound), so the classification is safe by construction."""
    rng = np.random.default_rng(31000 + seed)
    n = 400
    nu0 = rng.uniform(1.0, 20.0, n)
    P = float(rng.choice([1.0, 3.0]))
    lines = dict(nu0=nu0, A=10 ** rng.uniform(-8, -4, n), g_up=rng.integers(1, 9, n).astype(float),
                 E_low=rng.uniform(0, 500, n), gamma_air=10 ** rng.uniform(-4.5, -3.0, n), gamma_self=10 ** rng.uniform(-4.5, -3.0, n),
                 n_exp=rng.uniform(0.4, 0.8, n), delta=-rng.uniform(0.0, 0.5, n) * nu0 / P, iso=np.zeros(n, dtype=np.int32))
    lines["delta"][::7] *= -0.2                                   # a few shifted up as well
    cond = dict(T=float(rng.uniform(1500, 3000)), P_atm=P, P_self_atm=0.3 * P, isos=[(float(rng.choice([1.008, 2.016, 4.0])), 30.0, 1.0)])
    grid = (0.25, 21.0, 2.0e-5)
    cut = float(rng.choice([0.05, 0.4]))
    dl = {k: torch.as_tensor(v).cuda() for k, v in lines.items()}
    op = B.Opacity(*grid)
    op.set_conditions_hitran(cond["T"], cond["P_atm"], cond["P_self_atm"], cond["isos"])
    k = op.compute_hitran(dl, cut)
    torch.cuda.synchronize()
    st = op.stats()
    S0, gL0, aD0, ctr, valid = O.line_params_hitran(lines, cond)
    a_bins = aD0 / grid[2]
    assert a_bins.max() > 8.0 and (np.abs(lines["delta"]) * P).max() > 2.0          # cores hundreds of bins across, shifts of cm^-1
    k_ref, evals = O.opacity_grid_hitran(lines, cond, grid, cut)
    assert st["n_evals"] == evals
    rel, ab, frac = check_parity(k.cpu().numpy(), k_ref, what=f"pressure shift {seed}")
    print(f"pressure shift {seed}: rel={rel:.2e} abs={ab:.2e} alpha_D up to {a_bins.max():.1f} bins, levels {st['n_levels']}")
    op.close()


@pytest.mark.parametrize("mode,factor", [("lorentz", 500.0), ("lorentz", 40.0), ("doppler", 3000.0)])
@pytest.mark.parametrize("case", ["config2", "config3", "resolved"])
def test_width_relative_cutting_length(B, case, mode, factor):
    """hk_set_cut_mode: the cutting length of a line is a multiple of its own Lorentz
    or Doppler half-width.  Integer extents exact, k(nu) at the north_star tolerance, with and without plinth removal."""
    if case == "config2":
        lines, cond, grid, _ = _mini(2, 20_000)
    elif case == "config3":
        lines, cond, grid, _ = _mini(3, 100_000)
    else:
        rng = np.random.default_rng(23)
        n = 1500
        lines = _simple_lines(np.sort(rng.uniform(995.0, 1025.0, n)), A=10 ** rng.uniform(-3, 2, n),
                              E_low=rng.uniform(0, 4000, n), gamma_ref=rng.uniform(0.01, 0.2, n))
        cond, grid = COND, (1000.0, 1020.5, 0.001)
    dl = _to_cuda(lines)
    S, gL, aD, valid = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    hw = gL if mode == "lorentz" else aD * np.sqrt(np.log(2.0))
    N = O.grid_size(*grid)
    for plinth in (False, True):
        op = B.Opacity(*grid)
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        op.set_cut_mode(mode)
        op.set_plinth(plinth)
        k = op.compute(dl, factor)
        torch.cuda.synchronize()
        st = op.stats()
        k_ref, evals = O.opacity_grid(lines, cond, grid, factor, plinth=plinth, cut_mode=mode)
        assert st["n_evals"] == evals and st["n_lines"] == len(hw)
        g_ilo, g_ihi, _ = (t.cpu().numpy().astype(np.int64) for t in op.extents(dl))
        # the oracle's extent formula with each line's own cutting length
        c = factor * hw
        ilo = np.maximum(np.ceil((lines["nu0"] - c - grid[0]) / grid[2]), 0).astype(np.int64)
        ihi = np.minimum(np.floor((lines["nu0"] + c - grid[0]) / grid[2]), N - 1).astype(np.int64)
        empty = ilo > ihi
        assert np.array_equal(g_ilo, np.where(empty, 0, ilo)) and np.array_equal(g_ihi, np.where(empty, -1, ihi))
        assert int((g_ihi - g_ilo + 1).sum()) == evals
        if plinth:
            k_raw, _ = O.opacity_grid(lines, cond, grid, factor, cut_mode=mode)
            # (40 Gamma_L puts the cut inside the core, |z| < 25, of every line with y < 0.6: counted by the library)
            (rel, n_in), ab = _check_plinth(op, k.cpu().numpy(), k_ref, k_raw, f"cut {mode} x{factor} {case} plinth"), 0.0
        else:
            rel, ab, frac = check_parity(k.cpu().numpy(), k_ref, what=f"cut {mode} x{factor} {case} plinth={plinth}")
        print(f"cut {mode} x{factor} {case} plinth={plinth}: rel={rel:.2e} abs={ab:.2e} cuts {c.min():.3g}..{c.max():.3g} cm^-1")
        op.close()


def test_bands_of_different_resolution(B):
    """hk_compute_bands: three bands at 0.05 / 0.01 / 0.1 cm^-1; every band against the oracle on its own
    grid (lines near a band edge reach into both bands)."""
    lines, cond, _, cut = _mini(2, 20_000)
    bands = [(0.0, 3000.0, 0.05), (3000.0, 4200.0, 0.01), (4200.0, 10000.0, 0.1)]
    ops = []
    for g in bands:
        op = B.Opacity(*g)
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        ops.append(op)
    outs = B.compute_bands(ops, _to_cuda(lines), cut)
    torch.cuda.synchronize()
    total = 0
    for g, op, k in zip(bands, ops, outs):
        k_ref, evals = O.opacity_grid(lines, cond, g, cut)
        assert op.stats()["n_evals"] == evals
        total += evals
        check_parity(k.cpu().numpy(), k_ref, what=f"band {g}")
    assert total > 0
    with pytest.raises(B.HKError) as e:
        B.compute_bands(ops + [B.Opacity(0.0, 1.0, 0.1)], _to_cuda(lines), cut)      # a band without conditions
    assert e.value.status == B.HK_ESTATE
    for op in ops:
        op.close()


@pytest.mark.parametrize("seed", range(N_FUZZ))
def test_randomised_small_cases(B, seed):
    """Differential fuzz: random grids (offset, span, resolution from 1e-3 to 1 cm^-1), cuts from below a bin to beyond
    the grid or none, conditions, line densities from one line to dense, every tile geometry and both extent-end paths,
    against the oracle on all bins at the north_star tolerance, with exact integer work counts."""
    rng = np.random.default_rng(1000 + seed)
    dnu = float(10 ** rng.uniform(-3, 0))
    nbins = int(rng.integers(1, 60_000))
    numin = float(rng.choice([0.0, rng.uniform(0.0, 2.0e4)]))
    grid = (numin, numin + nbins * dnu, dnu)
    span = nbins * dnu
    cut = float(rng.choice([0.0, 10 ** rng.uniform(np.log10(0.3 * dnu), np.log10(3.0 * span + 10 * dnu))]))
    n = int(rng.choice([1, 2, 30, 400, 3000]))
    if seed % 4 == 3:                                  # dense: many lines per tile (the 8-warp centre kernel, long chunks)
        n = 20_000
        if nbins > 1500:
            nbins = int(rng.integers(1, 1500))
            grid = (numin, numin + nbins * dnu, dnu)
            span = nbins * dnu
    pad = min(cut if cut > 0 else 5.0, 50.0)
    nu0 = np.abs(rng.uniform(numin - pad, numin + span + pad, n)) + 1e-3
    if rng.random() < 0.3:
        nu0[: n // 2] = numin + dnu * rng.integers(0, nbins, n // 2)          # centres exactly on grid points
    lines = _simple_lines(nu0, A=10 ** rng.uniform(-6, 4, n), g_up=rng.integers(1, 30, n).astype(float),
                          E_low=rng.uniform(0, 8000, n), gamma_ref=10 ** rng.uniform(-3, -0.3, n),
                          n_exp=rng.uniform(0.4, 0.8, n))
    cond = dict(T=float(rng.uniform(200, 3000)), P_atm=float(10 ** rng.uniform(-3, 1.7)),
                mass_amu=float(rng.uniform(2, 200)), Q=float(10 ** rng.uniform(0, 4)))
    profile = str(rng.choice(["voigt", "voigt", "lorentz"]))
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_profile(profile)
    op.set_tile_bins(int(rng.choice([0, 2, 4, 8])))
    op.set_edge_nodes(bool(rng.integers(0, 2)))
    dl = _to_cuda(lines)
    k = op.compute(dl, cut)
    torch.cuda.synchronize()
    st = op.stats()
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut, profile=profile)
    ext = tuple(t.cpu().numpy() for t in op.extents(dl))
    assert _check_extents(ext, lines, cond, grid, cut) == evals == st["n_evals"]
    if k_ref.max() > 0:
        check_parity(k.cpu().numpy(), k_ref, what=f"fuzz {seed}: grid {grid} cut {cut:g} n {n} {profile} {cond}")
    else:
        assert float(k.abs().max()) == 0.0
    op.close()


@pytest.mark.parametrize("seed", range(N_FUZZ))
def test_randomised_variants(B, seed):
    """Differential fuzz of the variants: every profile, plinth removal, width-relative cutting lengths, in random
    combinations on random small problems, at the north_star tolerance (with plinth removal: the opacity before removal
    is the reference magnitude, R27)."""
    rng = np.random.default_rng(5000 + seed)
    dnu = float(10 ** rng.uniform(-3, -0.5))
    nbins = int(rng.integers(200, 40_000))
    numin = float(rng.choice([0.0, rng.uniform(0.0, 2.0e4)]))
    grid = (numin, numin + nbins * dnu, dnu)
    span = nbins * dnu
    n = int(rng.choice([3, 50, 800, 3000]))
    nu0 = np.abs(rng.uniform(numin - 2.0, numin + span + 2.0, n)) + 1e-3
    lines = _simple_lines(nu0, A=10 ** rng.uniform(-6, 4, n), g_up=rng.integers(1, 30, n).astype(float),
                          E_low=rng.uniform(0, 8000, n), gamma_ref=10 ** rng.uniform(-2.5, -0.3, n),
                          n_exp=rng.uniform(0.4, 0.8, n))
    cond = dict(T=float(rng.uniform(200, 3000)), P_atm=float(10 ** rng.uniform(-2, 1.7)),
                mass_amu=float(rng.uniform(2, 200)), Q=float(10 ** rng.uniform(0, 4)))
    profile = str(rng.choice(["voigt", "lorentz", "doppler", "binned_gaussian"]))
    plinth = bool(rng.integers(0, 2))
    mode = str(rng.choice(["fixed", "lorentz", "doppler"]))
    cut = float(10 ** rng.uniform(np.log10(2 * dnu), np.log10(span))) if mode == "fixed" else float(10 ** rng.uniform(1, 3.5))
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_profile(profile)
    op.set_plinth(plinth)
    op.set_cut_mode(mode)
    dl = _to_cuda(lines)
    k = op.compute(dl, cut).cpu().numpy()
    torch.cuda.synchronize()
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut, plinth=plinth, profile=profile, cut_mode=mode)
    what = f"variants {seed}: {profile} plinth={plinth} cut {mode} {cut:g} grid {grid} n {n} {cond}"
    assert op.stats()["n_evals"] == evals, what
    assert np.all(np.isfinite(k)), what
    if profile in ("doppler", "binned_gaussian"):
        # dynamic range of one launch (hk.h, R22): amplitudes carry one power-of-two scale, the largest
        # Gaussian amplitude at 2^100, so a term below 2^-226 (1e-68) of the largest line peak is flushed to zero.  A
        # spectrum that lies entirely below that -- no grid point within 12.5 Doppler widths of any line -- is all zero.
        peak = float((lambda S, gL, aD, v: (S / (aD * np.sqrt(np.pi))).max())(*O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])))
        k_unsub = k_ref if not plinth else O.opacity_grid(lines, cond, grid, cut, profile=profile, cut_mode=mode)[0]
        if k_unsub.max() < 1e-58 * peak:
            assert float(np.abs(k).max()) <= 1e-58 * peak
            op.close()
            return
    if plinth:
        k_raw = O.opacity_grid(lines, cond, grid, cut, profile=profile, cut_mode=mode)[0]
        if k_raw.max() > 0:
            _check_plinth(op, k, k_ref, k_raw, what)
        else:
            assert float(np.abs(k).max()) == 0.0
    elif k_ref.max() > 0:
        check_parity(k, k_ref, what=what)
    else:
        assert float(np.abs(k).max()) == 0.0
    op.close()


@pytest.mark.parametrize("seed", range(N_FUZZ))
def test_randomised_hitran(B, seed):
    """Differential fuzz of the HITRAN-style entry point: random self / air pressures, shifts of many bins, 1-4
    isotopologues, against the oracle (extent counts exact, north_star tolerance)."""
    rng = np.random.default_rng(9000 + seed)
    dnu = float(10 ** rng.uniform(-3, -0.5))
    nbins = int(rng.integers(50, 30_000))
    numin = float(rng.choice([0.0, rng.uniform(0.0, 2.0e4)]))
    grid = (numin, numin + nbins * dnu, dnu)
    span = nbins * dnu
    n = int(rng.choice([5, 300, 3000]))
    n_iso = int(rng.integers(1, 5))
    isos = [(float(rng.uniform(2, 200)), float(10 ** rng.uniform(0, 4)), float(10 ** rng.uniform(-4, 0))) for _ in range(n_iso)]
    P = float(10 ** rng.uniform(-3, 1.7))
    cond = dict(T=float(rng.uniform(200, 3000)), P_atm=P, P_self_atm=float(rng.uniform(0, 1) * P), isos=isos)
    lines = dict(nu0=np.abs(rng.uniform(numin - 3.0, numin + span + 3.0, n)) + 1e-3, A=10 ** rng.uniform(-6, 4, n),
                 g_up=rng.integers(1, 30, n).astype(float), E_low=rng.uniform(0, 8000, n),
                 gamma_air=10 ** rng.uniform(-2.5, -0.3, n), gamma_self=10 ** rng.uniform(-2.5, 0.0, n),
                 n_exp=rng.uniform(0.3, 0.9, n), delta=rng.uniform(-0.05, 0.05, n),
                 iso=rng.integers(0, n_iso + (1 if seed % 5 == 0 else 0), n).astype(np.int32))   # some outside the table
    cut = float(rng.choice([0.0, 10 ** rng.uniform(np.log10(2 * dnu), np.log10(span + 1.0))]))
    op = B.Opacity(*grid)
    op.set_conditions_hitran(cond["T"], cond["P_atm"], cond["P_self_atm"], isos)
    dl = {k2: torch.as_tensor(v2).cuda() for k2, v2 in lines.items()}
    k = op.compute_hitran(dl, cut).cpu().numpy()
    torch.cuda.synchronize()
    k_ref, evals = O.opacity_grid_hitran(lines, cond, grid, cut)
    what = f"hitran fuzz {seed}: grid {grid} cut {cut:g} n {n} {cond}"
    st = op.stats()
    assert st["n_evals"] == evals and st["n_skipped"] == int((lines["iso"] >= n_iso).sum()), what
    if k_ref.max() > 0:
        check_parity(k, k_ref, what=what)
    else:
        assert float(np.abs(k).max()) == 0.0
    op.close()


@pytest.mark.parametrize("seed", range(max(4, N_FUZZ // 4)))
def test_randomised_entry_points(B, seed):
    """The other entry points on random small problems: block-wise hk_accumulate, hk_compute_host with a random block
    size, hk_compute_batch with three conditions, hk_compute_bands -- each against the oracle."""
    rng = np.random.default_rng(13000 + seed)
    dnu = float(10 ** rng.uniform(-2.5, -0.5))
    nbins = int(rng.integers(100, 20_000))
    numin = float(rng.choice([0.0, rng.uniform(0.0, 1.0e4)]))
    grid = (numin, numin + nbins * dnu, dnu)
    span = nbins * dnu
    n = int(rng.choice([7, 500, 4000]))
    lines = _simple_lines(np.abs(rng.uniform(numin - 2.0, numin + span + 2.0, n)) + 1e-3, A=10 ** rng.uniform(-6, 4, n),
                          g_up=rng.integers(1, 30, n).astype(float), E_low=rng.uniform(0, 8000, n),
                          gamma_ref=10 ** rng.uniform(-2.5, -0.3, n), n_exp=rng.uniform(0.4, 0.8, n))
    cond = dict(T=float(rng.uniform(200, 3000)), P_atm=float(10 ** rng.uniform(-2, 1.7)),
                mass_amu=float(rng.uniform(2, 200)), Q=float(10 ** rng.uniform(0, 4)))
    cut = float(rng.choice([0.0, 10 ** rng.uniform(np.log10(2 * dnu), np.log10(span))]))
    plinth = bool(rng.integers(0, 2))
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut, plinth=plinth)
    k_raw = k_ref if not plinth else O.opacity_grid(lines, cond, grid, cut)[0]
    in_core0 = _oracle_illcond(lines, cond, grid, cut, 1.01) if (plinth and cut > 0) else 0

    def ok(k, ref=k_ref, raw=k_raw, what="", in_core=in_core0):
        tag = f"entry points {seed} {what}: cut {cut:g} plinth {plinth} grid {grid} n {n}"
        if plinth and in_core > 0:       # the contract of hk_set_plinth (hk.h): cut inside a line's core
            check_parity_plinth(np.asarray(k), ref, raw, what=tag)
        elif plinth and ref.max() > 0:   # ... and for well-conditioned lines: the subtracted value, up to the rounding of its terms
            check_parity_subtracted(np.asarray(k), ref, raw, what=tag)
        elif ref.max() > 0:
            check_parity(np.asarray(k), ref, what=tag)

    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_plinth(plinth)
    dl = _to_cuda(lines)
    # blocks through hk_accumulate
    k = torch.zeros(op.N, dtype=torch.float64, device="cuda")
    cuts = sorted(set([0, n] + [int(x) for x in rng.integers(0, n + 1, 3)]))
    for a0, a1 in zip(cuts[:-1], cuts[1:]):
        op.compute({f: v[a0:a1].contiguous() for f, v in dl.items()}, cut, out=k, accumulate=True)
    torch.cuda.synchronize()
    ok(k.cpu().numpy(), what="accumulate")
    # host pipeline
    hl = {f: torch.as_tensor(v).pin_memory() for f, v in lines.items()}
    kh = op.compute_host(hl, cut, block_lines=int(rng.integers(1, n + 5)))
    assert op.stats()["n_evals"] == evals
    ok(kh.numpy(), what="host")
    # batch: the handle's own condition in the middle
    Ts, Ps, Qs = [cond["T"] * 0.5, cond["T"], cond["T"] * 1.3], [cond["P_atm"] * 2, cond["P_atm"], 0.0], [cond["Q"], cond["Q"], 7.0]
    kb = op.compute_batch(dl, cut, Ts, Ps, Qs).cpu().numpy()
    ok(kb[1], what="batch[1]")
    for c in (0, 2):
        cc = dict(T=Ts[c], P_atm=Ps[c], mass_amu=cond["mass_amu"], Q=Qs[c])
        r = O.opacity_grid(lines, cc, grid, cut, plinth=plinth)[0]
        rr = r if not plinth else O.opacity_grid(lines, cc, grid, cut)[0]
        if rr.max() > 0:
            ok(kb[c], ref=r, raw=rr, what=f"batch[{c}]", in_core=_oracle_illcond(lines, cc, grid, cut, 1.01) if (plinth and cut > 0) else 0)
    op.close()


@pytest.mark.parametrize("cut", [25.0, 0.0])
def test_large_grid_few_lines(B, cut):
    """2e7 bins (beyond the 1 GiB budget of the per-bin extent-end accumulators: the direct edge kernel takes over, and
    the node hierarchy grows to its deepest), a few thousand lines; sampled bins against the oracle."""
    grid = (0.0, 20000.0, 0.001)
    n = 3000 if cut > 0 else 300
    lines = W.to_numpy(W.make_lines(2, n=n, seed=3))
    lines["nu0"] = lines["nu0"] * 2.0                      # spread over the whole grid
    cond = W.conditions(2)
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    k = op.compute(_to_cuda(lines), cut)
    torch.cuda.synchronize()
    st = op.stats()
    N = op.N
    assert N == 20_000_000 and st["n_pairs_edge_node"] == 0 and st["n_levels"] >= 5
    rng = np.random.default_rng(8)
    bins = set(rng.integers(0, N, 4000).tolist()) | {0, 1, N - 2, N - 1}
    S, _, _, _ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    for l in np.argsort(S)[-6:]:
        jc = int(lines["nu0"][l] / grid[2])
        for off in (0, int(cut / grid[2]) if cut > 0 else 5000):
            bins |= set(range(max(0, jc + off - 40), min(N, jc + off + 40))) | set(range(max(0, jc - off - 40), min(N, jc - off + 40)))
    jmax = int(k.argmax())
    bins |= set(range(max(0, jmax - 8), min(N, jmax + 8)))
    bins = np.array(sorted(bins), dtype=np.int64)
    k_ref, _ = O.opacity_bins(lines, cond, grid, cut, bins)
    kmax = float(k_ref.max())                    # the oracle's maximum (the GPU's argmax bin is sampled)
    assert float(k.max()) <= kmax * (1 + 1e-4)
    check_parity(k[torch.as_tensor(bins, device="cuda")].cpu().numpy(), k_ref, kmax=kmax, what=f"large grid cut {cut}")
    ilo, ihi, _ = op.extents(_to_cuda(lines))
    assert int((ihi.long() - ilo.long() + 1).sum()) == st["n_evals"]
    op.close()


@pytest.mark.parametrize("cut", [25.0, 0.0])
def test_billion_bin_grid(B, cut):
    """Towards the maximum grid size (N < 2^31): 1.2e9 bins at 1e-5 cm^-1, 500 lines; uncut that is 6e11 (line, bin)
    terms through 22 levels of the node hierarchy.  Sampled bins against the oracle."""
    free, _ = torch.cuda.mem_get_info()
    if free < 30e9:
        pytest.skip("needs ~16 GB of device memory")
    grid = (0.0, 12000.0, 1e-5)
    lines = W.to_numpy(W.make_lines(2, n=500, seed=4))
    cond = W.conditions(2)
    op = B.Opacity(*grid)
    assert op.N == 1_200_000_000
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    k = op.compute(_to_cuda(lines), cut)
    torch.cuda.synchronize()
    st = op.stats()
    assert st["n_evals"] == (500 * op.N if cut == 0.0 else st["n_evals"]) and st["n_levels"] >= 14
    rng = np.random.default_rng(1)
    jmax = int(k.argmax())
    bins = np.unique(np.concatenate([rng.integers(0, op.N, 3000), [0, op.N - 1], (lines["nu0"][:20] / grid[2]).astype(np.int64),
                                     np.arange(max(0, jmax - 8), min(op.N, jmax + 8))]))
    k_ref, _ = O.opacity_bins(lines, cond, grid, cut, bins)
    kmax = float(k_ref.max())                    # the oracle's maximum (the GPU's argmax bin is sampled)
    assert float(k.max()) <= kmax * (1 + 1e-4)
    check_parity(k[torch.as_tensor(bins, device="cuda")].cpu().numpy(), k_ref, kmax=kmax, what=f"1.2e9 bins cut {cut}")
    op.close()
    del k
    torch.cuda.empty_cache()


# ---- per-line parameters (step a1) ----------------------------------------------------

@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_line_params_and_extents(B, cfg):
    lines, cond, grid, cut = _mini(cfg, 100_000 if cfg != 1 else None)
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    dl = _to_cuda(lines)
    S, gL, aD = (t.cpu().numpy() for t in op.line_params(dl))
    S0, gL0, aD0, valid = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    assert valid.all()
    assert np.abs(S / S0 - 1).max() <= 1e-12
    assert np.abs(gL / gL0 - 1).max() <= 1e-12
    assert np.abs(aD / aD0 - 1).max() <= 1e-13
    op.compute(dl, cut)
    ext = tuple(t.cpu().numpy() for t in op.extents(dl))
    _check_extents(ext, lines, cond, grid, cut)
    op.close()


# ---- edge cases -------------------------------------------------------------------------

def _simple_lines(nu0, **kw):
    n = len(nu0)
    d = dict(nu0=np.asarray(nu0, dtype=np.float64), A=np.full(n, 1.0), g_up=np.full(n, 3.0),
             E_low=np.full(n, 100.0), gamma_ref=np.full(n, 0.05), n_exp=np.full(n, 0.6))
    d.update({k: np.asarray(v, dtype=np.float64) for k, v in kw.items()})
    return d


COND = dict(T=1200.0, P_atm=0.7, mass_amu=28.0, Q=300.0)


def test_empty_input(B):
    op = B.Opacity(0.0, 100.0, 0.1)
    op.set_conditions(1000.0, 1.0, 18.0, 100.0)
    lines = {k: torch.empty(0, dtype=torch.float64, device="cuda") for k in B.FIELDS}
    k = op.compute(lines, 25.0, out=torch.full((op.N,), 7.0, dtype=torch.float64, device="cuda"))
    torch.cuda.synchronize()
    assert float(k.abs().max()) == 0.0
    assert op.stats()["n_evals"] == 0


@pytest.mark.parametrize("grid,cut", [
    ((0.0, 0.1, 0.1), 25.0),            # N = 1
    ((100.0, 437.3, 0.1), 25.0),        # ragged tail (N = 3373), numin != 0
    ((100.0, 437.3, 0.1), 0.05),        # cut smaller than dnu: most extents empty or one bin
    ((100.0, 437.3, 0.1), 1.0e4),       # cut larger than the grid
    ((100.0, 437.3, 0.1), 0.0),         # uncut
    ((1000.0, 1020.5, 0.001), 3.0),     # fine grid, resolved lines (20500 bins)
    ((5.0, 3000.0, 1.0), 25.0),         # dnu >> widths
])
def test_edge_grids(B, grid, cut):
    rng = np.random.default_rng(11)
    numin, numax, dnu = grid
    span = numax - numin
    nu0 = np.concatenate([
        rng.uniform(numin - 30.0, numax + 30.0, 3000),          # includes off-grid centres whose wings reach in
        [numin, numax, numin + dnu * 7, numin + 0.5 * dnu, numax - dnu, numin - 25.0, numax + 25.0],
        numin + dnu * rng.integers(0, max(1, int(span / dnu)), 50),   # centres exactly on grid points
    ])
    nu0 = np.abs(nu0) + 1e-3
    n = nu0.size
    lines = _simple_lines(nu0, A=10 ** rng.uniform(-4, 3, n), g_up=rng.integers(1, 20, n).astype(float),
                          E_low=rng.uniform(0, 5000, n), gamma_ref=rng.uniform(0.01, 0.2, n),
                          n_exp=rng.uniform(0.5, 0.75, n))
    k_gpu, st, ext = _gpu_k(B, lines, COND, grid, cut)
    k_ref, evals = O.opacity_grid(lines, COND, grid, cut)
    assert _check_extents(ext, lines, COND, grid, cut) == evals == st["n_evals"]
    check_parity(k_gpu, k_ref, what=f"grid {grid} cut {cut}")


def test_bad_lines_are_skipped(B):
    rng = np.random.default_rng(3)
    n = 500
    lines = _simple_lines(rng.uniform(1.0, 200.0, n))
    bad = {0: ("nu0", 0.0), 1: ("nu0", -5.0), 2: ("nu0", np.nan), 3: ("A", -1.0), 4: ("A", np.inf),
           5: ("g_up", np.nan), 6: ("E_low", np.inf), 7: ("gamma_ref", np.nan), 8: ("n_exp", -np.inf)}
    for i, (f, v) in bad.items():
        lines[f][i] = v
    grid, cut = (0.0, 200.0, 0.05), 10.0
    k_gpu, st, ext = _gpu_k(B, lines, COND, grid, cut)
    assert st["n_skipped"] == len(bad)
    good = {k: np.delete(v, list(bad)) for k, v in lines.items()}
    k_ref, evals = O.opacity_grid(good, COND, grid, cut)
    assert st["n_evals"] == evals
    check_parity(k_gpu, k_ref, what="bad lines")
    k_all, _ = O.opacity_grid(lines, COND, grid, cut)          # the oracle applies the same rule (R14)
    assert np.array_equal(k_all, k_ref)
    _check_extents(ext, lines, COND, grid, cut)


def test_order_independence_and_linearity(B):
    lines, cond, grid, cut = _mini(2, 8000)
    k0, _, _ = _gpu_k(B, lines, cond, grid, cut)
    perm = np.random.default_rng(1).permutation(8000)
    k1, _, _ = _gpu_k(B, {k: v[perm] for k, v in lines.items()}, cond, grid, cut)
    big = k0 >= 1e-8 * k0.max()
    assert np.abs(k1[big] / k0[big] - 1).max() <= 1e-6                      # R16: order changes rounding only
    ka, _, _ = _gpu_k(B, {k: v[:3000] for k, v in lines.items()}, cond, grid, cut)
    kb, _, _ = _gpu_k(B, {k: v[3000:] for k, v in lines.items()}, cond, grid, cut)
    assert np.abs((ka + kb)[big] / k0[big] - 1).max() <= 1e-6


def test_strong_and_weak_lines_dynamic_range(B):
    """35 decades of line strength in one launch: the weak lines' bins fall in
    the absolute regime, but a launch of the weak lines alone must still be right."""
    rng = np.random.default_rng(9)
    n = 2000
    nu0 = np.sort(rng.uniform(50.0, 950.0, n))
    A = 10 ** rng.uniform(-10, 3, n)
    E = rng.uniform(0, 40000, n)
    lines = _simple_lines(nu0, A=A, E_low=E)
    grid, cut = (0.0, 1000.0, 0.01), 25.0
    cond = dict(T=700.0, P_atm=1.0, mass_amu=18.0, Q=1000.0)
    k_gpu, _, _ = _gpu_k(B, lines, cond, grid, cut)
    k_ref, _ = O.opacity_grid(lines, cond, grid, cut)
    check_parity(k_gpu, k_ref, what="35 decades")
    S, _, _, _ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    weak = S < np.quantile(S, 0.2)
    lw = {k: v[weak] for k, v in lines.items()}
    k_gpu, _, _ = _gpu_k(B, lw, cond, grid, cut)
    k_ref, _ = O.opacity_grid(lw, cond, grid, cut)
    check_parity(k_gpu, k_ref, what="weak lines alone")


def test_error_codes_on_device_box(B):
    op = B.Opacity(0.0, 10.0, 0.1)
    lines = _to_cuda(_simple_lines([1.0, 2.0]))
    with pytest.raises(B.HKError) as e:
        op.compute(lines, 1.0)                       # no conditions yet
    assert e.value.status == B.HK_ESTATE
    with pytest.raises(B.HKError) as e:
        op.set_conditions(-1.0, 1.0, 18.0, 1.0)
    assert e.value.status == B.HK_EINVAL
    op.set_conditions(300.0, 1.0, 18.0, 1.0)
    ws = torch.empty(256, dtype=torch.uint8, device="cuda")
    assert B._lib.hk_set_workspace(op._ctx, ws.data_ptr(), 256) == 0
    ls, n = B._lines_struct(lines)
    out = torch.empty(op.N, dtype=torch.float64, device="cuda")
    import ctypes as C
    assert B._lib.hk_compute(op._ctx, C.byref(ls), n, 1.0, out.data_ptr(), None) == B.HK_ENOSPC


# ---- the fp32 evaluator: measured accuracy map (our counterpart of Fig. 4) ------

def test_evaluator_accuracy_map(B):
    """Re w(x+iy) through the shipped fp32 device functions on a log lattice and at the
    region boundaries, against the oracle's w.  Budget per region: 3e-5."""
    xs = np.concatenate([[0.0], np.logspace(-3, 7, 640)])
    ys = np.logspace(-2, 7, 576)
    X, Y = np.meshgrid(xs, ys, indexing="ij")
    # region boundaries +- a few ulp
    for z2 in (B.HK_Z1, B.HK_Z2, B.HK_Z4, 36.0, B.HK_Z3, 21.0, 50.0, 88.0):
        for yv in np.logspace(-2, math.log10(math.sqrt(z2)) - 1e-3, 64):
            xb = math.sqrt(z2 - yv * yv)
            xe = xb * (1 + np.array([-4, -2, -1, 0, 1, 2, 4]) * 6e-8)
            X = np.concatenate([X.ravel(), xe])
            Y = np.concatenate([Y.ravel(), np.full(xe.size, yv)])
    # the values of y at which the rings change (z3_for, z4_for, HK_Y10: hk_device.cuh), from both sides, x dense across the core
    for yb in (1.0, 1.5, 1.8, 3.0, 4.5):
        for yv in (yb * (1 - 1e-6), yb, yb * (1 + 1e-6), yb * 1.03):
            xe = np.linspace(0.0, 8.0, 801)
            X = np.concatenate([X.ravel(), xe])
            Y = np.concatenate([Y.ravel(), np.full(xe.size, yv)])
    x32 = X.ravel().astype(np.float32)
    y32 = Y.ravel().astype(np.float32)
    out, reg = B.eval_voigt_f32(torch.from_numpy(x32).cuda(), torch.from_numpy(y32).cuda(), with_region=True)
    got = out.cpu().numpy().astype(np.float64)
    reg = reg.cpu().numpy()
    ref = O.voigt_K(x32.astype(np.float64), y32.astype(np.float64))
    ok = ref > 1e-30                     # below that the term is far under any bin's tolerance
    rel = np.abs(got - ref) / np.maximum(ref, 1e-300)
    for r, name in enumerate(("far", "mid", "gauss-hermite 4", "gauss-hermite 6", "trapezoid", "gauss-hermite 10")):
        m = ok & (reg == r)
        assert m.any()
        worst = rel[m].max()
        p999 = np.quantile(rel[m], 0.999)
        print(f"evaluator region {name}: n={m.sum()} max rel={worst:.2e} p99.9={p999:.2e}")
        assert worst <= 3e-5, (name, worst, x32[m][rel[m].argmax()], y32[m][rel[m].argmax()])


# ---- bench-size parity on sampled outputs ----------------------------------------------

def _full_size_sampled(B, cfg, n_windows, width, n=None, plinth=False, cut_override=None, special=False, twice=False):
    """The CUDA path on the whole workload; the oracle on sampled windows of contiguous bins, every bin summed over all
    lines within its cut.  Windows: stratified over the grid, always the first and the last; with special=True also the
    densest region of the list, the window holding the GPU's maximum and the bins at +- cut of the strongest line
    (SURVEY.md 8(d)).  max(k) of the tolerance is the ORACLE's value at the bin where the GPU has its maximum (checked
    to agree first), not a number taken from the GPU alone."""
    c = W.CONFIGS[cfg]
    cond, grid, cut = W.conditions(cfg), c["grid"], c["cut"]
    if cut_override is not None:
        cut = cut_override
    dl = W.make_lines(cfg, n=n, seed=0, device="cuda")
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_plinth(plinth)
    k = op.compute(dl, cut)
    torch.cuda.synchronize()
    st = op.stats()
    if twice:
        # what bench.py times is a REPEATED compute on one workspace: for a sorted list that is the single-pass
        # preprocess (line_sorted_kernel).  The windows below check that second result; the first one must agree with it.
        k_first = k.clone()
        st_first = st
        k = op.compute(dl, cut, out=k)
        torch.cuda.synchronize()
        st = op.stats()
        assert st_first["single_pass"] == 0 and st["single_pass"] == 1
        assert _stat_ints(st) == _stat_ints(st_first) and st["scale_exp"] == st_first["scale_exp"]
        assert float((k - k_first).abs().max() / k.max()) <= 2e-6      # (fp32 partial sums of <= 128 terms in another order)
        del k_first
    N = op.N
    rng = np.random.default_rng(cfg)
    wins = sample_windows(N, n_windows, width, rng)
    nu0 = dl["nu0"]
    sorted_in = bool((nu0[1:] >= nu0[:-1]).all())

    def clip(b0):
        b0 = int(max(0, min(N - width, b0)))
        return (b0, min(N, b0 + width))

    def oracle_window(b0, b1):
        if cut > 0:
            lo, hi = grid[0] + b0 * grid[2] - cut - 2 * grid[2], grid[0] + (b1 - 1) * grid[2] + cut + 2 * grid[2]
            if sorted_in:
                i0 = int(torch.searchsorted(nu0, torch.tensor([lo], dtype=torch.float64, device="cuda")))
                i1 = int(torch.searchsorted(nu0, torch.tensor([hi], dtype=torch.float64, device="cuda"), right=True))
                sub = {f: v[i0:i1].cpu().numpy() for f, v in dl.items()}
            else:
                sel = (nu0 >= lo) & (nu0 <= hi)
                sub = {f: v[sel].cpu().numpy() for f, v in dl.items()}
        else:
            sub = {f: v.cpu().numpy() for f, v in dl.items()}
        return O.opacity_bins(sub, cond, grid, cut, np.arange(b0, b1, dtype=np.int64), plinth=plinth)[0]

    # max(k): the oracle at the GPU's argmax window
    jmax = int(k.argmax())
    wmax = clip(jmax - width // 2)
    k_ref_max = oracle_window(*wmax)
    kmax = float(k_ref_max.max())
    assert abs(float(k[jmax]) / float(k_ref_max[jmax - wmax[0]]) - 1.0) <= 1e-4, "GPU maximum disagrees with the oracle"
    assert float(k.max()) <= kmax * (1.0 + 1e-4)
    check_parity(k[wmax[0]:wmax[1]].cpu().numpy(), k_ref_max, kmax=kmax, what=f"config {cfg} window of the maximum")
    if special:
        # densest region of the list: the window around the median centre of the densest 1/64 of the grid
        hist = torch.histc(nu0, bins=64, min=grid[0], max=grid[1])
        dens = int(hist.argmax())
        wins.append(clip(int((dens + 0.5) * N / 64) - width // 2))
        # the strongest line: its centre and the bins at +- cut
        S, _, _ = op.line_params(dl)
        ls = int(S.argmax())
        jc = int((float(nu0[ls]) - grid[0]) / grid[2])
        del S
        wins.append(clip(jc - width // 2))
        if cut > 0:
            cb = int(round(cut / grid[2]))
            wins.append(clip(jc - cb - width // 2))
            wins.append(clip(jc + cb - width // 2))
    worst = 0.0
    for b0, b1 in sorted(set(wins)):
        k_ref = oracle_window(b0, b1)
        rel, _, _ = check_parity(k[b0:b1].cpu().numpy(), k_ref, kmax=kmax, what=f"config {cfg} window {b0}")
        worst = max(worst, rel)
    # exact integer work count from the extents, all lines (O(n))
    ilo, ihi, _ = op.extents(dl)
    assert int((ihi.long() - ilo.long() + 1).sum()) == st["n_evals"]
    op.close()
    return worst, st


def test_config2_full_size_sampled(B):
    worst, st = _full_size_sampled(B, 2, 24, 64)
    print(f"config 2 full: worst rel {worst:.2e}, evals {st['n_evals']:.3e}")


def test_config5_full_size_sampled(B):
    worst, st = _full_size_sampled(B, 5, 12, 32)
    assert st["n_evals"] == 200_000 * 5_000_000
    print(f"config 5 full: worst rel {worst:.2e}")


@pytest.mark.parametrize("cfg,plinth,cut", [(3, False, None), (4, False, None), (3, True, None), (3, False, 25.037), (4, False, 99.99631)])
def test_bt2_shaped_full_size_sampled(B, cfg, plinth, cut):
    """The bench workload (config 4) and its coarse twin (config 3) at 5e8 lines, in the launch
    configuration bench.py times; the oracle sums every line within the cut on sampled bins."""
    import gc
    gc.collect()
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 120e9:
        pytest.skip("needs ~110 GB of device memory")
    if not plinth and cut is None:
        # the plain headline configs: 64 windows x 64 bins, with the special windows
        worst, st = _full_size_sampled(B, cfg, 60, 64, special=True, twice=True)
    else:
        worst, st = _full_size_sampled(B, cfg, 6 if cfg == 4 else 10, 8 if cfg == 4 else 32, plinth=plinth, cut_override=cut)
    print(f"config {cfg} full (plinth {plinth}): worst rel {worst:.2e}, evals {st['n_evals']:.3e}")


# ---- degenerate widths and the far end of the Gaussian ---------------------------------

@pytest.mark.parametrize("profile", ["lorentz", "voigt"])
def test_zero_width_line_on_a_grid_point(B, profile):
    """A line of zero Lorentz width (A = 0, P = 0) centred exactly on a grid point: 1/q is not finite there.  Its
    strength is zero (A = 0), so the spectrum is that of the other lines -- and must stay finite."""
    rng = np.random.default_rng(31)
    grid, cut = (100.0, 140.0, 0.01), 5.0
    nu0 = np.concatenate([rng.uniform(100.0, 140.0, 200), 100.0 + 0.01 * rng.integers(0, 4000, 20)])
    A = np.concatenate([10 ** rng.uniform(-2, 2, 200), np.zeros(20)])
    lines = _simple_lines(nu0, A=A)
    cond = dict(T=900.0, P_atm=0.0, mass_amu=30.0, Q=100.0)          # P = 0: Gamma_L = A/(4 pi c), zero for A = 0
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_profile(profile)
    k = op.compute(_to_cuda(lines), cut).cpu().numpy()
    assert np.all(np.isfinite(k))
    live = {f: v[:200] for f, v in lines.items()}
    k_ref, _ = O.opacity_grid(live, cond, grid, cut, profile=profile)
    check_parity(k, k_ref, what=f"zero-width line on a grid point, {profile}")
    op.close()


@pytest.mark.parametrize("mix", ["y_large", "y_tiny", "mixed"])
def test_lane_candidate_range_follows_the_widest_inner_region(B, mix):
    """range_kernel lists, per tile, the lines that can have innermost (lane-pass) bins there, from the largest
    z3_for(y^2) over the launch's lines: 30.25 where y^2 >= 1e-6 throughout, 50 once a line lies below that (157 with a
    pure Gaussian: the Doppler-profile tests).  Wide lines (alpha_D ~ 15 bins: the inner region spans several level-0
    tiles) of either kind, alone and mixed in one list, all bins against the oracle -- a range one class too tight
    would drop the outer part of the inner region of the tiny-y lines."""
    rng = np.random.default_rng(77)
    grid, cut = (20000.0, 20060.0, 0.005), 6.0
    n = 240
    nu0 = np.sort(rng.uniform(20000.5, 20059.5, n))
    tiny = {"y_large": np.zeros(n, bool), "y_tiny": np.ones(n, bool), "mixed": rng.random(n) < 0.1}[mix]
    # beta = sqrt(2 k T / m)/c = 3.7e-6 at 3000 K, m = 40: alpha_D = 0.074 cm^-1 = 15 bins; y = 0.17 or 7e-5
    cond = dict(T=3000.0, P_atm=1.0, mass_amu=40.0, Q=10.0)
    lines = _simple_lines(nu0, A=10 ** rng.uniform(-1, 1, n), gamma_ref=np.where(tiny, 2.0e-5, 0.05))
    _, gL, aD, _ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    y2 = (gL / aD) ** 2
    assert np.all(y2[tiny] < 1e-6) and np.all(y2[~tiny] > 1e-3) and 10 < np.median(aD) / grid[2] < 20
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    k = op.compute(_to_cuda(lines), cut).cpu().numpy()
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut)
    st = op.stats()
    assert st["n_evals"] == evals and st["n_evals_trap"] > 0
    rel, ab, _ = check_parity(k, k_ref, what=f"lane candidate range, {mix}")
    print(f"lane candidate range {mix}: rel={rel:.2e} abs={ab:.2e}, innermost evaluations {st['n_evals_trap']}")
    op.close()


def test_binned_gaussian_narrow_lines_at_bin_edges(B):
    """Lines 3000 times narrower than a bin whose centres lie within a few alpha_D of a bin edge (R26): the
    neighbouring bin's share, erfc((edge - nu0)/alpha_D)/2, needs the sub-bin offset to better than one fp32."""
    cond = dict(T=100.0, P_atm=0.5, mass_amu=200.0, Q=50.0)
    grid, cut = (900.0, 1100.0, 1.0), 30.0
    aD = 1000.0 / 2.99792458e10 * math.sqrt(2 * 1.380649e-16 * 100.0 / (200.0 / 6.02214076e23))
    ks = np.linspace(-4.5, 4.5, 37)
    nu0 = 900.0 + (np.arange(ks.size) * 5 + 7 + 0.5) * 1.0 + ks * aD      # isolated lines, one per 5 bins
    lines = _simple_lines(nu0, A=np.full(ks.size, 3.0))
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_profile("binned_gaussian")
    k = op.compute(_to_cuda(lines), cut).cpu().numpy()
    k_ref, evals = O.opacity_grid(lines, cond, grid, cut, profile="binned_gaussian")
    assert op.stats()["n_evals"] == evals
    assert ((k_ref > 1e-8 * k_ref.max()) & (k_ref < 1e-3 * k_ref.max())).sum() >= 10       # small edge shares are there
    rel, ab, frac = check_parity(k, k_ref, what="binned Gaussian at bin edges")
    print(f"binned Gaussian, narrow lines at bin edges: rel={rel:.2e}")
    op.close()


@pytest.mark.parametrize("xnear", [6.0, 9.5, 12.0])
def test_doppler_far_tail(B, xnear):
    """Pure Doppler lines whose nearest grid point is xnear Doppler widths away: the whole spectrum is the far Gaussian
    tail (e^-36 ... e^-144 of the peaks), inside the dynamic range of one launch (hk.h), so it must still be right."""
    cond = dict(T=300.0, P_atm=1.0, mass_amu=40.0, Q=10.0)
    grid, cut = (2000.0, 2040.0, 0.1), 3.0
    beta = math.sqrt(2 * 1.380649e-16 * 300.0 / (40.0 / 6.02214076e23)) / 2.99792458e10
    gp = 2000.0 + 0.1 * (np.arange(20) * 17 + 11)                  # grid points, one line next to each
    nu0 = gp + xnear * beta * gp * np.where(np.arange(20) % 2 == 0, 1.0, -1.0)      # xnear alpha_D (< half a bin) away
    lines = _simple_lines(nu0, A=10 ** np.linspace(-1, 3, 20))
    op = B.Opacity(*grid)
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    op.set_profile("doppler")
    k = op.compute(_to_cuda(lines), cut).cpu().numpy()
    k_ref, _ = O.opacity_grid(lines, cond, grid, cut, profile="doppler")
    S, _, aDl, _ = O.line_params(lines, cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    peak = (S / (aDl * np.sqrt(np.pi))).max()
    assert 1e-66 * peak < k_ref.max() < 1e-12 * peak
    rel, ab, frac = check_parity(k, k_ref, what=f"Doppler far tail x = {xnear}")
    print(f"Doppler far tail x={xnear}: max k / peak = {k_ref.max() / peak:.2e}, rel={rel:.2e}")
    op.close()
