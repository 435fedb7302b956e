"""hk_compute_static (include/hk.h): the hot path on the library's static device workspace, for callers that cannot
allocate device memory.  Collected last (the name sorts after every other test file): checked against hk_compute on the
same inputs, at the tolerance of the parity tests, on two calls in a row -- and against the oracle on all bins."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

from oracle import hk_oracle as O
from workload import linelists as W

from parity_util import check_parity

pytestmark = pytest.mark.gpu


def _cuda(lines_np):
    return {k: torch.as_tensor(np.ascontiguousarray(v), dtype=torch.float64).cuda() for k, v in lines_np.items()}


def test_static_workspace_matches_hk_compute_twice_in_a_row():
    from paper_2101_02005_b200 import binding as B
    # config 1 at full size (1e4 lines, 2e4 bins) and a second, different problem on the same static array: config 2's
    # generator (unsorted list) on a window of its grid, most lines off the grid
    c1 = W.CONFIGS[1]
    cases = [(W.to_numpy(W.make_lines(1, seed=0)), W.conditions(1), c1["grid"], c1["cut"]),
             (W.to_numpy(W.make_lines(2, n=60_000, seed=3)), W.conditions(2), (3600.0, 3900.0, 0.01), 25.0)]
    for lines, cond, grid, cut in cases:
        n = len(lines["nu0"])
        dl = _cuda(lines)
        ref_op = B.Opacity(*grid)
        ref_op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        assert ref_op.workspace_bytes(n) <= B.HK_STATIC_WS_BYTES
        k_ref_gpu = ref_op.compute(dl, cut).cpu().numpy()          # the existing path, on a workspace of its own
        st_ref = ref_op.stats()
        ref_op.close()
        k_oracle, evals = O.opacity_grid(lines, cond, grid, cut)

        op = B.Opacity(*grid)                                      # no workspace is ever bound to this context
        op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
        out = torch.full((op.N,), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        free = []
        for call in range(2):
            out.fill_(float("nan"))                                # the call overwrites every bin
            torch.cuda.synchronize()
            free.append(torch.cuda.mem_get_info()[0])
            op.compute_static(dl, cut, out)
            torch.cuda.synchronize()
            free.append(torch.cuda.mem_get_info()[0])
            k = out.cpu().numpy()
            st = op.stats()
            assert op._ws is None
            assert st["n_evals"] == evals == st_ref["n_evals"] and st["n_skipped"] == st_ref["n_skipped"]
            assert st["n_off_grid"] == st_ref["n_off_grid"] and st["single_pass"] == 0
            # against the existing path: same kernels, same arithmetic (fp32 partial sums and fp64 atomics in another order)
            rel, ab, _ = check_parity(k, k_ref_gpu, what=f"hk_compute_static call {call} vs hk_compute")
            assert np.abs(k - k_ref_gpu).max() <= 2e-6 * k_ref_gpu.max()
            # ... and against the oracle
            rel_o, ab_o, _ = check_parity(k, k_oracle, what=f"hk_compute_static call {call} vs oracle")
            print(f"n={n} N={op.N} call {call}: vs hk_compute rel={rel:.1e}, vs oracle rel={rel_o:.1e} abs={ab_o:.1e}")
        # the second call changed nothing in the device's free memory (the first may have loaded the module lazily)
        assert free[3] == free[2], free
        op.close()


def test_static_workspace_limits_and_errors():
    from paper_2101_02005_b200 import binding as B
    grid = W.CONFIGS[2]["grid"]                                    # 1e6 bins: ~200 MB of per-bin accumulators
    cond = W.conditions(2)
    op = B.Opacity(*grid)
    dl = _cuda(W.to_numpy(W.make_lines(2, n=1000, seed=0)))
    out = torch.zeros(op.N, dtype=torch.float64, device="cuda")
    with pytest.raises(B.HKError) as e:                            # conditions first
        op.compute_static(dl, 25.0, out)
    assert e.value.status == B.HK_ESTATE
    op.set_conditions(cond["T"], cond["P_atm"], cond["mass_amu"], cond["Q"])
    assert op.workspace_bytes(1000) > B.HK_STATIC_WS_BYTES
    with pytest.raises(B.HKError) as e:                            # beyond the static array: refused, nothing enqueued
        op.compute_static(dl, 25.0, out)
    assert e.value.status == B.HK_ENOSPC
    assert float(out.abs().max()) == 0.0
    op.close()
    # a workspace bound with hk_set_workspace stays bound (and its single-pass hint intact) across a static call
    c1 = W.CONFIGS[1]
    lines = W.to_numpy(W.make_lines(1, seed=0))
    d1 = _cuda(lines)
    op = B.Opacity(*c1["grid"])
    cd = W.conditions(1)
    op.set_conditions(cd["T"], cd["P_atm"], cd["mass_amu"], cd["Q"])
    k0 = op.compute(d1, c1["cut"]).clone()
    ws = op._ws
    out = torch.empty(op.N, dtype=torch.float64, device="cuda")
    op.compute_static(d1, c1["cut"], out)
    k1 = op.compute(d1, c1["cut"])
    torch.cuda.synchronize()
    assert op._ws is ws
    assert float((k1 - k0).abs().max()) <= 2e-6 * float(k0.max()) and float((out - k0).abs().max()) <= 2e-6 * float(k0.max())
    op.set_cut_mode("lorentz")
    with pytest.raises(B.HKError) as e:                            # width-relative cuts synchronise: not on this path
        op.compute_static(d1, 40.0, out)
    assert e.value.status == B.HK_ESTATE
    op.close()
