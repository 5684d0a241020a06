"""spiir_rank_static — the ranking chain (Eq. 13-15) without a caller-supplied workspace.

Some users of the library cannot allocate device memory at the point where candidates are ranked: an online search
process has by then given the whole GPU to the filter banks' workspaces and SNR rings, a late cudaMalloc would at best
stall the streams that are filtering, and a component hosted inside another process may simply be forbidden to
allocate after start-up.  For them `spiir_rank_static` keeps the histogram / R / FAP tables in an array that is part
of the library image (one per GPU, at most SPIIR_RANK_STATIC_MAX_BINS bins, shared by every call).

The test checks the new call against the existing workspace path (Ranker: reset, accumulate, finalize, candidates)
on two calls in a row with DIFFERENT inputs — the second one smaller and on coarser bins, so that anything the first
call left behind in the shared array would show.  Both paths run the same kernels on integer counts, so the
results must agree bit for bit (the tolerance of test_rank_statistic_fap_far's tables).

The file sorts last on purpose (pytest -x stops at the first failure; this call is an add-on, not part of the
hot path), and it must pass alone in a fresh process as well as after the other tests: it takes nothing from them.
"""
import ctypes as C

import numpy as np
import pytest


@pytest.fixture(scope="module")
def sp():
    import paper_2011_06787_b200 as sp
    sp.lib()                                    # fails loudly if the CUDA library is missing
    return sp


def _events(sp, rng, n_slots, n_slides):
    """Seeded triggers, background events [n_slots][n_slides] and foreground candidates [n_slots], shaped like a
    chunk's (rho_C^2 = trigger power + scaled chi^2_4, xi^2 a reduced chi^2, a tenth unused, some empty slots)."""
    snr = rng.uniform(4.0, 7.0, n_slots).astype(np.float32)
    trig = np.zeros(n_slots, sp.TRIGGER_DTYPE)
    trig["valid"] = 1; trig["snr"] = snr; trig["tmpl"] = np.arange(n_slots)
    trig["valid"][::7] = 0

    def draw(per_slot):
        n = n_slots * per_slot
        res = np.zeros(n, sp.RESULT_DTYPE)
        xi = np.zeros(n, sp.XI2_DTYPE)
        used = (rng.random(n) < 0.9).astype(np.int32)
        res["coh2"] = (np.repeat(snr, per_slot) ** 2 + rng.chisquare(4, n) * rng.uniform(0.5, 6.0, n)).astype(np.float32)
        res["tot2"] = res["coh2"]
        res["pix"] = np.where(used == 1, 5, -1)
        xi["xi2_c"] = (rng.chisquare(30, n) / 30 * rng.choice([1.0, 1.0, 3.0], n)).astype(np.float32)
        xi["used"] = used
        return res, xi

    bg, bg_xi = draw(n_slides)
    fg, fg_xi = draw(1)
    fg["coh2"][: n_slots // 16] *= 6.0           # a few loud candidates: R and FAP reach 0
    return trig, bg, bg_xi, fg, fg_xi


@pytest.mark.gpu
def test_rank_static_matches_the_workspace_path_on_two_calls_in_a_row(sp):
    import torch
    to_dev = lambda a: torch.from_numpy(a.view(np.uint8).reshape(len(a), -1).copy()).cuda()
    rng = np.random.default_rng(20261106)
    # first call: the largest binning the built-in array takes; second: fewer events, coarser bins, other ranges
    cases = [((64, 64, 4.0, 7.5, -1.0, 2.0), 900, 11, 11.0 * 5.0),
             ((12, 9, 4.5, 7.0, -0.5, 1.5), 130, 3, 3.0 * 2.0)]
    assert cases[0][0][0] * cases[0][0][1] == sp.SPIIR_RANK_STATIC_MAX_BINS
    n_selected = []
    for bins, n_slots, S, t_b in cases:
        trig, bg, bg_xi, fg, fg_xi = _events(sp, rng, n_slots, S)
        d = [to_dev(a) for a in (trig, bg, bg_xi, fg, fg_xi)]
        # the existing path, on a workspace of its own
        rk = sp.Ranker(*bins)
        rk.accumulate(d[0], d[1], d[2], n_slots, S)
        rk.finalize()
        want = sp.rank_to_numpy(rk.candidates(d[0], d[3], d[4], n_slots, t_b))
        # the new entry point: inputs and outputs only
        out = torch.full((n_slots, 16), 0xA5, dtype=torch.uint8, device="cuda")      # every byte must be written
        got = sp.rank_to_numpy(sp.rank_static(bins, d[0], d[1], d[2], n_slots, S, d[0], d[3], d[4], n_slots, t_b, out=out))
        torch.cuda.synchronize()
        assert got.tobytes() == want.tobytes()
        for f in ("rank", "fap", "far", "selected"):
            assert np.array_equal(got[f], want[f]), f
        n_selected.append(int(want["selected"].sum()))
        assert (want["fap"][want["selected"] == 1] > 0).any()                          # the comparison is not 0 == 0
    assert n_selected[0] > 100 and n_selected[1] > 10
    # an empty background: every selected candidate gets zeros, as from a freshly reset workspace
    bins, n_slots, S, t_b = cases[1]
    rk = sp.Ranker(*bins)
    rk.finalize()
    want = sp.rank_to_numpy(rk.candidates(d[0], d[3], d[4], n_slots, t_b))
    got = sp.rank_to_numpy(sp.rank_static(bins, None, None, None, 0, S, d[0], d[3], d[4], n_slots, t_b))
    torch.cuda.synchronize()
    assert got.tobytes() == want.tobytes() and not got["rank"].any() and got["selected"].sum() == n_selected[1]


def test_rank_static_refuses_binnings_beyond_the_built_in_array(sp):
    """Sizes are checked before any CUDA call, so this runs without a GPU."""
    call = lambda b, *a: sp.spiir_rank_static(C.cast(C.byref(b), C.c_void_p), *a)
    rest = (None, None, None, 0, 1, None, None, None, 0, 1.0, None, None)
    too_many = sp.spiir_rank_bins(64, 65, 4.0, 7.5, -1.0, 2.0)
    assert call(too_many, *rest) == sp.SPIIR_EINVAL
    msg = sp.last_error()
    assert "SPIIR_RANK_STATIC_MAX_BINS" in msg and "4160" in msg
    n = C.c_size_t(0)                            # the workspace path still takes this binning
    assert sp.spiir_rank_workspace_bytes(C.cast(C.byref(too_many), C.c_void_p), C.byref(n)) == sp.SPIIR_OK
    ok_bins = sp.spiir_rank_bins(64, 64, 4.0, 7.5, -1.0, 2.0)
    assert call(ok_bins, None, None, None, 0, 0, None, None, None, 0, 1.0, None, None) == sp.SPIIR_EINVAL   # n_slides < 1
    assert call(ok_bins, None, None, None, 5, 1, None, None, None, 0, 1.0, None, None) == sp.SPIIR_EINVAL   # NULL background
    assert call(ok_bins, None, None, None, 0, 1, None, None, None, 5, 1.0, None, None) == sp.SPIIR_EINVAL   # NULL foreground
    assert call(ok_bins, None, None, None, 0, 1, None, None, None, 0, 0.0, None, None) == sp.SPIIR_EINVAL   # T_b = 0
