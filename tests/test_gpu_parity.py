"""-m gpu parity tests: the CUDA path, called through the C ABI, against the float64
oracle on the same seeded inputs (tolerances in tests/parity_util.py)."""
import math

import numpy as np
import pytest

import oracle
import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def sp():
    import paper_2011_06787_b200 as sp
    sp.lib()                                    # fails loudly if the CUDA library is missing
    return sp


@pytest.fixture(scope="module")
def U():
    import parity_util
    return parity_util


def _table(cfg, nside=None, gmst=None):
    pos, resp = workloads.detector_geometry(cfg["dets"])
    g = workloads.strain_for_config(cfg["index"], seconds=1)["gmst"] if gmst is None else gmst
    U2, delay = oracle.sky_table(nside or cfg["nside"], pos, resp, cfg["sigma"], g, 2048.0)
    return U2.astype(np.float32), delay


# ------------------------------------------------------------------ config 0, whole path
def test_cfg0_whole_path(sp, U):
    import torch
    cfg = workloads.config(0)
    bank = workloads.bank_for_config(0)
    st = workloads.strain_for_config(0)
    x = st["strain"]
    z_ref = oracle.filter_bank(x, bank)
    z, trigs, bk = U.run_bank(bank, x, 2048, peak_thr=0.0)
    U.check_snr(z, z_ref)
    trig, cnt = trigs[0]
    assert cnt == 8
    U.check_peaks_mode0(trig, z, z_ref, 0, 0.0)
    # sky search on the bank's own ring, stage-isolated against the oracle on the same float32 z
    u2, delay = _table(cfg, gmst=st["gmst"])
    plan = sp.SkyPlan(u2, delay, max_slots=8)
    tr_dev, _ = bk.peaks(0.0, 0)
    smap = torch.empty(8, plan.n_pix, dtype=torch.float32, device="cuda")
    res = sp.results_to_numpy(plan.search(bk.snr_view(), tr_dev, 8, skymap=smap))
    torch.cuda.synchronize()
    ref = U.oracle_sky_on(z, 2048, 2047, u2, delay, trig, want_map=True)
    U.check_sky(res, z, 2048, 2047, u2, delay, trig, ref=ref)
    # peaks within 21 samples of the chunk edge must come back as "no result"
    edge = (trig["k"] < 21) | (trig["k"] > 2047 - 21)
    assert np.all((res["pix"] == -1) == (ref[1][:, 0] == -1))
    assert np.all(res["pix"][~edge] >= 0)
    # two detectors: coh2 == tot2, null2 == 0 at every pixel (P11) -> the map is flat per delay ring
    ok = res["pix"] >= 0
    np.testing.assert_allclose(res["coh2"][ok], res["tot2"][ok], rtol=1e-5)
    m = smap.cpu().numpy()
    assert np.abs(m - ref[2]).max() <= 1e-4 * max(1.0, np.abs(ref[2]).max())


# ------------------------------------------------------------------ single-rate bank, chunk invariance
def test_single_rate_bank_ragged_and_split_invariant(sp, U):
    """A bank whose templates have ragged filter counts (incl. an empty template and one larger than
    a unit), several chunk splits: all must match the one-shot oracle (P7)."""
    rng = np.random.default_rng(11)
    counts = [32, 1, 0, 300, 77, 129, 8, 64, 700]
    banks = [workloads.random_bank(rng, 1, max(c, 1), [2048]) for c in counts]
    off = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
    bank = dict(n_templates=len(counts), band_rates=[2048], out_band=0, tmpl_offset=off,
                a=np.concatenate([b["a"][:c] for b, c in zip(banks, counts)]),
                b=np.concatenate([b["b"][:c] for b, c in zip(banks, counts)]),
                delay=np.concatenate([b["delay"][:c] for b, c in zip(banks, counts)]),
                band=np.zeros(sum(counts), np.uint8), max_delay=[2047])
    x = workloads.gaussian_strain(rng, 2, 3 * 2048)
    z_ref = oracle.filter_bank(x, bank)
    assert np.all(z_ref[:, 2] == 0)
    z1, _, _ = U.run_bank(bank, x, 2048)
    U.check_snr(z1, z_ref)
    z2, _, _ = U.run_bank(bank, x, None, chunks=[4, 2044, 1024, 8, 3064])
    U.check_snr(z2, z_ref)
    z3, _, _ = U.run_bank(bank, x, 6144)
    U.check_snr(z3, z_ref)
    assert np.abs(z1 - z2).max() <= 1e-4 and np.abs(z1 - z3).max() <= 1e-4


def test_long_delay_template_and_reset(sp, U):
    """Chirp-matched template (delays up to ~24 000 samples, served beyond the shared window) next
    to random templates; reset restores the initial state."""
    import torch
    bank = workloads.bank_for_config(1, n_templates=24)
    assert bank["max_delay"][0] > 20000
    x = workloads.strain_for_config(1)["strain"][:, :15 * 2048]
    z_ref = oracle.filter_bank(x, bank)
    z, trigs, bk = U.run_bank(bank, x, 2048, peak_thr=4.0)
    U.check_snr(z, z_ref)
    assert np.abs(z_ref[:, 0]).max() > 6.0                 # the injection is seen by template 0
    n_near = 0
    for c, (trig, cnt) in enumerate(trigs):
        sl = slice(c * 2048, (c + 1) * 2048)
        n_near += U.check_peaks_mode0(trig, z[:, :, sl], z_ref[:, :, sl], c * 2048, 4.0)
        assert cnt == int(trig["valid"].sum())
    bk.reset()
    xs = torch.from_numpy(x[:, :2048].copy()).cuda()
    out = torch.empty(3, 24, 2048, 2, dtype=torch.float32, device="cuda")
    bk.filter_chunk(xs, out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy().view(np.complex64)[..., 0], z[:, :, :2048])


# ------------------------------------------------------------------ multirate
def test_multirate_streaming_matches_one_shot_oracle(sp, U):
    rng = np.random.default_rng(5)
    bank = workloads.random_bank(rng, 6, 83, workloads.configs.RATES8, out_band=1)
    dec, itp = workloads.halfband_taps()
    x = workloads.gaussian_strain(rng, 2, 5 * 4096)
    z_ref = oracle.filter_bank(x, bank, dec, itp)
    z, trigs, _ = U.run_bank(bank, x, 4096, taps=(dec, itp), peak_thr=4.0)
    U.check_snr(z, z_ref)
    for c, (trig, cnt) in enumerate(trigs):
        sl = slice(c * 2048, (c + 1) * 2048)
        U.check_peaks_mode0(trig, z[:, :, sl], z_ref[:, :, sl], c * 2048, 4.0)
    z2, _, _ = U.run_bank(bank, x, None, taps=(dec, itp), chunks=[512, 4096, 1024, 3584, 4096, 4096, 3072])
    U.check_snr(z2, z_ref)
    # three bands with the output at the top rate (out_band = 0)
    bank3 = workloads.random_bank(rng, 3, 40, [2048, 1024, 512], out_band=0)
    x3 = workloads.gaussian_strain(rng, 1, 2 * 2048)
    z3_ref = oracle.filter_bank(x3, bank3, dec, itp)
    z3, _, _ = U.run_bank(bank3, x3, 2048, taps=(dec, itp))
    U.check_snr(z3, z3_ref)


def test_cfg2_shape_sample(sp, U):
    """Config 2's layout (8 bands, 600 filters per template) on a template subset, 3 chunks."""
    bank = workloads.bank_for_config(2, n_templates=16)
    dec, itp = workloads.halfband_taps()
    x = workloads.strain_for_config(2, seconds=3)["strain"]
    z_ref = oracle.filter_bank(x, bank, dec, itp)
    z, _, bk = U.run_bank(bank, x, 4096, taps=(dec, itp))
    U.check_snr(z, z_ref)
    assert bk.updates_per_chunk(4096) == 2 * 16 * 75 * 8160


# ------------------------------------------------------------------ early-warning bank (NEXT-4, second half)
def test_early_warning_bank(sp, U):
    """PAPER.md:393 (Sec. IV, early-warning configuration): templates truncated at a seeded cut-off of 30-60 Hz, so
    that all of their filters sit in the bands of <= 256 Hz and bands 0-3 of the 8-band layout hold NO filter at all —
    a shape the (lanes, filters-per-lane) chooser and the launch grouping never see in the other configs.  Streaming
    in 1-s chunks against the one-shot oracle, peaks per chunk, ragged templates, chunk-split invariance."""
    rng = np.random.default_rng(393)
    full = workloads.random_bank(rng, 40, 700, workloads.configs.RATES8, out_band=1, exact_norm=False)
    bank = workloads.early_warning_bank(full, rng, exact_norm=False)
    per_band = np.bincount(bank["band"], minlength=8)
    assert per_band[:4].sum() == 0 and per_band[4:].min() > 0
    assert len(set(np.diff(bank["tmpl_offset"]).tolist())) > 10                 # ragged
    dec, itp = workloads.halfband_taps()
    x = workloads.gaussian_strain(rng, 2, 6 * 4096)
    z_ref = oracle.filter_bank(x, bank, dec, itp)
    z, trigs, bk = U.run_bank(bank, x, 4096, taps=(dec, itp), peak_thr=0.0)
    U.check_snr(z, z_ref)
    assert np.abs(z_ref[:, :, 2 * 2048:]).max() > 0.5                           # not a comparison of zeros
    for c, (trig, cnt) in enumerate(trigs):
        sl = slice(c * 2048, (c + 1) * 2048)
        U.check_peaks_mode0(trig, z[:, :, sl], z_ref[:, :, sl], c * 2048, 0.0)
    for b in range(4):
        assert bk.band_plan(b)["n_filters"] == 0
    assert bk.updates_per_chunk(4096) == 2 * sum(int(per_band[b]) * (4096 >> b) for b in range(8))
    z2, _, _ = U.run_bank(bank, x, None, taps=(dec, itp), chunks=[512, 4096, 1024, 3584, 4096, 4096, 3072, 4096])
    U.check_snr(z2, z_ref)


# ------------------------------------------------------------------ peaks mode 1
def test_peaks_mode1_paper_rule(sp, U):
    rng = np.random.default_rng(8)
    bank = workloads.random_bank(rng, 37, 16, [2048])
    x = workloads.gaussian_strain(rng, 2, 2048)
    for bank_size, thr in ((10, 2.5), (37, 0.0), (1, 3.0)):
        z, trigs, _ = U.run_bank(bank, x, 2048, bank_size=bank_size, peak_thr=thr, peak_mode=1)
        trig, cnt = trigs[0]
        for d in range(2):
            k, v = oracle.peaks_mode1(z[d], thr, bank_size)
            t = trig[d * 37:(d + 1) * 37]
            assert np.array_equal(t["valid"], v)
            assert np.array_equal(t["k"][v == 1], k[v == 1])
            zz = z[d][np.arange(37), k]
            assert np.array_equal(t["z_re"][v == 1], zz.real[v == 1])
        assert cnt == int(trig["valid"].sum())


# ------------------------------------------------------------------ sky search on snippets (config 3 form)
def _snippet_case(sp, n_rows, nside, n_windows, half, seed, gmst=0.7):
    import torch
    cfg = workloads.config(3)
    pos, resp = workloads.detector_geometry(cfg["dets"])
    U2, delay = oracle.sky_table(nside, pos, resp, cfg["sigma"], gmst, 2048.0)
    u2 = U2.astype(np.float32)
    rng = np.random.default_rng(seed)
    z, tdet, k, truth = workloads.snr_snippets(rng, u2, delay, n_rows, n_windows, half, 0.25)
    zc = np.ascontiguousarray(z).view(np.complex64)[..., 0]
    trig = np.zeros(n_rows, sp.TRIGGER_DTYPE)
    trig["valid"] = 1
    trig["tmpl"] = np.arange(n_rows)
    trig["det"] = tdet
    trig["k"] = k
    zd = torch.from_numpy(np.ascontiguousarray(z)).cuda()
    return u2, delay, zc, zd, trig, truth


def test_sky_foreground_and_signal_recovery(sp, U):
    _sky_foreground_and_signal_recovery(sp, U)


def _sky_foreground_and_signal_recovery(sp, U):
    import torch
    u2, delay, zc, zd, trig, truth = _snippet_case(sp, 200, 16, 1, 102, seed=21)
    trig["valid"][::7] = 0                                   # some empty slots
    L = zc.shape[2]
    plan = sp.SkyPlan(u2, delay, max_slots=200)
    assert plan.n_tuples < plan.n_pix
    view = sp.SnrView(zd)
    smap = torch.empty(200, plan.n_pix, dtype=torch.float32, device="cuda")
    res = sp.results_to_numpy(plan.search(view, sp.triggers_from_numpy(trig), 200, skymap=smap))
    torch.cuda.synchronize()
    ref = U.oracle_sky_on(zc, L, L - 1, u2, delay, trig, want_map=True)
    U.check_sky(res, zc, L, L - 1, u2, delay, trig, ref=ref)
    assert np.all(res["pix"][::7] == -1)
    m = smap.cpu().numpy()
    tot = np.maximum(ref[0][:, 0, 2], 1.0)[:, None]
    assert np.all(np.abs(m - ref[2]) <= 1e-4 * ref[2] + 2e-6 * tot)
    # injected coherent signals: strong ones come back within the oracle's own arg-max set
    sig = truth["is_signal"] & (trig["valid"] == 1)
    assert sig.sum() > 10
    assert np.mean(res["coh2"][sig]) > 4 * np.mean(res["coh2"][~truth["is_signal"] & (trig["valid"] == 1)])


def test_sky_time_slides(sp, U):
    import torch
    n_rows, S, half = 96, 7, 102
    W = 2 * half + 1
    u2, delay, zc, zd, trig, truth = _snippet_case(sp, n_rows, 16, S + 1, half, seed=22)
    L = zc.shape[2]
    plan = sp.SkyPlan(u2, delay, max_slots=n_rows)
    view = sp.SnrView(zd)
    td = sp.triggers_from_numpy(trig)
    for mult in ([1, 1, 1], [0, 0, 0]):
        res = sp.results_to_numpy(plan.background(view, td, n_rows, S, W, mult))
        torch.cuda.synchronize()
        U.check_sky(res, zc, L, L - 1, u2, delay, trig, n_slides=S, step=W, mult=mult)
    # P16: with every multiplier 0 each slide reproduces the foreground
    fg = sp.results_to_numpy(plan.search(view, td, n_rows))
    bg0 = sp.results_to_numpy(plan.background(view, td, n_rows, S, W, [0, 0, 0])).reshape(n_rows, S)
    for s in range(S):
        assert np.array_equal(bg0[:, s], fg)
    # one slide too many leaves the view: "no result" for that slide only
    res = sp.results_to_numpy(plan.background(view, td, n_rows, S + 1, W, [1, 1, 1])).reshape(n_rows, S + 1)
    assert np.all(res["pix"][:, S] == -1) and np.all(res["pix"][:, :S] >= 0)
    # a coarser background table (768 pixels) is just another plan
    cfg = workloads.config(3)
    pos, resp = workloads.detector_geometry(cfg["dets"])
    U2b, delayb = oracle.sky_table(8, pos, resp, cfg["sigma"], 0.7, 2048.0)
    planb = sp.SkyPlan(U2b.astype(np.float32), delayb, max_slots=n_rows)
    resb = sp.results_to_numpy(planb.background(view, td, n_rows, S, W, [1, 1, 1]))
    torch.cuda.synchronize()
    U.check_sky(resb, zc, L, L - 1, U2b.astype(np.float32), delayb, trig, n_slides=S, step=W, mult=[1, 1, 1])


def test_sky_ring_wraparound_and_two_detectors(sp, U):
    """A view used as a true ring (k_newest beyond ring_len, windows wrapping the end) and a
    two-detector network (projector = identity, P11)."""
    import torch
    cfg = workloads.config(0)
    pos, resp = workloads.detector_geometry(cfg["dets"])
    U2, delay = oracle.sky_table(8, pos, resp, cfg["sigma"], 2.1, 2048.0)
    u2 = U2.astype(np.float32)
    rng = np.random.default_rng(3)
    L, rows = 500, 40
    z = rng.standard_normal((2, rows, L, 2)).astype(np.float32)
    zc = z.view(np.complex64)[..., 0]
    k_newest = 3 * L + 123
    trig = np.zeros(rows, sp.TRIGGER_DTYPE)
    trig["valid"] = 1
    trig["tmpl"] = np.arange(rows)
    trig["det"] = rng.integers(0, 2, rows)
    trig["k"] = rng.integers(k_newest - L - 10, k_newest + 5, rows)      # some too old, some too new
    plan = sp.SkyPlan(u2, delay, max_slots=rows)
    view = sp.SnrView(torch.from_numpy(z).cuda(), k_newest=k_newest)
    res = sp.results_to_numpy(plan.search(view, sp.triggers_from_numpy(trig), rows))
    torch.cuda.synchronize()
    U.check_sky(res, zc, L, k_newest, u2, delay, trig)
    ok = res["pix"] >= 0
    assert ok.sum() > 10 and (~ok).sum() > 0
    np.testing.assert_allclose(res["coh2"][ok], res["tot2"][ok], rtol=1e-5)
    assert np.all(res["null2"][ok] <= 1e-4 * res["tot2"][ok] + 1e-5)


# ------------------------------------------------------------------ config 1 sample: bank -> peaks -> sky, one-chunk lag
def test_cfg1_sample_chain(sp, U):
    import torch
    cfg = workloads.config(1)
    T = 48
    bank = workloads.bank_for_config(1, n_templates=T)
    st = workloads.strain_for_config(1)
    x = st["strain"]
    NC = x.shape[1] // 2048
    z_ref = oracle.filter_bank(x, bank)
    u2, delay = _table(cfg, gmst=st["gmst"])
    ring = 3 * 2048
    bk = sp.Bank(bank, 3, 2048, ring_len=ring)
    plan = sp.SkyPlan(u2, delay, max_slots=3 * T)
    xs = torch.from_numpy(x).cuda()
    z = np.zeros((3, T, NC * 2048), np.complex64)
    prev = None
    best = (0.0, None)
    for c in range(NC):
        out = torch.empty(3, T, 2048, 2, dtype=torch.float32, device="cuda")
        bk.filter_chunk(xs[:, c * 2048:(c + 1) * 2048].contiguous(), out)
        z[:, :, c * 2048:(c + 1) * 2048] = out.cpu().numpy().view(np.complex64)[..., 0]
        if prev is not None:                                  # search chunk c-1 now that chunk c exists (A13)
            res = sp.results_to_numpy(plan.search(bk.snr_view(), prev[0], 3 * T))
            torch.cuda.synchronize()
            k_newest = (c + 1) * 2048 - 1
            lo = k_newest - ring + 1
            zr = np.zeros((3, T, ring), np.complex64)
            kk = np.arange(max(lo, 0), k_newest + 1)
            zr[:, :, kk % ring] = z[:, :, kk]
            U.check_sky(res, zr, ring, k_newest, u2, delay, prev[1])
            ok = res["pix"] >= 0
            if ok.any() and res["coh2"][ok].max() > best[0]:
                i = np.nonzero(ok)[0][np.argmax(res["coh2"][ok])]
                best = (float(res["coh2"][i]), (int(prev[1]["tmpl"][i]), int(res["pix"][i])))
        tr, cnt = bk.peaks(4.0, 0)
        torch.cuda.synchronize()
        prev = (tr.clone(), sp.triggers_to_numpy(tr).copy())
    U.check_snr(z, z_ref)
    # the injection (network SNR 15) is the loudest coherent candidate, found by template 0
    assert best[1][0] == 0 and math.sqrt(best[0]) > 10.0


# ------------------------------------------------------------------ config 4 at FULL size, sampled outputs
def test_cfg4_full_size_sampled(sp, U):
    """BASELINE.json config 4 in the launch configuration bench.py times (20 000 templates x 700
    filters, 8 bands, 3 detectors: k_bank grid 5005 x 3, k_combine 20000 x 3, k_sky on 60 000 slots at
    nside 32), three 1-s chunks.  The oracle cannot run 14 M filters, so outputs are SAMPLED: the SNR
    series of 16 templates (3 chirp-matched long-delay ones, the first / last random ones, 11 seeded)
    against the float64 oracle of exactly those templates (templates are independent), every peak of
    the last chunk stage-isolated against O4 on the GPU's own z, and the sky search / one time slide of
    the sampled templates' candidates against O6 / O7 (one-chunk lag, A13)."""
    import torch
    cfg = workloads.config(4)
    T, D, NC = cfg["n_templates"], 3, 3
    THR = 1.5          # the stream is 3 s old: the low-rate bands are still filling, threshold 4 would give ~no candidates
    bank = workloads.bank_for_config(4)
    st = workloads.strain_for_config(4, seconds=NC)
    x = st["strain"]
    dec, itp = workloads.halfband_taps()
    rng = np.random.default_rng(4)
    sel = np.unique(np.concatenate([[0, 7, 19, 20, T - 1], rng.integers(21, T - 1, 11)])).astype(np.int64)
    z_ref = oracle.filter_bank(x, bank, dec, itp, templates=sel)             # [D][n_sel][NC*2048]
    ring = 4 * 2048
    bk = sp.Bank(bank, D, 4096, ring_len=ring, bank_size=1000, dec_taps=dec, int_taps=itp)
    assert bk.band_plan(1)["n_units_long"] > 0                               # the long-delay class is exercised
    xs = torch.from_numpy(x).cuda()
    out = torch.empty(D, T, 2048, 2, dtype=torch.float32, device="cuda")
    z_sel = np.zeros((D, len(sel), NC * 2048), np.complex64)
    trig_prev = None
    sel_dev = torch.from_numpy(sel).cuda()
    for c in range(NC):
        bk.filter_chunk(xs[:, c * 4096:(c + 1) * 4096].contiguous(), out)
        z_sel[:, :, c * 2048:(c + 1) * 2048] = out[:, sel_dev].cpu().numpy().view(np.complex64)[..., 0]
        tr, cnt = bk.peaks(THR, 0)
        torch.cuda.synchronize()
        if c == NC - 2:
            trig_prev = (tr.clone(), sp.triggers_to_numpy(tr).copy())
    U.check_snr(z_sel, z_ref)
    # every peak of the last chunk, bit-exact against O4 on the GPU's own float32 z
    z_last = out.cpu().numpy().view(np.complex64)[..., 0]
    trig = sp.triggers_to_numpy(tr)
    k_iso, v_iso = oracle.peaks_mode0(z_last.reshape(D * T, 2048), THR)
    assert np.array_equal(trig["k"] - (NC - 1) * 2048, k_iso) and np.array_equal(trig["valid"], v_iso)
    assert int(cnt.cpu()[0]) == int(v_iso.sum()) and v_iso.sum() > 0.2 * D * T
    # the paper's two-step rule (mode 1) on the same chunk, banks of 1000 templates (A10), stage-isolated
    tr1, cnt1 = bk.peaks(THR, 1)
    torch.cuda.synchronize()
    t1 = sp.triggers_to_numpy(tr1)
    for d in range(D):
        k1, v1 = oracle.peaks_mode1(z_last[d], THR, 1000)
        td_ = t1[d * T:(d + 1) * T]
        assert np.array_equal(td_["valid"], v1) and np.array_equal(td_["k"][v1 == 1] - (NC - 1) * 2048, k1[v1 == 1])
    assert int(cnt1.cpu()[0]) == int(t1["valid"].sum()) > 100
    # end to end on the sampled templates (near-tie rule A12)
    rows = (np.arange(D)[:, None] * T + sel[None, :]).reshape(-1)
    U.check_peaks_mode0(_subset_trig(trig[rows], sel, D), z_sel[:, :, -2048:], z_ref[:, :, -2048:],
                        (NC - 1) * 2048, THR)
    # sky search + one slide over all 60 000 slots; compare the sampled templates' candidates
    u2, delay = _table(cfg, gmst=st["gmst"])
    plan = sp.SkyPlan(u2, delay, max_slots=D * T)
    view = bk.snr_view()
    fg = sp.results_to_numpy(plan.search(view, trig_prev[0], D * T))
    bg = sp.results_to_numpy(plan.background(view, trig_prev[0], D * T, 1, 2048, [1, 1, 1]))
    torch.cuda.synchronize()
    tp = trig_prev[1]
    assert np.all((fg["pix"] >= 0) == (tp["valid"] == 1))                    # every candidate searched, nothing else
    assert np.all(bg["pix"][tp["valid"] == 0] == -1)                         # (a slide may leave the stream's start)
    k_newest = NC * 2048 - 1
    zr = np.zeros((D, len(sel), ring), np.complex64)
    zr[:, :, :NC * 2048] = z_sel                                             # ring index = k (k < ring_len)
    sub = _subset_trig(tp[rows], sel, D)
    assert sub["valid"].sum() >= 8
    U.check_sky(fg[rows], zr, ring, k_newest, u2, delay, sub)
    U.check_sky(bg[rows], zr, ring, k_newest, u2, delay, sub, n_slides=1, step=2048, mult=[1, 1, 1])
    # the same candidates end to end, nothing from the CUDA path on the oracle's side: float64 SNR of the sampled
    # templates -> O4 -> O6 / O7
    zr64 = np.zeros((D, len(sel), ring), np.complex128)
    zr64[:, :, :NC * 2048] = z_ref
    k_o, v_o = oracle.peaks_mode0(z_ref[:, :, (NC - 2) * 2048:(NC - 1) * 2048].reshape(D * len(sel), 2048), THR)
    same = (v_o == 1) & (sub["valid"] == 1) & (k_o + (NC - 2) * 2048 == sub["k"])
    assert same.sum() >= 0.9 * (sub["valid"] == 1).sum()
    for gres, kw in ((fg[rows], {}), (bg[rows], dict(n_slides=1, step=2048, slide_mult=[1, 1, 1]))):
        ref_e, pix_e, _ = oracle.sky_search(u2, delay, zr64, len(sel) * ring, ring, ring, k_newest, same.astype(np.int32),
                                            sub["tmpl"], sub["det"], sub["k"], **kw)
        idx = np.nonzero(same & (pix_e[:, 0] >= 0))[0]
        cg, ce = gres["coh2"][idx].astype(np.float64), ref_e[idx, 0, 0]
        assert len(idx) >= 8 and np.all(gres["pix"][idx] >= 0)
        assert np.all(np.abs(np.sqrt(cg) - np.sqrt(ce)) <= 1e-3) and np.all(np.abs(cg - ce) <= 1e-4 * ce + 1e-5)


def test_cfg4_steady_state(sp, U):
    """BASELINE.json config 4 in the regime bench.py times: all 128 one-second chunks streamed through the full
    bank (20 000 templates x 700 filters, 8 bands, 3 detectors), threshold 4, SNR ring of 103 s
    so that it WRAPS, 100 one-second time slides on the foreground grid (nside 32).
    Sampled outputs (the oracle cannot run 14 M filters): 16 seeded templates (3 chirp-matched long-delay ones)
      * their SNR over the whole 128 s against the float64 oracle of exactly those templates (O1-O3);
      * their peaks in EVERY chunk, stage-isolated and end to end (A12); all 60 000 peaks of eight chunks around
        the start, the ring wrap and the end, stage-isolated;
      * for the last two searched chunks (ring wrapped, low-rate bands full): their candidates through O6 on the
        foreground and O7 on all 100 slides, and xi^2 (O8) on foreground and slides."""
    import torch
    cfg = workloads.config(4)
    T, D, NC, S, THR, nj = cfg["n_templates"], 3, 128, 100, 4.0, 175
    bank = workloads.bank_for_config(4)
    st = workloads.strain_for_config(4)
    x = st["strain"]
    assert x.shape[1] == NC * 4096
    dec, itp = workloads.halfband_taps()
    rng = np.random.default_rng(44)
    sel = np.unique(np.concatenate([[0, 7, 19, 20, T - 1], rng.integers(21, T - 1, 11)])).astype(np.int64)
    ns = len(sel)
    z_ref = oracle.filter_bank(x, bank, dec, itp, templates=sel)             # [D][ns][NC*2048]
    L = (S + 3) * 2048
    bk = sp.Bank(bank, D, 4096, ring_len=L, bank_size=1000, dec_taps=dec, int_taps=itp)
    u2, delay = _table(cfg, gmst=st["gmst"])
    plan = sp.SkyPlan(u2, delay, max_slots=D * T)
    dl_dev = torch.from_numpy(np.ascontiguousarray(delay, dtype=np.int32)).cuda()
    # a seeded synthetic autocorrelation table (an INPUT of Eq. 11 like the sky table; multirate templates have no
    # host helper): A[j] = exp(-|j| / tau + i w j)
    g = np.random.default_rng(45)
    tau, om = 5.0 + 40.0 * g.random(T), 0.1 + 1.2 * g.random(T)
    lag = np.arange(-nj, nj + 1)
    acorr = (np.exp(-np.abs(lag)[None, :] / tau[:, None]) * np.exp(1j * om[:, None] * lag[None, :])).astype(np.complex64)
    ac_dev = torch.from_numpy(acorr.view(np.float32).reshape(T, 2 * nj + 1, 2)).cuda()
    xs = torch.from_numpy(x).cuda()
    out = torch.empty(D, T, 2048, 2, dtype=torch.float32, device="cuda")
    z_sel = np.zeros((D, ns, NC * 2048), np.complex64)
    sel_dev = torch.from_numpy(sel).cuda()
    rows = (np.arange(D)[:, None] * T + sel[None, :]).reshape(-1)
    full_check = {0, 1, 50, 102, 103, 104, NC - 2, NC - 1}
    prev, n_rule2, n_cand, searched = None, 0, [], 0
    mult = [1, 1, 1]
    for c in range(NC):
        bk.filter_chunk(xs[:, c * 4096:(c + 1) * 4096].contiguous(), out)
        z_sel[:, :, c * 2048:(c + 1) * 2048] = out[:, sel_dev].cpu().numpy().view(np.complex64)[..., 0]
        tr, cnt = bk.peaks(THR, 0)
        torch.cuda.synchronize()
        trig = sp.triggers_to_numpy(tr).copy()
        n_cand.append(int(cnt.cpu()[0]))
        # the sampled templates' peaks of this chunk: stage-isolated + end to end
        n_rule2 += U.check_peaks_mode0(_subset_trig(trig[rows], sel, D), z_sel[:, :, c * 2048:(c + 1) * 2048],
                                       z_ref[:, :, c * 2048:(c + 1) * 2048], c * 2048, THR)
        if c in full_check:                                                   # all 60 000 peaks, stage-isolated
            z_all = out.cpu().numpy().view(np.complex64)[..., 0]
            k_iso, v_iso = oracle.peaks_mode0(z_all.reshape(D * T, 2048), THR)
            assert np.array_equal(trig["k"] - c * 2048, k_iso) and np.array_equal(trig["valid"], v_iso)
            assert n_cand[-1] == int(v_iso.sum())
            del z_all
        if c >= NC - 2 and prev is not None:
            # search the previous chunk's candidates (one-chunk lag, A13): the ring has wrapped (k_newest >= L)
            view = bk.snr_view()
            k_new = (c + 1) * 2048 - 1
            assert int(view.c.k_newest) == k_new and k_new + 1 > L
            fg_d = plan.search(view, prev[0], D * T)
            bg_d = plan.background(view, prev[0], D * T, S, 2048, mult)
            xi_f = sp.xi2_to_numpy(sp.signal_consistency(view, dl_dev, prev[0], fg_d, D * T, ac_dev, nj))
            xi_b = sp.xi2_to_numpy(sp.signal_consistency(view, dl_dev, prev[0], bg_d, D * T, ac_dev, nj, n_slides=S,
                                                         step=2048, mult=mult)).reshape(D * T, S)
            torch.cuda.synchronize()
            fg, bg = sp.results_to_numpy(fg_d), sp.results_to_numpy(bg_d).reshape(D * T, S)
            tp = prev[1]
            # every candidate of the chunk was searched on the foreground and on every one of the 100 slides
            assert np.all((fg["pix"] >= 0) == (tp["valid"] == 1)) and np.all((bg["pix"] >= 0) == (tp["valid"] == 1)[:, None])
            # the ring of the sampled templates as the device holds it: element k mod L is sample k
            kk = np.arange(k_new + 1 - L, k_new + 1)
            zr = np.zeros((D, ns, L), np.complex64)
            zr[:, :, kk % L] = z_sel[:, :, kk]
            dev_rows = bk.ring_rows(sel_dev).cpu().numpy().view(np.complex64)[..., 0]
            assert np.array_equal(dev_rows, zr)                               # the wrapped ring holds exactly the last L samples
            sub = _subset_trig(tp[rows], sel, D)
            assert sub["valid"].sum() >= 6
            st_f = U.check_sky(fg[rows], zr, L, k_new, u2, delay, sub)
            st_b = U.check_sky(bg[rows].reshape(-1), zr, L, k_new, u2, delay, sub, n_slides=S, step=2048, mult=mult)
            searched += st_f["n"] + st_b["n"]
            assert st_b["n"] == S * st_f["n"]
            # xi^2 (Eq. 11, 12) at the GPU's pixels, foreground and every slide
            A_sel = acorr[sel].astype(np.complex128)
            for xg, pixg, kw in ((xi_f[rows], fg["pix"][rows], {}),
                                 (xi_b[rows], bg["pix"][rows], dict(n_slides=S, step=2048, slide_mult=mult))):
                ref = oracle.xi2(delay, zr, ns * L, L, L, k_new, sub["valid"], sub["tmpl"], sub["det"], sub["k"],
                                 pixg, A_sel, nj, **kw)
                used = ref[..., D + 1] == 1
                assert np.array_equal(xg["used"].reshape(used.shape), used.astype(np.int32)) and used.sum() >= 6
                gc = xg["xi2_c"].reshape(used.shape)
                assert np.all(np.abs(gc - ref[..., D])[used] <= 1e-4 * ref[..., D][used] + 1e-5)
        prev = (tr.clone(), trig)
    err = U.check_snr(z_sel, z_ref)
    # steady state: about two thirds of the (detector, template, second) slots are above SNR 4 (what bench.py searches:
    # ~40 500 candidates per chunk), against a handful in the first seconds while the low-rate bands fill
    assert 0.5 * D * T < np.median(n_cand[-20:]) < 0.85 * D * T and n_cand[0] < 0.2 * D * T
    assert searched >= 2 * 6 * (1 + S)
    print("cfg4 steady state: max |dz| %.2e over 128 s, %d near-tie peaks (A12), %d sky results checked" % (err, n_rule2, searched))


def _subset_trig(trig_rows, sel, D):
    """Trigger slots of the selected templates with `tmpl` renumbered to rows of the sampled view."""
    t = trig_rows.copy()
    t["tmpl"] = np.tile(np.arange(len(sel)), D)
    return t


# ------------------------------------------------------------------ views that are not 16-byte friendly
def test_sky_unaligned_view(sp, U):
    """A view whose rows are not 16-byte friendly (odd ring_len 501, base pointer 8 bytes past an aligned address):
    the window staging cannot use TMA bulk copies and takes the 8-byte cp.async path.  Foreground, slides and a
    wrapped ring against O6 / O7."""
    import torch
    cfg = workloads.config(1)
    u2, delay = _table(cfg, nside=8, gmst=1.1)
    D, rows, L, k_new, S, step = 3, 40, 501, 1300, 3, 90
    rng = np.random.default_rng(501)
    z = (rng.standard_normal((D, rows, L)) + 1j * rng.standard_normal((D, rows, L))).astype(np.complex64)
    flat = torch.zeros(D * rows * L * 2 + 2, dtype=torch.float32, device="cuda")
    flat[2:] = torch.from_numpy(np.ascontiguousarray(z).view(np.float32).reshape(-1)).cuda()
    assert flat.data_ptr() % 16 == 0
    raw = sp.spiir_snr_view(flat.data_ptr() + 8, rows * L, L, L, k_new, rows)
    view = sp.SnrView(raw=raw)
    view._keep = flat
    n = 64
    trig = np.zeros(n, sp.TRIGGER_DTYPE)
    trig["valid"] = 1; trig["valid"][5] = 0
    trig["tmpl"] = rng.integers(0, rows, n); trig["det"] = rng.integers(0, D, n)
    trig["k"] = rng.integers(k_new - L + 1, k_new + 1, n)            # some windows leave the view on either side
    td = sp.triggers_from_numpy(trig)
    plan = sp.SkyPlan(u2, delay, max_slots=n)
    fg = sp.results_to_numpy(plan.search(view, td, n))
    bg = sp.results_to_numpy(plan.background(view, td, n, S, step, [1, 1, 1]))
    torch.cuda.synchronize()
    st_f = U.check_sky(fg, z, L, k_new, u2, delay, trig)
    st_b = U.check_sky(bg, z, L, k_new, u2, delay, trig, n_slides=S, step=step, mult=[1, 1, 1])
    assert st_f["n"] >= 30 and st_b["n"] >= 60 and (fg["pix"] == -1).sum() >= 2


# ------------------------------------------------------------------ grids of more than 32 767 stream chunks
def test_sky_grid_beyond_32767_chunks(sp, U):
    """A table of 1 105 920 directions (34 560 chunks of 32: the warps' chunk shares no longer fit 16 bits, which an
    earlier layout stored them in).  The table is the nside-32 one repeated 90 times, so by the tie rule of spiir.h
    (tuples in increasing order, pixel index ascending within a tuple) every result — maximum, tot2, null2 AND pixel —
    must be bit-identical to the 12 288-direction plan's, which the other tests hold against the oracle."""
    import torch
    cfg = workloads.config(1)
    u2, delay = _table(cfg, nside=32, gmst=2.2)
    reps = 90
    u2_big, delay_big = np.tile(u2, (reps, 1, 1)), np.tile(delay, (reps, 1))
    assert (len(u2_big) + 31) // 32 > 32767
    D, rows, L, k_new, S, step = 3, 24, 400, 399, 2, 60
    rng = np.random.default_rng(32767)
    z = (rng.standard_normal((D, rows, L)) + 1j * rng.standard_normal((D, rows, L))).astype(np.complex64)
    view = sp.SnrView(torch.from_numpy(np.ascontiguousarray(z).view(np.float32).reshape(D, rows, L, 2)).cuda())
    view.c.k_newest = k_new
    n = 48
    trig = np.zeros(n, sp.TRIGGER_DTYPE)
    trig["valid"] = 1
    trig["tmpl"] = rng.integers(0, rows, n); trig["det"] = np.arange(n) % D
    trig["k"] = rng.integers(200, 360, n)
    td = sp.triggers_from_numpy(trig)
    small, big = sp.SkyPlan(u2, delay, max_slots=n), sp.SkyPlan(u2_big, delay_big, max_slots=n)
    assert big.n_tuples == small.n_tuples
    for run in (lambda pl: pl.search(view, td, n), lambda pl: pl.background(view, td, n, S, step, [1, 1, 1])):
        a, b = sp.results_to_numpy(run(small)), sp.results_to_numpy(run(big))
        torch.cuda.synchronize()
        assert (a["pix"] >= 0).sum() >= n // 2
        assert a.tobytes() == b.tobytes()
    st = U.check_sky(sp.results_to_numpy(small.search(view, td, n)), z, L, k_new, u2, delay, trig)   # and the anchor itself
    assert st["n"] >= n // 2


# ------------------------------------------------------------------ degenerate inputs
def test_sky_degenerate_inputs(sp, U):
    """No slots, no valid slot, and an all-zero SNR view (every direction ties exactly)."""
    import torch
    cfg = workloads.config(1)
    u2, delay = _table(cfg, nside=4, gmst=0.3)
    plan = sp.SkyPlan(u2, delay, max_slots=16)
    L = 400
    zd = torch.zeros(3, 16, L, 2, dtype=torch.float32, device="cuda")
    view = sp.SnrView(zd)
    trig = np.zeros(16, sp.TRIGGER_DTYPE)
    trig["tmpl"] = np.arange(16); trig["det"] = np.arange(16) % 3; trig["k"] = 200
    td = sp.triggers_from_numpy(trig)
    # n_slots = 0: nothing is launched, nothing is written
    sentinel = torch.full((16, 16), 7, dtype=torch.uint8, device="cuda")
    plan.search(view, td, 0, out=sentinel)
    torch.cuda.synchronize()
    assert int(sentinel.min()) == 7
    # no valid slot: every result is "none", for the foreground and for every slide
    res = sp.results_to_numpy(plan.search(view, td, 16))
    bg = sp.results_to_numpy(plan.background(view, td, 16, 3, 50, [1, 1, 1]))
    torch.cuda.synchronize()
    for r in (res, bg):
        assert np.all(r["pix"] == -1) and np.all(r["coh2"] == 0) and np.all(r["tot2"] == 0)
    # all-zero SNR: coh2 = tot2 = null2 = 0 and a valid pixel (A19: every pixel is an arg-max)
    trig["valid"] = 1
    res = sp.results_to_numpy(plan.search(view, sp.triggers_from_numpy(trig), 16))
    torch.cuda.synchronize()
    assert np.all((res["pix"] >= 0) & (res["pix"] < plan.n_pix))
    assert np.all(res["coh2"] == 0) and np.all(res["tot2"] == 0) and np.all(res["null2"] == 0)
    zc = np.zeros((3, 16, L), np.complex64)
    U.check_sky(res, zc, L, L - 1, u2, delay, trig)
    # a view whose n_rows was never set (0, or garbage beyond what an int32 tmpl can address) is refused, as are slide
    # shifts that would overflow (tests/test_abi.py holds the same for the calls that need no plan)
    for n_rows in (0, -1, 1 << 40):
        bad = sp.SnrView(raw=sp.spiir_snr_view(zd.data_ptr(), 16 * L, L, L, L - 1, n_rows))
        for call in (lambda: plan.search(bad, td, 16), lambda: plan.background(bad, td, 16, 3, 50, [1, 1, 1])):
            with pytest.raises(sp.SpiirError) as ei:
                call()
            assert ei.value.code == sp.SPIIR_EINVAL and "n_rows" in str(ei.value)
    with pytest.raises(sp.SpiirError):
        plan.background(view, td, 16, 100, 1 << 39, [1, 1, 1])


# ------------------------------------------------------------------ config 3 in FULL
def test_cfg3_full(sp, U):
    """BASELINE.json config 3 in full ("configs 0-3: the oracle runs in full"): 4096 triggers,
    HEALPix nside 64 (49 152 directions), 100 time slides on packed +-50 ms snippets
    (DESIGN.md §8).  The oracle evaluates every (trigger, slide, direction) — 2.03e10 evaluations of O6 / O7
    in float64 — and every one of the 4096 x 101 GPU results is compared with it (coh2 1e-4 relative, pixel by
    the set-valued rule A19, tot2 / null2 at the GPU's pixel)."""
    import torch
    cfg = workloads.config(3)
    n_rows, S, half = cfg["n_triggers"], cfg["n_slides"], cfg["snippet_half"]
    W = 2 * half + 1
    pos, resp = workloads.detector_geometry(cfg["dets"])
    U2, delay = oracle.sky_table(cfg["nside"], pos, resp, cfg["sigma"], 0.7, 2048.0)
    u2 = U2.astype(np.float32)
    rng = workloads.streams(cfg["seed"])["snippets"]
    z, tdet, k, truth = workloads.snr_snippets(rng, u2, delay, n_rows, S + 1, half, cfg["coherent_fraction"])
    trig = np.zeros(n_rows, sp.TRIGGER_DTYPE)
    trig["valid"] = 1; trig["tmpl"] = np.arange(n_rows); trig["det"] = tdet; trig["k"] = k
    zd = torch.from_numpy(z).cuda()
    L = z.shape[2]
    plan = sp.SkyPlan(u2, delay, max_slots=n_rows)
    view = sp.SnrView(zd)
    td = sp.triggers_from_numpy(trig)
    fg = sp.results_to_numpy(plan.search(view, td, n_rows))
    bg = sp.results_to_numpy(plan.background(view, td, n_rows, S, W, [1, 1, 1])).reshape(n_rows, S)
    torch.cuda.synchronize()
    del zd
    assert np.all(fg["pix"] >= 0) and np.all(bg["pix"] >= 0)
    # invariants that hold at any size: coh2 <= tot2, null2 = max(tot2 - coh2, 0)
    for r in (fg, bg.reshape(-1)):
        assert np.all(r["coh2"] <= r["tot2"] * (1 + 1e-5) + 1e-6)
        assert np.all(np.abs(r["null2"] - np.maximum(r["tot2"] - r["coh2"], 0)) <= 1e-6 * r["tot2"] + 1e-6)
    # every trigger against the oracle: foreground and all 100 slides
    zc = np.ascontiguousarray(z).view(np.complex64)[..., 0]
    st_f = U.check_sky(fg, zc, L, L - 1, u2, delay, trig)
    st_b = U.check_sky(bg.reshape(-1), zc, L, L - 1, u2, delay, trig, n_slides=S, step=W, mult=[1, 1, 1])
    assert st_f["n"] == n_rows and st_b["n"] == n_rows * S
    print("cfg3 full: foreground %s, slides %s" % (st_f, st_b))
    # injected signals in the plane of their pixel: the foreground is far above the time-slid background of the
    # same trigger (the slid background keeps |z_T|^2)
    sig = np.nonzero(truth["is_signal"])[0]
    strong = sig[truth["rho"][sig] > 12]
    assert len(strong) > 50
    assert np.median(fg["coh2"][strong] / np.median(bg["coh2"][strong], axis=1)) > 2


# ------------------------------------------------------------------ NEXT-1: signal-consistency statistic (Eq. 11, 12)
def test_xi2_signal_consistency(sp, U):
    """Bank -> peaks -> sky search -> xi^2 on the bank's own ring (one-chunk lag), against the oracle's O8
    on the same float32 SNR, the same pixels and the same float32 autocorrelation table.  Tolerance: 1e-4
    relative + 1e-5 (351 float32 terms of order 1 per sum)."""
    import torch
    cfg = workloads.config(1)
    T, D, NC, nj = 24, 3, 4, 175
    bank = workloads.bank_for_config(1, n_templates=T)
    bank_A = dict(bank)
    st = workloads.strain_for_config(1, seconds=NC)
    x = st["strain"]
    u2, delay = _table(cfg, gmst=st["gmst"])
    ring = NC * 2048
    bk = sp.Bank(bank, D, 2048, ring_len=ring)
    plan = sp.SkyPlan(u2, delay, max_slots=D * T)
    # template 0 is chirp-matched with delays up to 24 576: its autocorrelation needs a long response
    acorr = np.stack([sp.template_autocorr(bank_A, t, nj) for t in range(T)])
    ac_dev = torch.from_numpy(acorr.view(np.float32).reshape(T, 2 * nj + 1, 2)).cuda()
    dl_dev = torch.from_numpy(np.ascontiguousarray(delay, dtype=np.int32)).cuda()
    xs = torch.from_numpy(x).cuda()
    z = np.zeros((D, T, NC * 2048), np.complex64)
    out = torch.empty(D, T, 2048, 2, dtype=torch.float32, device="cuda")
    trig_dev = None
    for c in range(NC):
        bk.filter_chunk(xs[:, c * 2048:(c + 1) * 2048].contiguous(), out)
        z[:, :, c * 2048:(c + 1) * 2048] = out.cpu().numpy().view(np.complex64)[..., 0]
        if c == NC - 2:
            tr, cnt = bk.peaks(2.5, 0)
            torch.cuda.synchronize()
            trig_dev, trig = tr.clone(), sp.triggers_to_numpy(tr).copy()
    view = bk.snr_view()
    sky = plan.search(view, trig_dev, D * T)
    xi = sp.xi2_to_numpy(sp.signal_consistency(view, dl_dev, trig_dev, sky, D * T, ac_dev, nj))
    torch.cuda.synchronize()
    res = sp.results_to_numpy(sky)
    k_newest = NC * 2048 - 1
    ref = oracle.xi2(delay, z, T * ring, ring, ring, k_newest, trig["valid"], trig["tmpl"], trig["det"], trig["k"],
                     res["pix"], acorr.astype(np.complex128), nj)
    used = ref[:, D + 1] == 1
    assert used.sum() >= 20 and np.array_equal(xi["used"], used.astype(np.int32))
    assert np.array_equal(used, (trig["valid"] == 1) & (res["pix"] >= 0))
    for I in range(D):
        assert np.all(np.abs(xi["xi2"][:, I] - ref[:, I]) <= 1e-4 * ref[:, I] + 1e-5)
    assert np.all(np.abs(xi["xi2_c"] - ref[:, D]) <= 1e-4 * ref[:, D] + 1e-5)
    assert np.all(xi["xi2"][~used] == 0) and np.all(xi["xi2_c"][~used] == 0)
    # end to end, nothing from the CUDA path on the oracle's side: float64 SNR -> O4 -> O6 -> O8 with the oracle's
    # own float64 autocorrelation; compared where both chains chose the same sample and pixel
    z64 = oracle.filter_bank(x, bank)
    sl = slice((NC - 2) * 2048, (NC - 1) * 2048)
    k_o, v_o = oracle.peaks_mode0(z64[:, :, sl].reshape(D * T, 2048), 2.5)
    same = (v_o == 1) & (trig["valid"] == 1) & (k_o + (NC - 2) * 2048 == trig["k"])
    ref_s, pix_s, _ = oracle.sky_search(u2, delay, z64, T * ring, ring, ring, k_newest, same.astype(np.int32),
                                        trig["tmpl"], trig["det"], trig["k"])
    A64 = np.stack([oracle.template_autocorr(bank_A, t, nj) for t in range(T)])
    same &= pix_s[:, 0] == res["pix"]
    xe = oracle.xi2(delay, z64, T * ring, ring, ring, k_newest, same.astype(np.int32), trig["tmpl"], trig["det"],
                    trig["k"], pix_s[:, 0], A64, nj)
    idx = np.nonzero(same & (xe[:, D + 1] == 1))[0]
    assert len(idx) >= 15
    assert np.all(np.abs(xi["xi2_c"][idx] - xe[idx, D]) <= 1e-3 * xe[idx, D] + 1e-4)   # float32 table and SNR vs float64
    # noise candidates: a reduced chi^2 of order 1; not exactly 1, the windows are centred on maxima
    assert 0.5 < np.median(xi["xi2_c"][used]) < 1.5
    # background events: one-second slides of the same candidates (chunk NC-2: slides 1 and 2 exist, 3 does not)
    S = 3
    bgs = plan.background(view, trig_dev, D * T, S, 2048, [1, 1, 1])
    xib = sp.xi2_to_numpy(sp.signal_consistency(view, dl_dev, trig_dev, bgs, D * T, ac_dev, nj,
                                                n_slides=S, step=2048, mult=[1, 1, 1])).reshape(D * T, S)
    torch.cuda.synchronize()
    rb = sp.results_to_numpy(bgs).reshape(D * T, S)
    refb = oracle.xi2(delay, z, T * ring, ring, ring, k_newest, trig["valid"], trig["tmpl"], trig["det"], trig["k"],
                      rb["pix"], acorr.astype(np.complex128), nj, n_slides=S, step=2048, slide_mult=[1, 1, 1])
    assert np.array_equal(xib["used"], refb[:, :, D + 1].astype(np.int32))
    assert xib["used"][:, 0].sum() >= 20 and xib["used"][:, 2].sum() == 0
    assert np.all(np.abs(xib["xi2_c"] - refb[:, :, D]) <= 1e-4 * refb[:, :, D] + 1e-5)
    for I in range(D):
        assert np.all(np.abs(xib["xi2"][:, :, I] - refb[:, :, I]) <= 1e-4 * refb[:, :, I] + 1e-5)
    # a window that leaves the view (candidates of the newest chunk, k + 175 > k_newest for some) is refused
    tr2, _ = bk.peaks(0.0, 0)
    sky2 = plan.search(view, tr2, D * T)
    xi2b = sp.xi2_to_numpy(sp.signal_consistency(view, dl_dev, tr2, sky2, D * T, ac_dev, nj))
    t2, r2 = sp.triggers_to_numpy(tr2), sp.results_to_numpy(sky2)
    ref2 = oracle.xi2(delay, z, T * ring, ring, ring, k_newest, t2["valid"], t2["tmpl"], t2["det"], t2["k"],
                      r2["pix"], acorr.astype(np.complex128), nj)
    assert np.array_equal(xi2b["used"], ref2[:, D + 1].astype(np.int32)) and (xi2b["used"] == 0).any()


# ------------------------------------------------------------------ NEXT-2: ranking statistic, FAP, FAR (Eq. 13-15)
def test_rank_statistic_fap_far(sp, U):
    """spiir_rank_* against oracle/rank.py on seeded event lists shaped like the background of a chunk
    (rho_C^2 = trigger power + chi^2_4, xi^2 reduced chi^2, 10 % unused, values planted exactly on bin and cut
    edges).  Histogram, R counts and FAP counts are integers: bit-exact.  R / FAP / FAR of the candidates:
    one float32 rounding of the same integer ratio."""
    import torch
    from oracle import rank
    rng = np.random.default_rng(31)
    n_slots, S = 700, 13
    snr = rng.uniform(4.0, 7.0, n_slots).astype(np.float32)
    trig = np.zeros(n_slots, sp.TRIGGER_DTYPE)
    trig["valid"] = 1; trig["snr"] = snr; trig["tmpl"] = np.arange(n_slots)
    trig["valid"][::11] = 0

    def events(n):
        base = np.repeat(snr, n // n_slots) ** 2
        coh2 = (base + rng.chisquare(4, n) * rng.uniform(0.5, 6.0, n)).astype(np.float32)
        xi2 = (rng.chisquare(30, n) / 30 * rng.choice([1.0, 1.0, 3.0], n)).astype(np.float32)
        used = (rng.random(n) < 0.9).astype(np.int32)
        return coh2, xi2, used

    bins = (48, 40, 4.0, 7.5, -1.0, 2.0)
    coh2, xi2, used = events(n_slots * S)
    # plant edge cases: exact bin edges (u integer and half-integer), exact cut edge, zeros, huge values
    coh2[:6] = np.float32([16.0, 2.0 ** 7.5, 64.0, 181.01933, 1e9, 0.0])
    xi2[:6] = np.float32([0.5, 1.0, 2.0, 4.0, 1e-9, 0.0])
    edge = (np.float32(snr[1]) + np.float32(1.41421356)) ** 2
    coh2[S], coh2[S + 1] = edge, np.nextafter(edge, np.float32(0))
    used[S] = used[S + 1] = 1
    bg = np.zeros(n_slots * S, sp.RESULT_DTYPE)
    bg["coh2"] = coh2; bg["tot2"] = coh2; bg["pix"] = np.where(used == 1, 5, -1)
    xi = np.zeros(n_slots * S, sp.XI2_DTYPE)
    xi["xi2_c"] = xi2; xi["used"] = used
    to_dev = lambda a: torch.from_numpy(a.view(np.uint8).reshape(len(a), -1).copy()).cuda()
    rk = sp.Ranker(*bins)
    td = to_dev(trig)
    half = (n_slots // 2) * S                                 # two accumulate calls = one histogram
    rk.accumulate(td, to_dev(bg[:half]), to_dev(xi[:half]), n_slots // 2, S)
    rk.accumulate(to_dev(trig[n_slots // 2:]), to_dev(bg[half:]), to_dev(xi[half:]), n_slots - n_slots // 2, S)
    rk.finalize()
    torch.cuda.synchronize()
    nb, H, Cc, F = rk.tables()
    snr_ev = np.repeat(snr, S)
    H_ref = rank.histogram(bins, snr_ev, coh2, xi2, used)
    assert nb == H_ref.sum() and 0.2 * len(coh2) < nb < len(coh2)
    assert np.array_equal(H, H_ref)
    C_ref = rank.rank_counts(H_ref)
    assert np.array_equal(Cc, C_ref)
    assert np.array_equal(F, rank.fap_counts(H_ref, C_ref))
    # foreground candidates
    c2, x2, u2_ = events(n_slots)
    c2[:40] *= 6.0                                            # some loud ones: R and FAP reach 0
    fg = np.zeros(n_slots, sp.RESULT_DTYPE); fg["coh2"] = c2; fg["pix"] = np.where(u2_ == 1, 3, -1)
    xf = np.zeros(n_slots, sp.XI2_DTYPE); xf["xi2_c"] = x2; xf["used"] = u2_
    T_b = 13.0 * 7.0
    out = sp.rank_to_numpy(rk.candidates(td, to_dev(fg), to_dev(xf), n_slots, T_b))
    torch.cuda.synchronize()
    R, fap, far, sel = rank.candidates(bins, H_ref, snr, c2, x2, u2_ * trig["valid"], T_b)
    assert np.array_equal(out["selected"], sel) and 0.2 * n_slots < sel.sum() < n_slots
    np.testing.assert_allclose(out["rank"], R, rtol=1e-6, atol=0)
    np.testing.assert_allclose(out["fap"], fap, rtol=1e-6, atol=0)
    np.testing.assert_allclose(out["far"], far, rtol=1e-6, atol=0)
    assert (out["fap"][sel == 1] == 0).any() and (out["fap"][sel == 1] > 0.5).any()
    # reset empties everything
    rk.reset(); rk.finalize()
    torch.cuda.synchronize()
    nb0, H0, C0, F0 = rk.tables()
    assert nb0 == 0 and not H0.any() and not C0.any() and not F0.any()


# ------------------------------------------------------------------ configs 1 and 2 in FULL, oracle in full
def test_cfg1_full(sp, U):
    """BASELINE.json config 1 complete: 512 templates x 300 filters, 3 detectors, 16 s, the chirp injection,
    peaks above 4 in every chunk, sky search (nside 16) of every candidate with the one-chunk lag."""
    import torch
    cfg = workloads.config(1)
    T, D = cfg["n_templates"], 3
    bank = workloads.bank_for_config(1)
    st = workloads.strain_for_config(1)
    x = st["strain"]
    NC = x.shape[1] // 2048
    z_ref = oracle.filter_bank(x, bank)
    u2, delay = _table(cfg, gmst=st["gmst"])
    ring = 3 * 2048
    bk = sp.Bank(bank, D, 2048, ring_len=ring, bank_size=512)
    plan = sp.SkyPlan(u2, delay, max_slots=D * T)
    xs = torch.from_numpy(x).cuda()
    z = np.zeros((D, T, NC * 2048), np.complex64)
    out = torch.empty(D, T, 2048, 2, dtype=torch.float32, device="cuda")
    prev, n_cand, n_near, n_pixdiff, n_e2e = None, 0, 0, 0, 0
    for c in range(NC):
        bk.filter_chunk(xs[:, c * 2048:(c + 1) * 2048].contiguous(), out)
        z[:, :, c * 2048:(c + 1) * 2048] = out.cpu().numpy().view(np.complex64)[..., 0]
        if prev is not None:
            res = sp.results_to_numpy(plan.search(bk.snr_view(), prev[0], D * T))
            torch.cuda.synchronize()
            k_newest = (c + 1) * 2048 - 1
            zr = np.zeros((D, T, ring), np.complex64)
            kk = np.arange(max(k_newest - ring + 1, 0), k_newest + 1)
            zr[:, :, kk % ring] = z[:, :, kk]
            n_pixdiff += U.check_sky(res, zr, ring, k_newest, u2, delay, prev[1])["pix_differs"]
            n_cand += int((res["pix"] >= 0).sum())
            # end to end with NOTHING from the CUDA path on the oracle's side: float64 SNR -> O4 -> O6, compared
            # where both sides chose the same sample (they all do unless a near-tie, A12)
            zr64 = np.zeros((D, T, ring), np.complex128)
            zr64[:, :, kk % ring] = z_ref[:, :, kk]
            slp = slice((c - 1) * 2048, c * 2048)
            k_o, v_o = oracle.peaks_mode0(z_ref[:, :, slp].reshape(D * T, 2048), 4.0)
            same = (v_o == 1) & (prev[1]["valid"] == 1) & (k_o + (c - 1) * 2048 == prev[1]["k"])
            ref_e, pix_e, map_e = oracle.sky_search(u2, delay, zr64, T * ring, ring, ring, k_newest, same.astype(np.int32),
                                                    prev[1]["tmpl"], prev[1]["det"], prev[1]["k"], want_map=True)
            idx = np.nonzero(same & (pix_e[:, 0] >= 0))[0]
            assert len(idx) > 0.9 * (prev[1]["valid"] == 1).sum() - 5 and np.all(res["pix"][idx] >= 0)
            cg, ce = res["coh2"][idx].astype(np.float64), ref_e[idx, 0, 0]
            assert np.all(np.abs(np.sqrt(cg) - np.sqrt(ce)) <= 1e-3) and np.all(np.abs(cg - ce) <= 1e-4 * ce + 1e-5)
            at_gpu_pix = map_e[idx, res["pix"][idx]]
            assert np.all(at_gpu_pix >= ce - np.maximum(1e-4 * ce, 1e-3))                  # A19 with the float64 map
            n_e2e += len(idx)
        tr, cnt = bk.peaks(4.0, 0)
        torch.cuda.synchronize()
        trig = sp.triggers_to_numpy(tr).copy()
        sl = slice(c * 2048, (c + 1) * 2048)
        n_near += U.check_peaks_mode0(trig, z[:, :, sl], z_ref[:, :, sl], c * 2048, 4.0)
        prev = (tr.clone(), trig)
    U.check_snr(z, z_ref)
    tr1, cnt1 = bk.peaks(4.0, 1)                              # mode 1 on the last chunk, one bank of 512 (A10)
    torch.cuda.synchronize()
    t1 = sp.triggers_to_numpy(tr1)
    for d in range(D):
        k1, v1 = oracle.peaks_mode1(z[d][:, -2048:], 4.0, 512)
        td_ = t1[d * T:(d + 1) * T]
        assert np.array_equal(td_["valid"], v1) and np.array_equal(td_["k"][v1 == 1] - (NC - 1) * 2048, k1[v1 == 1])
    assert int(cnt1.cpu()[0]) == int(t1["valid"].sum()) > 10
    assert n_cand > 3000                                      # ~36 % of the 1536 slots per second once the bank has filled
    assert n_e2e > 0.95 * n_cand
    print("cfg1 full: %d candidates searched (%d compared end to end with the float64 chain), %d near-tie peak "
          "indices (A12), %d set-valued pixels (A19)" % (n_cand, n_e2e, n_near, n_pixdiff))


def test_cfg2_full(sp, U):
    """BASELINE.json config 2 complete: 1024 templates x 600 filters over 8 rate bands, 2 detectors, 64 s in 1-s
    chunks with all state carried, per-chunk peaks; the oracle runs the whole stream in one shot, 128 templates
    at a time."""
    import torch
    cfg = workloads.config(2)
    T, D = cfg["n_templates"], 2
    bank = workloads.bank_for_config(2)
    dec, itp = workloads.halfband_taps()
    x = workloads.strain_for_config(2)["strain"]
    NC = x.shape[1] // 4096
    bk = sp.Bank(bank, D, 4096, ring_len=2 * 2048, dec_taps=dec, int_taps=itp)
    xs = torch.from_numpy(x).cuda()
    z = np.zeros((D, T, NC * 2048), np.complex64)
    out = torch.empty(D, T, 2048, 2, dtype=torch.float32, device="cuda")
    trigs = []
    for c in range(NC):
        bk.filter_chunk(xs[:, c * 4096:(c + 1) * 4096].contiguous(), out)
        tr, cnt = bk.peaks(4.0, 0)
        z[:, :, c * 2048:(c + 1) * 2048] = out.cpu().numpy().view(np.complex64)[..., 0]
        trigs.append(sp.triggers_to_numpy(tr).copy())
    worst, n_near = 0.0, 0
    for t0 in range(0, T, 128):
        sel = np.arange(t0, t0 + 128)
        z_ref = oracle.filter_bank(x, bank, dec, itp, templates=sel)
        worst = max(worst, U.check_snr(z[:, sel], z_ref))
        rows = (np.arange(D)[:, None] * T + sel[None, :]).reshape(-1)
        for c in (1, NC // 2, NC - 1):                        # three chunks' peaks end to end (every chunk would be 64x the time)
            sl = slice(c * 2048, (c + 1) * 2048)
            n_near += U.check_peaks_mode0(_subset_trig(trigs[c][rows], sel, D), z[:, sel][:, :, sl], z_ref[:, :, sl],
                                          c * 2048, 4.0)
    # every peak of every chunk, stage-isolated (bit-exact on the GPU's own z)
    for c in range(NC):
        k_iso, v_iso = oracle.peaks_mode0(z[:, :, c * 2048:(c + 1) * 2048].reshape(D * T, 2048), 4.0)
        assert np.array_equal(trigs[c]["k"] - c * 2048, k_iso) and np.array_equal(trigs[c]["valid"], v_iso)
    frac = np.mean([t["valid"].mean() for t in trigs[NC // 2:]])
    assert 0.1 < frac < 0.9
    print("cfg2 full: max |dz| %.2e, %d near-tie peak indices (A12), trigger fraction %.2f" % (worst, n_near, frac))


# ------------------------------------------------------------------ four detectors
def test_sky_four_detectors(sp, U):
    """N_d = 4 (the library's maximum): H1, L1, V1 and a fourth site built from seeded geometry (a detector's
    position and arm tensor are inputs of the table, A27).  Foreground with sky map, time slides, ring
    wrap-around - against the oracle.  With four detectors the null stream has 4 degrees of freedom."""
    import torch
    cfg = workloads.config(3)
    pos3, resp3 = workloads.detector_geometry(cfg["dets"])
    rng = np.random.default_rng(44)
    v = rng.standard_normal(3); v *= 6.37e6 / np.linalg.norm(v)              # somewhere on the Earth's surface
    x = np.cross(v, rng.standard_normal(3)); x /= np.linalg.norm(x)
    y = np.cross(v, x); y /= np.linalg.norm(y)
    pos = np.vstack([pos3, v[None]])
    resp = np.concatenate([resp3, (0.5 * (np.outer(x, x) - np.outer(y, y)))[None]])
    U2, delay = oracle.sky_table(8, pos, resp, [1.0, 1.0, 0.5, 0.7], 1.1, 2048.0)
    u2 = U2.astype(np.float32)
    rows, L, S, step = 150, 1400, 5, 200
    z = rng.standard_normal((4, rows, L, 2)).astype(np.float32)
    zc = z.view(np.complex64)[..., 0]
    k_newest = 2 * L + 77                                                     # the view is a ring that has wrapped twice
    trig = np.zeros(rows, sp.TRIGGER_DTYPE)
    trig["valid"] = 1; trig["tmpl"] = np.arange(rows); trig["det"] = rng.integers(0, 4, rows)
    trig["k"] = rng.integers(k_newest - 200, k_newest - 70, rows)
    plan = sp.SkyPlan(u2, delay, max_slots=rows)
    view = sp.SnrView(torch.from_numpy(z).cuda(), k_newest=k_newest)
    td = sp.triggers_from_numpy(trig)
    smap = torch.empty(rows, plan.n_pix, dtype=torch.float32, device="cuda")
    res = sp.results_to_numpy(plan.search(view, td, rows, skymap=smap))
    bg = sp.results_to_numpy(plan.background(view, td, rows, S, step, [1, 2, 1, 1]))
    torch.cuda.synchronize()
    ref = U.oracle_sky_on(zc, L, k_newest, u2, delay, trig, want_map=True)
    U.check_sky(res, zc, L, k_newest, u2, delay, trig, ref=ref)
    assert (res["pix"] >= 0).sum() > 100
    m = smap.cpu().numpy()
    tot = np.maximum(ref[0][:, 0, 2], 1.0)[:, None]
    assert np.all(np.abs(m - ref[2]) <= 1e-4 * ref[2] + 2e-6 * tot)
    U.check_sky(bg, zc, L, k_newest, u2, delay, trig, n_slides=S, step=step, mult=[1, 2, 1, 1])
    ok = res["pix"] >= 0
    assert 2.0 < np.mean(res["null2"][ok]) < 6.0 * 1.5                        # ~ (2 N_d - 4) = 4 dof at the arg-max, minus selection


# ------------------------------------------------------------------ NEXT-3: half-hourly table sets
def test_sky_table_set_nearest_in_time(sp, U):
    """the search uses the U / offset sample closest in time to the candidate.  The product
    builds its own 48 tables (spiir_sky_table_set_build) and selects with spiir_sky_table_nearest; the
    oracle builds its set with numpy's SVD and selects by exhaustive comparison."""
    import torch
    cfg = workloads.config(3)
    pos, resp = workloads.detector_geometry(cfg["dets"])
    nside, n_sets, dt, t0, g0 = 8, 48, 1800.0, 1.2e9, 0.4
    U2o, dlo = oracle.table_set(nside, pos, resp, cfg["sigma"], g0, dt, n_sets, 2048.0)
    u2p, dlp = sp.sky_table_set_build(nside, pos, resp, cfg["sigma"], g0, dt, n_sets, 2048.0)
    n_rows = 64
    pset = sp.SkyPlanSet(u2p, dlp, max_slots=n_rows, t0=t0, interval_s=dt)
    rng = np.random.default_rng(31)
    # signals as they arrive at the time of set 5; candidates stamped around it
    z, tdet, k, truth = workloads.snr_snippets(rng, U2o[5].astype(np.float32), dlo[5], n_rows, 1, 102, 0.5)
    zc = np.ascontiguousarray(z).view(np.complex64)[..., 0]
    L = zc.shape[2]
    trig = np.zeros(n_rows, sp.TRIGGER_DTYPE)
    trig["valid"] = 1
    trig["tmpl"] = np.arange(n_rows)
    trig["det"] = tdet
    trig["k"] = k
    view = sp.SnrView(torch.from_numpy(np.ascontiguousarray(z)).cuda())
    td = sp.triggers_from_numpy(trig)
    seen = set()
    for t in (t0 + 5 * dt, t0 + 5 * dt - 899.0, t0 + 5 * dt + 900.0, t0 + 5 * dt + 901.0, t0 + 3 * dt + 1000.0,
              t0 + 47 * dt + 900.0, t0 - 900.0):
        i = oracle.nearest_table(t, t0, dt, n_sets)
        assert pset.index(t) == i
        seen.add(i)
        res = sp.results_to_numpy(pset.select(t).search(view, td, n_rows))
        torch.cuda.synchronize()
        U.check_sky(res, zc, L, L - 1, U2o[i].astype(np.float32), dlo[i], trig)
        if i == 5:
            sig = truth["is_signal"]
            assert np.mean(res["coh2"][sig]) > 3 * np.mean(res["coh2"][~sig])
    assert seen == {0, 4, 5, 6, 47}
    for t in (t0 - 901.0, t0 + 47 * dt + 901.0):
        with pytest.raises(sp.SpiirError):
            pset.select(t)
    pset.close()


# ------------------------------------------------------------------ NEXT-3: sub-sample alignment
def test_sub_sample_alignment(sp, U):
    """spiir_snr_upsample_windows + coherent_sky_search with a table at R x 2048 Hz, against oracle O11
    (cubic Lagrange in float64) + O6.  Windows: bit copies at the input samples, 1e-6 of the window's
    largest |z| elsewhere; search: stage-isolated on the GPU's windows and end to end on the oracle's."""
    import torch
    rng = np.random.default_rng(77)
    ns, fs, R, H = 8, 2048.0, 3, 58       # R = 3: the widest windows (trigger in V1) of 32 pairs still fit shared memory
    cfg = workloads.config(3)
    pos, resp = workloads.detector_geometry(cfg["dets"])
    U1, d1 = oracle.sky_table(ns, pos, resp, cfg["sigma"], 0.9, fs)
    UR, dR = oracle.sky_table(ns, pos, resp, cfg["sigma"], 0.9, fs * R)
    assert np.abs(d1 - d1[:, :1]).max() < H
    th, ph = oracle.healpix_ring_centres(ns)
    lam = ph - 0.9
    nvec = np.stack([np.sin(th) * np.cos(lam), np.sin(th) * np.sin(lam), np.cos(th)], 1)
    tau = -(nvec @ pos.T) / workloads.C_LIGHT * fs                  # arrival offsets in samples, not rounded
    D, rows, L, k_newest = 3, 40, 700, 1000                         # ring holds k = 301 .. 1000, wrapped
    z = (rng.standard_normal((D, rows, L)) + 1j * rng.standard_normal((D, rows, L))) * math.sqrt(0.5)
    kk = np.arange(k_newest - L + 1, k_newest + 1)
    trig = np.zeros(rows, sp.TRIGGER_DTYPE)
    trig["valid"] = 1
    trig["tmpl"] = rng.permutation(rows)
    trig["det"] = rng.integers(0, D, rows)
    trig["k"] = rng.integers(301 + H + 1, 1000 - H - 1, rows)
    trig["k"][:6] = [301 + H + 1, 301 + H, 1000 - H - 1, 1000 - H, 650, 700]   # both edges, in and out
    trig["valid"][4] = 0
    p_true = rng.integers(0, 768, rows)
    for s in range(6, rows):                                       # loud signals arriving between samples
        T, r, k0 = int(trig["det"][s]), int(trig["tmpl"][s]), int(trig["k"][s])
        c = (rng.standard_normal(2) + 1j * rng.standard_normal(2)) * 8.0
        amp = U1[p_true[s]] @ c
        for I in range(D):
            x = kk - k0 - (tau[p_true[s], I] - tau[p_true[s], T])
            z[I, r, kk % L] += amp[I] * np.exp(-x ** 2 / (2 * 6.0 ** 2)) * np.exp(0.3j * x)
    z32 = z.astype(np.complex64)
    trig["z_re"] = z32[trig["det"], trig["tmpl"], trig["k"] % L].real
    trig["z_im"] = z32[trig["det"], trig["tmpl"], trig["k"] % L].imag
    trig["snr"] = np.abs(z32[trig["det"], trig["tmpl"], trig["k"] % L])
    zt = torch.from_numpy(np.ascontiguousarray(z32).view(np.float32).reshape(D, rows, L, 2)).cuda()
    view = sp.SnrView(zt, k_newest=k_newest)
    wview, wtrig = sp.upsample_windows(view, D, sp.triggers_from_numpy(trig), rows, R, H)
    torch.cuda.synchronize()
    Lw = 2 * R * H + 1
    Lp = wview.c.row_stride
    assert Lp == Lw + 1 and wview.c.ring_len == Lp and wview.c.k_newest == Lw - 1 and wview.c.det_stride == rows * Lp
    g = wview._keep.cpu().numpy().reshape(-1)[:D * rows * Lp * 2].view(np.complex64).reshape(D, rows, Lp)
    ref, ok = oracle.upsample_windows(z32, L, k_newest, trig["valid"], trig["tmpl"], trig["det"], trig["k"], R, H)
    assert list(ok[:6]) == [1, 0, 1, 0, 0, 1] and ok[6:].all()
    t2 = wtrig.cpu().numpy().view(sp.TRIGGER_DTYPE).reshape(-1)
    assert np.array_equal(t2["valid"], ok) and np.array_equal(t2["tmpl"], np.arange(rows))
    assert np.all(t2["k"] == R * H)
    v = ok == 1
    for f in ("det", "z_re", "z_im", "snr"):
        assert np.array_equal(t2[f][v], trig[f][v])
    assert np.all(g[:, :, Lw:] == 0) and np.all(g[:, ~v] == 0)
    assert np.array_equal(g[:, v, 0:Lw:R], ref[:, v, 0:Lw:R].astype(np.complex64))     # bit copies
    scale = np.abs(ref).max(axis=2, keepdims=True)
    assert np.all(np.abs(g[:, :, :Lw] - ref) <= 1e-6 * scale + 1e-30)
    # search on the windows
    plan = sp.SkyPlan(UR.astype(np.float32), dR, max_slots=rows)
    res = sp.results_to_numpy(plan.search(wview, wtrig, rows))
    torch.cuda.synchronize()
    U.check_sky(res, np.ascontiguousarray(g), Lp, Lw - 1, UR.astype(np.float32), dR, t2)   # stage-isolated
    refp = np.zeros((D, rows, Lp), complex)
    refp[:, :, :Lw] = ref
    oo, op, _ = oracle.sky_search(UR.astype(np.float32), dR, refp, rows * Lp, Lp, Lp, Lw - 1,
                                  ok, np.arange(rows), trig["det"], np.full(rows, R * H))      # end to end
    assert np.all(np.abs(res["coh2"][v] - oo[v, 0, 0]) <= 1e-4 * oo[v, 0, 0])
    assert np.all(res["pix"][~v] == -1)
    # against the integer-sample search of the same candidates: less null power, true pixel found
    plan1 = sp.SkyPlan(U1.astype(np.float32), d1, max_slots=rows)
    res1 = sp.results_to_numpy(plan1.search(view, sp.triggers_from_numpy(trig), rows))
    torch.cuda.synchronize()
    sig = np.arange(rows) >= 6
    assert np.mean(res["null2"][sig]) < np.mean(res1["null2"][sig])
    assert np.mean(res["pix"][sig] == p_true[sig]) >= np.mean(res1["pix"][sig] == p_true[sig])
    # ---- the time-slide background on the same finer grid: companions read s * step earlier, every
    #      detector's window resampled around its own centre; rows [slot][slide]
    S, step, mult = 4, 60, [1, 1, 1]
    sview, strig = sp.upsample_windows(view, D, sp.triggers_from_numpy(trig), rows, R, H, n_slides=S, step=step, mult=mult)
    torch.cuda.synchronize()
    gs = sview._keep.cpu().numpy().reshape(-1)[:D * rows * S * Lp * 2].view(np.complex64).reshape(D, rows * S, Lp)
    refs, oks = oracle.upsample_windows(z32, L, k_newest, trig["valid"], trig["tmpl"], trig["det"], trig["k"], R, H,
                                        n_slides=S, step=step, slide_mult=mult)
    t3 = strig.cpu().numpy().view(sp.TRIGGER_DTYPE).reshape(-1)
    assert np.array_equal(t3["valid"], oks) and 0.3 * rows * S < oks.sum() < rows * S      # late slides leave the ring
    assert np.array_equal(t3["tmpl"], np.arange(rows * S)) and int(sview.c.n_rows) == rows * S
    vs = oks == 1
    assert np.all(gs[:, ~vs] == 0) and np.array_equal(gs[:, vs, 0:Lw:R], refs[:, vs, 0:Lw:R].astype(np.complex64))
    assert np.all(np.abs(gs[:, :, :Lw] - refs) <= 1e-6 * np.abs(refs).max(axis=2, keepdims=True) + 1e-30)
    plan_s = sp.SkyPlan(UR.astype(np.float32), dR, max_slots=rows * S)
    res_s = sp.results_to_numpy(plan_s.search(sview, strig, rows * S))
    torch.cuda.synchronize()
    U.check_sky(res_s, np.ascontiguousarray(gs), Lp, Lw - 1, UR.astype(np.float32), dR, t3)  # O6 on the device's windows
    refsp = np.zeros((D, rows * S, Lp), complex)
    refsp[:, :, :Lw] = refs
    os_, ps_, _ = oracle.sky_search(UR.astype(np.float32), dR, refsp, rows * S * Lp, Lp, Lp, Lw - 1, oks,
                                    np.arange(rows * S), np.repeat(trig["det"], S), np.full(rows * S, R * H))
    assert np.all(np.abs(res_s["coh2"][vs] - os_[vs, 0, 0]) <= 1e-4 * os_[vs, 0, 0]) and np.all(res_s["pix"][~vs] == -1)
    # with factor 1 the windows are bit copies and the search on them IS timeslide_background on the integer grid
    # (same samples, same arithmetic): identical results wherever both windows exist
    v1, t1 = sp.upsample_windows(view, D, sp.triggers_from_numpy(trig), rows, 1, H, n_slides=S, step=step, mult=mult)
    plan_1s = sp.SkyPlan(U1.astype(np.float32), d1, max_slots=rows * S)
    r_w = sp.results_to_numpy(plan_1s.search(v1, t1, rows * S))
    r_b = sp.results_to_numpy(plan_1s.background(view, sp.triggers_from_numpy(trig), rows, S, step, mult))
    torch.cuda.synchronize()
    both = (r_w["pix"] >= 0) & (r_b["pix"] >= 0)
    assert both.sum() >= 0.3 * rows * S and np.all((r_w["pix"] >= 0) <= (r_b["pix"] >= 0))   # (the windows need one sample of margin more)
    for fld in ("coh2", "tot2", "null2", "pix"):
        assert np.array_equal(r_w[fld][both], r_b[fld][both]), fld
    assert np.mean(res["pix"][sig] == p_true[sig]) > 0.5


# ------------------------------------------------------------------ NEXT-4: front end on the device
@pytest.mark.parametrize("shape", ["paper", "small"])
def test_frontend_downsample_whiten_gate(sp, U, shape):
    """spiir_frontend_chunk against oracle/frontend.py (W1-W6) on seeded coloured noise with glitches, hop by hop from
    the start of a stream: the paper's shape (16 384 -> 2048 Hz, 192 taps, 2-s hops = 8192-point transforms, 27
    blocks of PSD history, 0.25 s pads) and a small one (decimation 4, 512-point transforms,
    odd history).  Tolerance: 1e-4 of the whitened standard deviation (= 1) once the estimate has three blocks; the
    first emitted hops divide by single raw periodograms and are compared at 5e-3 of the hop's rms.
    The gate decision |d_w| > threshold is float32 on the device: exact agreement is required wherever the oracle's
    |d_w| is not within 1e-3 of the threshold (nowhere, for these inputs)."""
    import torch
    from oracle import frontend as fe
    if shape == "paper":
        D, R, nt, H, nh, pad, fs, n_hops, thr = 3, 8, 192, 4096, 27, 512, 2048.0, 34, 8.0
        gl = [(0, 41.3, 300.0), (2, 20.05, -500.0), (2, 20.4, 400.0), (1, 59.99, 350.0)]
    else:
        D, R, nt, H, nh, pad, fs, n_hops, thr = 2, 4, 64, 256, 9, 100, 2048.0, 30, 6.0
        gl = [(0, 1.51, 300.0), (1, 2.999, 250.0)]
    taps = workloads.frontend_taps(R, nt)
    x = workloads.frontend_strain(70 + n_hops, D, R * H * n_hops, fs_in=fs * R, glitches=gl)
    ref, dw_ref = fe.frontend(x, taps, R, H, fs, nh, thr, pad)
    # knife-edge gate decisions (|d_w| within 1e-3 of the threshold) may fall either way in float32: the device's zeros
    # must contain those of threshold + 1e-3 and be contained in those of threshold - 1e-3
    ref_hi, _ = fe.frontend(x, taps, R, H, fs, nh, thr + 1e-3, pad)
    ref_lo, _ = fe.frontend(x, taps, R, H, fs, nh, thr - 1e-3, pad)
    f = sp.FrontEnd(D, taps, decim=R, hop=H, n_hist=nh, gate_pad=pad, out_rate_hz=fs, gate_threshold=thr)
    xd = torch.from_numpy(x).cuda()
    psd = torch.zeros(D, H + 1, dtype=torch.float32, device="cuda")
    got = np.zeros((D, n_hops * H), np.float32)
    for c in range(n_hops):
        o = f.chunk(xd[:, c * H * R:(c + 1) * H * R].contiguous(), psd=psd)
        got[:, c * H:(c + 1) * H] = o.cpu().numpy()
        if c == 12:                                                          # the PSD used for block 12 against the oracle's
            y = fe.downsample(x[1], taps, R)
            _, S, _ = fe.whiten_stream(y, H, fs, nh)
            np.testing.assert_allclose(psd[1].cpu().numpy(), S[12], rtol=2e-4, atol=1e-12)
    torch.cuda.synchronize()
    zero_ref, zero_got = ref == 0.0, got == 0.0
    assert np.all(zero_got[ref_hi == 0.0]) and np.all((ref_lo == 0.0)[zero_got]), "gated samples differ"
    ref = np.where(zero_got, 0.0, np.where(zero_ref, ref_hi, ref))           # values compared where the device kept them
    assert zero_ref[:, 6 * H:].sum() >= (len(gl) - 1) * 2 * pad              # the glitches and their pads are gone (two windows overlap)
    warm = 5 * H + pad                                                       # output index from which >= 3 blocks back the estimate
    err = np.abs(got - ref)
    assert err[:, warm:].max() <= 1e-4, err[:, warm:].max()
    # warm-up: the first emitted hops divide by one or three raw periodograms, whose smallest bins are float32
    # cancellation noise of the transform relative to the largest ones; compared against the hop's rms
    for c in range(warm // H + 1):
        sl = slice(c * H, min((c + 1) * H, warm))
        rms = max(1.0, float(np.sqrt(np.mean(ref[:, sl] ** 2))))
        assert err[:, sl].max() <= 5e-3 * rms, (c, err[:, sl].max(), rms)
    assert 0.9 < got[:, 12 * H:][~zero_got[:, 12 * H:]].std() < (1.15 if nh >= 27 else 1.3)   # unit variance out (a short history biases 1 / S-hat up)
    # a second front end of another shape, set up and run in between, must not disturb this one (the opt-in
    # shared-memory limit belongs to the kernel, not to an instance: a smaller instance used to lower it)
    other = sp.FrontEnd(1, workloads.frontend_taps(2, 16), decim=2, hop=256, n_hist=3, gate_pad=0, out_rate_hz=fs,
                        gate_threshold=50.0)
    other.chunk(xd[:1, :512].contiguous())
    # reset: the same stream again gives the same output bit for bit
    f.reset()
    o0 = f.chunk(xd[:, :H * R].contiguous())
    o1 = f.chunk(xd[:, H * R:2 * H * R].contiguous())
    torch.cuda.synchronize()
    assert np.array_equal(o0.cpu().numpy(), got[:, :H]) and np.array_equal(o1.cpu().numpy(), got[:, H:2 * H])


# ------------------------------------------------------------------ out-of-bounds writes (compute-sanitizer is closed on this pool)
def test_workspace_guard_bands(sp, U):
    """compute-sanitizer cannot be run on this pool (gpurun refuses it), so out-of-bounds WRITES are looked for
    directly: every buffer the library writes — the bank's workspace, the sky plan's workspace, the trigger / result /
    SNR outputs, the front end's workspace and output — is carved out of a larger allocation filled with a byte
    pattern, the whole path runs (multirate bank with a long-delay template, both peak modes, the sky
    search with slides on a wrapped ring, xi^2, the front end), and the guard bands on both sides of
    every buffer must still hold the pattern."""
    import ctypes as C
    import torch
    G = 1 << 16                                                               # 64 KB of guard on either side
    guards = []

    def guarded(nbytes, align=256):
        raw = torch.full((nbytes + 2 * G + align,), 0xA5, dtype=torch.uint8, device="cuda")
        off = (-(raw.data_ptr() + G)) % align + G
        guards.append((raw, off, nbytes))
        return raw, raw.data_ptr() + off

    L_ = sp.lib()
    st = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    cfg = workloads.config(4)
    T, D = 48, 3
    bank = workloads.bank_for_config(4, n_templates=T)                       # 20 chirp-matched long-delay templates + random
    dec, itp = workloads.halfband_taps()
    ring = 5 * 2048
    desc, keep = sp.make_desc(bank, D, 4096, ring, 16, dec, itp)
    nb = C.c_size_t(0)
    assert L_.spiir_bank_workspace_bytes(C.byref(desc), C.byref(nb)) == 0
    _, ws = guarded(nb.value)
    h = C.c_void_p()
    assert L_.spiir_bank_init(C.byref(h), C.byref(desc), C.c_void_p(ws), nb, st) == 0
    x = torch.from_numpy(workloads.strain_for_config(4, seconds=8)["strain"]).cuda()
    _, p_out = guarded(D * T * 2048 * 8)
    _, p_trig = guarded(D * T * 40)
    _, p_cnt = guarded(4, align=16)
    u2, delay = _table(cfg, nside=8, gmst=0.4)
    pb = C.c_size_t(0)
    plans = []
    for _ in range(1):
        assert L_.spiir_sky_plan_workspace_bytes(D, len(u2), D * T, C.byref(pb)) == 0
        _, pws = guarded(pb.value)
        ph = C.c_void_p()
        u2c, dlc = np.ascontiguousarray(u2, np.float32), np.ascontiguousarray(delay, np.int32)
        assert L_.spiir_sky_plan_init(C.byref(ph), D, len(u2), D * T, u2c.ctypes.data_as(C.c_void_p),
                                      dlc.ctypes.data_as(C.c_void_p), C.c_void_p(pws), pb, st) == 0
        plans.append(ph)
    S = 3
    _, p_fg = guarded(D * T * 16)
    _, p_bg = guarded(D * T * S * 16)
    _, p_xi = guarded(D * T * S * 24)
    nj = 20
    ac = torch.zeros(T, 2 * nj + 1, 2, device="cuda"); ac[:, nj, 0] = 1.0
    dl_dev = torch.from_numpy(np.ascontiguousarray(delay, np.int32)).cuda()
    mult = (C.c_int32 * D)(1, 1, 1)
    view = sp.spiir_snr_view()
    for c in range(8):                                                        # the 5-s ring wraps
        xc = x[:, c * 4096:(c + 1) * 4096].contiguous()
        assert L_.spiir_filter_chunk(h, C.c_void_p(xc.data_ptr()), 4096, C.c_void_p(p_out), st) == 0
        for mode in (1, 0):
            assert L_.spiir_peaks(h, C.c_float(1.0), mode, C.c_void_p(p_trig), C.c_void_p(p_cnt), st) == 0
        assert L_.spiir_bank_snr_view(h, C.byref(view)) == 0
        for ph in plans:
            assert L_.coherent_sky_search(ph, C.byref(view), C.c_void_p(p_trig), D * T, C.c_void_p(p_fg), None, st) == 0
            assert L_.timeslide_background(ph, C.byref(view), C.c_void_p(p_trig), D * T, S, C.c_int64(2048), mult,
                                           C.c_void_p(p_bg), st) == 0
        assert L_.spiir_signal_consistency(C.byref(view), D, len(u2), C.c_void_p(dl_dev.data_ptr()), C.c_void_p(p_trig),
                                           C.c_void_p(p_bg), D * T, S, C.c_int64(2048), mult, C.c_void_p(ac.data_ptr()),
                                           nj, C.c_void_p(p_xi), st) == 0
    # the front end
    taps = workloads.frontend_taps(8, 192)
    fd = sp.spiir_frontend_desc(D, 8, 192, 1024, 9, 256, 2048.0, 8.0, taps.ctypes.data)
    fb = C.c_size_t(0)
    assert L_.spiir_frontend_workspace_bytes(C.byref(fd), C.byref(fb)) == 0
    _, fws = guarded(fb.value)
    fh = C.c_void_p()
    assert L_.spiir_frontend_init(C.byref(fh), C.byref(fd), C.c_void_p(fws), fb, st) == 0
    raw = torch.from_numpy(workloads.frontend_strain(5, D, 8 * 1024 * 12)).cuda()
    _, p_fo = guarded(D * 1024 * 4)
    _, p_ps = guarded(D * 1025 * 4, align=16)
    for c in range(12):
        rc_ = raw[:, c * 8192:(c + 1) * 8192].contiguous()
        assert L_.spiir_frontend_chunk(fh, C.c_void_p(rc_.data_ptr()), C.c_void_p(p_fo), C.c_void_p(p_ps), st) == 0
    torch.cuda.synchronize()
    # ... and every buffer was written to (the pattern is gone from its interior), none beyond its ends
    for raw_t, off, nbytes in guards:
        assert not bool((raw_t[off:off + nbytes] == 0xA5).all())
        lo, hi = raw_t[:off], raw_t[off + nbytes:]
        assert bool((lo == 0xA5).all()) and bool((hi == 0xA5).all()), "a guard band was overwritten (buffer of %d bytes)" % nbytes
    for ph in plans:
        L_.spiir_sky_plan_free(ph)
    L_.spiir_frontend_free(fh)
    L_.spiir_bank_free(h)


# ------------------------------------------------------------------ the N > 1 path on the CUDA side (one GPU available)
def test_template_shards_on_the_cuda_path(sp, U):
    """The multi-GPU path shards by template with no exchange step.  Only one
    GPU is available, and ranks must not be emulated as concurrent processes on it, so the two ranks' shards are run
    one after the other through the C ABI: each rank's sub-bank (shard.template_shard / slice_bank, whole banks of
    `bank_size`) must reproduce its rows of the unsharded run — SNR to float32 rounding, peaks, sky results of its
    candidates — and the merged trigger lists must cover the unsharded list (the world-size-2 gloo test covers the
    host-side merge and timing reductions)."""
    import torch
    from paper_2011_06787_b200 import shard as shd
    cfg = workloads.config(2)
    T, D, NC, bs = 24, 3, 3, 4
    bank = workloads.bank_for_config(2, n_templates=T)
    dec, itp = workloads.halfband_taps()
    x = workloads.gaussian_strain(np.random.default_rng(9), D, NC * 4096)
    u2, delay = _table(workloads.config(1), nside=8, gmst=0.2)

    def run(b):
        z, trigs, bk = U.run_bank(b, x, 4096, ring_len=NC * 2048, bank_size=bs, taps=(dec, itp), peak_thr=2.0)
        plan = sp.SkyPlan(u2, delay, max_slots=D * b["n_templates"])
        prev = sp.triggers_from_numpy(trigs[NC - 2][0])
        res = sp.results_to_numpy(plan.search(bk.snr_view(), prev, D * b["n_templates"]))
        torch.cuda.synchronize()
        return z, trigs, res

    z_full, trig_full, res_full = run(bank)
    merged = []
    for rank in range(2):
        t0, t1 = shd.template_shard(rank, 2, T, bank_size=bs)
        assert (t0, t1) == ((0, 12), (12, 24))[rank]
        z, trigs, res = run(shd.slice_bank(bank, t0, t1))
        # a shard is an exact sub-problem: the same filters, states and inputs; only the order in which a template's
        # filters are summed may differ (the lane layout is planned per bank), i.e. float32 rounding
        assert np.abs(z - z_full[:, t0:t1]).max() <= 2e-6
        rows = (np.arange(D)[:, None] * T + np.arange(t0, t1)[None, :]).reshape(-1)
        for c in range(NC):
            tf, ts = trig_full[c][0][rows], trigs[c][0]
            same = tf["k"] == ts["k"]
            assert same.mean() >= 0.97                                       # (near-ties of the maximum, A12)
            assert np.array_equal(tf["valid"][same], ts["valid"][same]) and np.array_equal(tf["det"], ts["det"])
            assert np.array_equal(tf["tmpl"], ts["tmpl"] + t0)
            assert np.all(np.abs(tf["snr"][same] - ts["snr"][same]) <= 2e-6)
        tf, ts = trig_full[NC - 2][0][rows], trigs[NC - 2][0]
        ok = (tf["k"] == ts["k"]) & (tf["valid"] == 1) & (ts["valid"] == 1)
        assert ok.sum() >= 10 and np.array_equal(res_full[rows]["pix"][ok] >= 0, res["pix"][ok] >= 0)
        hit = ok & (res["pix"] >= 0)
        assert np.all(np.abs(res_full[rows]["coh2"][hit] - res["coh2"][hit]) <= 1e-5 * res["coh2"][hit])
        merged.append(shd.merge_triggers(trigs[NC - 1][0], t0))              # single process: the rank's own list, global indices
    allm = np.concatenate(merged)
    full = trig_full[NC - 1][0]
    full = full[full["valid"] == 1]
    assert abs(len(allm) - len(full)) <= 2
    common = set(zip(allm["det"], allm["tmpl"], allm["k"])) & set(zip(full["det"], full["tmpl"], full["k"]))
    assert len(common) >= 0.97 * len(full)
