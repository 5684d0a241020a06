"""CPU-only checks of the C-ABI library: it builds, loads, exports every symbol that
include/spiir.h declares, and rejects bad arguments before touching a device.
(No compute calls here; parity lives in the -m gpu tests.)"""
import ctypes as C
import os
import re

import numpy as np
import pytest

import workloads

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def sp():
    from paper_2011_06787_b200 import build
    build.build()
    import paper_2011_06787_b200 as sp
    sp.lib()
    return sp


def _declared():
    txt = open(os.path.join(ROOT, "include", "spiir.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    names = re.findall(r"\b([a-z][a-z0-9_]*)\s*\(", txt)
    return sorted({n for n in names if n.startswith("spiir_") or n in ("coherent_sky_search", "timeslide_background")})


def test_every_declared_symbol_is_exported(sp):
    L = C.CDLL(sp.LIB_PATH)
    decl = _declared()
    assert {"spiir_bank_init", "spiir_filter_chunk", "spiir_peaks", "coherent_sky_search",
            "timeslide_background"} <= set(decl)
    for n in decl:
        assert hasattr(L, n), n
    assert sorted(sp.EXPORTS) == decl                      # the binding names the same set


def test_struct_sizes_match_the_header(sp):
    assert C.sizeof(sp.spiir_snr_view) == 48
    assert C.sizeof(sp.spiir_bank_desc) == 16 + 32 + 32 + 8 + 7 * 8 + 8 + 8
    assert sp.TRIGGER_DTYPE.itemsize == 40 and sp.RESULT_DTYPE.itemsize == 16 and sp.XI2_DTYPE.itemsize == 24
    assert sp.RANK_DTYPE.itemsize == 16 and C.sizeof(sp.spiir_rank_bins) == 24


def test_workspace_query_and_bad_arguments(sp):
    bank = workloads.bank_for_config(0)
    d, keep = sp.make_desc(bank, 2, 2048, 2048)
    n = C.c_size_t(0)
    assert sp.spiir_bank_workspace_bytes(C.byref(d), C.byref(n)) == sp.SPIIR_OK and n.value > 0
    # each of these must be refused with EINVAL and a message
    def bad(mut):
        d2, k2 = sp.make_desc(bank, 2, 2048, 2048)
        mut(d2)
        rc = sp.spiir_bank_workspace_bytes(C.byref(d2), C.byref(n))
        assert rc == sp.SPIIR_EINVAL and sp.last_error()
    bad(lambda d: setattr(d, "n_det", 0))
    bad(lambda d: setattr(d, "n_det", 5))
    bad(lambda d: setattr(d, "n_bands", 9))
    bad(lambda d: setattr(d, "out_band", 1))               # single band: out_band must be 0
    bad(lambda d: setattr(d, "max_chunk_samples", 2050))   # not a multiple of 4
    bad(lambda d: setattr(d, "ring_len", 100))             # shorter than one chunk
    bad(lambda d: setattr(d, "host_a", None))
    bad(lambda d: setattr(d, "bank_size", 0))
    def small_delay(d):
        d.max_delay[0] = 5                                  # filters with larger delays exist
    bad(small_delay)
    def negative_band(d):
        band = np.array(bank["band"], dtype=np.int32).copy()
        band[3] = -1
        negative_band.keep = band                            # the descriptor holds a bare pointer
        d.host_band = band.ctypes.data
    bad(negative_band)
    assert sp.spiir_bank_workspace_bytes(None, C.byref(n)) == sp.SPIIR_EINVAL
    # band rates must halve
    bank8 = workloads.random_bank(np.random.default_rng(0), 2, 16, [4096, 2048, 1000], out_band=1)
    dec, itp = workloads.halfband_taps()
    d3, k3 = sp.make_desc(bank8, 2, 4096, 2048, dec_taps=dec, int_taps=itp)
    assert sp.spiir_bank_workspace_bytes(C.byref(d3), C.byref(n)) == sp.SPIIR_EINVAL


def test_null_handles_are_refused(sp):
    assert sp.spiir_bank_reset(None, None) == sp.SPIIR_EINVAL
    assert sp.spiir_bank_free(None) == sp.SPIIR_EINVAL
    assert sp.spiir_filter_chunk(None, None, 2048, None, None) == sp.SPIIR_EINVAL
    assert sp.spiir_peaks(None, C.c_float(4.0), 0, None, None, None) == sp.SPIIR_EINVAL
    assert sp.coherent_sky_search(None, None, None, 1, None, None, None) == sp.SPIIR_EINVAL
    assert sp.timeslide_background(None, None, None, 1, 1, 2048, None, None, None) == sp.SPIIR_EINVAL
    n = C.c_size_t(0)
    assert sp.spiir_sky_plan_workspace_bytes(1, 192, 8, C.byref(n)) == sp.SPIIR_EINVAL
    assert sp.spiir_sky_plan_workspace_bytes(3, 3072, 1536, C.byref(n)) == sp.SPIIR_OK and n.value > 3072 * 32


def test_host_table_builder_matches_the_oracle_table(sp):
    """spiir_sky_table_build (own closed-form SVD) vs oracle/sky.py (numpy SVD): delays
    exactly, projectors U2 U2^T to float32 rounding (A20: only the projector is unique)."""
    import oracle
    for dets, sigma, nside in ((["H1", "L1", "V1"], [1.0, 1.0, 0.5], 16), (["H1", "L1"], [1.0, 1.0], 4),
                               (["H1", "L1", "V1"], [1.0, 1.0, 0.5], 1)):
        pos, resp = workloads.detector_geometry(dets)
        u2, dl = sp.sky_table_build(nside, pos, resp, sigma, 1.2345, 2048.0)
        U2o, dlo = oracle.sky_table(nside, pos, resp, sigma, 1.2345, 2048.0)
        assert np.array_equal(dl, dlo)
        P = np.einsum("pik,pjk->pij", u2.astype(float), u2.astype(float))
        Po = np.einsum("pik,pjk->pij", U2o, U2o)
        assert np.abs(P - Po).max() < 1e-6


def test_table_set_and_nearest_selection_match_the_oracle(sp):
    """spiir_sky_table_set_build / spiir_sky_table_nearest (NEXT-3) vs oracle.table_set /
    oracle.nearest_table: delays exactly, projectors to float32 rounding, indices exactly."""
    import oracle
    pos, resp = workloads.detector_geometry(["H1", "L1", "V1"])
    sigma = [1.0, 0.9, 0.4]
    u2, dl = sp.sky_table_set_build(8, pos, resp, sigma, 2.5, 1800.0, 48, 2048.0)
    U2o, dlo = oracle.table_set(8, pos, resp, sigma, 2.5, 1800.0, 48, 2048.0)
    assert u2.shape == (48, 768, 3, 2) and np.array_equal(dl, dlo)
    P = np.einsum("spik,spjk->spij", u2.astype(float), u2.astype(float))
    Po = np.einsum("spik,spjk->spij", U2o, U2o)
    assert np.abs(P - Po).max() < 1e-6
    assert not np.array_equal(dl[0], dl[1])                      # half an hour does move the offsets
    rng = np.random.default_rng(8)
    t0 = 1.26e9
    ts = np.concatenate([t0 + rng.uniform(-2000, 48 * 1800 + 2000, 4000),
                         t0 + 1800.0 * np.arange(-1, 49) + 900.0,          # every midpoint (ties)
                         t0 + 1800.0 * np.arange(-1, 49), [t0 - 1e15, t0 + 1e15]])
    for t in ts:
        assert sp.sky_table_nearest(t, t0, 1800.0, 48) == oracle.nearest_table(t, t0, 1800.0, 48), t
    for n, dt in ((1, 10.0), (7, 0.3), (48, 1795.0)):
        for t in rng.uniform(-3 * dt, (n + 2) * dt, 500):
            assert sp.sky_table_nearest(t, 0.0, dt, n) == oracle.nearest_table(t, 0.0, dt, n)
    idx = C.c_int32(0)
    assert sp.lib().spiir_sky_table_nearest(0.0, 0.0, -1.0, 4, C.byref(idx)) != sp.SPIIR_OK
    assert sp.lib().spiir_sky_table_nearest(float("nan"), 0.0, 1.0, 4, C.byref(idx)) != sp.SPIIR_OK


def test_upsample_window_sizing_and_argument_checks(sp):
    """spiir_snr_upsample_elems (host only): [n_det][n_slots][2 R H + 1 padded to even] complex elements."""
    n = C.c_size_t(0)
    for D, S, R, H in ((3, 10, 4, 58), (2, 0, 1, 1), (4, 7, 16, 5), (1, 3, 3, 2)):
        assert sp.lib().spiir_snr_upsample_elems(D, S, R, H, C.byref(n)) == sp.SPIIR_OK
        Lw = 2 * R * H + 1
        assert n.value == D * S * (Lw + (Lw & 1))
    for D, S, R, H in ((0, 1, 2, 2), (5, 1, 2, 2), (3, -1, 2, 2), (3, 1, 0, 2), (3, 1, 17, 2), (3, 1, 2, 0)):
        assert sp.lib().spiir_snr_upsample_elems(D, S, R, H, C.byref(n)) == sp.SPIIR_EINVAL
    assert sp.lib().spiir_snr_upsample_elems(3, 1, 2, 2, None) == sp.SPIIR_EINVAL
    # NULL view / buffers are refused before any device work
    assert sp.lib().spiir_snr_upsample_windows(None, 3, None, 1, 2, 2, None, None, None, None) == sp.SPIIR_EINVAL


def test_bad_views_and_slide_arguments_are_refused_before_any_device_work(sp):
    """spiir_snr_view has no size field: a caller that leaves n_rows unset passes 0 or stack garbage.  Every entry
    point that takes a view refuses n_rows outside 1..2^31-1, a NULL dev_z, ring_len < 1 and negative strides; slide
    shifts that would overflow int64 are refused too.  The device pointers below are never dereferenced: the checks
    come first (coherent_sky_search / timeslide_background need a plan, hence a device: their arm is in the -m gpu
    test_sky_degenerate_inputs)."""
    L = sp.lib()
    fake = C.c_void_p(4096)                                                  # stands for device memory; not touched
    mult = (C.c_int32 * 3)(1, 1, 1)
    ov = sp.spiir_snr_view()

    def xi2(view, n_slides=0, step=0, m=mult):
        return L.spiir_signal_consistency(C.byref(view), 3, 768, fake, fake, fake, 4, n_slides, step, m, fake, 10, fake, None)

    def ups(view, n_slides=1, step=10, m=mult):
        return L.spiir_snr_upsample_windows_slides(C.byref(view), 3, fake, 4, n_slides, step, m, 2, 30, fake, fake,
                                                   C.byref(ov), None)

    def ups_fg(view):
        return L.spiir_snr_upsample_windows(C.byref(view), 3, fake, 4, 2, 30, fake, fake, C.byref(ov), None)

    good = dict(dev_z=4096, det_stride=1000, row_stride=100, ring_len=100, k_newest=99, n_rows=10)
    for bad in (dict(n_rows=0), dict(n_rows=-3), dict(n_rows=1 << 31), dict(n_rows=0x7F7F7F7F7F7F7F7F), dict(dev_z=None),
                dict(ring_len=0), dict(det_stride=-1), dict(row_stride=-100)):
        v = sp.spiir_snr_view(**{**good, **bad})
        for call in (xi2, ups, ups_fg):
            assert call(v) == sp.SPIIR_EINVAL, (bad, call.__name__)
            assert "view" in sp.last_error(), sp.last_error()
    v = sp.spiir_snr_view(**good)
    huge = (C.c_int32 * 3)(1, -(1 << 31), 1)
    for call in (xi2, ups):
        assert call(v, 100, 1 << 39, mult) == sp.SPIIR_EINVAL and "2^40" in sp.last_error()
        assert call(v, 100, 1 << 20, huge) == sp.SPIIR_EINVAL and "2^40" in sp.last_error()
        assert call(v, 1, 10, None) == sp.SPIIR_EINVAL
        assert call(v, 1, -1, mult) == sp.SPIIR_EINVAL
        assert call(v, -1, 10, mult) == sp.SPIIR_EINVAL


def test_early_warning_bank_shape_and_host_planning(sp):
    """workloads.early_warning_bank: only bands of <= 256 Hz keep filters, each filter below its
    template's seeded cut-off, CSR consistent, the input bank untouched; the library's host-side planner accepts a
    descriptor whose upper four bands are empty (no device needed for the workspace query)."""
    rng = np.random.default_rng(7)
    full = workloads.random_bank(rng, 30, 240, workloads.configs.RATES8, out_band=1, exact_norm=False)
    before = {k: np.array(full[k]).copy() for k in ("a", "b", "delay", "band", "tmpl_offset")}
    ew = workloads.early_warning_bank(full, rng, exact_norm=False)
    for k, v in before.items():
        assert np.array_equal(np.array(full[k]), v)
    off = ew["tmpl_offset"]
    assert off[0] == 0 and off[-1] == len(ew["a"]) == len(ew["b"]) == len(ew["delay"]) == len(ew["band"])
    rates = np.array(ew["band_rates"], float)
    assert ew["band"].min() >= 4 and rates[ew["band"]].max() <= 256
    f = np.abs(np.angle(ew["a"].astype(np.complex128))) * rates[ew["band"]] / (2 * np.pi)
    t_of = np.repeat(np.arange(30), np.diff(off))
    assert np.all(f <= ew["f_cut"][t_of] + 1e-9) and np.all((ew["f_cut"] >= 30) & (ew["f_cut"] <= 60))
    assert np.all(np.diff(ew["band"].astype(int))[np.diff(t_of) == 0] >= 0)           # still sorted by band inside a template
    # every dropped filter is in a band above 256 Hz or above the cut-off: nothing else went missing
    fa = np.abs(np.angle(full["a"].astype(np.complex128))) * rates[full["band"]] / (2 * np.pi)
    want = (rates[full["band"]] <= 256) & (fa <= np.repeat(ew["f_cut"], 240))
    assert want.sum() == len(ew["a"]) and np.array_equal(full["a"][want], ew["a"])
    dec, itp = workloads.halfband_taps()
    d, keep = sp.make_desc(ew, 3, 4096, 4096, 1000, dec, itp)
    n = C.c_size_t(0)
    assert sp.spiir_bank_workspace_bytes(C.byref(d), C.byref(n)) == sp.SPIIR_OK, sp.last_error()
    assert n.value > 0


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2011_06787_b200")
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                txt = open(os.path.join(dp, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "libspiir_oracle" not in txt and "spiir_oracle" not in txt, f


def test_host_autocorrelation_matches_the_oracle(sp):
    """spiir_template_autocorr (library, float64 host helper) against the oracle's own autocorrelation of the
    same templates, and its refusal of unstable filters."""
    import oracle
    bank = workloads.bank_for_config(0)
    for t in range(bank["n_templates"]):
        A = sp.template_autocorr(bank, t, 60)
        ref = oracle.template_autocorr(bank, t, 60)
        assert abs(A[60] - 1) < 1e-6 and np.abs(A - ref).max() < 5e-7
    a = np.array([1.0 + 0j], np.complex64); b = np.array([1.0 + 0j], np.complex64); d = np.zeros(1, np.int32)
    out = np.zeros(3, np.complex64)
    rc = sp.spiir_template_autocorr(1, a.ctypes.data, b.ctypes.data, d.ctypes.data, 1, out.ctypes.data)
    assert rc == sp.SPIIR_EINVAL and sp.last_error()
