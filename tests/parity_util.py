"""Shared helpers of the -m gpu parity tests (CUDA path through the C ABI vs oracle/).

Tolerances (BASELINE.json north_star / DESIGN.md §7):
  * |z_gpu - z_oracle| <= 1e-3 absolute on unit-noise-normalised SNR;
  * sample / trigger indices exact, with the set-valued near-tie rule A12;
  * coh2 within 1e-4 relative (1e-3 absolute on rho_c); null2 within 1e-4*tot2 + 1e-5 (A25);
  * pixel by the set-valued rule A19.
"""
import numpy as np
import torch

import oracle
import paper_2011_06787_b200 as sp

TOL_SNR = 1e-3
TOL_COH2_REL = 1e-4


def run_bank(bank, strain, chunk, n_det=None, ring_len=None, bank_size=1000, taps=(None, None),
             peak_thr=None, peak_mode=0, chunks=None):
    """Streams `strain` [n_det][n0] through spiir_filter_chunk in chunks; returns
    (z complex64 [n_det][T][n_out], list of per-chunk trigger arrays, Bank)."""
    strain = np.ascontiguousarray(strain, dtype=np.float32)
    D, n0 = strain.shape
    ob = int(bank["out_band"])
    T = int(bank["n_templates"])
    sizes = chunks if chunks is not None else [chunk] * (n0 // chunk)
    assert sum(sizes) == n0
    bk = sp.Bank(bank, D, max(sizes), ring_len=ring_len, bank_size=bank_size, dec_taps=taps[0], int_taps=taps[1])
    xs = torch.from_numpy(strain).cuda()
    z = np.zeros((D, T, n0 >> ob), np.complex64)
    trigs = []
    pos = 0
    for n in sizes:
        x = xs[:, pos:pos + n].contiguous()
        out = torch.empty(D, T, n >> ob, 2, dtype=torch.float32, device="cuda")
        bk.filter_chunk(x, out)
        if peak_thr is not None:
            tr, cnt = bk.peaks(peak_thr, peak_mode)
            trigs.append((sp.triggers_to_numpy(tr).copy(), int(cnt.cpu()[0])))
        torch.cuda.synchronize()
        z[:, :, pos >> ob:(pos + n) >> ob] = out.cpu().numpy().view(np.complex64)[..., 0]
        pos += n
    return z, trigs, bk


def check_snr(z_gpu, z_ref, tol=TOL_SNR):
    err = np.abs(z_gpu.astype(np.complex128) - z_ref)
    assert err.max() <= tol, "max |z_gpu - z_oracle| = %.3e > %.1e" % (err.max(), tol)
    return float(err.max())


def check_peaks_mode0(trig, z_gpu_chunk, z_ref_chunk, k0, thr, tol=TOL_SNR):
    """trig: TRIGGER_DTYPE [D*T] of one chunk; z_*_chunk [D][T][n].
    (i) stage-isolated: the oracle's O4 on the GPU's own float32 z must give the GPU's indices exactly;
    (ii) end-to-end: where the float64 oracle's arg-max differs, its |z| at the GPU's index must be
    within 2*tol of its maximum (near-tie rule A12).  Returns the number of rule-(ii) cases."""
    D, T, n = z_gpu_chunk.shape
    k_iso, v_iso = oracle.peaks_mode0(z_gpu_chunk.reshape(D * T, n), thr)
    assert np.array_equal(trig["k"] - k0, k_iso), "peak indices differ from O4 on the GPU's own z"
    assert np.array_equal(trig["valid"], v_iso)
    assert np.array_equal(trig["tmpl"], np.tile(np.arange(T), D))
    assert np.array_equal(trig["det"], np.repeat(np.arange(D), T))
    zz = z_gpu_chunk.reshape(D * T, n)[np.arange(D * T), k_iso]
    assert np.array_equal(trig["z_re"], zz.real) and np.array_equal(trig["z_im"], zz.imag)
    np.testing.assert_allclose(trig["snr"], np.abs(zz), rtol=1e-6)
    k_ref, v_ref = oracle.peaks_mode0(z_ref_chunk.reshape(D * T, n), thr)
    zr = np.abs(z_ref_chunk.reshape(D * T, n))
    diff = np.nonzero(k_ref != k_iso)[0]
    for i in diff:
        assert zr[i, k_ref[i]] - zr[i, k_iso[i]] <= 2 * tol, "trigger index differs beyond the near-tie rule"
    # validity may only differ when the maximum sits within tol of the threshold
    for i in np.nonzero(v_ref != v_iso)[0]:
        assert abs(zr[i, k_ref[i]] - thr) <= 2 * tol
    return len(diff)


def oracle_sky_on(view_z, ring_len, k_newest, u2, delay, trig, n_slides=0, step=0, mult=None, want_map=False):
    """Oracle O6/O7 on a float32 SNR array [D][rows][ring_len] (complex64) and a trigger array."""
    D, rows, L = view_z.shape
    return oracle.sky_search(u2, delay, view_z, rows * L, L, ring_len, k_newest,
                             trig["valid"], trig["tmpl"], trig["det"], trig["k"],
                             n_slides=n_slides, step=step, slide_mult=mult, want_map=want_map)


def check_sky(res_gpu, view_z, ring_len, k_newest, u2, delay, trig, n_slides=0, step=0, mult=None,
              ref=None):
    """res_gpu: RESULT_DTYPE [n_trig*S].  Set-valued pixel rule A19; values compared with the oracle
    at the GPU's own pixel and maxima compared with each other.  Returns statistics."""
    S = max(1, n_slides)
    n_trig = len(trig)
    if ref is None:
        ref = oracle_sky_on(view_z, ring_len, k_newest, u2, delay, trig, n_slides, step, mult)
    out, pix, _ = ref
    g = res_gpu.reshape(n_trig, S)
    D, rows, L = view_z.shape
    gp = g["pix"].astype(np.int64)
    gc, gt, gn = g["coh2"].astype(np.float64), g["tot2"].astype(np.float64), g["null2"].astype(np.float64)
    none = pix < 0
    assert np.all(gp[none] == -1) and np.all(gc[none] == 0) and np.all(gt[none] == 0) and np.all(gn[none] == 0)
    has = ~none
    bad = has & (gp < 0)
    assert not bad.any(), "GPU reports no result where the oracle has one (trigger, slide) %s" % (np.argwhere(bad)[:4].tolist(),)
    cmax = out[..., 0]
    tol = np.maximum(TOL_COH2_REL * cmax, 1e-6)
    err = np.abs(gc - cmax)
    assert np.all(err[has] <= tol[has]), "coh2 differs: worst %s" % (np.argwhere(has & (err > tol))[:4].tolist(),)
    assert np.all(np.abs(np.sqrt(gc[has]) - np.sqrt(cmax[has])) <= 1e-3)
    # at the oracle's own pixel the three values compare directly; elsewhere the GPU's pixel must be a valid
    # arg-max (A19) and the values are compared with the oracle evaluated AT THAT PIXEL
    c_at, tot_at = cmax.copy(), out[..., 2].copy()
    differs = np.argwhere(has & (gp != pix))
    for i, s in differs:
        ok, c, nul, tot = oracle.sky_eval(u2, delay, view_z, rows * L, L, ring_len, k_newest,
                                          int(trig["tmpl"][i]), int(trig["det"][i]), int(trig["k"][i]), int(gp[i, s]),
                                          s=(s + 1 if n_slides else 0), step=step, slide_mult=mult)
        assert ok
        assert c >= cmax[i, s] - max(1e-4 * cmax[i, s], 1e-3), "GPU pixel is not a valid arg-max (A19)"
        c_at[i, s], tot_at[i, s] = c, tot
    assert np.all(np.abs(gt - tot_at)[has] <= (1e-5 * tot_at + 1e-6)[has])
    assert np.all(np.abs(gn - np.maximum(tot_at - c_at, 0.0))[has] <= (1e-4 * tot_at + 1e-5)[has])
    rel = np.where(has, err / np.maximum(cmax, 1e-30), 0.0)
    return dict(pix_differs=int(len(differs)), n=int(has.sum()), max_rel_err_coh2=float(rel.max()) if has.any() else 0.0)
