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
    n_pixdiff = 0
    for i in range(n_trig):
        for s in range(S):
            gp = int(g["pix"][i, s])
            if pix[i, s] < 0:
                assert gp == -1 and g["coh2"][i, s] == 0 and g["tot2"][i, s] == 0 and g["null2"][i, s] == 0
                continue
            assert gp >= 0, "GPU reports no result where the oracle has one (trigger %d slide %d)" % (i, s)
            cmax = out[i, s, 0]
            tol = max(TOL_COH2_REL * cmax, 1e-6)
            assert abs(g["coh2"][i, s] - cmax) <= tol, (i, s, g["coh2"][i, s], cmax)
            assert abs(np.sqrt(g["coh2"][i, s]) - np.sqrt(cmax)) <= 1e-3
            if gp != pix[i, s]:
                n_pixdiff += 1
                ok, c, nul, tot = oracle.sky_eval(u2, delay, view_z, rows * L, L, ring_len, k_newest,
                                                  int(trig["tmpl"][i]), int(trig["det"][i]), int(trig["k"][i]), gp,
                                                  s=(s + 1 if n_slides else 0), step=step, slide_mult=mult)
                assert ok
                assert c >= cmax - max(1e-4 * cmax, 1e-3), "GPU pixel is not a valid arg-max (A19)"
            else:
                c, tot = cmax, out[i, s, 2]
            assert abs(g["tot2"][i, s] - tot) <= 1e-5 * tot + 1e-6
            assert abs(g["null2"][i, s] - max(tot - c, 0.0)) <= 1e-4 * tot + 1e-5
    return dict(pix_differs=n_pixdiff)
