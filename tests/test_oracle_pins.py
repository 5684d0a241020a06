"""Pins for the float64 oracle (no GPU): closed forms, brute force, library
routines, invariants and the values the paper prints.  P-numbers refer to
SURVEY.md §8(c) / DESIGN.md "What pins each part of the oracle".
A plausible mistake anywhere in oracle/ (dropped term, wrong sign or index,
transposed operand) must fail at least one of these.
"""
import math
import os

import numpy as np
import pytest
import scipy.signal

import oracle
import workloads

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden():
    out = {}
    for line in open(os.path.join(HERE, "golden", "paper_values.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            out[line[0]] = float(line[1])
    return out


def _rand_filters(rng, n, dmax=40, tau=(3.0, 60.0)):
    t = rng.uniform(*tau, size=n)
    w = rng.uniform(0.01, 1.5, size=n)
    a = np.exp(-1.0 / t + 1j * w).astype(np.complex64)
    b = ((rng.standard_normal(n) + 1j * rng.standard_normal(n)) / math.sqrt(2)).astype(np.complex64)
    d = rng.integers(0, dmax + 1, size=n).astype(np.int32)
    return a, b, d


# ---- P1: single-filter impulse response is b a^(k-d) after the delay --------
def test_p1_impulse_response_closed_form():
    a = np.array([np.exp(-1 / 50.0 + 0.3j)], np.complex64)
    b = np.array([0.7 - 0.2j], np.complex64)
    d = np.array([17], np.int32)
    x = np.zeros(400)
    x[0] = 1.0
    y = oracle.band_sum(x, a, b, d)
    k = np.arange(400)
    a64, b64 = complex(a[0]), complex(b[0])
    want = np.where(k >= 17, b64 * a64 ** np.maximum(k - 17, 0), 0.0)
    assert np.all(y[:17] == 0)
    np.testing.assert_allclose(y, want, rtol=0, atol=1e-13)


# ---- P2: tiny bank == direct convolution with truncated impulse responses ---
def test_p2_bank_equals_direct_convolution():
    rng = np.random.default_rng(2)
    n = 300
    x = rng.standard_normal(n)
    for nf in (1, 3, 5):
        a, b, d = _rand_filters(rng, nf)
        s = oracle.band_sum(x, a, b, d)
        h = np.zeros(n, complex)
        for l in range(nf):
            kk = np.arange(n - d[l])
            h[d[l]:] += complex(b[l]) * complex(a[l]) ** kk
        want = np.array([np.sum(h[:m + 1][::-1] * x[:m + 1]) for m in range(n)])
        np.testing.assert_allclose(s, want, rtol=0, atol=1e-11)


# ---- the recursion reduces to scipy.signal.lfilter (library routine) --------
def test_recursion_equals_scipy_lfilter():
    rng = np.random.default_rng(3)
    x = rng.standard_normal(500)
    a, b, d = _rand_filters(rng, 4)
    want = np.zeros(500, complex)
    for l in range(4):
        xd = np.concatenate([np.zeros(d[l]), x])[:500]
        want += scipy.signal.lfilter([complex(b[l])], [1.0, -complex(a[l])], xd)
    np.testing.assert_allclose(oracle.band_sum(x, a, b, d), want, rtol=0, atol=1e-11)


# ---- P3: closed-form noise variance used by the generator -------------------
def test_p3_noise_variance_closed_form_and_normalisation():
    from workloads.gen import _noise_variance
    rng = np.random.default_rng(4)
    a, b, d = _rand_filters(rng, 6, dmax=30, tau=(3.0, 25.0))
    n = 4000
    h = np.zeros(n, complex)
    for l in range(6):
        h[d[l]:] += complex(b[l]) * complex(a[l]) ** np.arange(n - d[l])
    V = _noise_variance(a.astype(complex)[None], b.astype(complex)[None], d[None])[0]
    assert abs(V - np.sum(np.abs(h) ** 2)) < 1e-9 * V
    # generated banks are scaled to E|z|^2 = 2 (A8): measure it through the oracle
    bank = workloads.random_bank(np.random.default_rng(5), 6, 24, [2048], tau_range=(5.0, 60.0), max_delay=100)
    x = np.random.default_rng(6).standard_normal((1, 60000)).astype(np.float32)
    z = oracle.filter_bank(x, bank)[0]
    m = np.mean(np.abs(z[:, 2000:]) ** 2)
    assert abs(m - 2.0) < 0.12


# ---- P4: linearity and shift invariance -------------------------------------
def test_p4_linearity_and_shift():
    rng = np.random.default_rng(7)
    a, b, d = _rand_filters(rng, 5)
    x1, x2 = rng.standard_normal(256), rng.standard_normal(256)
    z1, z2 = oracle.band_sum(x1, a, b, d), oracle.band_sum(x2, a, b, d)
    z12 = oracle.band_sum(2.5 * x1 - 0.75 * x2, a, b, d)
    np.testing.assert_allclose(z12, 2.5 * z1 - 0.75 * z2, atol=1e-12)
    xs = np.concatenate([np.zeros(13), x1])[:256]
    zs = oracle.band_sum(xs, a, b, d)
    np.testing.assert_allclose(zs[13:], z1[:-13], atol=1e-13)
    assert np.all(zs[:13] == 0)


# ---- P5: decimator / interpolator reduce to scipy routines ------------------
def test_p5_decimator_is_lfilter_odd_phase():
    dec, itp = workloads.halfband_taps()
    rng = np.random.default_rng(8)
    x = rng.standard_normal(1024)
    y = oracle.decimate(x, dec.astype(np.float64))
    want = scipy.signal.lfilter(dec.astype(np.float64), 1.0, x)[1::2]
    np.testing.assert_allclose(y, want, atol=1e-13)
    assert abs(np.sum(dec.astype(np.float64) ** 2) - 1.0) < 1e-6      # M2 noise gain
    assert abs(np.sum(itp.astype(np.float64)) - 2.0) < 1e-6           # M4 DC gain after zero-stuffing


def test_p5_interpolator_is_upfirdn():
    dec, itp = workloads.halfband_taps()
    rng = np.random.default_rng(9)
    acc = rng.standard_normal(200) + 1j * rng.standard_normal(200)
    s = rng.standard_normal(400) + 1j * rng.standard_normal(400)
    got = oracle.interp_add(acc, itp.astype(np.float64), s)
    want = scipy.signal.upfirdn(itp.astype(np.float64), acc, up=2)[:400] + s
    np.testing.assert_allclose(got, want, atol=1e-12)
    got0 = oracle.interp_add(acc, itp.astype(np.float64), None)
    np.testing.assert_allclose(got0, want - s, atol=1e-12)


def _small_multirate_bank(rng, T=3, L=8, rates=(4096, 2048, 1024, 512), out_band=1):
    return workloads.random_bank(rng, T, L, list(rates), out_band, tau_range=(4.0, 40.0), max_delay=30)


# ---- multirate composition written out with scipy (M1-M5 restated) ----------
def test_multirate_bank_equals_scipy_composition():
    rng = np.random.default_rng(10)
    dec, itp = workloads.halfband_taps()
    bank = _small_multirate_bank(rng)
    x = rng.standard_normal((1, 2048)).astype(np.float32)
    z = oracle.filter_bank(x, bank, dec, itp)[0]
    g, h = dec.astype(np.float64), itp.astype(np.float64)
    xb = [x[0].astype(np.float64)]
    for _ in range(3):
        xb.append(scipy.signal.lfilter(g, 1.0, xb[-1])[1::2])
    for t in range(3):
        sl = slice(bank["tmpl_offset"][t], bank["tmpl_offset"][t + 1])
        a, b, d, bd = bank["a"][sl], bank["b"][sl], bank["delay"][sl], bank["band"][sl]
        s = []
        for bnd in range(4):
            m = bd == bnd
            sb = np.zeros(len(xb[bnd]), complex)
            for l in np.nonzero(m)[0]:
                xd = np.concatenate([np.zeros(d[l]), xb[bnd]])[:len(xb[bnd])]
                sb += scipy.signal.lfilter([complex(b[l])], [1.0, -complex(a[l])], xd)
            s.append(sb)
        acc = s[3]
        for bnd in (2, 1):
            acc = s[bnd] + scipy.signal.upfirdn(h, acc, up=2)[:len(s[bnd])]
        want = acc + s[0][1::2]
        np.testing.assert_allclose(z[t], want, atol=1e-10)


# ---- P6: periodic shift invariance of the multirate path --------------------
def test_p6_multirate_periodic_shift_invariance():
    rng = np.random.default_rng(11)
    dec, itp = workloads.halfband_taps()
    bank = _small_multirate_bank(rng)            # B = 4 -> period 2^(B-1) = 8 top-rate samples
    x = rng.standard_normal(1024).astype(np.float32)
    q = 3
    xs = np.concatenate([np.zeros(8 * q, np.float32), x])[:1024]
    z = oracle.filter_bank(x[None], bank, dec, itp)[0]
    zs = oracle.filter_bank(xs[None], bank, dec, itp)[0]
    sh = 4 * q                                   # output is at half the input rate
    np.testing.assert_allclose(zs[:, sh:], z[:, :-sh], atol=1e-12)
    assert np.all(zs[:, :sh] == 0)


# ---- P8: B = 1 multirate plumbing == plain single-rate sum ------------------
def test_p8_single_band_path_is_plain_sum():
    rng = np.random.default_rng(12)
    bank = workloads.random_bank(rng, 3, 7, [2048], 0, tau_range=(4.0, 40.0), max_delay=30)
    x = rng.standard_normal((2, 512)).astype(np.float32)
    z = oracle.filter_bank(x, bank)
    for D in range(2):
        for t in range(3):
            sl = slice(bank["tmpl_offset"][t], bank["tmpl_offset"][t + 1])
            s = oracle.band_sum(x[D].astype(np.float64), bank["a"][sl], bank["b"][sl], bank["delay"][sl])
            assert np.array_equal(z[D, t], s)
    # a template subset is the same numbers as the full run (templates are independent)
    zs = oracle.filter_bank(x, bank, templates=[2, 0])
    assert np.array_equal(zs[:, 0], z[:, 2]) and np.array_equal(zs[:, 1], z[:, 0])


# ---- P9: peak finder against brute force, with planted exact ties -----------
@pytest.mark.parametrize("dtype", [np.complex128, np.complex64])
def test_p9_peaks_mode0_bruteforce_with_ties(dtype):
    rng = np.random.default_rng(13)
    z = (rng.standard_normal((9, 300)) + 1j * rng.standard_normal((9, 300))).astype(dtype)
    z[2, 250] = z[2, 40] = 9.0 + 0j              # exact tie -> lowest index wins
    z[5] *= 0.01                                 # below threshold
    k, v = oracle.peaks_mode0(z, 1.0)
    m2 = (z.real.astype(dtype(0).real.dtype) ** 2 + z.imag.astype(dtype(0).real.dtype) ** 2)
    for r in range(9):
        assert k[r] == int(np.argmax(m2[r]))     # numpy argmax returns the first maximum
        assert v[r] == int(m2[r].max() > 1.0)
    assert k[2] == 40 and v[5] == 0


def test_p9_peaks_mode1_bruteforce_and_guarantees():
    rng = np.random.default_rng(14)
    T, n, bs = 10, 200, 4
    z = (rng.standard_normal((T, n)) + 1j * rng.standard_normal((T, n))) * 1.2
    z[1, 50] = z[3, 50] = 5.0                    # tie across templates at one sample -> lowest t
    z[6, 10] = z[6, 120] = 6.0                   # tie in time within a template -> lowest k
    thr = 2.0
    k, v = oracle.peaks_mode1(z, thr, bs)
    m2 = np.abs(z) ** 2
    for t0 in range(0, T, bs):
        blk = m2[t0:t0 + bs]
        tstar = np.argmax(blk, axis=0)           # first maximum = lowest t
        kept = blk.max(axis=0) > thr * thr
        for t in range(t0, min(T, t0 + bs)):
            cand = [kk for kk in range(n) if kept[kk] and tstar[kk] == t - t0]
            if not cand:
                assert v[t] == 0
                continue
            best = max(cand, key=lambda kk: (m2[t, kk], -kk))
            assert v[t] == 1 and k[t] == best
        # at most one candidate per sample per bank
        ks = [k[t] for t in range(t0, min(T, t0 + bs)) if v[t]]
        assert len(ks) == len(set(ks))
    assert v[1] == 1 and (v[3] == 0 or k[3] != 50)
    assert k[6] == 10


# ---- sky table: P15 -----------------------------------------------------------
def _table(nside, dets, sigma, gmst=1.234):
    pos, resp = workloads.detector_geometry(dets)
    U2, dl = oracle.sky_table(nside, pos, resp, sigma, gmst, 2048.0)
    return pos, resp, U2, dl


def test_p15_healpix_and_table_invariants():
    g = _golden()
    assert 12 * 16 * 16 == g["sky_pixels_foreground"] and 12 * 8 * 8 == g["sky_pixels_background"]
    for ns in (1, 2, 4, 8):
        th, ph = oracle.healpix_ring_centres(ns)
        assert len(th) == 12 * ns * ns
        v = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)], 1)
        assert np.abs(v.sum(0)).max() < 1e-12                      # centres sum to zero
        assert len(np.unique(np.round(np.cos(th), 12))) == 4 * ns - 1   # 4 nside - 1 rings
        assert np.all(np.diff(np.cos(th)) <= 1e-15)                # RING order: north to south
        d = v @ v.T
        np.fill_diagonal(d, -1)
        assert d.max() < 1 - 1e-6                                  # all distinct
    # equal-area pixels: nearest-neighbour spacing ~ sqrt(4 pi / npix); PAPER.md:171 max 1.9 deg at nside 16
    th, ph = oracle.healpix_ring_centres(16)
    v = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)], 1)
    nn = np.degrees(np.arccos(np.clip(np.sort(v @ v.T, axis=1)[:, -2], -1, 1)))
    assert 2.5 < nn.min() and nn.max() < 2 * 2.0 * 1.9
    assert abs((1 - math.cos(math.radians(g["pixel_max_angle_deg"]))) * 100 - g["pixel_max_snr_loss_percent"]) < 0.01
    pos, resp, U2, dl = _table(8, ["H1", "L1", "V1"], [1, 1, 0.5])
    P = U2 @ U2.transpose(0, 2, 1)
    np.testing.assert_allclose(U2.transpose(0, 2, 1) @ U2, np.broadcast_to(np.eye(2), (768, 2, 2)), atol=1e-12)
    np.testing.assert_allclose(P @ P, P, atol=1e-12)
    np.testing.assert_allclose(np.trace(P, axis1=1, axis2=2), 2.0, atol=1e-12)
    for i in range(3):
        for j in range(i + 1, 3):
            lt = np.linalg.norm(pos[i] - pos[j]) / workloads.C_LIGHT
            assert np.abs(dl[:, i] - dl[:, j]).max() <= lt * 2048.0 + 1.0
            assert np.abs(dl[:, i] - dl[:, j]).max() >= lt * 2048.0 * 0.95 - 1.0
    lts = sorted(np.linalg.norm(pos[i] - pos[j]) / workloads.C_LIGHT * 1e3 for i in range(3) for j in range(i + 1, 3))
    np.testing.assert_allclose(lts, [10.01, 26.45, 27.29], atol=0.05)   # known light-travel times (ms)


def test_table_signs_against_plane_wave():
    """A delta-like pulse arriving from direction p0 hits detector I at geocentre
    time + tau_I: the detector CLOSER to the source (larger r.n) is hit earlier,
    so its delay is more negative.  Pins the sign of the delay table."""
    pos, resp, U2, dl = _table(4, ["H1", "L1", "V1"], [1, 1, 1])
    th, ph = oracle.healpix_ring_centres(4)
    lam = ph - 1.234
    n = np.stack([np.sin(th) * np.cos(lam), np.sin(th) * np.sin(lam), np.cos(th)], 1)
    proj = n @ pos.T
    for p in range(0, 192, 7):
        order_geo = np.argsort(-proj[p])
        assert np.all(np.diff(dl[p][order_geo]) >= 0)
    # projector equals the projector onto the column space of G_sigma (pinv form, Eq. 25)
    G, _ = oracle.g_sigma(th, ph, resp, [1, 1, 1], 1.234)
    for p in (0, 50, 191):
        Pg = G[p] @ np.linalg.pinv(G[p])
        np.testing.assert_allclose(U2[p] @ U2[p].T, Pg, atol=1e-10)


def test_antenna_pattern_textbook_special_cases():
    """A detector with arms along x, y at the origin: overhead source (theta=0)
    gives |F+|^2+|Fx|^2 = 1; a source in the detector plane along an arm gives
    1/4; along the bisector gives 0 (textbook interferometer pattern)."""
    resp = np.zeros((1, 3, 3))
    resp[0, 0, 0], resp[0, 1, 1] = 0.5, -0.5
    def power(theta, phi):
        G, _ = oracle.g_sigma(np.array([theta]), np.array([phi]), resp, [1.0], 0.0)
        return float(np.sum(G[0, 0] ** 2))
    assert abs(power(0.0, 0.3) - 1.0) < 1e-12
    assert abs(power(math.pi / 2, 0.0) - 0.25) < 1e-12
    assert abs(power(math.pi / 2, math.pi / 4) - 0.0) < 1e-12
    # 1/4 (1+cos^2)^2 cos^2(2phi) + cos^2 sin^2(2phi)
    th, ph = 0.7, 0.4
    want = 0.25 * (1 + math.cos(th) ** 2) ** 2 * math.cos(2 * ph) ** 2 + math.cos(th) ** 2 * math.sin(2 * ph) ** 2
    assert abs(power(th, ph) - want) < 1e-12


def _dense_view(z):
    """z complex [D][R][n] -> view args for a linear (non-wrapping) buffer."""
    D, R, n = z.shape
    return dict(det_stride=R * n, row_stride=n, ring_len=n, k_newest=n - 1)


# ---- P10 / P11 / P12 / P13: coherent statistic --------------------------------
def test_p10_p11_identity_and_two_detector_case():
    rng = np.random.default_rng(20)
    pos, resp, U2, dl = _table(4, ["H1", "L1"], [1, 1])
    z = rng.standard_normal((2, 3, 400)) + 1j * rng.standard_normal((2, 3, 400))
    k = np.array([200, 150, 300])
    res, pix, mp = oracle.sky_search(U2.astype(np.float32), dl, z, trig_valid=[1, 1, 1], trig_row=[0, 1, 2],
                                     trig_det=[0, 1, 0], trig_k=k, want_map=True, **_dense_view(z))
    for i, (T, r) in enumerate(zip([0, 1, 0], [0, 1, 2])):
        O = 1 - T
        for p in range(192):
            tot = abs(z[T, r, k[i]]) ** 2 + abs(z[O, r, k[i] + dl[p, O] - dl[p, T]]) ** 2
            assert abs(mp[i, p] - tot) < 1e-6 * tot          # N_d = 2: coh2 = sum |z|^2 (fp32 U2 rounding)
    # fp32-rounded U2 is orthonormal to ~1e-7 only, so coh2 may exceed tot2 by that much (null clamps at 0)
    np.testing.assert_allclose(res[:, 0, 0] + res[:, 0, 1], res[:, 0, 2], rtol=1e-6)
    assert np.all(res[:, 0, 1] < 1e-5 * res[:, 0, 2])


def test_p10_identity_three_detectors_and_manual_formula():
    rng = np.random.default_rng(21)
    pos, resp, U2, dl = _table(4, ["H1", "L1", "V1"], [1, 1, 0.5])
    u2 = U2.astype(np.float32)
    z = rng.standard_normal((3, 2, 600)) + 1j * rng.standard_normal((3, 2, 600))
    v = _dense_view(z)
    for (row, T, k) in [(0, 1, 300), (1, 2, 222)]:
        for p in (0, 17, 100, 191):
            ok, coh2, null2, tot2 = oracle.sky_eval(u2, dl, z, row=row, det=T, k=k, p=p, **v)
            vec = np.array([z[I, row, k + dl[p, I] - dl[p, T]] for I in range(3)])
            c = u2[p].astype(np.float64).T @ vec
            assert ok and abs(coh2 - np.sum(np.abs(c) ** 2)) < 1e-12
            assert abs(tot2 - np.sum(np.abs(vec) ** 2)) < 1e-12 and abs(coh2 + null2 - tot2) < 1e-12
            assert coh2 <= tot2 * (1 + 1e-6)


def test_p12_noise_expectations_four_and_two_dof():
    g = _golden()
    rng = np.random.default_rng(22)
    pos, resp, U2, dl = _table(2, ["H1", "L1", "V1"], [1, 1, 0.5])
    n = 120000
    z = rng.standard_normal((3, 1, n)) + 1j * rng.standard_normal((3, 1, n))     # unit variance per quadrature
    ks = np.arange(100, n - 100, 3)
    acc_c, acc_n = 0.0, 0.0
    u2 = U2.astype(np.float32)
    v = _dense_view(z)
    for k in ks[:20000]:
        ok, coh2, null2, tot2 = oracle.sky_eval(u2, dl, z, row=0, det=0, k=int(k), p=11, **v)
        acc_c += coh2
        acc_n += null2
    assert abs(acc_c / 20000 - g["coh_dof"]) < 0.08                          # E coh2 = 4
    assert abs(acc_n / 20000 - (2 * 3 - 4)) < 0.06                           # E null2 = 2 N_d - 4


def test_p13_injected_signal_recovers_its_pixel_and_zero_null():
    rng = np.random.default_rng(23)
    pos, resp, U2, dl = _table(8, ["H1", "L1", "V1"], [1, 1, 0.5])
    u2 = U2.astype(np.float32)
    n = 800
    for p0, T in [(5, 0), (300, 1), (700, 2)]:
        z = np.zeros((3, 1, n), complex)
        c = rng.standard_normal(2) + 1j * rng.standard_normal(2)
        amp = u2[p0].astype(np.float64) @ c
        o = np.arange(-20, 21)
        env = np.exp(-o ** 2 / (2 * 6.0 ** 2)) * np.exp(0.6j * o)
        k0 = 400
        for I in range(3):
            z[I, 0, k0 + dl[p0, I] - dl[p0, T] + o] = amp[I] * env
        res, pix, mp = oracle.sky_search(u2, dl, z, trig_valid=[1], trig_row=[0], trig_det=[T], trig_k=[k0],
                                         want_map=True, **_dense_view(z))
        tot = np.sum(np.abs(amp) ** 2)
        assert abs(mp[0, p0] - tot) < 1e-6 * tot                 # all power in the signal plane
        same = [p for p in range(768) if np.array_equal(dl[p] - dl[p, T], dl[p0] - dl[p0, T])]
        assert pix[0, 0] in same                                 # unique up to pixels sharing the delay tuple
        assert res[0, 0, 1] < 1e-5 * tot                         # null = 0 at the true pixel


def test_out_of_range_and_invalid_triggers():
    rng = np.random.default_rng(24)
    pos, resp, U2, dl = _table(2, ["H1", "L1", "V1"], [1, 1, 1])
    z = rng.standard_normal((3, 1, 300)) + 1j * rng.standard_normal((3, 1, 300))
    res, pix, _ = oracle.sky_search(U2.astype(np.float32), dl, z, trig_valid=[1, 1, 0, 1], trig_row=[0] * 4,
                                    trig_det=[0] * 4, trig_k=[10, 295, 150, 150], **_dense_view(z))
    assert list(pix[:, 0][:3]) == [-1, -1, -1] and pix[3, 0] >= 0
    assert np.all(res[:3] == 0)


# ---- P16: time slides ----------------------------------------------------------
def test_p16_time_slides_special_cases():
    rng = np.random.default_rng(25)
    pos, resp, U2, dl = _table(4, ["H1", "L1", "V1"], [1, 1, 0.5])
    u2 = U2.astype(np.float32)
    step, S = 128, 5
    base = rng.standard_normal((3, 2, step)) + 1j * rng.standard_normal((3, 2, step))
    z = np.tile(base, (1, 1, 8))                                 # periodic with period = step
    n = z.shape[2]
    tr = dict(trig_valid=[1, 1], trig_row=[0, 1], trig_det=[0, 2], trig_k=[n - 100, n - 90])
    fg, fpix, _ = oracle.sky_search(u2, dl, z, **tr, **_dense_view(z))
    bg, bpix, _ = oracle.sky_search(u2, dl, z, n_slides=S, step=step, slide_mult=[1, 1, 1], **tr, **_dense_view(z))
    for s in range(S):                                           # periodic ring: every slide == foreground
        np.testing.assert_allclose(bg[:, s], fg[:, 0], rtol=1e-12)
        assert np.array_equal(bpix[:, s], fpix[:, 0])
    z2 = rng.standard_normal((3, 2, n)) + 1j * rng.standard_normal((3, 2, n))
    fg2, fpix2, _ = oracle.sky_search(u2, dl, z2, **tr, **_dense_view(z2))
    bg0, bpix0, _ = oracle.sky_search(u2, dl, z2, n_slides=3, step=step, slide_mult=[0, 0, 0], **tr, **_dense_view(z2))
    for s in range(3):                                           # multipliers 0: slide == foreground
        assert np.array_equal(bg0[:, s], fg2[:, 0]) and np.array_equal(bpix0[:, s], fpix2[:, 0])
    # a genuine slide equals the foreground of a manually shifted copy (companions moved later by s*step)
    bg1, bpix1, _ = oracle.sky_search(u2, dl, z2, n_slides=2, step=step, slide_mult=[1, 1, 1], **tr, **_dense_view(z2))
    for s in (1, 2):
        for i, T in enumerate([0, 2]):
            zz = np.roll(z2, s * step, axis=2)
            zz[T] = z2[T]
            f, fp, _ = oracle.sky_search(u2, dl, zz, trig_valid=[1], trig_row=[i], trig_det=[T],
                                         trig_k=[tr["trig_k"][i]], **_dense_view(zz))
            np.testing.assert_allclose(bg1[i, s - 1], f[0, 0], rtol=1e-12)
            assert bpix1[i, s - 1] == fp[0, 0]


# ---- P17: the paper's printed arithmetic ---------------------------------------
def test_p17_paper_cost_arithmetic():
    g = _golden()
    flops = g["flop_per_filter_sample"] * g["o3_filters_per_template"] * g["o3_templates"] * g["o3_sample_rate"] * g["o3_detectors"]
    assert abs(flops / 1e12 - g["o3_filter_tflops"]) < 0.05
    assert abs(flops / (g["cpu_core_gflops"] * 1e9) - g["o3_cpu_cores"]) < 20
    nd = g["o3_detectors"]
    coh = 4 * nd ** 3 * g["o3_templates"] * (g["sky_pixels_foreground"] + g["n_time_shifts"] * g["sky_pixels_background"])
    assert abs(coh / 1e12 - g["coherent_worst_case_tflops"]) < 0.06
    # Table I: network SNR = quadrature sum of the detector SNRs
    for rl, rh, rv, net in [(13.8, 8.9, 3.8, 16.9), (24.4, 19.4, 3.7, 31.5), (9.9, 4.4, 4.1, 11.6)]:
        assert abs(math.sqrt(rl ** 2 + rh ** 2 + rv ** 2) - net) < 0.15
    # the update counted by the paper: 2 mul + 4 fma + 2 add = 12 flop in 8 instructions
    assert 2 * 1 + 4 * 2 + 2 * 1 == g["flop_per_filter_sample"]


# ---- generator sanity (inputs only) ---------------------------------------------
def test_generator_is_seeded_and_shaped():
    b0 = workloads.bank_for_config(0)
    b0b = workloads.bank_for_config(0)
    assert np.array_equal(b0["a"], b0b["a"]) and np.array_equal(b0["delay"], b0b["delay"])
    assert b0["n_templates"] == 4 and len(b0["a"]) == 128 and b0["delay"].max() <= 2047
    assert np.all(np.abs(b0["a"]) < 1)
    s0 = workloads.strain_for_config(0)
    assert s0["strain"].shape == (2, 2048) and s0["strain"].dtype == np.float32
    b2 = workloads.bank_for_config(2, n_templates=2)
    cnt = np.bincount(b2["band"][:600], minlength=8)
    assert list(cnt) == [75] * 8 and np.all(np.diff(b2["band"][:600].astype(int)) >= 0)
    from workloads.gen import _split_over_bands
    assert _split_over_bands(700, 8) == [87, 87, 87, 87, 88, 88, 88, 88]


# ---- O8 (NEXT-1): signal-consistency statistic, PAPER.md:177-188 (Eq. 11, 12) -------------
def _one_template_bank(a, b, d):
    return dict(n_templates=1, band_rates=[2048], out_band=0, tmpl_offset=np.array([0, len(a)], np.int64),
                a=a, b=b, delay=d, band=np.zeros(len(a), np.uint8), max_delay=[int(d.max())])


def test_p18_autocorrelation_closed_forms():
    # one filter: h[n] = b a^(n-d)  ->  A[j] = a^j (j >= 0), conj(a)^|j| (j < 0), whatever b and d
    a = np.array([np.exp(-1 / 37.0 + 0.83j)], np.complex64)
    b = np.array([0.3 - 1.1j], np.complex64)
    bank = _one_template_bank(a, b, np.array([11], np.int32))
    A = oracle.template_autocorr(bank, 0, 20)
    a64 = complex(a[0])
    for j in range(-20, 21):
        ref = a64 ** j if j >= 0 else np.conj(a64) ** (-j)
        assert abs(A[j + 20] - ref) < 1e-12
    # several filters with delays: the double sum over filter pairs of geometric series (P3's kernel at lag j)
    rng = np.random.default_rng(18)
    a, b, d = _rand_filters(rng, 6, dmax=25)
    A = oracle.template_autocorr(_one_template_bank(a, b, d), 0, 45)
    aa, bb = a.astype(np.complex128), b.astype(np.complex128)
    def R(j):
        tot = 0.0
        for l in range(6):
            for m in range(6):
                n0 = max(int(d[l]) - j, int(d[m]))
                tot += bb[l] * np.conj(bb[m]) * aa[l] ** (n0 + j - int(d[l])) * np.conj(aa[m]) ** (n0 - int(d[m])) \
                       / (1 - aa[l] * np.conj(aa[m]))
        return tot
    r0 = R(0)
    for j in (-45, -7, -1, 0, 1, 3, 40):
        assert abs(A[j + 45] - R(j) / r0) < 1e-10
    assert abs(A[45] - 1) < 1e-14 and np.allclose(A[::-1], np.conj(A))       # Hermitian, A[0] = 1


def test_p19_xi2_exact_signal_and_single_outlier():
    """z_I[c_I + j] = z0_I A[j] gives xi^2 = 0; one extra sample e at lag j1 != 0 in one detector gives
    xi_I^2 = |e|^2 / sum_j (2 - 2|A[j]|^2) there and xi_C^2 = that / N_d (Eq. 11, 12 by hand)."""
    nj, D, L = 12, 3, 200
    rng = np.random.default_rng(19)
    A = np.zeros((2, 2 * nj + 1), np.complex128)
    for r in range(2):
        aa = np.exp(-1 / (5.0 + 3 * r) + 1j * (0.4 + 0.5 * r))
        A[r] = [aa ** j if j >= 0 else np.conj(aa) ** (-j) for j in range(-nj, nj + 1)]
    delay = np.array([[0, 3, -5], [2, -4, 1]], np.int32)                     # two "pixels"
    z = np.zeros((D, 2, L), np.complex128)
    k, T, pix, row = 100, 1, 1, 1
    z0 = rng.standard_normal(D) + 1j * rng.standard_normal(D)
    for I in range(D):
        c = k + delay[pix, I] - delay[pix, T]
        z[I, row, c - nj:c + nj + 1] = z0[I] * A[row]
    args = dict(trig_valid=[1], trig_row=[row], trig_det=[T], trig_k=[k], pix=[pix], acorr=A, nj=nj)
    out = oracle.xi2(delay, z, 2 * L, L, L, L - 1, **args)
    assert np.all(np.abs(out[0, :D + 1]) < 1e-28) and out[0, D + 1] == 1
    e, j1, I1 = 0.7 - 0.2j, 5, 2
    z[I1, row, k + delay[pix, I1] - delay[pix, T] + j1] += e
    out = oracle.xi2(delay, z, 2 * L, L, L, L - 1, **args)
    den = np.sum(2 - 2 * np.abs(A[row]) ** 2)
    assert abs(out[0, I1] - abs(e) ** 2 / den) < 1e-14 and abs(out[0, D] - abs(e) ** 2 / den / D) < 1e-14
    assert out[0, 0] < 1e-28 and out[0, 1] < 1e-28
    # wrong pixel (other delays) no longer lines the windows up: the statistic is large
    bad = dict(args); bad["pix"] = [0]
    assert oracle.xi2(delay, z, 2 * L, L, L, L - 1, **bad)[0, D] > 1e-3
    # invalid slot, no pixel, window leaving the view: zeros and used = 0
    for kw in (dict(trig_valid=[0]), dict(pix=[-1]), dict(trig_k=[L - 3]), dict(trig_k=[nj - 1])):
        a2 = dict(args); a2.update(kw)
        assert np.all(oracle.xi2(delay, z, 2 * L, L, L, L - 1, **a2) == 0)


def test_p20_xi2_has_mean_one_in_gaussian_noise():
    """"a reduced chi^2 with a mean value of 1" - unit white noise through the oracle's own
    bank, A from the oracle's autocorrelation of the same templates."""
    rng = np.random.default_rng(20)
    bank = workloads.random_bank(rng, 6, 24, [2048], tau_range=(5.0, 60.0), max_delay=100)
    n, nj = 60000, 60
    x = rng.standard_normal((2, n)).astype(np.float32)
    z = oracle.filter_bank(x, bank)                                           # E|z|^2 = 2 (A8)
    A = np.stack([oracle.template_autocorr(bank, t, nj) for t in range(6)])
    ks = np.arange(2000, n - 200, 150)
    rows = np.repeat(np.arange(6), len(ks)); kk = np.tile(ks, 6)
    m = len(kk)
    delay = np.zeros((1, 2), np.int32)
    out = oracle.xi2(delay, z, 6 * n, n, n, n - 1, np.ones(m, np.int32), rows, np.zeros(m, np.int32), kk,
                     np.zeros(m, np.int32), A, nj)
    assert np.all(out[:, 3] == 1)
    assert abs(out[:, :2].mean() - 1.0) < 0.03                               # ~4600 windows of ~120 dof each
    assert np.allclose(out[:, 2], out[:, :2].mean(axis=1))                   # Eq. 12


def test_p21_xi2_on_time_slides():
    """O8 on the time-slid companions of O7: multipliers 0 reproduce the foreground on every slide; an exact
    signal whose companions sit s*step earlier gives 0 on slide s only; out-of-range slides are unused."""
    nj, D, L, step = 8, 3, 400, 50
    rng = np.random.default_rng(21)
    aa = np.exp(-1 / 4.0 + 0.7j)
    A = np.array([[aa ** j if j >= 0 else np.conj(aa) ** (-j) for j in range(-nj, nj + 1)]])
    delay = np.array([[1, -2, 4]], np.int32)
    z = (rng.standard_normal((D, 1, L)) + 1j * rng.standard_normal((D, 1, L)))
    k, T, S = 300, 0, 5
    base = dict(trig_valid=[1], trig_row=[0], trig_det=[T], trig_k=[k], acorr=A, nj=nj)
    fg = oracle.xi2(delay, z, L, L, L, L - 1, pix=[0], **base)
    bg0 = oracle.xi2(delay, z, L, L, L, L - 1, pix=np.zeros((1, S), np.int32), n_slides=S, step=step,
                     slide_mult=[0, 0, 0], **base)
    for s in range(S):
        assert np.array_equal(bg0[0, s], fg[0])
    # plant an exact signal: trigger detector at k, companions 3 slides earlier
    s0 = 3
    z0 = rng.standard_normal(D) + 1j * rng.standard_normal(D)
    for I in range(D):
        c = k + delay[0, I] - delay[0, T] - (s0 * step if I != T else 0)
        z[I, 0, c - nj:c + nj + 1] = z0[I] * A[0]
    bg = oracle.xi2(delay, z, L, L, L, L - 1, pix=np.zeros((1, S), np.int32), n_slides=S, step=step,
                    slide_mult=[1, 1, 1], **base)
    assert bg[0, s0 - 1, D] < 1e-28 and bg[0, s0 - 1, D + 1] == 1
    others = [s for s in range(S) if s != s0 - 1]
    assert np.all(bg[0, others, D] > 0.05)
    assert np.all(bg[0, :, T] < 1e-28)                                       # the trigger detector does not move
    # the sixth slide of step 50 from k = 300 with nj = 8 and delay -2 needs sample 300-300-2-8 < 0: unused
    bg6 = oracle.xi2(delay, z, L, L, L, L - 1, pix=np.zeros((1, 6), np.int32), n_slides=6, step=step,
                     slide_mult=[1, 1, 1], **base)
    assert bg6[0, 5, D + 1] == 0 and np.all(bg6[0, 5] == 0) and np.all(bg6[0, :5, D + 1] == 1)


# ---- NEXT-2: ranking statistic / FAP from the background (Eq. 13-15) ------------------
def test_p22_pseudo_log_binning():
    from oracle import rank
    x = np.float32(2.0) ** np.arange(-20, 21, dtype=np.float32)
    assert np.array_equal(rank.pseudo_log2(x), np.arange(-20, 21, dtype=np.float32))      # exact at powers of two
    xs = np.sort(np.random.default_rng(22).uniform(1e-3, 1e4, 5000).astype(np.float32))
    u = rank.pseudo_log2(xs)
    assert np.all(np.diff(u) >= 0)                                                        # monotone
    err = np.log2(xs.astype(np.float64)) - u
    assert err.min() > -1e-6 and err.max() < 0.0861                                       # chord under the log, max gap 0.0860
    assert abs(rank.pseudo_log2(np.float32([3.0]))[0] - 1.5) < 1e-7                       # 3 = 1.5 * 2^1 -> 1 + 0.5
    # bins: 8 bins over u in [0, 4): x = 1, 2, 3, 4, 15.9, and the clamped outsiders 0.3, 16, 100, 0, -1
    b = rank.bin_index(np.float32([1, 2, 3, 4, 15.9, 0.3, 16, 100, 0, -1]), 0.0, 4.0, 8)
    assert b.tolist() == [0, 2, 3, 4, 7, 0, 7, 7, 0, 0]


def test_p23_rank_and_fap_by_hand_and_by_counting_events():
    from oracle import rank
    # by hand: 2 x 2 bins (rho^2 axis u in [4, 8): edge at 2^6 = 64; xi^2 axis u in [-2, 2): edge at 1).
    bins = (2, 2, 4.0, 8.0, -2.0, 2.0)
    coh2 = np.float32([20, 30, 100, 150, 200, 70])          # rho-bins 0 0 1 1 1 1
    xi2 = np.float32([0.5, 3.0, 0.5, 0.7, 2.0, 0.9])       # xi-bins  0 1 0 0 1 0
    snr = np.float32([1, 1, 1, 1, 1, 1])
    H = rank.histogram(bins, snr, coh2, xi2, np.ones(6, np.int32))
    assert H.tolist() == [[1, 1], [3, 1]]
    Cc = rank.rank_counts(H)
    assert Cc.tolist() == [[4, 6], [3, 4]]                  # e.g. R(low rho, high xi) = everything = 6/6
    F = rank.fap_counts(H, Cc)
    assert F.tolist() == [[3, 5], [0, 3]]                   # bins with smaller R: (1,0) alone for C = 4; all but itself for C = 6
    R, fap, far, sel = rank.candidates(bins, H, np.float32([1, 20]), np.float32([120, 120]), np.float32([0.6, 0.6]),
                                       np.ones(2, np.int32), 50.0)
    assert sel.tolist() == [1, 0] and R[0] == 3 / 6 and fap[0] == 0.0 and far[0] == 0.0 and R[1] == 0
    # the cut rho_C >= rho_I + sqrt(2) decided in float32
    s = np.float32(5.0)
    edge = np.float32(s + np.float32(1.41421356)) ** 2
    assert rank.select([s, s], [np.nextafter(edge, np.float32(100)), np.nextafter(edge, np.float32(0)) * np.float32(0.999)],
                       [1, 1]).tolist() == [True, False]
    assert rank.select([s], [edge * 2], [0]).tolist() == [False]
    # by counting events: R and FAP from the event list itself, no histogram arithmetic
    rng = np.random.default_rng(23)
    n = 4000
    coh2 = (rng.chisquare(4, n) + 30).astype(np.float32)
    xi2 = (rng.chisquare(20, n) / 20).astype(np.float32)
    snr = rng.uniform(4, 5.5, n).astype(np.float32)
    used = (rng.random(n) < 0.9).astype(np.int32)
    bins = (12, 9, 4.5, 7.0, -1.5, 1.5)
    H = rank.histogram(bins, snr, coh2, xi2, used)
    sel = rank.select(snr, coh2, used)
    bi, bj = rank.bin_index(coh2, 4.5, 7.0, 12)[sel], rank.bin_index(xi2, -1.5, 1.5, 9)[sel]
    assert H.sum() == sel.sum() and 0.1 * n < sel.sum() < n
    Cc = rank.rank_counts(H)
    for i in range(12):
        for j in range(9):
            assert Cc[i, j] == np.sum((bi >= i) & (bj <= j))
    assert Cc[0, 8] == sel.sum() and np.all(np.diff(Cc, axis=0) <= 0) and np.all(np.diff(Cc, axis=1) >= 0)
    F = rank.fap_counts(H, Cc)
    r_event = Cc[bi, bj]
    for i in range(12):
        for j in range(9):
            assert F[i, j] == np.sum(r_event < Cc[i, j])
    # Eq. 14 is the cumulative distribution of R under the background: for background events themselves
    # FAP + P(same R) / 2 is uniform-like, mean 1/2
    same = np.array([np.sum(r_event == r) for r in r_event])
    assert abs(np.mean((F[bi, bj] + 0.5 * same) / sel.sum()) - 0.5) < 1e-9


# ---- P28 / P29: the two pins round 1 lacked (VERDICT r1 "What's weak" 1) --------------------------------
def _mutant(func, old, new):
    """The oracle function `func` with one source fragment replaced (a deliberately broken oracle): a pin
    earns its name only if such a plausible mistake turns it red."""
    import inspect
    import textwrap
    src = textwrap.dedent(inspect.getsource(func))
    assert src.count(old) == 1, "mutation target not found exactly once: %r" % old
    ns = dict(func.__globals__)
    exec(compile(src.replace(old, new), "<mutant of %s>" % func.__name__, "exec"), ns)
    return ns[func.__name__]


def _healpix_golden():
    rows = []
    for line in open(os.path.join(HERE, "golden", "healpix_ring_centres.txt")):
        f = line.split("#")[0].split()
        if len(f) == 4:
            rows.append((int(f[0]), int(f[1]), float(f[2]), float(f[3])))
    return rows


def _healpix_matches_golden(centres):
    for nside, pix, z, phi_over_pi in _healpix_golden():
        theta, phi = centres(nside)
        if abs(math.cos(theta[pix]) - z) > 1e-12 or abs(phi[pix] / math.pi - phi_over_pi) > 1e-12:
            return False
    return True


def test_p28_healpix_ring_centres_golden_values():
    """The in-ring phase of the HEALPix RING centres (the half-pixel shift of alternate belt rings, the
    j - 1/2 of the caps) against the base-pixel centres of ref. [46], typed into
    tests/golden/healpix_ring_centres.txt.  P15's invariants (sum of centres, ring count, spacing) are
    blind to that phase: the mutants below pass P15's checks and must fail here."""
    from oracle import sky
    rows = _healpix_golden()
    assert sum(1 for r in rows if r[0] == 1) == 12 and {r[1] for r in rows if r[0] == 2} >= {0, 4, 12, 20, 28, 44}
    assert _healpix_matches_golden(sky.healpix_ring_centres)
    # deliberately broken oracles: the belt's alternation swapped; the caps' half-pixel offset dropped
    swapped = _mutant(sky.healpix_ring_centres, "0.5 if (i + N) % 2 == 0 else 1.0", "1.0 if (i + N) % 2 == 0 else 0.5")
    assert not _healpix_matches_golden(swapped)
    th, ph = swapped(2)                                                       # ... while P15-style invariants still hold
    v = np.stack([np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph), np.cos(th)], axis=1)
    assert np.abs(v.sum(axis=0)).max() < 1e-12 and len(np.unique(np.round(np.cos(th), 12))) == 7
    no_half = _mutant(sky.healpix_ring_centres, "            z = 1.0 - i * i / (3.0 * N * N)\n            f = (j - 0.5)",
                      "            z = 1.0 - i * i / (3.0 * N * N)\n            f = (j - 1.0)")
    assert not _healpix_matches_golden(no_half)
    south = _mutant(sky.healpix_ring_centres, "j = 4 * i + 1 - (ps - 2 * i * (i - 1))", "j = ps - 2 * i * (i - 1)")
    assert not _healpix_matches_golden(south)                                 # a mirrored south cap is caught by pixels 44 / 47


def test_p29_far_by_hand_eq15():
    """Eq. 15: FAR = FAP N_b / T_b.  P23's 2 x 2 background (N_b = 6; H = [[1,1],[3,1]],
    R counts [[4,6],[3,4]], FAP counts [[3,5],[0,3]]) with T_b = 50 s:
      candidate in bin (0,0): R = 4/6, FAP = 3/6, FAR = 3/50 = 0.06 Hz;
      candidate in bin (0,1): R = 6/6, FAP = 5/6, FAR = 5/50 = 0.10 Hz  (N_b = 6, F = 5, T_b = 50 all differ,
      so a swapped or dropped factor gives another number)."""
    from oracle import rank
    bins = (2, 2, 4.0, 8.0, -2.0, 2.0)
    H = rank.histogram(bins, np.float32([1] * 6), np.float32([20, 30, 100, 150, 200, 70]),
                       np.float32([0.5, 3.0, 0.5, 0.7, 2.0, 0.9]), np.ones(6, np.int32))
    args = (bins, H, np.float32([1, 1, 1]), np.float32([30, 40, 100]), np.float32([0.5, 3.0, 0.6]), np.ones(3, np.int32), 50.0)

    def check(fn):
        R, fap, far, sel = fn(*args)
        return (sel.tolist() == [1, 1, 1]
                and np.allclose(R, [4 / 6, 1.0, 3 / 6], rtol=0, atol=1e-15)
                and np.allclose(fap, [3 / 6, 5 / 6, 0.0], rtol=0, atol=1e-15)
                and np.allclose(far, [0.06, 0.10, 0.0], rtol=0, atol=1e-15))

    assert check(rank.candidates)
    # deliberately broken oracles: N_b dropped (FAR = FAP / T_b), N_b applied twice, T_b ignored
    assert not check(_mutant(rank.candidates, "F[i, j] / float(background_seconds)",
                             "F[i, j] / max(nb, 1) / float(background_seconds)"))
    assert not check(_mutant(rank.candidates, "F[i, j] / float(background_seconds)",
                             "F[i, j] * nb / float(background_seconds)"))
    assert not check(_mutant(rank.candidates, "F[i, j] / float(background_seconds)", "F[i, j] / 1.0"))
    # T_b scales FAR inversely and leaves R and FAP alone
    far100 = rank.candidates(*args[:-1], 100.0)[2]
    assert np.allclose(far100, [0.03, 0.05, 0.0], rtol=0, atol=1e-15)


# ---- P14: strain-domain injection through a chirp-matched template (end-to-end sanity, loose by nature) ----
def test_p14_strain_injection_recovers_its_direction_or_the_mirror_image():
    """BASELINE.json config 1: the chirp injected into three detectors with the true arrival delays, filtered
    by the chirp-matched SPIIR template (O2-O3), searched over nside 16 (O5-O6).  With integer delays at
    2048 Hz (A18) the maximum lands within ~2 pixel widths of the true direction or of its mirror image
    through the plane of the three detectors; the true pixel is among the best few % and nearly as loud."""
    cfg = workloads.config(1)
    bank = workloads.bank_for_config(1, n_templates=1)                       # the chirp-matched template alone
    st = workloads.strain_for_config(1)
    inj = st["injections"][0]
    z = oracle.filter_bank(st["strain"], bank)                               # [3][1][n]
    k_true = int(round(inj["t_merge"] * 2048))
    net = np.sum(np.abs(z[:, 0]) ** 2, axis=0)
    # the loudest single-detector peak near the merger is the trigger
    lo, hi = k_true - 400, k_true + 400
    T = int(np.argmax([np.abs(z[I, 0, lo:hi]).max() for I in range(3)]))
    k = lo + int(np.argmax(np.abs(z[T, 0, lo:hi])))
    assert abs(k - k_true) < 100 and np.abs(z[T, 0, k]) > 6 and net[lo:hi].max() > 100   # network SNR 15 -> ~225
    pos, resp = workloads.detector_geometry(cfg["dets"])
    U2, delay = oracle.sky_table(16, pos, resp, cfg["sigma"], st["gmst"], 2048.0)
    n = z.shape[2]
    res, pix, mp = oracle.sky_search(U2.astype(np.float32), delay, z, n, n, n, n - 1, [1], [0], [T], [k],
                                     want_map=True)
    assert pix[0, 0] >= 0
    theta, phi = oracle.healpix_ring_centres(16)
    vec = np.stack([np.sin(theta) * np.cos(phi), np.sin(theta) * np.sin(phi), np.cos(theta)], axis=1)
    tv = np.array([math.sin(inj["theta"]) * math.cos(inj["phi"]), math.sin(inj["theta"]) * math.sin(inj["phi"]),
                   math.cos(inj["theta"])])
    # mirror image through the plane of the three detectors (same delays): reflect the source vector, in the
    # Earth-fixed frame the detector positions live in (longitude = phi - gmst)
    def earth(v, sign):
        c, s = math.cos(sign * st["gmst"]), math.sin(sign * st["gmst"])
        return np.array([c * v[0] + s * v[1], -s * v[0] + c * v[1], v[2]])
    nrm = np.cross(pos[1] - pos[0], pos[2] - pos[0]); nrm /= np.linalg.norm(nrm)
    te = earth(tv, +1)
    mv = earth(te - 2 * np.dot(te, nrm) * nrm, -1)
    best = vec[pix[0, 0]]
    ang = np.degrees(np.arccos(np.clip([best @ tv, best @ mv], -1, 1)))
    assert ang.min() < 7.5, ang
    p_true = int(np.argmax(vec @ tv))
    rank_true = int(np.sum(mp[0] > mp[0, p_true]))
    assert rank_true < 0.03 * len(vec)
    assert math.sqrt(mp[0, p_true]) >= 0.97 * math.sqrt(res[0, 0, 0])
    assert 12.0 < math.sqrt(res[0, 0, 0]) < 18.0                             # injected network SNR 15 in unit noise


# ----------------------------------------------------------------------------- NEXT-3: table sets
def _rings(nside):
    """(start, length) of every HEALPix ring, from the ring structure itself: 4 i pixels in the caps,
    4 nside in the belt."""
    out, s = [], 0
    lens = [4 * i for i in range(1, nside)] + [4 * nside] * (2 * nside + 1) + [4 * i for i in range(nside - 1, 0, -1)]
    for n in lens:
        out.append((s, n))
        s += n
    assert s == 12 * nside * nside
    return out


def test_p24_table_set_follows_the_earths_rotation():
    """U and the offsets are sampled every half hour over 24 h 'to accommodate the change
    of detector locations due to Earth's rotation'.  A quarter turn of the Earth (gmst + pi/2) moves every
    table entry a quarter of its ring to the east (every ring has a multiple of 4 pixels), a full sidereal
    day brings the set back, and a solar day leaves the 3 min 56 s that make the daily refresh necessary."""
    ns = 4
    pos, resp = workloads.detector_geometry(["H1", "L1", "V1"])
    sig = [1.0, 0.8, 0.5]
    U0, d0 = oracle.sky_table(ns, pos, resp, sig, 0.7, 2048.0)
    U1, d1 = oracle.sky_table(ns, pos, resp, sig, 0.7 + np.pi / 2, 2048.0)
    P0, P1 = U0 @ U0.transpose(0, 2, 1), U1 @ U1.transpose(0, 2, 1)
    for s, n in _rings(ns):
        j = np.arange(n)
        src = s + (j - n // 4) % n                              # entry now at phi was at phi - pi/2
        np.testing.assert_allclose(P1[s + j], P0[src], atol=1e-10)
        assert np.array_equal(d1[s + j], d0[src])
    assert not np.allclose(P1, P0, atol=1e-3)                   # and it is not the identity
    # the set: 49 samples a 48th of a sidereal day apart close on themselves, each is sky_table at its angle
    Us, ds = oracle.table_set(ns, pos, resp, sig, 0.7, oracle.sky.SIDEREAL_DAY_S / 48, 49, 2048.0)
    Ps = Us @ Us.transpose(0, 1, 3, 2)
    np.testing.assert_allclose(Ps[48], Ps[0], atol=1e-9)
    assert np.array_equal(ds[48], ds[0])
    np.testing.assert_allclose(Ps[12], P1, atol=1e-9)           # 12/48 of a turn = pi/2
    assert np.array_equal(ds[12], d1)
    omega = 7.2921150e-5                                        # Earth's rotation rate, rad/s (IERS)
    Ua, da = oracle.sky_table(ns, pos, resp, sig, 0.7 + omega * 5 * 1800.0, 2048.0)
    Ub, db = oracle.table_set(ns, pos, resp, sig, 0.7, 1800.0, 6, 2048.0)
    np.testing.assert_allclose(Ub[5] @ Ub[5].transpose(0, 2, 1), Ua @ Ua.transpose(0, 2, 1), atol=1e-6)
    assert np.mean(db[5] != da) < 0.01
    drift = (86400.0 / oracle.sky.SIDEREAL_DAY_S - 1.0) * 86400.0
    assert abs(drift - 236.6) < 0.5                             # seconds per solar day


def test_p25_nearest_table_and_the_east_west_statement():
    """'closest in the time to the triggering candidate' and 'the maximum coherent SNR value would not be
    affected but the detected sky direction ... could be off ... up to 15-min in the East-West direction'
    (PAPER.md:173)."""
    rng = np.random.default_rng(5)
    t0, dt, n = 1.0e9, 1800.0, 48
    for t in np.concatenate([t0 + rng.uniform(-900, 47 * 1800 + 900, 500), [t0, t0 + 47 * 1800.0]]):
        i = oracle.nearest_table(t, t0, dt, n)
        assert 0 <= i < n and abs(t - (t0 + i * dt)) <= 900.0   # never further than 15 min
        assert all(abs(t - (t0 + i * dt)) <= abs(t - (t0 + k * dt)) for k in (i - 1, i + 1))
    assert oracle.nearest_table(t0 + 2700.0, t0, dt, n) == 1    # exact tie: the earlier set
    assert oracle.nearest_table(t0 - 900.0, t0, dt, n) == 0
    assert oracle.nearest_table(t0 - 900.5, t0, dt, n) == -1    # stale on either side
    assert oracle.nearest_table(t0 + 47 * 1800 + 900.5, t0, dt, n) == -1
    # a signal built with the table of its own time, searched with a table k belt pixels of rotation
    # away: same maximum, found k pixels further east in the same ring
    ns, k = 8, 3
    pos, resp = workloads.detector_geometry(["H1", "L1", "V1"])
    sig = [1.0, 1.0, 0.5]
    Ut, dlt = oracle.sky_table(ns, pos, resp, sig, 1.234, 2048.0)
    Uo, dlo = oracle.sky_table(ns, pos, resp, sig, 1.234 + k * 2 * np.pi / (4 * ns), 2048.0)
    rings = _rings(ns)
    for ring in (ns + 1, 2 * ns, 3 * ns - 2):                   # belt rings
        s, nr = rings[ring]
        j0 = int(rng.integers(nr))
        p0 = s + j0
        z = np.zeros((3, 1, 800), complex)
        c = rng.standard_normal(2) + 1j * rng.standard_normal(2)
        amp = Ut[p0] @ c
        o = np.arange(-20, 21)
        env = np.exp(-o ** 2 / (2 * 6.0 ** 2)) * np.exp(0.6j * o)
        for I in range(3):
            z[I, 0, 400 + dlt[p0, I] - dlt[p0, 0] + o] = amp[I] * env
        kw = dict(trig_valid=[1], trig_row=[0], trig_det=[0], trig_k=[400], want_map=True, **_dense_view(z))
        rt, pt, mt = oracle.sky_search(Ut.astype(np.float32), dlt, z, **kw)
        ro, po, mo = oracle.sky_search(Uo.astype(np.float32), dlo, z, **kw)
        assert abs(ro[0, 0, 0] - rt[0, 0, 0]) < 1e-5 * rt[0, 0, 0]          # maximum not affected
        np.testing.assert_allclose(mo[0, s + (np.arange(nr) + k) % nr], mt[0, s:s + nr], rtol=1e-5, atol=1e-9)
        same_o = [p for p in range(12 * ns * ns) if np.array_equal(dlo[p] - dlo[p, 0], dlt[p0] - dlt[p0, 0])]
        assert po[0, 0] in same_o and (s + (j0 + k) % nr) in same_o


# ----------------------------------------------------------------------------- NEXT-3: sub-sample alignment
def test_p26_cubic_interpolator():
    """The 4-tap interpolator: textbook half-sample weights (-1, 9, 9, -1)/16, partition of unity,
    exact on cubics, sample-preserving, and accurate on a slow complex exponential."""
    np.testing.assert_allclose(oracle.lagrange4(0.5), np.array([-1, 9, 9, -1]) / 16.0, atol=1e-15)
    np.testing.assert_allclose(oracle.lagrange4(0.25), np.array([-7, 105, 35, -5]) / 128.0, atol=1e-15)
    for mu in np.linspace(0, 1, 11)[:-1]:
        w = oracle.lagrange4(mu)
        assert abs(w.sum() - 1) < 1e-14
        for deg in range(4):                                        # reproduces t^deg at t = mu
            assert abs(np.dot(w, np.array([-1.0, 0.0, 1.0, 2.0]) ** deg) - mu ** deg) < 1e-13
    # windows: layout, sample preservation, validity at the ring's edges, wrap-around
    rng = np.random.default_rng(3)
    D, rows, L, R, H = 2, 3, 64, 4, 5
    k_newest = 100                                                  # ring holds k = 37 .. 100
    t = np.arange(k_newest - L + 1, k_newest + 1)
    poly = lambda x: 0.3 + 0.1 * x - 0.02 * x ** 2 + 0.001j * x ** 3   # noqa: E731
    z = np.zeros((D, rows, L), complex)
    z[:, :, t % L] = poly(t - 70.0)
    trig_k = [70, 43, 42, 94, 95, 60]
    valid = [1, 1, 1, 1, 1, 0]
    rows_of = [0, 1, 2, 0, 1, 2]
    out, ok = oracle.upsample_windows(z, L, k_newest, valid, rows_of, [0, 1, 0, 1, 0, 1], trig_k, R, H)
    assert out.shape == (D, 6, 2 * R * H + 1)
    assert list(ok) == [1, 1, 0, 1, 0, 0]                           # k-H-1 >= 37 and k+H+1 <= 100
    for s in (0, 1, 3):
        tt = trig_k[s] - H + np.arange(2 * R * H + 1) / R
        np.testing.assert_allclose(out[0, s], poly(tt - 70.0), atol=1e-12)   # a cubic is reproduced exactly
        assert np.array_equal(out[1, s, ::R], z[1, rows_of[s], (trig_k[s] - H + np.arange(2 * H + 1)) % L])
    assert np.all(out[:, [2, 4, 5]] == 0)
    # a complex exponential at 0.05 cycles per sample (100 Hz at 2048 Hz): error below 1e-3
    zz = np.exp(2j * np.pi * 0.05 * np.arange(200))[None, None, :]
    o2, _ = oracle.upsample_windows(zz, 200, 199, [1], [0], [0], [100], 8, 20)
    tt = 80 + np.arange(321) / 8
    err = np.abs(o2[0, 0] - np.exp(2j * np.pi * 0.05 * tt)).max()
    assert 1e-5 < err < 1e-3
    # textbook remainder of cubic interpolation: |f''''| / 4! * max |(mu+1) mu (mu-1) (mu-2)| = w^4 / 24 * 9/16
    assert err <= (2 * np.pi * 0.05) ** 4 / 24 * 9 / 16 * 1.01


def test_p27_sub_sample_alignment_removes_the_integer_delay_loss():
    """Reading A18's probe: with delays rounded to the 2048 Hz grid a coherent signal leaks into the null
    stream; resampling the windows 4 times finer and searching with a table at 4 x 2048 Hz brings the
    null stream down by an order of magnitude and the coherent SNR back to the total."""
    rng = np.random.default_rng(41)
    ns, fs, R, H = 8, 2048.0, 4, 60
    pos, resp = workloads.detector_geometry(["H1", "L1", "V1"])
    sig = [1.0, 1.0, 0.5]
    U1, d1 = oracle.sky_table(ns, pos, resp, sig, 1.234, fs)
    UR, dR = oracle.sky_table(ns, pos, resp, sig, 1.234, fs * R)
    assert np.abs(dR - R * d1).max() <= R // 2 + 1                  # the same offsets on a finer grid
    th, ph = oracle.healpix_ring_centres(ns)
    lam = ph - 1.234
    nvec = np.stack([np.sin(th) * np.cos(lam), np.sin(th) * np.sin(lam), np.cos(th)], 1)
    tau = -(nvec @ pos.T) / workloads.C_LIGHT * fs                  # arrival offsets in samples, not rounded
    env = lambda x: np.exp(-x ** 2 / (2 * 6.0 ** 2)) * np.exp(0.3j * x)   # noqa: E731  (98 Hz carrier)
    n, k0 = 400, 200
    null_int, null_fine, loss_int, loss_fine = [], [], [], []
    for p0 in rng.choice(768, 12, replace=False):
        c = rng.standard_normal(2) + 1j * rng.standard_normal(2)
        amp = U1[p0] @ c
        tot = np.sum(np.abs(amp) ** 2)
        z = np.zeros((3, 1, n), complex)
        for I in range(3):
            z[I, 0] = amp[I] * env(np.arange(n) - k0 - (tau[p0, I] - tau[p0, 0]))
        kw = dict(trig_valid=[1], trig_row=[0], trig_det=[0], trig_k=[k0])
        r1, p1, _ = oracle.sky_search(U1.astype(np.float32), d1, z, **kw, **_dense_view(z))
        zu, ok = oracle.upsample_windows(z, n, n - 1, [1], [0], [0], [k0], R, H)
        assert ok[0] == 1
        r4, p4, _ = oracle.sky_search(UR.astype(np.float32), dR, zu, trig_valid=[1], trig_row=[0], trig_det=[0],
                                      trig_k=[R * H], **_dense_view(zu))
        assert p4[0, 0] == p0                                       # the fine search finds the true pixel
        null_int.append(r1[0, 0, 1] / tot); null_fine.append(r4[0, 0, 1] / tot)
        loss_int.append(1 - r1[0, 0, 0] / tot); loss_fine.append(1 - r4[0, 0, 0] / tot)
    assert np.mean(null_fine) < 0.1 * np.mean(null_int)
    assert np.mean(loss_fine) < 0.25 * np.mean(loss_int) and np.max(loss_fine) < 5e-3
    assert np.mean(loss_int) > 2e-3                                 # the loss being removed is real


# ---- NEXT-4: front end — pins P30-P35 of oracle/frontend.py ---------------------------------
def test_p30_downsampler_is_scipy_lfilter_decimated():
    """W1 reduces to a library routine: y = lfilter(h, 1, x)[R-1::R]."""
    from oracle import frontend as fe
    rng = np.random.default_rng(30)
    for R, nt in ((8, 192), (4, 64), (1, 5)):
        h = rng.standard_normal(nt)
        x = rng.standard_normal(R * 300)
        y = fe.downsample(x, h, R)
        np.testing.assert_allclose(y, scipy.signal.lfilter(h, 1.0, x)[R - 1::R], rtol=0, atol=1e-12)
    # a unit impulse at n = 5 comes out as the taps sampled every R-th with that offset
    h = np.arange(1.0, 25.0)
    x = np.zeros(80); x[5] = 1.0
    y = fe.downsample(x, h, 8)
    want = np.array([h[8 * m + 7 - 5] if 0 <= 8 * m + 7 - 5 < 24 else 0.0 for m in range(10)])
    assert np.array_equal(y, want)


def test_p31_whitener_is_the_identity_for_a_flat_psd_and_scales_a_line():
    """W2-W3: with S_n f_s / 2 = 1 the Hann blocks overlap-add back to the input exactly (window sum = 1, forward and
    inverse transform normalised); a sinusoid on a bin of known S_n comes out divided by sqrt(S_n f_s / 2)."""
    from oracle import frontend as fe
    rng = np.random.default_rng(31)
    H, fs = 128, 2048.0
    d = rng.standard_normal(H * 9)
    dw, S, P = fe.whiten_stream(d, H, fs, 27, psd_true=np.full(H + 1, 2.0 / fs))
    np.testing.assert_allclose(dw[:-H], d[:-H], rtol=0, atol=1e-13)          # (the last hop is only half added)
    w = fe.hann_periodic(2 * H)
    np.testing.assert_allclose(w[:H] + w[H:], 1.0, rtol=0, atol=1e-15)
    k0 = 20
    psd = np.full(H + 1, 2.0 / fs); psd[k0] = 9.0 * 2.0 / fs                 # S_n f_s / 2 = 9 on that bin: amplitude / 3
    t = np.arange(H * 9)
    line = np.cos(2 * np.pi * k0 * t / (2 * H))
    dw, _, _ = fe.whiten_stream(line, H, fs, 27, psd_true=psd)
    # the Hann window spreads a block's line over bins k0 - 1 .. k0 + 1 (amplitudes -1/4, 1/2, -1/4); only the central one
    # is divided by 3, and the side terms of two half-overlapped blocks cancel (their windows' cosines are in anti-phase):
    # what is left is the line itself, divided by 3
    want = line / 3.0
    np.testing.assert_allclose(dw[H:-H], want[H:-H], rtol=0, atol=1e-12)
    # Parseval on one block: sum |D|^2 = N sum (w d)^2, and the one-sided periodogram integrates to the windowed power
    blk = rng.standard_normal(2 * H) * w
    D = np.fft.rfft(blk)
    p1 = 2.0 * np.abs(D) ** 2 / (fs * np.sum(w * w))
    p1[0] /= 2; p1[-1] /= 2
    assert abs(p1.sum() * fs / (2 * H) - np.sum(blk ** 2) / np.sum(w * w)) < 1e-12


def test_p32_median_bias_and_unit_variance_out_of_white_noise():
    """W4: b(n) = sum (-1)^(i+1) / i is the textbook bias of the median of n exponential variates (b(1) = 1,
    b(3) = 5/6, -> ln 2), checked against a Monte-Carlo median; white noise of variance 9 is whitened to unit
    variance by the running estimate ("converges quickly"), with the small upward bias of 1 / S-hat."""
    from oracle import frontend as fe
    assert fe.median_bias(1) == 1.0 and abs(fe.median_bias(3) - 5.0 / 6.0) < 1e-15
    assert abs(fe.median_bias(27) - 0.71132) < 1e-5 and abs(fe.median_bias(9999) - math.log(2)) < 1e-4
    rng = np.random.default_rng(32)
    for n in (3, 9, 27):
        med = np.median(rng.exponential(1.0, size=(40000, n)), axis=1).mean()
        assert abs(med - fe.median_bias(n)) < 0.01
    H, fs = 256, 2048.0
    d = 3.0 * rng.standard_normal(H * 160)
    dw, S, P = fe.whiten_stream(d, H, fs, 27)
    assert np.all(S[0] == 0) and np.all(P[0] > 0) and np.all(S[1] == P[0])   # block 0 has no past: it only feeds the estimate
    assert abs((S[40:] * fs / 2).mean() - 9.0) < 0.2                         # the PSD estimate is unbiased
    assert 0.98 < dw[30 * H:-H].var() < 1.15                                 # unit variance (E 1/S-hat > 1/S by a few %)
    # one loud glitch in the history does not move the median estimate ("robust against glitches")
    d2 = d.copy(); d2[50 * H:50 * H + 40] += 500.0
    _, S2, _ = fe.whiten_stream(d2, H, fs, 27)
    _, _, P2 = fe.whiten_stream(d2, H, fs, 27)
    r = S2[60] / S[60]                           # two of the 27 blocks hold the glitch: the median moves by a rank, the mean by > 20 x
    assert np.median(r) < 1.2 and r.max() < 2.5 and np.median((P2[33:60].mean(axis=0) / P[33:60].mean(axis=0))[:20]) > 20


def test_p33_coloured_noise_comes_out_flat():
    """Eq. 1 on noise of KNOWN spectrum (AR(1) down-sampled): the whitened stream's Welch spectrum is flat at the
    unit-variance level 2 / f_s within the estimator's scatter, while the input's varies by a factor > 5."""
    from oracle import frontend as fe
    R, H, fs = 8, 256, 2048.0
    taps = workloads.frontend_taps(R, 192)
    x = workloads.frontend_strain(33, 1, R * H * 150)[0]
    y = fe.downsample(x, taps, R)
    dw, S, P = fe.whiten_stream(y, H, fs, 27)
    f, pin = scipy.signal.welch(y[40 * H:], fs=fs, nperseg=512)
    f, pout = scipy.signal.welch(dw[40 * H:-H], fs=fs, nperseg=512)
    band = (f > 20) & (f < 850)                                             # inside the down-sampler's pass band
    assert pin[band].max() / pin[band].min() > 5.0
    flat = pout[band] * fs / 2.0
    assert abs(flat.mean() - 1.05) < 0.1 and flat.std() < 0.12
    # and the estimate itself follows the known PSD of the generator (averaged over 8 adjacent bins of the 110 blocks;
    # below 650 Hz, where the down-sampler's response is flat)
    fk = np.arange(H + 1) * fs / (2 * H)
    lo = (fk > 20) & (fk < 650)
    ratio = (np.mean(S[40:], axis=0) / workloads.frontend_psd(fk))[lo]
    ratio = ratio[:len(ratio) // 8 * 8].reshape(-1, 8).mean(axis=1)
    assert np.all(np.abs(ratio - 1.0) < 0.12)


def test_p34_gate_zeroes_exactly_the_excursion_and_its_pads():
    """W5: with excursions on samples t0..t1 exactly [t0 - pad, t1 + pad] is zeroed, nothing else;
    two excursions closer than 2 pad merge; the stream's edges clip the window."""
    from oracle import frontend as fe
    d = np.ones(4000) * 0.5
    d[1000:1003] = 50.0; d[2500] = -60.0; d[2600] = 70.0; d[10] = 99.0
    m = fe.gate_mask(d, 8.0, 64)
    want = np.zeros(4000, bool)
    want[1000 - 64:1002 + 64 + 1] = True; want[2500 - 64:2600 + 64 + 1] = True; want[0:10 + 64 + 1] = True
    assert np.array_equal(m, want)
    assert not fe.gate_mask(np.full(100, 8.0), 8.0, 5).any()                 # strict: |d_w| > threshold


def test_p35_frontend_stream_latency_and_glitch_removal():
    """W6: the stream the front end emits is the gated whitened stream delayed by one hop plus the pad; a glitch in
    the raw data is gone from the output together with its pads, and nothing else is touched."""
    from oracle import frontend as fe
    R, H, fs, pad = 4, 256, 2048.0, 64
    taps = workloads.frontend_taps(R, 96)
    n_hops = 40
    x = workloads.frontend_strain(35, 2, R * H * n_hops, fs_in=fs * R, glitches=[(1, 30.3 * H / fs, 400.0)])
    out, dw = fe.frontend(x, taps, R, H, fs, 27, 8.0, pad)
    lag = H + pad
    for I in range(2):
        m = fe.gate_mask(dw[I, :(n_hops - 1) * H], 8.0, pad)
        want = np.where(m, 0.0, dw[I, :(n_hops - 1) * H])
        assert np.array_equal(out[I, lag:], want[:n_hops * H - lag]) and np.all(out[I, :lag] == 0)
    # once the PSD estimate has a few blocks (the first ones are whitened by one or three raw periodograms and gate
    # themselves), the only zeros are the glitch and its pads
    g0, warm = int(30.3 * H), 12 * H                                         # the glitch in output samples
    m1 = fe.gate_mask(dw[1, :(n_hops - 1) * H], 8.0, pad)
    z = np.nonzero(m1[warm:])[0] + warm
    assert z.min() <= g0 - pad + 12 and z.max() >= g0 + pad and z.max() - z.min() < 2 * pad + 40 and abs(z.mean() - g0) < 20
    assert not fe.gate_mask(dw[0, :(n_hops - 1) * H], 8.0, pad)[warm:].any()
