"""Seeded input generators (numpy only).  See package docstring for the rules.

Everything is drawn in float64 and rounded ONCE to float32 / complex64; the
rounded arrays are what both the oracle and the CUDA path consume.

Citations: PAPER.md:122 (a SPIIR filter = feed-forward b, feedback a, delay
t_d), PAPER.md:162 (SNR threshold 4), PAPER.md:489/:495 (unit variance per
quadrature, hence E|z|^2 = 2 — SURVEY.md §8(c) A8), BASELINE.json configs.
"""
import math
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
from scipy.signal import lfilter

from .configs import config, streams

C_LIGHT = 299792458.0
_N_THREADS = max(1, min(32, len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)))

# --------------------------------------------------------------------------
# FIR taps for the multirate layout (BASELINE.json config 2: "32-tap Kaiser
# (beta=5) windowed-sinc halfband FIR"; normalisation readings M2/M4).
# --------------------------------------------------------------------------

def halfband_taps(ntaps=32, beta=5.0):
    """Returns (dec_taps, int_taps) as float32[ntaps].

    g0[j] = 1/2 sinc((j - (ntaps-1)/2)/2) * kaiser[j].
    dec_taps = g0 / sqrt(sum g0^2)   (unit noise gain per decimation stage, M2)
    int_taps = 2 g0 / sum g0         (unity DC gain after zero-stuffing, M4)
    """
    j = np.arange(ntaps, dtype=np.float64)
    g0 = 0.5 * np.sinc(0.5 * (j - 0.5 * (ntaps - 1))) * np.kaiser(ntaps, beta)
    dec = g0 / math.sqrt(float(np.sum(g0 * g0)))
    itp = 2.0 * g0 / float(np.sum(g0))
    return dec.astype(np.float32), itp.astype(np.float32)


# --------------------------------------------------------------------------
# Detector geometry — an INPUT of the method.
# (lat deg, lon deg, height m, x-arm azimuth deg clockwise from north, y-arm)
# --------------------------------------------------------------------------
_DETECTORS = {
    "H1": (46.4551, -119.4077, 142.6, 324.0006, 234.0006),
    "L1": (30.5629, -90.7742, -6.6, 252.2835, 162.2835),
    "V1": (43.6314, 10.5045, 51.9, 19.4326, 289.4326),
}
_WGS84_A = 6378137.0
_WGS84_F = 1.0 / 298.257223563


def detector_geometry(names):
    """Earth-fixed positions [n,3] in metres and response tensors [n,3,3]
    D = (x x^T - y y^T)/2 from the arm unit vectors."""
    e2 = _WGS84_F * (2.0 - _WGS84_F)
    pos = np.zeros((len(names), 3))
    resp = np.zeros((len(names), 3, 3))
    for i, nm in enumerate(names):
        lat, lon, h, azx, azy = _DETECTORS[nm]
        la, lo = math.radians(lat), math.radians(lon)
        N = _WGS84_A / math.sqrt(1.0 - e2 * math.sin(la) ** 2)
        pos[i] = [(N + h) * math.cos(la) * math.cos(lo),
                  (N + h) * math.cos(la) * math.sin(lo),
                  (N * (1.0 - e2) + h) * math.sin(la)]
        east = np.array([-math.sin(lo), math.cos(lo), 0.0])
        north = np.array([-math.sin(la) * math.cos(lo), -math.sin(la) * math.sin(lo), math.cos(la)])
        x = math.sin(math.radians(azx)) * east + math.cos(math.radians(azx)) * north
        y = math.sin(math.radians(azy)) * east + math.cos(math.radians(azy)) * north
        resp[i] = 0.5 * (np.outer(x, x) - np.outer(y, y))
    return pos, resp


def _source_frame(theta, phi, gmst):
    lam = phi - gmst
    st, ct = math.sin(theta), math.cos(theta)
    n = np.array([st * math.cos(lam), st * math.sin(lam), ct])
    X = np.array([math.sin(lam), -math.cos(lam), 0.0])
    Y = np.array([-ct * math.cos(lam), -ct * math.sin(lam), st])
    return n, X, Y


def antenna_response(resp, theta, phi, gmst, psi):
    """Physical simulation of an injected signal: F+, Fx of each detector for a
    source at co-declination theta, right ascension phi, polarisation psi
    (F = rotation by 2 psi of (G+, Gx))."""
    n, X, Y = _source_frame(theta, phi, gmst)
    ep = np.outer(X, X) - np.outer(Y, Y)
    ec = np.outer(X, Y) + np.outer(Y, X)
    gp = np.einsum("dij,ij->d", resp, ep)
    gc = np.einsum("dij,ij->d", resp, ec)
    c2, s2 = math.cos(2 * psi), math.sin(2 * psi)
    return c2 * gp + s2 * gc, -s2 * gp + c2 * gc


def arrival_time(pos, theta, phi, gmst):
    """Arrival time at each detector relative to the geocentre, seconds."""
    n, _, _ = _source_frame(theta, phi, gmst)
    return -(pos @ n) / C_LIGHT


# --------------------------------------------------------------------------
# Filter banks
# --------------------------------------------------------------------------

def _split_over_bands(L, B):
    """M7: floor(L/B) per band, remainder to the lowest-rate bands first."""
    base = [L // B] * B
    for i in range(L % B):
        base[B - 1 - i] += 1
    return base


def _noise_variance(a, b, d, block_bytes=24 << 20):
    """Closed-form E|z|^2 of sum_l y_l in unit white noise, per template.

    a, b: complex128 [T, n]; d: int [T, n].  V = sum_{l,m} b_l conj(b_m) K_lm,
    K_lm = a_l^(d_m-d_l) / (1 - a_l conj(a_m))      if d_m >= d_l
         = conj(a_m)^(d_l-d_m) / (1 - a_l conj(a_m)) otherwise.
    Used only to scale the generated b (input normalisation, A8).
    """
    T, n = a.shape
    out = np.zeros(T)
    if n == 0:
        return out
    step = max(1, int(block_bytes // (n * n * 16 * 4)))
    la = np.log(a)

    def block(s):
        e = min(T, s + step)
        dd = (d[s:e, None, :] - d[s:e, :, None]).astype(np.float64)       # d_m - d_l  [T,l,m]
        pos = dd >= 0
        ex = np.where(pos, la[s:e, :, None] * dd, np.conj(la[s:e, None, :]) * (-dd))
        K = np.exp(ex) / (1.0 - a[s:e, :, None] * np.conj(a[s:e, None, :]))
        out[s:e] = np.real(np.einsum("tl,tm,tlm->t", b[s:e], np.conj(b[s:e]), K))

    # blocks are independent and their size does not depend on the thread count, so the
    # result is the same however many threads run them (numpy releases the GIL)
    starts = list(range(0, T, step))
    if len(starts) > 1 and _N_THREADS > 1:
        with ThreadPoolExecutor(_N_THREADS) as ex_:
            list(ex_.map(block, starts))
    else:
        for s in starts:
            block(s)
    return out


def random_bank(rng, n_templates, filters_per_template, band_rates, out_band=0,
                tau_range=(20.0, 2000.0), omega_range=(0.01, 1.5), max_delay=2047,
                exact_norm=True):
    """Random SPIIR bank (BASELINE.json config 0 recipe, per band M8).

    Returns a dict with CSR ``tmpl_offset`` int64[T+1], ``a``/``b`` complex64[n],
    ``delay`` int32[n] (samples of the filter's own band), ``band`` uint8[n];
    filters of a template are stored sorted by band.
    """
    B = len(band_rates)
    per_band = _split_over_bands(filters_per_template, B)
    L = filters_per_template
    T = n_templates
    tau = rng.uniform(*tau_range, size=(T, L))
    om = rng.uniform(*omega_range, size=(T, L))
    bre = rng.standard_normal((T, L))
    bim = rng.standard_normal((T, L))
    d = rng.integers(0, max_delay + 1, size=(T, L)).astype(np.int32)
    a32 = np.exp(-1.0 / tau + 1j * om).astype(np.complex64)
    a = a32.astype(np.complex128)
    b = (bre + 1j * bim) / math.sqrt(2.0)
    band = np.repeat(np.arange(B, dtype=np.uint8), per_band)[None, :].repeat(T, 0)
    V = np.zeros(T)
    o = 0
    for nb in per_band:
        sl = slice(o, o + nb)
        if exact_norm:
            V += _noise_variance(a[:, sl], b[:, sl], d[:, sl])
        else:  # diagonal approximation (cross terms of random phases dropped)
            V += np.sum(np.abs(b[:, sl]) ** 2 / (1.0 - np.abs(a[:, sl]) ** 2), axis=1)
        o += nb
    b = b * np.sqrt(2.0 / V)[:, None]
    return dict(
        n_templates=T, band_rates=list(band_rates), out_band=out_band,
        tmpl_offset=(np.arange(T + 1, dtype=np.int64) * L),
        a=a32.reshape(-1), b=b.astype(np.complex64).reshape(-1),
        delay=d.reshape(-1), band=band.reshape(-1).astype(np.uint8),
        max_delay=[max_delay] * B,
    )


def early_warning_bank(bank, rng, f_cut_range=(30.0, 60.0), max_rate_hz=256, exact_norm=True):
    """Early-warning variant of a multirate ``random_bank`` ("the early-warning configuration of the
    pipeline"): templates truncated before merger, so that a candidate exists while
    the signal is still in band.  Every template gets a seeded cut-off f_c ~ U[f_cut_range] Hz and keeps only the
    filters that (i) sit in a band of rate <= ``max_rate_hz`` and (ii) have a centre frequency arg(a) rate / (2 pi)
    <= f_c; b is rescaled so that the truncated template has unit noise variance again (A8: E|z|^2 = 2 in the
    steady state, i.e. once the longest delay line, 2047 samples of the 32 Hz band = 64 s, has filled).  The
    result is ragged (CSR) and leaves the bands above ``max_rate_hz`` without any filter.  Returns the new bank dict
    (plus ``f_cut`` [T]); the input is not modified."""
    T = int(bank["n_templates"])
    off = np.asarray(bank["tmpl_offset"])
    L = int(off[1] - off[0]) if T else 0
    assert np.array_equal(off, np.arange(T + 1, dtype=np.int64) * L), "needs the dense layout random_bank returns"
    rates = np.asarray(bank["band_rates"], dtype=np.float64)
    a = bank["a"].reshape(T, L).astype(np.complex128)
    b = bank["b"].reshape(T, L).astype(np.complex128)
    d = bank["delay"].reshape(T, L)
    band = bank["band"].reshape(T, L)
    f_cut = rng.uniform(*f_cut_range, size=T)
    f_centre = np.abs(np.angle(a)) * rates[band] / (2.0 * np.pi)
    keep = (rates[band] <= max_rate_hz) & (f_centre <= f_cut[:, None])
    bz = np.where(keep, b, 0.0)
    V = np.zeros(T)
    for bi in range(len(rates)):                               # filters of a template are stored sorted by band
        cols = np.nonzero(band[0] == bi)[0]
        if cols.size == 0 or not keep[:, cols].any():
            continue
        sl = slice(cols[0], cols[-1] + 1)
        # every band sees unit-variance noise (the decimation taps have unit noise gain, M2), as in random_bank
        if exact_norm:
            V += _noise_variance(a[:, sl], bz[:, sl], d[:, sl])
        else:
            V += np.sum(np.abs(bz[:, sl]) ** 2 / (1.0 - np.abs(a[:, sl]) ** 2), axis=1)
    scale = np.where(V > 0, np.sqrt(2.0 / np.where(V > 0, V, 1.0)), 1.0)
    b = b * scale[:, None]
    counts = keep.sum(axis=1)
    out = dict(bank)
    out.update(
        tmpl_offset=np.concatenate([[0], np.cumsum(counts)]).astype(np.int64),
        a=bank["a"].reshape(T, L)[keep], b=b.astype(np.complex64)[keep],
        delay=d[keep].astype(np.int32), band=band[keep].astype(np.uint8),
        max_delay=list(bank["max_delay"]), f_cut=f_cut,
    )
    out.pop("chirp_overlap", None)
    return out


# --------------------------------------------------------------------------
# Chirp (BASELINE.json config 1) and a naive SPIIR fit to it (generator only)
# --------------------------------------------------------------------------

def chirp_waveform(f0, tc, fs, f_cut=1000.0):
    """Complex h+ + i hx = A e^{i phi} sampled at fs from t=0 up to f=f_cut.
    f(t)=f0(1-t/tc)^(-3/8), phi=2 pi f0 tc (8/5)[1-(1-t/tc)^(5/8)], A=(f/f0)^(2/3)."""
    t_cut = tc * (1.0 - (f0 / f_cut) ** (8.0 / 3.0))
    K = int(math.floor(t_cut * fs))
    t = np.arange(K + 1) / fs
    u = 1.0 - t / tc
    f = f0 * u ** (-3.0 / 8.0)
    phi = 2 * math.pi * f0 * tc * (8.0 / 5.0) * (1.0 - u ** (5.0 / 8.0))
    A = (f / f0) ** (2.0 / 3.0)
    return A * np.exp(1j * phi), t, f


def chirp_matched_template(f0, tc, fs, n_filters, f_cut=1000.0):
    """Naive SPIIR approximation of the chirp: nodes walked
    backwards from the cut-off with spacing ~ tau, linear least squares for b.
    Returns (a complex64[n], b complex64[n], delay int32[n], overlap float)."""
    h, t, f = chirp_waveform(f0, tc, fs, f_cut)
    K = len(h) - 1
    target = np.conj(h[::-1])                               # g[n] = conj(h[K-n])

    def nodes(step):
        out = []
        tl = t[-1]
        while tl > 0 and len(out) < 4 * n_filters:
            fl = f0 * (1 - tl / tc) ** (-3.0 / 8.0)
            fdot = (3.0 / 8.0) * f0 / tc * (1 - tl / tc) ** (-11.0 / 8.0)
            tau = fs * math.sqrt(1.0 / (math.pi * fdot))
            out.append((tl, 2 * math.pi * fl / fs, tau))
            tl -= step * tau / fs
        return out

    lo, hi = 0.02, 2.0                                       # bisect the spacing for n_filters nodes
    for _ in range(40):
        mid = 0.5 * (lo + hi)
        if len(nodes(mid)) > n_filters:
            lo = mid
        else:
            hi = mid
    nd = nodes(hi)[:n_filters]
    while len(nd) < n_filters:                               # pad by repeating the earliest node shifted
        tl, om, tau = nd[-1]
        nd.append((max(tl - 0.5 * tau / fs, 0.0), om, tau))
    om = np.array([x[1] for x in nd])
    tau = np.array([x[2] for x in nd])
    d = np.array([K - int(round(x[0] * fs)) for x in nd], dtype=np.int32)
    a32 = np.exp(-1.0 / tau + 1j * om).astype(np.complex64)
    a = a32.astype(np.complex128)
    # Linear least squares for b against tgt[n] = target[n] (n <= K), through the normal
    # equations G b = r of the basis h_l[n] = a_l^(n-d_l) [n >= d_l], both in closed form:
    #   G_lm = sum_n conj(h_l[n]) h_m[n] = conj(a_l)^(d_m-d_l) / (1 - conj(a_l) a_m)   (d_m >= d_l)
    #                                    = a_m^(d_l-d_m)       / (1 - conj(a_l) a_m)   (d_m <  d_l)
    #   r_l  = sum_{n >= d_l} conj(a_l)^(n-d_l) target[n]   (a backward one-pole recursion)
    # The nodes oversample the chirp, so G is numerically singular: a tiny ridge picks the
    # small-norm solution.
    la = np.log(a)
    dd = (d[None, :] - d[:, None]).astype(np.float64)                  # d_m - d_l  [l, m]
    ex = np.where(dd >= 0, np.conj(la)[:, None] * dd, la[None, :] * (-dd))
    G = np.exp(ex) / (1.0 - np.conj(a)[:, None] * a[None, :])
    r = np.zeros(n_filters, complex)
    rev = target[::-1]
    for l in range(n_filters):
        # s[n] = target[n] + conj(a_l) s[n+1], evaluated at n = d_l (lfilter over the reversed series)
        seg = rev[:K + 1 - d[l]] if d[l] <= K else rev[:0]
        if len(seg):
            r[l] = lfilter([1.0], [1.0, -np.conj(a[l])], seg)[-1]
    ridge = 1e-9 * float(np.mean(np.real(np.diag(G))))
    b = np.linalg.solve(G + ridge * np.eye(n_filters), r)
    V = float(np.real(np.vdot(b, G @ b)))                    # E|z|^2 in unit white noise = sum |h|^2
    ov = abs(np.vdot(b, r)) / math.sqrt(V * float(np.vdot(target, target).real))
    b = b * math.sqrt(2.0 / V)
    return a32, b.astype(np.complex64), d, float(ov)


# --------------------------------------------------------------------------
# Strain
# --------------------------------------------------------------------------

def gaussian_strain(rng, n_det, n_samples):
    return rng.standard_normal((n_det, n_samples)).astype(np.float32)


def inject_chirp(strain, fs, pos, resp, sigma, f0, tc, t_start, snr, theta, phi, psi, gmst):
    """Adds sigma_I [F+ h+(t - tau_I) + Fx hx(t - tau_I)] scaled to a network
    optimal SNR ``snr`` (quadrature sum over detectors in unit white noise).
    Returns the float32 strain and a dict describing the injection."""
    h, t, _ = chirp_waveform(f0, tc, fs)
    fp, fc = antenna_response(resp, theta, phi, gmst, psi)
    tau = arrival_time(pos, theta, phi, gmst)
    n_det, n = strain.shape
    sig = np.zeros((n_det, n))
    grid = np.arange(n) / fs
    for i in range(n_det):
        tt = grid - t_start - tau[i]                         # source time at each detector sample
        hp = np.interp(tt, t, h.real, left=0.0, right=0.0)
        hc = np.interp(tt, t, h.imag, left=0.0, right=0.0)
        sig[i] = sigma[i] * (fp[i] * hp + fc[i] * hc)
    scale = snr / math.sqrt(float(np.sum(sig * sig)))
    out = (strain.astype(np.float64) + scale * sig).astype(np.float32)
    info = dict(theta=theta, phi=phi, psi=psi, gmst=gmst, t_merge=t_start + t[-1], tau=tau,
                det_snr=[float(scale * math.sqrt(np.sum(sig[i] ** 2))) for i in range(n_det)])
    return out, info


# --------------------------------------------------------------------------
# SNR snippets for the sky-search stress configuration (config 3)
# --------------------------------------------------------------------------

def snr_snippets(rng, u2, delay, n_rows, n_windows, half, coherent_fraction,
                 snr_range=(8.0, 20.0), env_sigma=6.0, env_omega=0.6):
    """Packed SNR view: float32 [n_det][n_rows][n_windows*(2*half+1)][2].

    Noise CN(0,2) (unit variance per quadrature).  ``coherent_fraction`` of the
    rows carry, in the LAST window, a signal lying in the plane spanned by the
    table's two projection vectors at a seeded pixel p0 (P13 form):
    z_I[k + (delta_I - delta_T) + o] += (U2(p0) c)_I e(o),  |e| peaked at o=0.
    ``u2``/``delay`` are the look-up table handed in as data (float32 [P][D][2],
    int32 [P][D]); no projection arithmetic happens here.
    Returns (z, trig_det int32[n_rows], k int64[n_rows], truth dict).
    """
    n_pix, n_det, _ = u2.shape
    W = 2 * half + 1
    n = n_windows * W
    z = rng.standard_normal((n_det, n_rows, n, 2)).astype(np.float32)
    trig_det = rng.integers(0, n_det, size=n_rows).astype(np.int32)
    k = np.full(n_rows, (n_windows - 1) * W + half, dtype=np.int64)
    is_sig = rng.random(n_rows) < coherent_fraction
    p0 = rng.integers(0, n_pix, size=n_rows)
    rho = rng.uniform(*snr_range, size=n_rows)
    c = (rng.standard_normal((n_rows, 2)) + 1j * rng.standard_normal((n_rows, 2)))
    o = np.arange(-4 * int(env_sigma), 4 * int(env_sigma) + 1)
    env = np.exp(-o ** 2 / (2 * env_sigma ** 2)) * np.exp(1j * env_omega * o)
    for r in np.nonzero(is_sig)[0]:
        amp = u2[p0[r]].astype(np.float64) @ c[r]
        amp *= rho[r] / np.linalg.norm(amp)
        for i in range(n_det):
            kk = int(k[r]) + int(delay[p0[r], i] - delay[p0[r], trig_det[r]]) + o
            s = amp[i] * env
            z[i, r, kk, 0] += s.real.astype(np.float32)
            z[i, r, kk, 1] += s.imag.astype(np.float32)
    return z, trig_det, k, dict(is_signal=is_sig, pix=p0, rho=rho)


# --------------------------------------------------------------------------
# Per-configuration assembly
# --------------------------------------------------------------------------

def bank_for_config(idx, n_templates=None, exact_norm=True, shard=0):
    """The filter bank of config ``idx`` (optionally with fewer templates —
    templates are independent, so a prefix is an exact sub-problem).  ``shard`` > 0
    draws the random templates of another template shard of the same shape (one
    shard per GPU: independent nodes of 4000 templates each)."""
    c = config(idx)
    rng = streams(c["seed"] + 7919 * int(shard))["bank"]
    T = c["n_templates"] if n_templates is None else n_templates
    bank = random_bank(rng, T, c["filters_per_template"], c["band_rates"], c["out_band"],
                       exact_norm=exact_norm)
    n_chirp = min(c["n_chirp_templates"], T)
    if n_chirp:
        inj_rng = streams(c["seed"])["injections"]
        params = chirp_params_for_config(c, inj_rng)
        L = c["filters_per_template"]
        band_of_2048 = c["band_rates"].index(2048)
        fits = [chirp_matched_template(params[t]["f0"], params[t]["tc"], 2048.0, L) for t in range(n_chirp)]
        for t, (a, b, d, ov) in enumerate(fits):
            sl = slice(t * L, (t + 1) * L)
            bank["a"][sl], bank["b"][sl], bank["delay"][sl] = a, b, d
            bank["band"][sl] = band_of_2048
            bank["max_delay"][band_of_2048] = max(bank["max_delay"][band_of_2048], int(d.max()))
            bank.setdefault("chirp_overlap", []).append(ov)
    return bank


def chirp_params_for_config(c, inj_rng):
    """Injection parameters: config 1 has one fixed chirp; config 4 draws 20."""
    n = c["injections"]
    out = []
    if c["index"] == 1:
        ch = c["chirp"]
        out.append(dict(f0=ch["f0"], tc=ch["tc"], t_start=ch["t_start"], snr=ch["snr"]))
    else:
        f0 = inj_rng.uniform(25.0, 40.0, size=n)
        tc = inj_rng.uniform(2.0, 12.0, size=n)
        snr = inj_rng.uniform(10.0, 20.0, size=n)
        slot = c["seconds"] / max(n, 1)
        for i in range(n):
            t0 = i * slot + 0.05 * slot
            out.append(dict(f0=float(f0[i]), tc=float(tc[i]), t_start=float(t0), snr=float(snr[i])))
    return out


def strain_for_config(idx, seconds=None):
    """float32 strain [n_det][seconds*f0] plus injection info and geometry."""
    c = config(idx)
    st = streams(c["seed"])
    secs = c["seconds"] if seconds is None else seconds
    f_in = c["band_rates"][0]
    x = gaussian_strain(st["strain"], len(c["dets"]), secs * f_in)
    pos, resp = detector_geometry(c["dets"])
    gmst = float(st["sky"].uniform(0, 2 * math.pi))
    infos = []
    if c["injections"]:
        params = chirp_params_for_config(c, st["injections"])
        for p in params:
            ct = st["sky"].uniform(-1, 1)
            theta, phi = math.acos(ct), float(st["sky"].uniform(0, 2 * math.pi))
            psi = float(st["sky"].uniform(0, math.pi))
            if p["t_start"] + p["tc"] + 0.1 > secs:
                continue
            x, info = inject_chirp(x, float(f_in), pos, resp, c["sigma"], p["f0"], p["tc"],
                                   p["t_start"], p["snr"], theta, phi, psi, gmst)
            infos.append(info)
    return dict(strain=x, pos=pos, resp=resp, gmst=gmst, sigma=np.array(c["sigma"], float),
                injections=infos, f_in=f_in)


# ----------------------------------------------------------------------------- NEXT-4: front-end inputs
def frontend_taps(decim=8, n_taps=192, beta=8.0):
    """Down-sampling FIR (an INPUT of the front end): Kaiser-windowed sinc, cut-off at 90 % of the output Nyquist
    frequency, unit DC gain.  PAPER.md:354: N_FIR-D ~ 192."""
    j = np.arange(n_taps) - 0.5 * (n_taps - 1)
    h = np.sinc(0.9 * j / decim) * np.kaiser(n_taps, beta)
    return (h / h.sum()).astype(np.float32)


def frontend_psd(f, fs_in=16384.0, rho=0.9, sigma=1.0):
    """One-sided PSD (per Hz) of the AR(1) noise `frontend_strain` draws: sigma^2 (2 / fs) / |1 - rho e^{-i w}|^2."""
    w = 2.0 * np.pi * np.asarray(f, float) / fs_in
    return sigma ** 2 * (2.0 / fs_in) / (1.0 - 2.0 * rho * np.cos(w) + rho * rho)


def frontend_strain(seed, n_det, n_samples, fs_in=16384.0, rho=0.9, sigma=1.0, glitches=()):
    """Raw strain for the front end: stationary coloured noise x[n] = rho x[n-1] + sigma e[n] (a known PSD of modest
    dynamic range standing in for a detector's spectrum, which is not available here) per detector, plus short
    glitches (detector, time in s, amplitude): a few samples wide, far above the noise.  float32 [n_det][n_samples]."""
    rng = np.random.default_rng(seed)
    import scipy.signal
    x = np.zeros((n_det, n_samples))
    for I in range(n_det):
        e = rng.standard_normal(n_samples + 2000)
        x[I] = scipy.signal.lfilter([sigma], [1.0, -rho], e)[2000:]
    for I, t, amp in glitches:
        i = int(round(t * fs_in))
        x[I, i:i + 24] += amp * np.hanning(24)
    return x.astype(np.float32)
