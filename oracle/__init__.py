"""float64 CPU ORACLE — test infrastructure only (see spiir_oracle.c header).

ctypes binding of oracle/libspiir_oracle.so (plain C, gcc) plus the numpy
look-up-table build O5 (oracle/sky.py).  Only tests/, bench.py's cpu_baseline /
--impl reference legs and __graft_entry__.smoke() may import this package; the
product package never does.
"""
import ctypes as C
import numpy as np

from .build import build as _build
from .sky import healpix_ring_centres, sky_table, g_sigma, table_set, nearest_table  # noqa: F401
from .upsample import lagrange4, upsample_windows  # noqa: F401
from . import frontend  # noqa: F401

_lib = None


_timed = False


def use_timed_build(threads=None):
    """bench.py only: switch to the -O3 -march=native build of the same source (compiled here, on this box) and
    set the OpenMP thread count (default: the physical cores).  Returns the thread count in use."""
    global _lib, _timed
    from .build import physical_cores
    _timed, _lib = True, None
    n = int(threads) if threads else physical_cores()
    lib().spiir_oracle_set_threads(C.c_int(n))
    return n


def set_threads(n):
    lib().spiir_oracle_set_threads(C.c_int(int(n)))


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build(timed=_timed))
        _lib.spiir_oracle_bank.restype = C.c_int
        _lib.spiir_oracle_sky.restype = C.c_int
        _lib.spiir_oracle_sky_eval.restype = C.c_int
        _lib.spiir_oracle_num_threads.restype = C.c_int
    return _lib


def _p(arr):
    return arr.ctypes.data_as(C.c_void_p) if arr is not None else None


def _f32c(x):
    """complex64 / float32 pairs -> contiguous float32 [...,2] view."""
    x = np.ascontiguousarray(x)
    if np.iscomplexobj(x):
        x = x.astype(np.complex64, copy=False).view(np.float32)
    return np.ascontiguousarray(x, dtype=np.float32)


def num_threads():
    return int(lib().spiir_oracle_num_threads())


def decimate(x, g):
    x = np.ascontiguousarray(x, dtype=np.float64)
    g = np.ascontiguousarray(g, dtype=np.float64)
    y = np.zeros(len(x) // 2)
    lib().spiir_oracle_decimate(_p(x), C.c_int64(len(x)), _p(g), C.c_int(len(g)), _p(y))
    return y


def band_sum(x, a, b, d):
    """s[m] = sum_l y_l[m] for one template in one band (O2+O3). complex128[n]."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    a, b = _f32c(a), _f32c(b)
    d = np.ascontiguousarray(d, dtype=np.int32)
    s = np.zeros((len(x), 2))
    lib().spiir_oracle_band_sum(_p(x), C.c_int64(len(x)), C.c_int64(len(d)), _p(a), _p(b), _p(d), _p(s))
    return s[:, 0] + 1j * s[:, 1]


def interp_add(acc_next, h, s=None):
    an = np.ascontiguousarray(acc_next, dtype=np.complex128).view(np.float64)
    n = 2 * len(acc_next)
    h = np.ascontiguousarray(h, dtype=np.float64)
    sv = None if s is None else np.ascontiguousarray(s, dtype=np.complex128).view(np.float64)
    acc = np.zeros((n, 2))
    lib().spiir_oracle_interp_add(_p(an), C.c_int64(n), _p(h), C.c_int(len(h)), _p(sv), _p(acc))
    return acc[:, 0] + 1j * acc[:, 1]


def filter_bank(strain, bank, dec_taps=None, int_taps=None, templates=None):
    """One-shot O1-O3 over the whole stream. Returns complex128 [n_det][n_sel][n_out]."""
    strain = np.ascontiguousarray(strain, dtype=np.float32)
    n_det, n0 = strain.shape
    B = len(bank["band_rates"])
    ob = int(bank["out_band"])
    T = int(bank["n_templates"])
    sel = np.arange(T, dtype=np.int64) if templates is None else np.ascontiguousarray(templates, dtype=np.int64)
    off = np.ascontiguousarray(bank["tmpl_offset"], dtype=np.int64)
    a, b = _f32c(bank["a"]), _f32c(bank["b"])
    d = np.ascontiguousarray(bank["delay"], dtype=np.int32)
    bnd = np.ascontiguousarray(bank["band"], dtype=np.uint8)
    if B > 1:
        assert dec_taps is not None and int_taps is not None
    dt = np.zeros(32, np.float32) if dec_taps is None else np.ascontiguousarray(dec_taps, dtype=np.float32)
    it = np.zeros(32, np.float32) if int_taps is None else np.ascontiguousarray(int_taps, dtype=np.float32)
    n_out = n0 >> ob
    z = np.zeros((n_det, len(sel), n_out, 2))
    rc = lib().spiir_oracle_bank(C.c_int(n_det), C.c_int64(n0), _p(strain), C.c_int(B), C.c_int(ob),
                                 C.c_int64(len(sel)), _p(sel), _p(off), _p(a), _p(b), _p(d), _p(bnd),
                                 _p(dt), _p(it), C.c_int(len(dt)), _p(z))
    if rc != 0:
        raise ValueError("spiir_oracle_bank: bad arguments")
    return z[..., 0] + 1j * z[..., 1]


def _zbuf(z):
    """Accepts complex128/float64[...,2] (double path) or complex64/float32[...,2] (fp32 decision path)."""
    z = np.ascontiguousarray(z)
    if z.dtype == np.complex128:
        return z.view(np.float64), 0
    if z.dtype == np.complex64:
        return z.view(np.float32), 1
    if z.dtype == np.float64:
        return z, 0
    if z.dtype == np.float32:
        return z, 1
    raise TypeError(z.dtype)


def peaks_mode0(z, thr):
    """z: [n_rows][n] complex. Returns (k int64[n_rows], valid int32[n_rows])."""
    buf, f32 = _zbuf(z)
    n_rows, n = z.shape[0], z.shape[1]
    k = np.zeros(n_rows, np.int64)
    v = np.zeros(n_rows, np.int32)
    lib().spiir_oracle_peaks_mode0(C.c_int64(n_rows), C.c_int64(n), _p(buf), C.c_int(f32),
                                   C.c_double(thr), _p(k), _p(v))
    return k, v


def peaks_mode1(z, thr, bank_size):
    buf, f32 = _zbuf(z)
    T, n = z.shape[0], z.shape[1]
    k = np.zeros(T, np.int64)
    v = np.zeros(T, np.int32)
    lib().spiir_oracle_peaks_mode1(C.c_int64(T), C.c_int64(n), C.c_int64(bank_size), _p(buf), C.c_int(f32),
                                   C.c_double(thr), _p(k), _p(v))
    return k, v


def _view_args(z, det_stride, row_stride, ring_len, k_newest):
    buf, f32 = _zbuf(z)
    return buf, [_p(buf), C.c_int(f32), C.c_int64(det_stride), C.c_int64(row_stride),
                 C.c_int64(ring_len), C.c_int64(k_newest)]


def sky_search(u2, delay, z, det_stride, row_stride, ring_len, k_newest,
               trig_valid, trig_row, trig_det, trig_k,
               n_slides=0, step=0, slide_mult=None, want_map=False):
    """O6 (n_slides=0) / O7.  u2 float32 [P][D][2], delay int32 [P][D].
    Returns (res float64 [n_trig][S][3] = coh2,null2,tot2; pix int32 [n_trig][S]; map or None)."""
    u2 = np.ascontiguousarray(u2, dtype=np.float32)
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    n_pix, n_det, _ = u2.shape
    n_trig = len(trig_k)
    S = max(1, n_slides)
    tv = np.ascontiguousarray(trig_valid, dtype=np.int32)
    tr = np.ascontiguousarray(trig_row, dtype=np.int32)
    td = np.ascontiguousarray(trig_det, dtype=np.int32)
    tk = np.ascontiguousarray(trig_k, dtype=np.int64)
    sm = np.ascontiguousarray(slide_mult if slide_mult is not None else np.zeros(n_det), dtype=np.int32)
    out = np.zeros((n_trig, S, 3))
    pix = np.zeros((n_trig, S), np.int32)
    mp = np.zeros((n_trig, n_pix)) if (want_map and n_slides == 0) else None
    buf, va = _view_args(z, det_stride, row_stride, ring_len, k_newest)
    rc = lib().spiir_oracle_sky(C.c_int(n_det), C.c_int64(n_pix), _p(u2), _p(delay), *va,
                                C.c_int64(n_trig), _p(tv), _p(tr), _p(td), _p(tk),
                                C.c_int(n_slides), C.c_int64(step), _p(sm), _p(out), _p(pix), _p(mp))
    if rc != 0:
        raise ValueError("spiir_oracle_sky: bad arguments")
    return out, pix, mp


def sky_eval(u2, delay, z, det_stride, row_stride, ring_len, k_newest, row, det, k, p,
             s=0, step=0, slide_mult=None):
    """One evaluation at pixel p (slide s, 0 = foreground): (ok, coh2, tot2-coh2, tot2)."""
    u2 = np.ascontiguousarray(u2, dtype=np.float32)
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    n_pix, n_det, _ = u2.shape
    sm = np.ascontiguousarray(slide_mult if slide_mult is not None else np.zeros(n_det), dtype=np.int32)
    res = np.zeros(3)
    buf, va = _view_args(z, det_stride, row_stride, ring_len, k_newest)
    ok = lib().spiir_oracle_sky_eval(C.c_int(n_det), C.c_int64(n_pix), _p(u2), _p(delay), *va,
                                     C.c_int32(row), C.c_int32(det), C.c_int64(k),
                                     C.c_int(s), C.c_int64(step), _p(sm), C.c_int64(p), _p(res))
    return bool(ok), res[0], res[1], res[2]


def template_autocorr(bank, t, nj, n_response=None):
    """Normalised autocorrelation A[j] = sum_n h[n+j] conj(h[n]) / sum_n |h[n]|^2, j = -nj..nj, of the
    impulse response h of template ``t`` (a single-band template at the output rate)
    ("the correlation function of a template with itself").  h is obtained by running the oracle's
    own recursion (O2+O3) on a unit impulse; the sums are written out directly.  complex128[2*nj+1]."""
    off = np.asarray(bank["tmpl_offset"])
    sl = slice(int(off[t]), int(off[t + 1]))
    a, b, d = np.asarray(bank["a"])[sl], np.asarray(bank["b"])[sl], np.asarray(bank["delay"])[sl]
    if len(set(np.asarray(bank["band"])[sl].tolist())) > 1:
        raise ValueError("template_autocorr: single-band templates only")
    if n_response is None:
        tau = -1.0 / np.log(np.abs(a.astype(np.complex128)))
        n_response = int(d.max() + 25.0 * tau.max()) + nj + 8
    x = np.zeros(n_response)
    x[0] = 1.0
    h = band_sum(x, a, b, d)
    norm = np.sum(np.abs(h) ** 2)
    A = np.zeros(2 * nj + 1, np.complex128)
    for j in range(-nj, nj + 1):
        if j >= 0:
            A[j + nj] = np.sum(h[j:] * np.conj(h[:len(h) - j]))
        else:
            A[j + nj] = np.sum(h[:len(h) + j] * np.conj(h[-j:]))
    return A / norm


def xi2(delay, z, det_stride, row_stride, ring_len, k_newest, trig_valid, trig_row, trig_det, trig_k, pix,
        acorr, nj, n_slides=0, step=0, slide_mult=None):
    """O8 (Eq. 11, 12).  acorr complex128 [rows][2*nj+1]; pix int32 [n_trig] (foreground) or
    [n_trig][n_slides].  Returns float64 [n_trig][n_det+2] (or [n_trig][n_slides][n_det+2]) =
    xi_I^2 per detector, xi_C^2, used flag."""
    delay = np.ascontiguousarray(delay, dtype=np.int32)
    n_det = delay.shape[1]
    n_trig = len(trig_k)
    S = max(1, n_slides)
    tv = np.ascontiguousarray(trig_valid, dtype=np.int32)
    tr = np.ascontiguousarray(trig_row, dtype=np.int32)
    td = np.ascontiguousarray(trig_det, dtype=np.int32)
    tk = np.ascontiguousarray(trig_k, dtype=np.int64)
    px = np.ascontiguousarray(pix, dtype=np.int32).reshape(n_trig, S)
    sm = np.ascontiguousarray(slide_mult if slide_mult is not None else np.zeros(n_det), dtype=np.int32)
    ac = np.ascontiguousarray(acorr, dtype=np.complex128)
    assert ac.shape[1] == 2 * nj + 1
    out = np.zeros((n_trig, S, n_det + 2))
    buf, va = _view_args(z, det_stride, row_stride, ring_len, k_newest)
    rc = lib().spiir_oracle_xi2(C.c_int(n_det), _p(delay), *va, C.c_int64(n_trig), _p(tv), _p(tr), _p(td),
                                _p(tk), _p(px), C.c_int(n_slides), C.c_int64(step), _p(sm),
                                _p(ac.view(np.float64)), C.c_int(nj), _p(out))
    if rc != 0:
        raise ValueError("spiir_oracle_xi2: bad arguments")
    return out if n_slides > 0 else out[:, 0]
