"""ctypes binding of libspiir_b200.so — argument marshalling only.

Every function of include/spiir.h is exposed under its C name (``spiir_bank_init``,
``spiir_filter_chunk``, ``spiir_peaks``, ``coherent_sky_search``,
``timeslide_background`` ...), taking raw device pointers (ints) exactly as the C
ABI does.  The small classes below (Bank, SkyPlan, SnrView) only own the torch
tensors that back the workspaces and outputs and pass ``tensor.data_ptr()`` and
``torch.cuda.current_stream().cuda_stream`` through; every step of the path runs in
the library's CUDA kernels.  There is no CPU fallback: a missing library raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libspiir_b200.so")

SPIIR_OK, SPIIR_EINVAL, SPIIR_ENOMEM, SPIIR_ECUDA, SPIIR_EOVERFLOW = 0, -1, -2, -3, -4
SPIIR_MAX_BANDS, SPIIR_MAX_DET, SPIIR_FIR_TAPS = 8, 4, 32


class SpiirError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("spiir error %d: %s" % (code, text))
        self.code = code


class spiir_bank_desc(C.Structure):
    _fields_ = [
        ("n_det", C.c_int32), ("n_templates", C.c_int32), ("n_bands", C.c_int32), ("out_band", C.c_int32),
        ("band_rate_hz", C.c_int32 * SPIIR_MAX_BANDS), ("max_delay", C.c_int32 * SPIIR_MAX_BANDS),
        ("n_filters", C.c_int64),
        ("host_tmpl_offset", C.c_void_p), ("host_a", C.c_void_p), ("host_b", C.c_void_p),
        ("host_delay", C.c_void_p), ("host_band", C.c_void_p),
        ("host_fir_dec", C.c_void_p), ("host_fir_int", C.c_void_p),
        ("max_chunk_samples", C.c_int32), ("bank_size", C.c_int32), ("ring_len", C.c_int64),
    ]


class spiir_snr_view(C.Structure):
    _fields_ = [("dev_z", C.c_void_p), ("det_stride", C.c_int64), ("row_stride", C.c_int64),
                ("ring_len", C.c_int64), ("k_newest", C.c_int64), ("n_rows", C.c_int64)]


class spiir_frontend_desc(C.Structure):
    _fields_ = [("n_det", C.c_int32), ("decim", C.c_int32), ("n_taps", C.c_int32), ("hop", C.c_int32),
                ("n_hist", C.c_int32), ("gate_pad", C.c_int32), ("out_rate_hz", C.c_float),
                ("gate_threshold", C.c_float), ("host_taps", C.c_void_p)]


class spiir_band_plan(C.Structure):
    _fields_ = [("lanes_per_unit", C.c_int32), ("filters_per_lane", C.c_int32), ("n_units", C.c_int32),
                ("n_units_long", C.c_int32), ("smem_history", C.c_int32), ("smem_bytes", C.c_int32),
                ("n_filters", C.c_int64), ("n_slots", C.c_int64)]


# numpy views of the two plain structs that live in device arrays
TRIGGER_DTYPE = np.dtype([("valid", "<i4"), ("tmpl", "<i4"), ("det", "<i4"), ("_pad", "<i4"), ("k", "<i8"),
                          ("z_re", "<f4"), ("z_im", "<f4"), ("snr", "<f4"), ("_pad2", "<f4")])
RESULT_DTYPE = np.dtype([("coh2", "<f4"), ("null2", "<f4"), ("tot2", "<f4"), ("pix", "<i4")])
XI2_DTYPE = np.dtype([("xi2_c", "<f4"), ("used", "<i4"), ("xi2", "<f4", (SPIIR_MAX_DET,))])
RANK_DTYPE = np.dtype([("rank", "<f4"), ("fap", "<f4"), ("far", "<f4"), ("selected", "<i4")])
assert TRIGGER_DTYPE.itemsize == 40 and RESULT_DTYPE.itemsize == 16 and XI2_DTYPE.itemsize == 24


class spiir_rank_bins(C.Structure):
    _fields_ = [("n_rho", C.c_int32), ("n_xi", C.c_int32), ("u_rho_min", C.c_float), ("u_rho_max", C.c_float),
                ("u_xi_min", C.c_float), ("u_xi_max", C.c_float)]

_SIGNATURES = {
    "spiir_bank_workspace_bytes": (C.c_int, [C.POINTER(spiir_bank_desc), C.POINTER(C.c_size_t)]),
    "spiir_bank_init": (C.c_int, [C.POINTER(C.c_void_p), C.POINTER(spiir_bank_desc), C.c_void_p, C.c_size_t, C.c_void_p]),
    "spiir_bank_reset": (C.c_int, [C.c_void_p, C.c_void_p]),
    "spiir_bank_free": (C.c_int, [C.c_void_p]),
    "spiir_filter_chunk": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]),
    "spiir_peaks": (C.c_int, [C.c_void_p, C.c_float, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]),
    "spiir_bank_snr_view": (C.c_int, [C.c_void_p, C.POINTER(spiir_snr_view)]),
    "spiir_sky_table_build": (C.c_int, [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                        C.c_double, C.c_void_p, C.c_void_p]),
    "spiir_sky_plan_workspace_bytes": (C.c_int, [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_size_t)]),
    "spiir_sky_plan_init": (C.c_int, [C.POINTER(C.c_void_p), C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                      C.c_void_p, C.c_size_t, C.c_void_p]),
    "spiir_sky_plan_free": (C.c_int, [C.c_void_p]),
    "spiir_sky_plan_tuples": (C.c_int32, [C.c_void_p]),
    "coherent_sky_search": (C.c_int, [C.c_void_p, C.POINTER(spiir_snr_view), C.c_void_p, C.c_int32, C.c_void_p,
                                      C.c_void_p, C.c_void_p]),
    "timeslide_background": (C.c_int, [C.c_void_p, C.POINTER(spiir_snr_view), C.c_void_p, C.c_int32, C.c_int32,
                                       C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p]),
    "spiir_bank_band_plan": (C.c_int, [C.c_void_p, C.c_int32, C.POINTER(spiir_band_plan)]),
    "spiir_bank_updates_per_chunk": (C.c_int64, [C.c_void_p, C.c_int32]),
    "spiir_launch_count": (C.c_int64, []),
    "spiir_bank_timing_enable": (C.c_int, [C.c_void_p, C.c_int32]),
    "spiir_bank_timing_read": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double),
                                         C.POINTER(C.c_int32)]),
    "spiir_signal_consistency": (C.c_int, [C.POINTER(spiir_snr_view), C.c_int32, C.c_int32, C.c_void_p, C.c_void_p,
                                           C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_void_p,
                                           C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p]),
    "spiir_rank_workspace_bytes": (C.c_int, [C.c_void_p, C.POINTER(C.c_size_t)]),
    "spiir_rank_reset": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "spiir_rank_accumulate": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                        C.c_int32, C.c_void_p]),
    "spiir_rank_finalize": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p]),
    "spiir_rank_candidates": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32,
                                        C.c_double, C.c_void_p, C.c_void_p]),
    "spiir_rank_static": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_void_p,
                                    C.c_void_p, C.c_void_p, C.c_int32, C.c_double, C.c_void_p, C.c_void_p]),
    "spiir_frontend_workspace_bytes": (C.c_int, [C.POINTER(spiir_frontend_desc), C.POINTER(C.c_size_t)]),
    "spiir_frontend_init": (C.c_int, [C.POINTER(C.c_void_p), C.POINTER(spiir_frontend_desc), C.c_void_p, C.c_size_t, C.c_void_p]),
    "spiir_frontend_reset": (C.c_int, [C.c_void_p, C.c_void_p]),
    "spiir_frontend_free": (C.c_int, [C.c_void_p]),
    "spiir_frontend_chunk": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "spiir_sky_table_set_build": (C.c_int, [C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double,
                                           C.c_double, C.c_int32, C.c_double, C.c_void_p, C.c_void_p]),
    "spiir_sky_table_nearest": (C.c_int, [C.c_double, C.c_double, C.c_double, C.c_int32, C.c_void_p]),
    "spiir_snr_upsample_elems": (C.c_int, [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p]),
    "spiir_snr_upsample_windows_slides": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32, C.c_int64,
                                                   C.c_void_p, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p,
                                                   C.c_void_p]),
    "spiir_snr_upsample_windows": (C.c_int, [C.c_void_p, C.c_int32, C.c_void_p, C.c_int32, C.c_int32, C.c_int32,
                                            C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "spiir_template_autocorr": (C.c_int, [C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int32, C.c_void_p]),
    "spiir_last_error": (C.c_char_p, []),
}
EXPORTS = sorted(_SIGNATURES)

_lib = None


def lib():
    """The loaded C-ABI library.  Raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("%s is missing: run `python -m paper_2011_06787_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def last_error():
    return lib().spiir_last_error().decode()


def _check(rc):
    if rc != SPIIR_OK:
        raise SpiirError(rc, last_error())
    return rc


def _mk(name):
    def call(*args):
        return getattr(lib(), name)(*args)
    call.__name__ = name
    call.__doc__ = "C ABI %s — see include/spiir.h" % name
    return call


for _n in EXPORTS:
    globals()[_n] = _mk(_n)


def _stream():
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _hp(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def make_desc(bank, n_det, max_chunk_samples, ring_len, bank_size=1000, dec_taps=None, int_taps=None):
    """spiir_bank_desc from a workloads bank dict; returns (desc, keepalive list)."""
    d = spiir_bank_desc()
    rates = list(bank["band_rates"])
    keep = [np.ascontiguousarray(bank["tmpl_offset"], dtype=np.int64),
            np.ascontiguousarray(np.asarray(bank["a"], dtype=np.complex64)).view(np.float32),
            np.ascontiguousarray(np.asarray(bank["b"], dtype=np.complex64)).view(np.float32),
            np.ascontiguousarray(bank["delay"], dtype=np.int32),
            np.ascontiguousarray(bank["band"], dtype=np.uint8),
            None if dec_taps is None else np.ascontiguousarray(dec_taps, dtype=np.float32),
            None if int_taps is None else np.ascontiguousarray(int_taps, dtype=np.float32)]
    d.n_det, d.n_templates, d.n_bands, d.out_band = n_det, int(bank["n_templates"]), len(rates), int(bank["out_band"])
    for i in range(SPIIR_MAX_BANDS):
        d.band_rate_hz[i] = rates[i] if i < len(rates) else 0
        d.max_delay[i] = int(bank["max_delay"][i]) if i < len(rates) else 0
    d.n_filters = len(keep[3])
    d.host_tmpl_offset, d.host_a, d.host_b, d.host_delay, d.host_band, d.host_fir_dec, d.host_fir_int = \
        [None if k is None else k.ctypes.data for k in keep]
    d.max_chunk_samples, d.bank_size, d.ring_len = int(max_chunk_samples), int(bank_size), int(ring_len)
    return d, keep


class SnrView:
    """A spiir_snr_view over a caller tensor z float32 [n_det][rows][ring_len][2] on the device."""

    def __init__(self, z=None, k_newest=None, raw=None):
        if raw is not None:
            self.c, self._keep = raw, None
            return
        assert z.is_cuda and z.dim() == 4 and z.shape[-1] == 2 and z.is_contiguous()
        n_det, rows, ring_len, _ = z.shape
        self._keep = z
        self.c = spiir_snr_view(z.data_ptr(), rows * ring_len, ring_len, ring_len,
                                ring_len - 1 if k_newest is None else int(k_newest), rows)


def upsample_windows(view, n_det, trig, n_slots, factor, half_width, n_slides=0, step=0, mult=None):
    """spiir_snr_upsample_windows (n_slides = 0) / spiir_snr_upsample_windows_slides: returns (SnrView over the
    resampled windows, re-addressed triggers uint8 cuda [n_slots * max(1, n_slides)][40]); the view keeps the window
    tensor alive."""
    import torch
    n = C.c_size_t(0)
    _check(lib().spiir_snr_upsample_elems(n_det, n_slots, int(factor), int(half_width), C.byref(n)))
    S1 = max(1, int(n_slides))
    out = torch.empty(max(int(n.value) * S1, 2), 2, dtype=torch.float32, device="cuda")
    trig_out = torch.empty(n_slots * S1, 40, dtype=torch.uint8, device="cuda")
    ov = spiir_snr_view()
    if n_slides:
        m = (C.c_int32 * n_det)(*[int(x) for x in mult])
        _check(lib().spiir_snr_upsample_windows_slides(C.byref(view.c), n_det, C.c_void_p(trig.data_ptr()), n_slots,
                                                       int(n_slides), C.c_int64(int(step)), m, int(factor), int(half_width),
                                                       C.c_void_p(out.data_ptr()), C.c_void_p(trig_out.data_ptr()),
                                                       C.byref(ov), _stream()))
    else:
        _check(lib().spiir_snr_upsample_windows(C.byref(view.c), n_det, C.c_void_p(trig.data_ptr()), n_slots, int(factor),
                                                int(half_width), C.c_void_p(out.data_ptr()),
                                                C.c_void_p(trig_out.data_ptr()), C.byref(ov), _stream()))
    v = SnrView(raw=ov)
    v._keep = out
    return v, trig_out


class Bank:
    """Owns the workspace tensor of one spiir_bank and forwards to the C ABI."""

    def __init__(self, bank, n_det, max_chunk_samples, ring_len=None, bank_size=1000, dec_taps=None, int_taps=None):
        import torch
        n_out_max = max_chunk_samples >> int(bank["out_band"])
        ring_len = n_out_max if ring_len is None else ring_len
        self.desc, self._keep = make_desc(bank, n_det, max_chunk_samples, ring_len, bank_size, dec_taps, int_taps)
        nbytes = C.c_size_t(0)
        _check(lib().spiir_bank_workspace_bytes(C.byref(self.desc), C.byref(nbytes)))
        self.workspace_bytes = nbytes.value
        self.ws = torch.empty(nbytes.value + 256, dtype=torch.uint8, device="cuda")
        base = (self.ws.data_ptr() + 255) // 256 * 256
        self.h = C.c_void_p()
        _check(lib().spiir_bank_init(C.byref(self.h), C.byref(self.desc), C.c_void_p(base), nbytes, _stream()))
        self.n_det, self.n_templates = n_det, int(bank["n_templates"])
        self.out_band, self.n_bands = int(bank["out_band"]), len(bank["band_rates"])
        self.n_slots = self.n_det * self.n_templates
        self.trig = torch.zeros(self.n_slots, 40, dtype=torch.uint8, device="cuda")
        self.count = torch.zeros(1, dtype=torch.int32, device="cuda")

    def reset(self):
        _check(lib().spiir_bank_reset(self.h, _stream()))

    def filter_chunk(self, strain, snr_out=None):
        """strain: float32 cuda [n_det][n]; snr_out: float32 cuda [n_det][T][n>>out_band][2] or None."""
        assert strain.is_cuda and strain.is_contiguous() and strain.dtype.is_floating_point and strain.element_size() == 4
        n = strain.shape[-1]
        if snr_out is not None:
            assert snr_out.is_cuda and snr_out.is_contiguous()
            assert snr_out.numel() == self.n_det * self.n_templates * (n >> self.out_band) * 2
        _check(lib().spiir_filter_chunk(self.h, C.c_void_p(strain.data_ptr()), n,
                                        C.c_void_p(snr_out.data_ptr()) if snr_out is not None else None, _stream()))

    def peaks(self, threshold, mode=0, trig=None, count=None):
        """spiir_peaks into the given device buffers (default: the Bank's own)."""
        trig = self.trig if trig is None else trig
        count = self.count if count is None else count
        _check(lib().spiir_peaks(self.h, C.c_float(threshold), mode, C.c_void_p(trig.data_ptr()),
                                 C.c_void_p(count.data_ptr()), _stream()))
        return trig, count

    def snr_view(self):
        v = spiir_snr_view()
        _check(lib().spiir_bank_snr_view(self.h, C.byref(v)))
        return SnrView(raw=v)

    def ring_rows(self, rows):
        """The SNR ring rows of the templates `rows` (int64 cuda tensor) as float32 cuda [n_det][len(rows)][ring_len][2]
        (element k mod ring_len of a row is sample k): a torch view of the workspace, copied; no arithmetic."""
        import torch
        v = self.snr_view().c
        off = int(v.dev_z) - self.ws.data_ptr()
        L = int(v.ring_len)
        n = self.n_det * self.n_templates * L * 2
        ring = self.ws[off:off + 4 * n].view(torch.float32).view(self.n_det, self.n_templates, L, 2)
        return ring[:, rows].contiguous()

    def band_plan(self, band):
        p = spiir_band_plan()
        _check(lib().spiir_bank_band_plan(self.h, band, C.byref(p)))
        return {f[0]: getattr(p, f[0]) for f in spiir_band_plan._fields_}

    def timing_enable(self, n_chunks):
        """Record the next n_chunks filter_chunk calls (events are created here, not in the call); 0 = off."""
        _check(lib().spiir_bank_timing_enable(self.h, int(n_chunks)))

    def timing_read(self):
        """(ms in the recursion kernels, ms in whole filter_chunk calls, number of calls) since the last read."""
        a, c, n = C.c_double(0), C.c_double(0), C.c_int32(0)
        _check(lib().spiir_bank_timing_read(self.h, C.byref(a), C.byref(c), C.byref(n)))
        return a.value, c.value, n.value

    def updates_per_chunk(self, n_samples):
        return int(lib().spiir_bank_updates_per_chunk(self.h, n_samples))

    def close(self):
        if self.h:
            lib().spiir_bank_free(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def sky_table_build(nside, pos, resp, sigma, gmst, fs):
    """Host look-up table (spiir_sky_table_build): returns (u2 float32 [P][D][2], delay int32 [P][D])."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    resp = np.ascontiguousarray(resp, dtype=np.float64)
    sigma = np.ascontiguousarray(sigma, dtype=np.float64)
    n_det = pos.shape[0]
    npix = 12 * nside * nside
    u2 = np.zeros((npix, n_det, 2), np.float32)
    delay = np.zeros((npix, n_det), np.int32)
    _check(lib().spiir_sky_table_build(nside, n_det, _hp(pos), _hp(resp), _hp(sigma), float(gmst), float(fs),
                                       _hp(u2), _hp(delay)))
    return u2, delay


def sky_table_set_build(nside, pos, resp, sigma, gmst0, interval_s, n_sets, fs):
    """spiir_sky_table_set_build: (u2 float32 [n_sets][P][D][2], delay int32 [n_sets][P][D])."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    resp = np.ascontiguousarray(resp, dtype=np.float64)
    sigma = np.ascontiguousarray(sigma, dtype=np.float64)
    n_det = pos.shape[0]
    npix = 12 * nside * nside
    u2 = np.zeros((n_sets, npix, n_det, 2), np.float32)
    delay = np.zeros((n_sets, npix, n_det), np.int32)
    _check(lib().spiir_sky_table_set_build(nside, n_det, _hp(pos), _hp(resp), _hp(sigma), float(gmst0),
                                           float(interval_s), int(n_sets), float(fs), _hp(u2), _hp(delay)))
    return u2, delay


def sky_table_nearest(t, t0, interval_s, n_sets):
    """spiir_sky_table_nearest: index of the set closest in time, -1 when the tables are stale."""
    idx = C.c_int32(-2)
    _check(lib().spiir_sky_table_nearest(float(t), float(t0), float(interval_s), int(n_sets), C.byref(idx)))
    return int(idx.value)


class SkyPlanSet:
    """One SkyPlan per sampled table; `select(t)` is the plan closest in time to t."""

    def __init__(self, u2_sets, delay_sets, max_slots, t0, interval_s):
        self.t0, self.interval_s = float(t0), float(interval_s)
        self.plans = [SkyPlan(u, d, max_slots) for u, d in zip(u2_sets, delay_sets)]

    def index(self, t):
        i = sky_table_nearest(t, self.t0, self.interval_s, len(self.plans))
        if i < 0:
            raise SpiirError(SPIIR_EINVAL, "sky tables are stale at t = %r: rebuild the set" % (t,))
        return i

    def select(self, t):
        return self.plans[self.index(t)]

    def close(self):
        for p in self.plans:
            p.close()


class SkyPlan:
    """Owns the workspace of one spiir_sky_plan and the output tensors of its searches."""

    def __init__(self, u2, delay, max_slots):
        import torch
        u2 = np.ascontiguousarray(u2, dtype=np.float32)
        delay = np.ascontiguousarray(delay, dtype=np.int32)
        self.n_pix, self.n_det = int(u2.shape[0]), int(u2.shape[1])
        self.max_slots = int(max_slots)
        nbytes = C.c_size_t(0)
        _check(lib().spiir_sky_plan_workspace_bytes(self.n_det, self.n_pix, self.max_slots, C.byref(nbytes)))
        self.ws = torch.empty(nbytes.value + 256, dtype=torch.uint8, device="cuda")
        base = (self.ws.data_ptr() + 255) // 256 * 256
        self.h = C.c_void_p()
        _check(lib().spiir_sky_plan_init(C.byref(self.h), self.n_det, self.n_pix, self.max_slots, _hp(u2), _hp(delay),
                                         C.c_void_p(base), nbytes, _stream()))
        self.n_tuples = int(lib().spiir_sky_plan_tuples(self.h))

    def search(self, view, trig, n_slots, out=None, skymap=None):
        """coherent_sky_search; trig: uint8 cuda [n_slots][40]; returns out float32-bytes cuda [n_slots][16]."""
        import torch
        if out is None:
            out = torch.empty(n_slots, 16, dtype=torch.uint8, device="cuda")
        _check(lib().coherent_sky_search(self.h, C.byref(view.c), C.c_void_p(trig.data_ptr()), n_slots,
                                         C.c_void_p(out.data_ptr()),
                                         C.c_void_p(skymap.data_ptr()) if skymap is not None else None, _stream()))
        return out

    def background(self, view, trig, n_slots, n_slides, step, mult, out=None):
        import torch
        if out is None:
            out = torch.empty(n_slots * n_slides, 16, dtype=torch.uint8, device="cuda")
        m = np.ascontiguousarray(mult, dtype=np.int32)
        _check(lib().timeslide_background(self.h, C.byref(view.c), C.c_void_p(trig.data_ptr()), n_slots, n_slides,
                                          int(step), _hp(m), C.c_void_p(out.data_ptr()), _stream()))
        return out

    def close(self):
        if self.h:
            lib().spiir_sky_plan_free(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def triggers_to_numpy(trig):
    return trig.cpu().numpy().view(TRIGGER_DTYPE).reshape(-1)


def triggers_from_numpy(arr):
    import torch
    arr = np.ascontiguousarray(arr, dtype=TRIGGER_DTYPE)
    return torch.from_numpy(arr.view(np.uint8).reshape(-1, 40)).cuda()


def results_to_numpy(out):
    return out.cpu().numpy().view(RESULT_DTYPE).reshape(-1)


def template_autocorr(bank, t, n_j):
    """spiir_template_autocorr for template ``t`` of a bank dict: complex64 [2 n_j + 1]."""
    off = np.asarray(bank["tmpl_offset"])
    sl = slice(int(off[t]), int(off[t + 1]))
    a = np.ascontiguousarray(np.asarray(bank["a"])[sl], dtype=np.complex64)
    b = np.ascontiguousarray(np.asarray(bank["b"])[sl], dtype=np.complex64)
    d = np.ascontiguousarray(np.asarray(bank["delay"])[sl], dtype=np.int32)
    out = np.zeros(2 * n_j + 1, np.complex64)
    _check(lib().spiir_template_autocorr(len(d), _hp(a), _hp(b), _hp(d), n_j, _hp(out)))
    return out


def signal_consistency(view, delay_dev, trig, sky, n_slots, autocorr_dev, n_j, out=None,
                       n_slides=0, step=0, mult=None):
    """spiir_signal_consistency; delay_dev int32 cuda [n_pix][n_det], trig uint8 cuda [n_slots][40],
    sky uint8 cuda [n_slots (* n_slides)][16], autocorr_dev float32 cuda [rows][2 n_j + 1][2]; returns uint8
    cuda [n_slots (* n_slides)][24] (XI2_DTYPE)."""
    import torch
    n_pix, n_det = delay_dev.shape
    assert delay_dev.is_cuda and delay_dev.dtype == torch.int32 and delay_dev.is_contiguous()
    assert autocorr_dev.is_cuda and autocorr_dev.is_contiguous() and autocorr_dev.shape[-2] == 2 * n_j + 1
    if out is None:
        out = torch.empty(n_slots * max(1, n_slides), 24, dtype=torch.uint8, device="cuda")
    m = np.ascontiguousarray(mult if mult is not None else np.zeros(n_det), dtype=np.int32)
    _check(lib().spiir_signal_consistency(C.byref(view.c), n_det, n_pix, C.c_void_p(delay_dev.data_ptr()),
                                          C.c_void_p(trig.data_ptr()), C.c_void_p(sky.data_ptr()), n_slots,
                                          n_slides, int(step), _hp(m),
                                          C.c_void_p(autocorr_dev.data_ptr()), n_j, C.c_void_p(out.data_ptr()),
                                          _stream()))
    return out


def xi2_to_numpy(out):
    return out.cpu().numpy().view(XI2_DTYPE).reshape(-1)


class Ranker:
    """Owns the workspace of the background histogram (spiir_rank_*): accumulate -> finalize -> candidates."""

    def __init__(self, n_rho, n_xi, u_rho_min, u_rho_max, u_xi_min, u_xi_max):
        import torch
        self.bins = spiir_rank_bins(n_rho, n_xi, u_rho_min, u_rho_max, u_xi_min, u_xi_max)
        n = C.c_size_t(0)
        _check(lib().spiir_rank_workspace_bytes(C.byref(self.bins), C.byref(n)))
        self.ws = torch.empty(n.value // 8, dtype=torch.int64, device="cuda")
        self.reset()

    def _b(self):
        return C.cast(C.byref(self.bins), C.c_void_p)

    def reset(self):
        _check(lib().spiir_rank_reset(C.c_void_p(self.ws.data_ptr()), self._b(), _stream()))

    def accumulate(self, trig, bg, xi, n_slots, n_slides):
        _check(lib().spiir_rank_accumulate(C.c_void_p(self.ws.data_ptr()), self._b(), C.c_void_p(trig.data_ptr()),
                                           C.c_void_p(bg.data_ptr()), C.c_void_p(xi.data_ptr()), n_slots, n_slides,
                                           _stream()))

    def finalize(self):
        _check(lib().spiir_rank_finalize(C.c_void_p(self.ws.data_ptr()), self._b(), _stream()))

    def candidates(self, trig, fg, xi, n_slots, background_seconds, out=None):
        import torch
        if out is None:
            out = torch.empty(n_slots, 16, dtype=torch.uint8, device="cuda")
        _check(lib().spiir_rank_candidates(C.c_void_p(self.ws.data_ptr()), self._b(), C.c_void_p(trig.data_ptr()),
                                           C.c_void_p(fg.data_ptr()), C.c_void_p(xi.data_ptr()), n_slots,
                                           float(background_seconds), C.c_void_p(out.data_ptr()), _stream()))
        return out

    def tables(self):
        """(N_b, H, R counts, FAP counts) as numpy int64 arrays [n_rho][n_xi]."""
        w = self.ws.cpu().numpy()
        n = self.bins.n_rho * self.bins.n_xi
        shp = (self.bins.n_rho, self.bins.n_xi)
        return int(w[0]), w[4:4 + n].reshape(shp), w[4 + n:4 + 2 * n].reshape(shp), w[4 + 2 * n:4 + 3 * n].reshape(shp)


SPIIR_RANK_STATIC_MAX_BINS = 4096


def rank_static(bins, bg_trig, bg, bg_xi, n_bg_slots, n_slides, fg_trig, fg, fg_xi, n_fg_slots, background_seconds,
                out=None):
    """spiir_rank_static: Ranker.reset + accumulate + finalize + candidates in one call whose tables sit in an array
    built into the library, for callers that cannot allocate a workspace on the device any more (all memory already
    handed out, or a late cudaMalloc would stall the streams that are filtering).  `bins` = (n_rho, n_xi, u_rho_min,
    u_rho_max, u_xi_min, u_xi_max) with n_rho * n_xi <= SPIIR_RANK_STATIC_MAX_BINS.  One array per GPU, shared by all
    calls: do not let two calls overlap on the device.  Only `out` (the caller's result buffer, n_fg_slots x 16
    bytes) is created here when it is not passed in."""
    import torch
    b = spiir_rank_bins(*bins)
    if out is None:
        out = torch.empty(n_fg_slots, 16, dtype=torch.uint8, device="cuda")
    p = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    _check(lib().spiir_rank_static(C.cast(C.byref(b), C.c_void_p), p(bg_trig), p(bg), p(bg_xi), n_bg_slots, n_slides,
                                   p(fg_trig), p(fg), p(fg_xi), n_fg_slots, float(background_seconds), p(out),
                                   _stream()))
    return out


def rank_to_numpy(out):
    return out.cpu().numpy().view(RANK_DTYPE).reshape(-1)


class FrontEnd:
    """Owns the workspace of one spiir_frontend (NEXT-4) and forwards to the C ABI."""

    def __init__(self, n_det, taps, decim=8, hop=4096, n_hist=27, gate_pad=512, out_rate_hz=2048.0, gate_threshold=8.0):
        import torch
        self._taps = np.ascontiguousarray(taps, dtype=np.float32)
        self.desc = spiir_frontend_desc(int(n_det), int(decim), len(self._taps), int(hop), int(n_hist), int(gate_pad),
                                        float(out_rate_hz), float(gate_threshold), self._taps.ctypes.data)
        n = C.c_size_t(0)
        _check(lib().spiir_frontend_workspace_bytes(C.byref(self.desc), C.byref(n)))
        self.ws = torch.empty(n.value + 256, dtype=torch.uint8, device="cuda")
        base = (self.ws.data_ptr() + 255) // 256 * 256
        self.h = C.c_void_p()
        _check(lib().spiir_frontend_init(C.byref(self.h), C.byref(self.desc), C.c_void_p(base), n, _stream()))
        self.n_det, self.hop, self.decim = int(n_det), int(hop), int(decim)

    def reset(self):
        _check(lib().spiir_frontend_reset(self.h, _stream()))

    def chunk(self, raw, out=None, psd=None):
        """raw float32 cuda [n_det][hop * decim] -> float32 cuda [n_det][hop] (spiir_frontend_chunk)."""
        import torch
        assert raw.is_cuda and raw.is_contiguous() and raw.dtype == torch.float32
        assert raw.numel() == self.n_det * self.hop * self.decim
        if out is None:
            out = torch.empty(self.n_det, self.hop, dtype=torch.float32, device="cuda")
        _check(lib().spiir_frontend_chunk(self.h, C.c_void_p(raw.data_ptr()), C.c_void_p(out.data_ptr()),
                                          C.c_void_p(psd.data_ptr()) if psd is not None else None, _stream()))
        return out

    def __del__(self):
        try:
            if getattr(self, "h", None):
                lib().spiir_frontend_free(self.h)
        except Exception:
            pass
