"""ctypes binding of ``libsft_b200.so`` (include/sft.h).  Argument marshalling only: every step
of the SFT inner product runs in the library's CUDA kernels.  There is NO CPU fallback: if the
library cannot be loaded, or no CUDA device is present, the calls raise.

Arrays may be numpy arrays (host) or torch CUDA tensors (device); all arrays of one call must
live in the same place.  torch is used only to allocate device memory and for its streams.
"""
import ctypes as C
import os
import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsft_b200.so")

MAX_CHANNELS = 4
NPARAM = 8
KERNEL = {"dirichlet": 0, "fresnel": 1}
RESPONSE = {"none": 0, "table": 1, "annual": 2}
PHASE = {"fp64": 0, "split32": 1}
MEM_HOST, MEM_DEVICE = 0, 1
PATHS = ("series0", "series1", "series2", "series3", "fresnel", "table", "table2")
EVALUATOR = {"auto": 0, "direct": 1, "table": 2}
STATUS = {0: "SFT_OK", 1: "SFT_EINVAL", 2: "SFT_ESHAPE", 3: "SFT_ENODATA", 4: "SFT_EUNSUPPORTED",
          5: "SFT_ECUDA", 6: "SFT_ENOMEM"}


class SftError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (STATUS.get(status, status), msg))
        self.status = status


class PlanDesc(C.Structure):
    """Mirror of ``sft_plan_desc``."""
    _fields_ = [("n_channels", C.c_int32), ("n_sft", C.c_int64),
                ("t_sft", C.c_double), ("fs", C.c_double), ("t0", C.c_double),
                ("k_lo", C.c_int32), ("k_hi", C.c_int32), ("K", C.c_int32),
                ("kernel", C.c_int32), ("waveform", C.c_int32), ("phase_path", C.c_int32),
                ("response", C.c_int32),
                ("f_lo", C.c_double), ("f_hi", C.c_double), ("f_ref", C.c_double),
                ("resp_period", C.c_double), ("resp_depth", C.c_double),
                ("resp_psi", C.c_double * MAX_CHANNELS), ("resp_chi", C.c_double * MAX_CHANNELS),
                ("evaluator", C.c_int32), ("include_dc", C.c_int32), ("device", C.c_int32), ("stream", C.c_void_p)]


EXPORTS = ["sft_plan_create", "sft_plan_destroy", "sft_load_data", "sft_inner_products",
           "sft_cumulative_snr", "sft_plan_sync", "sft_plan_launch_count", "sft_plan_last_kernel_ms",
           "sft_plan_set_chunk", "sft_plan_path_counts", "sft_compute_sfts", "sft_ingest_timeseries",
           "sft_tsft_rule", "sft_statistics", "sft_fstat", "sft_validity", "sft_append_sfts", "sft_estimate_psd_scale", "sft_plan_set_table_track", "sft_plan_table_bytes", "sft_last_error", "sft_version",
           "sft_measure_alu_peaks", "sft_static_setup", "sft_inner_products_static",
           "sft_plan_set_host_slab"]

_lib = None


def load_library(path=None):
    """dlopens the C-ABI library (never builds it, never falls back)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise ImportError("%s is missing: build it with `python -m paper_2502_11823_b200.build`" % path)
    lib = C.CDLL(path)
    vp, i32, i64, dbl = C.c_void_p, C.c_int32, C.c_int64, C.c_double
    lib.sft_plan_create.argtypes = [C.POINTER(PlanDesc), C.POINTER(vp)]
    lib.sft_plan_destroy.argtypes = [vp]
    lib.sft_load_data.argtypes = [vp, i32, vp, vp, vp, vp, i32]
    lib.sft_inner_products.argtypes = [vp, i64, vp, vp, vp, vp, vp, i32]
    lib.sft_cumulative_snr.argtypes = [vp, i64, vp, vp, vp, vp, i32]
    lib.sft_plan_sync.argtypes = [vp]
    lib.sft_plan_launch_count.argtypes = [vp]
    lib.sft_plan_launch_count.restype = i64
    lib.sft_plan_last_kernel_ms.argtypes = [vp]
    lib.sft_plan_last_kernel_ms.restype = dbl
    lib.sft_plan_set_chunk.argtypes = [vp, i32]
    lib.sft_plan_set_host_slab.argtypes = [vp, i64]
    lib.sft_plan_set_host_slab.restype = i32
    lib.sft_plan_path_counts.argtypes = [vp, C.POINTER(i64), i32]
    lib.sft_statistics.argtypes = [vp, i64, vp, vp, vp, vp, vp, i32]
    lib.sft_statistics.restype = i32
    lib.sft_fstat.argtypes = [vp, i64, vp, vp, vp, vp, i32]
    lib.sft_fstat.restype = i32
    lib.sft_validity.argtypes = [vp, i64, vp, dbl, vp, vp, i32]
    lib.sft_validity.restype = i32
    lib.sft_append_sfts.argtypes = [vp, i32, i64, i64, vp, vp, vp, i32]
    lib.sft_append_sfts.restype = i32
    lib.sft_estimate_psd_scale.argtypes = [i32, vp, vp, i64, i32, i32, i32, dbl, vp, i32, vp, i32]
    lib.sft_estimate_psd_scale.restype = i32
    lib.sft_plan_set_table_track.argtypes = [vp, vp, i32]
    lib.sft_plan_set_table_track.restype = i32
    lib.sft_plan_table_bytes.argtypes = [vp]
    lib.sft_plan_table_bytes.restype = i64
    lib.sft_tsft_rule.argtypes = [dbl, dbl, i32, dbl, dbl, C.POINTER(dbl), C.POINTER(dbl)]
    lib.sft_tsft_rule.restype = i32
    lib.sft_compute_sfts.argtypes = [i32, vp, vp, i64, i32, dbl, i32, i32, vp, i32]
    lib.sft_ingest_timeseries.argtypes = [vp, i32, vp, i64, vp, vp, vp, i32]
    lib.sft_measure_alu_peaks.argtypes = [i32, C.POINTER(dbl), i32]
    lib.sft_measure_alu_peaks.restype = i32
    lib.sft_static_setup.argtypes = [i32, C.POINTER(i64)]
    lib.sft_static_setup.restype = i32
    lib.sft_inner_products_static.argtypes = [vp, i64, vp, vp, vp, vp]
    lib.sft_inner_products_static.restype = i32
    lib.sft_last_error.argtypes = [vp]
    lib.sft_last_error.restype = C.c_char_p
    lib.sft_version.restype = C.c_char_p
    for f in ("sft_plan_create", "sft_plan_destroy", "sft_load_data", "sft_inner_products",
              "sft_cumulative_snr", "sft_plan_sync", "sft_plan_set_chunk", "sft_plan_path_counts",
              "sft_compute_sfts", "sft_ingest_timeseries"):
        getattr(lib, f).restype = i32
    _lib = lib
    return lib


def _is_torch(a):
    return a is not None and type(a).__module__.startswith("torch")


def _where(arrays):
    """MEM_HOST / MEM_DEVICE for a set of arrays (None entries ignored); mixing raises."""
    kinds = set()
    for a in arrays:
        if a is None:
            continue
        kinds.add(MEM_DEVICE if (_is_torch(a) and a.is_cuda) else MEM_HOST)
    if len(kinds) > 1:
        raise ValueError("all arrays of one call must be on the same side (host or device)")
    return kinds.pop() if kinds else MEM_HOST


def _ptr(a, dtype, shape=None, name="array"):
    """Checked raw pointer of a C-contiguous numpy array / torch tensor (or None)."""
    if a is None:
        return None
    if _is_torch(a):
        import torch
        want = {np.float32: torch.float32, np.float64: torch.float64, np.int32: torch.int32,
                np.complex64: torch.complex64, np.uint8: torch.uint8}[dtype]
        if a.dtype != want or not a.is_contiguous():
            raise TypeError("%s must be a contiguous %s tensor" % (name, want))
        if shape is not None and tuple(a.shape) != tuple(shape):
            raise ValueError("%s has shape %s, expected %s" % (name, tuple(a.shape), tuple(shape)))
        return C.c_void_p(a.data_ptr())
    if not isinstance(a, np.ndarray) or a.dtype != dtype or not a.flags.c_contiguous:
        raise TypeError("%s must be a C-contiguous numpy array of %s" % (name, np.dtype(dtype)))
    if shape is not None and tuple(a.shape) != tuple(shape):
        raise ValueError("%s has shape %s, expected %s" % (name, a.shape, tuple(shape)))
    return C.c_void_p(a.ctypes.data)


class Plan:
    """``sft_plan`` handle.  ``desc`` is a dict with the fields of ``sft_plan_desc``; ``kernel`` and
    ``response`` may be given by name, ``pn1`` (0/1) is accepted for ``waveform``."""

    def __init__(self, desc=None, device=0, stream=None, **kw):
        d = dict(desc or {})
        d.update(kw)
        self.lib = load_library()
        pd = PlanDesc()
        pd.n_channels = int(d["n_channels"])
        pd.n_sft = int(d["n_sft"])
        pd.t_sft, pd.fs, pd.t0 = float(d["t_sft"]), float(d["fs"]), float(d.get("t0", 0.0))
        pd.k_lo, pd.k_hi, pd.K = int(d["k_lo"]), int(d["k_hi"]), int(d["K"])
        k = d.get("kernel", "fresnel")
        pd.kernel = KERNEL[k] if isinstance(k, str) else int(k)
        pd.waveform = int(d.get("waveform", d.get("pn1", 0)))
        ph = d.get("phase_path", "fp64")
        pd.phase_path = PHASE[ph] if isinstance(ph, str) else int(ph)
        r = d.get("response", "none")
        pd.response = RESPONSE[r] if isinstance(r, str) else int(r)
        pd.f_lo = float(d.get("f_lo", 0.0))
        pd.f_hi = float(min(d.get("f_hi", 1e300), 1e300))
        pd.f_ref = float(d.get("f_ref", 1.0))
        pd.resp_period = float(d.get("resp_period", 31557600.0))
        pd.resp_depth = float(d.get("resp_depth", 0.0))
        for i, v in enumerate(d.get("resp_psi", ())):
            pd.resp_psi[i] = float(v)
        for i, v in enumerate(d.get("resp_chi", ())):
            pd.resp_chi[i] = float(v)
        ev = d.get("evaluator", "auto")
        pd.evaluator = EVALUATOR[ev] if isinstance(ev, str) else int(ev)
        pd.include_dc = int(d.get("include_dc", 0))
        pd.device = int(device)
        pd.stream = C.c_void_p(int(stream)) if stream else None
        self.desc = pd
        self.n_channels, self.n_sft, self.nb = pd.n_channels, pd.n_sft, pd.k_hi - pd.k_lo
        h = C.c_void_p()
        st = self.lib.sft_plan_create(C.byref(pd), C.byref(h))
        if st != 0:
            raise SftError(st, self.lib.sft_last_error(None).decode())
        self._h = h

    # -- helpers -----------------------------------------------------------------------------
    def _check(self, st):
        if st != 0:
            raise SftError(st, self.lib.sft_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self.lib.sft_plan_destroy(self._h)
            self._h = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    # -- the C ABI ---------------------------------------------------------------------------
    def load_data(self, channel, sft_bins, psd_scale, psd_shape=None, response=None):
        """``sft_load_data``: complex64 [n_sft][nb] bins, float64 [n_sft] scale, float64 [nb] shape."""
        mem = _where([sft_bins, psd_scale, psd_shape, response])
        self._check(self.lib.sft_load_data(
            self._h, int(channel),
            _ptr(sft_bins, np.complex64, (self.n_sft, self.nb), "sft_bins"),
            _ptr(psd_scale, np.float64, (self.n_sft,), "psd_scale"),
            _ptr(psd_shape, np.float64, (self.nb,), "psd_shape"),
            _ptr(response, np.complex64, (self.n_sft,), "response"), mem))

    def append_sfts(self, channel, first_sft, sft_bins, psd_scale, response=None):
        """``sft_append_sfts``: replaces slots [first_sft, first_sft + n_new) of a loaded channel in place."""
        n_new = int(sft_bins.shape[0])
        mem = _where([sft_bins, psd_scale, response])
        self._check(self.lib.sft_append_sfts(
            self._h, int(channel), int(first_sft), n_new, _ptr(sft_bins, np.complex64, (n_new, self.nb), "sft_bins"),
            _ptr(psd_scale, np.float64, (n_new,), "psd_scale"), _ptr(response, np.complex64, (n_new,), "response"), mem))

    def ingest_timeseries(self, channel, x, psd_scale=None, psd_shape=None, response=None):
        """``sft_ingest_timeseries``: float64 strain series [>= n_sft * n] instead of precomputed SFT bins."""
        mem = _where([x, psd_scale, psd_shape, response])
        ns = int(x.shape[0])
        self._check(self.lib.sft_ingest_timeseries(
            self._h, int(channel), _ptr(x, np.float64, (ns,), "x"), ns,
            _ptr(psd_scale, np.float64, (self.n_sft,), "psd_scale"),
            _ptr(psd_shape, np.float64, (self.nb,), "psd_shape"),
            _ptr(response, np.complex64, (self.n_sft,), "response"), mem))

    def inner_products(self, params, xh, hh, xh_im=None, kc_out=None):
        """``sft_inner_products`` into caller-allocated outputs."""
        nT = int(params.shape[0])
        mem = _where([params, xh, hh, xh_im, kc_out])
        self._check(self.lib.sft_inner_products(
            self._h, nT, _ptr(params, np.float64, (nT, NPARAM), "params"),
            _ptr(xh, np.float64, (nT,), "xh"), _ptr(hh, np.float64, (nT,), "hh"),
            _ptr(xh_im, np.float64, (nT,), "xh_im"),
            _ptr(kc_out, np.int32, (nT, self.n_channels, self.n_sft), "kc_out"), mem))

    def inner_products_static(self, params, xh, hh, xh_im=None):
        """``sft_inner_products_static``: the allocation-free call (device tensors only, at most STATIC_MAX_TEMPLATES rows)."""
        nT = int(params.shape[0])
        if _where([params, xh, hh, xh_im]) != MEM_DEVICE:
            raise ValueError("sft_inner_products_static takes device tensors only")
        self._check(self.lib.sft_inner_products_static(
            self._h, nT, _ptr(params, np.float64, (nT, NPARAM), "params"),
            _ptr(xh, np.float64, (nT,), "xh"), _ptr(hh, np.float64, (nT,), "hh"),
            _ptr(xh_im, np.float64, (nT,), "xh_im")))

    def cumulative_snr(self, params, snr=None, cum_xh=None, cum_hh=None):
        """``sft_cumulative_snr`` into caller-allocated float32 [nT][n_sft] outputs."""
        nT = int(params.shape[0])
        mem = _where([params, snr, cum_xh, cum_hh])
        shp = (nT, self.n_sft)
        self._check(self.lib.sft_cumulative_snr(
            self._h, nT, _ptr(params, np.float64, (nT, NPARAM), "params"),
            _ptr(snr, np.float32, shp, "snr"), _ptr(cum_xh, np.float32, shp, "cum_xh"),
            _ptr(cum_hh, np.float32, shp, "cum_hh"), mem))

    def statistics(self, xh, xh_im, hh, loglike=None, rho2_phase_max=None):
        """``sft_statistics``: log-likelihood and phase-maximised statistic from the inner products."""
        nT = int(xh.shape[0])
        mem = _where([xh, xh_im, hh, loglike, rho2_phase_max])
        self._check(self.lib.sft_statistics(
            self._h, nT, _ptr(xh, np.float64, (nT,), "xh"), _ptr(xh_im, np.float64, (nT,), "xh_im"),
            _ptr(hh, np.float64, (nT,), "hh"), _ptr(loglike, np.float64, (nT,), "loglike"),
            _ptr(rho2_phase_max, np.float64, (nT,), "rho2_phase_max"), mem))

    def fstat(self, params, twoF, xnu=None, mnu=None):
        """``sft_fstat``: 2F [nT] and optionally ([x,h_nu]) [4][nT], (([h_0,h_0]), ([h_1,h_1]), ([h_0,h_1])) [3][nT]."""
        nT = int(params.shape[0])
        mem = _where([params, twoF, xnu, mnu])
        self._check(self.lib.sft_fstat(
            self._h, nT, _ptr(params, np.float64, (nT, NPARAM), "params"), _ptr(twoF, np.float64, (nT,), "twoF"),
            _ptr(xnu, np.float64, (4, nT), "xnu"), _ptr(mnu, np.float64, (3, nT), "mnu"), mem))

    def validity(self, params, delta_max, delta_eff=None, flags=None):
        """``sft_validity``: delta_eff [nT] float64 and / or flags [nT] uint8 (delta_eff > delta_max)."""
        nT = int(params.shape[0])
        mem = _where([params, delta_eff, flags])
        self._check(self.lib.sft_validity(
            self._h, nT, _ptr(params, np.float64, (nT, NPARAM), "params"), float(delta_max),
            _ptr(delta_eff, np.float64, (nT,), "delta_eff"), _ptr(flags, np.uint8, (nT,), "flags"), mem))

    def set_table_track(self, fiducial_params, half_width):
        """``sft_plan_set_table_track``: tables only along the track of ``fiducial_params`` (+- half_width bins); None = full."""
        fp = None if fiducial_params is None else np.ascontiguousarray(fiducial_params, dtype=np.float64)
        self._check(self.lib.sft_plan_set_table_track(self._h, _ptr(fp, np.float64, (NPARAM,), "fiducial_params"), int(half_width)))

    def table_bytes(self):
        return int(self.lib.sft_plan_table_bytes(self._h))

    def sync(self):
        self._check(self.lib.sft_plan_sync(self._h))

    def launch_count(self):
        return int(self.lib.sft_plan_launch_count(self._h))

    def last_kernel_ms(self):
        return float(self.lib.sft_plan_last_kernel_ms(self._h))

    def set_chunk(self, sfts_per_unit):
        self._check(self.lib.sft_plan_set_chunk(self._h, int(sfts_per_unit)))

    def set_host_slab(self, templates_per_slab):
        """``sft_plan_set_host_slab``: templates per slab of ``cumulative_snr`` with host outputs (0 = automatic)."""
        self._check(self.lib.sft_plan_set_host_slab(self._h, int(templates_per_slab)))

    def path_counts(self):
        """``sft_plan_path_counts``: dict path name -> active pairs of the last call that had kc_out."""
        out = (C.c_int64 * 7)()
        self._check(self.lib.sft_plan_path_counts(self._h, out, 7))
        return dict(zip(PATHS, [int(v) for v in out]))


def plan_from_workload(w, device=0, stream=None, **override):
    """Creates a plan for a ``workloads.Workload`` and loads all its channels (host arrays)."""
    d = dict(w.desc)
    d.update(override)
    track = d.pop("table_track", None)               # (fiducial parameter row, half width in bins) or None
    plan = Plan(d, device=device, stream=stream)
    if track is not None:
        plan.set_table_track(track[0], track[1])
    for c in range(plan.n_channels):
        resp = None if w.response is None else np.ascontiguousarray(w.response[c], dtype=np.complex64)
        plan.load_data(c, np.ascontiguousarray(w.bins[c], dtype=np.complex64),
                       np.ascontiguousarray(w.psd_scale[c], dtype=np.float64),
                       np.ascontiguousarray(w.psd_shape[c], dtype=np.float64), resp)
    return plan


def tsft_rule(m_chirp, eta, f_max, delta, pn1=1):
    """``sft_tsft_rule``: (T_SFT [s], max fddot [Hz/s^2]) of Eq.(34) for this library's waveform.  No GPU needed."""
    lib = load_library()
    t, fdd = C.c_double(), C.c_double()
    st = lib.sft_tsft_rule(float(m_chirp), float(eta), int(pn1), float(f_max), float(delta), C.byref(t), C.byref(fdd))
    if st != 0:
        raise SftError(st, lib.sft_last_error(None).decode())
    return t.value, fdd.value


def compute_sfts(x, n_sft, n, dt, k_lo, k_hi, bins, device=0, stream=None):
    """``sft_compute_sfts``: band-limited data SFTs of a float64 series into complex64 ``bins`` [n_sft][k_hi-k_lo]."""
    lib = load_library()
    mem = _where([x, bins])
    if x is None or len(x.shape) != 1 or int(x.shape[0]) < int(n_sft) * int(n):
        raise ValueError("x must be a 1-D series of at least n_sft * n = %d samples" % (int(n_sft) * int(n)))
    st = lib.sft_compute_sfts(int(device), C.c_void_p(int(stream)) if stream else None,
                              _ptr(x, np.float64, None, "x"), int(n_sft), int(n), float(dt), int(k_lo), int(k_hi),
                              _ptr(bins, np.complex64, (int(n_sft), int(k_hi) - int(k_lo)), "bins"), mem)
    if st != 0:
        raise SftError(st, lib.sft_last_error(None).decode())


def estimate_psd_scale(sft_bins, k_lo, n_samp, t_sft, psd_shape=None, half_window=0, out=None, device=0, stream=None):
    """``sft_estimate_psd_scale``: per-SFT noise level [n_sft] (float64) from complex64 ``sft_bins`` [n_sft][nb]."""
    lib = load_library()
    n_sft, nb = int(sft_bins.shape[0]), int(sft_bins.shape[1])
    if out is None:
        if _is_torch(sft_bins):
            import torch
            out = torch.empty(n_sft, dtype=torch.float64, device=sft_bins.device)
        else:
            out = np.empty(n_sft, dtype=np.float64)
    mem = _where([sft_bins, psd_shape, out])
    st = lib.sft_estimate_psd_scale(int(device), C.c_void_p(int(stream)) if stream else None,
                                    _ptr(sft_bins, np.complex64, (n_sft, nb), "sft_bins"), n_sft, int(k_lo), int(k_lo) + nb,
                                    int(n_samp), float(t_sft), _ptr(psd_shape, np.float64, (nb,), "psd_shape"), int(half_window),
                                    _ptr(out, np.float64, (n_sft,), "psd_scale"), mem)
    if st != 0:
        raise SftError(st, lib.sft_last_error(None).decode())
    return out


def measure_alu_peaks(device=0):
    """``sft_measure_alu_peaks``: dict of measured pipe rates in Gop/s (lane operations)."""
    lib = load_library()
    out = (C.c_double * 6)()
    st = lib.sft_measure_alu_peaks(int(device), out, 6)
    if st != 0:
        raise SftError(st, lib.sft_last_error(None).decode())
    return dict(zip(("ffma", "ffma2", "dfma", "mufu_rcp", "ffma_mufu_mix", "table_mix_ipc"), [float(v) for v in out]))


STATIC_MAX_TEMPLATES = 4096          # SFT_STATIC_MAX_TEMPLATES of include/sft.h


def static_setup(device=0):
    """``sft_static_setup``: resolves the library's static scratch on ``device``; returns its size in bytes."""
    lib = load_library()
    n = C.c_int64(0)
    st = lib.sft_static_setup(int(device), C.byref(n))
    if st != 0:
        raise SftError(st, lib.sft_last_error(None).decode())
    return int(n.value)


def version():
    return load_library().sft_version().decode()
