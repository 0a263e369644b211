"""Thin ctypes binding of libdedisp_b200.so (include/dedisp.h): argument marshalling only.

PyTorch is used for device memory and streams; every arithmetic step runs in the library's CUDA
kernels.  There is no fallback: if the shared library is missing or a call fails this raises.
"""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdedisp_b200.so")

OK, EINVAL, ENOMEM, ECUDA, ESHAPE, ESTATE, ELIMIT = range(7)
F32, U8 = 0, 1
KERNEL_AUTO, KERNEL_NAIVE, KERNEL_DIRECT, KERNEL_WINDOW, KERNEL_LONG = range(5)

_c = ctypes
_vp, _i64, _int, _dbl = _c.c_void_p, _c.c_int64, _c.c_int, _c.c_double
_SIGS = {
    "dedisp_plan_create": (_int, [_c.POINTER(_vp), _int, _dbl, _dbl, _dbl, _c.POINTER(_dbl), _int, _int, _int]),
    "dedisp_plan_destroy": (_int, [_vp]),
    "dedisp_plan_max_delay": (_i64, [_vp]),
    "dedisp_plan_nchans": (_int, [_vp]),
    "dedisp_plan_ndm": (_int, [_vp]),
    "dedisp_plan_nsub": (_int, [_vp]),
    "dedisp_plan_nfine": (_int, [_vp]),
    "dedisp_plan_get_shifts": (_int, [_vp, _vp]),
    "dedisp_plan_get_subband_shifts": (_int, [_vp, _vp, _vp, _vp, _vp]),
    "dedisp_plan_set_kernel": (_int, [_vp, _int]),
    "dedisp_plan_resolved_kernel": (_int, [_vp, _int]),
    "dedisp_plan_last_kernel": (_int, [_vp]),
    "dedisp_plan_window_info": (_int, [_vp, _vp]),
    "dedisp_plan_set_window_geometry": (_int, [_vp, _int, _int, _int, _int]),
    "dedisp_plan_reserve": (_int, [_vp, _int, _i64, _int]),
    "dedisp_plan_scratch_bytes": (_i64, [_vp, _i64, _int]),
    "dedisp_execute": (_int, [_vp, _vp, _vp, _int, _i64, _i64, _i64, _int, _vp]),
    "dedisp_execute_host": (_int, [_vp, _vp, _vp, _int, _i64, _int, _vp]),
    "dedisp_stream_create": (_int, [_c.POINTER(_vp), _vp, _int, _i64, _int]),
    "dedisp_stream_push": (_int, [_vp, _vp, _vp, _vp]),
    "dedisp_stream_push_host": (_int, [_vp, _vp, _vp, _vp]),
    "dedisp_stream_reset": (_int, [_vp, _vp]),
    "dedisp_stream_destroy": (_int, [_vp]),
    "dedisp_plan_max_chunk": (_i64, [_vp, _int, _i64, _int]),
    "dedisp_plan_last_launches": (_int, [_vp]),
    "dedisp_plan_set_timing": (_int, [_vp, _int]),
    "dedisp_plan_last_kernel_ms": (_int, [_vp, _vp]),
    "dedisp_plan_last_stage_ms": (_int, [_vp, _vp]),
    "dedisp_plan_detect": (_int, [_vp, _vp, _int, _i64, _i64, _int, _dbl, _vp, _i64, _vp, _vp]),
    "dedisp_detect_static": (_int, [_vp, _int, _int, _i64, _i64, _int, _dbl, _vp, _i64, _vp, _vp]),
    "dedisp_detect_static_max_slots": (_i64, []),
    "dedisp_execute_detect": (_int, [_vp, _vp, _vp, _int, _i64, _i64, _i64, _int, _dbl, _vp, _i64, _vp, _vp]),
    "dedisp_plan_copy_host_output": (_int, [_vp, _vp, _i64, _vp]),
    "dedisp_execute_detect_host": (_int, [_vp, _vp, _int, _i64, _int, _dbl, _vp, _i64, _vp, _vp]),
    "dedisp_power_corner_turn": (_int, [_vp, _vp, _int, _i64, _i64, _i64, _vp]),
    "dedisp_bin": (_int, [_vp, _vp, _i64, _i64, _i64, _i64, _int, _vp]),
    "dedisp_survey_create": (_int, [_c.POINTER(_vp), _int, _dbl, _dbl, _dbl, _int, _vp, _int]),
    "dedisp_survey_destroy": (_int, [_vp]),
    "dedisp_survey_npass": (_int, [_vp]),
    "dedisp_survey_max_delay": (_i64, [_vp]),
    "dedisp_survey_pass_plan": (_vp, [_vp, _int]),
    "dedisp_survey_out_layout": (_int, [_vp, _i64, _int, _vp, _vp, _vp, _vp]),
    "dedisp_survey_reserve": (_int, [_vp, _i64, _int]),
    "dedisp_survey_execute": (_int, [_vp, _vp, _vp, _i64, _i64, _int, _vp]),
    "dedisp_survey_last_launches": (_int, [_vp]),
    "dedisp_fadd_microbench": (_int, [_int, _int, _int, _vp, _vp, _vp, _vp]),
    "dedisp_strerror": (_c.c_char_p, [_int]),
    "dedisp_version": (_c.c_char_p, []),
}
EXPORTS = tuple(_SIGS)
_lib = None


class DedispError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        msg = lib().dedisp_strerror(status).decode()
        super().__init__("%s: %s (status %d)" % (where, msg, status))


def lib():
    """Loads the C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("%s is missing: run `python -m paper_1107_2516_b200.build` "
                               "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in _SIGS.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _check(status, where):
    if status != OK:
        raise DedispError(status, where)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _dtype_of(t):
    import torch
    if t.dtype == torch.float32:
        return F32, torch.float32
    if t.dtype == torch.uint8:
        return U8, torch.int32
    raise TypeError("input must be float32 or uint8")


class Plan:
    """dedisp_plan_create(nchans, f_top, df, t_samp, dm_list[, nsub, nfine])."""

    def __init__(self, nchans, f_top_mhz, df_mhz, t_samp_ms, dm_list, nsub=0, nfine=0):
        dm = np.ascontiguousarray(dm_list, dtype=np.float64)
        h = _vp()
        _check(lib().dedisp_plan_create(ctypes.byref(h), int(nchans), float(f_top_mhz), float(df_mhz),
                                        float(t_samp_ms), dm.ctypes.data_as(_c.POINTER(_dbl)),
                                        int(dm.size), int(nsub), int(nfine)), "dedisp_plan_create")
        self._h = h
        self.nchans, self.ndm, self.nsub, self.nfine = int(nchans), int(dm.size), int(nsub), int(nfine)
        self._reserved = {}

    def reserve(self, dtype, nsamp_out, nbeams=1):
        """dedisp_plan_reserve: tables onto the current device, scratch for this shape (blocking)."""
        _check(lib().dedisp_plan_reserve(self._h, int(dtype), int(nsamp_out), int(nbeams)), "dedisp_plan_reserve")
        # the library's buffers only grow and their sizes rise with both arguments, so a shape is covered
        # exactly when ONE earlier reserve had both at least as large (not the maxima taken separately)
        self._reserved.setdefault(int(dtype), []).append((int(nsamp_out), int(nbeams)))

    def _ensure_reserved(self, dtype, nsamp_out, nbeams):
        # execute / detect never allocate (include/dedisp.h): the binding reserves the first time a
        # shape is seen, which keeps `plan.execute(x, n)` a one-liner
        if not any(n >= nsamp_out and b >= nbeams for n, b in self._reserved.get(int(dtype), ())):
            self.reserve(dtype, int(nsamp_out), int(nbeams))

    def close(self):
        if getattr(self, "_h", None):
            _check(lib().dedisp_plan_destroy(self._h), "dedisp_plan_destroy")
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def max_delay(self):
        return int(lib().dedisp_plan_max_delay(self._h))

    def shifts(self):
        out = np.empty((self.ndm, self.nchans), dtype=np.int32)
        _check(lib().dedisp_plan_get_shifts(self._h, out.ctypes.data), "dedisp_plan_get_shifts")
        return out

    def subband_shifts(self):
        nco = self.ndm // self.nfine if self.nfine else 0
        s1 = np.empty((nco, self.nchans), dtype=np.int32)
        s2 = np.empty((self.ndm, max(self.nsub, 1)), dtype=np.int32)
        nom = np.empty(nco, dtype=np.float64)
        m2 = np.empty(nco, dtype=np.int32)
        _check(lib().dedisp_plan_get_subband_shifts(self._h, s1.ctypes.data, s2.ctypes.data,
                                                    nom.ctypes.data, m2.ctypes.data),
               "dedisp_plan_get_subband_shifts")
        return s1, s2, nom, m2

    def set_kernel(self, kernel):
        _check(lib().dedisp_plan_set_kernel(self._h, int(kernel)), "dedisp_plan_set_kernel")
        self._reserved = {}          # the scratch a shape needs depends on the kernel

    def set_window_geometry(self, T, G, NT, D):
        _check(lib().dedisp_plan_set_window_geometry(self._h, int(T), int(G), int(NT), int(D)),
               "dedisp_plan_set_window_geometry")

    def resolved_kernel(self, dtype=F32):
        return int(lib().dedisp_plan_resolved_kernel(self._h, int(dtype)))

    def window_info(self):
        """dedisp_plan_window_info as a dict (geometry of the register-window kernel)."""
        a = np.zeros(14, dtype=np.int64)
        _check(lib().dedisp_plan_window_info(self._h, a.ctypes.data), "dedisp_plan_window_info")
        keys = ("ok", "Hb", "kmax", "lmax", "ntile_dm", "slots", "rows_per_block", "nband", "T", "G", "NT", "D",
                "stage_channels", "ring_stages")
        return dict(zip(keys, (int(v) for v in a)))

    def scratch_bytes(self, nsamp_out, nbeams=1):
        return int(lib().dedisp_plan_scratch_bytes(self._h, int(nsamp_out), int(nbeams)))

    def max_chunk(self, dtype, mem_bytes, nbeams=1):
        return int(lib().dedisp_plan_max_chunk(self._h, int(dtype), int(mem_bytes), int(nbeams)))

    def set_timing(self, on=True):
        _check(lib().dedisp_plan_set_timing(self._h, int(bool(on))), "dedisp_plan_set_timing")

    def last_kernel_ms(self):
        """Device time of the dominant kernel(s) of the last execute (needs set_timing(True))."""
        v = ctypes.c_float(0.0)
        _check(lib().dedisp_plan_last_kernel_ms(self._h, ctypes.addressof(v)), "dedisp_plan_last_kernel_ms")
        return float(v.value)

    def last_stage_ms(self):
        """Subband plans: (stage 1 ms, stage 2 ms) of the last execute (needs set_timing(True))."""
        v = (ctypes.c_float * 2)()
        _check(lib().dedisp_plan_last_stage_ms(self._h, ctypes.addressof(v)), "dedisp_plan_last_stage_ms")
        return float(v[0]), float(v[1])

    @property
    def last_launches(self):
        return int(lib().dedisp_plan_last_launches(self._h))

    @property
    def last_kernel(self):
        """dedisp_plan_last_kernel: the kernel the last execute / push really ran (KERNEL_*), -1 before any."""
        return int(lib().dedisp_plan_last_kernel(self._h))

    def execute(self, x, nsamp_out, out=None, stream=None):
        """x: CUDA tensor [nchans][n_in] or [nbeams][nchans][n_in] (float32 or uint8), last dim
        contiguous, row stride a multiple of 16 bytes.  Returns out [.. ndm][nsamp_out]."""
        import torch
        if not x.is_cuda:
            raise RuntimeError("dedisp_execute needs a CUDA tensor (there is no CPU fallback)")
        dt, odt = _dtype_of(x)
        x3 = x if x.dim() == 3 else x.unsqueeze(0)
        nb, nch, _ = x3.shape
        if nch != self.nchans or x3.stride(2) != 1 or (nb > 1 and x3.stride(0) != nch * x3.stride(1)):
            raise DedispError(ESHAPE, "dedisp_execute")
        if out is None:
            ostride = (int(nsamp_out) + 3) // 4 * 4
            buf = torch.empty((nb, self.ndm, ostride), dtype=odt, device=x.device)
            out3 = buf[:, :, :int(nsamp_out)]
        else:
            out3 = out if out.dim() == 3 else out.unsqueeze(0)
            if out3.dtype != odt or out3.stride(2) != 1 or out3.shape[1] != self.ndm or \
                    (nb > 1 and out3.stride(0) != self.ndm * out3.stride(1)):
                raise DedispError(ESHAPE, "dedisp_execute")
        self._ensure_reserved(dt, int(nsamp_out), int(nb))
        _check(lib().dedisp_execute(self._h, x3.data_ptr(), out3.data_ptr(), dt, int(nsamp_out),
                                    int(x3.stride(1)), int(out3.stride(1)), int(nb), _stream_ptr(stream)),
               "dedisp_execute")
        return out3 if x.dim() == 3 else out3[0]

    def detect(self, out, nsigma, capacity=1 << 20, stream=None):
        """dedisp_plan_detect on a CUDA tensor out[(nbeams,) ndm, n] as returned by execute.  Returns
        (results, events): per-beam dicts {mean, sigma, threshold, count} and numpy record arrays
        (t, dm, value) of the stored events (unordered)."""
        import torch
        o = out if out.dim() == 3 else out[None]
        assert o.is_cuda and o.stride(2) == 1 and o.shape[1] == self.ndm and o.stride(0) == o.stride(1) * self.ndm
        dt = F32 if o.dtype == torch.float32 else U8
        nb = o.shape[0]
        self._ensure_reserved(dt, 0, int(nb))
        ev = torch.zeros((nb, capacity, 4), dtype=torch.int32, device=o.device)     # 16-byte records
        res = torch.zeros((nb, 4), dtype=torch.float64, device=o.device)            # 32-byte records
        _check(lib().dedisp_plan_detect(self._h, o.data_ptr(), dt, int(o.shape[2]), int(o.stride(1)), int(nb),
                                        float(nsigma), ev.data_ptr(), int(capacity), res.data_ptr(),
                                        _stream_ptr(stream)), "dedisp_plan_detect")
        rh = res.cpu().numpy()
        counts = rh[:, 3].copy().view(np.int64)
        results = [dict(mean=float(rh[b, 0]), sigma=float(rh[b, 1]), threshold=float(rh[b, 2]), count=int(counts[b]))
                   for b in range(nb)]
        rec = np.dtype([("t", np.int64), ("dm", np.int32), ("value", np.float32)])
        events = [ev[b, :min(int(counts[b]), capacity)].cpu().numpy().view(rec).reshape(-1) for b in range(nb)]
        return results, events

    _REC = np.dtype([("t", np.int64), ("dm", np.int32), ("value", np.float32)])

    def execute_detect(self, x, nsamp_out, nsigma, capacity=1 << 20, out=None, stream=None):
        """dedisp_execute_detect: de-disperse x (as execute) and detect events in one call.  Returns
        (out, results, events) with results / events as detect returns them."""
        import torch
        if not x.is_cuda:
            raise RuntimeError("dedisp_execute_detect needs a CUDA tensor (there is no CPU fallback)")
        dt, odt = _dtype_of(x)
        x3 = x if x.dim() == 3 else x.unsqueeze(0)
        nb, nch, _ = x3.shape
        if nch != self.nchans or x3.stride(2) != 1 or (nb > 1 and x3.stride(0) != nch * x3.stride(1)):
            raise DedispError(ESHAPE, "dedisp_execute_detect")
        if out is None:
            ostride = (int(nsamp_out) + 3) // 4 * 4
            out3 = torch.empty((nb, self.ndm, ostride), dtype=odt, device=x.device)[:, :, :int(nsamp_out)]
        else:
            out3 = out if out.dim() == 3 else out.unsqueeze(0)
        self._ensure_reserved(dt, int(nsamp_out), int(nb))
        ev = torch.zeros((nb, capacity, 4), dtype=torch.int32, device=x.device)
        res = torch.zeros((nb, 4), dtype=torch.float64, device=x.device)
        _check(lib().dedisp_execute_detect(self._h, x3.data_ptr(), out3.data_ptr(), dt, int(nsamp_out),
                                           int(x3.stride(1)), int(out3.stride(1)), int(nb), float(nsigma),
                                           ev.data_ptr(), int(capacity), res.data_ptr(), _stream_ptr(stream)),
               "dedisp_execute_detect")
        rh = res.cpu().numpy()
        counts = rh[:, 3].copy().view(np.int64)
        results = [dict(mean=float(rh[b, 0]), sigma=float(rh[b, 1]), threshold=float(rh[b, 2]), count=int(counts[b]))
                   for b in range(nb)]
        events = [ev[b, :min(int(counts[b]), capacity)].cpu().numpy().view(self._REC).reshape(-1) for b in range(nb)]
        return (out3 if x.dim() == 3 else out3[0]), results, events

    def execute_detect_host(self, x, nsamp_out, nsigma, capacity=1 << 20, events=None, stream=None):
        """dedisp_execute_detect_host: x numpy / CPU tensor [nbeams][nchans][nsamp_out+max_delay]; only the
        events and the statistics come back.  `events`: optional (pinned) CPU tensor / array of
        nbeams*capacity*16 bytes to receive the triplets.  Returns (results, events)."""
        xa = x.numpy() if hasattr(x, "numpy") else np.asarray(x)
        xa = xa if xa.ndim == 3 else xa[None]
        assert xa.flags.c_contiguous and xa.shape[1] == self.nchans and xa.shape[2] == nsamp_out + self.max_delay
        dt = F32 if xa.dtype == np.float32 else U8
        nb = xa.shape[0]
        if events is None:
            events = np.zeros((nb, capacity), dtype=self._REC)
        ea = events.numpy() if hasattr(events, "numpy") else events
        res = np.zeros((nb, 4), dtype=np.float64)
        _check(lib().dedisp_execute_detect_host(self._h, xa.ctypes.data, dt, int(nsamp_out), int(nb), float(nsigma),
                                                ea.ctypes.data, int(capacity), res.ctypes.data, _stream_ptr(stream)),
               "dedisp_execute_detect_host")
        counts = res[:, 3].copy().view(np.int64)
        results = [dict(mean=float(res[b, 0]), sigma=float(res[b, 1]), threshold=float(res[b, 2]), count=int(counts[b]))
                   for b in range(nb)]
        ev = ea.view(np.uint8).reshape(nb, -1)[:, :capacity * 16].view(self._REC).reshape(nb, capacity)
        return results, [ev[b, :min(int(counts[b]), capacity)] for b in range(nb)]

    def host_output(self, nbeams, nsamp_out, dtype=F32, stream=None):
        """dedisp_plan_copy_host_output: the de-dispersed buffer of the last execute_host /
        execute_detect_host call as a CUDA tensor [nbeams][ndm][nsamp_out] (a copy)."""
        import torch
        t = torch.empty((int(nbeams), self.ndm, int(nsamp_out)), dtype=torch.float32 if dtype == F32 else torch.int32,
                        device="cuda")
        _check(lib().dedisp_plan_copy_host_output(self._h, t.data_ptr(), t.numel() * 4, _stream_ptr(stream)),
               "dedisp_plan_copy_host_output")
        return t

    def execute_host(self, x, nsamp_out, out=None, stream=None):
        """x: numpy / CPU tensor [nbeams][nchans][nsamp_out+max_delay] dense; returns numpy out."""
        xa = x.numpy() if hasattr(x, "numpy") else np.asarray(x)
        xa = xa if xa.ndim == 3 else xa[None]
        assert xa.flags.c_contiguous and xa.shape[1] == self.nchans
        assert xa.shape[2] == nsamp_out + self.max_delay
        dt = F32 if xa.dtype == np.float32 else U8
        if out is None:
            out = np.empty((xa.shape[0], self.ndm, nsamp_out), dtype=np.float32 if dt == F32 else np.int32)
        oa = out.numpy() if hasattr(out, "numpy") else out
        _check(lib().dedisp_execute_host(self._h, xa.ctypes.data, oa.ctypes.data, dt, int(nsamp_out),
                                         int(xa.shape[0]), _stream_ptr(stream)), "dedisp_execute_host")
        return out


def detect_static(out, nsigma, capacity=1 << 20, events=None, results=None, stream=None):
    """dedisp_detect_static: Plan.detect's numbers without a plan and without any allocation inside the
    library -- for a real-time loop that cannot take cudaMalloc's device-wide stall, or a process whose
    GPU memory is already fully claimed.  The per-block sums live in a fixed 296 KiB array inside the
    library (shared by all calls on a GPU: do not overlap two of them), so the shape is limited to
    nbeams * min(ndm, 1184) <= detect_static_max_slots(); beyond that DedispError(ELIMIT).

    out is a CUDA tensor [(nbeams,) ndm, n] as returned by execute.  Pass preallocated `events`
    (int32 [nbeams, capacity, 4]) and `results` (float64 [nbeams, 4]) CUDA tensors to keep this wrapper
    from allocating as well; by default torch allocates them.  Returns (results, events) as Plan.detect."""
    import torch
    o = out if out.dim() == 3 else out[None]
    assert o.is_cuda and o.stride(2) == 1 and o.stride(0) == o.stride(1) * o.shape[1]
    dt = F32 if o.dtype == torch.float32 else U8
    nb, ndm = int(o.shape[0]), int(o.shape[1])
    ev = events if events is not None else torch.zeros((nb, capacity, 4), dtype=torch.int32, device=o.device)
    res = results if results is not None else torch.zeros((nb, 4), dtype=torch.float64, device=o.device)
    assert ev.is_contiguous() and ev.dtype == torch.int32 and tuple(ev.shape) == (nb, capacity, 4)
    assert res.is_contiguous() and res.dtype == torch.float64 and tuple(res.shape) == (nb, 4)
    _check(lib().dedisp_detect_static(o.data_ptr(), dt, ndm, int(o.shape[2]), int(o.stride(1)), nb, float(nsigma),
                                      ev.data_ptr(), int(capacity), res.data_ptr(), _stream_ptr(stream)),
           "dedisp_detect_static")
    rh = res.cpu().numpy()
    counts = rh[:, 3].copy().view(np.int64)
    out_res = [dict(mean=float(rh[b, 0]), sigma=float(rh[b, 1]), threshold=float(rh[b, 2]), count=int(counts[b]))
               for b in range(nb)]
    out_ev = [ev[b, :min(int(counts[b]), capacity)].cpu().numpy().view(Plan._REC).reshape(-1) for b in range(nb)]
    return out_res, out_ev


def detect_static_max_slots():
    """dedisp_detect_static_max_slots: (beam, block) slots of the fixed scratch array."""
    return int(lib().dedisp_detect_static_max_slots())


def power_corner_turn(volt, out=None, stream=None):
    """dedisp_power_corner_turn: volt CUDA complex64 [nsamp][nchans] (row stride free) -> float32
    [nchans][nsamp] in the de-disperser's layout (row stride padded to 16 elements)."""
    import torch
    if not volt.is_cuda or volt.dtype != torch.complex64 or volt.dim() != 2 or volt.stride(1) != 1:
        raise DedispError(ESHAPE, "dedisp_power_corner_turn")
    nsamp, nchans = volt.shape
    if out is None:
        stride = (nsamp + 15) // 16 * 16
        out = torch.empty((nchans, stride), dtype=torch.float32, device=volt.device)[:, :nsamp]
    _check(lib().dedisp_power_corner_turn(volt.data_ptr(), out.data_ptr(), int(nchans), int(nsamp),
                                          int(volt.stride(0)), int(out.stride(0)), _stream_ptr(stream)),
           "dedisp_power_corner_turn")
    return out


def bin_samples(x, nb, stream=None):
    """dedisp_bin: x CUDA float32 [..., n] (last dim contiguous, uniform row stride) -> [..., n // nb]
    with a row stride padded to 16 elements (ready for dedisp_execute)."""
    import torch
    if not x.is_cuda or x.dtype != torch.float32 or x.stride(-1) != 1 or x.dim() < 2:
        raise DedispError(ESHAPE, "dedisp_bin")
    rows = 1
    for k in range(x.dim() - 1):
        rows *= x.shape[k]
    for k in range(x.dim() - 2):
        if x.stride(k) != x.stride(k + 1) * x.shape[k + 1]:
            raise DedispError(ESHAPE, "dedisp_bin")
    n = x.shape[-1]
    nout = n // int(nb)
    stride = max(16, (nout + 15) // 16 * 16)
    out = torch.empty(tuple(x.shape[:-1]) + (stride,), dtype=torch.float32, device=x.device)
    _check(lib().dedisp_bin(x.data_ptr(), out.data_ptr(), int(rows), int(n), int(x.stride(-2)), int(stride),
                            int(nb), _stream_ptr(stream)), "dedisp_bin")
    return out[..., :nout]


class Stream:
    """dedisp_stream_*: streaming chunk driver carrying the max_delay overlap between chunks."""

    def __init__(self, plan, dtype, chunk, nbeams=1):
        h = _vp()
        _check(lib().dedisp_stream_create(ctypes.byref(h), plan._h, int(dtype), int(chunk), int(nbeams)),
               "dedisp_stream_create")
        self._h, self.plan, self.dtype, self.chunk, self.nbeams = h, plan, int(dtype), int(chunk), int(nbeams)

    def push(self, chunk_in, out=None, stream=None):
        import torch
        if not chunk_in.is_cuda or not chunk_in.is_contiguous():
            raise RuntimeError("dedisp_stream_push needs a contiguous CUDA tensor")
        want = (self.nbeams, self.plan.nchans, self.chunk)
        if tuple(chunk_in.shape) != want:
            raise DedispError(ESHAPE, "dedisp_stream_push")
        if out is None:
            out = torch.empty((self.nbeams, self.plan.ndm, self.chunk), device=chunk_in.device,
                              dtype=torch.float32 if self.dtype == F32 else torch.int32)
        _check(lib().dedisp_stream_push(self._h, chunk_in.data_ptr(), out.data_ptr(), _stream_ptr(stream)),
               "dedisp_stream_push")
        return out

    def push_host(self, chunk_in, out, stream=None):
        ia = chunk_in.numpy() if hasattr(chunk_in, "numpy") else chunk_in
        oa = out.numpy() if hasattr(out, "numpy") else out
        assert ia.flags.c_contiguous and oa.flags.c_contiguous
        _check(lib().dedisp_stream_push_host(self._h, ia.ctypes.data, oa.ctypes.data, _stream_ptr(stream)),
               "dedisp_stream_push_host")
        return out

    def reset(self, stream=None):
        _check(lib().dedisp_stream_reset(self._h, _stream_ptr(stream)), "dedisp_stream_reset")

    def close(self):
        if getattr(self, "_h", None):
            _check(lib().dedisp_stream_destroy(self._h), "dedisp_stream_destroy")
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class _Pass(ctypes.Structure):
    _fields_ = [("dm_low", _dbl), ("dm_step", _dbl), ("ndm", _int), ("nfine", _int), ("bin", _int)]


class Survey:
    """dedisp_survey_*: passes = [(dm_low, dm_step, ndm, nfine, bin), ...] (Tables 1 / 4)."""

    def __init__(self, nchans, f_top_mhz, df_mhz, t_samp_ms, nsub, passes):
        arr = (_Pass * len(passes))(*[_Pass(float(a), float(b), int(c), int(d), int(e)) for (a, b, c, d, e) in passes])
        h = _vp()
        _check(lib().dedisp_survey_create(ctypes.byref(h), int(nchans), float(f_top_mhz), float(df_mhz), float(t_samp_ms),
                                          int(nsub), ctypes.addressof(arr), len(passes)), "dedisp_survey_create")
        self._h, self.nchans, self.nsub, self.passes = h, int(nchans), int(nsub), [tuple(p) for p in passes]
        self._reserved = (-1, 0)

    @property
    def max_delay(self):
        return int(lib().dedisp_survey_max_delay(self._h))

    @property
    def last_launches(self):
        return int(lib().dedisp_survey_last_launches(self._h))

    def pass_tables(self, i):
        """(s1, s2, nominal_dm, maxshift2, max_delay) of pass i's subband plan."""
        ph = lib().dedisp_survey_pass_plan(self._h, int(i))
        ndm, nfine = self.passes[i][2], self.passes[i][3]
        nco = ndm // nfine
        s1 = np.empty((nco, self.nchans), dtype=np.int32)
        s2 = np.empty((ndm, self.nsub), dtype=np.int32)
        nom = np.empty(nco, dtype=np.float64)
        m2 = np.empty(nco, dtype=np.int32)
        _check(lib().dedisp_plan_get_subband_shifts(ph, s1.ctypes.data, s2.ctypes.data, nom.ctypes.data, m2.ctypes.data),
               "dedisp_plan_get_subband_shifts")
        return s1, s2, nom, m2, int(lib().dedisp_plan_max_delay(ph))

    def out_layout(self, nsamp, nbeams=1):
        n = len(self.passes)
        off, st, no = (np.zeros(n, dtype=np.int64) for _ in range(3))
        tot = _i64(0)
        _check(lib().dedisp_survey_out_layout(self._h, int(nsamp), int(nbeams), off.ctypes.data, st.ctypes.data,
                                              no.ctypes.data, ctypes.addressof(tot)), "dedisp_survey_out_layout")
        return off, st, no, int(tot.value)

    def execute(self, x, nsamp, stream=None):
        """x: CUDA float32 [(nbeams,) nchans, >= nsamp + max_delay].  Returns one tensor view
        [(nbeams,) ndm_i, nsamp // bin_i] per pass (all inside one output buffer)."""
        import torch
        x3 = x if x.dim() == 3 else x.unsqueeze(0)
        if not x.is_cuda or x.dtype != torch.float32 or x3.shape[1] != self.nchans or x3.stride(2) != 1 or \
                (x3.shape[0] > 1 and x3.stride(0) != x3.shape[1] * x3.stride(1)):
            raise DedispError(ESHAPE, "dedisp_survey_execute")
        nb = x3.shape[0]
        if nsamp > self._reserved[0] or nb > self._reserved[1]:
            _check(lib().dedisp_survey_reserve(self._h, int(nsamp), int(nb)), "dedisp_survey_reserve")
            self._reserved = (max(self._reserved[0], int(nsamp)), max(self._reserved[1], int(nb)))
        off, st, no, tot = self.out_layout(nsamp, nb)
        out = torch.empty(max(tot, 4), dtype=torch.float32, device=x.device)
        _check(lib().dedisp_survey_execute(self._h, x3.data_ptr(), out.data_ptr(), int(nsamp), int(x3.stride(1)), int(nb),
                                           _stream_ptr(stream)), "dedisp_survey_execute")
        views = []
        for i, p in enumerate(self.passes):
            v = out[off[i]:off[i] + nb * p[2] * st[i]].view(nb, p[2], int(st[i]))[:, :, :int(no[i])]
            views.append(v if x.dim() == 3 else v[0])
        return views

    def close(self):
        if getattr(self, "_h", None):
            _check(lib().dedisp_survey_destroy(self._h), "dedisp_survey_destroy")
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fadd_microbench(packed=True, iters=20000, repeats=5, stream=None):
    """dedisp_fadd_microbench -> (milliseconds, adds executed, number of SMs)."""
    ms, adds, nsm = ctypes.c_float(0.0), ctypes.c_double(0.0), ctypes.c_int(0)
    _check(lib().dedisp_fadd_microbench(int(bool(packed)), int(iters), int(repeats), ctypes.addressof(ms),
                                        ctypes.addressof(adds), ctypes.addressof(nsm), _stream_ptr(stream)),
           "dedisp_fadd_microbench")
    return float(ms.value), float(adds.value), int(nsm.value)


def version():
    return lib().dedisp_version().decode()
