"""Thin Python binding of the C-ABI library (include/mf.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libmadflow_b200.so; PyTorch provides device memory
and streams.  There is NO fallback: if the library is missing or no CUDA device is present, calls raise.

The module-level functions carry the C names (mf_create_process, mf_vegas_iterate, mf_refine_grid,
mf_unweight, ...) and take raw integers (device pointers); `Process` wraps them for torch tensors.  The
integration driver (iteration loop, grid refinement schedule, w_max policy) that bench.py and the tests use is
`integrate.run_config`.
"""
import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmadflow_b200.so")
_lib = None

MF_OK, MF_EINVAL, MF_ECUDA, MF_EOVERFLOW, MF_ERANGE, MF_ENOMEM = 0, -1, -2, -3, -4, -5
_ERR = {MF_EINVAL: "MF_EINVAL", MF_ECUDA: "MF_ECUDA", MF_EOVERFLOW: "MF_EOVERFLOW", MF_ERANGE: "MF_ERANGE",
        MF_ENOMEM: "MF_ENOMEM"}

c_double_p = C.POINTER(C.c_double)

# every symbol include/mf.h declares (tests check the library exports each one)
EXPORTS = ["mf_create_process", "mf_destroy_process", "mf_n_dims", "mf_n_final", "mf_record_size",
           "mf_debug_row_len", "mf_last_error", "mf_launch_config", "mf_vegas_iterate", "mf_vegas_iterate_static", "mf_refine_grid",
           "mf_unweight", "mf_set_dynamic_scale", "mf_set_observables", "mf_debug_eval", "mf_debug_philox", "mf_debug_pdf", "mf_debug_me2",
           "mf_debug_me2_quark_gluon", "mf_measure_fp64_peak", "mf_measure_dmma_peak"]


class MfError(RuntimeError):
    pass


class ProcessDesc(C.Structure):
    """mf_process_desc"""
    _fields_ = [("process", C.c_int32), ("sqrt_s", C.c_double), ("alpha_em", C.c_double), ("alpha_s", C.c_double),
                ("m_top", C.c_double), ("mu2", C.c_double), ("ptmin", C.c_double), ("etamax", C.c_double),
                ("drmin", C.c_double), ("gev2_to_pb", C.c_double), ("n_bins", C.c_int32), ("pdf_nx", C.c_int32),
                ("pdf_nq", C.c_int32), ("pdf_lnx", c_double_p), ("pdf_lnq2", c_double_p), ("pdf_xf", c_double_p),
                ("pdf_nfl", C.c_int32)]


class IterResult(C.Structure):
    """mf_iter_result"""
    _fields_ = [("sum_w", C.c_double), ("sum_w2", C.c_double), ("max_abs_w", C.c_double), ("n_pass", C.c_uint64),
                ("n_accept", C.c_uint64)]


def lib():
    """Loads libmadflow_b200.so; raises (never falls back) if it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise MfError("%s not found: build it with `python -m paper_2106_10279_b200.build` "
                          "(there is no CPU fallback)" % LIB_PATH)
        L = C.CDLL(LIB_PATH)
        vp, u64, u32, i32p = C.c_void_p, C.c_uint64, C.c_uint32, C.POINTER(C.c_int32)
        L.mf_create_process.argtypes = [C.POINTER(ProcessDesc), C.POINTER(vp)]
        L.mf_destroy_process.argtypes = [vp]
        for f in ("mf_n_dims", "mf_n_final", "mf_record_size", "mf_debug_row_len"):
            getattr(L, f).argtypes = [vp, i32p]
        L.mf_last_error.argtypes = [vp]
        L.mf_last_error.restype = C.c_char_p
        L.mf_launch_config.argtypes = [vp, i32p, i32p]
        L.mf_vegas_iterate.argtypes = [vp, vp, u64, u32, u64, u64, vp, vp, vp]
        L.mf_vegas_iterate_static.argtypes = [vp, vp, u64, u32, u64, u64, vp, vp, vp]
        L.mf_refine_grid.argtypes = [vp, vp, vp, C.c_double, vp]
        L.mf_unweight.argtypes = [vp, vp, u64, u32, u64, u64, C.c_double, vp, u64, vp, vp, vp, vp]
        L.mf_set_observables.argtypes = [vp, vp, C.c_int32, C.c_double, C.c_double]
        L.mf_set_dynamic_scale.argtypes = [vp, C.c_int32]
        L.mf_debug_eval.argtypes = [vp, vp, u64, u32, u64, u64, vp, vp]
        L.mf_debug_philox.argtypes = [u64, u32, u64, u64, u32, vp, vp]
        L.mf_debug_pdf.argtypes = [vp, vp, vp, u64, vp, vp]
        L.mf_debug_me2.argtypes = [vp, vp, u64, vp, vp]
        L.mf_debug_me2_quark_gluon.argtypes = [C.c_int32, C.c_double, C.c_double, vp, u64, vp, vp]
        L.mf_measure_fp64_peak.argtypes = [C.c_int64, c_double_p, c_double_p]
        L.mf_measure_dmma_peak.argtypes = [C.c_int64, c_double_p, c_double_p]
        _lib = L
    return _lib


def _check(rc, handle=None, what=""):
    if rc != MF_OK:
        msg = lib().mf_last_error(handle).decode() if handle else ""
        raise MfError("%s failed: %s %s" % (what, _ERR.get(rc, rc), msg))


# ---- C names, raw arguments ---------------------------------------------------------------------------
def mf_create_process(desc):
    h = C.c_void_p()
    rc = lib().mf_create_process(C.byref(desc), C.byref(h))
    return rc, h


def mf_destroy_process(h):
    return lib().mf_destroy_process(h)


def mf_vegas_iterate(h, d_grid, seed, iteration, first_event, n_events, d_hist, d_result, stream=0):
    return lib().mf_vegas_iterate(h, d_grid, seed, iteration, first_event, n_events, d_hist, d_result, stream)


def mf_vegas_iterate_static(h, d_grid, seed, iteration, first_event, n_events, d_hist, d_result, stream=0):
    return lib().mf_vegas_iterate_static(h, d_grid, seed, iteration, first_event, n_events, d_hist, d_result, stream)


def mf_refine_grid(h, d_grid, d_hist, alpha, stream=0):
    return lib().mf_refine_grid(h, d_grid, d_hist, alpha, stream)


def mf_unweight(h, d_grid, seed, iteration, first_event, n_events, w_max, d_records, capacity, d_count, d_hist,
                d_result, stream=0):
    return lib().mf_unweight(h, d_grid, seed, iteration, first_event, n_events, w_max, d_records, capacity, d_count,
                             d_hist, d_result, stream)


def mf_set_observables(h, d_obs, n_bins, pt_max, eta_max):
    return lib().mf_set_observables(h, d_obs, n_bins, pt_max, eta_max)


def mf_debug_eval(h, d_grid, seed, iteration, first_event, n_events, d_out, stream=0):
    return lib().mf_debug_eval(h, d_grid, seed, iteration, first_event, n_events, d_out, stream)


def mf_debug_philox(seed, iteration, first_event, n_events, n_blocks, d_out, stream=0):
    return lib().mf_debug_philox(seed, iteration, first_event, n_events, n_blocks, d_out, stream)


def mf_debug_pdf(h, d_x, d_q2, n, d_out, stream=0):
    return lib().mf_debug_pdf(h, d_x, d_q2, n, d_out, stream)


def mf_debug_me2(h, d_mom, n, d_out, stream=0):
    return lib().mf_debug_me2(h, d_mom, n, d_out, stream)


def mf_measure_fp64_peak(iters=1 << 16):
    fl, ms = C.c_double(), C.c_double()
    _check(lib().mf_measure_fp64_peak(iters, C.byref(fl), C.byref(ms)), None, "mf_measure_fp64_peak")
    return fl.value, ms.value


def mf_measure_dmma_peak(iters=1 << 14):
    fl, ms = C.c_double(), C.c_double()
    _check(lib().mf_measure_dmma_peak(iters, C.byref(fl), C.byref(ms)), None, "mf_measure_dmma_peak")
    return fl.value, ms.value


def make_desc(wl, pdf=None):
    """mf_process_desc from a workloads.Workload; returns (desc, keepalive)."""
    d = ProcessDesc()
    for f in ("process", "sqrt_s", "alpha_em", "alpha_s", "m_top", "mu2", "ptmin", "etamax", "drmin", "gev2_to_pb",
              "n_bins"):
        setattr(d, f, getattr(wl, f))
    keep = None
    if wl.process != 0:
        if pdf is None:
            raise MfError("process %d needs a PDF table" % wl.process)
        keep = tuple(np.ascontiguousarray(a, dtype=np.float64) for a in pdf)
        d.pdf_nx, d.pdf_nq = len(keep[0]), len(keep[1])
        d.pdf_nfl = keep[2].shape[0] if keep[2].ndim == 3 else 1
        d.pdf_lnx, d.pdf_lnq2, d.pdf_xf = (a.ctypes.data_as(c_double_p) for a in keep)
    return d, keep


# ---- torch-tensor wrapper -----------------------------------------------------------------------------
def _torch():
    import torch
    if not torch.cuda.is_available():
        raise MfError("no CUDA device: the MadFlow hot path has no CPU fallback")
    return torch


def _stream_ptr(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


class Process:
    """A process handle plus helpers that take torch CUDA tensors.  `wl` is a workloads.Workload."""

    def __init__(self, wl, pdf=None):
        _torch()
        self.wl = wl
        desc, _keep = make_desc(wl, pdf)
        rc, h = mf_create_process(desc)
        if rc != MF_OK:
            raise MfError("mf_create_process failed: %s" % _ERR.get(rc, rc))
        self.h = h
        v, v2 = C.c_int32(), C.c_int32()
        L = lib()
        L.mf_n_dims(h, C.byref(v)); self.n_dims = v.value
        L.mf_n_final(h, C.byref(v)); self.n_final = v.value
        L.mf_record_size(h, C.byref(v)); self.record_size = v.value
        L.mf_debug_row_len(h, C.byref(v)); self.row_len = v.value
        L.mf_launch_config(h, C.byref(v), C.byref(v2)); self.blocks, self.threads = v.value, v2.value
        self.n_bins = wl.n_bins

    def close(self):
        if getattr(self, "h", None):
            mf_destroy_process(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- buffers -------------------------------------------------------------------------------------------
    def new_grid(self):
        torch = _torch()
        from . import workloads as W
        return torch.from_numpy(W.uniform_grid(self.n_dims, self.n_bins)).cuda()

    def new_hist(self):
        return _torch().zeros((self.n_dims, self.n_bins), dtype=_torch().float64, device="cuda")

    def new_result(self):
        return _torch().zeros(5, dtype=_torch().float64, device="cuda")

    @staticmethod
    def result_to_host(res):
        """mf_iter_result tensor (5 x 8 bytes) -> IterResult"""
        raw = res.cpu().numpy().tobytes()
        return IterResult.from_buffer_copy(raw)

    # -- hot calls (asynchronous on `stream`) -------------------------------------------------------------------
    def vegas_iterate(self, grid, seed, iteration, first_event, n_events, hist, result, stream=None):
        _check(mf_vegas_iterate(self.h, grid.data_ptr(), seed, iteration, first_event, n_events,
                                hist.data_ptr() if hist is not None else None, result.data_ptr(),
                                _stream_ptr(stream)), self.h, "mf_vegas_iterate")

    def vegas_iterate_static(self, grid, seed, iteration, first_event, n_events, hist, result, stream=None):
        """mf_vegas_iterate with the launch's scratch in the library's static device array: allocates nothing (include/mf.h)"""
        _check(mf_vegas_iterate_static(self.h, grid.data_ptr(), seed, iteration, first_event, n_events,
                                       hist.data_ptr() if hist is not None else None, result.data_ptr(),
                                       _stream_ptr(stream)), self.h, "mf_vegas_iterate_static")

    def refine_grid(self, grid, hist, alpha=1.5, stream=None):
        _check(mf_refine_grid(self.h, grid.data_ptr(), hist.data_ptr(), alpha, _stream_ptr(stream)), self.h,
               "mf_refine_grid")

    def unweight(self, grid, seed, iteration, first_event, n_events, w_max, records, capacity, count, hist, result,
                 stream=None):
        _check(mf_unweight(self.h, grid.data_ptr(), seed, iteration, first_event, n_events, w_max,
                           records.data_ptr() if records is not None else None, capacity, count.data_ptr(),
                           hist.data_ptr() if hist is not None else None, result.data_ptr(), _stream_ptr(stream)),
               self.h, "mf_unweight")

    def set_dynamic_scale(self, on):
        """mu^2 = m_t^2 + pT(top)^2 per event with one-loop running alpha_s (include/mf.h)"""
        _check(lib().mf_set_dynamic_scale(self.h, 1 if on else 0), self.h, "mf_set_dynamic_scale")

    def set_observables(self, obs, n_bins=0, pt_max=0.0, eta_max=0.0):
        """attach a zeroed float64 CUDA tensor [2, n_bins + 1] (pT and eta of the first final-state particle); None detaches"""
        if obs is not None:
            assert obs.is_cuda and obs.dtype == _torch().float64 and obs.numel() == 2 * (n_bins + 1) and obs.is_contiguous()
        _check(mf_set_observables(self.h, obs.data_ptr() if obs is not None else None, n_bins, pt_max, eta_max), self.h,
               "mf_set_observables")
        self._obs = obs          # keep the buffer alive while attached

    # -- diagnostics ---------------------------------------------------------------------------------------
    def debug_eval(self, grid, seed, iteration, first_event, n_events):
        torch = _torch()
        out = torch.empty((n_events, self.row_len), dtype=torch.float64, device="cuda")
        _check(mf_debug_eval(self.h, grid.data_ptr(), seed, iteration, first_event, n_events, out.data_ptr(),
                             _stream_ptr(None)), self.h, "mf_debug_eval")
        return out.cpu().numpy()

    def debug_pdf(self, x, q2):
        torch = _torch()
        xd = torch.as_tensor(np.ascontiguousarray(x, dtype=np.float64)).cuda()
        qd = torch.as_tensor(np.ascontiguousarray(q2, dtype=np.float64)).cuda()
        out = torch.empty_like(xd)
        _check(mf_debug_pdf(self.h, xd.data_ptr(), qd.data_ptr(), xd.numel(), out.data_ptr(), _stream_ptr(None)),
               self.h, "mf_debug_pdf")
        return out.cpu().numpy()

    def debug_me2(self, mom):
        torch = _torch()
        m = torch.as_tensor(np.ascontiguousarray(mom, dtype=np.float64)).cuda().reshape(-1, self.n_final + 2, 4)
        shape = (m.shape[0], 2) if self.wl.process == 4 else (m.shape[0],)     # MF_PP_TT: (gg, q qbar) per point
        out = torch.empty(shape, dtype=torch.float64, device="cuda")
        _check(mf_debug_me2(self.h, m.data_ptr(), m.shape[0], out.data_ptr(), _stream_ptr(None)), self.h,
               "mf_debug_me2")
        return out.cpu().numpy()

    def records_array(self, records, count):
        """Decode `count` AoS records (uint8 tensor) into a numpy structured array with fields mom[n+2][4], w, id and,
        for MF_PP_TT / MF_PP_TTG / MF_PP_TTGG, channel (include/mf.h)."""
        from .lhe import record_dtype
        dt = record_dtype(self.n_final, self.wl.process)
        assert dt.itemsize == self.record_size
        raw = records[:count * self.record_size].cpu().numpy().tobytes()
        return np.frombuffer(raw, dtype=dt)

    def records_view(self, records, count):
        """(momenta[count, n+2, 4], w[count], id[count]) of `count` records"""
        a = self.records_array(records, count)
        return a["mom"], a["w"], a["id"]


def debug_me2_quark_gluon(kind, m_top, alpha_s, mom):
    """|M|^2 of q qbar -> ttbar g (kind 0), q g -> ttbar q (1), qbar g -> ttbar qbar (2) at mom[n][5][4];
    kind 3: q qbar -> ttbar g g at mom[n][6][4]"""
    torch = _torch()
    m = torch.as_tensor(np.ascontiguousarray(mom, dtype=np.float64)).cuda().reshape(-1, 6 if kind == 3 else 5, 4)
    out = torch.empty(m.shape[0], dtype=torch.float64, device="cuda")
    _check(lib().mf_debug_me2_quark_gluon(kind, m_top, alpha_s, m.data_ptr(), m.shape[0], out.data_ptr(), _stream_ptr(None)),
           None, "mf_debug_me2_quark_gluon")
    return out.cpu().numpy()


def debug_philox(seed, iteration, first_event, n_events, n_blocks):
    torch = _torch()
    out = torch.empty((n_events, n_blocks, 4), dtype=torch.int32, device="cuda")
    _check(mf_debug_philox(seed, iteration, first_event, n_events, n_blocks, out.data_ptr(), _stream_ptr(None)), None,
           "mf_debug_philox")
    return out.cpu().numpy().view(np.uint32)
