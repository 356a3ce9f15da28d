"""ORACLE — TEST INFRASTRUCTURE ONLY.  ctypes binding of oracle/libmfo.so (the CPU oracle).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import this.
It shares nothing with the CUDA path and does not import the product package.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None

c_double_p = C.POINTER(C.c_double)
c_u32_p = C.POINTER(C.c_uint32)
c_i32_p = C.POINTER(C.c_int32)
c_u64_p = C.POINTER(C.c_uint64)


class ProcessDesc(C.Structure):
    _fields_ = [("process", C.c_int32), ("sqrt_s", C.c_double), ("alpha_em", C.c_double), ("alpha_s", C.c_double),
                ("m_top", C.c_double), ("mu2", C.c_double), ("ptmin", C.c_double), ("etamax", C.c_double),
                ("drmin", C.c_double), ("gev2_to_pb", C.c_double), ("n_bins", C.c_int32), ("pdf_nx", C.c_int32),
                ("pdf_nq", C.c_int32), ("pdf_lnx", c_double_p), ("pdf_lnq2", c_double_p), ("pdf_xf", c_double_p),
                ("pdf_nfl", C.c_int32)]


class IterResult(C.Structure):
    _fields_ = [("sum_w", C.c_double), ("sum_w2", C.c_double), ("max_abs_w", C.c_double), ("n_pass", C.c_uint64),
                ("n_accept", C.c_uint64)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        L = _lib
        L.mfo_uniform_from_words.restype = C.c_double
        L.mfo_vegas_map.restype = C.c_double
        L.mfo_two_body.restype = C.c_double
        L.mfo_rambo.restype = C.c_double
        L.mfo_two_pi_power.restype = C.c_double
        L.mfo_two_pi_power.argtypes = [C.c_int]
        L.mfo_pdf_xf.restype = C.c_double
        L.mfo_me2.restype = C.c_double
        L.mfo_pdf_xf.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_int]
        L.mfo_two_body.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, c_double_p]
        L.mfo_rambo.argtypes = [C.c_int, c_double_p, C.c_double, c_double_p, c_double_p, C.c_int]
        L.mfo_parton_fractions.argtypes = [C.c_double, C.c_double, C.c_double, C.c_double, c_double_p]
        L.mfo_cuts.argtypes = [C.c_int, c_double_p, C.c_double, C.c_double, C.c_double, c_double_p]
        L.mfo_boost_z.argtypes = [C.c_double, c_double_p, c_double_p]
        L.mfo_me2.argtypes = [C.c_void_p, c_double_p, C.c_int, C.c_int, c_double_p, c_double_p, C.c_int]
        L.mfo_vegas_iterate.argtypes = [C.c_void_p, c_double_p, C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint64,
                                        c_double_p, C.POINTER(IterResult), C.c_int]
        L.mfo_refine_grid.argtypes = [C.c_void_p, c_double_p, c_double_p, C.c_double, C.c_int]
        L.mfo_unweight.argtypes = [C.c_void_p, c_double_p, C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint64, C.c_double,
                                   C.c_void_p, C.c_uint64, c_u64_p, c_double_p, C.POINTER(IterResult), C.c_int]
        L.mfo_debug_eval.argtypes = [C.c_void_p, c_double_p, C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint64,
                                     c_double_p, C.c_int]
        L.mfo_philox_block.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64, C.c_uint32, c_u32_p]
        L.mfo_uniform_from_words.argtypes = [C.c_uint32, C.c_uint32]
        L.mfo_vegas_map.argtypes = [c_double_p, C.c_int, C.c_int, c_double_p, c_double_p, c_i32_p]
        L.mfo_dressed_amplitude.argtypes = [C.c_void_p, c_double_p, c_i32_p, c_i32_p, C.c_int, C.c_int, c_double_p]
        L.mfo_ordered_amplitude_coloured.argtypes = L.mfo_dressed_amplitude.argtypes
        L.mfo_spinor.argtypes = [c_double_p, C.c_double, C.c_int, C.c_int, C.c_int, c_double_p]
        L.mfo_polarisation.argtypes = [c_double_p, C.c_int, C.c_int, c_double_p]
        L.mfo_count_ops_me2.argtypes = [C.c_void_p, c_double_p, c_u64_p]
        L.mfo_count_ops_event.argtypes = [C.c_void_p, c_double_p, C.c_uint64, C.c_uint32, C.c_uint64, c_u64_p]
        L.mfo_colour_matrix.argtypes = [C.c_int, c_double_p]
        L.mfo_colour_matrix_entry.restype = C.c_double
        L.mfo_colour_matrix_entry.argtypes = [C.c_int, c_i32_p, c_i32_p]
        L.mfo_set_dynamic_scale.argtypes = [C.c_void_p, C.c_int32]
        L.mfo_me2_qq_ttbar_gg.restype = C.c_double
        L.mfo_me2_qq_ttbar_gg.argtypes = [c_double_p, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int]
        L.mfo_qq_ttbar_gg_amplitude.restype = None
        L.mfo_qq_ttbar_gg_amplitude.argtypes = [c_double_p, C.c_double, C.c_double, c_i32_p, C.c_int, c_i32_p, c_double_p]
        L.mfo_me2_light_line_ttbar_g.restype = C.c_double
        L.mfo_me2_light_line_ttbar_g.argtypes = [C.c_int, c_double_p, C.c_double, C.c_double, C.c_int, C.c_int, C.c_int]
        L.mfo_me2_qq.restype = C.c_double
        L.mfo_me2_qq.argtypes = [C.c_void_p, c_double_p, C.c_int, C.c_int]
        L.mfo_pdf_xf_table.restype = C.c_double
        L.mfo_pdf_xf_table.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int]
    return _lib


def _dp(a):
    return a.ctypes.data_as(c_double_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*ctr)
    k = (C.c_uint32 * 2)(*key)
    o = (C.c_uint32 * 4)()
    lib().mfo_philox4x32_10(c, k, o)
    return list(o)


def philox_block(seed, iteration, event, block):
    o = (C.c_uint32 * 4)()
    lib().mfo_philox_block(seed, iteration, event, block, o)
    return list(o)


def uniform_from_words(hi, lo):
    return lib().mfo_uniform_from_words(hi, lo)


def vegas_map(grid, u):
    grid = _f64(grid)
    u = _f64(u)
    D, nb = grid.shape[0], grid.shape[1] - 1
    x = np.empty(D)
    b = np.empty(D, dtype=np.int32)
    j = lib().mfo_vegas_map(_dp(grid), D, nb, _dp(u), _dp(x), b.ctypes.data_as(c_i32_p))
    return x, j, b


def parton_fractions(x0, x1, tau_min, s):
    out = np.empty(6)
    lib().mfo_parton_fractions(x0, x1, tau_min, s, _dp(out))
    return dict(zip(["tau", "y", "x1", "x2", "shat", "jac"], out))


def two_body(shat, m, xc, xphi):
    mom = np.empty((4, 4))
    w = lib().mfo_two_body(shat, m, xc, xphi, _dp(mom))
    return mom, w


def rambo(masses, w, rho, prec=0):
    masses = _f64(masses)
    rho = _f64(rho)
    n = len(masses)
    k = np.empty((n, 4))
    V = lib().mfo_rambo(n, _dp(masses), w, _dp(rho), _dp(k), prec)
    return k, V


def two_pi_power(n):
    """(2 pi)^(4 - 3 n), the oracle's own function (O6 step 6)"""
    return lib().mfo_two_pi_power(n)


def cuts(gluons_lab, ptmin, etamax, drmin):
    g = _f64(gluons_lab)
    obs = np.empty((g.shape[0], 3))
    ok = lib().mfo_cuts(g.shape[0], _dp(g), ptmin, etamax, drmin, _dp(obs))
    return bool(ok), obs


def boost_z(y, p):
    p = _f64(p)
    out = np.empty(4)
    lib().mfo_boost_z(y, _dp(p), _dp(out))
    return out


def me2_qq_ttbar_gg(mom, mt, alpha_s, basis=0, subst=-1, prec=0):
    """averaged |M|^2 of q qbar -> t tbar g g at mom[6][4] (36 diagrams, explicit colour tensors)"""
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    assert mom.shape == (6, 4)
    return lib().mfo_me2_qq_ttbar_gg(_dp(mom), mt, alpha_s, basis, subst, prec)


def qq_ttbar_gg_amplitude(mom, mt, gs, lam, col, basis=0):
    """(diagram sum, dressed recursion) of iM for helicities lam[6] and colours col[6] = (qbar, q, t, tbar, g, g)"""
    mom = np.ascontiguousarray(mom, dtype=np.float64)
    lam = np.ascontiguousarray(lam, dtype=np.int32)
    col = np.ascontiguousarray(col, dtype=np.int32)
    out = np.zeros(4)
    lib().mfo_qq_ttbar_gg_amplitude(_dp(mom), mt, gs, lam.ctypes.data_as(c_i32_p), basis, col.ctypes.data_as(c_i32_p), _dp(out))
    return complex(out[0], out[1]), complex(out[2], out[3])


def me2_light_line_ttbar_g(kind, mom, mt, alpha_s, basis=0, subst=0, prec=0):
    """kind 0: q qbar -> t tbar g; kind 1: q g -> t tbar q (mom: 5 x 4, the two incoming first); oracle/mfo.h"""
    mom = _f64(mom)
    return lib().mfo_me2_light_line_ttbar_g(kind, _dp(mom), mt, alpha_s, basis, subst, prec)


def colour_matrix(n):
    import math
    f = math.factorial(n)
    out = np.empty((f, f))
    rc = lib().mfo_colour_matrix(n, _dp(out))
    assert rc == 0
    return out


def colour_matrix_entry(n, sigma, tau):
    """C_{sigma tau} straight from its definition (sum over all 8^n colour assignments)"""
    s = np.ascontiguousarray(sigma, dtype=np.int32)
    t = np.ascontiguousarray(tau, dtype=np.int32)
    return lib().mfo_colour_matrix_entry(n, s.ctypes.data_as(c_i32_p), t.ctypes.data_as(c_i32_p))


def spinor(p, m, lam, basis=0, kind=0):
    p = _f64(p)
    out = np.empty(8)
    lib().mfo_spinor(_dp(p), m, lam, basis, kind, _dp(out))
    return out[0::2] + 1j * out[1::2]


def polarisation(p, lam, basis=0):
    p = _f64(p)
    out = np.empty(8)
    lib().mfo_polarisation(_dp(p), lam, basis, _dp(out))
    return out[0::2] + 1j * out[1::2]


class Process:
    """Handle on an oracle process (mfo_create_process).  `wl` is a workloads.Workload-like object."""

    def __init__(self, wl, pdf=None):
        self.wl = wl
        d = ProcessDesc()
        for f in ("process", "sqrt_s", "alpha_em", "alpha_s", "m_top", "mu2", "ptmin", "etamax", "drmin", "gev2_to_pb",
                  "n_bins"):
            setattr(d, f, getattr(wl, f))
        self._keep = None
        if wl.process != 0:
            lnx, lnq2, xf = (_f64(a) for a in pdf)
            self._keep = (lnx, lnq2, xf)
            d.pdf_nx, d.pdf_nq = len(lnx), len(lnq2)
            d.pdf_nfl = xf.shape[0] if xf.ndim == 3 else 1
            d.pdf_lnx, d.pdf_lnq2, d.pdf_xf = _dp(lnx), _dp(lnq2), _dp(xf)
        h = C.c_void_p()
        rc = lib().mfo_create_process(C.byref(d), C.byref(h))
        if rc != 0:
            raise ValueError("mfo_create_process failed: %d" % rc)
        self.h = h
        v = C.c_int32()
        lib().mfo_n_dims(h, C.byref(v)); self.n_dims = v.value
        lib().mfo_n_final(h, C.byref(v)); self.n_final = v.value
        lib().mfo_record_size(h, C.byref(v)); self.record_size = v.value
        lib().mfo_debug_row_len(h, C.byref(v)); self.row_len = v.value
        self.n_bins = wl.n_bins

    def __del__(self):
        try:
            if self.h:
                lib().mfo_destroy_process(self.h)
                self.h = None
        except Exception:
            pass

    def vegas_iterate(self, grid, seed, iteration, first_event, n_events, prec=0):
        grid = _f64(grid)
        hist = np.zeros((self.n_dims, self.n_bins))
        res = IterResult()
        rc = lib().mfo_vegas_iterate(self.h, _dp(grid), seed, iteration, first_event, n_events, _dp(hist), C.byref(res), prec)
        assert rc == 0
        return hist, res

    def refine_grid(self, grid, hist, alpha=1.5, prec=0):
        grid = _f64(grid).copy()
        hist = _f64(hist)
        rc = lib().mfo_refine_grid(self.h, _dp(grid), _dp(hist), alpha, prec)
        assert rc == 0
        return grid

    def unweight(self, grid, seed, iteration, first_event, n_events, w_max, capacity, count=0, prec=0):
        grid = _f64(grid)
        hist = np.zeros((self.n_dims, self.n_bins))
        res = IterResult()
        rec = np.zeros(max(capacity, 1) * self.record_size, dtype=np.uint8)
        cnt = C.c_uint64(count)
        rc = lib().mfo_unweight(self.h, _dp(grid), seed, iteration, first_event, n_events, w_max,
                                rec.ctypes.data_as(C.c_void_p), capacity, C.byref(cnt), _dp(hist), C.byref(res), prec)
        assert rc == 0
        return rec, cnt.value, hist, res

    def debug_eval(self, grid, seed, iteration, first_event, n_events, prec=0):
        grid = _f64(grid)
        out = np.empty((n_events, self.row_len))
        rc = lib().mfo_debug_eval(self.h, _dp(grid), seed, iteration, first_event, n_events, _dp(out), prec)
        assert rc == 0
        return out

    def set_dynamic_scale(self, on):
        assert lib().mfo_set_dynamic_scale(self.h, 1 if on else 0) == 0

    def pdf_xf(self, x, q2, prec=0):
        return lib().mfo_pdf_xf(self.h, x, q2, prec)

    def pdf_xf_table(self, table, x, q2, prec=0):
        return lib().mfo_pdf_xf_table(self.h, table, x, q2, prec)

    def me2_qq(self, mom, basis=0, prec=0):
        """averaged |M|^2 of q(mom[0]) qbar(mom[1]) -> t(mom[2]) tbar(mom[3]); process 4 only"""
        mom = _f64(mom)
        return lib().mfo_me2_qq(self.h, _dp(mom), basis, prec)

    def me2(self, mom, basis=0, subst_gluon=-1, prec=0, want_amps=False, want_per_hel=False):
        mom = _f64(mom)
        amps = per = None
        ap = pp = None
        if want_amps:
            import math
            ng = {1: 2, 2: 3, 3: 4, 4: 2, 5: 3, 6: 5, 7: 4}[self.wl.process]
            amps = np.zeros(((4 << ng), math.factorial(ng), 2))
            ap = _dp(amps)
        if want_per_hel:
            per = np.zeros(16)
            pp = _dp(per)
        v = lib().mfo_me2(self.h, _dp(mom), basis, subst_gluon, ap, pp, prec)
        if want_amps:
            return v, amps[..., 0] + 1j * amps[..., 1]
        if want_per_hel:
            return v, per
        return v

    def dressed_amplitude(self, mom, hel, col, icol, jcol):
        mom = _f64(mom)
        h = np.ascontiguousarray(hel, dtype=np.int32)
        c = np.ascontiguousarray(col, dtype=np.int32)
        out = np.empty(2)
        rc = lib().mfo_dressed_amplitude(self.h, _dp(mom), h.ctypes.data_as(c_i32_p), c.ctypes.data_as(c_i32_p), icol, jcol, _dp(out))
        assert rc == 0
        return out[0] + 1j * out[1]

    def ordered_amplitude_coloured(self, mom, hel, col, icol, jcol):
        mom = _f64(mom)
        h = np.ascontiguousarray(hel, dtype=np.int32)
        c = np.ascontiguousarray(col, dtype=np.int32)
        out = np.empty(2)
        rc = lib().mfo_ordered_amplitude_coloured(self.h, _dp(mom), h.ctypes.data_as(c_i32_p), c.ctypes.data_as(c_i32_p), icol, jcol, _dp(out))
        assert rc == 0
        return out[0] + 1j * out[1]

    def count_ops_me2(self, mom):
        mom = _f64(mom)
        out = (C.c_uint64 * 6)()
        lib().mfo_count_ops_me2(self.h, _dp(mom), out)
        return dict(zip(["add", "mul", "div", "sqrt", "trans", "cmp"], list(out)))

    def count_ops_event(self, grid, seed, iteration, event):
        grid = _f64(grid)
        out = (C.c_uint64 * 6)()
        lib().mfo_count_ops_event(self.h, _dp(grid), seed, iteration, event, out)
        return dict(zip(["add", "mul", "div", "sqrt", "trans", "cmp"], list(out)))

    def records_array(self, rec, count):
        """Decode `count` AoS records into a structured array: mom[n+2][4], w, id and, for process 4, channel."""
        fields = [("mom", np.float64, (self.n_final + 2, 4)), ("w", np.float64), ("id", np.uint64)]
        if self.wl.process in (4, 5, 7):
            fields.append(("channel", np.uint64))
        dt = np.dtype(fields)
        assert dt.itemsize == self.record_size
        return np.frombuffer(rec.tobytes()[:count * self.record_size], dtype=dt)

    def records_view(self, rec, count):
        """(momenta[count, n+2, 4], w[count], event_id[count])"""
        a = self.records_array(rec, count)
        return a["mom"], a["w"], a["id"]


def observable_histograms(rows, n_dims, n_final, n_bins, pt_max, eta_max):
    """ORACLE for the observable histograms of the fused pass ("histogram accumulation"; L109-119, Fig. 2:
    d sigma / d pT,top and d sigma / d eta,top), written out from their definition on the oracle's own per-event rows
    (debug_eval): for every event with w != 0 take the lab-frame momentum (E, px, py, pz) of the FIRST final-state
    particle, pT = sqrt(px^2 + py^2), eta = asinh(pz / pT), and add w to bin floor(pT / pt_max * n_bins) of row 0 and
    to bin floor((eta + eta_max) / (2 eta_max) * n_bins) of row 1; bin n_bins collects everything outside.
    Returns obs[2][n_bins + 1]."""
    rows = np.asarray(rows)
    o = n_dims + 4 * (n_final + 2)
    w = rows[:, o + 6]
    p = rows[:, n_dims + 8:n_dims + 12]                 # particle 2 = first final-state particle
    obs = np.zeros((2, n_bins + 1))
    for k in range(len(rows)):
        if w[k] == 0.0:
            continue
        pt = np.sqrt(p[k, 1] * p[k, 1] + p[k, 2] * p[k, 2])
        eta = np.arcsinh(p[k, 3] / pt)
        bp = pt / pt_max * n_bins
        be = (eta + eta_max) / (2.0 * eta_max) * n_bins
        ip = int(bp) if bp < n_bins else n_bins
        ie = int(be) if 0.0 <= be < n_bins else n_bins
        obs[0, ip] += w[k]
        obs[1, ie] += w[k]
    return obs
