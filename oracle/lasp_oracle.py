"""ctypes wrapper around oracle/lasp_oracle.c (the fp64 CPU oracle).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_2512_24840_b200/.
Argument marshalling only; all arithmetic is in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lasp_oracle.c")
_LIB = os.path.join(_HERE, "liblasp_oracle.so")

_f64p = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_u8p = C.POINTER(C.c_uint8)


class _Model(C.Structure):
    _fields_ = [
        ("n_pix", C.c_int32), ("n_seg", C.c_int32),
        ("seg_offset", _i32p), ("loglam", _f64p), ("seg_sigma_inst", _f64p),
        ("n_labels", C.c_int32), ("n_terms", C.c_int32),
        ("term_exps", _u8p), ("coeffs", _f64p), ("lo", _f64p), ("hi", _f64p),
        ("label_log10", _u8p), ("emu_a", _f64p), ("emu_b", _f64p),
        ("cont_degree", C.c_int32), ("seg_n_edge", _i32p),
        ("n_models", C.c_int32), ("term_model", _u8p), ("model_blend", _f64p),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


class Oracle:
    """The oracle bound to one model description (dict from synth.make_model_desc)."""

    def __init__(self, desc: dict):
        self.L = int(desc["n_labels"]); self.K = int(desc["n_terms"]); self.P = int(desc["n_pix"])
        self.NP = self.L + 2; self.D = int(desc["cont_degree"]); self.n_seg = int(desc["n_seg"])
        self.nc = self.n_seg * (self.D + 1)
        k = self._keep = {}
        k["seg_offset"] = np.ascontiguousarray(desc["seg_offset"], dtype=np.int32)
        k["loglam"] = np.ascontiguousarray(desc["loglam"], dtype=np.float64)
        k["seg_sigma_inst"] = np.ascontiguousarray(desc["seg_sigma_inst"], dtype=np.float64)
        k["term_exps"] = np.ascontiguousarray(desc["term_exps"], dtype=np.uint8)
        k["coeffs"] = np.ascontiguousarray(desc["coeffs"], dtype=np.float64)
        k["lo"] = np.ascontiguousarray(desc["lo"], dtype=np.float64)
        k["hi"] = np.ascontiguousarray(desc["hi"], dtype=np.float64)
        k["label_log10"] = np.ascontiguousarray(desc["label_log10"], dtype=np.uint8)
        k["emu_a"] = np.ascontiguousarray(desc["emu_a"], dtype=np.float64)
        k["emu_b"] = np.ascontiguousarray(desc["emu_b"], dtype=np.float64)
        k["seg_n_edge"] = np.ascontiguousarray(desc["seg_n_edge"], dtype=np.int32)
        self.n_models = int(desc.get("n_models", 0))
        k["term_model"] = np.ascontiguousarray(desc.get("term_model", np.zeros(self.K)), dtype=np.uint8)
        k["model_blend"] = np.ascontiguousarray(desc.get("model_blend", np.zeros(4)), dtype=np.float64).reshape(-1)
        self.m = _Model(self.P, self.n_seg, _p(k["seg_offset"], _i32p), _p(k["loglam"], _f64p),
                        _p(k["seg_sigma_inst"], _f64p), self.L, self.K, _p(k["term_exps"], _u8p),
                        _p(k["coeffs"], _f64p), _p(k["lo"], _f64p), _p(k["hi"], _f64p),
                        _p(k["label_log10"], _u8p), _p(k["emu_a"], _f64p), _p(k["emu_b"], _f64p),
                        self.D, _p(k["seg_n_edge"], _i32p), self.n_models, _p(k["term_model"], _u8p),
                        _p(k["model_blend"], _f64p))
        self.lo = k["lo"]; self.hi = k["hi"]

    # ---- helpers
    @staticmethod
    def _f64(a):
        return np.ascontiguousarray(a, dtype=np.float64)

    def norm_u(self, theta):
        return 2.0 * (self._f64(theta) - self.lo) / (self.hi - self.lo) - 1.0

    def denorm(self, u):
        return self.lo + (self._f64(u) + 1.0) * (self.hi - self.lo) * 0.5

    def pixel_kms(self):
        s = np.empty(self.P)
        lib().orc_pixel_kms(C.byref(self.m), _p(s, _f64p))
        return s

    # ---- pieces (for pins)
    def monomials(self, theta):
        theta = self._f64(theta)
        x = np.empty(self.L); phi = np.empty(self.K); dphi = np.empty((self.L, self.K)); dx = np.empty(self.L)
        lib().orc_monomials(C.byref(self.m), _p(theta, _f64p), _p(x, _f64p), _p(phi, _f64p),
                            _p(dphi, _f64p), _p(dx, _f64p))
        return x, phi, dphi, dx

    def blend_weight(self, r, theta0):
        w = C.c_double(0.0); dw = C.c_double(0.0)
        lib().orc_blend_weight(C.byref(self.m), C.c_int(r), C.c_double(theta0), C.byref(w), C.byref(dw))
        return w.value, dw.value

    @staticmethod
    def legendre(x, D):
        out = np.empty(D + 1)
        lib().orc_legendre(C.c_double(x), C.c_int(D), _p(out, _f64p))
        return out

    @staticmethod
    def kernel_weights(mu, sigma, Hcap=4096):
        g = np.empty(2 * Hcap + 1); gm = np.empty_like(g); gs = np.empty_like(g)
        f = lib().orc_kernel_weights
        f.restype = C.c_int
        H = f(C.c_double(mu), C.c_double(sigma), C.c_int(Hcap), _p(g, _f64p), _p(gm, _f64p), _p(gs, _f64p))
        if H < 0:
            raise ValueError("support exceeds Hcap")
        n = 2 * H + 1
        return H, g[:n].copy(), gm[:n].copy(), gs[:n].copy()

    @staticmethod
    def adam_step(u, m, v, g, t, lr, b1=0.9, b2=0.999, eps=1e-8):
        u = np.array(u, dtype=np.float64); m = np.array(m, dtype=np.float64)
        v = np.array(v, dtype=np.float64); g = np.ascontiguousarray(g, dtype=np.float64)
        lib().orc_adam_step(C.c_int(u.size), _p(u, _f64p), _p(m, _f64p), _p(v, _f64p), _p(g, _f64p),
                            C.c_int(t), C.c_double(lr), C.c_double(b1), C.c_double(b2), C.c_double(eps))
        return u, m, v

    def solve_continuum(self, S, y, w):
        S = self._f64(S); y = self._f64(y); w = self._f64(w)
        b = np.empty(self.nc); c = np.empty(self.P)
        f = lib().orc_solve_continuum
        f.restype = C.c_int
        st = f(C.byref(self.m), _p(S, _f64p), _p(y, _f64p), _p(w, _f64p), _p(b, _f64p), _p(c, _f64p))
        return b, c, st

    # ---- the entry points mirrored by include/lasp_gpu.h
    def eval_S(self, params):
        params = self._f64(params).reshape(-1, self.NP)
        out = np.empty((params.shape[0], self.P))
        lib().orc_eval_S(C.byref(self.m), C.c_int64(params.shape[0]), _p(params, _f64p), _p(out, _f64p))
        return out

    def eval_model(self, params, cont):
        params = self._f64(params).reshape(-1, self.NP)
        cont = self._f64(cont).reshape(-1, self.nc)
        out = np.empty((params.shape[0], self.P))
        lib().orc_eval_model(C.byref(self.m), C.c_int64(params.shape[0]), _p(params, _f64p),
                             _p(cont, _f64p), _p(out, _f64p))
        return out

    def _obs(self, flux, ivar, mask):
        flux = self._f64(flux).reshape(-1, self.P)
        ivar = self._f64(ivar).reshape(-1, self.P)
        if mask is not None:
            mask = np.ascontiguousarray(mask, dtype=np.uint8).reshape(-1, self.P)
        return flux, ivar, mask

    def eval_grad(self, flux, ivar, mask, params):
        flux, ivar, mask = self._obs(flux, ivar, mask)
        B = flux.shape[0]
        params = self._f64(params).reshape(B, self.NP)
        chi2 = np.empty(B); grad = np.empty((B, self.NP)); cont = np.empty((B, self.nc))
        status = np.zeros(B, dtype=np.int32)
        lib().orc_eval_grad(C.byref(self.m), C.c_int64(B), _p(flux, _f64p), _p(ivar, _f64p),
                            _p(mask, _u8p) if mask is not None else None, _p(params, _f64p),
                            _p(chi2, _f64p), _p(grad, _f64p), _p(cont, _f64p), _p(status, _i32p))
        return chi2, grad, cont, status

    def chi2_u(self, flux, ivar, mask, u):
        flux, ivar, mask = self._obs(flux, ivar, mask)
        u = self._f64(u)
        out = C.c_double(0.0)
        lib().orc_chi2_u(C.byref(self.m), _p(flux, _f64p), _p(ivar, _f64p),
                         _p(mask, _u8p) if mask is not None else None, _p(u, _f64p), C.byref(out))
        return out.value

    def fit(self, flux, ivar, mask, init, n_iter, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8,
            fd_h=1e-5, want_err=True, want_trace=False):
        flux, ivar, mask = self._obs(flux, ivar, mask)
        B = flux.shape[0]
        init = self._f64(init).reshape(B, self.NP)
        params = np.empty((B, self.NP)); cont = np.empty((B, self.nc)); chi2 = np.empty(B)
        err = np.empty((B, self.NP)) if want_err else None
        status = np.zeros(B, dtype=np.int32)
        trace = np.empty((B, n_iter + 1)) if want_trace else None
        lib().orc_fit(C.byref(self.m), C.c_int64(B), _p(flux, _f64p), _p(ivar, _f64p),
                      _p(mask, _u8p) if mask is not None else None, _p(init, _f64p), C.c_int(n_iter),
                      C.c_double(lr), C.c_double(beta1), C.c_double(beta2), C.c_double(eps),
                      C.c_double(fd_h), _p(params, _f64p), _p(cont, _f64p), _p(chi2, _f64p),
                      _p(err, _f64p) if want_err else None, _p(status, _i32p),
                      _p(trace, _f64p) if want_trace else None)
        out = dict(params=params, cont=cont, chi2=chi2, err=err, status=status)
        if want_trace:
            out["trace"] = trace
        return out


    def fit_stop(self, flux, ivar, mask, init, max_iter, lr=0.1, beta1=0.9, beta2=0.999, eps=1e-8, window=50,
                 tol=1e-5, fd_h=1e-5, want_err=True):
        """The fit with the paper's stopping rules (orc_fit_stop)."""
        flux, ivar, mask = self._obs(flux, ivar, mask)
        B = flux.shape[0]
        init = self._f64(init).reshape(B, self.NP)
        params = np.empty((B, self.NP)); cont = np.empty((B, self.nc)); chi2 = np.empty(B)
        err = np.empty((B, self.NP)) if want_err else None
        status = np.zeros(B, dtype=np.int32); n_steps = np.zeros(B, dtype=np.int32)
        lib().orc_fit_stop(C.byref(self.m), C.c_int64(B), _p(flux, _f64p), _p(ivar, _f64p),
                           _p(mask, _u8p) if mask is not None else None, _p(init, _f64p), C.c_int(max_iter),
                           C.c_double(lr), C.c_double(beta1), C.c_double(beta2), C.c_double(eps), C.c_int(window),
                           C.c_double(tol), C.c_double(fd_h), _p(params, _f64p), _p(cont, _f64p), _p(chi2, _f64p),
                           _p(err, _f64p) if want_err else None, _p(status, _i32p), _p(n_steps, _i32p))
        return dict(params=params, cont=cont, chi2=chi2, err=err, status=status, n_steps=n_steps)

    def fit_clean(self, flux, ivar, mask, init, n_iter, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8, every=30, max_updates=11,
                  window=0, tol=1e-5, fd_h=1e-5, want_err=True):
        """The fit with the Clean strategy (orc_fit_clean): fixed n_iter steps (window = 0) or the
        stopping rules of P:169-171 (window > 0, n_iter the maximum)."""
        flux, ivar, mask = self._obs(flux, ivar, mask)
        B = flux.shape[0]
        init = self._f64(init).reshape(B, self.NP)
        params = np.empty((B, self.NP)); cont = np.empty((B, self.nc)); chi2 = np.empty(B)
        err = np.empty((B, self.NP)) if want_err else None
        status = np.zeros(B, dtype=np.int32); n_clipped = np.zeros(B, dtype=np.int32); n_steps = np.zeros(B, dtype=np.int32)
        mask_out = np.zeros((B, self.P), dtype=np.uint8)
        lib().orc_fit_clean(C.byref(self.m), C.c_int64(B), _p(flux, _f64p), _p(ivar, _f64p),
                            _p(mask, _u8p) if mask is not None else None, _p(init, _f64p), C.c_int(n_iter),
                            C.c_double(lr), C.c_double(beta1), C.c_double(beta2), C.c_double(eps), C.c_int(every),
                            C.c_int(max_updates), C.c_int(window), C.c_double(tol), C.c_double(fd_h), _p(params, _f64p),
                            _p(cont, _f64p), _p(chi2, _f64p), _p(err, _f64p) if want_err else None, _p(status, _i32p),
                            _p(mask_out, _u8p), _p(n_clipped, _i32p), _p(n_steps, _i32p))
        return dict(params=params, cont=cont, chi2=chi2, err=err, status=status, mask=mask_out, n_clipped=n_clipped,
                    n_steps=n_steps)

    def fit_lm(self, flux, ivar, mask, init, n_iter, lambda0=1e-3, fd_h=1e-5, want_err=True, want_trace=False):
        """Levenberg-Marquardt on the NP x NP system (NEXT-4; orc_fit_lm): n_iter LM iterations from `init`."""
        flux, ivar, mask = self._obs(flux, ivar, mask)
        B = flux.shape[0]
        init = self._f64(init).reshape(B, self.NP)
        params = np.empty((B, self.NP)); cont = np.empty((B, self.nc)); chi2 = np.empty(B)
        err = np.empty((B, self.NP)) if want_err else None
        status = np.zeros(B, dtype=np.int32); n_steps = np.zeros(B, dtype=np.int32)
        trace = np.zeros((B, n_iter + 1)) if want_trace else None
        lib().orc_fit_lm(C.byref(self.m), C.c_int64(B), _p(flux, _f64p), _p(ivar, _f64p),
                         _p(mask, _u8p) if mask is not None else None, _p(init, _f64p), C.c_int(n_iter),
                         C.c_double(lambda0), C.c_double(fd_h), _p(params, _f64p), _p(cont, _f64p), _p(chi2, _f64p),
                         _p(err, _f64p) if want_err else None, _p(status, _i32p), _p(n_steps, _i32p),
                         _p(trace, _f64p) if want_trace else None)
        return dict(params=params, cont=cont, chi2=chi2, err=err, status=status, n_steps=n_steps, trace=trace)


def obs_nodes(loglam):
    """Observed integration nodes of P:92 for one segment (orc_obs_nodes)."""
    ll = np.ascontiguousarray(loglam, dtype=np.float64)
    out = np.empty(ll.size + 1)
    lib().orc_obs_nodes(_p(ll, _f64p), C.c_int(ll.size), _p(out, _f64p))
    return out


def resample(T, lam1, dlam1, nodes):
    """Flux-conserving resampling of one model spectrum (Eq. 2-4; orc_resample)."""
    T = np.ascontiguousarray(T, dtype=np.float64); nodes = np.ascontiguousarray(nodes, dtype=np.float64)
    out = np.empty(nodes.size - 1)
    lib().orc_resample(C.c_int(T.size), C.c_double(lam1), C.c_double(dlam1), _p(T, _f64p), C.c_int(out.size),
                       _p(nodes, _f64p), _p(out, _f64p))
    return out


def resample_coeffs(coef, lam1, dlam1, seg_offset, loglam):
    """Every row of a [K, q] coefficient table onto the observed grid (orc_resample_coeffs)."""
    coef = np.ascontiguousarray(coef, dtype=np.float64)
    seg = np.ascontiguousarray(seg_offset, dtype=np.int32); ll = np.ascontiguousarray(loglam, dtype=np.float64)
    out = np.empty((coef.shape[0], ll.size))
    lib().orc_resample_coeffs(C.c_int(coef.shape[0]), C.c_int(coef.shape[1]), C.c_double(lam1), C.c_double(dlam1),
                              _p(coef, _f64p), C.c_int(ll.size), C.c_int(seg.size - 1), _p(seg, _i32p), _p(ll, _f64p),
                              _p(out, _f64p))
    return out


def stop_rule(L, window=50, tol=1e-5):
    """First step t (1-based) at which criterion (2) or (3) of P:169-171 fires on the loss sequence L, and the rule
    (1 = neither within the sequence, then t = 0)."""
    L = np.ascontiguousarray(L, dtype=np.float64)
    rule = C.c_int(0)
    f = lib().orc_stop_rule
    f.restype = C.c_int
    t = f(_p(L, _f64p), C.c_int(L.size), C.c_int(window), C.c_double(tol), C.byref(rule))
    return int(t), int(rule.value)


def clean_update(r, M, w, seg_offset, fshift):
    """One Clean-strategy mask update (orc_clean_update): returns (new weights, number clipped, k used)."""
    r = np.ascontiguousarray(r, dtype=np.float64); M = np.ascontiguousarray(M, dtype=np.float64)
    w = np.array(w, dtype=np.float64)
    seg = np.ascontiguousarray(seg_offset, dtype=np.int32)
    k = C.c_int(0)
    f = lib().orc_clean_update
    f.restype = C.c_int
    n = f(C.c_int(r.size), C.c_int(seg.size - 1), _p(seg, _i32p), _p(r, _f64p), _p(M, _f64p), _p(w, _f64p),
          C.c_double(fshift), C.byref(k))
    return w, int(n), int(k.value)


def forward(desc, params, cont):
    """`forward` callable for synth.make_case: model spectra from the oracle."""
    return Oracle(desc).eval_model(params, cont)
