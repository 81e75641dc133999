"""Thin ctypes binding over include/lasp_gpu.h: argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in liblasp_gpu.so.
There is no CPU fallback: a missing library or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblasp_gpu.so")

SYMBOLS = ["lasp_create", "lasp_destroy", "lasp_reserve", "lasp_fit_batch", "lasp_fit_batch_host", "lasp_eval_model",
           "lasp_eval_grad", "lasp_eval_grad_static", "lasp_kernel_variant", "lasp_launch_info", "lasp_launch_count", "lasp_fma_per_spectrum_step",
           "lasp_fma_executed_per_spectrum_step", "lasp_last_fit_stats", "lasp_resample_coeffs", "lasp_last_error",
           "lasp_version"]

LASP_ST_NOT_SPD, LASP_ST_NONFINITE, LASP_ST_NEG_CONT, LASP_ST_ON_BOUND, LASP_ST_STOP_TOL, LASP_ST_STOP_RISE = 1, 2, 4, 8, 16, 32

_f32p = C.POINTER(C.c_float)
_f64p = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_u8p = C.POINTER(C.c_uint8)


class ModelDesc(C.Structure):
    _fields_ = [
        ("n_pix", C.c_int32), ("n_seg", C.c_int32),
        ("seg_offset", _i32p), ("loglam", _f64p), ("seg_sigma_inst", _f32p),
        ("n_labels", C.c_int32), ("n_terms", C.c_int32),
        ("term_exps", _u8p), ("coeffs", _f32p), ("lo", _f32p), ("hi", _f32p),
        ("label_log10", _u8p), ("emu_a", _f32p), ("emu_b", _f32p),
        ("cont_degree", C.c_int32), ("seg_n_edge", _i32p),
        ("n_models", C.c_int32), ("term_model", _u8p), ("model_blend", _f32p),
    ]


class FitOpts(C.Structure):
    _fields_ = [("n_iter", C.c_int32), ("lr", C.c_float), ("beta1", C.c_float), ("beta2", C.c_float),
                ("eps", C.c_float), ("variant", C.c_int32), ("emulator_path", C.c_int32),
                ("refresh", C.c_int32), ("warm", C.c_int32), ("fd_fresh", C.c_int32),
                ("stop_window", C.c_int32), ("stop_tol", C.c_float),
                ("clean_every", C.c_int32), ("clean_max", C.c_int32),
                ("optimizer", C.c_int32), ("lm_lambda0", C.c_float)]


class LaspError(RuntimeError):
    pass


_lib = None


def lib():
    """Load liblasp_gpu.so (built in-tree by paper_2512_24840_b200/build.py); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise LaspError(f"{LIB_PATH} is missing: run `python -m paper_2512_24840_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.lasp_create.argtypes = [C.POINTER(ModelDesc), C.c_int, C.POINTER(C.c_void_p)]
        L.lasp_create.restype = C.c_int
        L.lasp_destroy.argtypes = [C.c_void_p]
        L.lasp_reserve.argtypes = [C.c_void_p, C.c_int64]
        L.lasp_fit_batch.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 4 + [C.POINTER(FitOpts)] + \
                                    [C.c_void_p] * 8
        L.lasp_fit_batch_host.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 4 + [C.POINTER(FitOpts)] + \
                                         [C.c_void_p] * 7 + [C.c_int64]
        L.lasp_eval_model.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 2 + [C.POINTER(FitOpts)] + [C.c_void_p] * 2
        L.lasp_eval_grad.argtypes = [C.c_void_p, C.c_int64] + [C.c_void_p] * 4 + [C.POINTER(FitOpts)] + [C.c_void_p] * 5
        L.lasp_eval_grad_static.argtypes = L.lasp_eval_grad.argtypes
        L.lasp_resample_coeffs.argtypes = [C.c_int, C.c_int32, C.c_int32, C.c_double, C.c_double, C.c_void_p, C.c_int32,
                                           C.c_int32, _i32p, _f64p, C.c_void_p, C.c_void_p]
        L.lasp_kernel_variant.argtypes = [C.c_void_p]
        L.lasp_kernel_variant.restype = C.c_int
        L.lasp_launch_info.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int32)]
        L.lasp_fma_executed_per_spectrum_step.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.lasp_fma_executed_per_spectrum_step.restype = C.c_double
        L.lasp_last_fit_stats.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.lasp_launch_count.argtypes = [C.c_void_p]
        L.lasp_launch_count.restype = C.c_int64
        L.lasp_fma_per_spectrum_step.argtypes = [C.c_void_p, C.c_double]
        L.lasp_fma_per_spectrum_step.restype = C.c_double
        L.lasp_last_error.argtypes = [C.c_void_p]
        L.lasp_last_error.restype = C.c_char_p
        L.lasp_version.restype = C.c_int
        _lib = L
    return _lib


def _p(a, t):
    return a.ctypes.data_as(t)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def resample_coeffs(coef_model, lam1, dlam1, seg_offset, loglam, device: int = 0):
    """lasp_resample_coeffs: a [K, q] coefficient table (device tensor or numpy array) on the model's linear grid
    lam1 + m dlam1 -> a [K, n_pix] float32 device tensor on the observed grid (Eq. 2-4 of the paper)."""
    import torch
    if not torch.cuda.is_available():
        raise LaspError("no CUDA device: the LASP path runs only in its sm_100a kernels")
    dev = torch.device("cuda", device)
    if not isinstance(coef_model, torch.Tensor):
        coef_model = torch.from_numpy(np.ascontiguousarray(coef_model, dtype=np.float32))
    coef_model = coef_model.to(dev, torch.float32).contiguous()
    seg = np.ascontiguousarray(seg_offset, dtype=np.int32)
    ll = np.ascontiguousarray(loglam, dtype=np.float64)
    K, q = coef_model.shape
    out = torch.empty((K, ll.size), device=dev, dtype=torch.float32)
    st = C.c_void_p(torch.cuda.current_stream(dev).cuda_stream)
    rc = lib().lasp_resample_coeffs(device, K, q, float(lam1), float(dlam1), _ptr(coef_model), ll.size, seg.size - 1,
                                    _p(seg, _i32p), _p(ll, _f64p), _ptr(out), st)
    if rc != 0:
        raise LaspError(f"lasp_resample_coeffs failed ({rc}): {lib().lasp_last_error(None).decode()}")
    return out


class LaspModel:
    """A lasp_ctx bound to one model description (dict of numpy arrays, see synth.make_model_desc)."""

    def __init__(self, desc: dict, device: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise LaspError("no CUDA device: the LASP path runs only in its sm_100a kernels")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.L = int(desc["n_labels"]); self.K = int(desc["n_terms"]); self.P = int(desc["n_pix"])
        self.NP = self.L + 2; self.D = int(desc["cont_degree"]); self.n_seg = int(desc["n_seg"])
        self.nc = self.n_seg * (self.D + 1)
        k = self._keep = {}
        k["seg_offset"] = np.ascontiguousarray(desc["seg_offset"], dtype=np.int32)
        k["loglam"] = np.ascontiguousarray(desc["loglam"], dtype=np.float64)
        k["seg_sigma_inst"] = np.ascontiguousarray(desc["seg_sigma_inst"], dtype=np.float32)
        k["term_exps"] = np.ascontiguousarray(desc["term_exps"], dtype=np.uint8)
        k["coeffs"] = np.ascontiguousarray(desc["coeffs"], dtype=np.float32)
        k["lo"] = np.ascontiguousarray(desc["lo"], dtype=np.float32)
        k["hi"] = np.ascontiguousarray(desc["hi"], dtype=np.float32)
        k["label_log10"] = np.ascontiguousarray(desc["label_log10"], dtype=np.uint8)
        k["emu_a"] = np.ascontiguousarray(desc["emu_a"], dtype=np.float32)
        k["emu_b"] = np.ascontiguousarray(desc["emu_b"], dtype=np.float32)
        k["seg_n_edge"] = np.ascontiguousarray(desc["seg_n_edge"], dtype=np.int32)
        self.n_models = int(desc.get("n_models", 0))
        k["term_model"] = np.ascontiguousarray(desc.get("term_model", np.zeros(self.K)), dtype=np.uint8)
        k["model_blend"] = np.ascontiguousarray(desc.get("model_blend", np.zeros(4)), dtype=np.float32).reshape(-1)
        d = ModelDesc(self.P, self.n_seg, _p(k["seg_offset"], _i32p), _p(k["loglam"], _f64p),
                      _p(k["seg_sigma_inst"], _f32p), self.L, self.K, _p(k["term_exps"], _u8p),
                      _p(k["coeffs"], _f32p), _p(k["lo"], _f32p), _p(k["hi"], _f32p),
                      _p(k["label_log10"], _u8p), _p(k["emu_a"], _f32p), _p(k["emu_b"], _f32p),
                      self.D, _p(k["seg_n_edge"], _i32p), self.n_models, _p(k["term_model"], _u8p),
                      _p(k["model_blend"], _f32p))
        self.ctx = C.c_void_p()
        rc = lib().lasp_create(C.byref(d), device, C.byref(self.ctx))
        if rc != 0:
            raise LaspError(f"lasp_create failed ({rc}): {lib().lasp_last_error(None).decode()}")

    def close(self):
        if getattr(self, "ctx", None) is not None and self.ctx:
            lib().lasp_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != 0:
            raise LaspError(f"{what} failed ({rc}): {lib().lasp_last_error(self.ctx).decode()}")

    def _dev(self, a, dtype):
        t = self.torch
        if a is None:
            return None
        if not isinstance(a, t.Tensor):
            a = t.from_numpy(np.ascontiguousarray(a))
        return a.to(device=self.device, dtype=dtype).contiguous()

    def _stream(self):
        return C.c_void_p(self.torch.cuda.current_stream(self.device).cuda_stream)

    def reserve(self, B: int):
        self._check(lib().lasp_reserve(self.ctx, B), "lasp_reserve")

    def default_variant(self) -> int:
        """lasp_kernel_variant: 1 = the resident variant serves this model by default, 2 = streaming only."""
        return int(lib().lasp_kernel_variant(self.ctx))

    def launch_info(self, variant: int) -> dict:
        out = (C.c_int32 * 4)()
        self._check(lib().lasp_launch_info(self.ctx, variant, out), "lasp_launch_info")
        return dict(available=bool(out[0]), threads=int(out[1]), ctas_per_sm=int(out[2]), smem_bytes=int(out[3]))

    def fma_executed_per_spectrum_step(self, mean_taps: float, fresh_frac: float) -> float:
        return float(lib().lasp_fma_executed_per_spectrum_step(self.ctx, mean_taps, fresh_frac))

    def last_fit_stats(self) -> dict:
        out = (C.c_double * 2)()
        self._check(lib().lasp_last_fit_stats(self.ctx, out), "lasp_last_fit_stats")
        return dict(group_steps=out[0], fresh_steps=out[1], fresh_frac=(out[1] / out[0] if out[0] else 0.0))

    @staticmethod
    def _opts(n_iter=0, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8, variant=0, emulator_path=0, refresh=0, warm=0,
              fd_fresh=0, stop_window=0, stop_tol=1e-5, clean_every=0, clean_max=0, optimizer=0, lm_lambda0=0.0):
        return FitOpts(int(n_iter), lr, beta1, beta2, eps, int(variant), int(emulator_path), int(refresh), int(warm),
                       int(fd_fresh), int(stop_window), float(stop_tol), int(clean_every), int(clean_max), int(optimizer),
                       float(lm_lambda0))

    def launch_count(self) -> int:
        return int(lib().lasp_launch_count(self.ctx))

    def fma_per_spectrum_step(self, mean_taps: float) -> float:
        return float(lib().lasp_fma_per_spectrum_step(self.ctx, mean_taps))

    def fit_batch(self, flux, ivar, mask, init, n_iter, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8,
                  want_err=True, want_cont=True, out=None, emulator_path=0, variant=0, refresh=0, warm=0, fd_fresh=0,
                  stop_window=0, stop_tol=1e-5, clean_every=0, clean_max=0, optimizer=0, lm_lambda0=0.0):
        """lasp_fit_batch on device tensors; returns dict of device tensors (`mask_out`: the pixels that took part in
        the final evaluation; clean_every > 0 turns the Clean strategy on; optimizer = 1: Levenberg-Marquardt)."""
        t = self.torch
        flux = self._dev(flux, t.float32); ivar = self._dev(ivar, t.float32)
        mask = self._dev(mask, t.uint8); init = self._dev(init, t.float32)
        B = flux.shape[0]
        assert flux.shape == (B, self.P) and ivar.shape == (B, self.P) and init.shape == (B, self.NP)
        if out is None:
            out = dict(params=t.empty((B, self.NP), device=self.device, dtype=t.float32),
                       chi2=t.empty(B, device=self.device, dtype=t.float32),
                       status=t.empty(B, device=self.device, dtype=t.int32),
                       n_steps=t.empty(B, device=self.device, dtype=t.int32),
                       mask_out=t.empty((B, self.P), device=self.device, dtype=t.uint8),
                       cont=t.empty((B, self.nc), device=self.device, dtype=t.float32) if want_cont else None,
                       err=t.empty((B, self.NP), device=self.device, dtype=t.float32) if want_err else None)
        opts = self._opts(n_iter, lr, beta1, beta2, eps, variant, emulator_path, refresh, warm, fd_fresh, stop_window,
                          stop_tol, clean_every, clean_max, optimizer, lm_lambda0)
        rc = lib().lasp_fit_batch(self.ctx, B, _ptr(flux), _ptr(ivar), _ptr(mask), _ptr(init), C.byref(opts),
                                  _ptr(out["params"]), _ptr(out.get("cont")), _ptr(out["chi2"]),
                                  _ptr(out.get("err")), _ptr(out["status"]), _ptr(out.get("n_steps")),
                                  _ptr(out.get("mask_out")), self._stream())
        self._check(rc, "lasp_fit_batch")
        return out

    def fit_batch_host(self, flux, ivar, mask, init, n_iter, lr=1e-2, beta1=0.9, beta2=0.999, eps=1e-8,
                       want_err=True, want_cont=True, chunk=0, out=None, emulator_path=0, variant=0, refresh=0, warm=0,
                       fd_fresh=0, stop_window=0, stop_tol=1e-5, clean_every=0, clean_max=0, want_mask=False,
                       optimizer=0, lm_lambda0=0.0):
        """lasp_fit_batch_host on HOST tensors (torch CPU tensors, pinned for overlap); returns host tensors.
        The library cuts the batch into chunks and overlaps the copies with the fits."""
        t = self.torch

        def host(a, dtype):
            if a is None:
                return None
            if not isinstance(a, t.Tensor):
                a = t.from_numpy(np.ascontiguousarray(a))
            assert a.device.type == "cpu"
            return a.to(dtype).contiguous()

        flux = host(flux, t.float32); ivar = host(ivar, t.float32)
        mask = host(mask, t.uint8); init = host(init, t.float32)
        B = flux.shape[0]
        assert flux.shape == (B, self.P) and ivar.shape == (B, self.P) and init.shape == (B, self.NP)
        if out is None:
            pin = dict(pin_memory=True)
            out = dict(params=t.empty((B, self.NP), dtype=t.float32, **pin), chi2=t.empty(B, dtype=t.float32, **pin),
                       status=t.empty(B, dtype=t.int32, **pin), n_steps=t.empty(B, dtype=t.int32, **pin),
                       mask_out=t.empty((B, self.P), dtype=t.uint8, **pin) if want_mask else None,
                       cont=t.empty((B, self.nc), dtype=t.float32, **pin) if want_cont else None,
                       err=t.empty((B, self.NP), dtype=t.float32, **pin) if want_err else None)
        opts = self._opts(n_iter, lr, beta1, beta2, eps, variant, emulator_path, refresh, warm, fd_fresh, stop_window,
                          stop_tol, clean_every, clean_max, optimizer, lm_lambda0)
        rc = lib().lasp_fit_batch_host(self.ctx, B, _ptr(flux), _ptr(ivar), _ptr(mask), _ptr(init), C.byref(opts),
                                       _ptr(out["params"]), _ptr(out.get("cont")), _ptr(out["chi2"]),
                                       _ptr(out.get("err")), _ptr(out["status"]), _ptr(out.get("n_steps")),
                                       _ptr(out.get("mask_out")), int(chunk))
        self._check(rc, "lasp_fit_batch_host")
        return out

    def eval_model(self, params, cont, variant=0, emulator_path=0):
        t = self.torch
        params = self._dev(params, t.float32); cont = self._dev(cont, t.float32)
        B = params.shape[0]
        assert params.shape == (B, self.NP) and cont.shape == (B, self.nc)
        model = t.empty((B, self.P), device=self.device, dtype=t.float32)
        opts = self._opts(variant=variant, emulator_path=emulator_path)
        rc = lib().lasp_eval_model(self.ctx, B, _ptr(params), _ptr(cont), C.byref(opts), _ptr(model), self._stream())
        self._check(rc, "lasp_eval_model")
        return model

    def eval_grad(self, flux, ivar, mask, params, variant=0, emulator_path=0):
        t = self.torch
        flux = self._dev(flux, t.float32); ivar = self._dev(ivar, t.float32)
        mask = self._dev(mask, t.uint8); params = self._dev(params, t.float32)
        B = flux.shape[0]
        chi2 = t.empty(B, device=self.device, dtype=t.float32)
        grad = t.empty((B, self.NP), device=self.device, dtype=t.float32)
        cont = t.empty((B, self.nc), device=self.device, dtype=t.float32)
        status = t.empty(B, device=self.device, dtype=t.int32)
        opts = self._opts(variant=variant, emulator_path=emulator_path)
        rc = lib().lasp_eval_grad(self.ctx, B, _ptr(flux), _ptr(ivar), _ptr(mask), _ptr(params), C.byref(opts),
                                  _ptr(chi2), _ptr(grad), _ptr(cont), _ptr(status), self._stream())
        self._check(rc, "lasp_eval_grad")
        return dict(chi2=chi2, grad_u=grad, cont=cont, status=status)

    def eval_grad_static(self, flux, ivar, mask, params, variant=0, emulator_path=0, out=None):
        """lasp_eval_grad_static: as eval_grad, but the library allocates nothing (its scratch is a fixed 16 MiB device
        array: small batches only, and calls must not overlap on the GPU).  Pass `out` (dict of device tensors chi2,
        grad_u, cont, status) to keep this wrapper from allocating the outputs too."""
        t = self.torch
        flux = self._dev(flux, t.float32); ivar = self._dev(ivar, t.float32)
        mask = self._dev(mask, t.uint8); params = self._dev(params, t.float32)
        B = flux.shape[0]
        if out is None:
            out = dict(chi2=t.empty(B, device=self.device, dtype=t.float32),
                       grad_u=t.empty((B, self.NP), device=self.device, dtype=t.float32),
                       cont=t.empty((B, self.nc), device=self.device, dtype=t.float32),
                       status=t.empty(B, device=self.device, dtype=t.int32))
        opts = self._opts(variant=variant, emulator_path=emulator_path)
        rc = lib().lasp_eval_grad_static(self.ctx, B, _ptr(flux), _ptr(ivar), _ptr(mask), _ptr(params), C.byref(opts),
                                         _ptr(out["chi2"]), _ptr(out["grad_u"]), _ptr(out["cont"]), _ptr(out["status"]),
                                         self._stream())
        self._check(rc, "lasp_eval_grad_static")
        return out
