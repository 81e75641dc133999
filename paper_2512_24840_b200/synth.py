"""Seeded synthetic inputs shaped like the paper's workloads.

This module serves BOTH the fp64 oracle (tests) and the CUDA path (tests, bench): it only
draws random numbers and lays out arrays.  It holds none of the method's arithmetic -- model
spectra are produced by a ``forward`` callable the caller passes in (the oracle in the parity
tests, the parity-checked CUDA forward kernel for the bulk batches of ``bench.py``).

The inputs stand in for LAMOST DR10 (~1.3-1.5 k pixels on a log10 grid of step
1e-4) and DESI DR1 (three-arm format of BASELINE.json config 2), which are not available.

Recipe (master seed ``251224840 + 1000*cfg``, ``numpy.random.Generator(PCG64)``; draw order:
coefficients, truth, continuum, SNR, initial offsets, mask, noise):

* prior box: Teff [3500, 8000] K, log g [0, 6], [Fe/H] [-3, 1], abundances [-1, 1],
  RV [-400, 400] km/s, sigma* [20, 300] km/s;
* emulator inputs x_l = label mapped affinely to [-1, 1] over the box (Teff through log10);
* coefficients: C[0,:] = 1, C[k,:] = 0.3/sqrt(K-1) * N(0,1) / rms(phi_k), rms over
  x ~ U(-1,1)^L, so the flux is 1 +- 0.3 (BASELINE.json config 0);
* truth: Teff U(4000,7500), log g U(1,5), [Fe/H] U(-2.5,0.5), abundances U(-0.5,0.5),
  RV U(-200,200), sigma* U(50,150); continuum b_0 = 1, b_n ~ N(0, 0.05) per segment;
* initial guess: truth + U(+-500 K, +-1, +-0.5, +-100 km/s), sigma* = 100, abundances 0;
* noise: sigma = median(model)/SNR per spectrum (configs 0,1,3,4,S), or
  var_j = alpha*max(model_j,0) + rho^2 with rho^2 = 0.2 med^2/SNR^2, alpha = med/(1.25 SNR^2)
  (config 2); ivar = 1/var;
* masked pixels get mask = 0 AND flux = 1e3, so a leak of a masked pixel shows in chi2.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

C_KMS = 299792.458
MASTER_SEED = 251224840

BOX = {
    "teff": (3500.0, 8000.0),
    "logg": (0.0, 6.0),
    "feh": (-3.0, 1.0),
    "abund": (-1.0, 1.0),
    "rv": (-400.0, 400.0),
    "sigma": (20.0, 300.0),
}


@dataclass
class Config:
    """One workload of BASELINE.json `configs` (restated in SURVEY.md 8(d))."""

    cfg: int | str
    name: str
    B: int
    grid: str  # "log10" or "linear"
    lam_min: float
    lam_max: float
    step: float
    seg_bounds: tuple  # pixel offsets, len n_seg+1 (None -> single segment)
    sigma_inst: tuple
    K: int
    L: int
    D: int
    n_iter: int
    snr: tuple  # (lo, hi) log-uniform, or (v, v) fixed
    noise: str  # "const" | "poisson"
    mask_frac: float
    parity_B: int
    lr: float = 1e-2
    beta1: float = 0.9
    beta2: float = 0.999
    eps: float = 1e-8
    seed: int = field(default=0)
    # piecewise emulator (Eq. 1's f_1..f_5): terms per polynomial model, e.g. (25, 26, 19) for the
    # cold / warm / hot models of P:187, and for each model (lo0, lo1, hi0, hi1) in K: its weight rises over [lo0, lo1] and
    # falls over [hi0, hi1] (0, 0 = no ramp on that side).  Empty: one polynomial.
    models: tuple = ()
    model_blend: tuple = ()
    teff_box: tuple = ()       # prior box of Teff (default BOX["teff"])
    teff_truth: tuple = ()     # range of the true Teff (default 4000-7500 K)

    def __post_init__(self):
        idx = self.cfg if isinstance(self.cfg, int) else 9
        self.seed = MASTER_SEED + 1000 * idx


_DESI_SEGS = (0, 2744, 4932, 7781)

CONFIGS = {
    0: Config(0, "tiny-ref", 64, "log10", 3850.0, 5500.0, 1e-4, None, (0.0,), 26, 3, 10, 100,
              (30.0, 30.0), "const", 0.0, 64),
    1: Config(1, "lamost-like", 65536, "log10", 3850.0, 5500.0, 1e-4, None, (0.0,), 26, 3, 30, 500,
              (10.0, 200.0), "const", 0.03, 256),
    2: Config(2, "desi-like", 262144, "linear", 3600.0, 9824.0, 0.8, _DESI_SEGS, (70.0, 55.0, 45.0),
              26, 3, 30, 500, (5.0, 100.0), "poisson", 0.05, 64),
    3: Config(3, "survey-stream", 10_000_000, "log10", 3850.0, 5500.0, 1e-4, None, (0.0,), 26, 3, 30,
              500, (10.0, 200.0), "const", 0.03, 128),
    4: Config(4, "high-dim", 131072, "linear", 3600.0, 9824.0, 0.8, _DESI_SEGS, (70.0, 55.0, 45.0),
              105, 13, 30, 300, (50.0, 50.0), "const", 0.05, 64),
    "S": Config("S", "long-stream", 4096, "log10", 3600.0, 9800.0, 2.5e-5, None, (0.0,), 26, 3, 30,
                100, (50.0, 50.0), "const", 0.03, 16),
    # the paper's own emulator layout: three polynomial models with 25 / 26 / 19 terms (cold <= 4550 K, warm
    # 4000-9000 K, hot >= 7000 K) on the 1327 LAMOST pixels of 4200-5700 A; Teff spans all five regimes of P:72-76
    "E": Config("E", "elodie-like", 16384, "log10", 4200.0, 5700.0, 1e-4, None, (0.0,), 70, 3, 30, 500,
                (10.0, 200.0), "const", 0.03, 32, models=(25, 26, 19),
                model_blend=((0.0, 0.0, 4000.0, 4550.0), (4000.0, 4550.0, 7000.0, 9000.0), (7000.0, 9000.0, 0.0, 0.0)),
                teff_box=(3100.0, 12000.0), teff_truth=(3500.0, 11000.0)),
}


def loglam_grid(grid: str, lam_min: float, lam_max: float, step: float) -> np.ndarray:
    """log10(lambda/A) of the pixel centres.  P:227 / P:377: 4200-5700 A at log10 step 1e-4 is
    1327 pixels, n = floor(log10(max/min)/step) + 1."""
    if grid == "log10":
        n = int(math.floor(math.log10(lam_max / lam_min) / step + 1e-9)) + 1
        return math.log10(lam_min) + step * np.arange(n, dtype=np.float64)
    n = int(math.floor((lam_max - lam_min) / step + 1e-9)) + 1
    return np.log10(lam_min + step * np.arange(n, dtype=np.float64))


def monomial_exps(L: int, K: int) -> np.ndarray:
    """First K monomials of L variables in graded lexicographic order:
    degree 0, then x1, x2, ..; within a degree x1 exponents descend first."""
    def compositions(total, nvar):
        if nvar == 1:
            yield (total,)
            return
        for first in range(total, -1, -1):
            for rest in compositions(total - first, nvar - 1):
                yield (first,) + rest

    out = []
    deg = 0
    while len(out) < K:
        out.extend(compositions(deg, L))
        deg += 1
    return np.asarray(out[:K], dtype=np.uint8)


def param_names(L: int):
    base = ["teff", "logg", "feh"] + [f"x{i}" for i in range(L - 3)]
    return base + ["rv", "sigma"]


def make_model_desc(c: Config, seed: int | None = None) -> dict:
    """Everything `lasp_create` takes (include/lasp_gpu.h: lasp_model_desc) as numpy arrays."""
    rng = np.random.Generator(np.random.PCG64(c.seed if seed is None else seed))
    loglam = loglam_grid(c.grid, c.lam_min, c.lam_max, c.step)
    P = loglam.size
    seg = np.asarray(c.seg_bounds if c.seg_bounds is not None else (0, P), dtype=np.int32)
    assert seg[-1] == P, (seg, P)
    L, K = c.L, c.K
    if c.models:
        assert sum(c.models) == K
        exps = np.concatenate([monomial_exps(L, kr) for kr in c.models])
    else:
        exps = monomial_exps(L, K)
    tbox = c.teff_box if c.teff_box else BOX["teff"]
    lo = np.array([tbox[0], BOX["logg"][0], BOX["feh"][0]] + [BOX["abund"][0]] * (L - 3)
                  + [BOX["rv"][0], BOX["sigma"][0]], dtype=np.float32)
    hi = np.array([tbox[1], BOX["logg"][1], BOX["feh"][1]] + [BOX["abund"][1]] * (L - 3)
                  + [BOX["rv"][1], BOX["sigma"][1]], dtype=np.float32)
    label_log10 = np.zeros(L, dtype=np.uint8)
    label_log10[0] = 1
    tlo = lo[:L].astype(np.float64)
    thi = hi[:L].astype(np.float64)
    tlo[label_log10 == 1] = np.log10(tlo[label_log10 == 1])
    thi[label_log10 == 1] = np.log10(thi[label_log10 == 1])
    emu_a = (2.0 / (thi - tlo)).astype(np.float32)
    emu_b = (-(thi + tlo) / (thi - tlo)).astype(np.float32)
    # coefficients: flux 1 +- 0.3
    rms = np.prod(np.sqrt(1.0 / (2.0 * exps.astype(np.float64) + 1.0)), axis=1)
    extra = {}
    if c.models:
        # one master polynomial (the longest model's terms), and every model a copy of its leading terms with each term
        # scaled by 1 + 0.05 N(0,1): the models agree to a few percent where they overlap, as fitted models of one library do
        km = max(c.models)
        master = rng.standard_normal((km, P)) * (0.3 / math.sqrt(km - 1)) / rms[:km, None]
        master[0, :] = 1.0
        parts = []
        for kr in c.models:
            scale = 1.0 + 0.05 * rng.standard_normal(kr)
            scale[0] = 1.0
            parts.append(master[:kr] * scale[:, None])
        coeffs = np.concatenate(parts)
        extra = dict(n_models=len(c.models),
                     term_model=np.concatenate([np.full(kr, r, dtype=np.uint8) for r, kr in enumerate(c.models)]),
                     model_blend=np.asarray(c.model_blend, dtype=np.float32))
    else:
        coeffs = rng.standard_normal((K, P)) * (0.3 / math.sqrt(max(K - 1, 1))) / rms[:, None]
        coeffs[0, :] = 1.0
    # edge exclusion from the prior box: ceil((max|v| + 5 sigma_tot,max)/s_min)
    n_edge = np.zeros(seg.size - 1, dtype=np.int32)
    vmax = float(max(abs(lo[L]), abs(hi[L])))
    for s in range(seg.size - 1):
        ll = loglam[seg[s]:seg[s + 1]]
        smin = C_KMS * math.log(10.0) * float(np.min(np.diff(ll)))
        stot = math.hypot(float(hi[L + 1]), float(c.sigma_inst[s]))
        n_edge[s] = int(math.ceil((vmax + 5.0 * stot) / smin))
    return dict(
        n_pix=P, n_seg=int(seg.size - 1), seg_offset=seg, loglam=loglam,
        seg_sigma_inst=np.asarray(c.sigma_inst, dtype=np.float32),
        n_labels=L, n_terms=K, term_exps=exps, coeffs=coeffs.astype(np.float32),
        lo=lo, hi=hi, label_log10=label_log10, emu_a=emu_a, emu_b=emu_b,
        cont_degree=c.D, seg_n_edge=n_edge, _rng=rng, **extra,
    )


def draw_params(c: Config, desc: dict, B: int, rng: np.random.Generator) -> dict:
    """Truth, continuum coefficients, SNR and initial guesses for B spectra (draw order fixed)."""
    L = c.L
    truth = np.empty((B, L + 2), dtype=np.float64)
    tt = c.teff_truth if c.teff_truth else (4000.0, 7500.0)
    truth[:, 0] = rng.uniform(tt[0], tt[1], B)
    truth[:, 1] = rng.uniform(1.0, 5.0, B)
    truth[:, 2] = rng.uniform(-2.5, 0.5, B)
    for l in range(3, L):
        truth[:, l] = rng.uniform(-0.5, 0.5, B)
    truth[:, L] = rng.uniform(-200.0, 200.0, B)
    truth[:, L + 1] = rng.uniform(50.0, 150.0, B)
    n = c.D + 1
    cont = rng.standard_normal((B, desc["n_seg"], n)) * 0.05
    cont[:, :, 0] = 1.0
    if c.snr[0] == c.snr[1]:
        snr = np.full(B, c.snr[0])
    else:
        snr = np.exp(rng.uniform(math.log(c.snr[0]), math.log(c.snr[1]), B))
    init = truth.copy()
    init[:, 0] += rng.uniform(-500.0, 500.0, B)
    init[:, 1] += rng.uniform(-1.0, 1.0, B)
    init[:, 2] += rng.uniform(-0.5, 0.5, B)
    for l in range(3, L):
        init[:, l] = 0.0
    init[:, L] += rng.uniform(-100.0, 100.0, B)
    init[:, L + 1] = 100.0
    init = np.clip(init, desc["lo"].astype(np.float64), desc["hi"].astype(np.float64))
    return dict(truth=truth.astype(np.float32), cont=cont.reshape(B, -1).astype(np.float32),
                snr=snr, init=init.astype(np.float32))


def add_noise_numpy(c: Config, model: np.ndarray, snr: np.ndarray, rng: np.random.Generator):
    """mask, noise -> (flux f32, ivar f32, mask u8).  `model` is [B,P]."""
    B, P = model.shape
    mask = (rng.uniform(size=(B, P)) >= c.mask_frac).astype(np.uint8) if c.mask_frac > 0 else \
        np.ones((B, P), dtype=np.uint8)
    z = rng.standard_normal((B, P))
    med = np.median(model, axis=1)
    if c.noise == "poisson":
        rho2 = 0.2 * med ** 2 / snr ** 2
        alpha = med / (1.25 * snr ** 2)
        var = alpha[:, None] * np.maximum(model, 0.0) + rho2[:, None]
    else:
        var = np.broadcast_to(((med / snr) ** 2)[:, None], model.shape)
    flux = model + np.sqrt(var) * z
    flux = np.where(mask == 1, flux, 1e3)
    return flux.astype(np.float32), (1.0 / var).astype(np.float32), mask


def make_case(cfg, forward, B: int | None = None, noise_free: bool = False) -> dict:
    """A full parity case: model description + B spectra.  ``forward(desc, params, cont)`` must
    return the model spectra [B,P] for physical ``params`` [B,NP] and plain-Legendre ``cont``."""
    c = CONFIGS[cfg]
    B = c.parity_B if B is None else B
    desc = make_model_desc(c)
    rng = desc.pop("_rng")
    pr = draw_params(c, desc, B, rng)
    model = np.asarray(forward(desc, pr["truth"], pr["cont"]), dtype=np.float64)
    if noise_free:
        flux = model.astype(np.float32)
        ivar = np.ones_like(flux)
        mask = np.ones(model.shape, dtype=np.uint8)
    else:
        flux, ivar, mask = add_noise_numpy(c, model, pr["snr"], rng)
    return dict(config=c, desc=desc, B=B, flux=flux, ivar=ivar, mask=mask, model=model, **pr)
