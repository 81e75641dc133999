"""Parity of the CUDA path (through the C ABI) against the fp64 oracle, element by element on the
same seeded inputs.  Tolerances are BASELINE.json north_star's, made operational in SURVEY.md 8(c)
C.4:  flux <= 1e-5 * median|model|;  gradient <= 1e-4 * |g|_inf;  continuum ratio <= 1e-4 on fitted
pixels;  after the fit every parameter within 1e-3 of its prior range, chi2 within 1e-4 relative,
errors within 1e-2 relative, status words equal.

Every entry point is exercised on the kernels that are benchmarked: `lasp_eval_model`, `lasp_eval_grad` and
`lasp_fit_batch` all run the group kernels of csrc/lasp_fit_v1.cuh, in the resident variant (variant 1) and in the
streaming variant (variant 2), with the emulator on the FP32 pipe (emulator_path 1) and on the tensor pipe (2).
"""
import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

from helpers import make, small_config, two_arm_config, two_arm_log_config
from paper_2512_24840_b200 import synth

pytestmark = pytest.mark.gpu

TOL_FLUX, TOL_GRAD, TOL_CONT, TOL_PAR, TOL_CHI2, TOL_ERR = 1e-5, 1e-4, 1e-4, 1e-3, 1e-4, 1e-2


@pytest.fixture(scope="module")
def gpu():
    import torch
    from paper_2512_24840_b200 import binding, build
    build.build()
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return binding


def cont_values(desc, cont, i):
    """c_j from plain-Legendre coefficients at the paper's nodes, per segment."""
    n = desc["cont_degree"] + 1
    c = np.empty(desc["n_pix"])
    for k in range(desc["n_seg"]):
        a, b = desc["seg_offset"][k], desc["seg_offset"][k + 1]
        x = -1.0 + 2.0 * np.arange(b - a) / (b - a)
        c[a:b] = npleg.legval(x, cont[i, k * n:(k + 1) * n])
    return c


def fit_weights(case, i):
    d = case["desc"]
    w = case["ivar"][i].astype(np.float64) * case["mask"][i]
    for k in range(d["n_seg"]):
        a, b = d["seg_offset"][k], d["seg_offset"][k + 1]
        ne = d["seg_n_edge"][k]
        w[a:a + ne] = 0
        w[b - ne:b] = 0
    return w


def check_model(gpu, oracle_mod, case, params=None, **kw):
    """lasp_eval_model vs the oracle on EVERY pixel (edges included), at identical (theta, b)."""
    m = gpu.LaspModel(case["desc"])
    params = case["truth"] if params is None else params
    got = m.eval_model(params, case["cont"], **kw).cpu().numpy().astype(np.float64)
    ref = oracle_mod.Oracle(case["desc"]).eval_model(params, case["cont"])
    scale = np.median(np.abs(ref), axis=1, keepdims=True)
    err = np.abs(got - ref) / scale
    assert err.max() <= TOL_FLUX, err.max()
    m.close()
    return got


def check_grad(gpu, oracle_mod, case, params, **kw):
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    g = m.eval_grad(case["flux"], case["ivar"], case["mask"], params, **kw)
    chi2, grad, cont, st = o.eval_grad(case["flux"], case["ivar"], case["mask"], params)
    gg = g["grad_u"].cpu().numpy().astype(np.float64)
    assert np.allclose(g["chi2"].cpu().numpy(), chi2, rtol=TOL_CHI2)
    rel = np.abs(gg - grad).max(axis=1) / np.abs(grad).max(axis=1)
    assert rel.max() <= TOL_GRAD, rel
    gc = g["cont"].cpu().numpy().astype(np.float64)
    for i in range(case["B"]):
        w = fit_weights(case, i)
        ratio = cont_values(case["desc"], gc, i)[w > 0] / cont_values(case["desc"], cont, i)[w > 0]
        assert np.abs(ratio - 1).max() <= TOL_CONT
    assert np.array_equal(g["status"].cpu().numpy(), st)
    m.close()
    return gg


def compare_fit(case, o, r, ref, want_err=True, tol_par=TOL_PAR, tol_chi2=TOL_CHI2):
    par = r["params"].cpu().numpy().astype(np.float64)
    dpar = np.abs(par - ref["params"]) / (o.hi - o.lo)
    assert dpar.max() <= tol_par, dpar.max(axis=0)
    chi = r["chi2"].cpu().numpy().astype(np.float64)
    good = ref["chi2"] > 0
    assert np.abs(chi[good] / ref["chi2"][good] - 1).max() <= tol_chi2
    assert np.array_equal(r["status"].cpu().numpy(), ref["status"])
    # Continuum: the WLS solution is a function of the parameters, so like the flux it is compared AT IDENTICAL
    # PARAMETERS -- the oracle's solve at the parameters the kernel returned -- at 1e-4 on every fitted pixel.  (Against
    # the oracle's OWN final iterate a parameter difference the 1e-3 tolerance allows moves the edge of a degree-30
    # continuum by more than 1e-4: measured 1.9e-4 for dparam = 6e-4 on config-4 shapes with a fresh factor on every
    # step; that comparison is therefore held to the parameter tolerance, 1e-3.)
    n = ref["params"].shape[0]
    gc = r["cont"].cpu().numpy().astype(np.float64)
    same = o.eval_grad(case["flux"][:n], case["ivar"][:n], case["mask"][:n], par)[2]
    for i in range(n):
        w = fit_weights(case, i)
        if ref["status"][i] & 3 or not (w > 0).any():
            continue
        cg = cont_values(case["desc"], gc, i)[w > 0]
        ratio = cg / cont_values(case["desc"], same, i)[w > 0]
        assert np.abs(ratio - 1).max() <= TOL_CONT, (i, np.abs(ratio - 1).max())
        ratio = cg / cont_values(case["desc"], ref["cont"], i)[w > 0]
        assert np.abs(ratio - 1).max() <= max(TOL_PAR, tol_par), (i, np.abs(ratio - 1).max())
    if want_err:
        e = r["err"].cpu().numpy().astype(np.float64)
        ok = np.isfinite(ref["err"]).all(axis=1)
        assert np.array_equal(np.isfinite(e).all(axis=1), ok)
        assert np.abs(e[ok] / ref["err"][ok] - 1).max() <= TOL_ERR, np.abs(e[ok] / ref["err"][ok] - 1).max(axis=0)


def check_fit(gpu, oracle_mod, case, n_iter, lr=1e-2, want_err=True, **kw):
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    r = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], n_iter, lr=lr, want_err=want_err, **kw)
    ref = o.fit(case["flux"], case["ivar"], case["mask"], case["init"], n_iter, lr=lr, want_err=want_err)
    compare_fit(case, o, r, ref, want_err)
    m.close()
    return r, ref


def widest_params(case):
    """|v| and sigma* near the edge of the prior box: the widest supports the layout allows."""
    B, L = case["B"], case["desc"]["n_labels"]
    params = case["init"].copy()
    params[:, L] = np.where(np.arange(B) % 2 == 0, 390.0, -385.0)
    params[:, L + 1] = np.linspace(250.0, 298.0, B)
    return params


# ------------------------------------------------------------------ forward model (lasp_eval_model, group kernels)
# north_star: model flux relative error <= 1e-5, Eq. 5, Eq. 6

@pytest.mark.parametrize("path", [1, 2])
def test_model_flux_config0(gpu, oracle_mod, path):
    check_model(gpu, oracle_mod, synth.make_case(0, oracle_mod.forward, B=64), emulator_path=path)


@pytest.mark.parametrize("path", [1, 2])
def test_model_flux_config1_widest_support(gpu, oracle_mod, path):
    """config-1 shapes at the widest supports of the prior box (H = 28): the T range takes two sweeps of the CTA."""
    case = synth.make_case(1, oracle_mod.forward, B=9)
    check_model(gpu, oracle_mod, case, emulator_path=path)
    check_model(gpu, oracle_mod, case, params=widest_params(case), emulator_path=path)


@pytest.mark.parametrize("path", [1, 2])
def test_model_flux_two_arm_linear(gpu, oracle_mod, path):
    check_model(gpu, oracle_mod, make(two_arm_config(), oracle_mod, B=37), emulator_path=path)


@pytest.mark.parametrize("path", [1, 2])
def test_model_flux_config2_desi_shape(gpu, oracle_mod, path):
    case = synth.make_case(2, oracle_mod.forward, B=8)
    check_model(gpu, oracle_mod, case, emulator_path=path)
    check_model(gpu, oracle_mod, case, params=widest_params(case), emulator_path=path)


@pytest.mark.parametrize("path", [1, 2])
def test_model_flux_config4_high_dim(gpu, oracle_mod, path):
    check_model(gpu, oracle_mod, synth.make_case(4, oracle_mod.forward, B=6), emulator_path=path)


def test_model_flux_streaming_variant(gpu, oracle_mod):
    """variant 2 on shapes that also run resident: config 0, the two-arm linear grid, config 2, and bit-for-bit the same
    stencil inputs give the same flux to rounding order."""
    for case in (synth.make_case(0, oracle_mod.forward, B=13), make(two_arm_config(), oracle_mod, B=5),
                 synth.make_case(2, oracle_mod.forward, B=5)):
        a = check_model(gpu, oracle_mod, case, variant=2)
        b = check_model(gpu, oracle_mod, case, variant=1)
        assert np.abs(a - b).max() <= 2e-6 * np.abs(b).max()


# ------------------------------------------------------------------ chi2 + gradient

def test_grad_config0(gpu, oracle_mod):
    case = synth.make_case(0, oracle_mod.forward, B=64)
    check_grad(gpu, oracle_mod, case, case["init"])


def test_grad_config1_masked(gpu, oracle_mod):
    case = synth.make_case(1, oracle_mod.forward, B=40)  # ragged: ten groups of four
    check_grad(gpu, oracle_mod, case, case["init"])


def test_grad_two_arm_linear(gpu, oracle_mod):
    case = make(two_arm_config(), oracle_mod, B=5)
    check_grad(gpu, oracle_mod, case, case["init"])


def test_grad_config4_high_dim(gpu, oracle_mod):
    case = synth.make_case(4, oracle_mod.forward, B=4)
    check_grad(gpu, oracle_mod, case, case["init"])


def test_grad_widest_kernels_need_two_sweeps(gpu, oracle_mod):
    """|v| and sigma* near the edge of the prior box: support H = 28, the T range no longer fits one sweep of the
    CTA's 192 threads (config-1 shapes), so the emulator / adjoint loops take their second pass."""
    case = synth.make_case(1, oracle_mod.forward, B=9)
    check_grad(gpu, oracle_mod, case, widest_params(case))


def test_grad_two_arm_log_grid(gpu, oracle_mod):
    case = make(two_arm_log_config(), oracle_mod, B=6)   # several uniform segments: slots do not alias
    check_grad(gpu, oracle_mod, case, case["init"])


def test_grad_streaming_variant(gpu, oracle_mod):
    """variant 2 (rows in global scratch, shared-memory window per sweep) on config-1 shapes incl. the widest supports,
    on several uniform segments and on a linear grid."""
    case = synth.make_case(1, oracle_mod.forward, B=10)
    check_grad(gpu, oracle_mod, case, case["init"], variant=2)
    check_grad(gpu, oracle_mod, case, widest_params(case), variant=2)
    case = make(two_arm_log_config(), oracle_mod, B=6)
    check_grad(gpu, oracle_mod, case, case["init"], variant=2)
    case = make(two_arm_config(), oracle_mod, B=5)
    check_grad(gpu, oracle_mod, case, case["init"], variant=2)


# ------------------------------------------------------------------ full fits

def test_fit_config0_all_64(gpu, oracle_mod):
    case = synth.make_case(0, oracle_mod.forward)
    assert case["B"] == 64
    check_fit(gpu, oracle_mod, case, case["config"].n_iter)


def test_fit_config1_subset(gpu, oracle_mod):
    case = synth.make_case(1, oracle_mod.forward, B=48)
    check_fit(gpu, oracle_mod, case, case["config"].n_iter)


def test_fit_two_arm_linear(gpu, oracle_mod):
    case = make(two_arm_config(n_iter=120), oracle_mod, B=9)
    check_fit(gpu, oracle_mod, case, 120)


def test_fit_two_arm_log_grid(gpu, oracle_mod):
    case = make(two_arm_log_config(n_iter=60), oracle_mod, B=7)
    check_fit(gpu, oracle_mod, case, 60)


@pytest.mark.slow
def test_fit_config2_first_64_at_500_steps(gpu, oracle_mod):
    """config 2 (DESI three-arm, per-pixel kernels), first 64 spectra, all 500 Adam steps."""
    case = synth.make_case(2, oracle_mod.forward, B=64)
    check_fit(gpu, oracle_mod, case, case["config"].n_iter)


@pytest.mark.slow
@pytest.mark.parametrize("path", [1, 2])
def test_fit_config4_first_64_at_300_steps(gpu, oracle_mod, path):
    """config 4 (K = 105, 13 labels, three linear-grid arms), first 64 spectra, all 300 steps, emulator on
    the FP32 pipe and on the tensor pipe: the run crosses several mid-run re-factorisations."""
    case = synth.make_case(4, oracle_mod.forward, B=64)
    check_fit(gpu, oracle_mod, case, case["config"].n_iter, emulator_path=path)


# ------------------------------------------------------------------ the stale-factor steps

@pytest.mark.parametrize("policy", [dict(refresh=64), dict(refresh=0), dict(refresh=1)])
def test_iterates_across_refactorisations(gpu, oracle_mod, policy):
    """The iterate u_t itself (not only the end of the fit) against the oracle's at the same t, ten times inside the
    parameter tolerance, for step counts just before, at and after the re-factorisation steps of the fixed schedule
    (fresh on t <= 4 and t = 65, 129): t = 20, 40, 63, 64 end on stale steps up to 60 after a factor, 65, 66 and 129
    right after one.  chi2 at an iterate that has NOT converged magnifies a parameter difference by the (large)
    gradient there: with a stale factor it is held to 1e-3 mid-run (measured <= 3e-4 at t = 20..66, DESIGN.md
    "Stale Gram factor"), with a fresh factor on every step (refresh = 1, the method as written) to the 1e-4 of the
    converged fits."""
    case = synth.make_case(1, oracle_mod.forward, B=8)
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    for n_iter in (1, 5, 20, 40, 63, 64, 65, 66, 129):
        r = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], n_iter, **policy)
        ref = o.fit(case["flux"], case["ivar"], case["mask"], case["init"], n_iter)
        compare_fit(case, o, r, ref, tol_par=1e-4, tol_chi2=TOL_CHI2 if policy["refresh"] == 1 else 1e-3)
    st = m.last_fit_stats()
    assert st["group_steps"] == 2 * 129
    expect = {64: 2 * 6, 1: 2 * 129}.get(policy["refresh"])   # warm steps 1-4, then t = 65 and 129
    if expect is not None:
        assert st["fresh_steps"] == expect
    else:
        assert 2 * 5 <= st["fresh_steps"] <= 2 * 129
    m.close()


def test_fit_at_the_papers_learning_rate(gpu, oracle_mod):
    """lr = 0.1 for 80 steps, before Adam's late-time bursts make fp32 and fp64 trajectories diverge (SURVEY.md
    section 7): per-step changes are 10x those of the configs, so the adaptive policy must re-factorise far more
    often than every 64th step, and the fit stays inside the tolerances."""
    case = synth.make_case(1, oracle_mod.forward, B=16)
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    r = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 80, lr=0.1)
    ref = o.fit(case["flux"], case["ivar"], case["mask"], case["init"], 80, lr=0.1)
    compare_fit(case, o, r, ref)
    st = m.last_fit_stats()
    assert st["fresh_frac"] > 0.1
    m.close()


def test_fit_linear_grid_long_enough_to_refactor(gpu, oracle_mod):
    """A linear-grid (per-pixel-kernel) fit of 140 steps on config-2 shapes: crosses the re-factorisations at 65 and 129."""
    case = synth.make_case(2, oracle_mod.forward, B=4)
    check_fit(gpu, oracle_mod, case, 140, refresh=64)


# ------------------------------------------------------------------ edge cases

def test_zero_steps_returns_init_and_single_spectrum(gpu, oracle_mod):
    case = make(small_config(), oracle_mod, B=1)
    r, ref = check_fit(gpu, oracle_mod, case, 0, want_err=False)
    assert np.allclose(r["params"].cpu().numpy(), case["init"], rtol=1e-6)


def test_status_bits_and_all_masked(gpu, oracle_mod):
    case = make(small_config(n_iter=5), oracle_mod, B=3)
    o = oracle_mod.Oracle(case["desc"])
    case["mask"][0, :] = 0
    case["flux"][1, :] = -np.abs(case["flux"][1, :])
    case["init"][2, o.L] = 400.0
    r, ref = check_fit(gpu, oracle_mod, case, 0, want_err=False)
    st = r["status"].cpu().numpy()
    assert st[0] & 1 and st[1] & 4 and st[2] & 8
    assert r["chi2"][0].item() == 0.0
    assert np.all(r["cont"][0].cpu().numpy() == 0.0)


def test_masked_pixels_do_not_leak(gpu, oracle_mod):
    """Flux on pixels with w == 0 is never looked at -- not even when it is NaN or Inf (reading R-1)."""
    case = make(small_config(mask_frac=0.1), oracle_mod, B=2)
    m = gpu.LaspModel(case["desc"])
    a = m.eval_grad(case["flux"], case["ivar"], case["mask"], case["init"])
    f2 = case["flux"].copy()
    f2[case["mask"] == 0] = -77.0
    f2[0, np.flatnonzero(case["mask"][0] == 0)[:3]] = [np.nan, np.inf, -np.inf]
    f2[:, :5] = np.nan                       # excluded edge pixels
    b = m.eval_grad(f2, case["ivar"], case["mask"], case["init"])
    assert np.isfinite(a["chi2"].cpu().numpy()).all()
    assert np.array_equal(a["chi2"].cpu().numpy(), b["chi2"].cpu().numpy())
    assert np.array_equal(a["grad_u"].cpu().numpy(), b["grad_u"].cpu().numpy())
    m.close()


def test_nonfinite_input_sets_status_bit_2(gpu, oracle_mod):
    """LASP_ST_NONFINITE on both sides.  Spectrum 0: an infinite weight on a fitted pixel, no Adam step (chi2 = inf,
    system not positive definite).  Spectrum 1: a NaN flux on a fitted pixel with Adam steps -- the gradient is NaN and
    the iterate becomes NaN in the oracle (lasp_oracle.c orc_adam_step) and in the kernel alike: parameters and chi2
    come back NaN with the same status word.  Spectrum 2 is healthy and shares spectrum 1's CTA group: untouched."""
    case = make(small_config(), oracle_mod, B=3)
    o = oracle_mod.Oracle(case["desc"])
    j = case["desc"]["n_pix"] // 2
    case["mask"][:, j] = 1
    iv = case["ivar"].copy(); iv[0, j] = np.inf
    fl = case["flux"].copy(); fl[1, j] = np.nan
    m = gpu.LaspModel(case["desc"])
    for n_iter, flux, ivar in ((0, case["flux"], iv), (6, fl, case["ivar"])):
        r = m.fit_batch(flux, ivar, case["mask"], case["init"], n_iter)
        ref = o.fit(flux, ivar, case["mask"], case["init"], n_iter)
        st = r["status"].cpu().numpy()
        assert np.array_equal(st, ref["status"]), (st, ref["status"])
        bad = 0 if n_iter == 0 else 1
        assert st[bad] & gpu.LASP_ST_NONFINITE and not (st[2] & gpu.LASP_ST_NONFINITE)
        par = r["params"].cpu().numpy()
        assert np.array_equal(np.isnan(par), np.isnan(ref["params"]))
        assert not np.isfinite(r["chi2"][bad].item()) and not np.isfinite(ref["chi2"][bad])
        good = [i for i in range(3) if i != bad]
        assert (np.abs(par[good] - ref["params"][good]) / (o.hi - o.lo)).max() <= TOL_PAR
        assert np.abs(r["chi2"].cpu().numpy()[good] / ref["chi2"][good] - 1).max() <= TOL_CHI2
    m.close()


def test_bad_arguments_return_error_codes(gpu, oracle_mod):
    d = synth.make_model_desc(synth.CONFIGS[0]); d.pop("_rng")
    d2 = dict(d); d2["cont_degree"] = 40
    with pytest.raises(gpu.LaspError):
        gpu.LaspModel(d2)          # LASP_ERR_UNSUPPORTED
    d3 = dict(d); d3["hi"] = d["lo"].copy()
    with pytest.raises(gpu.LaspError):
        gpu.LaspModel(d3)          # lo >= hi
    case = make(small_config(), oracle_mod, B=2)
    m = gpu.LaspModel(case["desc"])
    for bad in (dict(variant=3), dict(emulator_path=3), dict(refresh=-1), dict(fd_fresh=2),
                dict(variant=2, emulator_path=2)):           # the tensor-pipe emulator exists in the resident variant only
        with pytest.raises(gpu.LaspError):
            m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 1, **bad)
    m.close()


# ------------------------------------------------------------------ emulator on the tensor pipe (emulator_path = 2)

def test_grad_tensor_pipe_emulator(gpu, oracle_mod):
    """chi2 / gradient / continuum with T = phi.C formed by mma.sync TF32 on split operands, ragged batch, masked pixels."""
    case = synth.make_case(1, oracle_mod.forward, B=40)
    g2 = check_grad(gpu, oracle_mod, case, case["init"], emulator_path=2)
    g1 = check_grad(gpu, oracle_mod, case, case["init"], emulator_path=1)
    assert not np.array_equal(g1, g2)      # the two paths round differently: path 2 did not silently run path 1
    case = synth.make_case(4, oracle_mod.forward, B=6)     # K = 105: 14 k-steps in four register chunks
    check_grad(gpu, oracle_mod, case, case["init"], emulator_path=2)


def test_fit_tensor_pipe_emulator(gpu, oracle_mod):
    case = synth.make_case(0, oracle_mod.forward)
    check_fit(gpu, oracle_mod, case, case["config"].n_iter, emulator_path=2)
    case = synth.make_case(1, oracle_mod.forward, B=24)
    r2, _ = check_fit(gpu, oracle_mod, case, case["config"].n_iter, emulator_path=2)
    m = gpu.LaspModel(case["desc"])
    r1 = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], case["config"].n_iter, emulator_path=1)
    assert not np.array_equal(r1["params"].cpu().numpy(), r2["params"].cpu().numpy())
    m.close()


# ------------------------------------------------------------------ host pipeline (config 3 path)

def test_fit_batch_host_matches_device_call(gpu, oracle_mod):
    """lasp_fit_batch_host (chunked H2D / fit / D2H) returns exactly what lasp_fit_batch returns, ragged chunks."""
    import torch
    case = synth.make_case(0, oracle_mod.forward, B=37)
    m = gpu.LaspModel(case["desc"])
    dev = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 25)
    host = m.fit_batch_host(torch.from_numpy(case["flux"]).pin_memory(), torch.from_numpy(case["ivar"]).pin_memory(),
                            torch.from_numpy(case["mask"]).pin_memory(), torch.from_numpy(case["init"]).pin_memory(),
                            25, chunk=16)
    for k in ("params", "chi2", "cont", "err", "status"):
        assert torch.equal(host[k], dev[k].cpu()), k
    nomask = m.fit_batch_host(case["flux"], case["ivar"], None, case["init"], 5, chunk=0, want_err=False, want_cont=False)
    assert nomask["err"] is None and torch.isfinite(nomask["chi2"]).all()
    # chunk = 0 (automatic) on a batch large enough for two chunks: 9,001 spectra -> 4,504 + 4,497, groups as in one call
    n = 9001
    tile = lambda a: np.tile(a, (n // 37 + 1, 1))[:n]
    big = {k: tile(case[k]) for k in ("flux", "ivar", "mask", "init")}
    dev = m.fit_batch(big["flux"], big["ivar"], big["mask"], big["init"], 6, want_err=False)
    host = m.fit_batch_host(big["flux"], big["ivar"], big["mask"], big["init"], 6, chunk=0, want_err=False)
    for k in ("params", "chi2", "cont", "status"):
        assert torch.equal(host[k], dev[k].cpu()), k
    m.close()


@pytest.mark.slow
def test_fit_config3_stream_first_and_last_chunk_vs_oracle(gpu, oracle_mod):
    """BASELINE.json config 3 in miniature: ten chunks streamed from pinned host memory through lasp_fit_batch_host, all
    500 Adam steps; the first 128 spectra of chunk 0 and of chunk 9 are compared with the oracle."""
    import torch
    cfg = synth.CONFIGS[3]
    base = synth.make_case(3, oracle_mod.forward, B=256)
    chunk, nchunk = 384, 10
    idx = np.arange(chunk * nchunk) % 256
    idx[:128] = np.arange(128)                                   # chunk 0 starts with base spectra 0..127
    idx[9 * chunk:9 * chunk + 128] = np.arange(128, 256)         # chunk 9 with base spectra 128..255
    m = gpu.LaspModel(base["desc"])
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a[idx])).pin_memory()
    r = m.fit_batch_host(pin(base["flux"]), pin(base["ivar"]), pin(base["mask"]), pin(base["init"]), cfg.n_iter,
                         lr=cfg.lr, chunk=chunk)
    o = oracle_mod.Oracle(base["desc"])
    ref = o.fit(base["flux"], base["ivar"], base["mask"], base["init"], cfg.n_iter, lr=cfg.lr)
    for lo, sel in ((0, slice(0, 128)), (9 * chunk, slice(128, 256))):
        sub = {k: (v[lo:lo + 128] if v is not None else None) for k, v in r.items()}
        subcase = dict(base, flux=base["flux"][sel], ivar=base["ivar"][sel], mask=base["mask"][sel])
        subref = {k: v[sel] for k, v in ref.items()}
        compare_fit(subcase, o, sub, subref)
    m.close()


# ------------------------------------------------------------------ full size, bench launch configuration

@pytest.mark.slow
def test_fit_config1_full_size_sampled(gpu, oracle_mod):
    """BASELINE.json config 1 at full size (B = 65,536, 500 Adam steps, the grid bench.py launches): the batch is 256
    DISTINCT oracle-generated spectra tiled 256 times; sampled rows across the batch (first, ragged middle, last CTA)
    are compared with the oracle one by one, and every copy of a spectrum must give the same result."""
    import torch
    cfg = synth.CONFIGS[1]
    nb = 256
    base = synth.make_case(1, oracle_mod.forward, B=nb)
    reps = cfg.B // nb
    m = gpu.LaspModel(base["desc"])
    dev = m.device
    tile = lambda a: torch.from_numpy(a).to(dev).repeat(reps, *([1] * (a.ndim - 1)))
    r = m.fit_batch(tile(base["flux"]), tile(base["ivar"]), tile(base["mask"]), tile(base["init"]), cfg.n_iter,
                    lr=cfg.lr)
    par = r["params"].cpu().numpy().astype(np.float64)
    chi = r["chi2"].cpu().numpy().astype(np.float64)
    err = r["err"].cpu().numpy().astype(np.float64)
    st = r["status"].cpu().numpy()
    # property that holds at any size: identical inputs give identical outputs wherever they sit in the grid
    assert np.array_equal(par.reshape(reps, nb, -1), np.broadcast_to(par[:nb], (reps, nb, par.shape[1])))
    assert np.array_equal(chi.reshape(reps, nb), np.broadcast_to(chi[:nb], (reps, nb)))
    sample = [0, 5, 77, 255, nb * 100 + 131, nb * 177 + 18, nb * 201 + 200, cfg.B - nb + 2, cfg.B - 1] + list(range(32, 64))
    idx = sorted({i % nb for i in sample})
    o = oracle_mod.Oracle(base["desc"])
    ref = o.fit(base["flux"][idx], base["ivar"][idx], base["mask"][idx], base["init"][idx], cfg.n_iter, lr=cfg.lr)
    pos = {j: n for n, j in enumerate(idx)}
    for i in sample:
        n = pos[i % nb]
        assert (np.abs(par[i] - ref["params"][n]) / (o.hi - o.lo)).max() <= TOL_PAR, i
        assert abs(chi[i] / ref["chi2"][n] - 1) <= TOL_CHI2, i
        assert np.abs(err[i] / ref["err"][n] - 1).max() <= TOL_ERR, i
        assert st[i] == ref["status"][n], i
    m.close()


# ------------------------------------------------------------------ streaming variant (rows too long for shared memory)

def test_streaming_variant_fits_match_oracle_on_resident_shapes(gpu, oracle_mod):
    """variant 2 forced on shapes the resident variant also takes: config 0 in full, a config-1 subset over all 500
    steps, a two-segment log grid and a linear grid."""
    case = synth.make_case(0, oracle_mod.forward)
    check_fit(gpu, oracle_mod, case, case["config"].n_iter, variant=2)
    case = synth.make_case(1, oracle_mod.forward, B=12)
    check_fit(gpu, oracle_mod, case, case["config"].n_iter, variant=2)
    case = make(two_arm_log_config(n_iter=60), oracle_mod, B=7)
    check_fit(gpu, oracle_mod, case, 60, variant=2)
    case = make(two_arm_config(n_iter=120), oracle_mod, B=9)
    check_fit(gpu, oracle_mod, case, 120, variant=2)


@pytest.mark.slow
def test_fit_long_spectrum_streaming_16_at_100_steps(gpu, oracle_mod):
    """SURVEY.md 8(d) shape "S" (one 17.4 k-pixel segment): its rows do not fit shared memory, so the default variant
    is the streaming one; first 16 spectra, 100 Adam steps, flux and gradient parity included."""
    case = synth.make_case("S", oracle_mod.forward, B=16)
    m = gpu.LaspModel(case["desc"])
    assert m.default_variant() == 2 and not m.launch_info(1)["available"]
    with pytest.raises(gpu.LaspError):
        m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 1, variant=1)
    m.close()
    check_model(gpu, oracle_mod, case)
    check_grad(gpu, oracle_mod, case, case["init"])
    check_fit(gpu, oracle_mod, case, case["config"].n_iter)
    m1 = gpu.LaspModel(synth.make_case(0, oracle_mod.forward, B=1)["desc"])
    assert m1.default_variant() == 1
    m1.close()


# ------------------------------------------------------------------ the paper's stopping rules (NEXT-2)

def test_stopping_rules_structure(gpu, oracle_mod):
    """stop_window = 50 with an infinite tolerance: every spectrum stops at the first testable step (t = 51, 50 updates,
    bit LASP_ST_STOP_TOL) and returns exactly the fixed-step fit of 50 steps; with stop_tol = 0 nothing fires, n_iter
    updates are applied and the result is exactly the fixed-step fit; both as the oracle's orc_fit_stop."""
    case = synth.make_case(1, oracle_mod.forward, B=10)
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    args = (case["flux"], case["ivar"], case["mask"], case["init"])
    r = m.fit_batch(*args, 200, lr=0.05, stop_window=50, stop_tol=1e30)
    fixed = m.fit_batch(*args, 50, lr=0.05)
    assert np.array_equal(r["n_steps"].cpu().numpy(), np.full(10, 50))
    st = r["status"].cpu().numpy()
    assert np.all(st & gpu.LASP_ST_STOP_TOL) and not np.any(st & gpu.LASP_ST_STOP_RISE)
    assert np.array_equal(r["params"].cpu().numpy(), fixed["params"].cpu().numpy())
    ref = o.fit_stop(*args, 200, lr=0.05, tol=1e30)
    compare_fit(case, o, r, ref)
    assert np.array_equal(ref["n_steps"], np.full(10, 50))
    r = m.fit_batch(*args, 70, lr=0.05, stop_window=50, stop_tol=0.0)
    fixed = m.fit_batch(*args, 70, lr=0.05)
    assert np.array_equal(r["n_steps"].cpu().numpy(), np.full(10, 70))
    assert not np.any(r["status"].cpu().numpy() & (gpu.LASP_ST_STOP_TOL | gpu.LASP_ST_STOP_RISE))
    assert np.array_equal(r["params"].cpu().numpy(), fixed["params"].cpu().numpy())
    assert np.array_equal(fixed["n_steps"].cpu().numpy(), np.full(10, 70))      # fixed-step mode reports n_iter
    m.close()


@pytest.mark.slow
def test_stopping_rules_at_the_papers_settings(gpu, oracle_mod):
    """lr = 0.1, at most 5000 iterations, window 50, tolerance 1e-5 on config-0 and config-1 subsets.
    The stop step is decided by a floating-point comparison on a loss that the two sides hold in different precision
    (fp32 / fp64), so it is unique only up to the step at which |L_t - L_(t-50)| crosses the tolerance within rounding:
    the rule that fired must be the same, the stop step within a few steps, and parameters / chi2 / status inside the
    usual tolerances.  Spectra of one CTA group stop at different steps (the stopped ones are frozen while the group
    runs on): each must equal the kernel's own fixed-step fit cut at its stop step."""
    for cfg_id, B in ((0, 24), (1, 24)):
        case = synth.make_case(cfg_id, oracle_mod.forward, B=B)
        m = gpu.LaspModel(case["desc"])
        o = oracle_mod.Oracle(case["desc"])
        args = (case["flux"], case["ivar"], case["mask"], case["init"])
        r = m.fit_batch(*args, 5000, lr=0.1, stop_window=50, stop_tol=1e-5)
        ref = o.fit_stop(*args, 5000, lr=0.1)
        ns, st = r["n_steps"].cpu().numpy(), r["status"].cpu().numpy()
        assert np.all(ref["n_steps"] < 5000) and np.all(ns < 5000)
        assert np.array_equal(st & 48, ref["status"] & 48)                      # the same criterion fired
        assert np.abs(ns - ref["n_steps"]).max() <= 5, (ns, ref["n_steps"])
        ref_cmp = dict(ref, status=ref["status"])
        compare_fit(case, o, r, ref_cmp)
        assert len(set(ns[:4].tolist())) > 1 or len(set(ns.tolist())) > 1         # stop steps do differ between spectra
        for n in sorted(set(ns.tolist()))[:3]:
            fixed = m.fit_batch(*args, int(n), lr=0.1)
            sel = ns == n
            assert np.array_equal(r["params"].cpu().numpy()[sel], fixed["params"].cpu().numpy()[sel])
        m.close()


# ------------------------------------------------------------------------------------------------
# Clean-strategy masking, against oracle/lasp_oracle.c orc_fit_clean
# ------------------------------------------------------------------------------------------------
def _contaminate(case, seed):
    """Cosmic-ray-like spikes and a few-pixel emission feature on every spectrum (what the Clean strategy is for)."""
    rng = np.random.default_rng(seed)
    flux = case["flux"].copy()
    P = case["desc"]["n_pix"]
    hits = []
    for i in range(case["B"]):
        j = rng.choice(np.arange(40, P - 40), size=6, replace=False)
        amp = rng.uniform(0.4, 2.0, size=6) * np.median(np.abs(flux[i]))
        flux[i, j] += amp.astype(flux.dtype)
        k = int(rng.integers(60, P - 60))
        bump = np.array([0.3, 0.8, 1.0, 0.7, 0.25]) * 0.9 * np.median(np.abs(flux[i]))
        flux[i, k:k + 5] += bump.astype(flux.dtype)
        hits.append(np.concatenate([j, [k + 1, k + 2, k + 3]]))
    return flux, hits


def _check_clean(gpu, oracle_mod, case, n_iter, lr, every=30, seed=5, min_same=0.75):
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    flux, hits = _contaminate(case, seed)
    args = (flux, case["ivar"], case["mask"], case["init"])
    r = m.fit_batch(*args, n_iter, lr=lr, clean_every=every)
    ref = o.fit_clean(*args, n_iter, lr=lr, every=every)
    mg = r["mask_out"].cpu().numpy()
    B, P = mg.shape
    # integer work: the masks.  The clipping thresholds compare float residuals (fp32 here, fp64 in the oracle) with
    # k sigma, so a pixel within rounding of a threshold may fall on either side: what is unique is compared exactly
    # (every pixel the oracle clips by a clear margin, every pixel it keeps by a clear margin), the rest must be few.
    w0 = np.stack([fit_weights(case, i) for i in range(B)]) > 0
    assert not np.any(mg & ~w0) and not np.any(ref["mask"] & ~w0)              # masks only shrink (R-9)
    diff = (mg != ref["mask"]).sum(axis=1)
    same = diff == 0
    assert same.mean() >= min_same, diff
    assert diff.sum() <= 2e-4 * B * P + 2, diff
    for i in range(B):
        inside = w0[i][hits[i]]
        assert np.all(mg[i][hits[i]][inside] == 0), i                           # the injected outliers are gone
    clipped = (w0 & (mg == 0)).sum(axis=1)
    assert np.all(clipped >= 6) and np.all(clipped < 0.06 * P)
    # the final evaluation, at identical parameters and identical mask: chi2 and continuum
    par = r["params"].cpu().numpy().astype(np.float64)
    chi_same, _, cont_same, st_same = o.eval_grad(flux, case["ivar"], mg, par)
    chi = r["chi2"].cpu().numpy().astype(np.float64)
    assert np.abs(chi / chi_same - 1).max() <= TOL_CHI2
    assert np.array_equal(r["status"].cpu().numpy(), st_same)
    gc = r["cont"].cpu().numpy().astype(np.float64)
    for i in range(B):
        keep = mg[i] > 0
        ratio = cont_values(case["desc"], gc, i)[keep] / cont_values(case["desc"], cont_same, i)[keep]
        assert np.abs(ratio - 1).max() <= TOL_CONT, (i, np.abs(ratio - 1).max())
    # the whole fit, where the two sides took the same clipping decisions
    dpar = np.abs(par - ref["params"]) / (o.hi - o.lo)
    assert dpar[same].max() <= TOL_PAR, dpar.max(axis=1)
    assert np.abs(chi[same] / ref["chi2"][same] - 1).max() <= 10 * TOL_CHI2
    e = r["err"].cpu().numpy().astype(np.float64)
    ok = same & np.isfinite(ref["err"]).all(axis=1)
    assert np.abs(e[ok] / ref["err"][ok] - 1).max() <= TOL_ERR
    # where a borderline pixel differs the fits still agree to a few tolerances (one pixel of ~1e3 changes little)
    assert dpar.max() <= 5 * TOL_PAR, dpar.max(axis=1)
    m.close()
    return r, ref, same


def test_clean_strategy_small_model(gpu, oracle_mod):
    """Config-0-like single-segment model, mask updates after steps 30, 60, 90, 120 of 150."""
    case = make(small_config(snr=(60.0, 60.0)), oracle_mod, B=18)     # 18: a ragged last group
    _check_clean(gpu, oracle_mod, case, 150, 0.03)


def test_clean_strategy_config1_shapes(gpu, oracle_mod):
    """LAMOST-like spectra (config 1 shapes), the paper's schedule (every 30 steps, at most 11 updates): 12 updates
    would fit into 360 steps, the 12th must not happen (the oracle stops at 11 too)."""
    case = synth.make_case(1, oracle_mod.forward, B=12)
    _check_clean(gpu, oracle_mod, case, 365, 0.02)


def test_clean_off_reports_the_input_mask(gpu, oracle_mod):
    """mask_out without Clean is the staged mask: ivar * mask != 0 away from the segment edges, on several segments too;
    and a fit with clean_every > n_iter is bit-identical to the fit without Clean."""
    for case in (make(two_arm_config(), oracle_mod), make(small_config(), oracle_mod, B=6)):
        m = gpu.LaspModel(case["desc"])
        args = (case["flux"], case["ivar"], case["mask"], case["init"])
        r = m.fit_batch(*args, 5)
        w0 = np.stack([fit_weights(case, i) for i in range(case["B"])]) > 0
        assert np.array_equal(r["mask_out"].cpu().numpy() > 0, w0)
        if case["desc"]["n_seg"] == 1:
            r2 = m.fit_batch(*args, 5, clean_every=30)
            for k in ("params", "chi2", "cont", "err", "mask_out"):
                assert np.array_equal(r[k].cpu().numpy(), r2[k].cpu().numpy(), equal_nan=True), k
        m.close()


def test_clean_unsupported_combinations(gpu, oracle_mod):
    """Several segments and the streaming variant: LASP_ERR_UNSUPPORTED."""
    case = make(two_arm_config(), oracle_mod)
    m = gpu.LaspModel(case["desc"])
    with pytest.raises(gpu.LaspError, match="Clean"):
        m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 5, clean_every=2)
    m.close()
    case = make(small_config(), oracle_mod, B=4)
    m = gpu.LaspModel(case["desc"])
    args = (case["flux"], case["ivar"], case["mask"], case["init"])
    with pytest.raises(gpu.LaspError, match="Clean"):
        m.fit_batch(*args, 5, clean_every=2, variant=2)
    with pytest.raises(gpu.LaspError):
        m.fit_batch(*args, 5, clean_every=-1)
    m.close()


def test_clean_strategy_with_stopping_rules(gpu, oracle_mod):
    """The paper's full loop: lr 0.1, stopping rules (window 50, tolerance 1e-5) and mask updates every 30
    steps in the same run, on contaminated config-1 shapes.  Stop steps are unique only up to the rounding of the
    tolerance test (as in test_stopping_rules_at_the_papers_settings), the masks up to threshold rounding."""
    case = synth.make_case(1, oracle_mod.forward, B=12)
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    flux, hits = _contaminate(case, 9)
    args = (flux, case["ivar"], case["mask"], case["init"])
    r = m.fit_batch(*args, 5000, lr=0.1, stop_window=50, stop_tol=1e-5, clean_every=30)
    ref = o.fit_clean(*args, 5000, lr=0.1, every=30, window=50, tol=1e-5)
    ns, st, mg = r["n_steps"].cpu().numpy(), r["status"].cpu().numpy(), r["mask_out"].cpu().numpy()
    assert np.all(ref["n_steps"] < 5000) and np.array_equal(st & 48, ref["status"] & 48)
    assert np.abs(ns - ref["n_steps"]).max() <= 5, (ns, ref["n_steps"])
    diff = (mg != ref["mask"]).sum(axis=1)
    assert (diff == 0).mean() >= 0.75 and diff.sum() <= 4, diff
    same = diff == 0
    par = r["params"].cpu().numpy().astype(np.float64)
    dpar = np.abs(par - ref["params"]) / (o.hi - o.lo)
    assert dpar[same].max() <= TOL_PAR, dpar.max(axis=1)
    chi = r["chi2"].cpu().numpy().astype(np.float64)
    assert np.abs(chi[same] / ref["chi2"][same] - 1).max() <= 10 * TOL_CHI2
    for i in range(case["B"]):
        assert np.all(mg[i][hits[i]] == 0) or not np.all(fit_weights(case, i)[hits[i]] > 0)
    # structure: infinite tolerance with window 40 = the fixed-step Clean fit of 40 steps (one mask update, after step 30)
    a = m.fit_batch(*args, 200, lr=0.05, stop_window=40, stop_tol=1e30, clean_every=30)
    b = m.fit_batch(*args, 40, lr=0.05, clean_every=30)
    assert np.array_equal(a["n_steps"].cpu().numpy(), np.full(12, 40))
    for k in ("params", "mask_out"):
        assert np.array_equal(a[k].cpu().numpy(), b[k].cpu().numpy()), k
    m.close()


# ------------------------------------------------------------------------------------------------
# Levenberg-Marquardt on the NP x NP system, against oracle/lasp_oracle.c orc_fit_lm
# ------------------------------------------------------------------------------------------------
def _check_lm(gpu, oracle_mod, case, n_iter, tol_chi2=TOL_CHI2, **kw):
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    args = (case["flux"], case["ivar"], case["mask"], case["init"])
    r = m.fit_batch(*args, n_iter, optimizer=1, **kw)
    ref = o.fit_lm(*args, n_iter)
    compare_fit(case, o, r, ref, tol_chi2=tol_chi2)
    # accepted steps: equal while chi2 still falls by more than rounding; at convergence the fp32 and fp64 sides may
    # accept or reject differently (chi2' < chi2 within rounding), so only the early count is unique
    ns = r["n_steps"].cpu().numpy()
    assert np.all(ns >= np.minimum(ref["n_steps"], 3)) and np.all(ns <= n_iter)
    m.close()
    return r, ref


def test_lm_first_iterations_match_oracle(gpu, oracle_mod):
    """1, 2 and 3 LM iterations from the initial guesses: far from convergence every step is accepted on both sides and
    the iterates agree to the parameter tolerance (the Jacobian is a central difference of step 2e-3 in fp32 here, 1e-5 in
    fp64 in the oracle: the truncation error of the step is O(h^2)).  The first step agrees to the strict chi2 tolerance;
    from the second on the iterates sit on a steep slope of chi2 (it still falls by tens of percent per step) and the step
    itself carries the fp32 rounding of J amplified by the conditioning of J^T J along the weakly determined directions
    (measured: du ~ 7e-5, chi2 4e-4 relative on the least converged spectrum, with or without fd_fresh), so chi2 there is
    held to 1e-3 as for the mid-run Adam iterates of test_iterates_across_refactorisations; parameters stay within 1e-3
    of the range throughout, and the minimum LM converges to meets every tolerance
    (test_lm_converged_fit_config1_and_linear_grid)."""
    case = make(small_config(snr=(60.0, 60.0)), oracle_mod, B=10)
    for n in (1, 2, 3):
        for fresh in (0, 1):
            r, ref = _check_lm(gpu, oracle_mod, case, n, tol_chi2=TOL_CHI2 if n == 1 else 1e-3, fd_fresh=fresh)
            assert np.array_equal(r["n_steps"].cpu().numpy(), ref["n_steps"])


def test_lm_converged_fit_config1_and_linear_grid(gpu, oracle_mod):
    """12 LM iterations: the minimiser of the oracle's LM (= MINPACK's, test_oracle_pins) within the usual tolerances, on
    config-1 shapes, on two linear-grid arms (per-pixel kernels) and on the streaming variant; and the same point the
    500-step Adam fit of the kernel reaches."""
    case = synth.make_case(1, oracle_mod.forward, B=14)
    r, ref = _check_lm(gpu, oracle_mod, case, 12)
    m = gpu.LaspModel(case["desc"])
    adam = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 500)
    o = oracle_mod.Oracle(case["desc"])
    d = np.abs(adam["params"].cpu().numpy() - r["params"].cpu().numpy()) / (o.hi - o.lo)
    assert d.max() <= TOL_PAR, d.max(axis=0)
    m.close()
    _check_lm(gpu, oracle_mod, make(two_arm_config(), oracle_mod), 12)
    _check_lm(gpu, oracle_mod, make(small_config(), oracle_mod, B=6), 10, variant=2)


def test_lm_zero_iterations_and_unsupported(gpu, oracle_mod):
    case = make(small_config(), oracle_mod, B=5)
    _check_lm(gpu, oracle_mod, case, 0)
    m = gpu.LaspModel(case["desc"])
    args = (case["flux"], case["ivar"], case["mask"], case["init"])
    with pytest.raises(gpu.LaspError, match="Levenberg"):
        m.fit_batch(*args, 3, optimizer=1, clean_every=2)
    with pytest.raises(gpu.LaspError, match="Levenberg"):
        m.fit_batch(*args, 3, optimizer=1, stop_window=2)
    with pytest.raises(gpu.LaspError):
        m.fit_batch(*args, 3, optimizer=2)
    m.close()


# ------------------------------------------------------------------------------------------------
# Flux-conserving resampler (step 3, Eq. 2-4), against orc_resample_coeffs
# ------------------------------------------------------------------------------------------------
def _elodie_like_table(K, seed):
    """A [K, 14501] coefficient table on the ELODIE grid (3900-6800 A, 0.2 A): smooth rows with narrow lines."""
    rng = np.random.default_rng(seed)
    q = 14501
    lam = 3900.0 + 0.2 * np.arange(q)
    C_ = np.empty((K, q))
    for k in range(K):
        base = rng.normal() * np.sin(lam / rng.uniform(40.0, 400.0) + rng.uniform(0, 6.28))
        lines = np.zeros(q)
        for c0 in rng.uniform(3900.0, 6800.0, 60):
            lines -= rng.uniform(0.05, 0.6) * np.exp(-0.5 * ((lam - c0) / rng.uniform(0.15, 0.8)) ** 2)
        C_[k] = (1.0 if k == 0 else 0.0) + 0.2 * base + lines
    return C_.astype(np.float32)


def test_resample_coeffs_lamost_grid(gpu, oracle_mod):
    """26 terms x 14,501 model pixels onto the 1327-pixel LAMOST grid of P:227 (4200-5700 A, log10 step 1e-4): every
    element within 1e-6 of the scale of its row (float output of an fp64 sum), flux conserved."""
    C_ = _elodie_like_table(26, 11)
    ll = synth.loglam_grid("log10", 4200.0, 5700.0, 1e-4)
    got = gpu.resample_coeffs(C_, 3900.0, 0.2, [0, ll.size], ll).cpu().numpy().astype(np.float64)
    ref = oracle_mod.resample_coeffs(C_.astype(np.float64), 3900.0, 0.2, [0, ll.size], ll)
    assert got.shape == ref.shape == (26, 1327)
    scale = np.abs(ref).max(axis=1, keepdims=True)
    assert (np.abs(got - ref) / scale).max() <= 1e-6
    nodes = oracle_mod.obs_nodes(ll)
    assert np.allclose((got * np.diff(nodes)).sum(axis=1), (ref * np.diff(nodes)).sum(axis=1), rtol=1e-6, atol=1e-4)


def test_resample_coeffs_segments_ragged_and_out_of_range(gpu, oracle_mod):
    """Three linear-grid arms (DESI-like, 0.8 A) reaching beyond both ends of the model grid, a one-pixel segment, a
    non-multiple-of-128 pixel count, and bins narrower than a model pixel (upsampling): all as the oracle; bins wholly
    outside the model carry zero."""
    C_ = _elodie_like_table(7, 12)
    lam = 3600.0 + 0.8 * np.arange(4200)                       # 3600 .. 6959 A: both ends beyond 3900-6800
    ll = np.log10(lam)
    seg = [0, 1500, 1501, 4200]
    got = gpu.resample_coeffs(C_, 3900.0, 0.2, seg, ll).cpu().numpy().astype(np.float64)
    ref = oracle_mod.resample_coeffs(C_.astype(np.float64), 3900.0, 0.2, seg, ll)
    scale = np.abs(ref).max(axis=1, keepdims=True)
    assert (np.abs(got - ref) / scale).max() <= 1e-6
    assert np.all(got[:, lam < 3899.0] == 0.0) and np.all(got[:, lam > 6801.0] == 0.0)
    fine = np.log10(4500.0 + 0.05 * np.arange(777))            # 0.05 A bins inside 0.2 A model pixels
    got = gpu.resample_coeffs(C_, 3900.0, 0.2, [0, 777], fine).cpu().numpy().astype(np.float64)
    ref = oracle_mod.resample_coeffs(C_.astype(np.float64), 3900.0, 0.2, [0, 777], fine)
    assert (np.abs(got - ref) / np.abs(ref).max(axis=1, keepdims=True)).max() <= 1e-6
    with pytest.raises(gpu.LaspError):
        gpu.resample_coeffs(C_, 3900.0, 0.0, [0, 777], fine)
    with pytest.raises(gpu.LaspError):
        gpu.resample_coeffs(C_, 3900.0, 0.2, [0, 700], fine)


# ------------------------------------------------------------------------------------------------
# Piecewise emulator: three polynomial models over five Teff regimes (Eq. 1; NEXT-3, reading R-15)
# ------------------------------------------------------------------------------------------------
def _regime_params(case):
    """Parameters that visit every regime, both overlaps and the four borders' neighbourhoods."""
    teff = np.array([3300.0, 3990.0, 4010.0, 4275.0, 4540.0, 4560.0, 5800.0, 6990.0, 7010.0, 8000.0, 8990.0, 9010.0, 11500.0])
    p = np.repeat(case["truth"][:1].astype(np.float64), teff.size, axis=0)
    p[:, 0] = teff
    return p


def test_piecewise_emulator_flux_and_gradient(gpu, oracle_mod):
    """Config E (25 / 26 / 19 terms, 1327 LAMOST pixels): lasp_eval_model within 1e-5 and lasp_eval_grad within 1e-4 of the
    oracle in every regime and inside both cross-fades (the Teff component carries the d omega / d Teff term)."""
    case = synth.make_case("E", oracle_mod.forward, B=13)
    params = _regime_params(case)
    for path in (1, 2):
        check_model(gpu, oracle_mod, case, emulator_path=path)
        check_model(gpu, oracle_mod, case, params=params, emulator_path=path)
    check_grad(gpu, oracle_mod, case, case["init"])
    check_grad(gpu, oracle_mod, case, params)
    check_grad(gpu, oracle_mod, case, params, variant=2)


def test_piecewise_emulator_fit(gpu, oracle_mod):
    """Fits on config E (Teff from 3500 to 11000 K, initial guesses up to 500 K away: iterates cross regime borders), 300
    Adam steps, and 10 LM iterations, against the oracle."""
    case = synth.make_case("E", oracle_mod.forward, B=24)
    check_fit(gpu, oracle_mod, case, 300)
    _check_lm(gpu, oracle_mod, case, 10)


def test_two_live_contexts_of_different_shapes(gpu, oracle_mod):
    """The dynamic shared-memory limit is an attribute of the kernel function, shared by every ctx on the device: creating
    a second ctx for a smaller model must not lower it under the first one's launches (cudaLaunchKernel: invalid argument),
    in either order of creation and use."""
    big = synth.make_case(1, oracle_mod.forward, B=6)
    small = make(small_config(), oracle_mod, B=5)
    m_big = gpu.LaspModel(big["desc"])
    m_small = gpu.LaspModel(small["desc"])                 # created after, launched before
    for m, case in ((m_small, small), (m_big, big), (m_small, small)):
        o = oracle_mod.Oracle(case["desc"])
        g = m.eval_grad(case["flux"], case["ivar"], case["mask"], case["init"])
        chi2, grad, _, _ = o.eval_grad(case["flux"], case["ivar"], case["mask"], case["init"])
        gg = g["grad_u"].cpu().numpy().astype(np.float64)
        assert (np.abs(gg - grad).max(axis=1) / np.abs(grad).max(axis=1)).max() <= TOL_GRAD
        r = m.fit_batch(case["flux"], case["ivar"], case["mask"], case["init"], 3)
        assert np.isfinite(r["chi2"].cpu().numpy()).all()
        m.eval_model(case["truth"], case["cont"])
    m_big.close(); m_small.close()


def test_config1_launch_stays_under_the_196k_carveout(gpu):
    """Two CTAs of the config-1 shape must fit the 196 KB shared-memory carveout (60 KB of L1 left; the next step, 228 KB,
    leaves 28 KB and costs 2 %): 2 x (dynamic + static block state <= 1792 + 1024 reserved) <= 200,704 B,
    without the stopping rules and with the paper's window of 50."""
    cfg = synth.CONFIGS[1]
    desc = synth.make_model_desc(cfg)
    desc.pop("_rng")
    m = gpu.LaspModel(desc)
    info = m.launch_info(1)
    assert info["available"] and info["ctas_per_sm"] == 2 and info["threads"] == 192
    for window in (0, 50):
        assert 2 * (info["smem_bytes"] + 16 * window + 1792 + 1024) <= 196 * 1024, info
    m.close()


def test_stopping_rules_streaming_variant_and_largest_window(gpu, oracle_mod):
    """The stopping rules on the streaming variant stop at the resident variant's steps (same arithmetic, other rounding
    order: parameters within the tolerance, same criterion), and the largest window (128: the launch then asks for the
    whole history ring, lasp_gpu.cu launch()) works."""
    case = synth.make_case(1, oracle_mod.forward, B=12)
    m = gpu.LaspModel(case["desc"])
    o = oracle_mod.Oracle(case["desc"])
    args = (case["flux"], case["ivar"], case["mask"], case["init"])
    a = m.fit_batch(*args, 5000, lr=0.1, stop_window=50, stop_tol=1e-5, variant=1)
    b = m.fit_batch(*args, 5000, lr=0.1, stop_window=50, stop_tol=1e-5, variant=2)
    na, nb = a["n_steps"].cpu().numpy(), b["n_steps"].cpu().numpy()
    assert np.abs(na - nb).max() <= 5 and np.array_equal(a["status"].cpu().numpy(), b["status"].cpu().numpy())
    d = np.abs(a["params"].cpu().numpy() - b["params"].cpu().numpy()) / (o.hi - o.lo)
    assert d.max() <= TOL_PAR
    c = m.fit_batch(*args, 400, lr=0.02, stop_window=128, stop_tol=1e-5)      # (a tolerance near the fp32 resolution of
    ref = o.fit_stop(*args, 400, lr=0.02, window=128, tol=1e-5)                # L ~ 1, e.g. 1e-7, moves the stop by ~10 steps)
    assert np.abs(c["n_steps"].cpu().numpy() - ref["n_steps"]).max() <= 5
    assert np.array_equal(c["status"].cpu().numpy() & 48, ref["status"] & 48)
    m.close()
