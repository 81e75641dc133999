"""Pins for the fp64 oracle (oracle/lasp_oracle.c) against things OTHER than itself:
values the paper prints (tests/golden/paper_values.txt), numpy library routines, closed forms,
finite differences, brute force and statistical invariants.
CPU only: `pytest -m "not gpu"`.
"""
import math
import os

import numpy as np
import pytest
from numpy.polynomial import legendre as npleg

from paper_2512_24840_b200 import synth

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def golden():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or "|" not in line:
            continue
        k, v, _ = [t.strip() for t in line.split("|", 2)]
        out[k] = float(v)
    return out


from helpers import make, small_config, two_arm_config  # noqa: E402


# ---------------------------------------------------------------- grid

def test_grid_pixel_counts_match_paper():
    g = golden()
    assert synth.loglam_grid("log10", 4200.0, 5700.0, 1e-4).size == g["grid_pixels_4200_5700_log10_1e-4"]
    assert synth.loglam_grid("log10", 3850.0, 5500.0, 1e-4).size == g["grid_pixels_3850_5500_log10_1e-4"]
    assert synth.loglam_grid("linear", 3600.0, 9824.0, 0.8).size == 7781  # BASELINE.json configs[4]


def test_pixel_velocity_scale(oracle_mod):
    g = golden()
    case = make(small_config(), oracle_mod, B=1)
    s = oracle_mod.Oracle(case["desc"]).pixel_kms()
    assert np.allclose(s, g["kms_per_pixel_log10_1e-4"], rtol=2e-6)
    # linear grid: s_j = c * dlambda/lambda (Appendix of SURVEY.md: 66.6 km/s at 3600 A, 24.4 at 9824 A)
    d = synth.make_model_desc(synth.CONFIGS[2]); d.pop("_rng")
    s2 = oracle_mod.Oracle(d).pixel_kms()
    lam = 10 ** d["loglam"]
    ends = np.zeros(lam.size, dtype=bool)
    ends[d["seg_offset"][:-1]] = True; ends[d["seg_offset"][1:] - 1] = True
    assert np.allclose(s2[~ends], synth.C_KMS * 0.8 / lam[~ends], rtol=1e-6)   # centred differences
    assert np.allclose(s2[ends], synth.C_KMS * 0.8 / lam[ends], rtol=2e-4)     # one-sided at segment ends
    assert abs(s2[0] - 66.6) < 0.05 and abs(s2[-1] - 24.4) < 0.05


def test_edge_exclusion_rule(oracle_mod):
    # 28 px for configs 0/1/3, 47/61/79 for the three DESI segments
    d = synth.make_model_desc(synth.CONFIGS[1]); d.pop("_rng")
    assert list(d["seg_n_edge"]) == [28]
    d2 = synth.make_model_desc(synth.CONFIGS[2]); d2.pop("_rng")
    assert list(d2["seg_n_edge"]) == [47, 61, 79]
    # and it really covers the largest support of the prior box
    o = oracle_mod.Oracle(d2)
    s = o.pixel_kms()
    for k in range(3):
        a, b = d2["seg_offset"][k], d2["seg_offset"][k + 1]
        st = math.hypot(300.0, float(d2["seg_sigma_inst"][k]))
        Hmax = math.ceil(400.0 / s[a:b].min() + 5 * st / s[a:b].min())
        assert d2["seg_n_edge"][k] >= Hmax


# ---------------------------------------------------------------- emulator (Eq. 1)

def test_term_tables():
    g = golden()
    e = synth.monomial_exps(13, 105)
    assert e.shape[0] == g["quadratic_terms_13_labels"] == 1 + 13 + 13 * 14 // 2
    assert e.sum(axis=1).max() == 2 and len({tuple(r) for r in e}) == 105
    e3 = synth.monomial_exps(3, 26)
    assert (e3[:20].sum(axis=1) <= 3).all() and len({tuple(r) for r in e3[:20]}) == 20
    # then x1^4, x1^3 x2, x1^3 x3, x1^2 x2^2, x1^2 x2 x3, x1^2 x3^2
    assert [tuple(r) for r in e3[20:]] == [(4, 0, 0), (3, 1, 0), (3, 0, 1), (2, 2, 0), (2, 1, 1), (2, 0, 2)]


def test_monomials_brute_force_and_fd(oracle_mod):
    d = synth.make_model_desc(synth.CONFIGS[4]); d.pop("_rng")
    o = oracle_mod.Oracle(d)
    rng = np.random.default_rng(1)
    theta = o.denorm(rng.uniform(-0.9, 0.9, o.NP))
    x, phi, dphi, dxdt = o.monomials(theta[: o.L])
    # x: Teff through log10, the rest affine; all inside [-1,1]
    tau = theta[: o.L].copy()
    tau[0] = math.log10(tau[0])  # only Teff goes through log10 (C.2-19)
    xe = d["emu_a"].astype(np.float64) * tau + d["emu_b"].astype(np.float64)
    assert np.allclose(x, xe, rtol=1e-13, atol=1e-13) and np.all(np.abs(x) <= 1)
    # phi: product definition through numpy power
    ref = np.prod(x[None, :] ** d["term_exps"].astype(np.float64), axis=1)
    assert np.allclose(phi, ref, rtol=1e-13)
    # dphi/dx_l by central differences of the numpy definition
    for l in range(o.L):
        h = 1e-6
        xp, xm = x.copy(), x.copy()
        xp[l] += h; xm[l] -= h
        fd = (np.prod(xp[None, :] ** d["term_exps"], axis=1) - np.prod(xm[None, :] ** d["term_exps"], axis=1)) / (2 * h)
        assert np.allclose(dphi[l], fd, rtol=1e-7, atol=1e-9)
    # chain factor d x / d theta
    assert np.isclose(dxdt[0], d["emu_a"][0] / (theta[0] * math.log(10.0)), rtol=1e-13)
    assert np.allclose(dxdt[1:], d["emu_a"][1:], rtol=1e-13)


def test_emulator_is_einsum_and_constant_term_at_origin(oracle_mod):
    case = make(small_config(), oracle_mod, B=1)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    # tiny broadening, zero shift => S == T to ~1e-12 (pure identity kernel: see test below)
    theta = o.denorm(np.zeros(o.NP))
    theta[o.L] = 0.0
    _, phi, _, _ = o.monomials(theta[: o.L])
    T = np.einsum("k,kp->p", phi, d["coeffs"].astype(np.float64))
    # x = 0 for every label at the box centre (in the emulator's variable) -> only the constant term
    x, phi0, _, _ = o.monomials(np.array([math.sqrt(3500.0 * 8000.0), 3.0, -1.0]))
    assert np.allclose(x, 0.0, atol=1e-6)
    assert np.isclose(phi0[0], 1.0) and np.allclose(phi0[1:], 0.0, atol=1e-6)
    # the oracle's own emulator_row, reached through eval_S with no shift and a vanishing width (sigma* = 1e-3 km/s:
    # H = 1 and the two side taps weigh exp(-1/(2 sigma^2)) = 0, an identity kernel, so S == T), against a brute-force
    # loop over terms with the monomials multiplied out by hand
    theta[o.L + 1] = 1e-3
    S = o.eval_S(theta)[0]
    xx = np.array([float(d["emu_a"][l]) * (math.log10(theta[l]) if d["label_log10"][l] else float(theta[l]))
                   + float(d["emu_b"][l]) for l in range(o.L)], dtype=np.float64)
    for j in list(range(7)) + [d["n_pix"] // 2, d["n_pix"] - 1]:
        acc = 0.0
        for k in range(o.K):
            mono = 1.0
            for l in range(o.L):
                for _ in range(int(d["term_exps"][k, l])):
                    mono *= xx[l]
            acc += mono * float(d["coeffs"][k, j])
        assert abs(acc - S[j]) < 1e-12 and abs(acc - T[j]) < 1e-12


# ---------------------------------------------------------------- kernel (Eq. 5)

def test_kernel_support_rule_and_unit_sum(oracle_mod):
    g = golden()
    H, w, _, _ = oracle_mod.Oracle.kernel_weights(1.3, 2.0)
    assert w.size == g["kernel_length_mu_1.3_sigma_2.0"] and H == 12
    H, w, _, _ = oracle_mod.Oracle.kernel_weights(-2.9, 0.72)
    assert w.size == g["kernel_length_mu_-2.9_sigma_0.72"]
    for mu, sg in [(0.0, 0.3), (2.5, 1.7), (-5.8, 4.3), (0.49, 0.29)]:
        H, w, wm, ws = oracle_mod.Oracle.kernel_weights(mu, sg)
        assert H == math.ceil(abs(mu) + 5 * sg) and w.size == 2 * H + 1
        assert abs(w.sum() - 1.0) < 1e-14
        assert abs(wm.sum()) < 1e-13 and abs(ws.sum()) < 1e-13  # derivatives of a unit-sum kernel
        k = np.arange(-H, H + 1)
        ref = np.exp(-0.5 * ((k - mu) / sg) ** 2)
        assert np.allclose(w, ref / ref.sum(), rtol=1e-13)
        assert np.argmax(w) == H + int(round(mu))  # centred at +mu (C.2-11)


def test_kernel_derivatives_vs_finite_differences(oracle_mod):
    kw = oracle_mod.Oracle.kernel_weights
    for mu, sg in [(0.37, 1.9), (-2.2, 0.8), (3.05, 3.3)]:
        H, w, wm, ws = kw(mu, sg)
        h = 1e-6
        # H held constant (C.2-15): rebuild the perturbed kernels on the same support by hand
        k = np.arange(-H, H + 1)

        def gk(m, s):
            e = np.exp(-0.5 * ((k - m) / s) ** 2)
            return e / e.sum()
        assert np.allclose(wm, (gk(mu + h, sg) - gk(mu - h, sg)) / (2 * h), rtol=1e-6, atol=1e-9)
        assert np.allclose(ws, (gk(mu, sg + h) - gk(mu, sg - h)) / (2 * h), rtol=1e-6, atol=1e-9)


def _line_model(oracle_mod, a_pix=6.0, depth=0.5, **cfgkw):
    """A model whose template is a single Gaussian absorption line: K=1 (constant term only),
    C[0,:] = 1 - depth*exp(-(j-j0)^2/(2 a^2))."""
    case = make(small_config(K=1, D=0, **cfgkw), oracle_mod, B=1)
    d = case["desc"]
    P = d["n_pix"]
    j = np.arange(P)
    d["coeffs"] = (1.0 - depth * np.exp(-0.5 * ((j - P // 2) / a_pix) ** 2))[None, :].astype(np.float32)
    return d, j


def test_shift_direction_and_width_addition(oracle_mod):
    # textbook: Gaussian (width a) convolved with Gaussian (width s) is Gaussian width sqrt(a^2+s^2),
    # centred at +mu: positive RV moves the line to LONGER wavelength (C.2-11, C.2-12).
    d, j = _line_model(oracle_mod, a_pix=6.0)
    o = oracle_mod.Oracle(d)
    s = o.pixel_kms()[0]
    v, sig = 150.0, 120.0
    S = o.eval_S(np.array([[5000.0, 3.0, -1.0, v, sig]]))[0]
    prof = 1.0 - S
    cen = (prof * j).sum() / prof.sum()
    wid = math.sqrt((prof * (j - cen) ** 2).sum() / prof.sum())
    assert abs(cen - (d["n_pix"] // 2 + v / s)) < 2e-3
    assert abs(wid - math.sqrt(6.0 ** 2 + (sig / s) ** 2)) < 2e-3
    assert abs(prof.sum() - 0.5 * 6.0 * math.sqrt(2 * math.pi)) < 1e-4  # flux preserved (C.2-9)


def test_constant_kernel_equals_numpy_convolve(oracle_mod):
    case = make(small_config(), oracle_mod, B=1)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    theta = case["truth"][0].astype(np.float64)
    _, phi, _, _ = o.monomials(theta[: o.L])
    T = phi @ d["coeffs"].astype(np.float64)
    s = o.pixel_kms()[0]
    H, w, _, _ = o.kernel_weights(theta[o.L] / s, theta[o.L + 1] / s)
    S = o.eval_S(theta[None, :])[0]
    ref = np.convolve(T, w, mode="valid")  # no padding involved: pixels H .. P-1-H
    assert np.allclose(S[H: d["n_pix"] - H], ref, rtol=1e-12, atol=1e-13)
    # replicate-edge clamp on the rest (C.2-16)
    Tpad = np.concatenate([np.full(H, T[0]), T, np.full(H, T[-1])])
    assert np.allclose(S, np.convolve(Tpad, w, mode="valid"), rtol=1e-12, atol=1e-13)
    # fitted pixels never read padding: n_edge >= H for anything in the prior box
    assert d["seg_n_edge"][0] >= H


def test_integer_shift_and_constant_template(oracle_mod):
    d, j = _line_model(oracle_mod, a_pix=3.0)
    o = oracle_mod.Oracle(d)
    s = o.pixel_kms()[0]
    T = d["coeffs"][0].astype(np.float64)
    # sigma -> small and integer mu: a pure integer shift (box lower bound is 20 km/s = 0.29 px:
    # neighbours carry exp(-1/(2*0.29^2)) = 2.6e-3, so allow that much smearing)
    S = o.eval_S(np.array([[5000.0, 3.0, -1.0, 2 * s, 1e-3 * s]]))[0]
    assert np.allclose(S[5:-5], T[3:-7], atol=1e-12)
    # a constant template stays constant whatever the kernel
    d["coeffs"][:] = 0.7
    S = oracle_mod.Oracle(d).eval_S(np.array([[5000.0, 3.0, -1.0, -133.0, 77.0]]))[0]
    assert np.allclose(S, np.float64(np.float32(0.7)), rtol=1e-14)


def test_per_pixel_kernel_on_linear_grid(oracle_mod):
    # C.2-13/14: sigma_tot = sqrt(sigma*^2 + sigma_inst^2), mu_j = v/s_j, per pixel, per segment.
    case = make(two_arm_config(), oracle_mod, B=1)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    theta = case["truth"][0].astype(np.float64)
    _, phi, _, _ = o.monomials(theta[: o.L])
    T = phi @ d["coeffs"].astype(np.float64)
    s = o.pixel_kms()
    S = o.eval_S(theta[None, :])[0]
    seg = d["seg_offset"]
    for j in (5, 200, 379, 380, 550, 699):
        k = 0 if j < seg[1] else 1
        a, b = seg[k], seg[k + 1]
        mu = theta[o.L] / s[j]
        sg = math.hypot(theta[o.L + 1], float(d["seg_sigma_inst"][k])) / s[j]
        H = math.ceil(abs(mu) + 5 * sg)
        t = np.arange(-H, H + 1)
        w = np.exp(-0.5 * ((t - mu) / sg) ** 2); w /= w.sum()
        ref = sum(w[i] * T[min(max(j - t[i], a), b - 1)] for i in range(t.size))  # never crosses a segment
        assert abs(S[j] - ref) < 1e-13


# ---------------------------------------------------------------- Legendre continuum (Eq. 6)

def test_legendre_matches_numpy(oracle_mod):
    g = golden()
    P = 1327
    x = -1.0 + 2.0 * np.arange(P) / P  # P:127, 0-based
    assert x[0] == g["legendre_node_first"] and abs(x[-1] - g["legendre_node_last_p1327"]) < 1e-15
    V = npleg.legvander(x, 50)
    assert V.shape[1] == g["legendre_table_columns"]
    for j in (0, 1, 500, 1326):
        assert np.allclose(oracle_mod.Oracle.legendre(float(x[j]), 50), V[j], rtol=1e-12, atol=1e-13)
    assert np.allclose(oracle_mod.Oracle.legendre(-1.0, 50), (-1.0) ** np.arange(51))


def test_wls_matches_lstsq_and_normal_equations(oracle_mod):
    case = make(two_arm_config(), oracle_mod, B=2)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    S = o.eval_S(case["truth"])
    n = o.D + 1
    for i in range(2):
        y = case["flux"][i].astype(np.float64)
        w = case["ivar"][i].astype(np.float64) * case["mask"][i]
        for k in range(o.n_seg):  # apply the edge exclusion by hand
            a, b = d["seg_offset"][k], d["seg_offset"][k + 1]
            w[a: a + d["seg_n_edge"][k]] = 0.0
            w[b - d["seg_n_edge"][k]: b] = 0.0
        bb, c, st = o.solve_continuum(S[i], y, w)
        assert st == 0
        for k in range(o.n_seg):
            a, b = d["seg_offset"][k], d["seg_offset"][k + 1]
            x = -1.0 + 2.0 * np.arange(b - a) / (b - a)
            Phi = S[i, a:b, None] * npleg.legvander(x, o.D)
            sw = np.sqrt(w[a:b])
            ref = np.linalg.lstsq(Phi * sw[:, None], y[a:b] * sw, rcond=None)[0]
            assert np.allclose(bb[k * n:(k + 1) * n], ref, rtol=1e-8, atol=1e-10)
            assert np.allclose(c[a:b], npleg.legval(x, bb[k * n:(k + 1) * n]), rtol=1e-12)  # C.2-8
            r = y[a:b] - c[a:b] * S[i, a:b]
            nrm = np.abs(Phi.T @ (w[a:b] * y[a:b])).max()
            assert np.abs(Phi.T @ (w[a:b] * r)).max() < 1e-9 * nrm  # Phi^T W r = 0


def test_wls_recovers_true_continuum_noise_free(oracle_mod):
    case = make(two_arm_config(), oracle_mod, B=2, noise_free=True)
    o = oracle_mod.Oracle(case["desc"])
    chi2, grad, cont, st = o.eval_grad(case["flux"], case["ivar"], case["mask"], case["truth"])
    # flux went through float32, so "exact" means float32 rounding of the data
    assert np.allclose(cont, case["cont"], atol=2e-6)
    assert np.all(st == 0)


# ---------------------------------------------------------------- gradient / envelope

@pytest.mark.parametrize("which", ["log1seg", "lin2seg"])
def test_gradient_vs_fd_of_resolved_chi2(oracle_mod, which):
    """north_star check 1 + SURVEY C.2-5: the analytic partial gradient at fixed b equals the
    central difference of chi2(u) WITH the continuum re-solved (envelope theorem), every
    parameter, both segment paths."""
    case = make(small_config() if which == "log1seg" else two_arm_config(), oracle_mod, B=2)
    o = oracle_mod.Oracle(case["desc"])
    chi2, grad, cont, st = o.eval_grad(case["flux"], case["ivar"], case["mask"], case["init"])
    for i in range(2):
        u = o.norm_u(case["init"][i])
        assert np.isclose(o.chi2_u(case["flux"][i], case["ivar"][i], case["mask"][i], u), chi2[i], rtol=1e-13)
        for p in range(o.NP):
            h = 1e-6
            up, um = u.copy(), u.copy()
            up[p] += h; um[p] -= h
            fd = (o.chi2_u(case["flux"][i], case["ivar"][i], case["mask"][i], up)
                  - o.chi2_u(case["flux"][i], case["ivar"][i], case["mask"][i], um)) / (2 * h)
            assert abs(fd - grad[i, p]) <= 2e-6 * np.abs(grad[i]).max(), (which, i, p, fd, grad[i, p])


def test_masked_pixels_do_not_leak(oracle_mod):
    case = make(small_config(mask_frac=0.1), oracle_mod, B=1)
    o = oracle_mod.Oracle(case["desc"])
    f2 = case["flux"].copy()
    assert (f2[case["mask"] == 0] == 1e3).all()
    f2[case["mask"] == 0] = -77.0
    # also scribble on the excluded edge pixels
    ne = case["desc"]["seg_n_edge"][0]
    f2[:, :ne] = 5.0; f2[:, -ne:] = -5.0
    a = o.eval_grad(case["flux"], case["ivar"], case["mask"], case["init"])
    b = o.eval_grad(f2, case["ivar"], case["mask"], case["init"])
    assert a[0][0] == b[0][0] and np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2])


def test_noise_free_stationarity_and_recovery(oracle_mod):
    """north_star check 2: at the truth on noise-free self-generated data chi2 = 0 and grad = 0
    (to the float32 rounding of the stored flux); from config-0 style offsets the fit returns."""
    case = make(small_config(D=4, n_iter=400), oracle_mod, B=4, noise_free=True)
    o = oracle_mod.Oracle(case["desc"])
    chi2, grad, _, _ = o.eval_grad(case["flux"], case["ivar"], None, case["truth"])
    npx = case["desc"]["n_pix"]
    assert np.all(chi2 < npx * (2e-7) ** 2 * 4)
    chi0, g0, _, _ = o.eval_grad(case["flux"], case["ivar"], None, case["init"])
    assert np.all(np.abs(grad).max(axis=1) < 1e-5 * np.abs(g0).max(axis=1))
    r = o.fit(case["flux"], case["ivar"], None, case["init"], 600, lr=0.03, want_err=False, want_trace=True)
    rngs = (o.hi - o.lo)
    assert np.all(r["chi2"] < 1e-6 * chi0)
    assert np.all(np.abs(r["params"] - case["truth"]) < 1e-3 * rngs)
    assert np.all(r["status"] == 0)


# ---------------------------------------------------------------- Adam

def test_adam_hand_computed_steps(oracle_mod):
    """north_star check 3.  Step 1: m^ = g, v^ = g^2 => du = -lr g/(|g|+eps).
    Step 2 from the closed forms of the bias-corrected moments with two given gradients."""
    g = golden()
    b1, b2, eps, lr = g["adam_beta1"], g["adam_beta2"], g["adam_eps"], 0.01
    u0 = np.array([0.2, -0.5, 0.0])
    g1 = np.array([3.0, -1e-3, 0.0])
    g2 = np.array([-1.0, 2e-3, 5.0])
    u1, m1, v1 = oracle_mod.Oracle.adam_step(u0, np.zeros(3), np.zeros(3), g1, 1, lr)
    assert np.allclose(u1, u0 - lr * g1 / (np.abs(g1) + eps), rtol=1e-14, atol=1e-16)
    assert u1[2] == u0[2]
    u2, m2, v2 = oracle_mod.Oracle.adam_step(u1, m1, v1, g2, 2, lr)
    mh = ((1 - b1) * (b1 * g1 + g2)) / (1 - b1 ** 2)
    vh = ((1 - b2) * (b2 * g1 ** 2 + g2 ** 2)) / (1 - b2 ** 2)
    assert np.allclose(u2, u1 - lr * mh / (np.sqrt(vh) + eps), rtol=1e-13, atol=1e-16)
    # clip to [-1,1] (C.2-18)
    u3, _, _ = oracle_mod.Oracle.adam_step(np.array([0.995]), np.zeros(1), np.zeros(1), np.array([-4.0]), 1, lr)
    assert u3[0] == 1.0


def test_adam_matches_torch_optimizer(oracle_mod):
    torch = pytest.importorskip("torch")
    A = np.array([[3.0, 0.5], [0.5, 1.0]]); c = np.array([0.3, -0.2])
    u = np.array([0.5, -0.4]); m = np.zeros(2); v = np.zeros(2)
    tu = torch.tensor(u, dtype=torch.float64, requires_grad=True)
    opt = torch.optim.Adam([tu], lr=0.02)  # defaults: betas (0.9, 0.999), eps 1e-8
    tA, tc = torch.tensor(A), torch.tensor(c)
    for t in range(1, 41):
        opt.zero_grad()
        loss = 0.5 * (tu - tc) @ tA @ (tu - tc)
        loss.backward()
        opt.step()
        u, m, v = oracle_mod.Oracle.adam_step(u, m, v, A @ (u - c), t, 0.02)
        assert np.allclose(u, tu.detach().numpy(), rtol=1e-12, atol=1e-14)


# ---------------------------------------------------------------- error estimate

def _numpy_rho(o, d, y, w, u):
    """Independent numpy restatement of rho(u) with the continuum re-solved (lstsq)."""
    S = o.eval_S(o.denorm(u)[None, :])[0]
    rho = np.zeros_like(S)
    for k in range(o.n_seg):
        a, b = d["seg_offset"][k], d["seg_offset"][k + 1]
        x = -1.0 + 2.0 * np.arange(b - a) / (b - a)
        Phi = S[a:b, None] * npleg.legvander(x, o.D)
        sw = np.sqrt(w[a:b])
        bb = np.linalg.lstsq(Phi * sw[:, None], y[a:b] * sw, rcond=None)[0]
        rho[a:b] = sw * (y[a:b] - Phi @ bb)
    return rho


def test_error_estimate_formula(oracle_mod):
    """Sigma = rho^T rho/(N_good-NP) (J^T J)^-1 with J from central differences of the re-solved
    whitened residual, rebuilt here in numpy from eval_S + lstsq."""
    case = make(small_config(n_iter=300, snr=(60.0, 60.0)), oracle_mod, B=2)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    r = o.fit(case["flux"], case["ivar"], case["mask"], case["init"], 300, lr=0.03)
    ne = d["seg_n_edge"][0]
    for i in range(2):
        y = case["flux"][i].astype(np.float64)
        w = case["ivar"][i].astype(np.float64) * case["mask"][i]
        w[:ne] = 0; w[-ne:] = 0
        u = o.norm_u(r["params"][i])
        h = 1e-5
        J = np.empty((d["n_pix"], o.NP))
        for p in range(o.NP):
            up, um = u.copy(), u.copy()
            up[p] += h; um[p] -= h
            J[:, p] = (_numpy_rho(o, d, y, w, up) - _numpy_rho(o, d, y, w, um)) / (2 * h)
        rho = _numpy_rho(o, d, y, w, u)
        ngood = int((w > 0).sum())
        cov = (rho @ rho) / (ngood - o.NP) * np.linalg.inv(J.T @ J)
        ref = np.sqrt(np.diag(cov)) * (o.hi - o.lo) / 2
        assert np.allclose(r["err"][i], ref, rtol=1e-5)
        assert np.isclose(rho @ rho, r["chi2"][i], rtol=1e-9)


def test_error_estimate_reduces_to_ols_covariance(oracle_mod):
    """Textbook special case: for small perturbations the model is linear in (u, b); the
    variable-projected J^T J is the Schur complement of the full Gauss-Newton matrix, so the
    oracle's errors equal sqrt(diag) of the u-block of s^2 (Jf^T Jf)^-1 with Jf = [d/du, d/db]."""
    case = make(small_config(n_iter=300, snr=(400.0, 400.0), mask_frac=0.0), oracle_mod, B=1)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    r = o.fit(case["flux"], case["ivar"], None, case["init"], 400, lr=0.03)
    ne = d["seg_n_edge"][0]
    y = case["flux"][0].astype(np.float64)
    w = case["ivar"][0].astype(np.float64).copy(); w[:ne] = 0; w[-ne:] = 0
    sw = np.sqrt(w)
    u = o.norm_u(r["params"][0])
    x = -1.0 + 2.0 * np.arange(d["n_pix"]) / d["n_pix"]
    V = npleg.legvander(x, o.D)
    b = r["cont"][0]
    S0 = o.eval_S(o.denorm(u)[None, :])[0]
    cols = []
    for p in range(o.NP):
        h = 1e-6
        up, um = u.copy(), u.copy(); up[p] += h; um[p] -= h
        dS = (o.eval_S(o.denorm(up)[None, :])[0] - o.eval_S(o.denorm(um)[None, :])[0]) / (2 * h)
        cols.append(-sw * (V @ b) * dS)
    Jf = np.column_stack(cols + [-sw * S0 * V[:, n] for n in range(o.D + 1)])
    ngood = int((w > 0).sum())
    cov = r["chi2"][0] / (ngood - o.NP) * np.linalg.inv(Jf.T @ Jf)
    ref = np.sqrt(np.diag(cov))[: o.NP] * (o.hi - o.lo) / 2
    # equal up to the O(residual) Golub-Pereyra term, tiny at SNR 400
    assert np.allclose(r["err"][0], ref, rtol=2e-3)


@pytest.mark.slow
def test_errors_match_monte_carlo_scatter(oracle_mod):
    """The paper's own validation idea: reported errors ~ scatter over noise realisations."""
    cfgobj = small_config(n_iter=250, snr=(40.0, 40.0), mask_frac=0.0, D=3)
    case = make(cfgobj, oracle_mod, B=1, noise_free=True)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    rng = np.random.default_rng(5)
    R = 160
    model = case["model"][0]
    sig = np.median(model) / 40.0
    flux = (model[None, :] + sig * rng.standard_normal((R, model.size))).astype(np.float32)
    ivar = np.full_like(flux, 1.0 / sig ** 2)
    init = np.repeat(case["truth"], R, axis=0)
    r = o.fit(flux, ivar, None, init, 250, lr=0.03)
    scatter = r["params"].std(axis=0, ddof=1)
    ratio = np.median(r["err"], axis=0) / scatter
    assert np.all(np.abs(ratio - 1.0) < 0.2), ratio
    ne = d["seg_n_edge"][0]
    dof = model.size - 2 * ne - o.NP - o.nc
    assert abs(np.mean(r["chi2"]) / dof - 1.0) < 0.03  # C.3: chi2/(N_good-NP-n_c) ~ 1


# ---------------------------------------------------------------- status bits (8(b))

def test_status_bits(oracle_mod):
    case = make(small_config(n_iter=5), oracle_mod, B=3)
    d = case["desc"]; o = oracle_mod.Oracle(d)
    mask = case["mask"].copy(); flux = case["flux"].copy(); init = case["init"].copy()
    mask[0, :] = 0                      # nothing to fit: continuum system is not positive definite
    flux[1, :] = -np.abs(flux[1, :])    # negative flux -> negative multiplicative correction
    init[2, o.L] = 400.0                # RV on its bound, gradient pushes outward or not: force bound
    r = o.fit(flux, case["ivar"], mask, init, 0, want_err=False)
    assert r["status"][0] & 1 and r["chi2"][0] == 0.0 and np.all(r["cont"][0] == 0.0)
    assert r["status"][1] & 4 and not (r["status"][1] & 1)
    assert r["status"][2] & 8
    assert np.allclose(r["params"][0], init[0], rtol=1e-12)  # zero steps: params = init


# ------------------------------------------------------------------ stopping rules (readings R-2..R-5)

def test_stop_rule_change_over_window_closed_form(oracle_mod):
    """Criterion (2), |L_t - L_{t-50}| < tol: for L_t = a r^t + c the difference is a r^(t-50) (1 - r^50), so the first
    firing step is known in closed form."""
    a, r, c, W, tol = 3.0, 0.93, 0.7, 50, 1e-5
    t = np.arange(1, 600)
    L = a * r ** t + c
    tstar = W + int(math.floor(math.log(tol / (a * (1 - r ** W))) / math.log(r))) + 1
    assert a * r ** (tstar - W) * (1 - r ** W) < tol <= a * r ** (tstar - 1 - W) * (1 - r ** W)
    assert oracle_mod.stop_rule(L, W, tol) == (tstar, 2)
    assert oracle_mod.stop_rule(L[:tstar - 1], W, tol) == (0, 1)          # the sequence ends one step early: nothing fires
    assert oracle_mod.stop_rule(L[:W], W, 1e30) == (0, 1)                 # not testable before t = W + 1 ...
    assert oracle_mod.stop_rule(L[:W + 1], W, 1e30) == (W + 1, 2)         # ... and fires there however loose the tolerance
    assert oracle_mod.stop_rule(L, 7, tol)[1] == 2 and oracle_mod.stop_rule(L, 7, tol)[0] < tstar


def test_stop_rule_monotone_rise(oracle_mod):
    """Criterion (3): 50 CONSECUTIVE increases.  A loss that falls for s steps and then rises every step fires at
    s + 50; one dip resets the count; (2) is tested before (3) when both hold."""
    W, s = 50, 13
    fall = 10.0 - 0.5 * np.arange(1, s + 1)              # L_1..L_s strictly falling
    rise = fall[-1] + 0.3 * np.arange(1, 200)            # then strictly rising: first increase at t = s + 1
    L = np.concatenate([fall, rise])
    assert oracle_mod.stop_rule(L, W, 1e-9) == (s + W, 3)
    L2 = L.copy()
    L2[s + 30 - 1] = L2[s + 30 - 2] - 1e-3               # a dip at t = s + 30: the run of increases restarts there
    assert oracle_mod.stop_rule(L2, W, 1e-9) == (s + 30 + W, 3)
    flat = np.concatenate([fall, fall[-1] + 1e-9 * np.arange(1, 200)])   # rising, but by less than tol per 50 steps
    assert oracle_mod.stop_rule(flat, W, 1e-5) == (s + W, 2)   # both hold first at t = s + W: (2) is tested first
    assert oracle_mod.stop_rule(np.ones(120), W, 1e-5) == (W + 1, 2)      # a constant loss is "no change", not a rise


def test_fit_with_stopping_rules_is_the_fixed_step_fit_cut_at_the_stop(oracle_mod):
    """orc_fit_stop against the pinned pieces: with an infinite tolerance every spectrum stops at the first testable
    step (t = 51: 50 updates, status bit 16); with tol = 0 and no sustained rise it runs to max_iter; and wherever it
    stops, the result is exactly orc_fit's after that many steps (same trajectory, R-5)."""
    case = make(small_config(), oracle_mod, B=3)
    o = oracle_mod.Oracle(case["desc"])
    args = (case["flux"], case["ivar"], case["mask"], case["init"])
    r = o.fit_stop(*args, 200, lr=0.05, tol=1e30)
    assert np.array_equal(r["n_steps"], [50, 50, 50]) and np.all(r["status"] & 16) and not np.any(r["status"] & 32)
    ref = o.fit(*args, 50, lr=0.05)
    for k in ("params", "chi2", "cont", "err"):
        assert np.array_equal(r[k], ref[k]), k
    r = o.fit_stop(*args, 70, lr=0.05, tol=0.0)
    assert np.array_equal(r["n_steps"], [70, 70, 70]) and not np.any(r["status"] & 48)
    assert np.array_equal(r["params"], o.fit(*args, 70, lr=0.05)["params"])
    # the paper's settings (lr 0.1, tol 1e-5, window 50): stops well before 5000, and the stop step is the one the
    # rule gives on the loss trace L_t = sqrt(chi2_t / p) of the fixed-step fit (R-2)
    r = o.fit_stop(*args, 5000, lr=0.1)
    assert np.all(r["n_steps"] < 2000) and np.all(r["status"] & 48)
    tr = o.fit(*args, int(r["n_steps"].max()) + 1, lr=0.1, want_trace=True, want_err=False)["trace"]
    for i in range(3):
        L = np.sqrt(tr[i, :-1] / case["desc"]["n_pix"])
        t, rule = oracle_mod.stop_rule(L, 50, 1e-5)
        assert t == r["n_steps"][i] + 1 and bool(r["status"][i] & (16 if rule == 2 else 32))
        assert np.array_equal(r["params"][i], o.fit(*[a[i:i + 1] for a in args], int(r["n_steps"][i]), lr=0.1,
                                                    want_err=False)["params"][0])


# ------------------------------------------------------------------ Clean-strategy masking (readings R-7..R-12)

def _baseline(n):
    """+1 on even pixels, -1 on odd ones: mean 0, mean square 1."""
    return np.where(np.arange(n) % 2 == 0, 1.0, -1.0)


def _sigma(eps, use):
    """Population standard deviation about the mean, written out (R-8)."""
    e = eps[use]
    mean = e.sum() / e.size
    return math.sqrt(((e - mean) ** 2).sum() / e.size)


def test_clean_primary_mask_and_threshold_escalation(oracle_mod):
    """Pass B: |eps| - f G > k sigma with k = 3, relaxed to 4, 5, 7 while more than 3 % would be clipped."""
    n = 400
    one, flat, seg = np.ones(n), np.zeros(n), [0, n]
    r = _baseline(n); r[100] = 10.0
    # sigma^2 = 499/400 - (9/400)^2: 3 sigma = 3.35 -> only the spike goes, its neighbours (-1: other sign, below every threshold) stay
    assert abs(_sigma(r, one > 0) - math.sqrt(499 / 400 - (9 / 400) ** 2)) < 1e-12
    w, nc, k = oracle_mod.clean_update(r, flat, one, seg, 0.5)
    assert (nc, k) == (1, 3) and np.array_equal(np.flatnonzero(w == 0), [100])
    # 16 spikes of 4.2 (4 % of the pixels): all above 3 sigma = 3.85, none above 4 sigma = 5.14 -> k = 4 clips nothing
    r = _baseline(n); r[20:340:20] = 4.2
    s = _sigma(r, one > 0)
    assert 3 * s < 4.2 < 4 * s
    w, nc, k = oracle_mod.clean_update(r, flat, one, seg, 0.5)
    assert (nc, k) == (0, 4) and np.all(w == 1)
    # 12 spikes of 5 and 4 of 9: k = 3 would clip all 16 (4 %), k = 4 only the four of 9 (1 %)
    r = _baseline(n); r[20:340:20] = 5.0; r[[40, 120, 200, 280]] = 9.0
    s = _sigma(r, one > 0)
    assert 3 * s < 5.0 < 4 * s < 9.0
    w, nc, k = oracle_mod.clean_update(r, flat, one, seg, 0.5)
    assert (nc, k) == (4, 4) and np.array_equal(np.flatnonzero(w == 0), [40, 120, 200, 280])
    # masked pixels (w = 0) are neither counted nor clipped, whatever their residual; weights whiten the residual (R-7)
    r = _baseline(n); r[100] = 10.0; r[250] = 1e6
    w0 = one.copy(); w0[250] = 0.0
    w, nc, k = oracle_mod.clean_update(r, flat, w0, seg, 0.5)
    assert nc == 1 and np.array_equal(np.flatnonzero(w == 0), [100, 250])
    r = _baseline(n); r[100] = 2.5; w4 = one.copy(); w4[100] = 16.0          # eps_100 = 4 * 2.5 = 10
    w, nc, k = oracle_mod.clean_update(r, flat, w4, seg, 0.5)
    assert nc == 1 and w[100] == 0


def test_clean_flux_gradient_allowance(oracle_mod):
    """G_j = max(|M_j - M_(j-1)|, |M_j - M_(j+1)|) excuses a residual that a small wavelength shift explains: at a step of
    8 in the model a residual of 6 passes with f_shift = 0.5 (6 - 4 = 2 < 3 sigma) and is clipped with 0.2 (6 - 1.6 = 4.4)."""
    n = 400
    M = np.where(np.arange(n) >= 200, 8.0, 0.0)
    r = _baseline(n); r[200] = 6.0
    s = _sigma(r, np.ones(n) > 0)
    assert 6 - 0.5 * 8 < 3 * s < 6 - 0.2 * 8
    w, nc, _ = oracle_mod.clean_update(r, M, np.ones(n), [0, n], 0.5)
    assert nc == 0
    w, nc, _ = oracle_mod.clean_update(r, M, np.ones(n), [0, n], 0.2)
    assert nc == 1 and w[200] == 0
    # only the neighbour that exists counts at a segment end: the step between pixels 199 | 200 is invisible when they
    # belong to different segments
    w, nc, _ = oracle_mod.clean_update(r, M, np.ones(n), [0, 200, n], 0.5)
    assert nc == 1 and w[200] == 0


def test_clean_adjacent_and_neighbourhood_masks(oracle_mod):
    """Pass C (2 sigma next to a primary outlier) and pass D (same sign, not larger, above sigma', repeated
    synchronously at most 20 times)."""
    n = 1000
    one, flat = np.ones(n), np.zeros(n)
    # C: 2.9 lies between 2 sigma and 3 sigma; next to the spike it is clipped, on its own (pixel 300) it is not;
    # across a segment boundary it is not a neighbour
    r = _baseline(n); r[100] = 10.0; r[101] = 2.9; r[300] = 2.9
    s = _sigma(r, one > 0)
    assert 2 * s < 2.9 < 3 * s
    w, nc, _ = oracle_mod.clean_update(r, flat, one, [0, n], 0.5)
    assert np.array_equal(np.flatnonzero(w == 0), [100, 101])
    w, nc, _ = oracle_mod.clean_update(r, flat, one, [0, 101, n], 0.5)
    assert np.array_equal(np.flatnonzero(w == 0), [100])
    # D: a ramp 1.98, 1.96, ... 1.40 behind a spike of 12: below 2 sigma (not C), above sigma', same sign, never larger than
    # the pixel before it -> one more pixel joins per iteration, and the 20-iteration cap leaves 521..530 in
    r = _baseline(n); r[500] = 12.0; r[501:531] = 2.0 - 0.02 * np.arange(1, 31)
    s = _sigma(r, one > 0)
    use = one > 0; use[500] = False
    s2 = _sigma(r, use)
    assert r[501] < 2 * s and r[530] > 1.05 * s2 and 1.0 < s2      # the +1 baseline pixels stay below sigma'
    w, nc, _ = oracle_mod.clean_update(r, flat, one, [0, n], 0.5)
    assert np.array_equal(np.flatnonzero(w == 0), np.arange(500, 521)) and nc == 21
    # the ramp is eaten only while it does not rise and keeps its sign
    r = _baseline(n); r[300] = 12.0; r[301] = 1.8; r[302] = 1.9; r[700] = 12.0; r[701] = 1.8; r[702] = -1.7
    w, nc, _ = oracle_mod.clean_update(r, flat, one, [0, n], 0.5)
    assert np.array_equal(np.flatnonzero(w == 0), [300, 301, 700, 701])
    # ... and on the other side of the spike too (descending towards lower pixels)
    r = _baseline(n); r[400] = 12.0; r[399] = 1.8; r[398] = 1.7; r[397] = 1.6
    w, nc, _ = oracle_mod.clean_update(r, flat, one, [0, n], 0.5)
    assert np.array_equal(np.flatnonzero(w == 0), [397, 398, 399, 400])


def test_fit_with_clean_strategy(oracle_mod):
    """orc_fit_clean against the pinned pieces: without updates it is orc_fit; its first update is orc_clean_update applied
    to the residuals of the pinned fit at that step with f_shift = 0.5; and on spectra hit by cosmic-ray-like spikes it
    clips those pixels and lands closer to the truth than the fit without Clean."""
    case = make(small_config(mask_frac=0.0, snr=(60.0, 60.0)), oracle_mod, B=4)
    o = oracle_mod.Oracle(case["desc"])
    flux = case["flux"].copy()
    P = case["desc"]["n_pix"]
    hit = np.array([150, 151, 152, 300, 420])
    flux[:, hit] += 1.5                                   # ~90 sigma at SNR 60
    args = (flux, case["ivar"], case["mask"], case["init"])
    plain = o.fit(*args, 60, lr=0.03)
    same = o.fit_clean(*args, 60, lr=0.03, every=0)
    for k in ("params", "chi2", "cont", "err"):
        assert np.array_equal(plain[k], same[k]), k
    assert np.array_equal(same["mask"], (case["ivar"] * case["mask"] != 0) & _not_edge(case))
    # first update after step 30
    at30 = o.fit(*args, 30, lr=0.03, want_err=False)
    M = o.eval_model(at30["params"], at30["cont"])
    one = o.fit_clean(*args, 30, lr=0.03, every=30, max_updates=1, want_err=False)
    for i in range(4):
        w0 = (case["ivar"][i].astype(np.float64) * case["mask"][i]) * _not_edge(case)[i]
        w1, nc, _ = oracle_mod.clean_update(flux[i].astype(np.float64) - M[i], M[i], w0, case["desc"]["seg_offset"], 0.5)
        assert np.array_equal(one["mask"][i], w1 != 0) and one["n_clipped"][i] == nc
        assert np.all(one["mask"][i][hit] == 0)
    assert np.array_equal(one["params"], at30["params"])
    # the paper's schedule (every 30 steps, up to 11 updates) over 400 steps
    clean = o.fit_clean(*args, 400, lr=0.03)
    dirty = o.fit(*args, 400, lr=0.03)
    rng = (o.hi - o.lo)
    e_clean = (np.abs(clean["params"] - case["truth"]) / rng).max()
    e_dirty = (np.abs(dirty["params"] - case["truth"]) / rng).max()
    assert np.all(clean["mask"][:, hit] == 0) and e_clean < 0.5 * e_dirty
    assert np.all(clean["n_clipped"] >= hit.size) and np.all(clean["n_clipped"] < 0.05 * P)


def test_fit_with_clean_strategy_and_stopping_rules(oracle_mod):
    """orc_fit_clean with window > 0 against the pinned pieces: without mask updates it is orc_fit_stop; with an infinite
    tolerance every spectrum stops at the first testable step (t = window + 1, `window` updates applied) and the result
    is the fixed-step Clean fit of `window` steps, the mask update after step 30 included; with tolerance 0 nothing
    fires and it is the fixed-step Clean fit; and a mask update postpones criterion (2): the clipped outliers make the
    loss drop, so the stop comes later than that of the same fit without Clean on clean data never would."""
    case = make(small_config(mask_frac=0.0, snr=(60.0, 60.0)), oracle_mod, B=3)
    o = oracle_mod.Oracle(case["desc"])
    flux = case["flux"].copy()
    flux[:, [150, 151, 300]] += 1.5
    args = (flux, case["ivar"], case["mask"], case["init"])
    a = o.fit_clean(*args, 120, lr=0.05, every=0, window=20, tol=1e-4)
    b = o.fit_stop(*args, 120, lr=0.05, window=20, tol=1e-4)
    for k in ("params", "chi2", "cont", "err", "status", "n_steps"):
        assert np.array_equal(a[k], b[k], equal_nan=True), k
    a = o.fit_clean(*args, 200, lr=0.05, every=30, window=40, tol=1e30)
    b = o.fit_clean(*args, 40, lr=0.05, every=30)
    assert np.array_equal(a["n_steps"], np.full(3, 40)) and np.all(a["status"] & 16)
    for k in ("params", "chi2", "cont", "err", "mask", "n_clipped"):
        assert np.array_equal(a[k], b[k], equal_nan=True), k
    assert np.all(a["n_clipped"] >= 3)
    a = o.fit_clean(*args, 70, lr=0.05, every=30, window=40, tol=0.0)
    b = o.fit_clean(*args, 70, lr=0.05, every=30)
    assert np.array_equal(a["n_steps"], np.full(3, 70)) and not np.any(a["status"] & 48)
    for k in ("params", "chi2", "cont", "err", "mask"):
        assert np.array_equal(a[k], b[k], equal_nan=True), k
    # a spectrum that has stopped gets no further mask update: stop at t = 21 (before the first update at step 30)
    a = o.fit_clean(*args, 200, lr=0.05, every=30, window=20, tol=1e30)
    assert np.array_equal(a["n_steps"], np.full(3, 20)) and np.all(a["n_clipped"] == 0)
    assert np.array_equal(a["mask"], (case["ivar"] * case["mask"] != 0) & _not_edge(case))


# ------------------------------------------------------------------------------------------------
# Levenberg-Marquardt on the NP x NP system (orc_fit_lm, reading R-13)
# ------------------------------------------------------------------------------------------------
def _lm_case(oracle_mod, **kw):
    case = make(small_config(snr=(60.0, 60.0), **kw), oracle_mod, B=3)
    d = case["desc"]
    o = oracle_mod.Oracle(d)
    ne = d["seg_n_edge"][0]
    ws = []
    for i in range(3):
        w = case["ivar"][i].astype(np.float64) * case["mask"][i]
        w[:ne] = 0; w[-ne:] = 0
        ws.append(w)
    return case, d, o, ws


def test_lm_first_step_is_marquardts_formula(oracle_mod):
    """One LM iteration rebuilt in numpy from the numpy residual of the error-estimate pins (eval_S + lstsq): J by central
    differences, delta = -(J^T J + lambda diag(J^T J))^-1 J^T rho, accepted because chi2 falls; a wrong sign, a missing
    diagonal scaling or an undamped step fails it.  lambda = 10 makes damping matter (a Gauss-Newton step differs)."""
    case, d, o, ws = _lm_case(oracle_mod)
    for lam in (1e-3, 10.0):
        r = o.fit_lm(case["flux"], case["ivar"], case["mask"], case["init"], 1, lambda0=lam, want_err=False, want_trace=True)
        for i in range(3):
            y = case["flux"][i].astype(np.float64)
            u = o.norm_u(case["init"][i])
            h = 1e-5
            J = np.empty((d["n_pix"], o.NP))
            for p in range(o.NP):
                up, um = u.copy(), u.copy()
                up[p] += h; um[p] -= h
                J[:, p] = (_numpy_rho(o, d, y, ws[i], up) - _numpy_rho(o, d, y, ws[i], um)) / (2 * h)
            rho = _numpy_rho(o, d, y, ws[i], u)
            A = J.T @ J
            delta = -np.linalg.solve(A + lam * np.diag(np.diag(A)), J.T @ rho)
            gn = -np.linalg.solve(A, J.T @ rho)
            un = np.clip(u + delta, -1, 1)
            rn = _numpy_rho(o, d, y, ws[i], un)
            assert rn @ rn < rho @ rho and r["n_steps"][i] == 1
            assert np.allclose(o.norm_u(r["params"][i]), un, atol=1e-9)
            assert np.isclose(r["trace"][i, 0], rho @ rho, rtol=1e-10) and np.isclose(r["trace"][i, 1], rn @ rn, rtol=1e-9)
            if lam == 10.0:
                assert np.abs(delta - gn).max() > 1e-3          # the damped step is not the Gauss-Newton step


def test_lm_converges_to_the_library_minimiser(oracle_mod):
    """The minimum orc_fit_lm reaches is the one scipy.optimize.least_squares(method="lm") (MINPACK) finds on the numpy
    residual, to 1e-6 of the prior range; chi2 never rises along the way; the analytic gradient of the oracle vanishes
    there; and the fixed-step Adam fit lands on the same point."""
    from scipy.optimize import least_squares
    case, d, o, ws = _lm_case(oracle_mod)
    r = o.fit_lm(case["flux"], case["ivar"], case["mask"], case["init"], 12, want_trace=True)
    assert np.all(np.diff(r["trace"], axis=1) <= 0) and np.all(r["n_steps"] >= 3) and np.all(r["n_steps"] <= 12)
    g0 = np.abs(o.eval_grad(case["flux"], case["ivar"], case["mask"], case["init"])[1]).max(axis=1)
    g1 = np.abs(o.eval_grad(case["flux"], case["ivar"], case["mask"], r["params"])[1]).max(axis=1)
    assert np.all(g1 < 1e-6 * g0)
    for i in range(3):
        y = case["flux"][i].astype(np.float64)
        sol = least_squares(lambda u: _numpy_rho(o, d, y, ws[i], u), o.norm_u(case["init"][i]), method="lm",
                            xtol=1e-14, ftol=1e-14, gtol=1e-14)
        assert np.abs(o.norm_u(r["params"][i]) - sol.x).max() < 2e-6, np.abs(o.norm_u(r["params"][i]) - sol.x)
        assert np.isclose(r["chi2"][i], 2 * sol.cost, rtol=1e-9)
    adam = o.fit(case["flux"], case["ivar"], case["mask"], case["init"], 1500, lr=0.02, want_err=False)
    assert (np.abs(adam["params"] - r["params"]) / (o.hi - o.lo)).max() < 1e-4
    # zero iterations: the evaluation at the initial guess
    z = o.fit_lm(case["flux"], case["ivar"], case["mask"], case["init"], 0, want_err=False)
    assert np.allclose(z["params"], case["init"]) and np.all(z["n_steps"] == 0)


def test_lm_noise_free_recovery_and_rejected_steps(oracle_mod):
    """On noise-free spectra LM returns the truth (chi2 -> 0) from the offset starts; and with a huge initial damping the
    first steps are tiny but accepted, while a start AT the minimum rejects everything (chi2 cannot fall): n_steps counts
    accepted steps only and the iterate never moves uphill."""
    case = make(small_config(mask_frac=0.0), oracle_mod, B=3, noise_free=True)
    o = oracle_mod.Oracle(case["desc"])
    r = o.fit_lm(case["flux"], case["ivar"], case["mask"], case["init"], 15, want_err=False)
    assert (np.abs(r["params"] - case["truth"]) / (o.hi - o.lo)).max() < 1e-6
    assert np.all(r["chi2"] < 1e-12 * o.fit_lm(case["flux"], case["ivar"], case["mask"], case["init"], 0, want_err=False)["chi2"])
    again = o.fit_lm(case["flux"], case["ivar"], case["mask"], r["params"], 4, want_err=False, want_trace=True)
    assert np.all(np.diff(again["trace"], axis=1) <= 0)
    assert (np.abs(again["params"] - r["params"]) / (o.hi - o.lo)).max() < 1e-7


def _not_edge(case):
    d = case["desc"]
    keep = np.ones((case["B"], d["n_pix"]), dtype=bool)
    for k in range(d["n_seg"]):
        a, b = d["seg_offset"][k], d["seg_offset"][k + 1]
        ne = d["seg_n_edge"][k]
        keep[:, a:a + ne] = False
        keep[:, b - ne:b] = False
    return keep


# ------------------------------------------------------------------------------------------------
# Flux-conserving resampler (step 3, Eq. 2-4): orc_obs_nodes, orc_resample
# ------------------------------------------------------------------------------------------------
ELODIE_LAM1, ELODIE_DLAM, ELODIE_Q = 3900.0, 0.2, 14501      # 3900-6800 A, 14,501 flux points


def test_resampler_nodes_are_the_papers(oracle_mod):
    """lambda''_i = exp(lambda_21 + (2i - 3) dlambda_2 / 2): on the LAMOST grid (log10 step 1e-4, 4200-5700 A, the
    1327 pixels of P:227) p + 1 nodes, each pixel centre the geometric mean of its two nodes, node ratio 10^1e-4."""
    ll = synth.loglam_grid("log10", 4200.0, 5700.0, 1e-4)
    assert ll.size == 1327
    n = oracle_mod.obs_nodes(ll)
    assert n.size == 1328
    assert np.allclose(np.sqrt(n[:-1] * n[1:]), 10.0 ** ll, rtol=1e-14)
    assert np.allclose(n[1:] / n[:-1], 10.0 ** 1e-4, rtol=1e-12)
    assert np.isclose(n[0], np.exp(np.log(4200.0) - 0.5 * 1e-4 * np.log(10.0)), rtol=1e-14)


def test_resampler_conserves_flux_and_reproduces_constants(oracle_mod):
    """Closed forms: a constant spectrum stays that constant; the integral over the observed bins equals the integral of
    the model over the same wavelength range (flux conservation, Carnall 2017); observed nodes equal to the model's nodes
    give the model back; merging aligned pairs of model pixels gives their means; and bins beyond the model's range
    receive only the flux inside it (R-14)."""
    rng = np.random.default_rng(3)
    T = 1.0 + 0.3 * rng.standard_normal(ELODIE_Q)
    nodes = oracle_mod.obs_nodes(synth.loglam_grid("log10", 4200.0, 5700.0, 1e-4))
    assert np.allclose(oracle_mod.resample(np.full(ELODIE_Q, 2.5), ELODIE_LAM1, ELODIE_DLAM, nodes), 2.5, rtol=1e-12)
    out = oracle_mod.resample(T, ELODIE_LAM1, ELODIE_DLAM, nodes)
    # brute force: the piecewise-constant model integrated over [nodes[0], nodes[-1]]
    edges = ELODIE_LAM1 + (np.arange(ELODIE_Q + 1) - 0.5) * ELODIE_DLAM
    ov = np.clip(np.minimum(edges[1:], nodes[-1]) - np.maximum(edges[:-1], nodes[0]), 0.0, None)
    assert np.isclose((out * np.diff(nodes)).sum(), (T * ov).sum(), rtol=1e-12)
    # every bin, brute force by overlaps
    for i in (0, 1, 500, 1326):
        o = np.clip(np.minimum(edges[1:], nodes[i + 1]) - np.maximum(edges[:-1], nodes[i]), 0.0, None)
        assert np.isclose(out[i], (T * o).sum() / (nodes[i + 1] - nodes[i]), rtol=1e-11)
    assert np.allclose(oracle_mod.resample(T, ELODIE_LAM1, ELODIE_DLAM, edges), T, rtol=1e-11)
    assert np.allclose(oracle_mod.resample(T[:1000], ELODIE_LAM1, ELODIE_DLAM, edges[:1001:2]),
                       0.5 * (T[0:1000:2] + T[1:1000:2]), rtol=1e-11)
    beyond = np.array([edges[0] - 1.0, edges[0] + 0.1, edges[0] + 0.3])
    got = oracle_mod.resample(T, ELODIE_LAM1, ELODIE_DLAM, beyond)
    assert np.isclose(got[0], T[0] * 0.1 / 1.1, rtol=1e-12) and np.isclose(got[1], (0.1 * T[0] + 0.1 * T[1]) / 0.2, rtol=1e-11)


def test_resampler_is_numpy_cumsum_interp_and_linear(oracle_mod):
    """The library-routine form of Eq. 2-4 (numpy cumsum + interp + diff), and Delta-4: resampling is linear, so
    resample(phi . C) = phi . resample(C) -- what lets the coefficient table be resampled once."""
    rng = np.random.default_rng(4)
    C_ = rng.standard_normal((5, ELODIE_Q))
    ll = synth.loglam_grid("log10", 4200.0, 5700.0, 1e-4)
    nodes = oracle_mod.obs_nodes(ll)
    edges = ELODIE_LAM1 + (np.arange(ELODIE_Q + 1) - 0.5) * ELODIE_DLAM
    for k in range(2):
        cum = np.concatenate([[0.0], np.cumsum(C_[k] * ELODIE_DLAM)])
        ref = np.diff(np.interp(nodes, edges, cum)) / np.diff(nodes)
        assert np.allclose(oracle_mod.resample(C_[k], ELODIE_LAM1, ELODIE_DLAM, nodes), ref, rtol=1e-9, atol=1e-12)
    phi = rng.standard_normal(5)
    R = oracle_mod.resample_coeffs(C_, ELODIE_LAM1, ELODIE_DLAM, [0, ll.size], ll)
    assert np.allclose(oracle_mod.resample(phi @ C_, ELODIE_LAM1, ELODIE_DLAM, nodes), phi @ R, rtol=1e-9, atol=1e-12)
    # two segments are resampled independently, each with its own end nodes
    R2 = oracle_mod.resample_coeffs(C_, ELODIE_LAM1, ELODIE_DLAM, [0, 700, ll.size], ll)
    assert np.allclose(R2[:, :699], R[:, :699], rtol=1e-12) and np.allclose(R2[:, 701:], R[:, 701:], rtol=1e-12)
    assert np.allclose(R2[:, 699:701], R[:, 699:701], rtol=1e-9)          # uniform log grid: the same nodes either way


# ------------------------------------------------------------------------------------------------
# Piecewise emulator: three polynomial models over five Teff regimes (Eq. 1; NEXT-3, reading R-15)
# ------------------------------------------------------------------------------------------------
def _single_model_desc(desc, r):
    """The description of model r alone (n_models = 0: the single-polynomial path pinned above)."""
    sel = np.asarray(desc["term_model"]) == r
    d = {k: v for k, v in desc.items() if k not in ("n_models", "term_model", "model_blend")}
    d["n_terms"] = int(sel.sum())
    d["term_exps"] = np.asarray(desc["term_exps"])[sel]
    d["coeffs"] = np.asarray(desc["coeffs"])[sel]
    return d


def test_piecewise_emulator_regimes_and_blend(oracle_mod):
    """P:72-76 / P:187 on the three-model config: in the pure regimes (<= 4000 K, 4550-7000 K, > 9000 K) the spectrum is the
    one model's own polynomial (the single-polynomial path, built here from that model's terms alone); in the overlaps
    it is omega_a f_a + omega_b f_b with the weights linear in log10 Teff, retyped here; weights sum to one everywhere and
    the spectrum is continuous across the four regime borders."""
    case = synth.make_case("E", oracle_mod.forward, B=1)
    d = case["desc"]
    o = oracle_mod.Oracle(d)
    singles = [oracle_mod.Oracle(_single_model_desc(d, r)) for r in range(3)]
    assert [s.K for s in singles] == [25, 26, 19]                       # 25, 26, 19 non-zero coefficients
    base = np.array([5000.0, 3.1, -0.7, 35.0, 80.0])

    def S(orc, teff):
        p = base.copy(); p[0] = teff
        return orc.eval_S(p[None, :])[0]

    for teff, r in ((3300.0, 0), (4000.0, 0), (4550.0, 1), (6000.0, 1), (7000.0, 1), (9000.0, 2), (11500.0, 2)):
        assert np.allclose(S(o, teff), S(singles[r], teff), rtol=1e-12, atol=1e-14), teff
    for teff, (a, b), (t0, t1) in ((4200.0, (0, 1), (4000.0, 4550.0)), (4500.0, (0, 1), (4000.0, 4550.0)),
                                   (7300.0, (1, 2), (7000.0, 9000.0)), (8800.0, (1, 2), (7000.0, 9000.0))):
        wb = (np.log10(teff) - np.log10(t0)) / (np.log10(t1) - np.log10(t0))
        ref = (1.0 - wb) * S(singles[a], teff) + wb * S(singles[b], teff)
        assert np.allclose(S(o, teff), ref, rtol=1e-12, atol=1e-14), teff
        assert not np.allclose(S(o, teff), S(singles[a], teff), rtol=1e-4)        # the blend is not one model
    for teff in np.linspace(3100.0, 12000.0, 90):
        w = [o.blend_weight(r, teff)[0] for r in range(3)]
        assert abs(sum(w) - 1.0) < 1e-14 and min(w) >= 0.0
    for border in (4000.0, 4550.0, 7000.0, 9000.0):
        assert np.abs(S(o, border * (1 + 1e-9)) - S(o, border * (1 - 1e-9))).max() < 1e-6


def test_piecewise_emulator_gradient_vs_fd(oracle_mod):
    """The analytic gradient with the d omega / d Teff term against central differences of the re-solved chi2, inside both
    overlaps and in a pure regime (a dropped or mis-signed weight derivative fails the Teff component)."""
    case = synth.make_case("E", oracle_mod.forward, B=3)
    o = oracle_mod.Oracle(case["desc"])
    init = case["init"].astype(np.float64).copy()
    init[:, 0] = (4300.0, 8000.0, 5600.0)
    chi2, grad, cont, st = o.eval_grad(case["flux"], case["ivar"], case["mask"], init)
    for i in range(3):
        u = o.norm_u(init[i])
        for p in range(o.NP):
            h = 1e-6
            up, um = u.copy(), u.copy()
            up[p] += h; um[p] -= h
            fd = (o.chi2_u(case["flux"][i], case["ivar"][i], case["mask"][i], up)
                  - o.chi2_u(case["flux"][i], case["ivar"][i], case["mask"][i], um)) / (2 * h)
            assert abs(fd - grad[i, p]) <= 2e-6 * np.abs(grad[i]).max(), (i, p, fd, grad[i, p])
    # the weight derivative matters: without it the Teff component would be off by more than the tolerance
    w, dw = o.blend_weight(0, 4300.0)
    assert dw < 0 and abs(dw * 4300.0 * np.log(10.0) * (np.log10(4550.0) - np.log10(4000.0)) + 1.0) < 1e-12
