/*
 * lasp_oracle.c -- plain, slow, fp64 CPU oracle for the LASP-Adam-GPU hot path.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
 * It shares no code, header, table or constant generator with the CUDA path under
 * paper_2512_24840_b200/csrc/.
 *
 * Every function follows /root/reference/PAPER.md ("P:n" = line n) in the reading
 * fixed by SURVEY.md section 8(c) ("C.1" = the definition block, "C.2-n" = row n of the
 * table of readings).  Nothing is blocked, fused or reordered beyond what the
 * definition states: one spectrum at a time, one pixel at a time, one tap at a time.
 *
 *   emulator            Eq. 1   P:67-76, P:187     orc_monomials, emulator_row
 *   shift + broadening  Eq. 5   P:111-119          orc_kernel_weights, stencil
 *   Legendre continuum  Eq. 6   P:121-129          orc_legendre, orc_solve_continuum
 *   residual            Eq. 7   P:133              chi2 / rho
 *   objective           Eq. 9   P:163-167          sum_j w_j r_j^2 (C.2-2, C.2-3)
 *   Adam                step 8  P:169              orc_adam_step
 *   stopping rules      step 8  P:169-171          orc_stop_rule, orc_fit_stop
 *   Clean masking       step 6  P:137-161, P:171   orc_clean_update, orc_fit_clean
 *   resampler           step 3  Eq. 2-4, P:78-109  orc_obs_nodes, orc_resample, orc_resample_coeffs
 *   piecewise emulator  Eq. 1   P:72-76, P:187     orc_blend_weight (R-15, parity unpinned), orc_monomials
 *   LM optimiser        NEXT-4  P:54-58, P:397     orc_fit_lm (Marquardt's method written out; R-13)
 *   error estimate      step 9  P:173              errors_one
 *
 * Parity pins (tests/test_oracle_*.py): numpy legvander/legval, numpy lstsq,
 * numpy convolve, central finite differences of chi2 (with re-solve), closed-form
 * first Adam step and torch.optim.Adam, textbook OLS covariance, Monte-Carlo
 * scatter, noise-free recovery, the 1327-pixel grid of P:227; closed-form stop steps;
 * constructed outlier patterns for the Clean passes; scipy least_squares (MINPACK) for the
 * LM minimiser; flux conservation and numpy cumsum + interp for the resampler.
 * PARITY UNPINNED (against the paper): orc_blend_weight -- the paper gives the regimes and
 * the three models but not the weights inside the overlaps; reading R-15 of
 * DESIGN.md is pinned to its own definition only.  No other function is unpinned.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o liblasp_oracle.so lasp_oracle.c -lm
 * (threads run over spectra only; each spectrum is computed serially.)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_C_KMS 299792.458 /* speed of light, km/s (C.1) */

typedef struct {
    int32_t n_pix, n_seg;
    const int32_t *seg_offset;    /* [n_seg+1] */
    const double *loglam;         /* [n_pix] log10(lambda/A) */
    const double *seg_sigma_inst; /* [n_seg] km/s */
    int32_t n_labels, n_terms;    /* L, K */
    const uint8_t *term_exps;     /* [K*L] */
    const double *coeffs;         /* [K*n_pix] row-major */
    const double *lo, *hi;        /* [NP], NP = L+2: labels..., rv, sigma */
    const uint8_t *label_log10;   /* [L] */
    const double *emu_a, *emu_b;  /* [L] */
    int32_t cont_degree;          /* D */
    const int32_t *seg_n_edge;    /* [n_seg] */
    /* piecewise emulator (Eq. 1's f_1..f_5; NEXT-3): n_models polynomial models share the term table,
     * term k belongs to model term_model[k]; model r has weight omega_r(theta_0) (orc_blend_weight).  n_models <= 1:
     * one polynomial (Delta-5), the two pointers are not read. */
    int32_t n_models;
    const uint8_t *term_model;    /* [K] */
    const double *model_blend;    /* [n_models*4]: lo0, lo1, hi0, hi1 in the units of label 0 */
} orc_model;

/* ------------------------------------------------------------------ grid */

/* C.1: s_j = c ln10 (loglam_{j+1}-loglam_{j-1})/2, one-sided at segment ends. */
static double pixel_kms(const orc_model *m, int seg, int j)
{
    int o = m->seg_offset[seg], e = m->seg_offset[seg + 1];
    double d;
    if (e - o < 2) return ORC_C_KMS * log(10.0) * 1e-4;
    if (j == o) d = m->loglam[j + 1] - m->loglam[j];
    else if (j == e - 1) d = m->loglam[j] - m->loglam[j - 1];
    else d = 0.5 * (m->loglam[j + 1] - m->loglam[j - 1]);
    return ORC_C_KMS * log(10.0) * d;
}

void orc_pixel_kms(const orc_model *m, double *s_out)
{
    for (int s = 0; s < m->n_seg; ++s)
        for (int j = m->seg_offset[s]; j < m->seg_offset[s + 1]; ++j) s_out[j] = pixel_kms(m, s, j);
}

/* P:127 (0-based, per segment, C.2-7): x_j = -1 + 2 (j-o_s)/P_s ; never reaches +1. */
static double node_x(const orc_model *m, int seg, int j)
{
    int o = m->seg_offset[seg], n = m->seg_offset[seg + 1] - o;
    return -1.0 + 2.0 * (double)(j - o) / (double)n;
}

/* --------------------------------------------------------------- Legendre */

/* P_0..P_D at x by Bonnet's recurrence (n+1)P_{n+1} = (2n+1) x P_n - n P_{n-1}. */
void orc_legendre(double x, int D, double *P)
{
    P[0] = 1.0;
    if (D >= 1) P[1] = x;
    for (int n = 1; n < D; ++n) P[n + 1] = ((2.0 * n + 1.0) * x * P[n] - n * P[n - 1]) / (n + 1.0);
}

/* --------------------------------------------------------------- emulator */

/* C.1: theta = lo + (u+1)(hi-lo)/2 */
static void denorm(const orc_model *m, const double *u, double *theta)
{
    int NP = m->n_labels + 2;
    for (int p = 0; p < NP; ++p) theta[p] = m->lo[p] + (u[p] + 1.0) * (m->hi[p] - m->lo[p]) * 0.5;
}

static void norm_u(const orc_model *m, const double *theta, double *u)
{
    int NP = m->n_labels + 2;
    for (int p = 0; p < NP; ++p) u[p] = 2.0 * (theta[p] - m->lo[p]) / (m->hi[p] - m->lo[p]) - 1.0;
}

/* Weight of model r of the piecewise emulator at label 0 = theta0 (Eq. 1: the five Teff regimes of P:72-76 are three
 * polynomial models, cold <= 4550 K, warm 4000-9000 K, hot >= 7000 K, that overlap in 4000-4550 K and 7000-9000 K).
 * The paper does not say how the two models of an overlap are combined.  Reading R-15 (PARITY UNPINNED against
 * the paper, pinned only to its own definition): a cross-fade linear in tau(theta0) (log10 Teff) --
 *   omega_r = up * down,  up = clamp((tau - tau(lo0)) / (tau(lo1) - tau(lo0)), 0, 1)  (1 when lo1 <= lo0),
 *                         down = clamp((tau(hi1) - tau) / (tau(hi1) - tau(hi0)), 0, 1)  (1 when hi1 <= hi0);
 * the derivative is the slope strictly inside a ramp and 0 elsewhere (the kinks at the regime borders are the gradient
 * discontinuities the paper blames for Adam's instability near log Teff = 3.95). */
void orc_blend_weight(const orc_model *m, int r, double theta0, double *w, double *dw_dtheta)
{
    const double *bl = m->model_blend + 4 * r;
    int lg = m->label_log10[0];
    double tau = lg ? log10(theta0) : theta0, dtau = lg ? 1.0 / (theta0 * log(10.0)) : 1.0;
    double up = 1.0, dup = 0.0, dn = 1.0, ddn = 0.0;
    if (bl[1] > bl[0]) {
        double a = lg ? log10(bl[0]) : bl[0], b = lg ? log10(bl[1]) : bl[1], t = (tau - a) / (b - a);
        if (t <= 0.0) up = 0.0; else if (t >= 1.0) up = 1.0; else { up = t; dup = dtau / (b - a); }
    }
    if (bl[3] > bl[2]) {
        double a = lg ? log10(bl[2]) : bl[2], b = lg ? log10(bl[3]) : bl[3], t = (b - tau) / (b - a);
        if (t <= 0.0) dn = 0.0; else if (t >= 1.0) dn = 1.0; else { dn = t; ddn = -dtau / (b - a); }
    }
    *w = up * dn;
    *dw_dtheta = dup * dn + up * ddn;
}

/* Eq. 1: x_l = a_l tau_l(theta_l) + b_l ; phi_k = omega_r(k) prod_l x_l^{e_kl} (omega = 1 in the single-polynomial
 * reading, Delta-5) ; dphi[l*K+k] = d phi_k / d x_l ; dx_dtheta[l] (C.1 last line). */
void orc_monomials(const orc_model *m, const double *theta, double *x, double *phi, double *dphi,
                   double *dx_dtheta)
{
    int L = m->n_labels, K = m->n_terms;
    for (int l = 0; l < L; ++l) {
        if (m->label_log10[l]) {
            x[l] = m->emu_a[l] * log10(theta[l]) + m->emu_b[l];
            dx_dtheta[l] = m->emu_a[l] / (theta[l] * log(10.0));
        } else {
            x[l] = m->emu_a[l] * theta[l] + m->emu_b[l];
            dx_dtheta[l] = m->emu_a[l];
        }
    }
    for (int k = 0; k < K; ++k) {
        double v = 1.0;
        for (int l = 0; l < L; ++l)
            for (int e = 0; e < m->term_exps[k * L + l]; ++e) v *= x[l];
        phi[k] = v;
        for (int l = 0; l < L; ++l) {
            int el = m->term_exps[k * L + l];
            double d = 0.0;
            if (el > 0) {
                d = (double)el;
                for (int l2 = 0; l2 < L; ++l2) {
                    int e2 = m->term_exps[k * L + l2] - (l2 == l ? 1 : 0);
                    for (int e = 0; e < e2; ++e) d *= x[l2];
                }
            }
            dphi[l * K + k] = d;
        }
    }
    if (m->n_models > 1) {
        for (int k = 0; k < K; ++k) {
            double w, dw;
            orc_blend_weight(m, m->term_model[k], theta[0], &w, &dw);
            for (int l = 0; l < L; ++l) dphi[l * K + k] *= w;
            dphi[0 * K + k] += dw / dx_dtheta[0] * phi[k];      /* d omega / d x_0, chain rule through theta_0 */
            phi[k] *= w;
        }
    }
}

/* T_j = sum_k c_k C[k,j]  (Eq. 1 with the term vector c = phi or dphi/dx_l) */
static void emulator_row(const orc_model *m, const double *c, double *T)
{
    int P = m->n_pix, K = m->n_terms;
    for (int j = 0; j < P; ++j) {
        double acc = 0.0;
        for (int k = 0; k < K; ++k) acc += c[k] * m->coeffs[(size_t)k * P + j];
        T[j] = acc;
    }
}

/* ---------------------------------------------------------- kernel weights */

/* Eq. 5 / P:115 with readings C.2-9, -10, -15: H = ceil(|mu| + 5 sigma); point-sampled
 * Gaussian at integer offsets k = -H..H centred at +mu, unit sum over the truncated
 * support; analytic d g/d mu and d g/d sigma with H held constant (C.1).
 * Arrays hold 2H+1 entries, entry i is offset k = i - H.  Returns H. */
int orc_kernel_weights(double mu, double sigma, int Hcap, double *g, double *dg_dmu, double *dg_dsig)
{
    if (!isfinite(mu) || !isfinite(sigma)) return -1; /* non-finite parameters: no kernel; the caller's S is NaN */
    int H = (int)ceil(fabs(mu) + 5.0 * sigma);
    if (H > Hcap) return -H; /* caller sized the buffers too small */
    double sum = 0.0;
    for (int k = -H; k <= H; ++k) {
        double e = exp(-(k - mu) * (k - mu) / (2.0 * sigma * sigma));
        g[k + H] = e;
        sum += e;
    }
    double kbar = 0.0, m2 = 0.0;
    for (int k = -H; k <= H; ++k) {
        g[k + H] /= sum;
        kbar += g[k + H] * k;
        m2 += g[k + H] * (k - mu) * (k - mu);
    }
    for (int k = -H; k <= H; ++k) {
        if (dg_dmu) dg_dmu[k + H] = g[k + H] * (k - kbar) / (sigma * sigma);
        if (dg_dsig) dg_dsig[k + H] = g[k + H] * ((k - mu) * (k - mu) - m2) / (sigma * sigma * sigma);
    }
    return H;
}

static int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

/* Largest support over the prior box, used only to size scratch buffers. */
static int support_cap(const orc_model *m)
{
    int L = m->n_labels;
    double vmax = fmax(fabs(m->lo[L]), fabs(m->hi[L])) * 1.5 + 1.0;
    double smax = fmax(fabs(m->lo[L + 1]), fabs(m->hi[L + 1])) * 1.5 + 1.0;
    int cap = 0;
    for (int s = 0; s < m->n_seg; ++s)
        for (int j = m->seg_offset[s]; j < m->seg_offset[s + 1]; ++j) {
            double sj = pixel_kms(m, s, j);
            double st = sqrt(smax * smax + m->seg_sigma_inst[s] * m->seg_sigma_inst[s]);
            int H = (int)ceil(vmax / sj + 5.0 * st / sj) + 2;
            if (H > cap) cap = H;
        }
    return cap;
}

/* ------------------------------------------------------------ forward model */

typedef struct {
    int P, K, L, NP, D, nc, Hcap;
    double *theta, *x, *phi, *dphi, *dxdt;
    double *T, *dT;       /* [P], [L*P] */
    double *S, *dS;       /* [P], [NP*P]  dS = d S / d u_p */
    double *g, *gm, *gs;  /* [2Hcap+1] */
    double *w, *c, *r;    /* [P] */
    double *Pl;           /* [D+1] */
    double *A, *rhs;      /* [(D+1)^2], [D+1] */
    double *b;            /* [nc] */
} work_t;

static work_t *work_new(const orc_model *m)
{
    work_t *k = (work_t *)calloc(1, sizeof(work_t));
    k->P = m->n_pix; k->K = m->n_terms; k->L = m->n_labels; k->NP = k->L + 2;
    k->D = m->cont_degree; k->nc = m->n_seg * (k->D + 1); k->Hcap = support_cap(m);
    int P = k->P, K = k->K, L = k->L, NP = k->NP, D = k->D;
    k->theta = calloc(NP, 8); k->x = calloc(L, 8); k->phi = calloc(K, 8);
    k->dphi = calloc((size_t)L * K, 8); k->dxdt = calloc(L, 8);
    k->T = calloc(P, 8); k->dT = calloc((size_t)L * P, 8);
    k->S = calloc(P, 8); k->dS = calloc((size_t)NP * P, 8);
    k->g = calloc(2 * k->Hcap + 1, 8); k->gm = calloc(2 * k->Hcap + 1, 8); k->gs = calloc(2 * k->Hcap + 1, 8);
    k->w = calloc(P, 8); k->c = calloc(P, 8); k->r = calloc(P, 8);
    k->Pl = calloc(D + 1, 8); k->A = calloc((size_t)(D + 1) * (D + 1), 8); k->rhs = calloc(D + 1, 8);
    k->b = calloc(k->nc, 8);
    return k;
}

static void work_free(work_t *k)
{
    free(k->theta); free(k->x); free(k->phi); free(k->dphi); free(k->dxdt); free(k->T); free(k->dT);
    free(k->S); free(k->dS); free(k->g); free(k->gm); free(k->gs); free(k->w); free(k->c); free(k->r);
    free(k->Pl); free(k->A); free(k->rhs); free(k->b); free(k);
}

/* model(u) of C.1: fills k->S; with want_grad also k->dS[p][j] = dS_j/du_p (forward mode,
 * one parameter at a time -- the plain derivative of the definition). */
static void model_S(const orc_model *m, work_t *k, const double *u, int want_grad)
{
    int P = k->P, K = k->K, L = k->L;
    denorm(m, u, k->theta);
    orc_monomials(m, k->theta, k->x, k->phi, k->dphi, k->dxdt);
    emulator_row(m, k->phi, k->T);
    if (want_grad)
        for (int l = 0; l < L; ++l) emulator_row(m, k->dphi + (size_t)l * K, k->dT + (size_t)l * P);
    double v = k->theta[L], sig = k->theta[L + 1];
    for (int s = 0; s < m->n_seg; ++s) {
        int o = m->seg_offset[s], e = m->seg_offset[s + 1];
        double si = m->seg_sigma_inst[s];
        double stot = sqrt(sig * sig + si * si); /* C.2-13 */
        for (int j = o; j < e; ++j) {
            double sj = pixel_kms(m, s, j);
            double mu = v / sj, sg = stot / sj; /* C.2-12, C.2-14 */
            int H = orc_kernel_weights(mu, sg, k->Hcap, k->g, want_grad ? k->gm : NULL,
                                       want_grad ? k->gs : NULL);
            if (H < 0) { k->S[j] = NAN; continue; }
            double acc = 0.0;
            for (int t = -H; t <= H; ++t) acc += k->g[t + H] * k->T[clampi(j - t, o, e - 1)]; /* C.2-11, -16 */
            k->S[j] = acc;
            if (want_grad) {
                double am = 0.0, as = 0.0;
                for (int t = -H; t <= H; ++t) {
                    double Tv = k->T[clampi(j - t, o, e - 1)];
                    am += k->gm[t + H] * Tv;
                    as += k->gs[t + H] * Tv;
                }
                for (int l = 0; l < L; ++l) {
                    double al = 0.0;
                    for (int t = -H; t <= H; ++t)
                        al += k->g[t + H] * k->dT[(size_t)l * P + clampi(j - t, o, e - 1)];
                    k->dS[(size_t)l * P + j] = al * k->dxdt[l] * (m->hi[l] - m->lo[l]) * 0.5;
                }
                k->dS[(size_t)L * P + j] = am / sj * (m->hi[L] - m->lo[L]) * 0.5;
                k->dS[(size_t)(L + 1) * P + j] =
                    as * (sig / (stot * sj)) * (m->hi[L + 1] - m->lo[L + 1]) * 0.5;
            }
        }
    }
}

/* a0: w_j = mask_j ivar_j, zero on the n_edge first/last pixels of each segment (Eq. 8 P:161,
 * edge exclusion P:167, C.2-2, -17). */
static void make_weights(const orc_model *m, const double *ivar, const uint8_t *mask, double *w)
{
    for (int s = 0; s < m->n_seg; ++s) {
        int o = m->seg_offset[s], e = m->seg_offset[s + 1], ne = m->seg_n_edge[s];
        for (int j = o; j < e; ++j) {
            double v = ivar[j] * ((mask == NULL || mask[j]) ? 1.0 : 0.0);
            if (j - o < ne || e - 1 - j < ne) v = 0.0;
            w[j] = v;
        }
    }
}

/* Cholesky A = G G^T in place (lower), returns 0 if SPD else 1.  n <= 64. */
static int cholesky(double *A, int n)
{
    for (int i = 0; i < n; ++i) {
        for (int j = 0; j <= i; ++j) {
            double s = A[i * n + j];
            for (int t = 0; t < j; ++t) s -= A[i * n + t] * A[j * n + t];
            if (i == j) {
                if (!(s > 0.0)) return 1;
                A[i * n + i] = sqrt(s);
            } else
                A[i * n + j] = s / A[j * n + j];
        }
    }
    return 0;
}

static void chol_solve(const double *G, int n, double *x)
{
    for (int i = 0; i < n; ++i) {
        double s = x[i];
        for (int t = 0; t < i; ++t) s -= G[i * n + t] * x[t];
        x[i] = s / G[i * n + i];
    }
    for (int i = n - 1; i >= 0; --i) {
        double s = x[i];
        for (int t = i + 1; t < n; ++t) s -= G[t * n + i] * x[t];
        x[i] = s / G[i * n + i];
    }
}

/* solve(S) of C.1 (Eq. 6; C.2-4, -6): per segment
 *   A = Phi^T diag(w) Phi, rhs = Phi^T diag(w) y, Phi_jn = S_j P_n(x_j); b = A^-1 rhs.
 * A segment whose A is not positive definite gets b = 0 and status bit 1.
 * Then c_j = sum_n b_n P_n(x_j).  Returns status bits. */
static int solve_continuum(const orc_model *m, work_t *k, const double *y)
{
    int D = k->D, n = D + 1, status = 0;
    for (int s = 0; s < m->n_seg; ++s) {
        int o = m->seg_offset[s], e = m->seg_offset[s + 1];
        memset(k->A, 0, sizeof(double) * n * n);
        memset(k->rhs, 0, sizeof(double) * n);
        for (int j = o; j < e; ++j) {
            if (k->w[j] == 0.0) continue;
            orc_legendre(node_x(m, s, j), D, k->Pl);
            for (int a = 0; a < n; ++a) {
                double fa = k->S[j] * k->Pl[a];
                k->rhs[a] += fa * k->w[j] * y[j];
                for (int b2 = 0; b2 < n; ++b2) k->A[a * n + b2] += fa * k->w[j] * k->S[j] * k->Pl[b2];
            }
        }
        double *bs = k->b + s * n;
        if (cholesky(k->A, n)) {
            status |= 1;
            for (int a = 0; a < n; ++a) bs[a] = 0.0;
        } else {
            for (int a = 0; a < n; ++a) bs[a] = k->rhs[a];
            chol_solve(k->A, n, bs);
        }
        for (int j = o; j < e; ++j) {
            orc_legendre(node_x(m, s, j), D, k->Pl);
            double c = 0.0;
            for (int a = 0; a < n; ++a) c += bs[a] * k->Pl[a];
            k->c[j] = c;
        }
    }
    return status;
}

/* chi2(u) of C.1: S = model(u); b = solve(S); r = y - c S; chi2 = sum w r^2.  k->w must be set. */
static double chi2_at(const orc_model *m, work_t *k, const double *u, const double *y, int want_grad,
                      int *status)
{
    model_S(m, k, u, want_grad);
    int st = solve_continuum(m, k, y);
    double chi2 = 0.0;
    for (int j = 0; j < k->P; ++j) {
        k->r[j] = y[j] - k->c[j] * k->S[j];
        if (k->w[j] != 0.0) chi2 += k->w[j] * k->r[j] * k->r[j];
    }
    if (status) *status |= st;
    return chi2;
}

/* grad(u) of C.1: d chi2/d u_p = sum_j (-2 w_j r_j c_j) dS_j/du_p with b held (C.2-5). */
static void grad_from_work(const work_t *k, double *grad)
{
    for (int p = 0; p < k->NP; ++p) {
        double acc = 0.0;
        for (int j = 0; j < k->P; ++j)
            if (k->w[j] != 0.0) acc += -2.0 * k->w[j] * k->r[j] * k->c[j] * k->dS[(size_t)p * k->P + j];
        grad[p] = acc;
    }
}

/* One Adam update (step 8; C.2-18, -20): t starts at 1, bias-corrected, eps outside
 * the sqrt of the bias-corrected second moment, then clip to [-1,1]. */
void orc_adam_step(int n, double *u, double *mom, double *vel, const double *g, int t, double lr,
                   double b1, double b2, double eps)
{
    for (int p = 0; p < n; ++p) {
        mom[p] = b1 * mom[p] + (1.0 - b1) * g[p];
        vel[p] = b2 * vel[p] + (1.0 - b2) * g[p] * g[p];
        double mh = mom[p] / (1.0 - pow(b1, (double)t));
        double vh = vel[p] / (1.0 - pow(b2, (double)t));
        double un = u[p] - lr * mh / (sqrt(vh) + eps);
        u[p] = un < -1.0 ? -1.0 : (un > 1.0 ? 1.0 : un);
    }
}

static int finite_all(const double *v, int n)
{
    for (int i = 0; i < n; ++i)
        if (!isfinite(v[i])) return 0;
    return 1;
}

/* Step 9 (C.2-22, -23): rho(u) = sqrt(w) (y - c S) with the continuum re-solved,
 * J by central differences of step h in u, Sigma = rho^T rho/(N_good-NP) (J^T J)^-1,
 * err_p = sqrt(Sigma_pp) (hi_p-lo_p)/2.  Non-invertible J^T J gives NaN errors. */
static void errors_one(const orc_model *m, work_t *k, const double *u, const double *y, double h,
                       double *err)
{
    int P = k->P, NP = k->NP;
    double *J = calloc((size_t)NP * P, 8), *up = calloc(NP, 8), *rp = calloc(P, 8);
    double *N = calloc((size_t)NP * NP, 8);
    for (int p = 0; p < NP; ++p) {
        memcpy(up, u, 8 * NP);
        up[p] = u[p] + h;
        chi2_at(m, k, up, y, 0, NULL);
        for (int j = 0; j < P; ++j) rp[j] = sqrt(k->w[j]) * k->r[j];
        up[p] = u[p] - h;
        chi2_at(m, k, up, y, 0, NULL);
        for (int j = 0; j < P; ++j) J[(size_t)p * P + j] = (rp[j] - sqrt(k->w[j]) * k->r[j]) / (2.0 * h);
    }
    double ss = chi2_at(m, k, u, y, 0, NULL);
    int ngood = 0;
    for (int j = 0; j < P; ++j) ngood += (k->w[j] > 0.0);
    for (int a = 0; a < NP; ++a)
        for (int b = 0; b < NP; ++b) {
            double acc = 0.0;
            for (int j = 0; j < P; ++j) acc += J[(size_t)a * P + j] * J[(size_t)b * P + j];
            N[a * NP + b] = acc;
        }
    double s2 = ss / (double)(ngood - NP);
    if (ngood <= NP || cholesky(N, NP)) {
        for (int p = 0; p < NP; ++p) err[p] = NAN;
    } else {
        /* diag of (J^T J)^-1: solve N z = e_p */
        for (int p = 0; p < NP; ++p) {
            memset(up, 0, 8 * NP);
            up[p] = 1.0;
            chol_solve(N, NP, up);
            err[p] = sqrt(s2 * up[p]) * (m->hi[p] - m->lo[p]) * 0.5;
        }
    }
    free(J); free(up); free(rp); free(N);
}

/* status bits of SURVEY 8(b): 1 not SPD, 2 non-finite, 4 continuum <= 0 on a fitted pixel
 * (the paper's failure criterion), 8 parameter on its bound. */
static int final_status(const work_t *k, const double *u, double chi2, int st)
{
    if (!isfinite(chi2) || !finite_all(u, k->NP) || !finite_all(k->b, k->nc)) st |= 2;
    for (int j = 0; j < k->P; ++j)
        if (k->w[j] > 0.0 && k->c[j] <= 0.0) { st |= 4; break; }
    for (int p = 0; p < k->NP; ++p)
        if (u[p] <= -1.0 || u[p] >= 1.0) st |= 8;
    return st;
}

/* ------------------------------------------------------------- public API */

/* lasp_eval_model: model_j = c_j S_j at given physical params and plain-Legendre cont. */
int orc_eval_model(const orc_model *m, int64_t B, const double *params, const double *cont,
                   double *model)
{
    int NP = m->n_labels + 2, P = m->n_pix, n = m->cont_degree + 1, nc = m->n_seg * n;
#pragma omp parallel
    {
        work_t *k = work_new(m);
        double *u = calloc(NP, 8);
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < B; ++i) {
            norm_u(m, params + i * NP, u);
            model_S(m, k, u, 0);
            for (int s = 0; s < m->n_seg; ++s)
                for (int j = m->seg_offset[s]; j < m->seg_offset[s + 1]; ++j) {
                    orc_legendre(node_x(m, s, j), m->cont_degree, k->Pl);
                    double c = 0.0;
                    for (int a = 0; a < n; ++a) c += cont[i * nc + s * n + a] * k->Pl[a];
                    model[i * P + j] = c * k->S[j];
                }
        }
        free(u);
        work_free(k);
    }
    return 0;
}

/* The bare broadened template S (no continuum), for pins. */
int orc_eval_S(const orc_model *m, int64_t B, const double *params, double *S)
{
    int NP = m->n_labels + 2, P = m->n_pix;
    work_t *k = work_new(m);
    double *u = calloc(NP, 8);
    for (int64_t i = 0; i < B; ++i) {
        norm_u(m, params + i * NP, u);
        model_S(m, k, u, 0);
        memcpy(S + i * P, k->S, 8 * (size_t)P);
    }
    free(u);
    work_free(k);
    return 0;
}

/* lasp_eval_grad: chi2, d chi2/d u, continuum coefficients, status bit 1 at given params. */
int orc_eval_grad(const orc_model *m, int64_t B, const double *flux, const double *ivar,
                  const uint8_t *mask, const double *params, double *chi2, double *grad_u,
                  double *cont, int32_t *status)
{
    int NP = m->n_labels + 2, P = m->n_pix, nc = m->n_seg * (m->cont_degree + 1);
#pragma omp parallel
    {
        work_t *k = work_new(m);
        double *u = calloc(NP, 8);
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < B; ++i) {
            int st = 0;
            make_weights(m, ivar + i * P, mask ? mask + i * P : NULL, k->w);
            norm_u(m, params + i * NP, u);
            chi2[i] = chi2_at(m, k, u, flux + i * P, 1, &st);
            grad_from_work(k, grad_u + i * NP);
            if (cont) memcpy(cont + i * nc, k->b, 8 * (size_t)nc);
            if (status) status[i] = st;
        }
        free(u);
        work_free(k);
    }
    return 0;
}

/* chi2 only (re-solving the continuum), at normalised u -- used by the finite-difference pins. */
int orc_chi2_u(const orc_model *m, const double *flux, const double *ivar, const uint8_t *mask,
               const double *u, double *chi2)
{
    work_t *k = work_new(m);
    make_weights(m, ivar, mask, k->w);
    *chi2 = chi2_at(m, k, u, flux, 0, NULL);
    work_free(k);
    return 0;
}

/* lasp_fit_batch (fit + outputs + errors of C.1).  trace may be NULL, else [B*(n_iter+1)]
 * receives chi2 at every iterate (trace[t] = chi2 at the u the t-th gradient was taken at,
 * trace[n_iter] = final). */
int orc_fit(const orc_model *m, int64_t B, const double *flux, const double *ivar,
            const uint8_t *mask, const double *init, int n_iter, double lr, double b1, double b2,
            double eps, double fd_h, double *params, double *cont, double *chi2, double *err,
            int32_t *status, double *trace)
{
    int NP = m->n_labels + 2, P = m->n_pix, nc = m->n_seg * (m->cont_degree + 1);
#pragma omp parallel
    {
        work_t *k = work_new(m);
        double *u = calloc(NP, 8), *mom = calloc(NP, 8), *vel = calloc(NP, 8), *g = calloc(NP, 8);
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < B; ++i) {
            const double *y = flux + i * P;
            make_weights(m, ivar + i * P, mask ? mask + i * P : NULL, k->w);
            norm_u(m, init + i * NP, u);
            memset(mom, 0, 8 * NP);
            memset(vel, 0, 8 * NP);
            for (int t = 1; t <= n_iter; ++t) {
                double c2 = chi2_at(m, k, u, y, 1, NULL);
                if (trace) trace[i * (n_iter + 1) + (t - 1)] = c2;
                grad_from_work(k, g);
                orc_adam_step(NP, u, mom, vel, g, t, lr, b1, b2, eps);
            }
            int st = 0;
            double c2 = chi2_at(m, k, u, y, 0, &st); /* one more evaluation at the final u (C.2-21) */
            if (trace) trace[i * (n_iter + 1) + n_iter] = c2;
            chi2[i] = c2;
            denorm(m, u, params + i * NP);
            if (cont) memcpy(cont + i * nc, k->b, 8 * (size_t)nc);
            st = final_status(k, u, c2, st);
            if (status) status[i] = st;
            if (err) errors_one(m, k, u, y, fd_h, err + i * NP);
        }
        free(u); free(mom); free(vel); free(g);
        work_free(k);
    }
    return 0;
}

/* ------------------------------------------------------- stopping rules (step 8)
 *
 * "The optimization is considered converged when any of the following three criteria is satisfied: (1) a maximum of
 * 5000 iterations is reached; (2) the change in loss over 50 consecutive steps is less than 1e-5; or (3) the loss
 * increases monotonically over 50 consecutive steps."  Readings (R-2..R-5):
 *   R-2  the loss of one spectrum is Eq. 9 restricted to it, L = sqrt(chi2 / p) with p = n_pix (Delta-2: the hot path
 *        minimises sum_i chi2_i, so every spectrum stops on its own loss; with ivar = 1 this is the paper's L for N = 1);
 *   R-3  criterion (2) is |L_t - L_{t-W}| < tol, W = 50, first testable at t = W + 1;
 *   R-4  criterion (3) is W consecutive increases L_t > L_{t-1} > ... > L_{t-W};
 *   R-5  L_t is the loss at the iterate the t-th gradient is taken at (t = 1, 2, ...); the rules are tested, (2)
 *        before (3), BEFORE update t is applied, and a spectrum that stops at t keeps that iterate: t - 1 updates.
 *        Criterion (1): after max_iter updates nothing more is applied.
 * orc_stop_rule scans a loss sequence L[0..n-1] (L[t-1] = L_t) and returns the first t at which (2) or (3) fires
 * (*rule = 2 or 3), or 0 with *rule = 1 when neither fires within the sequence. */
int orc_stop_rule(const double *L, int n, int window, double tol, int *rule)
{
    int rise = 0;
    for (int t = 1; t <= n; ++t) {
        if (t > 1 && L[t - 1] > L[t - 2]) ++rise; else rise = 0;
        if (t > window && fabs(L[t - 1] - L[t - 1 - window]) < tol) { *rule = 2; return t; }
        if (rise >= window) { *rule = 3; return t; }
    }
    *rule = 1;
    return 0;
}

/* lasp_fit_batch with the paper's stopping rules: as orc_fit, but every spectrum stops by R-2..R-5.
 * n_steps[i] = Adam updates applied; status gets bit 16 (stopped by criterion 2) or 32 (criterion 3). */
int orc_fit_stop(const orc_model *m, int64_t B, const double *flux, const double *ivar,
                 const uint8_t *mask, const double *init, int max_iter, double lr, double b1, double b2,
                 double eps, int window, double tol, double fd_h, double *params, double *cont,
                 double *chi2, double *err, int32_t *status, int32_t *n_steps)
{
    int NP = m->n_labels + 2, P = m->n_pix, nc = m->n_seg * (m->cont_degree + 1);
#pragma omp parallel
    {
        work_t *k = work_new(m);
        double *u = calloc(NP, 8), *mom = calloc(NP, 8), *vel = calloc(NP, 8), *g = calloc(NP, 8);
        double *hist = calloc((size_t)max_iter + 1, 8);
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < B; ++i) {
            const double *y = flux + i * P;
            make_weights(m, ivar + i * P, mask ? mask + i * P : NULL, k->w);
            norm_u(m, init + i * NP, u);
            memset(mom, 0, 8 * NP);
            memset(vel, 0, 8 * NP);
            int rule = 1, rise = 0, applied = 0;
            for (int t = 1; t <= max_iter; ++t) {
                double c2 = chi2_at(m, k, u, y, 1, NULL);
                double L = sqrt(c2 / (double)P);                     /* R-2 */
                hist[t] = L;
                if (t > 1 && L > hist[t - 1]) ++rise; else rise = 0;
                if (t > window && fabs(L - hist[t - window]) < tol) { rule = 2; break; }   /* R-3 */
                if (rise >= window) { rule = 3; break; }                                    /* R-4 */
                grad_from_work(k, g);
                orc_adam_step(NP, u, mom, vel, g, t, lr, b1, b2, eps);
                applied = t;
            }
            int st = 0;
            double c2 = chi2_at(m, k, u, y, 0, &st);
            chi2[i] = c2;
            denorm(m, u, params + i * NP);
            if (cont) memcpy(cont + i * nc, k->b, 8 * (size_t)nc);
            st = final_status(k, u, c2, st);
            if (rule == 2) st |= 16;
            if (rule == 3) st |= 32;
            if (status) status[i] = st;
            if (n_steps) n_steps[i] = applied;
            if (err) errors_one(m, k, u, y, fd_h, err + i * NP);
        }
        free(u); free(mom); free(vel); free(g); free(hist);
        work_free(k);
    }
    return 0;
}

/* ------------------------------------------------------- Clean-strategy masking (step 6, Eq. 8)
 *
 * One mask update of one spectrum, from the residuals at the current iterate.  Readings (R-7..R-12):
 *   R-7  eps_j = sqrt(w_j) r_j, r = y - c S (Eq. 7 in the weighted form of Delta-1; the paper's case is w = 1), and the
 *        flux-gradient allowance G_j = sqrt(w_j) max(|M_j - M_(j-1)|, |M_j - M_(j+1)|), M = c S (the corrected model of
 *        Eq. 7), with only the neighbour that exists at a segment end; the unmasked pixels U are those with w_j > 0;
 *   R-8  sigma_eps = population standard deviation (about the mean) of eps over U; sigma'_eps the same over U without the
 *        pixels clipped by B and C;
 *   R-9  masks accumulate: a pixel clipped by an update stays clipped (A <- A B C D);
 *   R-10 B: excess_j = |eps_j| - f_shift G_j > k sigma, k = 3; if more than 3 % of U is clipped, k = 4, then 5, then 7
 *        (the first k that clips at most 3 %, else 7);
 *   R-11 C: the neighbours j' = j +- 1 (same segment, in U, not in B) of every j in B with excess_j' > 2 sigma;
 *   R-12 D: starting from O = B + C, synchronously: every neighbour j' (same segment, in U, not in O) of a j in O with
 *        eps_j eps_j' > 0, |eps_j'| <= |eps_j| and excess_j' > sigma' joins O; repeated until nothing joins, at most 20 times.
 * w is updated in place (clipped pixels get 0); returns the number of pixels clipped by this update, *k_used the k of B. */
static double pop_std(const double *eps, const uint8_t *use, int P, int *n_out)
{
    double s = 0.0, s2 = 0.0;
    int n = 0;
    for (int j = 0; j < P; ++j)
        if (use[j]) { s += eps[j]; ++n; }
    if (n_out) *n_out = n;
    if (n == 0) return 0.0;
    double mean = s / n;
    for (int j = 0; j < P; ++j)
        if (use[j]) s2 += (eps[j] - mean) * (eps[j] - mean);
    return sqrt(s2 / n);
}

int orc_clean_update(int P, int n_seg, const int32_t *seg_offset, const double *r, const double *M, double *w,
                     double fshift, int *k_used)
{
    double *eps = calloc(P, 8), *exc = calloc(P, 8);
    uint8_t *U = calloc(P, 1), *O = calloc(P, 1), *use = calloc(P, 1), *add = calloc(P, 1);
    int *seg = calloc(P, sizeof(int));
    for (int s = 0; s < n_seg; ++s)
        for (int j = seg_offset[s]; j < seg_offset[s + 1]; ++j) seg[j] = s;
    for (int j = 0; j < P; ++j) {
        U[j] = w[j] > 0.0;
        double sw = U[j] ? sqrt(w[j]) : 0.0;
        int s = seg[j], o = seg_offset[s], e = seg_offset[s + 1];
        double g = 0.0;
        if (j - 1 >= o) g = fmax(g, fabs(M[j] - M[j - 1]));
        if (j + 1 < e) g = fmax(g, fabs(M[j] - M[j + 1]));
        eps[j] = sw * r[j];
        exc[j] = fabs(eps[j]) - fshift * sw * g;                    /* R-7 */
    }
    int nU = 0;
    double sigma = pop_std(eps, U, P, &nU);                          /* R-8 */
    static const double ks[4] = {3.0, 4.0, 5.0, 7.0};
    int kk = 3;
    for (int t = 0; t < 4; ++t) {                                    /* R-10 */
        int n = 0;
        for (int j = 0; j < P; ++j) n += U[j] && exc[j] > ks[t] * sigma;
        kk = (int)ks[t];
        if ((double)n <= 0.03 * (double)nU) break;
    }
    if (k_used) *k_used = kk;
    for (int j = 0; j < P; ++j) O[j] = U[j] && exc[j] > (double)kk * sigma;
    memcpy(add, O, P);
    for (int j = 0; j < P; ++j) {                                    /* R-11 */
        if (!O[j]) continue;
        int s = seg[j], o = seg_offset[s], e = seg_offset[s + 1];
        for (int d = -1; d <= 1; d += 2) {
            int q = j + d;
            if (q < o || q >= e || !U[q] || O[q]) continue;
            if (exc[q] > 2.0 * sigma) add[q] = 1;
        }
    }
    memcpy(O, add, P);
    for (int j = 0; j < P; ++j) use[j] = U[j] && !O[j];
    double sigma2 = pop_std(eps, use, P, NULL);
    for (int it = 0; it < 20; ++it) {                                /* R-12 */
        int changed = 0;
        memcpy(add, O, P);
        for (int j = 0; j < P; ++j) {
            if (!O[j]) continue;
            int s = seg[j], o = seg_offset[s], e = seg_offset[s + 1];
            for (int d = -1; d <= 1; d += 2) {
                int q = j + d;
                if (q < o || q >= e || !U[q] || O[q]) continue;
                if (eps[j] * eps[q] > 0.0 && fabs(eps[q]) <= fabs(eps[j]) && exc[q] > sigma2) { add[q] = 1; changed = 1; }
            }
        }
        memcpy(O, add, P);
        if (!changed) break;
    }
    int n = 0;
    for (int j = 0; j < P; ++j)
        if (O[j]) { w[j] = 0.0; ++n; }                               /* R-9 */
    free(eps); free(exc); free(U); free(O); free(use); free(add); free(seg);
    return n;
}

/* lasp_fit_batch with the Clean strategy: as orc_fit (window = 0: fixed n_iter steps) or as orc_fit_stop (window > 0:
 * the stopping rules of P:169-171, R-2..R-5, n_iter the maximum), and after update t, t = every, 2 every, ...
 * (at most max_updates times; the paper: every 30 steps, up to 11) the mask is updated from the residuals at
 * the new iterate, with f_shift = 0.5 for the first update and 0.2 afterwards.  A spectrum that has stopped
 * gets no further mask update (its optimisation is over, "during the optimization").  The loss of R-2 keeps its
 * denominator n_pix when pixels are clipped (Eq. 9 divides by p N, not by the number of unmasked pixels).
 * mask_out[i*P+j] = 1 where the pixel still takes part at the end; n_steps[i] = Adam updates applied. */
int orc_fit_clean(const orc_model *m, int64_t B, const double *flux, const double *ivar,
                  const uint8_t *mask, const double *init, int n_iter, double lr, double b1, double b2,
                  double eps_adam, int every, int max_updates, int window, double tol, double fd_h, double *params,
                  double *cont, double *chi2, double *err, int32_t *status, uint8_t *mask_out, int32_t *n_clipped,
                  int32_t *n_steps)
{
    int NP = m->n_labels + 2, P = m->n_pix, nc = m->n_seg * (m->cont_degree + 1);
#pragma omp parallel
    {
        work_t *k = work_new(m);
        double *u = calloc(NP, 8), *mom = calloc(NP, 8), *vel = calloc(NP, 8), *g = calloc(NP, 8);
        double *Mod = calloc(P, 8);
        double *hist = calloc((size_t)n_iter + 1, 8);
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < B; ++i) {
            const double *y = flux + i * P;
            make_weights(m, ivar + i * P, mask ? mask + i * P : NULL, k->w);
            norm_u(m, init + i * NP, u);
            memset(mom, 0, 8 * NP);
            memset(vel, 0, 8 * NP);
            int updates = 0, clipped = 0, rule = 1, rise = 0, applied = 0;
            for (int t = 1; t <= n_iter; ++t) {
                double c2t = chi2_at(m, k, u, y, 1, NULL);
                if (window > 0) {                                    /* as orc_fit_stop */
                    double L = sqrt(c2t / (double)P);
                    hist[t] = L;
                    if (t > 1 && L > hist[t - 1]) ++rise; else rise = 0;
                    if (t > window && fabs(L - hist[t - window]) < tol) { rule = 2; break; }
                    if (rise >= window) { rule = 3; break; }
                }
                grad_from_work(k, g);
                orc_adam_step(NP, u, mom, vel, g, t, lr, b1, b2, eps_adam);
                applied = t;
                if (every > 0 && t % every == 0 && updates < max_updates) {
                    chi2_at(m, k, u, y, 0, NULL);                    /* residuals at the new iterate */
                    for (int j = 0; j < P; ++j) Mod[j] = k->c[j] * k->S[j];
                    clipped += orc_clean_update(P, m->n_seg, m->seg_offset, k->r, Mod, k->w, updates == 0 ? 0.5 : 0.2, NULL);
                    ++updates;
                }
            }
            int st = 0;
            double c2 = chi2_at(m, k, u, y, 0, &st);
            chi2[i] = c2;
            denorm(m, u, params + i * NP);
            if (cont) memcpy(cont + i * nc, k->b, 8 * (size_t)nc);
            st = final_status(k, u, c2, st);
            if (rule == 2) st |= 16;
            if (rule == 3) st |= 32;
            if (status) status[i] = st;
            if (n_steps) n_steps[i] = applied;
            if (mask_out) for (int j = 0; j < P; ++j) mask_out[i * P + j] = k->w[j] != 0.0;
            if (n_clipped) n_clipped[i] = clipped;
            if (err) errors_one(m, k, u, y, fd_h, err + i * NP);
        }
        free(u); free(mom); free(vel); free(g); free(Mod); free(hist);
        work_free(k);
    }
    return 0;
}

/* ------------------------------------------------------- Levenberg-Marquardt on the NP x NP system
 *
 * The paper's LASP-CurveFit minimises the same chi2 with scipy.optimize.curve_fit, and its future work asks
 * for "curvature awareness" in LASP-Adam-GPU.  Neither passage states an algorithm; this is Marquardt's method
 * written out on the objective of steps 5-7 (reading R-13 of DESIGN.md):
 *   rho(u) = sqrt(w) (y - c(u) S(u)) with the continuum re-solved at every u (variable projection, as step 9);
 *   J by central differences of step h in u (as errors_one), A = J^T J, g = J^T rho;
 *   lambda = lambda0; chi2 = |rho(u)|^2; then n_iter times:
 *     solve (A + lambda diag(A)) delta = -g  (Cholesky; delta = 0 when it is not positive definite);
 *     u' = clip(u + delta, [-1, 1]); chi2' = |rho(u')|^2;
 *     chi2' < chi2: u = u', chi2 = chi2', lambda = max(lambda / 10, 1e-10), one more accepted step;
 *     otherwise (NaN included): u stays, lambda = min(10 lambda, 1e10).
 * Then the final evaluation, status and error estimate of orc_fit.  n_steps[i] = accepted steps. */
static void lm_residual(const orc_model *m, work_t *k, const double *u, const double *y, double *rho, double *c2)
{
    *c2 = chi2_at(m, k, u, y, 0, NULL);
    for (int j = 0; j < k->P; ++j) rho[j] = sqrt(k->w[j]) * k->r[j];
}

int orc_fit_lm(const orc_model *m, int64_t B, const double *flux, const double *ivar,
               const uint8_t *mask, const double *init, int n_iter, double lambda0, double fd_h,
               double *params, double *cont, double *chi2, double *err, int32_t *status, int32_t *n_steps,
               double *trace)
{
    int NP = m->n_labels + 2, P = m->n_pix, nc = m->n_seg * (m->cont_degree + 1);
#pragma omp parallel
    {
        work_t *k = work_new(m);
        double *u = calloc(NP, 8), *ut = calloc(NP, 8), *up = calloc(NP, 8), *g = calloc(NP, 8);
        double *J = calloc((size_t)NP * P, 8), *rho = calloc(P, 8), *rp = calloc(P, 8), *rm = calloc(P, 8);
        double *A = calloc((size_t)NP * NP, 8), *N = calloc((size_t)NP * NP, 8);
#pragma omp for schedule(dynamic, 1)
        for (int64_t i = 0; i < B; ++i) {
            const double *y = flux + i * P;
            make_weights(m, ivar + i * P, mask ? mask + i * P : NULL, k->w);
            norm_u(m, init + i * NP, u);
            double lam = lambda0, c2;
            int accepted = 0;
            lm_residual(m, k, u, y, rho, &c2);
            if (trace) trace[i * (n_iter + 1)] = c2;
            for (int t = 1; t <= n_iter; ++t) {
                for (int p = 0; p < NP; ++p) {
                    double cc;
                    memcpy(up, u, 8 * NP);
                    up[p] = u[p] + fd_h;
                    lm_residual(m, k, up, y, rp, &cc);
                    up[p] = u[p] - fd_h;
                    lm_residual(m, k, up, y, rm, &cc);
                    for (int j = 0; j < P; ++j) J[(size_t)p * P + j] = (rp[j] - rm[j]) / (2.0 * fd_h);
                }
                for (int a = 0; a < NP; ++a) {
                    double s = 0.0;
                    for (int j = 0; j < P; ++j) s += J[(size_t)a * P + j] * rho[j];
                    g[a] = s;
                    for (int b = 0; b < NP; ++b) {
                        double acc = 0.0;
                        for (int j = 0; j < P; ++j) acc += J[(size_t)a * P + j] * J[(size_t)b * P + j];
                        A[a * NP + b] = acc;
                    }
                }
                memcpy(N, A, 8 * (size_t)NP * NP);
                for (int a = 0; a < NP; ++a) N[a * NP + a] += lam * A[a * NP + a];
                memcpy(ut, u, 8 * NP);
                if (!cholesky(N, NP)) {
                    for (int a = 0; a < NP; ++a) up[a] = -g[a];
                    chol_solve(N, NP, up);
                    for (int a = 0; a < NP; ++a) {
                        double v = u[a] + up[a];
                        ut[a] = v < -1.0 ? -1.0 : (v > 1.0 ? 1.0 : v);
                    }
                }
                double c2t;
                lm_residual(m, k, ut, y, rp, &c2t);
                if (c2t < c2) {
                    memcpy(u, ut, 8 * NP);
                    memcpy(rho, rp, 8 * (size_t)P);
                    c2 = c2t;
                    lam = fmax(lam / 10.0, 1e-10);
                    ++accepted;
                } else
                    lam = fmin(lam * 10.0, 1e10);
                if (trace) trace[i * (n_iter + 1) + t] = c2;
            }
            int st = 0;
            double cf = chi2_at(m, k, u, y, 0, &st);
            chi2[i] = cf;
            denorm(m, u, params + i * NP);
            if (cont) memcpy(cont + i * nc, k->b, 8 * (size_t)nc);
            st = final_status(k, u, cf, st);
            if (status) status[i] = st;
            if (n_steps) n_steps[i] = accepted;
            if (err) errors_one(m, k, u, y, fd_h, err + i * NP);
        }
        free(u); free(ut); free(up); free(g); free(J); free(rho); free(rp); free(rm); free(A); free(N);
        work_free(k);
    }
    return 0;
}

/* ------------------------------------------------------- flux-conserving resampler (step 3, Eq. 2-4; NEXT-3)
 *
 * The model spectrum T_1..T_q lives on a linear grid lam1 + (m-1) dlam1; its integration nodes are lam1 + (m - 1/2) dlam1,
 * m = 0..q.  Eq. 2: the cumulative integral 0, T_1 dlam1, ..., sum T_i dlam1 on those nodes; Eq. 3: linear
 * interpolation of it onto the observed integration nodes; Eq. 4: T'_i = (F(node_(i+1)) - F(node_i)) / (node_(i+1) - node_i).
 * Reading R-14: outside the model's nodes the integrated flux is held at its end values (the clamp of the
 * usual interp routines), i.e. the model carries no flux there.  orc_obs_nodes: the observed integration nodes of P:92,
 * lambda'' = exp(lambda_2i -+ dlambda_2 / 2) in the base the grid is stored in (log10 here): per segment, nodes at the
 * midpoints in log-wavelength of neighbouring pixels and half a step beyond the first and the last pixel -- on a uniform
 * log grid exactly the paper's. */
void orc_obs_nodes(const double *loglam, int p, double *nodes)
{
    if (p == 1) { nodes[0] = pow(10.0, loglam[0] - 0.5e-4); nodes[1] = pow(10.0, loglam[0] + 0.5e-4); return; }
    nodes[0] = pow(10.0, loglam[0] - 0.5 * (loglam[1] - loglam[0]));
    for (int i = 1; i < p; ++i) nodes[i] = pow(10.0, 0.5 * (loglam[i - 1] + loglam[i]));
    nodes[p] = pow(10.0, loglam[p - 1] + 0.5 * (loglam[p - 1] - loglam[p - 2]));
}

void orc_resample(int q, double lam1, double dlam1, const double *T, int p, const double *nodes, double *out)
{
    double *cum = calloc((size_t)q + 1, 8), *F = calloc((size_t)p + 1, 8);
    for (int m = 1; m <= q; ++m) cum[m] = cum[m - 1] + T[m - 1] * dlam1;             /* Eq. 2 */
    for (int i = 0; i <= p; ++i) {                                                   /* Eq. 3 */
        double t = (nodes[i] - (lam1 - 0.5 * dlam1)) / dlam1;                        /* position in units of model nodes */
        if (t <= 0.0) F[i] = cum[0];
        else if (t >= (double)q) F[i] = cum[q];
        else {
            int m = (int)floor(t);
            F[i] = cum[m] + (cum[m + 1] - cum[m]) * (t - (double)m);
        }
    }
    for (int i = 0; i < p; ++i) out[i] = (F[i + 1] - F[i]) / (nodes[i + 1] - nodes[i]);   /* Eq. 4 */
    free(cum); free(F);
}

/* The resampler applied to every row of a coefficient table [K][q] -> [K][n_pix] (Delta-4: it is linear and does not
 * depend on the parameters, so resampling the coefficients once equals resampling every model spectrum). */
void orc_resample_coeffs(int K, int q, double lam1, double dlam1, const double *coef, int n_pix, int n_seg,
                         const int32_t *seg_offset, const double *loglam, double *out)
{
    double *nodes = calloc((size_t)n_pix + 1, 8);
    for (int s = 0; s < n_seg; ++s) {
        int o = seg_offset[s], ps = seg_offset[s + 1] - o;
        orc_obs_nodes(loglam + o, ps, nodes);
        for (int k = 0; k < K; ++k) orc_resample(q, lam1, dlam1, coef + (size_t)k * q, ps, nodes, out + (size_t)k * n_pix + o);
    }
    free(nodes);
}

/* Pins call these two directly. */
int orc_solve_continuum(const orc_model *m, const double *S, const double *y, const double *w,
                        double *b, double *c)
{
    work_t *k = work_new(m);
    memcpy(k->S, S, 8 * (size_t)k->P);
    memcpy(k->w, w, 8 * (size_t)k->P);
    int st = solve_continuum(m, k, y);
    memcpy(b, k->b, 8 * (size_t)k->nc);
    if (c) memcpy(c, k->c, 8 * (size_t)k->P);
    work_free(k);
    return st;
}

int orc_support_cap(const orc_model *m) { return support_cap(m); }
