// lasp_device.cuh -- device code of the LASP-Adam fitting hot path for sm_100a.
//
// Mapping: ONE WARP LANE = ONE SPECTRUM.  A warp owns a tile of 32
// spectra and walks the pixels in chunks of CH; every per-spectrum quantity is private to its
// lane, so there is no cross-thread reduction anywhere on the per-pixel path.  Spectrum-
// independent operands (emulator coefficients C, Chebyshev nodes, pixel scales) are warp-uniform
// loads.  Per-lane small state (Adam moments, phi, continuum moments, tap weights) lives in shared
// memory as rows of 32 lanes with stride RS=33 (conflict-free both lane-wise and for the
// warp-cooperative Cholesky that reads one lane's column across rows).
//
// Paper / survey references: Eq. n and P:n are /root/reference/PAPER.md; C.2-n are the readings of
// SURVEY.md 8(c); a0..a9 are the steps of SURVEY.md 8(a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lasp_gpu.h"

#define CH 8   // pixels per register chunk
#define RS 33  // shared-memory row stride (floats)
#define FULL 0xffffffffu
#define LASP_NPMAX (LASP_MAX_LABELS + 2)

// scratch arrays, each [Ppad][32] floats per warp slot
enum { A_T = 0, A_S, A_DSV, A_DSS, A_CP, A_A, A_EI, A_TT, A_X, A_J0 };

struct SegDev {
    int po;       // first padded pixel of the segment (multiple of CH)
    int len;      // padded length = halo + roundup(P,CH) + halo
    int halo;     // replicated-edge columns on each side (multiple of CH, >= largest support H)
    int P, o;     // real length and real offset
    int fit_lo, fit_hi;  // chunk-aligned padded range containing every pixel that can have w>0
    int uniform;  // 1: constant km/s per pixel (log grid) -> one kernel per spectrum per step
    float inv_s;  // 1/s (pixels per km/s) when uniform, else the LARGEST 1/s_j of the segment
    float sig_inst;
    float ta, tb; // Chebyshev node t = ta*(jp - po - halo) + tb, t in [-1,1] over the fitted pixels
};

struct ModelDev {
    int n_seg, L, K, NP, D, n1, nmom, Ppad, P, nc, Hmax;
    SegDev seg[LASP_MAX_SEG];
    const float *C;        // [K][Ppad] emulator coefficients in the padded layout (halos replicate edges)
    const float *inv_s;    // [Ppad] 1/s_j
    const uint8_t *exps;   // [K][L]
    const double *conv;    // [n_seg][n1][n1] internal Chebyshev(t) -> plain Legendre(x^) (C.2-8)
    float lo[LASP_NPMAX], hi[LASP_NPMAX];
    float emu_a[LASP_MAX_LABELS], emu_b[LASP_MAX_LABELS];
    uint8_t label_log10[LASP_MAX_LABELS];
    // shared-memory row offsets (per warp)
    int r_U, r_M, r_V, r_PHI, r_Q, r_G, r_MOM, r_RHS, r_B, rows;
    int nscr;  // scratch arrays per warp slot
};

#define SMR(r) sm[(r) * RS + lane]

__device__ __forceinline__ int warp_max_i(int v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = max(v, __shfl_xor_sync(FULL, v, o));
    return v;
}
__device__ __forceinline__ float warp_sum_f(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(FULL, v, o);
    return v;
}

// ------------------------------------------------------------------------------------------
// a1: de-normalise, emulator inputs, monomials phi_k -> shared memory (Eq. 1, C.2-18/19)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float label_x(const ModelDev &M, int l, float theta)
{
    return M.emu_a[l] * (M.label_log10[l] ? log10f(theta) : theta) + M.emu_b[l];
}

__device__ void setup_params(const ModelDev &M, float *sm, int lane, float *x, float &v, float &sigstar)
{
    for (int l = 0; l < M.L; ++l) {
        float u = SMR(M.r_U + l);
        float th = M.lo[l] + (u + 1.f) * (M.hi[l] - M.lo[l]) * 0.5f;
        x[l] = label_x(M, l, th);
    }
    {
        float u = SMR(M.r_U + M.L);
        v = M.lo[M.L] + (u + 1.f) * (M.hi[M.L] - M.lo[M.L]) * 0.5f;
        u = SMR(M.r_U + M.L + 1);
        sigstar = M.lo[M.L + 1] + (u + 1.f) * (M.hi[M.L + 1] - M.lo[M.L + 1]) * 0.5f;
    }
    for (int k = 0; k < M.K; ++k) {
        float p = 1.f;
        for (int l = 0; l < M.L; ++l) {
            int e = M.exps[k * M.L + l];
            for (int q = 0; q < e; ++q) p *= x[l];
        }
        SMR(M.r_PHI + k) = p;
    }
}

// a2: T_j = sum_k phi_k C[k,j] over the padded range [lo,hi) -> scratch T  (Eq. 1)
__device__ void phase_T(const ModelDev &M, const float *sm, int lane, float *scr, int lo, int hi)
{
    float *Tcol = scr + (size_t)A_T * M.Ppad * 32 + lane;
    for (int jp0 = lo; jp0 < hi; jp0 += CH) {
        float T[CH];
#pragma unroll
        for (int i = 0; i < CH; ++i) T[i] = 0.f;
        const float *c = M.C + jp0;
        for (int k = 0; k < M.K; ++k) {
            float ph = SMR(M.r_PHI + k);
            const float4 a = __ldg((const float4 *)(c + (size_t)k * M.Ppad));
            const float4 b = __ldg((const float4 *)(c + (size_t)k * M.Ppad) + 1);
            T[0] = fmaf(ph, a.x, T[0]); T[1] = fmaf(ph, a.y, T[1]);
            T[2] = fmaf(ph, a.z, T[2]); T[3] = fmaf(ph, a.w, T[3]);
            T[4] = fmaf(ph, b.x, T[4]); T[5] = fmaf(ph, b.y, T[5]);
            T[6] = fmaf(ph, b.z, T[6]); T[7] = fmaf(ph, b.w, T[7]);
        }
#pragma unroll
        for (int i = 0; i < CH; ++i) Tcol[(size_t)(jp0 + i) * 32] = T[i];
    }
}

// ------------------------------------------------------------------------------------------
// a3: kernel weights of a uniform (log-grid) segment: one Gaussian per spectrum per step
// (Eq. 5; C.2-9/10/15).  Row m of G holds g_k for k = m - Hw, zero outside the lane's
// own support |k| <= H.  Returns the warp-wide largest support Hw.
// ------------------------------------------------------------------------------------------
struct UniW {
    float mu, e1n, e2n, cmu, csig;  // moments of the normalised kernel and derivative scalings
};

__device__ int setup_weights_uniform(const ModelDev &M, const SegDev &sg, float *sm, int lane, float v,
                                     float sigstar, UniW &w)
{
    float sigtot = sqrtf(sigstar * sigstar + sg.sig_inst * sg.sig_inst);
    float mu = v * sg.inv_s, s = sigtot * sg.inv_s;
    int H = (int)ceilf(fabsf(mu) + 5.f * s);
    H = min(max(H, 0), sg.halo);  // memory safety for parameters outside the prior box
    int Hw = warp_max_i(H);
    float i2 = 0.5f / (s * s);
    float sum = 0.f, s1 = 0.f, s2 = 0.f;
    for (int k = -H; k <= H; ++k) {
        float d = (float)k - mu;
        float e = expf(-d * d * i2);
        sum += e; s1 = fmaf(e, d, s1); s2 = fmaf(e * d, d, s2);
    }
    float inv = 1.f / sum;
    for (int m = 0; m <= 2 * Hw; ++m) {
        int k = m - Hw;
        float d = (float)k - mu;
        SMR(M.r_G + m) = (k >= -H && k <= H) ? expf(-d * d * i2) * inv : 0.f;
    }
    w.mu = mu;
    w.e1n = s1 * inv;            // kbar - mu
    w.e2n = s2 * inv;            // second moment about mu
    float is2 = 2.f * i2;        // 1/sigma^2 (pixels)
    w.cmu = is2 * sg.inv_s;      // dS/dv     = (1/s)   sum_k dg_k/dmu    T   (C.1)
    w.csig = is2 * sqrtf(is2) * (sigstar / sigtot) * sg.inv_s;  // dS/dsigma* = sigma*/(sigtot s) sum_k dg_k/dsigma T
    return Hw;
}

// a4: sliding-window stencil for CH outputs with one shared kernel (uniform segment).
// Output i sits at padded pixel jp0+i; tap m has offset k = m-Hw and reads T[jp0+i-k].  The window
// p[] is rotated statically inside the unrolled block, so each tap costs one new load.
template <bool DERIV>
__device__ __forceinline__ void stencil_uniform_chunk(const float *__restrict__ Tcol, const float *smG,
                                                      int jp0, int Hw, const UniW &w, float (&A0)[CH],
                                                      float (&A1)[CH], float (&A2)[CH])
{
    float p[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        p[i] = Tcol[(size_t)(jp0 + Hw + i) * 32];
        A0[i] = 0.f; A1[i] = 0.f; A2[i] = 0.f;
    }
    const int ntap = 2 * Hw + 1;
    for (int mb = 0; mb < ntap; mb += CH) {
        float nw[CH];
#pragma unroll
        for (int s = 0; s < CH; ++s) {
            int m1 = mb + s + 1;
            nw[s] = (m1 < ntap) ? Tcol[(size_t)(jp0 + Hw - m1) * 32] : 0.f;
        }
#pragma unroll
        for (int s = 0; s < CH; ++s) {
            int m = mb + s;
            if (m < ntap) {
                float g = smG[m * RS];
                float w1 = 0.f, w2 = 0.f;
                if (DERIV) {
                    float d = (float)(m - Hw) - w.mu;
                    w1 = g * (d - w.e1n) * w.cmu;
                    w2 = g * (d * d - w.e2n) * w.csig;
                }
#pragma unroll
                for (int i = 0; i < CH; ++i) {
                    float r = p[(i - s + CH) % CH];
                    A0[i] = fmaf(g, r, A0[i]);
                    if (DERIV) { A1[i] = fmaf(w1, r, A1[i]); A2[i] = fmaf(w2, r, A2[i]); }
                }
                p[(CH - 1 - s) % CH] = nw[s];
            }
        }
    }
}

// a3+a4 for a segment with a per-pixel kernel (linear grid; C.2-14): weights are generated on the
// fly for every (pixel, tap).  Outputs S, dS/dv, dS/dsigma*, and 1/E0 (needed by the adjoint).
template <bool DERIV>
__device__ __forceinline__ void stencil_general_chunk(const ModelDev &M, const SegDev &sg,
                                                      const float *__restrict__ Tcol, int jp0, float v,
                                                      float sigstar, float sigtot, float (&S)[CH],
                                                      float (&DSV)[CH], float (&DSS)[CH], float (&EI)[CH])
{
    float mu[CH], i2[CH], Hf[CH], is[CH];
    int Hc = 0;
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        is[i] = __ldg(M.inv_s + jp0 + i);
        mu[i] = v * is[i];
        float s = sigtot * is[i];
        int H = (int)ceilf(fabsf(mu[i]) + 5.f * s);
        H = min(max(H, 0), sg.halo);
        Hf[i] = (float)H;
        i2[i] = 0.5f / (s * s);
        Hc = max(Hc, H);
    }
    Hc = warp_max_i(Hc);
    float p[CH], E0[CH], E1[CH], E2[CH], A0[CH], A1[CH], A2[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        p[i] = Tcol[(size_t)(jp0 + Hc + i) * 32];
        E0[i] = E1[i] = E2[i] = A0[i] = A1[i] = A2[i] = 0.f;
    }
    const int ntap = 2 * Hc + 1;
    for (int mb = 0; mb < ntap; mb += CH) {
        float nw[CH];
#pragma unroll
        for (int s = 0; s < CH; ++s) {
            int m1 = mb + s + 1;
            nw[s] = (m1 < ntap) ? Tcol[(size_t)(jp0 + Hc - m1) * 32] : 0.f;
        }
#pragma unroll
        for (int s = 0; s < CH; ++s) {
            int m = mb + s;
            if (m < ntap) {
                float kf = (float)(m - Hc);
#pragma unroll
                for (int i = 0; i < CH; ++i) {
                    float d = kf - mu[i];
                    float e = (fabsf(kf) <= Hf[i]) ? __expf(-d * d * i2[i]) : 0.f;
                    float r = p[(i - s + CH) % CH];
                    E0[i] += e;
                    A0[i] = fmaf(e, r, A0[i]);
                    if (DERIV) {
                        float ed = e * d, edd = ed * d;
                        E1[i] += ed; E2[i] += edd;
                        A1[i] = fmaf(ed, r, A1[i]);
                        A2[i] = fmaf(edd, r, A2[i]);
                    }
                }
                p[(CH - 1 - s) % CH] = nw[s];
            }
        }
    }
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        float inv = 1.f / E0[i];
        S[i] = A0[i] * inv;
        EI[i] = inv;
        if (DERIV) {
            float is2 = 2.f * i2[i];
            float smu = (A1[i] * inv - E1[i] * inv * S[i]) * is2;
            float ssg = (A2[i] * inv - E2[i] * inv * S[i]) * is2 * sqrtf(is2);
            DSV[i] = smu * is[i];
            DSS[i] = ssg * (sigstar / sigtot) * is[i];
        } else {
            DSV[i] = 0.f; DSS[i] = 0.f;
        }
    }
}

// ------------------------------------------------------------------------------------------
// a5: continuum.  Internal basis: Chebyshev T_n(t), t rescaled to the FITTED pixel range of the
// segment, which keeps the weighted Gram matrix at cond ~30 in fp32.
// Any basis of the degree-D polynomials gives the same WLS continuum (Eq. 6); coefficients are
// converted to the paper's plain Legendre basis on output (C.2-8).
// The Gram matrix is never accumulated: T_m T_n = (T_{m+n} + T_{|m-n|})/2, so the 2D+1 moments
//   mom_n = sum_j w_j S_j^2 T_n(t_j)           (SURVEY.md section 7 "moment route")
// determine it, and the right-hand side is residual-based (iterative-refinement form):
//   rhs_n = sum_j w_j S_j (y_j - cprev_j S_j) T_n(t_j),   b = bprev + A^-1 rhs.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ void moments_chunk(const ModelDev &M, const SegDev &sg, float *sm, int lane,
                                              int jp0, const float (&S)[CH], const float2 *__restrict__ ywcol,
                                              const float *__restrict__ cpcol)
{
    float u[CH], vv[CH], a[CH], b[CH], x2[CH];
    float pm = 0.f, pr = 0.f;
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        float2 yw = ywcol[(size_t)(jp0 + i) * 32];
        float cp = cpcol[(size_t)(jp0 + i) * 32];
        float ws = yw.y * S[i];
        u[i] = ws * S[i];
        vv[i] = ws * fmaf(-cp, S[i], yw.x);
        float t = fmaf(sg.ta, (float)(jp0 + i - sg.po - sg.halo), sg.tb);
        a[i] = 1.f; b[i] = t; x2[i] = 2.f * t;
        pm += u[i]; pr += vv[i];
    }
    SMR(M.r_MOM) += pm;
    SMR(M.r_RHS) += pr;
    for (int n = 1; n < M.nmom; ++n) {
        pm = 0.f;
#pragma unroll
        for (int i = 0; i < CH; ++i) pm = fmaf(u[i], b[i], pm);
        SMR(M.r_MOM + n) += pm;
        if (n < M.n1) {
            pr = 0.f;
#pragma unroll
            for (int i = 0; i < CH; ++i) pr = fmaf(vv[i], b[i], pr);
            SMR(M.r_RHS + n) += pr;
        }
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            float nx = fmaf(x2[i], b[i], -a[i]);
            a[i] = b[i]; b[i] = nx;
        }
    }
}

// c_j = sum_n b_n T_n(t_j) for the CH pixels at jp0
__device__ __forceinline__ void cont_chunk(const ModelDev &M, const SegDev &sg, const float *sm, int lane,
                                           int rowB, int jp0, float (&c)[CH])
{
    float a[CH], b[CH], x2[CH];
    float b0 = SMR(rowB);
#pragma unroll
    for (int i = 0; i < CH; ++i) {
        float t = fmaf(sg.ta, (float)(jp0 + i - sg.po - sg.halo), sg.tb);
        a[i] = 1.f; b[i] = t; x2[i] = 2.f * t;
        c[i] = b0;
    }
    for (int n = 1; n < M.n1; ++n) {
        float bn = SMR(rowB + n);
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            c[i] = fmaf(bn, b[i], c[i]);
            float nx = fmaf(x2[i], b[i], -a[i]);
            a[i] = b[i]; b[i] = nx;
        }
    }
}

// Warp-cooperative Cholesky solve of the 32 lanes' systems, one spectrum at a time, lanes = rows.
// A_ij = (mom_{i+j} + mom_{|i-j|})/2 ; b += A^-1 rhs.  Returns a bit mask of spectra whose system
// was not positive definite (their b is set to 0; status bit LASP_ST_NOT_SPD).
__device__ unsigned warp_solve_segment(const ModelDev &M, float *sm, int lane, int rowB)
{
    const int n1 = M.n1;
    unsigned fail = 0;
    __syncwarp();
    for (int sp = 0; sp < 32; ++sp) {
        float row[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) {
            float a = (j == lane) ? 1.f : 0.f;
            if (j < n1 && lane < n1) {
                int d = lane - j;
                d = d < 0 ? -d : d;
                a = 0.5f * (sm[(M.r_MOM + lane + j) * RS + sp] + sm[(M.r_MOM + d) * RS + sp]);
            }
            row[j] = a;
        }
        float r = (lane < n1) ? sm[(M.r_RHS + lane) * RS + sp] : 0.f;
        bool ok = true;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if (k < n1) {
                float d0 = 0.5f * (sm[(M.r_MOM + 2 * k) * RS + sp] + sm[M.r_MOM * RS + sp]);
                float d = __shfl_sync(FULL, row[k], k);
                if (!(d > 1e-6f * d0)) ok = false;
                float rinv = rsqrtf(d);
                float lik = row[k] * rinv;
                row[k] = lik;
#pragma unroll
                for (int j = k + 1; j < 32; ++j) {
                    if (j < n1) {
                        float ljk = __shfl_sync(FULL, lik, j);
                        row[j] = fmaf(-lik, ljk, row[j]);
                    }
                }
            }
        }
        // forward substitution L y = rhs
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if (k < n1) {
                float diag = __shfl_sync(FULL, row[k], k);
                float yk = __shfl_sync(FULL, r, k) / diag;
                if (lane > k) r = fmaf(-row[k], yk, r);
                else if (lane == k) r = yk;
            }
        }
        // back substitution L^T x = y
#pragma unroll
        for (int k = 31; k >= 0; --k) {
            if (k < n1) {
                float part = (lane > k && lane < n1) ? row[k] * r : 0.f;
                part = warp_sum_f(part);
                float diag = __shfl_sync(FULL, row[k], k);
                float xk = (__shfl_sync(FULL, r, k) - part) / diag;
                if (lane == k) r = xk;
            }
        }
        if (lane < n1) {
            if (ok) sm[(rowB + lane) * RS + sp] += r;
            else sm[(rowB + lane) * RS + sp] = 0.f;
        }
        if (!ok) fail |= (1u << sp);
    }
    __syncwarp();
    return fail;
}

// ------------------------------------------------------------------------------------------
// Per-segment passes
// ------------------------------------------------------------------------------------------
struct SegCtx {  // per-step, per-segment lane state
    int Hw;      // warp-wide support bound used for the T range
    int loT, hiT;
    UniW w;
    float sigtot;
};

__device__ __forceinline__ int roundup_ch(int v) { return (v + CH - 1) / CH * CH; }

// weights + T range + emulator
__device__ void seg_prepare(const ModelDev &M, const SegDev &sg, float *sm, int lane, float *scr, float v,
                            float sigstar, int out_lo, int out_hi, SegCtx &c)
{
    c.sigtot = sqrtf(sigstar * sigstar + sg.sig_inst * sg.sig_inst);
    if (sg.uniform) {
        c.Hw = setup_weights_uniform(M, sg, sm, lane, v, sigstar, c.w);
    } else {
        int H = (int)ceilf((fabsf(v) + 5.f * c.sigtot) * sg.inv_s);  // inv_s = largest 1/s_j of the segment
        c.Hw = warp_max_i(min(max(H, 0), sg.halo));
    }
    int Hr = roundup_ch(c.Hw);
    c.loT = max(sg.po, out_lo - Hr);
    c.hiT = min(sg.po + sg.len, out_hi + Hr);
    phase_T(M, sm, lane, scr, c.loT, c.hiT);
}

// stencil over the chunks of [lo,hi): writes S (and dS/dv, dS/dsigma*, 1/E0) to scratch
template <bool DERIV>
__device__ void seg_stencil(const ModelDev &M, const SegDev &sg, const float *sm, int lane, float *scr,
                            float v, float sigstar, const SegCtx &c, int lo, int hi)
{
    const size_t AS = (size_t)M.Ppad * 32;
    const float *Tcol = scr + A_T * AS + lane;
    float *Sc = scr + A_S * AS + lane, *Vc = scr + A_DSV * AS + lane, *Gc = scr + A_DSS * AS + lane;
    float *Ec = scr + A_EI * AS + lane;
    for (int jp0 = lo; jp0 < hi; jp0 += CH) {
        float S[CH], DV[CH], DS[CH];
        if (sg.uniform) {
            stencil_uniform_chunk<DERIV>(Tcol, sm + M.r_G * RS + lane, jp0, c.Hw, c.w, S, DV, DS);
        } else {
            float EI[CH];
            stencil_general_chunk<DERIV>(M, sg, Tcol, jp0, v, sigstar, c.sigtot, S, DV, DS, EI);
#pragma unroll
            for (int i = 0; i < CH; ++i) Ec[(size_t)(jp0 + i) * 32] = EI[i];
        }
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            Sc[(size_t)(jp0 + i) * 32] = S[i];
            if (DERIV) { Vc[(size_t)(jp0 + i) * 32] = DV[i]; Gc[(size_t)(jp0 + i) * 32] = DS[i]; }
        }
    }
}

// moments + solve: b += A^-1 Phi^T W (y - cprev S).  Returns the not-SPD mask.
__device__ unsigned seg_solve(const ModelDev &M, const SegDev &sg, float *sm, int lane, const float *scr,
                              const float2 *ywcol, int rowB)
{
    const size_t AS = (size_t)M.Ppad * 32;
    const float *Sc = scr + A_S * AS + lane, *Cc = scr + A_CP * AS + lane;
    for (int n = 0; n < M.nmom; ++n) SMR(M.r_MOM + n) = 0.f;
    for (int n = 0; n < M.n1; ++n) SMR(M.r_RHS + n) = 0.f;
    for (int jp0 = sg.fit_lo; jp0 < sg.fit_hi; jp0 += CH) {
        float S[CH];
#pragma unroll
        for (int i = 0; i < CH; ++i) S[i] = Sc[(size_t)(jp0 + i) * 32];
        moments_chunk(M, sg, sm, lane, jp0, S, ywcol, Cc);
    }
    return warp_solve_segment(M, sm, lane, rowB);
}

// c from the current b -> scratch CP (used between the two solves of a cold start)
__device__ void seg_ceval(const ModelDev &M, const SegDev &sg, const float *sm, int lane, float *scr, int rowB)
{
    float *Cc = scr + (size_t)A_CP * M.Ppad * 32 + lane;
    for (int jp0 = sg.fit_lo; jp0 < sg.fit_hi; jp0 += CH) {
        float c[CH];
        cont_chunk(M, sg, sm, lane, rowB, jp0, c);
#pragma unroll
        for (int i = 0; i < CH; ++i) Cc[(size_t)(jp0 + i) * 32] = c[i];
    }
}

struct Acc {  // per-lane accumulators of one evaluation
    float chi2, gv, gs, cmin;
    int ngood;
};

// a6: residual, chi2, adjoint a_j = -2 w r c, dchi2/dv, dchi2/dsigma*; stores c (-> cprev of the
// next step) and a.  MODE 0: gradient evaluation; MODE 1: store rho = sqrt(w) r into array `xarr`.
template <int MODE>
__device__ void seg_residual(const ModelDev &M, const SegDev &sg, const float *sm, int lane, float *scr,
                             const float2 *ywcol, int rowB, Acc &acc, int xarr)
{
    const size_t AS = (size_t)M.Ppad * 32;
    const float *Sc = scr + A_S * AS + lane, *Vc = scr + A_DSV * AS + lane, *Gc = scr + A_DSS * AS + lane;
    const float *Ec = scr + A_EI * AS + lane;
    float *Cc = scr + A_CP * AS + lane, *Ac = scr + A_A * AS + lane;
    float *Xc = scr + (size_t)xarr * AS + lane;
    for (int jp0 = sg.fit_lo; jp0 < sg.fit_hi; jp0 += CH) {
        float c[CH];
        cont_chunk(M, sg, sm, lane, rowB, jp0, c);
        float chi = 0.f, gv = 0.f, gs = 0.f;
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            size_t o = (size_t)(jp0 + i) * 32;
            float2 yw = ywcol[o];
            float S = Sc[o];
            float r = fmaf(-c[i], S, yw.x);
            float wr = yw.y * r;
            chi = fmaf(wr, r, chi);
            Cc[o] = c[i];
            if (yw.y > 0.f) { acc.cmin = fminf(acc.cmin, c[i]); acc.ngood++; }
            if (MODE == 0) {
                float a = -2.f * wr * c[i];
                gv = fmaf(a, Vc[o], gv);
                gs = fmaf(a, Gc[o], gs);
                Ac[o] = sg.uniform ? a : a * Ec[o];
            } else {
                Xc[o] = sqrtf(yw.y) * r;
            }
        }
        acc.chi2 += chi; acc.gv += gv; acc.gs += gs;
    }
}

__device__ __forceinline__ void q_accum_chunk(const ModelDev &M, float *sm, int lane, int jp0,
                                              const float (&t)[CH])
{
    const float *c = M.C + jp0;
    for (int k = 0; k < M.K; ++k) {
        const float4 a = __ldg((const float4 *)(c + (size_t)k * M.Ppad));
        const float4 b = __ldg((const float4 *)(c + (size_t)k * M.Ppad) + 1);
        float s = t[0] * a.x;
        s = fmaf(t[1], a.y, s); s = fmaf(t[2], a.z, s); s = fmaf(t[3], a.w, s);
        s = fmaf(t[4], b.x, s); s = fmaf(t[5], b.y, s); s = fmaf(t[6], b.z, s); s = fmaf(t[7], b.w, s);
        SMR(M.r_Q + k) += s;
    }
}

// a7: adjoint stencil t_i = sum_j a_j g_{j,j-i} and q_k = sum_i t_i C[k,i]  (reverse mode)
__device__ void seg_adjoint(const ModelDev &M, const SegDev &sg, float *sm, int lane, float *scr, float v,
                            float sigstar, const SegCtx &c)
{
    const size_t AS = (size_t)M.Ppad * 32;
    const float *Ac = scr + A_A * AS + lane;
    if (sg.uniform) {
        // gather form: t_i = sum_k g_k a_{i+k}; a is zero outside the fitted range
        const float *smG = sm + M.r_G * RS + lane;
        const int Hw = c.Hw, ntap = 2 * Hw + 1;
        const int flo = sg.fit_lo, fhi = sg.fit_hi;
        for (int jp0 = c.loT; jp0 < c.hiT; jp0 += CH) {
            float p[CH], t[CH];
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                int idx = jp0 - Hw + i;
                p[i] = (idx >= flo && idx < fhi) ? Ac[(size_t)idx * 32] : 0.f;
                t[i] = 0.f;
            }
            for (int mb = 0; mb < ntap; mb += CH) {
                float nw[CH];
#pragma unroll
                for (int s = 0; s < CH; ++s) {
                    int idx = jp0 + CH - Hw + mb + s;
                    nw[s] = (mb + s + 1 < ntap && idx >= flo && idx < fhi) ? Ac[(size_t)idx * 32] : 0.f;
                }
#pragma unroll
                for (int s = 0; s < CH; ++s) {
                    int m = mb + s;
                    if (m < ntap) {
                        float g = smG[m * RS];
#pragma unroll
                        for (int i = 0; i < CH; ++i) t[i] = fmaf(g, p[(i + s) % CH], t[i]);
                        p[s % CH] = nw[s];
                    }
                }
            }
            q_accum_chunk(M, sm, lane, jp0, t);
        }
    } else {
        // scatter form: source pixel j (weights of ITS kernel, normalised by its 1/E0 already folded
        // into a) adds a_j e_{j,k} to t_{j-k}; t accumulates in scratch TT, then q in a second pass.
        float *Tt = scr + A_TT * AS + lane;
        for (int jp = c.loT; jp < c.hiT; ++jp) Tt[(size_t)jp * 32] = 0.f;
        for (int jp0 = sg.fit_lo; jp0 < sg.fit_hi; jp0 += CH) {
            float mu[CH], i2[CH], Hf[CH], av[CH], ac[CH];
            int Hc = 0;
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                float is = __ldg(M.inv_s + jp0 + i);
                mu[i] = v * is;
                float s = c.sigtot * is;
                int H = (int)ceilf(fabsf(mu[i]) + 5.f * s);
                H = min(max(H, 0), sg.halo);
                Hf[i] = (float)H;
                i2[i] = 0.5f / (s * s);
                Hc = max(Hc, H);
                av[i] = Ac[(size_t)(jp0 + i) * 32];
                ac[i] = 0.f;
            }
            Hc = warp_max_i(Hc);
            const int ntap_pad = roundup_ch(2 * Hc + 1);
            for (int mb = 0; mb < ntap_pad; mb += CH) {
#pragma unroll
                for (int s = 0; s < CH; ++s) {
                    int m = mb + s;
                    float kf = (float)(m - Hc);
#pragma unroll
                    for (int i = 0; i < CH; ++i) {
                        float d = kf - mu[i];
                        float e = (fabsf(kf) <= Hf[i]) ? __expf(-d * d * i2[i]) : 0.f;
                        ac[(i - s + CH) % CH] = fmaf(av[i], e, ac[(i - s + CH) % CH]);
                    }
                    // logical CH-1 (target jp0+CH-1+Hc-m) is complete for this chunk: retire it
                    int tgt = jp0 + CH - 1 + Hc - m;
                    float val = ac[(CH - 1 - s) % CH];
                    if (tgt >= c.loT && tgt < c.hiT) Tt[(size_t)tgt * 32] += val;
                    ac[(CH - 1 - s) % CH] = 0.f;
                }
            }
            // after ntap_pad taps the rotation is back to identity; flush the rest
#pragma unroll
            for (int i = 0; i < CH - 1; ++i) {
                int tgt = jp0 + i + Hc - ntap_pad;
                if (tgt >= c.loT && tgt < c.hiT) Tt[(size_t)tgt * 32] += ac[i];
            }
        }
        for (int jp0 = c.loT; jp0 < c.hiT; jp0 += CH) {
            float t[CH];
#pragma unroll
            for (int i = 0; i < CH; ++i) t[i] = Tt[(size_t)(jp0 + i) * 32];
            q_accum_chunk(M, sm, lane, jp0, t);
        }
    }
}

// ------------------------------------------------------------------------------------------
// One evaluation of chi2 (+ gradient) at the u held in shared memory.
//   COLD: the continuum starts from b = 0 and is solved twice (solve + one refinement);
//   otherwise b, cprev are warm from the previous evaluation and one residual-based solve suffices.
//   MODE 0: chi2 + gradient wrt u -> grad[] ; MODE 1: chi2 + rho -> scratch array xarr.
// ------------------------------------------------------------------------------------------
template <int MODE>
__device__ __noinline__ void evaluate(const ModelDev &M, float *sm, int lane, float *scr, const float2 *ywcol, bool cold,
                         Acc &acc, float *grad, unsigned &failmask, int xarr)
{
    float x[LASP_MAX_LABELS];
    float v, sigstar;
    setup_params(M, sm, lane, x, v, sigstar);
    acc.chi2 = 0.f; acc.gv = 0.f; acc.gs = 0.f; acc.cmin = 3.0e38f; acc.ngood = 0;
    failmask = 0;
    if (MODE == 0)
        for (int k = 0; k < M.K; ++k) SMR(M.r_Q + k) = 0.f;
    for (int s = 0; s < M.n_seg; ++s) {
        const SegDev &sg = M.seg[s];
        const int rowB = M.r_B + s * M.n1;
        if (sg.fit_hi <= sg.fit_lo) continue;
        SegCtx c;
        seg_prepare(M, sg, sm, lane, scr, v, sigstar, sg.fit_lo, sg.fit_hi, c);
        seg_stencil<MODE == 0>(M, sg, sm, lane, scr, v, sigstar, c, sg.fit_lo, sg.fit_hi);
        if (cold) {
            for (int n = 0; n < M.n1; ++n) SMR(rowB + n) = 0.f;
            seg_ceval(M, sg, sm, lane, scr, rowB);
            failmask |= seg_solve(M, sg, sm, lane, scr, ywcol, rowB);
            seg_ceval(M, sg, sm, lane, scr, rowB);
        }
        failmask |= seg_solve(M, sg, sm, lane, scr, ywcol, rowB);
        seg_residual<MODE>(M, sg, sm, lane, scr, ywcol, rowB, acc, xarr);
        if (MODE == 0) seg_adjoint(M, sg, sm, lane, scr, v, sigstar, c);
    }
    if (MODE == 0) {
        // chain rule to u: labels through dphi/dx, dx/dtheta, (hi-lo)/2 ; v and sigma* directly (C.1)
        for (int l = 0; l < M.L; ++l) {
            float gx = 0.f;
            for (int k = 0; k < M.K; ++k) {
                int el = M.exps[k * M.L + l];
                if (el == 0) continue;
                float d = (float)el;
                for (int l2 = 0; l2 < M.L; ++l2) {
                    int e2 = M.exps[k * M.L + l2] - (l2 == l ? 1 : 0);
                    for (int q = 0; q < e2; ++q) d *= x[l2];
                }
                gx = fmaf(d, SMR(M.r_Q + k), gx);
            }
            float u = SMR(M.r_U + l);
            float half = (M.hi[l] - M.lo[l]) * 0.5f;
            float th = M.lo[l] + (u + 1.f) * half;
            float dxdt = M.label_log10[l] ? M.emu_a[l] / (th * 2.302585093f) : M.emu_a[l];
            grad[l] = gx * dxdt * half;
        }
        grad[M.L] = acc.gv * (M.hi[M.L] - M.lo[M.L]) * 0.5f;
        grad[M.L + 1] = acc.gs * (M.hi[M.L + 1] - M.lo[M.L + 1]) * 0.5f;
    }
}
