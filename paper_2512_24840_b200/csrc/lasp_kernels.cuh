// lasp_kernels.cuh -- the __global__ entry points built on lasp_device.cuh.
#pragma once
#include "lasp_device.cuh"

struct FitArgs {
    const float2 *YW;  // staged {flux, w} in [tile][Ppad][32] layout
    float *scratch;    // [warp slot][nscr][Ppad][32]
    long long B;
    int tiles;
    const float *init;
    int n_iter;
    float lr, b1, b2, eps, fd_h;
    float *params, *cont, *chi2, *err;
    int *status;
    // lasp_eval_grad
    const float *gparams;
    float *grad_u;
    // lasp_eval_model
    const float *mcont;
    float *model;
};

// ------------------------------------------------------------------------------------------
// a0: stage.  w = mask*ivar, zero on the n_edge pixels at each end of each segment (Eq. 8 P:161,
// P:167), non-finite or non-positive ivar treated as masked; transpose to lane-major tiles so that
// the fit kernel's per-pixel loads are 256-byte coalesced.  YW is pre-zeroed (halos, tails).
// grid (ceil(P/32), tiles), block (32, 8).
// ------------------------------------------------------------------------------------------
__global__ void lasp_stage_kernel(const __grid_constant__ ModelDev M, const float *__restrict__ flux,
                                  const float *__restrict__ ivar, const uint8_t *__restrict__ mask,
                                  long long B, float2 *__restrict__ YW)
{
    __shared__ float2 tile[32][33];
    const int j = blockIdx.x * 32 + threadIdx.x;
    const long long t = blockIdx.y;
    for (int r = threadIdx.y; r < 32; r += 8) {
        long long i = t * 32 + r;
        float2 v = make_float2(0.f, 0.f);
        if (i < B && j < M.P) {
            size_t o = (size_t)i * M.P + j;
            float y = flux[o], w = ivar[o];
            if (mask && mask[o] == 0) w = 0.f;
            if (!(w > 0.f) || !isfinite(w) || !isfinite(y)) { w = 0.f; y = 0.f; }
            v = make_float2(y, w);
        }
        tile[r][threadIdx.x] = v;
    }
    __syncthreads();
    for (int c = threadIdx.y; c < 32; c += 8) {
        int jj = blockIdx.x * 32 + c;
        if (jj >= M.P) continue;
        int s = 0;
        while (s + 1 < M.n_seg && jj >= M.seg[s + 1].o) ++s;
        const SegDev &sg = M.seg[s];
        int rel = jj - sg.o;
        float2 v = tile[threadIdx.x][c];
        int jp = sg.po + sg.halo + rel;
        YW[((size_t)t * M.Ppad + jp) * 32 + threadIdx.x] = v;
    }
}

// Zero the weights on the excluded edge pixels (separate tiny pass keeps the transpose simple).
// grid (tiles), block 32: lane = spectrum.
__global__ void lasp_edge_kernel(const __grid_constant__ ModelDev M, const int *__restrict__ n_edge,
                                 float2 *__restrict__ YW)
{
    const size_t t = blockIdx.x;
    const int lane = threadIdx.x;
    for (int s = 0; s < M.n_seg; ++s) {
        const SegDev &sg = M.seg[s];
        int ne = min(n_edge[s], sg.P);
        for (int q = 0; q < ne; ++q) {
            int jp = sg.po + sg.halo + q;
            YW[(t * M.Ppad + jp) * 32 + lane].y = 0.f;
            jp = sg.po + sg.halo + sg.P - 1 - q;
            YW[(t * M.Ppad + jp) * 32 + lane].y = 0.f;
        }
    }
}

// ------------------------------------------------------------------------------------------
// helpers shared by the entry points
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float *warp_smem(const ModelDev &M, float *smem)
{
    return smem + (size_t)(threadIdx.x >> 5) * M.rows * RS;
}

__device__ __forceinline__ float *warp_scratch(const ModelDev &M, float *scratch)
{
    size_t slot = (size_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    return scratch + slot * (size_t)M.nscr * M.Ppad * 32;
}

// internal Chebyshev(t) coefficients -> plain Legendre(x^) (C.2-8), fp64
__device__ void write_cont(const ModelDev &M, const float *sm, int lane, float *out)
{
    for (int s = 0; s < M.n_seg; ++s) {
        const double *cv = M.conv + (size_t)s * M.n1 * M.n1;
        for (int m = 0; m < M.n1; ++m) {
            double acc = 0.0;
            for (int n = 0; n < M.n1; ++n) acc += cv[m * M.n1 + n] * (double)SMR(M.r_B + s * M.n1 + n);
            out[s * M.n1 + m] = (float)acc;
        }
    }
}

// ------------------------------------------------------------------------------------------
// lasp_fit_batch: a1-a9 for one tile of 32 spectra per warp
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 1)
lasp_fit_kernel(const __grid_constant__ ModelDev M, const FitArgs a)
{
    extern __shared__ float smem[];
    float *sm = warp_smem(M, smem);
    float *scr = warp_scratch(M, a.scratch);
    const int lane = threadIdx.x & 31;
    const int wpb = blockDim.x >> 5;
    const int NP = M.NP;
    for (int tile = blockIdx.x * wpb + (threadIdx.x >> 5); tile < a.tiles; tile += gridDim.x * wpb) {
        const long long i = (long long)tile * 32 + lane;
        const bool valid = i < a.B;
        const long long ic = valid ? i : a.B - 1;
        const float2 *ywcol = a.YW + (size_t)tile * M.Ppad * 32 + lane;
        for (int p = 0; p < NP; ++p) {
            float th = a.init[ic * NP + p];
            float u = 2.f * (th - M.lo[p]) / (M.hi[p] - M.lo[p]) - 1.f;
            SMR(M.r_U + p) = fminf(fmaxf(u, -1.f), 1.f);
            SMR(M.r_M + p) = 0.f;
            SMR(M.r_V + p) = 0.f;
        }
        Acc acc;
        unsigned fail = 0;
        float grad[LASP_NPMAX];
        float pb1 = 1.f, pb2 = 1.f;
        for (int t = 1; t <= a.n_iter; ++t) {
            evaluate<0>(M, sm, lane, scr, ywcol, t == 1, acc, grad, fail, A_X);
            pb1 *= a.b1; pb2 *= a.b2;
            // a8: Adam (C.2-20), then clip to the prior box (C.2-18)
            for (int p = 0; p < NP; ++p) {
                float g = grad[p];
                float m = a.b1 * SMR(M.r_M + p) + (1.f - a.b1) * g;
                float v = a.b2 * SMR(M.r_V + p) + (1.f - a.b2) * g * g;
                SMR(M.r_M + p) = m; SMR(M.r_V + p) = v;
                float mh = m / (1.f - pb1), vh = v / (1.f - pb2);
                float u = SMR(M.r_U + p) - a.lr * mh / (sqrtf(vh) + a.eps);
                if (!(u == u)) u = SMR(M.r_U + p);  // keep the iterate if the gradient was NaN
                SMR(M.r_U + p) = fminf(fmaxf(u, -1.f), 1.f);
            }
        }
        // a9: one more evaluation at the final iterate (C.2-21)
        evaluate<1>(M, sm, lane, scr, ywcol, a.n_iter == 0, acc, grad, fail, A_X);
        const float chi2 = acc.chi2;
        const int ngood = acc.ngood;
        int st = 0;
        if ((fail >> lane) & 1u) st |= LASP_ST_NOT_SPD;
        bool fin = isfinite(chi2);
        for (int p = 0; p < NP; ++p) {
            float u = SMR(M.r_U + p);
            fin = fin && isfinite(u);
            if (u <= -1.f || u >= 1.f) st |= LASP_ST_ON_BOUND;
        }
        for (int n = 0; n < M.nc; ++n) fin = fin && isfinite(SMR(M.r_B + n));
        if (!fin) st |= LASP_ST_NONFINITE;
        if (ngood > 0 && acc.cmin <= 0.f) st |= LASP_ST_NEG_CONT;
        if (valid) {
            for (int p = 0; p < NP; ++p)
                a.params[i * NP + p] = M.lo[p] + (SMR(M.r_U + p) + 1.f) * (M.hi[p] - M.lo[p]) * 0.5f;
            a.chi2[i] = chi2;
            if (a.status) a.status[i] = st;
            if (a.cont) write_cont(M, sm, lane, a.cont + i * M.nc);
        }
        if (a.err) {
            // step 9 (C.2-22/23): J by central differences of the re-solved whitened residual
            const size_t AS = (size_t)M.Ppad * 32;
            for (int p = 0; p < NP; ++p) {
                float u0 = SMR(M.r_U + p);
                float up = u0 + a.fd_h, um = u0 - a.fd_h;
                SMR(M.r_U + p) = up;
                evaluate<1>(M, sm, lane, scr, ywcol, false, acc, grad, fail, A_X);
                SMR(M.r_U + p) = um;
                evaluate<1>(M, sm, lane, scr, ywcol, false, acc, grad, fail, A_J0 + p);
                SMR(M.r_U + p) = u0;
                float inv = 1.f / (up - um);
                float *Jc = scr + (size_t)(A_J0 + p) * AS + lane;
                const float *Xc = scr + (size_t)A_X * AS + lane;
                for (int s = 0; s < M.n_seg; ++s)
                    for (int jp = M.seg[s].fit_lo; jp < M.seg[s].fit_hi; ++jp)
                        Jc[(size_t)jp * 32] = (Xc[(size_t)jp * 32] - Jc[(size_t)jp * 32]) * inv;
            }
            double N[LASP_NPMAX * (LASP_NPMAX + 1) / 2];
            for (int p = 0; p < NP; ++p)
                for (int q = 0; q <= p; ++q) {
                    const float *Jp = scr + (size_t)(A_J0 + p) * AS + lane;
                    const float *Jq = scr + (size_t)(A_J0 + q) * AS + lane;
                    double s0 = 0.0, s1 = 0.0;
                    for (int s = 0; s < M.n_seg; ++s)
                        for (int jp = M.seg[s].fit_lo; jp < M.seg[s].fit_hi; jp += 2) {
                            s0 += (double)Jp[(size_t)jp * 32] * (double)Jq[(size_t)jp * 32];
                            s1 += (double)Jp[(size_t)(jp + 1) * 32] * (double)Jq[(size_t)(jp + 1) * 32];
                        }
                    N[p * (p + 1) / 2 + q] = s0 + s1;
                }
            // Cholesky of J^T J (packed lower), then (J^T J)^-1_pp = |L^-1 e_p|^2
            bool ok = ngood > NP;
            for (int p = 0; p < NP && ok; ++p)
                for (int q = 0; q <= p; ++q) {
                    double s = N[p * (p + 1) / 2 + q];
                    for (int k = 0; k < q; ++k) s -= N[p * (p + 1) / 2 + k] * N[q * (q + 1) / 2 + k];
                    if (p == q) {
                        if (!(s > 0.0)) { ok = false; break; }
                        N[p * (p + 1) / 2 + p] = sqrt(s);
                    } else
                        N[p * (p + 1) / 2 + q] = s / N[q * (q + 1) / 2 + q];
                }
            const double s2 = (double)chi2 / (double)(ngood - NP);
            for (int p = 0; p < NP; ++p) {
                float e = __int_as_float(0x7fc00000);
                if (ok) {
                    double y[LASP_NPMAX];
                    double nrm = 0.0;
                    for (int r = p; r < NP; ++r) {
                        double s = (r == p) ? 1.0 : 0.0;
                        for (int k = p; k < r; ++k) s -= N[r * (r + 1) / 2 + k] * y[k];
                        y[r] = s / N[r * (r + 1) / 2 + r];
                        nrm += y[r] * y[r];
                    }
                    e = (float)(sqrt(s2 * nrm) * (double)(M.hi[p] - M.lo[p]) * 0.5);
                }
                if (valid) a.err[i * NP + p] = e;
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// lasp_eval_grad: one cold evaluation of chi2 and d chi2/d u at given physical parameters
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 1)
lasp_grad_kernel(const __grid_constant__ ModelDev M, const FitArgs a)
{
    extern __shared__ float smem[];
    float *sm = warp_smem(M, smem);
    float *scr = warp_scratch(M, a.scratch);
    const int lane = threadIdx.x & 31;
    const int wpb = blockDim.x >> 5;
    const int NP = M.NP;
    for (int tile = blockIdx.x * wpb + (threadIdx.x >> 5); tile < a.tiles; tile += gridDim.x * wpb) {
        const long long i = (long long)tile * 32 + lane;
        const bool valid = i < a.B;
        const long long ic = valid ? i : a.B - 1;
        const float2 *ywcol = a.YW + (size_t)tile * M.Ppad * 32 + lane;
        for (int p = 0; p < NP; ++p)
            SMR(M.r_U + p) = 2.f * (a.gparams[ic * NP + p] - M.lo[p]) / (M.hi[p] - M.lo[p]) - 1.f;
        Acc acc;
        unsigned fail = 0;
        float grad[LASP_NPMAX];
        evaluate<0>(M, sm, lane, scr, ywcol, true, acc, grad, fail, A_X);
        if (valid) {
            a.chi2[i] = acc.chi2;
            for (int p = 0; p < NP; ++p) a.grad_u[i * NP + p] = grad[p];
            if (a.status) a.status[i] = ((fail >> lane) & 1u) ? LASP_ST_NOT_SPD : 0;
            if (a.cont) write_cont(M, sm, lane, a.cont + i * M.nc);
        }
    }
}

// ------------------------------------------------------------------------------------------
// lasp_eval_model: model_j = c_j S_j with the continuum given as plain-Legendre coefficients
// ------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256, 1)
lasp_model_kernel(const __grid_constant__ ModelDev M, const FitArgs a)
{
    extern __shared__ float smem[];
    float *sm = warp_smem(M, smem);
    float *scr = warp_scratch(M, a.scratch);
    const int lane = threadIdx.x & 31;
    const int wpb = blockDim.x >> 5;
    const int NP = M.NP;
    const size_t AS = (size_t)M.Ppad * 32;
    for (int tile = blockIdx.x * wpb + (threadIdx.x >> 5); tile < a.tiles; tile += gridDim.x * wpb) {
        const long long i = (long long)tile * 32 + lane;
        const bool valid = i < a.B;
        const long long ic = valid ? i : a.B - 1;
        for (int p = 0; p < NP; ++p)
            SMR(M.r_U + p) = 2.f * (a.gparams[ic * NP + p] - M.lo[p]) / (M.hi[p] - M.lo[p]) - 1.f;
        for (int n = 0; n < M.nc; ++n) SMR(M.r_B + n) = a.mcont[ic * M.nc + n];
        float x[LASP_MAX_LABELS], v, sigstar;
        setup_params(M, sm, lane, x, v, sigstar);
        for (int s = 0; s < M.n_seg; ++s) {
            const SegDev &sg = M.seg[s];
            const int lo = sg.po + sg.halo, hi = sg.po + sg.len - sg.halo;
            SegCtx c;
            seg_prepare(M, sg, sm, lane, scr, v, sigstar, lo, hi, c);
            seg_stencil<false>(M, sg, sm, lane, scr, v, sigstar, c, lo, hi);
            const float *Sc = scr + A_S * AS + lane;
            for (int j = 0; j < sg.P; ++j) {
                // plain Legendre at the paper's nodes x_j = -1 + 2 j/P_s, Bonnet recurrence
                float xx = -1.f + 2.f * (float)j / (float)sg.P;
                float p0 = 1.f, p1 = xx;
                float cc = SMR(M.r_B + s * M.n1);
                if (M.n1 > 1) cc = fmaf(SMR(M.r_B + s * M.n1 + 1), xx, cc);
                for (int n = 1; n + 1 < M.n1; ++n) {
                    float p2 = ((2.f * n + 1.f) * xx * p1 - (float)n * p0) / (float)(n + 1);
                    cc = fmaf(SMR(M.r_B + s * M.n1 + n + 1), p2, cc);
                    p0 = p1; p1 = p2;
                }
                if (valid) a.model[i * M.P + sg.o + j] = cc * Sc[(size_t)(lo + j) * 32];
            }
        }
    }
}
