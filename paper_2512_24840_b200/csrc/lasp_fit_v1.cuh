// lasp_fit_v1.cuh -- the fused LASP-Adam fitting kernel for sm_100a.
//
// Mapping.  A CTA advances a GROUP of GS = 4 spectra in lockstep through every Adam step.  Threads
// own pixels: thread t owns the octet (8 consecutive padded pixels) t of the range being swept, for
// all 4 spectra, so that every spectrum-independent operand (an emulator coefficient C[k,j], a
// continuum basis value) is fetched once and used for 4 spectra x 8 pixels from registers, and every
// per-spectrum scalar (phi_k, b_n, a tap weight) is one broadcast LDS.128 for the 4 spectra.  The
// emulator output T and the adjoint a live in shared-memory rows (neighbour access by the stencils);
// flux/weight rows are re-read from global memory, where the few hundred groups in flight keep them
// L2-resident.  Sums over pixels (continuum moments, chi2, gradient) are reduced with a register
// transpose over warp shuffles (32 values x 32 lanes in 31 shuffles) and one shared-memory slot per
// warp; the continuum system is solved by one warp per spectrum (lanes = rows).
//
// Two variants of every kernel (template parameter STREAM):
//   resident  (STREAM = false): rows T and A of the whole longest segment stay in shared memory;
//   streaming (STREAM = true) : for spectra too long for that.  Rows T and A live in per-CTA global scratch
//       (L2-resident); each sweep of the CTA over nt*8 pixels first copies the window [jb - guard, jb + nt*8 + guard)
//       of the row the stencil needs into ONE shared-memory window buffer (coalesced 128-bit loads, halo re-read),
//       everything that touches only the thread's own octet goes to the global rows directly.
//
// Citations: Eq. n and P:n are /root/reference/PAPER.md; C.2-n the readings of SURVEY.md 8()
// (restated in DESIGN.md); a0..a9 the steps of SURVEY.md 8(a).
#pragma once
#include "lasp_common.cuh"

// All shared memory is addressed from this symbol so that the compiler emits LDS/STS (a pointer carried
// in a struct is generic and costs LD/ST with global-memory scoreboarding).
extern __shared__ float4 v1_smem4[];
#define V1SM ((float *)v1_smem4)

// 128-bit accesses to the shared rows go at a stride of two float4 between lanes (one octet per thread), which
// would be a two-way bank conflict; flipping the low index bit of every other group of eight float4 makes the
// eight lanes of a quarter-warp hit eight different 16-byte bank groups.  Applied to EVERY access of rows T / A.
#define SW4(q) ((q) ^ (((q) >> 3) & 1))

#define GS 4    // spectra per CTA group
#define OCT 8   // pixels per thread tile

struct V1Lay {
    int RL, GUARD;          // shared-memory row length and guard (floats); row index = jp - po + GUARD
    int NA;                 // largest number of 4-tap groups of a kernel
    int Kq;                 // K+2 rounded to 8: rows of the zero-padded coefficient table the loops sweep
    int n1r, nmomr, VR;     // n1 rounded to 4; moments rounded; reduction slots per warp (x GS)
    int NW;                 // warps per CTA
    int Hm;                 // support clamp (memory safety outside the prior box)
    int fastw;              // 1: v1_update_fast also prepares the next step's kernel weights (one uniform segment)
    int fastupd;            // 1: v1_update_fast applies (L <= 4, K + 2 <= 32, NW <= 12)
    int lfseg;              // 1: one factor slot per segment (0: one slot, re-factored every step when n_seg > 1)
    int nt8;                // pixels per sweep of the CTA (threads x 8): the streaming window holds nt8 + 2 GUARD
    int SL;                 // longest padded segment: row length of the per-pixel-kernel scratch planes
    // shared-memory offsets (floats)
    int oT, oA, oU, oM, oV, oX, oPHI, oGW, oGR, oTAP, oMOM, oRHS, oB, oRED, oLF, oQ, oSC, oEXP, oXP, oDPHI, oGSC, oEW, oNP, oHIST, oTM, total;
    int emax;               // largest exponent of the monomial table
};

struct V1Args {
    const float *Y, *W;   // staged flux and weight planes [B][Ppad] (halos and tails zero), split-octet layout
    const float *C1;      // emulator coefficients [Kq+16][Ppad], zero past K, split-octet layout
    float *CP;            // [cta][GS][Ppad] previous continuum c_prev (a5, refinement form)
    float *XJ;            // [cta][(1+NP)][GS][Ppad] rho and Jacobian columns (a9), may be null
    long long B;
    int ngroups;
    const float *init;
    int n_iter;
    float lr, b1, b2, eps, fd_h;
    float *params, *cont, *chi2, *err;
    int *status;
    const float *gparams;  // lasp_eval_grad, lasp_eval_model: physical parameters [B][NP]
    float *grad_u;
    const float *mcont;    // lasp_eval_model: plain-Legendre continuum coefficients [B][nc]
    float *model;          // lasp_eval_model: output [B][P]
    float *TG, *AG;        // streaming variant: per-CTA global rows [cta][GS][Ppad] of T and of S / a
    // Gram re-factorisation policy (lasp_fit_opts.refresh / .warm / .fd_fresh)
    int warm;              // the first `warm` steps always re-factor
    int refresh;           // >= 1: re-factor every `refresh`-th step;  0: adaptive (drift monitor, at most every 64th)
    int fdfresh;           // 1: re-factor in every finite-difference evaluation of the error estimate
    float drift_tol;       // adaptive: re-factor when (sum of |du|_inf since the last factor) x |du|_inf exceeds this
    // the paper's stopping rules (lasp_fit_opts.stop_window / .stop_tol): 0 = fixed number of steps
    int stop_window;       // W <= V1_WMAX
    float stop_tol;
    int *nsteps;           // [B] Adam updates applied per spectrum (may be null)
    // Clean strategy (lasp_fit_opts.clean_every / .clean_max): 0 = No Clean
    int clean_every, clean_max;
    float lm_lambda0;      // lasp_fit_opts.optimizer = 1 (the LM instantiation of the fit kernel): initial damping
    unsigned char *mask_out;   // [B][P] 1 where the pixel still takes part at the end (may be null)
    unsigned long long *dbg;   // optional per-phase cycle counters (LASP_TIMING=1), else null
    // per-pixel broadening kernels (linear grids, C.2-14): 1/s_j and s_j with V1_TPAD replicated entries on
    // both sides, and per-CTA scratch [3][GS][Ppad] for dS/dv, dS/dsigma*, 1/E0 (thread-private pixels)
    const float *IS, *SJ;
    float *DS;
    unsigned int *queue;   // work-queue counter for the fit kernel (zeroed before the launch), may be null
    unsigned long long *stats;   // [0] += Adam group-steps, [1] += those with a fresh Gram factor (may be null)
    const float4 *CF;      // coefficient table as tf32 [hi|lo] MMA fragments (null: FP32-pipe emulator)
    int ksteps;            // k-steps of 8 terms in CF (<= 16)
};
#define V1_TPAD 256
#define V1_WMAX 128    // largest stopping-rule window (loss history ring per spectrum)

struct V1Np {          // per-spectrum scalars of a per-pixel-kernel segment
    float v, sigstar, sigtot, hn, hbv, hcap;   // hn = -log2(e)/(2 sigma_tot^2); hbv = |v| + 5 sigma_tot (km/s)
    float an;                                  // sqrt(log2(e)/2) / sigma_tot: a_j = an s_j scales offsets so that the weight is 2^(-d^2)
};


// slots of the per-warp reduction area (each slot holds GS floats)
#define SLOT_MOM(L_, n) (n)
#define SLOT_RHS(L_, n) ((L_).nmomr + (n))
#define SLOT_Q(L_, k) ((L_).nmomr + (L_).n1r + (k))
#define SLOT_STAT(L_) ((L_).VR - 6)   // chi2, ngood, min c, dchi2/dv and dchi2/dsigma* of per-pixel-kernel segments

// per-spectrum scalars in shared memory: SC[idx][GS]
enum { SC_V = 0, SC_SIG, SC_CHI, SC_NGOOD, SC_CMIN, SC_GV, SC_GS, SC_FAIL, SC_PB1, SC_PB2, SC_N };   // SC_PB*: beta1^t, beta2^t

// 32 values per lane -> lane l returns the warp total of value l (31 shuffles)
__device__ __forceinline__ float xreduce32(float (&x)[32], int lane)
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
        const bool up = (lane & s) != 0;
#pragma unroll
        for (int i = 0; i < s; ++i) {
            float send = up ? x[i] : x[i + s];
            float keep = up ? x[i + s] : x[i];
            x[i] = keep + __shfl_xor_sync(FULL, send, s);
        }
    }
    return x[0];
}

// 16 values per lane -> lane l returns the total of value (l & 15) over the 16 lanes of its half-warp (15 shuffles)
__device__ __forceinline__ float xreduce16(float (&x)[16], int lane)
{
#pragma unroll
    for (int s = 8; s >= 1; s >>= 1) {
        const bool up = (lane & s) != 0;
#pragma unroll
        for (int i = 0; i < s; ++i) {
            float send = up ? x[i] : x[i + s];
            float keep = up ? x[i + s] : x[i];
            x[i] = keep + __shfl_xor_sync(FULL, send, s);
        }
    }
    return x[0];
}

__device__ __forceinline__ float warp_min_f(float v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(FULL, v, o));
    return v;
}

// Block-wide state.  It lives in static shared memory and the per-thread indices are recomputed from
// threadIdx where needed: a context struct passed by reference to the (deliberately not inlined) phase
// functions would sit in LOCAL memory, and with shared memory carved out to ~190 KB per SM the remaining L1
// is thrashed by the coefficient stream, so every such access costs an L2 round trip.
struct V1Block {
    ModelDev M;
    V1Lay L;
    V1Args A;
    long long spec[GS];   // clamped spectrum indices of the group
    float *cp;            // this CTA's c_prev scratch
    float *ds;            // this CTA's dS/dv, dS/dsigma*, 1/E0 scratch (per-pixel-kernel segments)
    float *tg, *ag;       // streaming variant: this CTA's global rows of T and of S / a, [GS][Ppad]
    int next;             // next group of this CTA (dynamic work queue)
    // re-factorisation monitor: read and written by thread 0 only, which publishes its decision in `momflag`
    float drift;          // sum of |du|_inf over the steps since the last fresh Gram factor
    int since;            // steps since the last fresh Gram factor
    int momflag;          // this evaluation re-factorises (written after its first barrier, read after its second)
    int stepmax;          // max over the group of |du|_inf of the last update, as the bits of a non-negative float (atomicMax)
    unsigned failmask;    // bit seg * GS + g: the last factorisation of that system was not positive definite
    unsigned int nfresh;  // fresh Adam steps of the current group (statistics)
    int t;                // Adam step counter of the current group: evaluations of the Adam loop begun so far (thread 0
                          // advances it in v1_begin_eval).  The loop state lives here, not in registers: a register kept
                          // across the (non-inlined) evaluation and update calls is spilled and reloaded from local memory
    // stopping rules, per spectrum of the group (written by lane 0 of warp g)
    int stop_rule[GS];    // 0 = still optimising; 2 / 3 = stopped by criterion (2) / (3) of P:169-171
    int nsteps[GS];       // Adam updates applied
    int rise[GS];         // consecutive increases of the loss so far
    float lprev[GS];      // loss at the previous step
    // Clean strategy (thread 0)
    int force;            // the next Adam evaluation re-factorises whatever the policy says
    int nclean;           // mask updates done for the current group
    // Levenberg-Marquardt (lane 0 of warp g)
    float lm_lambda[GS], lm_chi2[GS];
    int lm_acc[GS];       // the last trial step was accepted
};
__shared__ V1Block v1_blk;
static_assert(sizeof(V1Block) <= 1792, "the block state is part of the shared-memory budget that keeps two config-1 CTAs under the 196 KB carveout (setup_variant in lasp_gpu.cu)");
#define V1_TID ((int)threadIdx.x)
#define V1_LANE ((int)(threadIdx.x & 31))
#define V1_WARP ((int)(threadIdx.x >> 5))
#define V1_NT ((int)blockDim.x)

#define SMV(off, idx, g) V1SM[(off) + (idx) * GS + (g)]

// ------------------------------------------------------------------------------------------
// a1: de-normalise, emulator inputs, monomials (Eq. 1, C.2-18/19).  Warp g, spectrum g.
// ------------------------------------------------------------------------------------------
// Piecewise emulator (Eq. 1's f_1..f_5; reading R-15): phi_k <- omega_r(k)(x_0) phi_k and the product rule
// on d phi_k / d x_0, omega_r = up * down with the two ramps linear in x_0; the derivative of a ramp is its slope strictly
// inside it and 0 elsewhere (as oracle/lasp_oracle.c orc_blend_weight).  Warp g, after phi and dphi have been written.
__device__ __forceinline__ void v1_blend(int g)
{
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int K = M.K, nl = M.L;
    const uint8_t *tm = (const uint8_t *)(V1SM + L.oTM);
    const float x0 = SMV(L.oX, 0, g);
    float w[LASP_MAX_MODELS], dw[LASP_MAX_MODELS];
#pragma unroll
    for (int r = 0; r < LASP_MAX_MODELS; ++r) {
        float up = 1.f, dup = 0.f, dn = 1.f, ddn = 0.f;
        if (r < M.n_models) {
            if (M.bl_ui[r] != 0.f) {
                const float t = (x0 - M.bl_u0[r]) * M.bl_ui[r];
                if (t <= 0.f) up = 0.f; else if (t < 1.f) { up = t; dup = M.bl_ui[r]; }
            }
            if (M.bl_di[r] != 0.f) {
                const float t = (M.bl_d1[r] - x0) * M.bl_di[r];
                if (t <= 0.f) dn = 0.f; else if (t < 1.f) { dn = t; ddn = -M.bl_di[r]; }
            }
        }
        w[r] = up * dn;
        dw[r] = dup * dn + up * ddn;
    }
    for (int k = V1_LANE; k < K; k += 32) {
        const int r = tm[k];
        float wr = w[0], dwr = dw[0];
#pragma unroll
        for (int q = 1; q < LASP_MAX_MODELS; ++q)
            if (r == q) { wr = w[q]; dwr = dw[q]; }
        const float ph = SMV(L.oPHI, k, g);
        SMV(L.oPHI, k, g) = wr * ph;
        for (int l = 0; l < nl; ++l) {
            const float d = SMV(L.oDPHI, l * K + k, g);
            SMV(L.oDPHI, l * K + k, g) = wr * d + (l == 0 ? dwr * ph : 0.f);
        }
    }
    __syncwarp();
}

__device__ __noinline__ void v1_param_setup(int g)
{
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int nl = M.L, K = M.K, ne = L.emax + 1;
    const uint8_t *ex = (const uint8_t *)(V1SM + L.oEXP);
    for (int p = V1_LANE; p < M.NP; p += 32) {
        const float u = SMV(L.oU, p, g);
        const float half = (M.hi[p] - M.lo[p]) * 0.5f;
        const float th = M.lo[p] + (u + 1.f) * half;
        float gsc = half;                       // d theta / d u
        if (p < nl) {
            SMV(L.oX, p, g) = label_x(M, p, th);
            gsc *= M.label_log10[p] ? M.emu_a[p] / (th * 2.302585093f) : M.emu_a[p];   // d x / d theta (C.1)
        } else
            SMV(L.oSC, p == nl ? SC_V : SC_SIG, g) = th;
        SMV(L.oGSC, p, g) = gsc;
    }
    __syncwarp();
    // powers x_l^e, e = 0..emax: XP[e*nl + l]
    for (int i = V1_LANE; i < nl * ne; i += 32) {
        const int e = i / nl, l = i - e * nl;
        const float x = SMV(L.oX, l, g);
        float pw = 1.f;
        for (int q = 0; q < e; ++q) pw *= x;
        SMV(L.oXP, i, g) = pw;
    }
    __syncwarp();
    // phi_k = prod_l x_l^e_kl and d phi_k / d x_l = e_kl x_l^(e_kl - 1) prod_{l2 != l} x_l2^e_kl2  (Eq. 1)
    if (nl <= 4) {
        // up to four labels: the exponents of term k come packed in one word (v1_init_block), so every table read of
        // a term issues at once instead of as a chain of byte loads (this phase is one warp's latency, nothing else)
        const unsigned *exw = (const unsigned *)(V1SM + L.oEXP);
        const float *xp = V1SM + L.oXP + g;
        for (int k = V1_LANE; k < K; k += 32) {
            const unsigned w = exw[k];
            float pe[4], pm[4];
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                const int e = (w >> (8 * l)) & 255;
                pe[l] = l < nl ? xp[(e * nl + l) * GS] : 1.f;
                pm[l] = (l < nl && e > 0) ? (float)e * xp[((e - 1) * nl + l) * GS] : 0.f;
            }
            float ph = 1.f;
#pragma unroll
            for (int l = 0; l < 4; ++l) ph *= pe[l];
            SMV(L.oPHI, k, g) = ph;
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                float d = pm[l];
#pragma unroll
                for (int l2 = 0; l2 < 4; ++l2)
                    if (l2 != l) d *= pe[l2];
                if (l < nl) SMV(L.oDPHI, l * K + k, g) = d;
            }
        }
        __syncwarp();
        if (M.n_models) v1_blend(g);
        return;
    }
    for (int k = V1_LANE; k < K; k += 32) {
        float p = 1.f;
        for (int l = 0; l < nl; ++l) p *= SMV(L.oXP, ex[k * nl + l] * nl + l, g);
        SMV(L.oPHI, k, g) = p;
        for (int l = 0; l < nl; ++l) {
            const int el = ex[k * nl + l];
            float d = 0.f;
            if (el > 0) {
                d = (float)el * SMV(L.oXP, (el - 1) * nl + l, g);
                for (int l2 = 0; l2 < nl; ++l2)
                    if (l2 != l) d *= SMV(L.oXP, ex[k * nl + l2] * nl + l2, g);
            }
            SMV(L.oDPHI, l * K + k, g) = d;
        }
    }
    __syncwarp();
    if (M.n_models) v1_blend(g);
}

// ------------------------------------------------------------------------------------------
// a3: kernel weights of a uniform (log-grid) segment (Eq. 5; C.2-9/10/15), in groups of
// four taps: group a holds taps k = 4a-3 .. 4a, a = a_lo .. a_lo+na-1, zero outside |k| <= H.
//   GW [g][a][4]       forward kernel g_k
//   GR [j][g][a][4]    reversed kernels for the adjoint pass: j=0: g_{-k}; j=1: d g_{-k}/dv;
//                      j=2: d g_{-k}/d sigma* (chain factors of C.1 folded in)
// ------------------------------------------------------------------------------------------
// Uniform segment, given (v, sigma*).  Lanes = table entries: entry idx is tap k = 4 (a_lo + idx/4) - 3 + idx%4, and the
// lane evaluates the exponential of its forward tap k and of its reversed tap -k itself, so nothing is exchanged
// between lanes except the three sums (this runs on one warp between two phases of all: its latency is the cost).
__device__ __forceinline__ void v1_weights_uniform(const SegDev &sg, int g, float v, float sigstar)
{
    const V1Lay &L = v1_blk.L;
    const float sig_inst = sg.sig_inst, inv_s = sg.inv_s;
    const int hcap = sg.halo - 18;
    float *gw = V1SM + L.oGW + g * L.NA * 4;
    float *gr = V1SM + L.oGR + g * L.NA * 4;
    const int rs = GS * L.NA * 4;
    const float sigtot = sqrtf(sigstar * sigstar + sig_inst * sig_inst);
    const float mu = v * inv_s, s = sigtot * inv_s;
    int H = (int)ceilf(fabsf(mu) + 5.f * s);
    H = min(max(H, 0), hcap);   // memory safety outside the prior box (halo >= Hmax + 18)
    const float i2 = 0.5f / (s * s);
    const int a_lo = -(H / 4), na = (H + 3) / 4 - a_lo + 1;
    const float is2 = 2.f * i2;                        // 1/sigma^2 (pixels)
    const float cmu = is2 * inv_s;                     // dS/dv      = (1/s) sum dg/dmu T
    const float csig = is2 * sqrtf(is2) * (sigstar / sigtot) * inv_s;
    if (na * 4 <= 64) {
        // the usual case (H <= 29): a lane owns at most two table entries; the forward tap k and the reversed tap -k of
        // an entry are exponentiated ONCE, kept in registers over the warp sums and scaled afterwards (this runs on one
        // warp between two phases of all: every dependent operation is latency on the step's critical path)
        float ef[2], er[2], df[2], dr[2];
        float sum = 0.f, s1 = 0.f, s2 = 0.f;
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int idx = it * 32 + V1_LANE;
            const int k = 4 * (a_lo + (idx >> 2)) - 3 + (idx & 3);
            const bool in = idx < na * 4 && k >= -H && k <= H;
            df[it] = (float)k - mu; dr[it] = (float)(-k) - mu;
            ef[it] = in ? expf(-df[it] * df[it] * i2) : 0.f;
            er[it] = in ? expf(-dr[it] * dr[it] * i2) : 0.f;
            sum += ef[it]; s1 = fmaf(ef[it], df[it], s1); s2 = fmaf(ef[it] * df[it], df[it], s2);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sum += __shfl_xor_sync(FULL, sum, o); s1 += __shfl_xor_sync(FULL, s1, o); s2 += __shfl_xor_sync(FULL, s2, o);
        }
        const float inv = 1.f / sum;
        const float e1n = s1 * inv, e2n = s2 * inv;       // kbar - mu ; second moment about mu
#pragma unroll
        for (int it = 0; it < 2; ++it) {
            const int idx = it * 32 + V1_LANE;
            if (idx < na * 4) {
                gw[idx] = ef[it] * inv;
                const float gg = er[it] * inv;
                gr[idx] = gg;
                gr[rs + idx] = gg * (dr[it] - e1n) * cmu;
                gr[2 * rs + idx] = gg * (dr[it] * dr[it] - e2n) * csig;
            }
        }
    } else {
        float sum = 0.f, s1 = 0.f, s2 = 0.f;
        for (int i0 = 0; i0 < na * 4; i0 += 32) {
            const int idx = i0 + V1_LANE;
            const int k = 4 * (a_lo + (idx >> 2)) - 3 + (idx & 3);
            const float d = (float)k - mu;
            const float e = (idx < na * 4 && k >= -H && k <= H) ? expf(-d * d * i2) : 0.f;
            sum += e; s1 = fmaf(e, d, s1); s2 = fmaf(e * d, d, s2);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            sum += __shfl_xor_sync(FULL, sum, o); s1 += __shfl_xor_sync(FULL, s1, o); s2 += __shfl_xor_sync(FULL, s2, o);
        }
        const float inv = 1.f / sum;
        const float e1n = s1 * inv, e2n = s2 * inv;       // kbar - mu ; second moment about mu
        for (int i0 = 0; i0 < na * 4; i0 += 32) {
            const int idx = i0 + V1_LANE;
            if (idx < na * 4) {
                const int k = 4 * (a_lo + (idx >> 2)) - 3 + (idx & 3);
                const bool in = (k >= -H) && (k <= H);
                const float df = (float)k - mu, dr = (float)(-k) - mu;
                gw[idx] = in ? expf(-df * df * i2) * inv : 0.f;
                const float gg = in ? expf(-dr * dr * i2) * inv : 0.f;
                gr[idx] = gg;
                gr[rs + idx] = gg * (dr - e1n) * cmu;
                gr[2 * rs + idx] = gg * (dr * dr - e2n) * csig;
            }
        }
    }
    if (V1_LANE == 0) {
        int *tap = (int *)(V1SM + L.oTAP);
        tap[g * 2] = a_lo; tap[g * 2 + 1] = na;
    }
    __syncwarp();
}

__device__ __noinline__ void v1_setup_weights(const SegDev &sg, int g)
{
    const V1Lay &L = v1_blk.L;
    const float v = SMV(L.oSC, SC_V, g), sigstar = SMV(L.oSC, SC_SIG, g);
    if (!sg.uniform) {
        // per-pixel kernels: only the spectrum's scalars and the segment-wide reach (sg.inv_s = largest 1/s_j)
        const float sigtot = sqrtf(sigstar * sigstar + sg.sig_inst * sg.sig_inst);
        if (V1_LANE == 0) {
            V1Np *np = (V1Np *)(V1SM + L.oNP) + g;
            np->v = v; np->sigstar = sigstar; np->sigtot = sigtot;
            np->hn = -0.72134752044f / (sigtot * sigtot);        // -log2(e)/2 / sigma_tot^2
            np->an = 0.84932180029f / sigtot;
            np->hbv = fabsf(v) + 5.f * sigtot;
            np->hcap = (float)(sg.halo - 18);
            const int H = (int)ceilf(fminf(np->hbv * sg.inv_s, np->hcap));
            int *tap = (int *)(V1SM + L.oTAP);
            tap[g * 2] = -(H / 4); tap[g * 2 + 1] = (H + 3) / 4 + (H / 4) + 1;
        }
        __syncwarp();
        return;
    }
    v1_weights_uniform(sg, g, v, sigstar);
}

// ------------------------------------------------------------------------------------------
// a4: sliding-window stencil for one octet and NK kernels sharing the window (Eq. 5).
//   out[n][i] = sum_k w_n[k] row[j0 + i - k],  taps in groups a: k = 4a-3..4a.
// row4 is the float4 view of a shared-memory row indexed by (padded pixel)/4; for group a the window
// is row[j0-4a .. j0-4a+11]: one new LDS.128 per group feeds 32*NK FMAs.
// ------------------------------------------------------------------------------------------
template <int NK>
__device__ __forceinline__ void v1_stencil_octet(const float4 *__restrict__ row4, int j0, int a_lo, int na,
                                                 const float4 *__restrict__ w0, int wstride4,
                                                 float (&acc)[NK][OCT])
{
#pragma unroll
    for (int n = 0; n < NK; ++n)
#pragma unroll
        for (int i = 0; i < OCT; ++i) acc[n][i] = 0.f;
    const int q = (j0 >> 2) - a_lo;
    float4 qb = row4[SW4(q + 1)], qc = row4[SW4(q + 2)];
#pragma unroll 1
    for (int ai = 0; ai < na; ++ai) {
        const float4 qa = row4[SW4(q - ai)];
        const float Wd[12] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y, qb.z, qb.w, qc.x, qc.y, qc.z, qc.w};
#pragma unroll
        for (int n = 0; n < NK; ++n) {
            const float4 w = w0[n * wstride4 + ai];
#pragma unroll
            for (int i = 0; i < OCT; ++i) {
                float s = acc[n][i];
                s = fmaf(w.x, Wd[i + 3], s);
                s = fmaf(w.y, Wd[i + 2], s);
                s = fmaf(w.z, Wd[i + 1], s);
                s = fmaf(w.w, Wd[i], s);
                acc[n][i] = s;
            }
        }
        qc = qb; qb = qa;
    }
}

// shared-memory row 0 of buffer `off` as a float pointer indexed by padded pixel jp (row g is + g * RL); `org` is the
// first padded pixel of the segment (resident rows) or of the sweep (streaming window)
__device__ __forceinline__ float *v1_rowp(int off, int org)
{
    return V1SM + off + v1_blk.L.GUARD - org;
}

// coefficient-table stream.  TNA (the steady-state step of the resident two-CTA shape, v1_step_hot): read through L2 without
// taking lines in the small L1, which the flux / weight / c_prev planes of the two resident CTAs re-use between the forward
// and the residual phase (config 1: +0.6 %).  Elsewhere the plain read-only path: with one CTA per SM or the streaming
// variant's global rows the same hint costs 2-5 % (config 4, shape S; measured).
template <bool TNA>
__device__ __forceinline__ float4 v1_ld_table(const float4 *p)
{
    if (!TNA) return __ldg(p);
    float4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(p));
    return v;
}

// streaming variant: copy padded pixels [jb - GUARD, jb + nt8 + GUARD) of the GS global rows `src` ([GS][Ppad], plain
// layout) into the window buffer with the SW4 addressing of the resident rows: 128-bit coalesced loads, the halo of
// 2 GUARD pixels is re-read by the neighbouring sweep.  Pixels outside [0, Ppad) read as zero.  Callers bracket it
// with __syncthreads (the rows were written by other threads of this CTA; __ldcg reads them at L2).
__device__ __forceinline__ void v1_window_load(const float *__restrict__ src, int jb)
{
    const int G = v1_blk.L.GUARD, RL = v1_blk.L.RL, P4 = v1_blk.M.Ppad >> 2;
    const int n4 = (v1_blk.L.nt8 + 2 * G) >> 2, q0 = (jb - G) >> 2;
#pragma unroll 1
    for (int g = 0; g < GS; ++g) {
        float4 *row4 = (float4 *)(V1SM + v1_blk.L.oT + g * RL + G - jb);
        const float4 *s4 = (const float4 *)(src + (size_t)g * v1_blk.M.Ppad);
        for (int i = V1_TID; i < n4; i += V1_NT) {
            const int q = q0 + i;
            float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
            if (q >= 0 && q < P4) v = __ldcg(s4 + q);
            row4[SW4(q)] = v;
        }
    }
}

// own-octet access to a row: shared memory (resident) or the CTA's global row (streaming), two float4
template <bool STREAM>
__device__ __forceinline__ void v1_oct_load(const float *rowsm, const float *rowgl, int g, int j0, float (&x)[OCT])
{
    float4 a, b;
    if (STREAM) {
        const float4 *p = (const float4 *)(rowgl + (size_t)g * v1_blk.M.Ppad + j0);
        a = __ldcg(p); b = __ldcg(p + 1);
    } else {
        const float4 *p = (const float4 *)(rowsm + g * v1_blk.L.RL);
        a = p[SW4(j0 >> 2)]; b = p[SW4((j0 >> 2) + 1)];
    }
    x[0] = a.x; x[1] = a.y; x[2] = a.z; x[3] = a.w; x[4] = b.x; x[5] = b.y; x[6] = b.z; x[7] = b.w;
}
template <bool STREAM>
__device__ __forceinline__ void v1_oct_store(float *rowsm, float *rowgl, int g, int j0, const float (&x)[OCT])
{
    const float4 a = make_float4(x[0], x[1], x[2], x[3]), b = make_float4(x[4], x[5], x[6], x[7]);
    if (STREAM) {
        float4 *p = (float4 *)(rowgl + (size_t)g * v1_blk.M.Ppad + j0);
        p[0] = a; p[1] = b;
    } else {
        float4 *p = (float4 *)(rowsm + g * v1_blk.L.RL);
        p[SW4(j0 >> 2)] = a; p[SW4((j0 >> 2) + 1)] = b;
    }
}

// ------------------------------------------------------------------------------------------
// a3 + a4 on a linear grid (C.2-14): every pixel j has its own kernel, mu_j = v/s_j, sigma_j = sigma_tot/s_j,
// H_j = ceil(|mu_j| + 5 sigma_j), e_jk = exp(-(k-mu_j)^2/(2 sigma_j^2)) on |k| <= H_j, normalised per pixel.
// Weights are generated on the fly (one ex2 per pixel and tap); |k| <= ceil(x)  <=>  |k| - 1 < x.
//   forward:  S_j = A0/E0, and dS_j/dv, dS_j/dsigma* from the first and second moments of e (C.1)
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float v1_ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// One group of four taps k = k0 .. k0 + 3 of the forward stencil for the thread's eight pixels.  The weight is
// e = 2^(-d^2) with d = (k - mu_i) a_i, a_i = sqrt(log2(e) / 2) / sigma_i (one FFMA, one FMUL, one ex2); the kernel moments
// are accumulated in the scaled offset d and rescaled once per pixel.  MASK = false: every tap of the group lies inside the
// support of every pixel of the (active part of the) warp, so the support test is left out.
template <bool MASK>
__device__ __forceinline__ void v1_np_taps_forward(const float (&Wd)[12], int k0, const float (&aa)[OCT], const float (&bb)[OCT],
                                                   const float (&hb)[OCT], float (&A0)[OCT], float (&A1)[OCT], float (&A2)[OCT],
                                                   float (&E0)[OCT], float (&E1)[OCT], float (&E2)[OCT])
{
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        const float kf = (float)(k0 + r);
        const float ak1 = fabsf(kf) - 1.f;
#pragma unroll
        for (int i = 0; i < OCT; ++i) {
            const float d = fmaf(kf, aa[i], -bb[i]);
            float e = v1_ex2(d * -d);
            if (MASK) e = (ak1 < hb[i]) ? e : 0.f;
            const float Tv = Wd[i + 3 - r];
            const float ed = e * d, edd = ed * d;
            E0[i] += e; E1[i] += ed; E2[i] += edd;
            A0[i] = fmaf(e, Tv, A0[i]); A1[i] = fmaf(ed, Tv, A1[i]); A2[i] = fmaf(edd, Tv, A2[i]);
        }
    }
}

__device__ __forceinline__ void v1_np_forward_octet(const float4 *__restrict__ row4, int j0, const V1Np &p,
                                                    const float (&is)[OCT], const float (&sj)[OCT],
                                                    float (&S)[OCT], float (&DSV)[OCT], float (&DSS)[OCT],
                                                    float (&EI)[OCT])
{
    float aa[OCT], bb[OCT], hb[OCT];
    float A0[OCT], A1[OCT], A2[OCT], E0[OCT], E1[OCT], E2[OCT];
    float hmx = 0.f, hmn = 3.0e38f;
#pragma unroll
    for (int i = 0; i < OCT; ++i) {
        aa[i] = p.an * sj[i];
        bb[i] = p.v * is[i] * aa[i];
        hb[i] = fminf(p.hbv * is[i], p.hcap);
        hmx = fmaxf(hmx, hb[i]);
        hmn = fminf(hmn, hb[i]);
        A0[i] = A1[i] = A2[i] = E0[i] = E1[i] = E2[i] = 0.f;
    }
    const int H = (int)ceilf(hmx);
    const int a_lo = -(H / 4), na = (H + 3) / 4 - a_lo + 1;
    const int q = (j0 >> 2) - a_lo;
    float4 qb = row4[SW4(q + 1)], qc = row4[SW4(q + 2)];
    for (int ai = 0; ai < na; ++ai) {
        const float4 qa = row4[SW4(q - ai)];
        const float Wd[12] = {qa.x, qa.y, qa.z, qa.w, qb.x, qb.y, qb.z, qb.w, qc.x, qc.y, qc.z, qc.w};
        const int k0 = 4 * (a_lo + ai) - 3;
        const bool inside = (float)(max(abs(k0), abs(k0 + 3)) - 1) < hmn;   // |k| <= ceil(x)  <=>  |k| - 1 < x
        if (__all_sync(__activemask(), inside)) v1_np_taps_forward<false>(Wd, k0, aa, bb, hb, A0, A1, A2, E0, E1, E2);
        else v1_np_taps_forward<true>(Wd, k0, aa, bb, hb, A0, A1, A2, E0, E1, E2);
        qc = qb; qb = qa;
    }
    const float rs = p.sigstar / p.sigtot;
#pragma unroll
    for (int i = 0; i < OCT; ++i) {
        const float inv = 1.f / E0[i];
        S[i] = A0[i] * inv;
        EI[i] = inv;
        // moments in the scaled offset: A1 = a A1', A2 = a^2 A2' (E likewise) and 1/sigma_j^2 = 2 ln2 a^2, so both
        // derivatives come out as (.)' times a constant times a
        const float smu = (A1[i] * inv - E1[i] * inv * S[i]) * (1.3862943611f * aa[i]);
        const float ssg = (A2[i] * inv - E2[i] * inv * S[i]) * (1.6322368749f * aa[i]);
        DSV[i] = smu * is[i];
        DSS[i] = ssg * rs * is[i];
    }
}

// adjoint:  t_i = sum_j a'_j e_{j,j-i},  a' = a/E0 (row A).  With k' = j... the window over SOURCE pixels slides
// like the forward one; each source carries its own (mu, sigma, H).  istab/sjtab point at padded pixel 0.
template <bool MASK>
__device__ __forceinline__ void v1_np_taps_adjoint(const float (&Wd)[12], int k0, const float (&aa)[12], const float (&bb)[12],
                                                   const float (&hb)[12], float (&t)[OCT])
{
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        // target i reads source m = i+3-r at lag k' = k0 + r: source j = i - k' contributes e_{j, k = j - i = -k'}
        const float kf = (float)(k0 + r);
        const float ak1 = fabsf(kf) - 1.f;
#pragma unroll
        for (int i = 0; i < OCT; ++i) {
            const int m = i + 3 - r;
            const float d = fmaf(-kf, aa[m], -bb[m]);
            float e = v1_ex2(d * -d);
            if (MASK) e = (ak1 < hb[m]) ? e : 0.f;
            t[i] = fmaf(Wd[m], e, t[i]);
        }
    }
}

__device__ __forceinline__ void v1_np_adjoint_octet(const float4 *__restrict__ row4, int j0, int H, const V1Np &p,
                                                    const float *__restrict__ istab, const float *__restrict__ sjtab,
                                                    float (&t)[OCT])
{
#pragma unroll
    for (int i = 0; i < OCT; ++i) t[i] = 0.f;
    const int a_lo = -(H / 4), na = (H + 3) / 4 - a_lo + 1;
    for (int ai = 0; ai < na; ++ai) {
        const int a = a_lo + ai;
        const int wb = j0 - 4 * a;                         // window base: sources wb .. wb+11
        const int q = wb >> 2;
        const float4 w0 = row4[SW4(q)], w1 = row4[SW4(q + 1)], w2 = row4[SW4(q + 2)];
        const float Wd[12] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w, w2.x, w2.y, w2.z, w2.w};
        float aa[12], bb[12], hb[12];
        float hmn = 3.0e38f;
#pragma unroll
        for (int m4 = 0; m4 < 3; ++m4) {
            const float4 i4 = __ldg((const float4 *)(istab + wb) + m4), s4 = __ldg((const float4 *)(sjtab + wb) + m4);
            const float ii[4] = {i4.x, i4.y, i4.z, i4.w}, ss[4] = {s4.x, s4.y, s4.z, s4.w};
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                aa[m4 * 4 + c] = p.an * ss[c];
                bb[m4 * 4 + c] = p.v * ii[c] * aa[m4 * 4 + c];
                hb[m4 * 4 + c] = fminf(p.hbv * ii[c], p.hcap);
                hmn = fminf(hmn, hb[m4 * 4 + c]);
            }
        }
        const int k0 = 4 * a - 3;
        const bool inside = (float)(max(abs(k0), abs(k0 + 3)) - 1) < hmn;
        if (__all_sync(__activemask(), inside)) v1_np_taps_adjoint<false>(Wd, k0, aa, bb, hb, t);
        else v1_np_taps_adjoint<true>(Wd, k0, aa, bb, hb, t);
    }
}

// Per-pixel kernels (linear grids): the stencil pass of spectra [g0, g1) for the octet at j0: S -> row A, and its two
// kernel-parameter derivatives and 1/E0 -> the scratch planes [3][GS][SL] (segment-relative, split-octet, L2-resident).
template <bool STREAM>
__device__ __forceinline__ void v1_np_forward_pass(const SegDev &sg, const float *rowT, float *rowA, int j0, int g0, int g1)
{
    const V1Lay &L = v1_blk.L;
    const float *ISg = v1_blk.A.IS + V1_TPAD, *SJg = v1_blk.A.SJ + V1_TPAD;
    float *dsg = v1_blk.ds;
    float isv[OCT], sjv[OCT];
    {
        const float4 a0 = __ldg((const float4 *)(ISg + j0)), a1 = __ldg((const float4 *)(ISg + j0) + 1);
        const float4 b0 = __ldg((const float4 *)(SJg + j0)), b1 = __ldg((const float4 *)(SJg + j0) + 1);
        isv[0] = a0.x; isv[1] = a0.y; isv[2] = a0.z; isv[3] = a0.w; isv[4] = a1.x; isv[5] = a1.y; isv[6] = a1.z; isv[7] = a1.w;
        sjv[0] = b0.x; sjv[1] = b0.y; sjv[2] = b0.z; sjv[3] = b0.w; sjv[4] = b1.x; sjv[5] = b1.y; sjv[6] = b1.z; sjv[7] = b1.w;
    }
    for (int g = g0; g < g1; ++g) {
        float Sg[OCT], DV[OCT], DG[OCT], EI[OCT];
        const V1Np np = ((const V1Np *)(V1SM + L.oNP))[g];
        v1_np_forward_octet((const float4 *)(rowT + g * L.RL), j0, np, isv, sjv, Sg, DV, DG, EI);
        v1_oct_store<STREAM>(rowA, v1_blk.ag, g, j0, Sg);
        float4 *d4 = (float4 *)(dsg + g * L.SL + ((j0 - sg.po) >> 1));
        const int S8 = L.SL >> 3, SP = GS * (L.SL >> 2);
        d4[0] = make_float4(DV[0], DV[1], DV[2], DV[3]); d4[S8] = make_float4(DV[4], DV[5], DV[6], DV[7]);
        d4 += SP;
        d4[0] = make_float4(DG[0], DG[1], DG[2], DG[3]); d4[S8] = make_float4(DG[4], DG[5], DG[6], DG[7]);
        d4 += SP;
        d4[0] = make_float4(EI[0], EI[1], EI[2], EI[3]); d4[S8] = make_float4(EI[4], EI[5], EI[6], EI[7]);
    }
}

// padded pixel range [lo,hi) on which T is needed by the forward stencils of the group's fitted octets
// (group a reads row[j0-4a .. j0-4a+11]); the adjoint pass runs on the same range.  Kept tight: config 1
// has 188 fitted octets and 192 threads, so 16 pixels of reach on each side still fit one sweep.
__device__ __forceinline__ void v1_group_range(const SegDev &sg, int &lo, int &hi)
{
    const int *tap = (const int *)(V1SM + v1_blk.L.oTAP);
    int rl = 0, rh = 0;
#pragma unroll
    for (int g = 0; g < GS; ++g) {
        const int a_lo = tap[2 * g], na = tap[2 * g + 1];
        rl = max(rl, 4 * (a_lo + na - 1));
        rh = max(rh, -4 * a_lo + 4);
    }
    lo = sg.fit_lo - (rl + OCT - 1) / OCT * OCT;
    hi = sg.fit_hi + (rh + OCT - 1) / OCT * OCT;
}


// T range of a phase: the fitted octets plus the group's reach (full = 0), or the whole segment plus the reach, inside
// the halo (full = 1: lasp_eval_model).  The phases take the segment INDEX and derive everything from the block state:
// a reference or a range passed in would have to be kept alive across the (non-inlined) phase calls by the caller,
// i.e. spilled to local memory and reloaded behind every call.
__device__ __forceinline__ void v1_phase_range(const SegDev &sg, int full, int &lo, int &hi)
{
    if (!full) { v1_group_range(sg, lo, hi); return; }
    const int *tap = (const int *)(V1SM + v1_blk.L.oTAP);
    int rl = 0, rh = 0;
#pragma unroll
    for (int q = 0; q < GS; ++q) {
        rl = max(rl, 4 * (tap[2 * q] + tap[2 * q + 1] - 1));
        rh = max(rh, -4 * tap[2 * q] + 4);
    }
    const int seg_lo = sg.po + sg.halo, seg_hi = seg_lo + (sg.P + OCT - 1) / OCT * OCT;
    lo = max(sg.po, seg_lo - (rl + OCT - 1) / OCT * OCT);
    hi = min(sg.po + sg.len, seg_hi + (rh + OCT - 1) / OCT * OCT);
}

// ------------------------------------------------------------------------------------------
// a2: T_j = sum_k phi_k C[k,j] over the padded range [lo,hi) -> shared row T (Eq. 1)
// ------------------------------------------------------------------------------------------
template <bool STREAM, bool TNA = false>
__device__ __noinline__ void v1_phase_emulator(int s_, int full)
{
    const SegDev &sg = v1_blk.M.seg[s_];
    int lo, hi;
    v1_phase_range(sg, full, lo, hi);
    // everything the loop needs is copied to registers first: the model lives in shared memory, and after
    // any shared-memory store the compiler would otherwise have to re-read it
    const float4 *phi4 = (const float4 *)(V1SM + v1_blk.L.oPHI);
    const int P4 = v1_blk.M.Ppad >> 2, P8 = v1_blk.M.Ppad >> 3, Kq = v1_blk.L.Kq, nt8 = V1_NT * OCT;
    const float *Cg = v1_blk.A.C1;
    float *rowT = v1_rowp(v1_blk.L.oT, sg.po);
    float *tg = v1_blk.tg;
    for (int j0 = lo + V1_TID * OCT; j0 < hi; j0 += nt8) {
        float acc[GS][OCT];
#pragma unroll
        for (int g = 0; g < GS; ++g)
#pragma unroll
            for (int i = 0; i < OCT; ++i) acc[g][i] = 0.f;
        // C[k, j0..j0+7] streams from L2/L1 in batches of 4 terms, the next batch in flight while this one is
        // multiplied (two register buffers).  The table has Kq = K+2 rounded to 8 rows plus 8 more, all zero
        // past K (and phi is zero there), so the loop has no bounds tests.
        const float4 *c4 = (const float4 *)Cg + (j0 >> 3);
        float4 bufA[8], bufB[8];
        auto load4 = [&](int k0, float4 (&buf)[8]) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                buf[2 * u] = v1_ld_table<TNA>(c4 + (k0 + u) * P4);
                buf[2 * u + 1] = v1_ld_table<TNA>(c4 + (k0 + u) * P4 + P8);
            }
        };
        auto mul4 = [&](int k0, const float4 (&buf)[8]) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const float4 ph = phi4[k0 + u];
                const float4 ca = buf[2 * u], cb = buf[2 * u + 1];
                const float cc[OCT] = {ca.x, ca.y, ca.z, ca.w, cb.x, cb.y, cb.z, cb.w};
                const float pg[GS] = {ph.x, ph.y, ph.z, ph.w};
#pragma unroll
                for (int g = 0; g < GS; ++g)
#pragma unroll
                    for (int i = 0; i < OCT; ++i) acc[g][i] = fmaf(pg[g], cc[i], acc[g][i]);
            }
        };
        // three buffers: two batches (16 x 128-bit loads per thread) are in flight while one is multiplied --
        // an L2 hit costs ~1000 cycles under this load, a batch of FMAs ~150
        float4 bufC[8];
        load4(0, bufA);
        load4(4, bufB);
        for (int k0 = 0; k0 < Kq; k0 += 12) {
            load4(k0 + 8, bufC);
            mul4(k0, bufA);
            if (k0 + 4 >= Kq) break;
            load4(k0 + 12, bufA);
            mul4(k0 + 4, bufB);
            if (k0 + 8 >= Kq) break;
            load4(k0 + 16, bufB);
            mul4(k0 + 8, bufC);
        }
#pragma unroll
        for (int g = 0; g < GS; ++g) v1_oct_store<STREAM>(rowT, tg, g, j0, acc[g]);
    }
}

// ------------------------------------------------------------------------------------------
// a2 on the tensor pipe: the same contraction as mma.sync.m16n8k8 TF32 with both operands split in two
// (x = hi + lo, each a tf32 number): rows = 16 pixels, k = 8 terms, and the 8 columns carry [phi_hi | phi_lo] of the
// GS = 4 spectra, so that two MMAs (table hi, table lo) form all four partial products in FP32 accumulators.
// Warp w owns pixels [lo + 256 w, lo + 256 w + 256) of every sweep; the table comes pre-split in fragment order
// (lasp_gpu.cu), one LDG.128 per (octet, k-step).  Models with up to 128 terms (NCH <= 4).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float v1_tf32(float x)
{
    unsigned r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}

__device__ __forceinline__ void v1_mma_tf32(float (&d)[4], float a0, float a1, float a2, float a3, float b0, float b1)
{
    asm("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                 : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
                 : "r"(__float_as_uint(a0)), "r"(__float_as_uint(a1)), "r"(__float_as_uint(a2)), "r"(__float_as_uint(a3)),
                   "r"(__float_as_uint(b0)), "r"(__float_as_uint(b1)));
}

// NCH = number of chunks of four k-steps (32 terms) whose B fragments are held in registers: K <= 32 * NCH
template <int NCH>
__device__ __noinline__ void v1_phase_emulator_mma(int s_, int full)
{
    const SegDev &sg = v1_blk.M.seg[s_];
    int lo, hi;
    v1_phase_range(sg, full, lo, hi);
    const int lane = V1_LANE, gid = lane >> 2, tig = lane & 3, K = v1_blk.M.K, ks = v1_blk.A.ksteps;
    const int RL = v1_blk.L.RL, sweep = v1_blk.L.NW * 256;
    const float4 *CF = v1_blk.A.CF + lane;
    float *rowT = V1SM + v1_blk.L.oT + v1_blk.L.GUARD - sg.po;
    const float *phi = V1SM + v1_blk.L.oPHI + (gid & 3);
    // B fragments (k = term, n = column): columns 0..3 carry phi_hi of spectrum n, columns 4..7 phi_lo of spectrum n - 4
    float b0[4 * NCH], b1[4 * NCH];
#pragma unroll
    for (int s = 0; s < 4 * NCH; ++s) {
        const int k0 = 8 * s + tig, k1 = k0 + 4;
        const float p0 = k0 < K ? phi[k0 * GS] : 0.f, p1 = k1 < K ? phi[k1 * GS] : 0.f;
        const float h0 = v1_tf32(p0), h1 = v1_tf32(p1);
        b0[s] = gid < 4 ? h0 : v1_tf32(p0 - h0);
        b1[s] = gid < 4 ? h1 : v1_tf32(p1 - h1);
    }
    const int g0 = 2 * (tig & 1), half = tig >> 1;    // after the hi/lo fold: this lane stores spectra g0, g0+1 of octet o + half
    for (int base = lo + V1_WARP * 256; base < hi; base += sweep) {
        // two 16-pixel tiles per trip: the 16 LDG.128 of a chunk are all in flight before its first MMA, and the four
        // accumulation chains (tile x table hi/lo) are independent
#pragma unroll 1
        for (int mt = 0; mt < 16; mt += 2) {
            const int jA = base + mt * 16;
            if (jA >= hi) break;                           // warp-uniform
            const int jB = jA + 16 < hi ? jA + 16 : jA;    // odd tail: the second tile repeats the first (not stored)
            const float4 *fA = CF + (size_t)(jA >> 3) * ks * 32, *fB = CF + (size_t)(jB >> 3) * ks * 32;
            float ah[4] = {0.f, 0.f, 0.f, 0.f}, al[4] = {0.f, 0.f, 0.f, 0.f}, bh[4] = {0.f, 0.f, 0.f, 0.f}, bl[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
                float4 A0[4], A1[4], B0[4], B1[4];
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    const int sc = 4 * ch + s < ks ? 4 * ch + s : 0;   // k-steps past ks re-read step 0 (their B fragments are zero)
                    A0[s] = __ldg(fA + sc * 32); A1[s] = __ldg(fA + (ks + sc) * 32);
                    B0[s] = __ldg(fB + sc * 32); B1[s] = __ldg(fB + (ks + sc) * 32);
                }
#pragma unroll
                for (int s = 0; s < 4; ++s) {
                    v1_mma_tf32(ah, A0[s].x, A1[s].x, A0[s].y, A1[s].y, b0[4 * ch + s], b1[4 * ch + s]);   // table hi
                    v1_mma_tf32(bh, B0[s].x, B1[s].x, B0[s].y, B1[s].y, b0[4 * ch + s], b1[4 * ch + s]);
                    v1_mma_tf32(al, A0[s].z, A1[s].z, A0[s].w, A1[s].w, b0[4 * ch + s], b1[4 * ch + s]);   // table lo
                    v1_mma_tf32(bl, B0[s].z, B1[s].z, B0[s].w, B1[s].w, b0[4 * ch + s], b1[4 * ch + s]);
                }
            }
            // D[pixel][n]: lane holds n = 2 tig, 2 tig + 1 for pixels gid (d0, d1) and gid + 8 (d2, d3); T_g = D[g] + D[g+4]
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                ah[i] += al[i]; bh[i] += bl[i];
                ah[i] += __shfl_xor_sync(FULL, ah[i], 2); bh[i] += __shfl_xor_sync(FULL, bh[i], 2);
            }
            const int jpA = jA + half * 8 + gid, jpB = jB + half * 8 + gid;
            if (jpA < hi) {
                float *e0 = (float *)((float4 *)(rowT + g0 * RL) + SW4(jpA >> 2)) + (jpA & 3);
                float *e1 = (float *)((float4 *)(rowT + (g0 + 1) * RL) + SW4(jpA >> 2)) + (jpA & 3);
                *e0 = half ? ah[2] : ah[0]; *e1 = half ? ah[3] : ah[1];
            }
            if (jB != jA && jpB < hi) {
                float *e0 = (float *)((float4 *)(rowT + g0 * RL) + SW4(jpB >> 2)) + (jpB & 3);
                float *e1 = (float *)((float4 *)(rowT + (g0 + 1) * RL) + SW4(jpB >> 2)) + (jpB & 3);
                *e0 = half ? bh[2] : bh[0]; *e1 = half ? bh[3] : bh[1];
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// Which octet of the fitted range a thread owns in the phases that work with the continuum basis (forward, moments,
// residual), and the Chebyshev nodes.
//
// The internal basis T_n(t) lives on the symmetric nodes  t_j = (2 (j - fit_lo) - (N - 1)) / (N - 1), N = fit_hi - fit_lo
// (an even number of octets, lasp_gpu.cu), so that the pixel mirrored about the centre of the fitted range has the
// node -t_j EXACTLY (odd integer numerators), and T_n(-t) = (-1)^n T_n(t).
//
// SYM (resident variant): lanes l < 16 and 31 - l of a warp own the mirrored octets p and Noct - 1 - p (pair p = sweep *
// nt/2 + 16 warp + l).  A sum over both octets  sum_j v_j T_n(t_j)  is then  sum_i T_n(t_i) [v_i + (-1)^n v'_(7-i)]  in
// one lane's own nodes: lane l takes the even n with v + v', lane 31 - l the odd n with v' - v (its own nodes), each
// HALF of the basis; a continuum evaluation likewise splits into E(t) = sum_even b_n T_n, O(t) = sum_odd b_n T_n with
// c(t) = E + O, c(-t) = E - O.  The exchange is 32 shuffles with lane ^ 31.  Halves the FMAs, the recurrences and the
// transposes of the right-hand side, the moments and the continuum evaluation.
// !SYM (streaming variant: a sweep must be one contiguous window): thread tid owns octet sweep * nt + tid, full basis.
// ------------------------------------------------------------------------------------------
template <bool SYM>
__device__ __forceinline__ int v1_nsweep(const SegDev &sg)
{
    const int noct = (sg.fit_hi - sg.fit_lo) >> 3;
    return SYM ? ((noct >> 1) + (V1_NT >> 1) - 1) / (V1_NT >> 1) : (noct + V1_NT - 1) / V1_NT;
}

template <bool SYM>
__device__ __forceinline__ int v1_oct_of(const SegDev &sg, int sw, bool &act)
{
    const int noct = (sg.fit_hi - sg.fit_lo) >> 3;
    if (SYM) {
        const int lane = V1_LANE, p = sw * (V1_NT >> 1) + 16 * V1_WARP + (lane < 16 ? lane : 31 - lane);
        act = p < (noct >> 1);
        return sg.fit_lo + OCT * (act ? (lane < 16 ? p : noct - 1 - p) : 0);
    }
    const int o = sw * V1_NT + V1_TID;
    act = o < noct;
    return sg.fit_lo + OCT * o;   // inactive threads never dereference it
}

// Chebyshev recurrence state for the thread's octet.  Full basis: (pp, pc) = (T_-1, T_0) = (t, 1), step x2 = 2 t.
// SYM: lanes < 16 walk the even n: (T_-2, T_0) = (T_2, 1); lanes >= 16 the odd n: (T_-1, T_1) = (t, t); step 2 T_2
// (2 T_2 T_n = T_(n+2) + T_(n-2)).
template <bool SYM>
__device__ __forceinline__ void v1_cheb_init(const SegDev &sg, int j0, float (&pp)[OCT], float (&pc)[OCT], float (&x2)[OCT])
{
    const int nm1 = sg.fit_hi - sg.fit_lo - 1;
    const float tm = sg.ta;
    const bool hi = V1_LANE >= 16;
#pragma unroll
    for (int i = 0; i < OCT; ++i) {
        const float t = tm * (float)(2 * (j0 + i - sg.fit_lo) - nm1);
        if (SYM) {
            const float t2 = fmaf(2.f * t, t, -1.f);
            pp[i] = hi ? t : t2; pc[i] = hi ? t : 1.f; x2[i] = 2.f * t2;
        } else { pp[i] = t; pc[i] = 1.f; x2[i] = 2.f * t; }
    }
}

// sums  sum_i x[g][i] T_n(t_i)  for the basis the lane walks, reduced over the warp into this warp's slots slot0 + n:
// nred = number of n (rounded up to 8) of the full basis.  `first` overwrites the slots, else accumulates.
template <bool SYM>
__device__ __forceinline__ void v1_basis_sums(const float (&x)[GS][OCT], float (&pp)[OCT], float (&pc)[OCT], const float (&x2)[OCT],
                                              float *red, int slot0, int nred, bool first)
{
    const int lane = V1_LANE;
    if (SYM) {
        const int hi = lane >> 4;
        for (int n0 = 0; n0 < (nred >> 1); n0 += 4) {      // four n of this lane's parity per transpose: value (nn, g) at nn*4 + g
            float X[16];
#pragma unroll
            for (int nn = 0; nn < 4; ++nn) {
#pragma unroll
                for (int g = 0; g < GS; ++g) {
                    float sr = 0.f;
#pragma unroll
                    for (int i = 0; i < OCT; ++i) sr = fmaf(x[g][i], pc[i], sr);
                    X[nn * 4 + g] = sr;
                }
#pragma unroll
                for (int i = 0; i < OCT; ++i) { const float nx = fmaf(x2[i], pc[i], -pp[i]); pp[i] = pc[i]; pc[i] = nx; }
            }
            const float tot = xreduce16(X, lane);
            float *r = red + (slot0 + 2 * (n0 + ((lane & 15) >> 2)) + hi) * GS + (lane & 3);
            if (first) *r = tot; else *r += tot;
        }
    } else {
        for (int n0 = 0; n0 < nred; n0 += 8) {             // eight n per transpose
            float X[32];
#pragma unroll
            for (int nn = 0; nn < 8; ++nn) {
#pragma unroll
                for (int g = 0; g < GS; ++g) {
                    float sr = 0.f;
#pragma unroll
                    for (int i = 0; i < OCT; ++i) sr = fmaf(x[g][i], pc[i], sr);
                    X[nn * 4 + g] = sr;
                }
#pragma unroll
                for (int i = 0; i < OCT; ++i) { const float nx = fmaf(x2[i], pc[i], -pp[i]); pp[i] = pc[i]; pc[i] = nx; }
            }
            const float tot = xreduce32(X, lane);
            float *r = red + (slot0 + n0 + (lane >> 2)) * GS + (lane & 3);
            if (first) *r = tot; else *r += tot;
        }
    }
}

// SYM: x <- x + (-1)^n x(mirror) for the parity this lane walks (lanes < 16: +, lanes >= 16: -); pixel i of this octet
// mirrors pixel 7 - i of lane ^ 31's octet
__device__ __forceinline__ void v1_mirror_combine(float (&x)[GS][OCT])
{
    const bool hi = V1_LANE >= 16;
#pragma unroll
    for (int g = 0; g < GS; ++g)
#pragma unroll
        for (int i = 0; i < OCT / 2; ++i) {
            const float ra = __shfl_xor_sync(FULL, x[g][OCT - 1 - i], 31), rb = __shfl_xor_sync(FULL, x[g][i], 31);
            x[g][i] = hi ? x[g][i] - ra : x[g][i] + ra;
            x[g][OCT - 1 - i] = hi ? x[g][OCT - 1 - i] - rb : x[g][OCT - 1 - i] + rb;
        }
}

// ------------------------------------------------------------------------------------------
// a4 + a5 (accumulation part).  For the thread's octet of the fitted range:
//   S = G (*) T (or re-read from row A when `stencil` is false), stored to row A;
//   u = w S^2, v = w S (y - c_prev S);
//   Chebyshev moments  mom_n = sum_j u_j T_n(t_j), n < 2D+1 (only when `mom`), and the residual-form
//   right-hand side    rhs_n = sum_j v_j T_n(t_j), n <= D      (SURVEY.md section 7 "moment route";
//   T_m T_n = (T_{m+n} + T_{|m-n|})/2 turns the moments into the Gram matrix of Eq. 6's WLS).
// Partial sums over the thread's 8 pixels are reduced over the warp by register transposes and
// land in this warp's reduction slots.
// ------------------------------------------------------------------------------------------
template <bool UNI, bool STREAM>
__device__ __noinline__ void v1_phase_forward(int s_, bool stencil)
{
    const SegDev &sg = v1_blk.M.seg[s_];
    const V1Args &a = v1_blk.A;
    const V1Lay &L = v1_blk.L;
    const int *tap = (const int *)(V1SM + L.oTAP);
    float *red = V1SM + L.oRED + V1_WARP * L.VR * GS;
    // hoisted to registers (the model sits in shared memory; see v1_phase_emulator)
    const int Ppad = v1_blk.M.Ppad, P8 = Ppad >> 3, RL = L.RL, NA = L.NA, n1r = L.n1r, nmomr = L.nmomr, nt8 = V1_NT * OCT;
    constexpr bool SYM = !STREAM;
    const int fit_lo = sg.fit_lo;
    float *rowA = v1_rowp(L.oA, sg.po);
    const float *rowT = v1_rowp(L.oT, sg.po);
    float *ag = v1_blk.ag;
    const float4 *gw4 = (const float4 *)(V1SM + L.oGW);
    const float *Yg = a.Y, *Wg = a.W;
    const float *cpg = v1_blk.cp;
    constexpr bool uniform = UNI;
    const float *ISg = a.IS + V1_TPAD, *SJg = a.SJ + V1_TPAD;
    float *dsg = v1_blk.ds;
    int alo[GS], nag[GS];
    size_t rowo[GS];
#pragma unroll
    for (int g = 0; g < GS; ++g) { alo[g] = tap[2 * g]; nag[g] = tap[2 * g + 1]; rowo[g] = (size_t)v1_blk.spec[g] * Ppad; }
    if (!uniform && stencil && !STREAM) {
        // Per-pixel kernels, resident rows: the stencil runs as two passes of its own ahead of the basis sums, thread t
        // on octet t for the first two spectra and on octet N - 1 - t for the other two.  On a linear grid the kernels
        // widen by 15-25 % from the blue to the red end of an arm: with the mirrored-pair mapping of the basis sums
        // (lanes < 16 blue, lanes >= 16 red, warp 0 at the two ends) half of every warp waits for the other half and every
        // warp for warp 0; here the lanes of a warp work on neighbouring octets and every thread gets one octet of each
        // half.  S goes through row A either way; the barrier hands it to the threads that sum it.
        const int noct = (sg.fit_hi - sg.fit_lo) / OCT;
        for (int pass = 0; pass < 2; ++pass)
            for (int ob = 0; ob < noct; ob += V1_NT) {
                const int o = pass ? noct - 1 - (ob + V1_TID) : ob + V1_TID;
                if (o >= 0 && o < noct) v1_np_forward_pass<STREAM>(sg, rowT, rowA, fit_lo + o * OCT, 2 * pass, 2 * pass + 2);
            }
        __syncthreads();
    }
    const int nsweep = v1_nsweep<SYM>(sg);
    for (int sw = 0; sw < nsweep; ++sw) {   // uniform trip count
        bool act;
        const int j0 = v1_oct_of<SYM>(sg, sw, act);
        const bool first = sw == 0;
        if (STREAM && stencil) {   // this sweep's window of T (written to the global rows by the emulator phase)
            const int jb = fit_lo + sw * nt8;
            __syncthreads();
            v1_window_load(v1_blk.tg, jb);
            __syncthreads();
            rowT = v1_rowp(L.oT, jb);
        }
        if (!uniform && stencil && STREAM && act) v1_np_forward_pass<STREAM>(sg, rowT, rowA, j0, 0, GS);
        float v[GS][OCT];
        if (act) {
#pragma unroll
            for (int g = 0; g < GS; ++g) {
                // flux / weight / c_prev rows come from L2: issue the loads first, the stencil hides them
                const size_t ro = rowo[g] + (j0 >> 1);   // split-octet layout: half h of octet o at h*Ppad/2 + 4 o
                const float4 y0 = __ldg((const float4 *)(Yg + ro)), y1 = __ldg((const float4 *)(Yg + ro) + P8);
                const float4 w0 = __ldcg((const float4 *)(Wg + ro)), w1 = __ldcg((const float4 *)(Wg + ro) + P8);
                const float4 *cp4 = (const float4 *)(cpg + g * Ppad + (j0 >> 1));
                const float4 c0 = __ldcg(cp4), c1 = __ldcg(cp4 + P8);
                float S[1][OCT];
                if (stencil && uniform) {
                    v1_stencil_octet<1>((const float4 *)(rowT + g * RL), j0, alo[g], nag[g], gw4 + g * NA, 0, S);
                    v1_oct_store<STREAM>(rowA, ag, g, j0, S[0]);
                } else
                    v1_oct_load<STREAM>(rowA, ag, g, j0, S[0]);
                const float yy[OCT] = {y0.x, y0.y, y0.z, y0.w, y1.x, y1.y, y1.z, y1.w};
                const float ww[OCT] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
                const float cc[OCT] = {c0.x, c0.y, c0.z, c0.w, c1.x, c1.y, c1.z, c1.w};
#pragma unroll
                for (int i = 0; i < OCT; ++i) {
                    v[g][i] = ww[i] * S[0][i] * fmaf(-cc[i], S[0][i], yy[i]);
                }
            }
        } else {
#pragma unroll
            for (int g = 0; g < GS; ++g)
#pragma unroll
                for (int i = 0; i < OCT; ++i) v[g][i] = 0.f;
        }
        // right-hand side  rhs_n = sum_j v_j T_n(t_j), n <= D
        float pp[OCT], pc[OCT], x2[OCT];
        v1_cheb_init<SYM>(sg, j0, pp, pc, x2);
        if (SYM) v1_mirror_combine(v);
        v1_basis_sums<SYM>(v, pp, pc, x2, red, nmomr, n1r, first);
    }
}

// ------------------------------------------------------------------------------------------
// a5, refresh steps only: Gram moments  mom_n = sum_j u_j T_n(t_j), u = w S^2, n < 2D+1  (S is in row A, w comes
// from L2 again).  Kept apart from v1_phase_forward so that the every-step code stays small.
// ------------------------------------------------------------------------------------------
template <bool STREAM>
__device__ __noinline__ void v1_phase_moments(int s_)
{
    const SegDev &sg = v1_blk.M.seg[s_];
    const V1Lay &L = v1_blk.L;
    float *red = V1SM + L.oRED + V1_WARP * L.VR * GS;
    constexpr bool SYM = !STREAM;
    const int Ppad = v1_blk.M.Ppad, P8 = Ppad >> 3, nmomr = L.nmomr;
    const float *rowA = v1_rowp(L.oA, sg.po);
    const float *ag = v1_blk.ag;
    const float *Wg = v1_blk.A.W;
    const int nsweep = v1_nsweep<SYM>(sg);
    for (int sw = 0; sw < nsweep; ++sw) {
        bool act;
        const int j0 = v1_oct_of<SYM>(sg, sw, act);
        float u[GS][OCT], pp[OCT], pc[OCT], x2[OCT];
#pragma unroll
        for (int g = 0; g < GS; ++g) {
#pragma unroll
            for (int i = 0; i < OCT; ++i) u[g][i] = 0.f;
            if (act) {
                const size_t ro = (size_t)v1_blk.spec[g] * Ppad + (j0 >> 1);
                const float4 w0 = __ldcg((const float4 *)(Wg + ro)), w1 = __ldcg((const float4 *)(Wg + ro) + P8);
                float SS[OCT];
                v1_oct_load<STREAM>(rowA, ag, g, j0, SS);
                const float ww[OCT] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
#pragma unroll
                for (int i = 0; i < OCT; ++i) u[g][i] = ww[i] * SS[i] * SS[i];
            }
        }
        v1_cheb_init<SYM>(sg, j0, pp, pc, x2);
        if (SYM) v1_mirror_combine(u);
        v1_basis_sums<SYM>(u, pp, pc, x2, red, 0, nmomr, sw == 0);
    }
}

// ------------------------------------------------------------------------------------------
// a5 (solve part), warp g for spectrum g, lanes = rows of the (D+1)x(D+1) system padded to 32 with
// the identity.  A_ij = (mom_{i+j} + mom_{|i-j|})/2 ; b += A^-1 rhs (one step of iterative
// refinement whose residual was formed from the pixel data).  With
// `refactor` false the Cholesky factor kept in shared memory from an earlier step is reused
// (the refinement's fixed point does not depend on it).
// LF[row*33 + col] holds the unit-diagonal factor Lt = L D^-1, then the 32 values 1/d^2.
// ------------------------------------------------------------------------------------------
#define V1_LFS (32 * 33 + 32)
#define V1_INVC 16       // columns of the inverse per pass

// Gram matrix from the moments, Cholesky with lanes = rows, factor kept in shared memory.  Its own function so that
// the every-step solve below stays a few hundred instructions.
__device__ __noinline__ void v1_refactor(int g, int seg)
{
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int n1 = M.n1, lane = V1_LANE;
    float *momS = V1SM + L.oMOM + g * L.nmomr;
    float *lf = V1SM + L.oLF + (seg * L.lfseg * GS + g) * V1_LFS;
    float *invd = lf + 32 * 33;
    const float *red = V1SM + L.oRED;
    const int wst = L.VR * GS;
    for (int n = lane; n < L.nmomr; n += 32) {
        float s = 0.f;
        for (int w = 0; w < L.NW; ++w) s += red[w * wst + SLOT_MOM(L, n) * GS + g];
        momS[n] = s;
    }
    __syncwarp();
    // This function runs once per `refresh` steps, so its instructions are never in the instruction cache when it
    // starts: everything is a short loop over shared memory (the fully unrolled register version spent most of its
    // time fetching 50 KB of straight-line code).  Row `lane` of A, identity padding beyond n1.
    float *own = lf + lane * 33;                  // this lane's row
#pragma unroll 1
    for (int j0 = 0; j0 < 32; j0 += 8) {
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int j = j0 + u;
            int d = lane - j;
            d = d < 0 ? -d : d;
            v[u] = (j < n1 && lane < n1) ? 0.5f * (momS[lane + j] + momS[d]) : (j == lane ? 1.f : 0.f);
        }
#pragma unroll
        for (int u = 0; u < 8; ++u) own[j0 + u] = v[u];
    }
    __syncwarp();
    const float m0 = momS[0];
    bool ok = true;
#pragma unroll 1
    for (int k = 0; k < n1; ++k) {            // right-looking Cholesky, lanes = rows; column k travels by shuffle
        const float d = lf[k * 33 + k];
        if (!(d > 1e-6f * 0.5f * (momS[2 * k] + m0))) ok = false;
        const float lik = lane >= k ? own[k] * rsqrtf(d) : 0.f;
        __syncwarp();
        own[k] = lik;
#pragma unroll 1
        for (int j0 = k + 1; j0 < n1; j0 += 8) {
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = own[min(j0 + u, 31)];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = fmaf(-lik, __shfl_sync(FULL, lik, (j0 + u) & 31), v[u]);
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (j0 + u < n1) own[j0 + u] = v[u];
        }
        __syncwarp();
    }
    const float mine = 1.f / own[lane];
    invd[lane] = mine;
    if (lane == 0) {
        SMV(L.oSC, SC_N + seg, g) = ok ? 0.f : 1.f;
        const unsigned bit = 1u << (seg * GS + g);   // the adaptive policy re-factorises every step while a system fails
        if (ok) atomicAnd(&v1_blk.failmask, ~bit); else atomicOr(&v1_blk.failmask, bit);
    }
    __syncwarp();
    // unit-diagonal factor Lt = L D^-1 (D = diag L) and 1/d^2:  A^-1 = Lt^-T D^-2 Lt^-1
#pragma unroll 1
    for (int j0 = 0; j0 < n1; j0 += 8) {
        float v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) v[u] = own[min(j0 + u, 31)] * invd[min(j0 + u, 31)];
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (j0 + u < n1) own[j0 + u] = v[u];
    }
    __syncwarp();
    invd[lane] = mine * mine;
    __syncwarp();
    // Explicit inverse X = A^-1 = Lt^-T D^-2 Lt^-1, V1_INVC columns at a time with lanes = rows (the same shuffle
    // chains as a triangular solve, V1_INVC of them interleaved).  X is symmetric: column c is parked in the unused
    // upper triangle of LF (rows < c) while the lower triangle still holds Lt, and mirrored at the end, so that
    // the solve of EVERY step is a 32x32 matrix-vector product without a serial chain.
    {
        const float id2 = invd[lane];
        float diag = 1.f;
#pragma unroll 1
        for (int c0 = 0; c0 < n1; c0 += V1_INVC) {
            float r[V1_INVC];
#pragma unroll
            for (int c = 0; c < V1_INVC; ++c) r[c] = (lane == c0 + c) ? 1.f : 0.f;
            for (int k = c0; k < n1; ++k) {          // Lt z = e_c: z is zero above row c
                const float lk = lf[lane * 33 + k];
#pragma unroll
                for (int c = 0; c < V1_INVC; ++c) {
                    const float zk = __shfl_sync(FULL, r[c], k);
                    if (lane > k) r[c] = fmaf(-lk, zk, r[c]);
                }
            }
#pragma unroll
            for (int c = 0; c < V1_INVC; ++c) r[c] *= id2;
            for (int k = n1 - 1; k > 0; --k) {       // Lt^T x = D^-2 z
                const float lk = lf[k * 33 + lane];
#pragma unroll
                for (int c = 0; c < V1_INVC; ++c) {
                    const float xk = __shfl_sync(FULL, r[c], k);
                    if (lane < k) r[c] = fmaf(-lk, xk, r[c]);
                }
            }
            __syncwarp();
#pragma unroll
            for (int c = 0; c < V1_INVC; ++c) {
                if (lane == c0 + c) diag = r[c];
                if (lane < c0 + c && c0 + c < 32) lf[lane * 33 + c0 + c] = r[c];
            }
            __syncwarp();
        }
        own[lane] = diag;
#pragma unroll 1
        for (int j0 = 0; j0 < n1; j0 += 8) {     // mirror: row `lane` left of the diagonal
            float v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = lf[min(j0 + u, 31) * 33 + lane];
#pragma unroll
            for (int u = 0; u < 8; ++u)
                if (j0 + u < n1 && j0 + u < lane) own[j0 + u] = v[u];
        }
        __syncwarp();
    }
}

__device__ __noinline__ void v1_phase_solve(int g, int seg, bool refactor)
{
#ifdef LASP_PHASE_TIMING
    unsigned long long *dbg_ = v1_blk.A.dbg;
    long long tk_ = clock64();
#define SOLVE_TICK(i) do { if (dbg_ && V1_TID == 0) { const long long t_ = clock64(); atomicAdd(dbg_ + (i), (unsigned long long)(t_ - tk_)); tk_ = t_; } } while (0)
#define SOLVE_COUNT(i) do { if (dbg_ && V1_TID == 0) atomicAdd(dbg_ + (i), 1ull); } while (0)
#else
#define SOLVE_COUNT(i) do { } while (0)
#define SOLVE_TICK(i) do { } while (0)
#endif
    if (refactor) { v1_refactor(g, seg); SOLVE_TICK(18); SOLVE_COUNT(21); }
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int n1 = M.n1, lane = V1_LANE, rowB = seg * M.n1;
    const float *lf = V1SM + L.oLF + (seg * L.lfseg * GS + g) * V1_LFS;
    const float *red = V1SM + L.oRED + SLOT_RHS(L, lane) * GS + g;
    const int wst = L.VR * GS, NW = L.NW;
    // one batch of loads: this lane's right-hand side over the warps' slots, its column of A^-1 (symmetric: row
    // reads are conflict-free; the identity beyond n1), the flag and the coefficient it updates
    float rp[12], xc[32];
#pragma unroll
    for (int w = 0; w < 12; ++w) rp[w] = (w < NW && lane < n1) ? red[w * wst] : 0.f;
#pragma unroll
    for (int j = 0; j < 32; ++j) xc[j] = lf[j * 33 + lane];
    const bool ok = SMV(L.oSC, SC_N + seg, g) == 0.f;
    const float b0 = SMV(L.oB, rowB + min(lane, n1 - 1), g);
    float rv = 0.f;
#pragma unroll
    for (int w = 0; w < 12; ++w) rv += rp[w];
    SOLVE_TICK(19);
    // x = A^-1 rhs, row `lane`; rhs_j travels by shuffle (zero beyond n1)
    float r0 = 0.f, r1 = 0.f, r2 = 0.f, r3 = 0.f;
#pragma unroll
    for (int j = 0; j < 32; j += 4) {
        r0 = fmaf(xc[j], __shfl_sync(FULL, rv, j), r0);
        r1 = fmaf(xc[j + 1], __shfl_sync(FULL, rv, j + 1), r1);
        r2 = fmaf(xc[j + 2], __shfl_sync(FULL, rv, j + 2), r2);
        r3 = fmaf(xc[j + 3], __shfl_sync(FULL, rv, j + 3), r3);
    }
    const float r = (r0 + r1) + (r2 + r3);
    if (lane < n1) SMV(L.oB, rowB + lane, g) = ok ? b0 + r : 0.f;
    __syncwarp();
    SOLVE_TICK(20);
}

// ------------------------------------------------------------------------------------------
// a5 (evaluation part) + a6.  c_j = sum_n b_n T_n(t_j) on the thread's octet -> c_prev scratch;
//   MODE 0: nothing else (between the two solves of a cold start);
//   MODE 1: r = y - c S, chi2, adjoint a = -2 w r c -> row A (replaces S), ngood, min c;
//   MODE 2: as 1, and rho = sqrt(w) r -> global row `xrow` (a9);
//   MODE 3: the adjoint only (Adam steps on uniform segments: chi2, ngood and min c are not needed until the final
//           evaluation, so their per-pixel updates and the reduction are left out).
// chi2 / ngood / cmin are reduced over the warp and accumulated in this warp's SLOT_STAT slots (zeroed by v1_evaluate).
// ------------------------------------------------------------------------------------------
template <int MODE, bool UNI, bool STREAM>
__device__ __noinline__ void v1_phase_residual(int s_, float *xrow)
{
    const SegDev &sg = v1_blk.M.seg[s_];
    const int rowB = s_ * v1_blk.M.n1;
    const V1Args &a = v1_blk.A;
    const V1Lay &L = v1_blk.L;
    const float4 *b4 = (const float4 *)(V1SM + L.oB) + rowB;
    constexpr bool SYM = !STREAM;
    const int Ppad = v1_blk.M.Ppad, P8 = Ppad >> 3, n1 = v1_blk.M.n1;
    float *rowA = v1_rowp(L.oA, sg.po);
    float *ag = v1_blk.ag;
    const float *Yg = a.Y, *Wg = a.W;
    float *cpg = v1_blk.cp;
    size_t rowo[GS];
#pragma unroll
    for (int g = 0; g < GS; ++g) rowo[g] = (size_t)v1_blk.spec[g] * Ppad;
    float chi[GS], ng[GS], cmin[GS], gvv[GS], gss[GS];
    constexpr bool uniform = UNI;
    const float *dsg = v1_blk.ds;
#pragma unroll
    for (int g = 0; g < GS; ++g) { chi[g] = 0.f; ng[g] = 0.f; cmin[g] = 3.0e38f; gvv[g] = 0.f; gss[g] = 0.f; }
    const int nsweep = v1_nsweep<SYM>(sg);
    for (int sw = 0; sw < nsweep; ++sw) {
        bool act;
        const int j0 = v1_oct_of<SYM>(sg, sw, act);
        if (!SYM && !act) continue;        // SYM: inactive lanes stay for the exchange (their partner is inactive too)
        float cc[GS][OCT], pp[OCT], pc[OCT], x2[OCT];
        float4 yq[GS][2], wq[GS][2];   // flux / weight from L2, issued before the basis loop hides them
        if (MODE != 0) {
#pragma unroll
            for (int g = 0; g < GS; ++g) {
                const size_t ro = rowo[g] + (j0 >> 1);
                yq[g][0] = __ldg((const float4 *)(Yg + ro)); yq[g][1] = __ldg((const float4 *)(Yg + ro) + P8);
                wq[g][0] = __ldcg((const float4 *)(Wg + ro)); wq[g][1] = __ldcg((const float4 *)(Wg + ro) + P8);
            }
        }
        v1_cheb_init<SYM>(sg, j0, pp, pc, x2);
#pragma unroll
        for (int g = 0; g < GS; ++g)
#pragma unroll
            for (int i = 0; i < OCT; ++i) cc[g][i] = 0.f;
        if (SYM) {
            // this lane's half of the basis at its own nodes: E = sum_even b_n T_n (lanes < 16) or O = sum_odd b_n T_n
            // (lanes >= 16); then c(t_i) = E_i - O'_(7-i) on lanes < 16 and c(t'_i) = E_(7-i) + O'_i on lanes >= 16,
            // the other half coming from lane ^ 31 (whose nodes are the negatives of this lane's)
            const int hi = V1_LANE >> 4;
            for (int n = hi; n < n1; n += 2) {
                const float4 b = b4[n];
                const float bg[GS] = {b.x, b.y, b.z, b.w};
#pragma unroll
                for (int g = 0; g < GS; ++g)
#pragma unroll
                    for (int i = 0; i < OCT; ++i) cc[g][i] = fmaf(bg[g], pc[i], cc[g][i]);
#pragma unroll
                for (int i = 0; i < OCT; ++i) { const float nx = fmaf(x2[i], pc[i], -pp[i]); pp[i] = pc[i]; pc[i] = nx; }
            }
#pragma unroll
            for (int g = 0; g < GS; ++g)
#pragma unroll
                for (int i = 0; i < OCT / 2; ++i) {
                    const float ra = __shfl_xor_sync(FULL, cc[g][OCT - 1 - i], 31), rb = __shfl_xor_sync(FULL, cc[g][i], 31);
                    cc[g][i] = hi ? cc[g][i] + ra : cc[g][i] - ra;
                    cc[g][OCT - 1 - i] = hi ? cc[g][OCT - 1 - i] + rb : cc[g][OCT - 1 - i] - rb;
                }
            if (!act) continue;
        } else {
            for (int n = 0; n < n1; ++n) {
                const float4 b = b4[n];
                const float bg[GS] = {b.x, b.y, b.z, b.w};
#pragma unroll
                for (int g = 0; g < GS; ++g)
#pragma unroll
                    for (int i = 0; i < OCT; ++i) cc[g][i] = fmaf(bg[g], pc[i], cc[g][i]);
#pragma unroll
                for (int i = 0; i < OCT; ++i) { const float nx = fmaf(x2[i], pc[i], -pp[i]); pp[i] = pc[i]; pc[i] = nx; }
            }
        }
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            float4 *cp4 = (float4 *)(cpg + g * Ppad + (j0 >> 1));
            cp4[0] = make_float4(cc[g][0], cc[g][1], cc[g][2], cc[g][3]);
            cp4[P8] = make_float4(cc[g][4], cc[g][5], cc[g][6], cc[g][7]);
            if (MODE == 0) continue;
            float SS[OCT];
            v1_oct_load<STREAM>(rowA, ag, g, j0, SS);
            const float4 y0 = yq[g][0], y1 = yq[g][1], w0 = wq[g][0], w1 = wq[g][1];
            const float yy[OCT] = {y0.x, y0.y, y0.z, y0.w, y1.x, y1.y, y1.z, y1.w};
            const float ww[OCT] = {w0.x, w0.y, w0.z, w0.w, w1.x, w1.y, w1.z, w1.w};
            float av[OCT], rho[OCT];
#pragma unroll
            for (int i = 0; i < OCT; ++i) {
                const float r = fmaf(-cc[g][i], SS[i], yy[i]);
                const float wr = ww[i] * r;
                if (MODE != 3) {
                    chi[g] = fmaf(wr, r, chi[g]);
                    if (ww[i] > 0.f) { cmin[g] = fminf(cmin[g], cc[g][i]); ng[g] += 1.f; }
                }
                av[i] = -2.f * wr * cc[g][i];
                if (MODE == 2) rho[i] = sqrtf(ww[i]) * r;
                if (MODE == 4) { av[i] = sqrtf(ww[i]) * r; rho[i] = cc[g][i] * SS[i]; }   // eps and M = c S for the mask update
            }
            if (MODE == 4) v1_oct_store<STREAM>(v1_rowp(L.oT, sg.po), v1_blk.tg, g, j0, rho);
            if (!uniform && MODE != 4) {
                // per-pixel kernels: the two kernel-parameter gradients close here (dS/dv, dS/dsigma* were kept by the
                // forward pass), and the adjoint handed to the stencil is a/E0 (each source pixel's own normalisation)
                const float4 *d4 = (const float4 *)(dsg + g * L.SL + ((j0 - sg.po) >> 1));
                const int S8 = L.SL >> 3, SP = GS * (L.SL >> 2);
                const float4 v0 = __ldcg(d4), v1 = __ldcg(d4 + S8);
                const float4 g0 = __ldcg(d4 + SP), g1 = __ldcg(d4 + SP + S8);
                const float4 e0 = __ldcg(d4 + 2 * SP), e1 = __ldcg(d4 + 2 * SP + S8);
                const float DV[OCT] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
                const float DG[OCT] = {g0.x, g0.y, g0.z, g0.w, g1.x, g1.y, g1.z, g1.w};
                const float EI[OCT] = {e0.x, e0.y, e0.z, e0.w, e1.x, e1.y, e1.z, e1.w};
#pragma unroll
                for (int i = 0; i < OCT; ++i) {
                    gvv[g] = fmaf(av[i], DV[i], gvv[g]);
                    gss[g] = fmaf(av[i], DG[i], gss[g]);
                    av[i] *= EI[i];
                }
            }
            v1_oct_store<STREAM>(rowA, ag, g, j0, av);
            if (MODE == 2) {
                float4 *x4 = (float4 *)(xrow + g * Ppad + j0);
                x4[0] = make_float4(rho[0], rho[1], rho[2], rho[3]);
                x4[1] = make_float4(rho[4], rho[5], rho[6], rho[7]);
            }
        }
    }
    if (MODE == 1 || MODE == 2) {
        // one register transpose for the sums (chi2, ngood, and the two kernel-parameter gradients of per-pixel
        // segments): value (kind, g) at kind*4 + g; the minimum of c by shuffles
        float *red = V1SM + L.oRED + V1_WARP * L.VR * GS;
        float X[32];
#pragma unroll
        for (int i = 0; i < 32; ++i) X[i] = 0.f;
#pragma unroll
        for (int g = 0; g < GS; ++g) { X[g] = chi[g]; X[4 + g] = ng[g]; X[12 + g] = gvv[g]; X[16 + g] = gss[g]; }
        const float tot = xreduce32(X, V1_LANE);
        if (V1_LANE < 20 && (V1_LANE < 8 || V1_LANE >= 12)) red[SLOT_STAT(L) * GS + V1_LANE] += tot;   // kinds 0,1,3,4
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            const float m = warp_min_f(cmin[g]);
            if (V1_LANE == 0) { float *st = red + (SLOT_STAT(L) + 2) * GS + g; *st = fminf(*st, m); }
        }
    }
}

// ------------------------------------------------------------------------------------------
// a7 (+ the two kernel-parameter gradients of a6), reverse mode.  For the thread's octet of the T range:
//   t_i   = sum_k g_k a_{i+k}            (adjoint stencil; a = 0 outside the fitted range)
//   tmu_i, tsg_i: the same with dg/dv, dg/dsigma*   =>  dchi2/dv = sum_i T_i tmu_i, dchi2/dsigma* likewise
//   q_k   = sum_i t_i C[k,i]
// Partial sums go through register transposes into this warp's Q slots (pseudo-terms K, K+1 carry
// the two kernel-parameter gradients), which v1_evaluate zeroed.
// ------------------------------------------------------------------------------------------
template <bool UNI, bool STREAM, bool TNA = false>
__device__ __noinline__ void v1_phase_adjoint(int s_)
{
    const SegDev &sg = v1_blk.M.seg[s_];
    int lo, hi;
    v1_phase_range(sg, 0, lo, hi);
    const V1Lay &L = v1_blk.L;
    const int *tap = (const int *)(V1SM + L.oTAP);
    const int P4 = v1_blk.M.Ppad >> 2, P8 = v1_blk.M.Ppad >> 3, K = v1_blk.M.K, Kq = L.Kq, NA = L.NA, RL = L.RL, nt8 = V1_NT * OCT;
    const int wstride4 = GS * NA;   // float4 stride between the three reversed kernels
    const int qslot0 = SLOT_Q(L, 0);
    float *red = V1SM + L.oRED + V1_WARP * L.VR * GS;
    const float *Cg = v1_blk.A.C1;
    const float *rowA = v1_rowp(L.oA, sg.po), *rowT = v1_rowp(L.oT, sg.po);
    const float4 *gr4 = (const float4 *)(V1SM + L.oGR);
    int alo[GS], nag[GS];
    constexpr bool uniform = UNI;
    const float *ISg = v1_blk.A.IS + V1_TPAD, *SJg = v1_blk.A.SJ + V1_TPAD;
    V1Np npp[UNI ? 1 : GS];
#pragma unroll
    for (int g = 0; g < GS; ++g) { alo[g] = tap[2 * g]; nag[g] = tap[2 * g + 1]; if (!UNI) npp[UNI ? 0 : g] = ((const V1Np *)(V1SM + L.oNP))[g]; }
    for (int jb = lo; jb < hi; jb += nt8) {
        const int j0 = jb + V1_TID * OCT;
        const bool act = j0 < hi;
        if (STREAM) {   // this sweep's window of the adjoint a (global rows, written by the residual phase)
            __syncthreads();
            v1_window_load(v1_blk.ag, jb);
            __syncthreads();
            rowA = v1_rowp(L.oA, jb);
        }
        float t[GS][OCT], gv[GS], gs[GS];
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            gv[g] = 0.f; gs[g] = 0.f;
            if (act && !uniform) {
                // sources up to H_seg above this octet carry the widest kernels (1/s_j grows with wavelength on
                // a linear grid): bound the loop by the kernel of the farthest source in reach
                const int hseg = 4 * (alo[g] + nag[g] - 1);
                const float hb = fminf(npp[UNI ? 0 : g].hbv * fmaxf(__ldg(ISg + j0 + OCT - 1 + hseg), __ldg(ISg + j0 - hseg)), npp[UNI ? 0 : g].hcap);
                v1_np_adjoint_octet((const float4 *)(rowA + g * RL), j0, (int)ceilf(hb), npp[UNI ? 0 : g], ISg, SJg, t[g]);
            } else if (act) {
                float acc[3][OCT];
                v1_stencil_octet<3>((const float4 *)(rowA + g * RL), j0, alo[g], nag[g], gr4 + g * NA, wstride4, acc);
                float TT[OCT];
                v1_oct_load<STREAM>(rowT, v1_blk.tg, g, j0, TT);
#pragma unroll
                for (int i = 0; i < OCT; ++i) {
                    t[g][i] = acc[0][i];
                    gv[g] = fmaf(TT[i], acc[1][i], gv[g]);
                    gs[g] = fmaf(TT[i], acc[2][i], gs[g]);
                }
            } else {
#pragma unroll
                for (int i = 0; i < OCT; ++i) t[g][i] = 0.f;
            }
        }
        // C[k, octet] in batches of 4 terms, the next batch in flight during the multiplies; the table is
        // zero past K, so rows K and K+1 are free to carry the two kernel-parameter gradients
        const float4 *c4 = (const float4 *)Cg + ((act ? j0 : lo) >> 3);
        float4 bufA[8], bufB[8];
        auto load4 = [&](int kb, float4 (&buf)[8]) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                buf[2 * u] = v1_ld_table<TNA>(c4 + (kb + u) * P4);
                buf[2 * u + 1] = v1_ld_table<TNA>(c4 + (kb + u) * P4 + P8);
            }
        };
        load4(0, bufA);
        for (int k0 = 0; k0 < Kq; k0 += 8) {
            float X[32];
            auto dot4 = [&](int xo, const float4 (&buf)[8]) {
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                    const float4 ca = buf[2 * u], cb = buf[2 * u + 1];
                    const float cc[OCT] = {ca.x, ca.y, ca.z, ca.w, cb.x, cb.y, cb.z, cb.w};
#pragma unroll
                    for (int g = 0; g < GS; ++g) {
                        float sacc = 0.f;
#pragma unroll
                        for (int i = 0; i < OCT; ++i) sacc = fmaf(t[g][i], cc[i], sacc);
                        X[xo + u * 4 + g] = sacc;
                    }
                }
            };
            load4(k0 + 4, bufB);
            dot4(0, bufA);
            load4(k0 + 8, bufA);
            if (k0 + 4 < Kq) dot4(16, bufB);
            else {
#pragma unroll
                for (int i = 16; i < 32; ++i) X[i] = 0.f;
            }
            if (k0 + 8 > K) {   // uniform: the block holding rows K and K+1 (K+1 < Kq always)
#pragma unroll
                for (int kk = 0; kk < 8; ++kk)
#pragma unroll
                    for (int g = 0; g < GS; ++g) X[kk * 4 + g] += (k0 + kk == K) ? gv[g] : ((k0 + kk == K + 1) ? gs[g] : 0.f);
            }
            const float tot = xreduce32(X, V1_LANE);
            red[(qslot0 + k0 + (V1_LANE >> 2)) * GS + (V1_LANE & 3)] += tot;
        }
    }
}

// After the first barrier of an evaluation: this warp's Q and statistics slots, which accumulate over sweeps and
// segments, are zeroed (only now have warps g < GS finished reading the previous evaluation's), and for the
// evaluations of the Adam loop thread 0 takes the Gram re-factorisation decision (momsel 0 / 1: as told; 2: adaptive,
// from what the update warps left before the barrier) and publishes it in v1_blk.momflag, read after the next barrier.
__device__ __forceinline__ void v1_begin_eval(int momsel, bool adam)
{
    const V1Lay &L = v1_blk.L;
    float *red = V1SM + L.oRED + V1_WARP * L.VR * GS;
    const int q0 = (L.nmomr + L.n1r) * GS;
    for (int i = q0 + V1_LANE; i < L.VR * GS; i += 32) red[i] = 0.f;
    __syncwarp();
    if (V1_LANE < GS) red[(SLOT_STAT(L) + 2) * GS + V1_LANE] = 3.0e38f;
    __syncwarp();
    if (V1_TID == 0 && adam) {
        const bool force = v1_blk.force != 0;   // the weights changed (Clean mask update)
        bool fresh = momsel == 1 || force;
        v1_blk.force = 0;
        if (momsel == 2) {
            const float step = __int_as_float(v1_blk.stepmax);
            const float drift = v1_blk.drift + step;
            const int since = v1_blk.since + 1;
            fresh = force || v1_blk.failmask != 0u || since >= 64 || drift * step > v1_blk.A.drift_tol;
            v1_blk.drift = fresh ? 0.f : drift;
            v1_blk.since = fresh ? 0 : since;
            v1_blk.stepmax = 0;
        }
        if (fresh) v1_blk.nfresh += 1;
        v1_blk.momflag = fresh ? 1 : 0;
        v1_blk.t += 1;
    }
}

// ------------------------------------------------------------------------------------------
// One evaluation of chi2 (+ gradient) at the u held in shared memory (warps g < GS have run
// v1_param_setup for their spectrum).  All threads of the CTA call this.
//   cold: b = 0, c_prev = 0, solve twice (solve + one refinement);  else b, c_prev are warm.
//   momsel: 1 = re-accumulate the Gram moments and re-factor (always when cold); 0 = reuse the stale factor;
//           2 = adaptive: decided by thread 0 after the first barrier from the drift monitor (DESIGN.md "Stale Gram
//               factor") and read by all after the second: fresh when a segment's system was flagged not positive
//               definite, when 64 steps have passed, or when (sum of |du|_inf since the last fresh factor) x
//               (|du|_inf of the last update) > drift_tol.  `adam` marks the evaluations of the Adam loop (statistics).
//   MODE 0: chi2 + gradient partials (Q slots) ; MODE 1: chi2 only ; MODE 2: chi2 + rho -> xrow ;
//   MODE 4: eps = sqrt(w) r -> row A and M = c S -> row T, for the Clean mask update (no statistics).
// On return (after the closing barrier) the per-warp reduction slots hold chi2 / ngood / min c (not with `stats`
// false on uniform segments: the Adam steps do not read them) and, for MODE 0, the q / dv / dsigma partials.
// ------------------------------------------------------------------------------------------
template <int MODE, bool STREAM>
__device__ __noinline__ void v1_evaluate(bool cold, int momsel, float *xrow, bool wready = false, bool stats = true, bool adam = false)
{
    const V1Args &a = v1_blk.A;
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    // This warp's Q and statistics slots accumulate over sweeps and segments.  They are zeroed after
    // the first barrier of the evaluation: only then have warps g < GS finished reading the previous
    // evaluation's slots (v1_gradient / v1_stats run between evaluations without a barrier).
#ifdef LASP_PHASE_TIMING
    long long tk = a.dbg ? clock64() : 0;
    auto tick = [&](int i) {
        if (a.dbg && V1_TID == 0) { const long long t = clock64(); atomicAdd(a.dbg + i, (unsigned long long)(t - tk)); tk = t; }
    };
#else
    auto tick = [](int) {};   // per-phase cycle counters: build with -DLASP_PHASE_TIMING
#endif
    if (M.n_seg > 1 && !L.lfseg) momsel = 1;   // one factor slot shared by the segments: never stale
    bool mom = momsel == 1;
    bool zeroed = false;
    auto zero_slots = [&]() { v1_begin_eval(momsel, adam); zeroed = true; };
    for (int s = 0; s < M.n_seg; ++s) {
        const SegDev &sg = M.seg[s];
        const int rowB = s * M.n1;
        if (sg.fit_hi <= sg.fit_lo) {
            if (V1_WARP < GS) {   // no fitted pixel: b = 0, not positive definite (as the oracle)
                for (int n = V1_LANE; n < M.n1; n += 32) SMV(L.oB, rowB + n, V1_WARP) = 0.f;
                if (V1_LANE == 0) SMV(L.oSC, SC_N + s, V1_WARP) = 1.f;
            }
            continue;
        }
        if (V1_WARP < GS) {
            if (!wready) v1_setup_weights(sg, V1_WARP);   // else v1_update_fast has left them in place
            if (cold) for (int n = V1_LANE; n < M.n1; n += 32) SMV(L.oB, rowB + n, V1_WARP) = 0.f;
        }
        if (STREAM) {
            // the global rows are indexed by absolute padded pixel: a stays zero outside the fitted ranges once cleared
            if (cold && s == 0)
                for (int i = V1_TID; i < GS * M.Ppad / 4; i += V1_NT) ((float4 *)v1_blk.ag)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        } else if (M.n_seg > 1 || cold) {
            // row A must be zero outside the fitted range of THIS segment (the adjoint stencil reads it)
            for (int i = V1_TID; i < GS * L.RL / 4; i += V1_NT) ((float4 *)(V1SM + L.oA))[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        if (cold) {
            if (s == 0)
                for (int i = V1_TID; i < GS * M.Ppad / 4; i += V1_NT) ((float4 *)v1_blk.cp)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        tick(0);
        __syncthreads();
        tick(1);
        if (!zeroed) zero_slots();
        if (!STREAM && v1_blk.A.CF) {
            const int ks = v1_blk.A.ksteps;
            if (ks <= 4) v1_phase_emulator_mma<1>(s, 0);
            else if (ks <= 8) v1_phase_emulator_mma<2>(s, 0);
            else v1_phase_emulator_mma<4>(s, 0);
        } else
            v1_phase_emulator<STREAM>(s, 0);
        tick(2);
        __syncthreads();
        tick(3);
        if (adam) mom = v1_blk.momflag != 0;
        if (sg.uniform) v1_phase_forward<true, STREAM>(s, true); else v1_phase_forward<false, STREAM>(s, true);
        if (mom || cold) v1_phase_moments<STREAM>(s);   // own octets of row A only: no barrier needed in between
        tick(4);
        __syncthreads();
        tick(5);
        if (V1_WARP < GS) v1_phase_solve(V1_WARP, s, mom || cold);
        tick(6);
        __syncthreads();
        tick(7);
        if (cold) {
            v1_phase_residual<0, true, STREAM>(s, nullptr);
            __syncthreads();   // c_prev written by this thread only, but keep phases aligned
            v1_phase_forward<true, STREAM>(s, false);   // S is re-read from row A: no stencil, either kind
            __syncthreads();
            if (V1_WARP < GS) v1_phase_solve(V1_WARP, s, false);
            __syncthreads();
        }
        if (MODE == 0 && !stats && sg.uniform) v1_phase_residual<3, true, STREAM>(s, xrow);   // Adam step: no statistics
        else if (sg.uniform) v1_phase_residual<(MODE == 2 || MODE == 4 ? MODE : 1), true, STREAM>(s, xrow);
        else v1_phase_residual<(MODE == 2 || MODE == 4 ? MODE : 1), false, STREAM>(s, xrow);
        tick(8);
        __syncthreads();
        tick(9);
        if (MODE == 0) {
            if (sg.uniform) v1_phase_adjoint<true, STREAM>(s); else v1_phase_adjoint<false, STREAM>(s);
            tick(10);
            __syncthreads();
            tick(11);
        }
    }
    if (!zeroed) {   // no segment had a fitted pixel
        __syncthreads();
        zero_slots();
        __syncthreads();
    }
}

// sums of the per-warp statistics for spectrum g (any lane may call; all return the same)
__device__ __forceinline__ void v1_stats(int g, float &chi2, float &ngood, float &cmin)
{
    const V1Lay &L = v1_blk.L;
    const float *red = V1SM + L.oRED + SLOT_STAT(L) * GS + g;
    chi2 = 0.f; ngood = 0.f; cmin = 3.0e38f;
    for (int w = 0; w < L.NW; ++w) {
        const float *r = red + w * L.VR * GS;
        chi2 += r[0]; ngood += r[GS]; cmin = fminf(cmin, r[2 * GS]);
    }
}

// a7 (tail) + chain rule to u (C.1 last lines).  Warp g; grad[p] valid on lane p afterwards.
__device__ __noinline__ float v1_gradient(int g)
{
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const float *red = V1SM + L.oRED;
    const int wst = L.VR * GS, nl = M.L, K = M.K, NW = L.NW, q0 = SLOT_Q(L, 0);
    float mine = 0.f;
    for (int l0 = 0; l0 < max(nl, 1); l0 += 4) {      // d chi2 / d x_l = sum_k (d phi_k / d x_l) q_k, four labels per butterfly
        float gx[4] = {0.f, 0.f, 0.f, 0.f};
        for (int k = V1_LANE; k < K + 2; k += 32) {
            float qk = 0.f;
            for (int w = 0; w < NW; ++w) qk += red[w * wst + (q0 + k) * GS + g];
            if (k >= K) { if (l0 == 0) SMV(L.oQ, k, g) = qk; }
            else {
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (l0 + u < nl) gx[u] = fmaf(SMV(L.oDPHI, (l0 + u) * K + k, g), qk, gx[u]);
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
            for (int u = 0; u < 4; ++u) gx[u] += __shfl_xor_sync(FULL, gx[u], o);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (V1_LANE == l0 + u) mine = gx[u];
    }
    __syncwarp();
    if (V1_LANE == nl || V1_LANE == nl + 1) {     // + the part closed in the residual phase (per-pixel kernels)
        const int which = V1_LANE - nl;
        float sx = SMV(L.oQ, K + which, g);
        for (int w = 0; w < NW; ++w) sx += red[w * wst + (SLOT_STAT(L) + 3 + which) * GS + g];
        mine = sx;
    }
    if (V1_LANE < M.NP) mine *= SMV(L.oGSC, V1_LANE, g);   // chain rule to u (C.1 last lines)
    return mine;
}

// ------------------------------------------------------------------------------------------
// a7 (tail) + a8 + a1 of the next step in one pass, for models with at most four labels and K + 2 <= 32
// (L.fastupd): lane k owns term k, lane p owns parameter p.  These phases are one warp's latency and every
// dependent shared-memory round trip costs it ~100 cycles while the other CTA's stencil keeps the LSU busy: all
// loads are issued together at the top, the labels travel by shuffle and x^e is formed in registers, so the chain
// is one load batch, one butterfly and one broadcast instead of ~40 round trips.  Same arithmetic, in the same
// order, as v1_gradient + the Adam lines of the fit loop + v1_param_setup.
// ------------------------------------------------------------------------------------------
__device__ __noinline__ void v1_update_fast(int g, float ib1, float ib2)
{
    const V1Args &a = v1_blk.A;
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int lane = V1_LANE;
#ifdef LASP_PHASE_TIMING
    long long tk_ = clock64();
#define UPD_TICK(i) do { if (a.dbg && V1_TID == 0) { const long long t_ = clock64(); atomicAdd(a.dbg + (i), (unsigned long long)(t_ - tk_)); tk_ = t_; } } while (0)
#else
#define UPD_TICK(i) do { } while (0)
#endif
    const int wst = L.VR * GS, nl = M.L, K = M.K, NW = L.NW, NP = M.NP, emax = L.emax;
    const float *redq = V1SM + L.oRED + (SLOT_Q(L, 0) + min(lane, K + 1)) * GS + g;
    const int which = min(max(lane - nl, 0), 1);
    const float *reds = V1SM + L.oRED + (SLOT_STAT(L) + 3 + which) * GS + g;
    const int pl = min(lane, NP - 1), kl = min(lane, K - 1), ll = min(lane, max(nl - 1, 0));
    // ---- one batch of loads
    float qp[12], sp[12];
#pragma unroll
    for (int w = 0; w < 12; ++w) {
        qp[w] = w < NW ? redq[w * wst] : 0.f;
        sp[w] = w < NW ? reds[w * wst] : 0.f;
    }
    float dphi[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) dphi[u] = u < nl ? SMV(L.oDPHI, u * K + kl, g) : 0.f;
    const float gsc = SMV(L.oGSC, pl, g), m0 = SMV(L.oM, pl, g), v0 = SMV(L.oV, pl, g), u0 = SMV(L.oU, pl, g);
    const unsigned exw = ((const unsigned *)(V1SM + L.oEXP))[kl];
    const float lo = M.lo[pl], hi = M.hi[pl], ea = M.emu_a[ll], eb = M.emu_b[ll];
    const bool lg = M.label_log10[ll] != 0;
    const float b1 = a.b1, b2 = a.b2, lr = a.lr, eps = a.eps;
    // ---- gradient (a7 tail): q_k, then d chi2 / d x_l = sum_k (d phi_k / d x_l) q_k
    float qk = 0.f, sx = 0.f;
#pragma unroll
    for (int w = 0; w < 12; ++w) { qk += qp[w]; sx += sp[w]; }
    UPD_TICK(16);
    float gx[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) gx[u] = lane < K ? dphi[u] * qk : 0.f;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int u = 0; u < 4; ++u) gx[u] += __shfl_xor_sync(FULL, gx[u], o);
    }
    const float qvs = __shfl_sync(FULL, qk, K + which);   // the v / sigma* sums live on lanes K, K+1
    float gr = lane < nl ? (lane == 0 ? gx[0] : lane == 1 ? gx[1] : lane == 2 ? gx[2] : gx[3]) : qvs + sx;
    gr *= gsc;                                              // chain rule to u (C.1 last lines)
    UPD_TICK(17);
    // ---- a8: Adam (C.2-20), clip to the prior box (C.2-18)
    const float mm = b1 * m0 + (1.f - b1) * gr;
    const float vv = b2 * v0 + (1.f - b2) * gr * gr;
    const float mh = mm * ib1, vh = vv * ib2;
    float u = u0 - __fdividef(lr * mh, sqrtf(vh) + eps);
    u = u < -1.f ? -1.f : (u > 1.f ? 1.f : u);              // clip (C.2-18); a NaN iterate stays NaN, as in the oracle
    {   // |du|_inf of this update, for the re-factorisation monitor (NaN does not count)
        float du = lane < NP ? fabsf(u - u0) : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) du = fmaxf(du, __shfl_xor_sync(FULL, du, o));
        if (lane == 0) atomicMax(&v1_blk.stepmax, __float_as_int(du));
    }
    // ---- a1: de-normalise, emulator inputs (C.2-18/19)
    const float half = (hi - lo) * 0.5f;
    const float th = lo + (u + 1.f) * half;
    float xv = 0.f, gscn = half;
    if (lane < nl) {
        xv = ea * (lg ? log10f(th) : th) + eb;
        gscn *= lg ? ea / (th * 2.302585093f) : ea;
    }
    if (lane < NP) {
        SMV(L.oM, lane, g) = mm; SMV(L.oV, lane, g) = vv; SMV(L.oU, lane, g) = u;
        SMV(L.oGSC, lane, g) = gscn;
        if (lane < nl) SMV(L.oX, lane, g) = xv;
        else SMV(L.oSC, lane == nl ? SC_V : SC_SIG, g) = th;
    }
    UPD_TICK(22);
    // ---- monomials (Eq. 1): x^e and e x^(e-1) by repeated multiplication, as the power table does
    float pe[4], pm[4];
#pragma unroll
    for (int l = 0; l < 4; ++l) {
        const float x = __shfl_sync(FULL, xv, l);
        const int e = (exw >> (8 * l)) & 255;
        float pw = 1.f, pwm = 0.f;
        for (int q = 0; q < emax; ++q)
            if (q < e) { pwm = pw; pw *= x; }
        pe[l] = l < nl ? pw : 1.f;
        pm[l] = l < nl ? (float)e * pwm : 0.f;
    }
    if (lane < K) {
        float ph = 1.f;
#pragma unroll
        for (int l = 0; l < 4; ++l) ph *= pe[l];
        SMV(L.oPHI, lane, g) = ph;
#pragma unroll
        for (int l = 0; l < 4; ++l) {
            float d = pm[l];
#pragma unroll
            for (int l2 = 0; l2 < 4; ++l2)
                if (l2 != l) d *= pe[l2];
            if (l < nl) SMV(L.oDPHI, l * K + lane, g) = d;
        }
    }
    UPD_TICK(23);
    if (L.fastw) {   // a3 of the next step (single uniform segment): v and sigma* are on lanes nl, nl+1
        const float vn = __shfl_sync(FULL, th, nl), sn = __shfl_sync(FULL, th, nl + 1);
        v1_weights_uniform(M.seg[0], g, vn, sn);
    }
    __syncwarp();
}

// internal Chebyshev(t) coefficients -> plain Legendre(x^) (C.2-8), fp64.  Warp g, lanes over rows.
__device__ __noinline__ void v1_write_cont(int g, float *out)
{
    const ModelDev &M = v1_blk.M;
    for (int s = 0; s < M.n_seg; ++s) {
        const double *cv = M.conv + (size_t)s * M.n1 * M.n1;
        for (int m = V1_LANE; m < M.n1; m += 32) {
            double acc = 0.0;
            for (int n = 0; n < M.n1; ++n) acc += cv[m * M.n1 + n] * (double)SMV(v1_blk.L.oB, s * M.n1 + n, g);
            out[s * M.n1 + m] = (float)acc;
        }
    }
}

// copy the kernel parameters into the block state (a pointer to a kernel parameter is a generic load from
// the parameter window; a struct passed by reference to a non-inlined function is a local-memory copy)
__device__ __forceinline__ void v1_init_block(const ModelDev &M, const V1Lay &L, const V1Args &a)
{
    for (int i = threadIdx.x; i < (int)(sizeof(ModelDev) / 4); i += blockDim.x) ((int *)&v1_blk.M)[i] = ((const int *)&M)[i];
    for (int i = threadIdx.x; i < (int)(sizeof(V1Lay) / 4); i += blockDim.x) ((int *)&v1_blk.L)[i] = ((const int *)&L)[i];
    for (int i = threadIdx.x; i < (int)(sizeof(V1Args) / 4); i += blockDim.x) ((int *)&v1_blk.A)[i] = ((const int *)&a)[i];
    if (threadIdx.x == 0) {
        v1_blk.cp = a.CP ? a.CP + (size_t)blockIdx.x * GS * M.Ppad : nullptr;
        v1_blk.ds = a.DS ? a.DS + (size_t)blockIdx.x * 3 * GS * L.SL : nullptr;
        v1_blk.tg = a.TG ? a.TG + (size_t)blockIdx.x * GS * M.Ppad : nullptr;
        v1_blk.ag = a.AG ? a.AG + (size_t)blockIdx.x * GS * M.Ppad : nullptr;
        v1_blk.drift = 0.f; v1_blk.since = 0; v1_blk.momflag = 0; v1_blk.nfresh = 0; v1_blk.stepmax = 0; v1_blk.failmask = 0u;
        v1_blk.t = 0;
    }
    if (M.L <= 4) {   // one word per term (v1_param_setup)
        for (int k = threadIdx.x; k < M.K; k += blockDim.x) {
            unsigned w = 0;
            for (int l = 0; l < M.L; ++l) w |= (unsigned)M.exps[k * M.L + l] << (8 * l);
            ((unsigned *)(V1SM + L.oEXP))[k] = w;
        }
    } else
        for (int i = threadIdx.x; i < M.K * M.L; i += blockDim.x) ((uint8_t *)(V1SM + L.oEXP))[i] = M.exps[i];
    if (M.n_models)
        for (int k = threadIdx.x; k < M.K; k += blockDim.x) ((uint8_t *)(V1SM + L.oTM))[k] = M.term_model[k];
    for (int i = threadIdx.x; i < GS * L.Kq; i += blockDim.x) V1SM[L.oPHI + i] = 0.f;   // phi is zero past K
    // rows T and A: zero-weight taps multiply whatever lies in the window, so it must at least be finite
    // (streaming: one window buffer, oA == oT, and the global rows, which may hold another launch's values)
    for (int i = threadIdx.x; i < (L.oA == L.oT ? 1 : 2) * GS * L.RL; i += blockDim.x) V1SM[L.oT + i] = 0.f;
    if (a.TG) {
        float *tg = a.TG + (size_t)blockIdx.x * GS * M.Ppad, *ag = a.AG + (size_t)blockIdx.x * GS * M.Ppad;
        for (int i = threadIdx.x; i < GS * M.Ppad; i += blockDim.x) { tg[i] = 0.f; ag[i] = 0.f; }
    }
    for (int i = threadIdx.x; i < GS * (SC_N + M.n_seg); i += blockDim.x) V1SM[L.oSC + i] = 0.f;
    __syncthreads();
}

__device__ __forceinline__ void v1_set_group(int grp)
{
    if (threadIdx.x < GS) {
        const long long i = (long long)grp * GS + threadIdx.x;
        v1_blk.spec[threadIdx.x] = i < v1_blk.A.B ? i : v1_blk.A.B - 1;
    }
    if (threadIdx.x == 0) {
        v1_blk.drift = 0.f; v1_blk.since = 0; v1_blk.momflag = 0; v1_blk.nfresh = 0; v1_blk.stepmax = 0; v1_blk.failmask = 0u;
        v1_blk.t = 0;
    }
}

// Jacobian of the re-solved whitened residual rho(u) by central differences of step fd_h in u (C.2-22):
// planes 1 .. NP of `xj` receive J_p on the fitted pixels (plane 0 is scratch).  `fresh_first`: the first of the 2 NP
// evaluations re-factorises whatever the fd_fresh option says (the LM loop calls this after a rejected trial step,
// when the factor and the warm start belong to another point).
template <bool STREAM>
__device__ __noinline__ void v1_jacobian(float *xj, bool fresh_first)
{
    const V1Args &a = v1_blk.A;
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int NP = M.NP;
    const size_t plane = (size_t)GS * M.Ppad;
    for (int p = 0; p < NP; ++p) {
        float u0 = 0.f;
        if (V1_WARP < GS) {
            u0 = SMV(L.oU, p, V1_WARP);
            __syncwarp();
            if (V1_LANE == 0) SMV(L.oU, p, V1_WARP) = u0 + a.fd_h;
            __syncwarp();
            v1_param_setup(V1_WARP);
        }
        // The factor of the final evaluation serves all 2 NP perturbed ones: a step of fd_h changes the Gram matrix
        // by a relative ~1e-3, so one refinement from the neighbouring solution leaves that fraction of the
        // continuum's response, far inside the 1e-2 the estimate is held to.
        v1_evaluate<2, STREAM>(false, (a.fdfresh != 0 || (fresh_first && p == 0)) ? 1 : 0, xj);
        if (V1_WARP < GS) {
            if (V1_LANE == 0) SMV(L.oU, p, V1_WARP) = u0 - a.fd_h;
            __syncwarp();
            v1_param_setup(V1_WARP);
        }
        v1_evaluate<2, STREAM>(false, a.fdfresh != 0, xj + (1 + p) * plane);
        if (V1_WARP < GS) {
            if (V1_LANE == 0) SMV(L.oU, p, V1_WARP) = u0;
            __syncwarp();
        }
        __syncthreads();
        // J_p = (rho+ - rho-)/(u+ - u-) on the pixels this thread owns (it wrote both)
        for (int s = 0; s < M.n_seg; ++s) {
            const SegDev &sg = M.seg[s];
            for (int j0 = sg.fit_lo + V1_TID * OCT; j0 < sg.fit_hi; j0 += V1_NT * OCT)
                for (int g = 0; g < GS; ++g) {
                    const float uu = SMV(L.oU, p, g);
                    const float inv = 1.f / ((uu + a.fd_h) - (uu - a.fd_h));
                    float4 *jp = (float4 *)(xj + (1 + p) * plane + (size_t)g * M.Ppad + j0);
                    const float4 *xp = (const float4 *)(xj + (size_t)g * M.Ppad + j0);
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        const float4 x = xp[h], m = jp[h];
                        jp[h] = make_float4((x.x - m.x) * inv, (x.y - m.y) * inv, (x.z - m.z) * inv, (x.w - m.w) * inv);
                    }
                }
        }
        __syncthreads();
    }
}

// N = X^T X (packed lower, N[g * npair + p (p + 1) / 2 + q]) of the first `ncol` columns X_p = plane 1 + p of `xj`, fp64
// accumulation across warps in shared memory (the factor area: the next evaluation that needs a factor re-factorises).
// ncol = NP: J^T J;  ncol = NP + 1 with rho(u) in plane 1 + NP: also J^T rho (row NP) and |rho|^2.
template <bool STREAM>
__device__ __noinline__ void v1_normal_eq(const float *xj, int ncol)
{
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const size_t plane = (size_t)GS * M.Ppad;
    double *N = (double *)(V1SM + L.oLF);
    const int npair = ncol * (ncol + 1) / 2;
    for (int i = V1_TID; i < GS * npair; i += V1_NT) N[i] = 0.0;
    __syncthreads();
    for (int s = 0; s < M.n_seg; ++s) {
        const SegDev &sg = M.seg[s];
        for (int jb = sg.fit_lo; jb < sg.fit_hi; jb += V1_NT * OCT) {
            const int j0 = jb + V1_TID * OCT;
            const bool act = j0 < sg.fit_hi;
            for (int pi0 = 0; pi0 < npair; pi0 += 8) {
                float X[32];
#pragma unroll
                for (int kk = 0; kk < 8; ++kk) {
                    const int pi = pi0 + kk;
                    int p = 0;
                    while ((p + 1) * (p + 2) / 2 <= pi) ++p;
                    const int q = pi - p * (p + 1) / 2;
#pragma unroll
                    for (int g = 0; g < GS; ++g) {
                        float sacc = 0.f;
                        if (act && pi < npair) {
                            const float4 *A4 = (const float4 *)(xj + (1 + p) * plane + (size_t)g * M.Ppad + j0);
                            const float4 *B4 = (const float4 *)(xj + (1 + q) * plane + (size_t)g * M.Ppad + j0);
                            const float4 a0 = A4[0], a1 = A4[1], b0 = B4[0], b1 = B4[1];
                            sacc = a0.x * b0.x + a0.y * b0.y + a0.z * b0.z + a0.w * b0.w +
                                   a1.x * b1.x + a1.y * b1.y + a1.z * b1.z + a1.w * b1.w;
                        }
                        X[kk * 4 + g] = sacc;
                    }
                }
                const float tot = xreduce32(X, V1_LANE);
                const int pi = pi0 + (V1_LANE >> 2);
                if (pi < npair) atomicAdd(&N[(V1_LANE & 3) * npair + pi], (double)tot);
            }
        }
    }
    __syncthreads();
}

// a9: error estimate (C.2-22/23).  J by central differences of the re-solved whitened
// residual rho(u), Sigma = rho^T rho/(N_good - NP) (J^T J)^-1, err_p = sqrt(Sigma_pp) (hi_p - lo_p)/2.
template <bool STREAM>
__device__ __noinline__ void v1_errors(float chi2_g, float ngood_g, bool valid_g)
{
    const V1Args &a = v1_blk.A;
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int NP = M.NP;
    const size_t plane = (size_t)GS * M.Ppad;
    float *xj = a.XJ + (size_t)blockIdx.x * (2 + NP) * plane;
    v1_jacobian<STREAM>(xj, false);
    v1_normal_eq<STREAM>(xj, NP);
    double *N = (double *)(V1SM + L.oLF);
    const int npair = NP * (NP + 1) / 2;
    if (V1_WARP < GS && V1_LANE == 0) {
        const int g = V1_WARP;
        double *Ng = N + g * npair;
        bool ok = ngood_g > (float)NP;
        for (int p = 0; p < NP && ok; ++p)
            for (int q = 0; q <= p; ++q) {
                double s = Ng[p * (p + 1) / 2 + q];
                for (int k = 0; k < q; ++k) s -= Ng[p * (p + 1) / 2 + k] * Ng[q * (q + 1) / 2 + k];
                if (p == q) {
                    if (!(s > 0.0)) { ok = false; break; }
                    Ng[p * (p + 1) / 2 + p] = sqrt(s);
                } else
                    Ng[p * (p + 1) / 2 + q] = s / Ng[q * (q + 1) / 2 + q];
            }
        const double s2 = (double)chi2_g / ((double)ngood_g - (double)NP);
        for (int p = 0; p < NP; ++p) {
            float e = __int_as_float(0x7fc00000);
            if (ok) {   // (J^T J)^-1_pp = |L^-1 e_p|^2
                double y[LASP_NPMAX];
                double nrm = 0.0;
                for (int r = p; r < NP; ++r) {
                    double s = (r == p) ? 1.0 : 0.0;
                    for (int k = p; k < r; ++k) s -= Ng[r * (r + 1) / 2 + k] * y[k];
                    y[r] = s / Ng[r * (r + 1) / 2 + r];
                    nrm += y[r] * y[r];
                }
                e = (float)(sqrt(s2 * nrm) * (double)(M.hi[p] - M.lo[p]) * 0.5);
            }
            if (valid_g) a.err[v1_blk.spec[g] * NP + p] = e;
        }
    }
    __syncthreads();
}

// ------------------------------------------------------------------------------------------
// Levenberg-Marquardt on the NP x NP system (reading R-13 of DESIGN.md, as
// oracle/lasp_oracle.c orc_fit_lm): one iteration = the Jacobian of the re-solved whitened residual (2 NP evaluations),
// the normal equations in fp64, the damped step (A + lambda diag A) delta = -g by Cholesky on lane 0 of the
// spectrum's warp, one trial evaluation, and the accept / reject decision per spectrum.
// Planes of xj: 0 trial residual / scratch, 1 .. NP the Jacobian, 1 + NP the residual at the current iterate.
// ------------------------------------------------------------------------------------------
template <bool STREAM>
__device__ __noinline__ void v1_lm_iteration(float *xj)
{
    const V1Args &a = v1_blk.A;
    const ModelDev &M = v1_blk.M;
    const V1Lay &L = v1_blk.L;
    const int NP = M.NP, g = V1_WARP;
    const size_t plane = (size_t)GS * M.Ppad;
    v1_jacobian<STREAM>(xj, true);
    v1_normal_eq<STREAM>(xj, NP + 1);
    if (g < GS) {
        if (V1_LANE == 0) {
            const int npair = (NP + 1) * (NP + 2) / 2;
            double *Ng = (double *)(V1SM + L.oLF) + g * npair;
            const double lam = (double)v1_blk.lm_lambda[g];
            double d[LASP_NPMAX];
            bool ok = true;
            for (int p = 0; p < NP; ++p) Ng[p * (p + 1) / 2 + p] *= 1.0 + lam;
            for (int p = 0; p < NP && ok; ++p)
                for (int q = 0; q <= p; ++q) {
                    double s = Ng[p * (p + 1) / 2 + q];
                    for (int k = 0; k < q; ++k) s -= Ng[p * (p + 1) / 2 + k] * Ng[q * (q + 1) / 2 + k];
                    if (p == q) {
                        if (!(s > 0.0)) { ok = false; break; }
                        Ng[p * (p + 1) / 2 + p] = sqrt(s);
                    } else
                        Ng[p * (p + 1) / 2 + q] = s / Ng[q * (q + 1) / 2 + q];
                }
            if (ok) {
                const double *gr = Ng + NP * (NP + 1) / 2;   // row NP: J^T rho
                for (int p = 0; p < NP; ++p) {               // L z = -g
                    double s = -gr[p];
                    for (int k = 0; k < p; ++k) s -= Ng[p * (p + 1) / 2 + k] * d[k];
                    d[p] = s / Ng[p * (p + 1) / 2 + p];
                }
                for (int p = NP - 1; p >= 0; --p) {          // L^T delta = z
                    double s = d[p];
                    for (int k = p + 1; k < NP; ++k) s -= Ng[k * (k + 1) / 2 + p] * d[k];
                    d[p] = s / Ng[p * (p + 1) / 2 + p];
                }
            }
            for (int p = 0; p < NP; ++p) {
                const float u0 = SMV(L.oU, p, g);
                SMV(L.oM, p, g) = u0;                        // the Adam moments are not used here: the iterate to fall back to
                float u = ok ? (float)((double)u0 + d[p]) : u0;
                u = u < -1.f ? -1.f : (u > 1.f ? 1.f : u);
                SMV(L.oU, p, g) = u;
            }
        }
        __syncwarp();
        v1_param_setup(g);
    }
    v1_evaluate<2, STREAM>(false, 1, xj);
    if (g < GS) {
        float c2t, ngood, cmin;
        v1_stats(g, c2t, ngood, cmin);
        const bool acc = c2t < v1_blk.lm_chi2[g];            // NaN: rejected
        __syncwarp();
        if (V1_LANE == 0) {
            v1_blk.lm_acc[g] = acc ? 1 : 0;
            if (acc) {
                v1_blk.lm_chi2[g] = c2t;
                v1_blk.lm_lambda[g] = fmaxf(v1_blk.lm_lambda[g] * 0.1f, 1e-10f);
                v1_blk.nsteps[g] += 1;
            } else {
                v1_blk.lm_lambda[g] = fminf(v1_blk.lm_lambda[g] * 10.f, 1e10f);
                for (int p = 0; p < NP; ++p) SMV(L.oU, p, g) = SMV(L.oM, p, g);
            }
        }
        __syncwarp();
        if (!acc) v1_param_setup(g);
    }
    __syncthreads();
    // the accepted trial residuals become the residual at the iterate
    for (int g2 = 0; g2 < GS; ++g2) {
        if (!v1_blk.lm_acc[g2]) continue;
        for (int s = 0; s < M.n_seg; ++s) {
            const SegDev &sg = M.seg[s];
            const float4 *src = (const float4 *)(xj + (size_t)g2 * M.Ppad);
            float4 *dst = (float4 *)(xj + (1 + NP) * plane + (size_t)g2 * M.Ppad);
            for (int q = (sg.fit_lo >> 2) + V1_TID; q < (sg.fit_hi >> 2); q += V1_NT) dst[q] = src[q];
        }
    }
    __syncthreads();
}

// ------------------------------------------------------------------------------------------
// One evaluation of the Adam loop in the common case -- ONE uniform (log-grid) segment, warm start, the kernel weights
// already prepared by v1_update_fast -- as a straight line of phase calls that keeps NOTHING alive across them: what a
// later phase needs (the re-factorisation flag, whether statistics are wanted) is re-read from the block state.  In the
// general v1_evaluate every value kept across a call is spilled to local memory and reloaded behind it, a round trip
// that misses the small L1 and sits on the critical path six times per step (profiles/r02_ncu.md).
// ------------------------------------------------------------------------------------------
template <bool STREAM>
__device__ __noinline__ void v1_step_hot(int momsel)
{
    __syncthreads();
    v1_begin_eval(momsel, true);
    v1_phase_emulator<STREAM, !STREAM>(0, 0);
    __syncthreads();
    v1_phase_forward<true, STREAM>(0, true);
    if (v1_blk.momflag != 0) v1_phase_moments<STREAM>(0);
    __syncthreads();
    if (V1_WARP < GS) v1_phase_solve(V1_WARP, 0, v1_blk.momflag != 0);
    __syncthreads();
    if (v1_blk.A.stop_window > 0) v1_phase_residual<1, true, STREAM>(0, nullptr);   // stopping rules read chi2
    else v1_phase_residual<3, true, STREAM>(0, nullptr);
    __syncthreads();
    v1_phase_adjoint<true, STREAM, !STREAM>(0);
    __syncthreads();
}

// ------------------------------------------------------------------------------------------
// Clean-strategy mask update (step 6, Eq. 8; the schedule of P:171), readings R-7..R-12 of DESIGN.md as
// oracle/lasp_oracle.c orc_clean_update states them.  One resident segment whose fitted range is one sweep of the
// CTA: thread t owns octet t of the fitted range and keeps eps, the excess and its flags in registers; neighbours
// across octets are read from row T, which holds eps_j for the pixels clipped so far by this update and 0 elsewhere.
// On entry (after v1_evaluate<4>) row A holds eps = sqrt(w) r and row T the corrected model M = c S at the current
// iterate.  The decisions (sigma, thresholds) are taken in double from the float residuals.  Clipped pixels get w = 0
// in the staged weight plane, for good (R-9); the next Adam step re-factorises the Gram matrix.
// ------------------------------------------------------------------------------------------
template <int NV>
__device__ __forceinline__ void v1_block_sum(double (&x)[NV][GS])
{
    const V1Lay &L = v1_blk.L;
    // the Q slots of the reduction area are free between an evaluation and the next one's first barrier
    double *red = (double *)(V1SM + L.oRED + (L.nmomr + L.n1r) * GS);
    const int wst = L.VR * GS / 2;
#pragma unroll
    for (int v = 0; v < NV; ++v)
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            double s = x[v][g];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(FULL, s, o);
            if (V1_LANE == 0) red[V1_WARP * wst + v * GS + g] = s;
        }
    __syncthreads();
#pragma unroll
    for (int v = 0; v < NV; ++v)
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            double s = 0.0;
            for (int w = 0; w < L.NW; ++w) s += red[w * wst + v * GS + g];
            x[v][g] = s;
        }
    __syncthreads();
}

__device__ __forceinline__ float v1_row_elem(const float *rowsm, int g, int jp)
{
    const float4 *p = (const float4 *)(rowsm + g * v1_blk.L.RL);
    return ((const float *)&p[SW4(jp >> 2)])[jp & 3];
}

// population standard deviation of eps over the pixels flagged in `use` (bit g*8+i), per spectrum (R-8)
__device__ __forceinline__ void v1_clean_sigma(const float (&eps)[GS][OCT], unsigned use, double (&sigma)[GS], double (&n)[GS])
{
    double s[2][GS];
#pragma unroll
    for (int g = 0; g < GS; ++g) {
        s[0][g] = 0.0; s[1][g] = 0.0;
#pragma unroll
        for (int i = 0; i < OCT; ++i)
            if ((use >> (g * OCT + i)) & 1u) { s[0][g] += (double)eps[g][i]; s[1][g] += 1.0; }
    }
    v1_block_sum<2>(s);
    double d[1][GS];
#pragma unroll
    for (int g = 0; g < GS; ++g) {
        n[g] = s[1][g];
        const double mean = n[g] > 0.0 ? s[0][g] / n[g] : 0.0;
        d[0][g] = 0.0;
#pragma unroll
        for (int i = 0; i < OCT; ++i)
            if ((use >> (g * OCT + i)) & 1u) { const double e = (double)eps[g][i] - mean; d[0][g] += e * e; }
    }
    v1_block_sum<1>(d);
#pragma unroll
    for (int g = 0; g < GS; ++g) sigma[g] = n[g] > 0.0 ? sqrt(d[0][g] / n[g]) : 0.0;
}

__device__ __noinline__ void v1_clean_update(float fshift)
{
    const SegDev &sg = v1_blk.M.seg[0];
    const V1Lay &L = v1_blk.L;
    const int Ppad = v1_blk.M.Ppad, P8 = Ppad >> 3;
    const int j0 = sg.fit_lo + V1_TID * OCT;
    const bool act = j0 < sg.fit_hi;
    const int r0 = j0 - (sg.po + sg.halo);   // real index of this octet's first pixel
    float *rowA = v1_rowp(L.oA, sg.po), *rowT = v1_rowp(L.oT, sg.po);
    float *Wg = const_cast<float *>(v1_blk.A.W);
    float eps[GS][OCT], exc[GS][OCT];
    unsigned U = 0u, O = 0u;   // bit g * 8 + i
#pragma unroll
    for (int g = 0; g < GS; ++g) {
#pragma unroll
        for (int i = 0; i < OCT; ++i) { eps[g][i] = 0.f; exc[g][i] = 0.f; }
        if (!act) continue;
        float Mv[OCT + 2], ww[OCT];
        {
            float m8[OCT];
            v1_oct_load<false>(rowA, nullptr, g, j0, eps[g]);
            v1_oct_load<false>(rowT, nullptr, g, j0, m8);
            Mv[0] = v1_row_elem(rowT, g, j0 - 1);
            Mv[OCT + 1] = v1_row_elem(rowT, g, j0 + OCT);
#pragma unroll
            for (int i = 0; i < OCT; ++i) Mv[i + 1] = m8[i];
            const float4 *w4 = (const float4 *)(Wg + (size_t)v1_blk.spec[g] * Ppad + (j0 >> 1));
            const float4 w0 = __ldcg(w4), w1 = __ldcg(w4 + P8);
            ww[0] = w0.x; ww[1] = w0.y; ww[2] = w0.z; ww[3] = w0.w; ww[4] = w1.x; ww[5] = w1.y; ww[6] = w1.z; ww[7] = w1.w;
        }
#pragma unroll
        for (int i = 0; i < OCT; ++i) {
            const int jr = r0 + i;
            float gm = 0.f;   // R-7: only the neighbour that exists at a segment end
            if (jr >= 1) gm = fabsf(Mv[i + 1] - Mv[i]);
            if (jr + 1 < sg.P) gm = fmaxf(gm, fabsf(Mv[i + 1] - Mv[i + 2]));
            if (ww[i] > 0.f) U |= 1u << (g * OCT + i);
            exc[g][i] = fabsf(eps[g][i]) - fshift * sqrtf(ww[i]) * gm;
        }
    }
    double sigma[GS], nU[GS];
    v1_clean_sigma(eps, U, sigma, nU);      // (its barriers also end every thread's reads of M in row T)
    // B (R-10): k = 3, escalated to 4, 5, 7 while more than 3 % of U would be clipped
    double cnt[4][GS];
    const double ks[4] = {3.0, 4.0, 5.0, 7.0};
#pragma unroll
    for (int t = 0; t < 4; ++t)
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            cnt[t][g] = 0.0;
#pragma unroll
            for (int i = 0; i < OCT; ++i)
                if (((U >> (g * OCT + i)) & 1u) && (double)exc[g][i] > ks[t] * sigma[g]) cnt[t][g] += 1.0;
        }
    v1_block_sum<4>(cnt);
#pragma unroll
    for (int g = 0; g < GS; ++g) {
        double kk = 7.0;
        if (cnt[0][g] <= 0.03 * nU[g]) kk = 3.0;
        else if (cnt[1][g] <= 0.03 * nU[g]) kk = 4.0;
        else if (cnt[2][g] <= 0.03 * nU[g]) kk = 5.0;
#pragma unroll
        for (int i = 0; i < OCT; ++i)
            if (((U >> (g * OCT + i)) & 1u) && (double)exc[g][i] > kk * sigma[g]) O |= 1u << (g * OCT + i);
    }
    // row T <- eps of the clipped pixels, 0 elsewhere (guards and the rest of the row included)
    for (int i = V1_TID; i < GS * L.RL / 4; i += V1_NT) ((float4 *)(V1SM + L.oT))[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    __syncthreads();
    auto publish = [&]() {
        if (!act) return;
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            float f[OCT];
#pragma unroll
            for (int i = 0; i < OCT; ++i) f[i] = ((O >> (g * OCT + i)) & 1u) ? eps[g][i] : 0.f;
            v1_oct_store<false>(rowT, nullptr, g, j0, f);
        }
    };
    // flags of the octet's pixels and of the two pixels beside it
    auto flags = [&](int g, float (&f)[OCT + 2]) {
        f[0] = v1_row_elem(rowT, g, j0 - 1);
        f[OCT + 1] = v1_row_elem(rowT, g, j0 + OCT);
#pragma unroll
        for (int i = 0; i < OCT; ++i) f[i + 1] = ((O >> (g * OCT + i)) & 1u) ? eps[g][i] : 0.f;
    };
    publish();
    __syncthreads();
    // C (R-11): neighbours of B with excess > 2 sigma
    {
        unsigned add = 0u;
        if (act) {
#pragma unroll
            for (int g = 0; g < GS; ++g) {
                float f[OCT + 2];
                flags(g, f);
#pragma unroll
                for (int i = 0; i < OCT; ++i) {
                    const unsigned bit = 1u << (g * OCT + i);
                    if ((U & bit) && !(O & bit) && (f[i] != 0.f || f[i + 2] != 0.f) && (double)exc[g][i] > 2.0 * sigma[g]) add |= bit;
                }
            }
        }
        __syncthreads();   // every thread has read the B flags
        O |= add;
        publish();
        __syncthreads();
    }
    double sigma2[GS], n2[GS];
    v1_clean_sigma(eps, U & ~O, sigma2, n2);
    // D (R-12): synchronous growth along same-sign, non-increasing |eps| with excess > sigma', at most 20 rounds
    for (int it = 0; it < 20; ++it) {
        unsigned add = 0u;
        if (act) {
#pragma unroll
            for (int g = 0; g < GS; ++g) {
                float f[OCT + 2];
                flags(g, f);
#pragma unroll
                for (int i = 0; i < OCT; ++i) {
                    const unsigned bit = 1u << (g * OCT + i);
                    if (!(U & bit) || (O & bit) || !((double)exc[g][i] > sigma2[g])) continue;
                    const float e = eps[g][i], l = f[i], r = f[i + 2];
                    if ((l != 0.f && l * e > 0.f && fabsf(e) <= fabsf(l)) || (r != 0.f && r * e > 0.f && fabsf(e) <= fabsf(r))) add |= bit;
                }
            }
        }
        const int changed = __syncthreads_or(add != 0u);   // also: every thread has read this round's flags
        O |= add;
        if (add) publish();
        __syncthreads();
        if (!changed) break;
    }
    // R-9: the clipped pixels leave the fit for good
    if (act && O) {
#pragma unroll
        for (int g = 0; g < GS; ++g) {
            if (!((O >> (g * OCT)) & 0xffu) || v1_blk.stop_rule[g] != 0) continue;   // a stopped spectrum keeps its mask
            float4 *w4 = (float4 *)(Wg + (size_t)v1_blk.spec[g] * Ppad + (j0 >> 1));
            float4 w0 = __ldcg(w4), w1 = __ldcg(w4 + P8);
            const unsigned o = O >> (g * OCT);
            if (o & 1u) w0.x = 0.f;  if (o & 2u) w0.y = 0.f;  if (o & 4u) w0.z = 0.f;  if (o & 8u) w0.w = 0.f;
            if (o & 16u) w1.x = 0.f; if (o & 32u) w1.y = 0.f; if (o & 64u) w1.z = 0.f; if (o & 128u) w1.w = 0.f;
            w4[0] = w0; w4[P8] = w1;
        }
    }
    if (V1_TID == 0) { v1_blk.force = 1; v1_blk.nclean += 1; }
    __syncthreads();
}

// ------------------------------------------------------------------------------------------
// The paper's stopping rules (step 8), per spectrum (Delta-2), warp g for spectrum g, called after the t-th
// evaluation and before update t (readings R-2..R-5 of DESIGN.md, as oracle/lasp_oracle.c orc_fit_stop):
//   loss L_t = sqrt(chi2_t / n_pix) (Eq. 9 restricted to one spectrum);
//   (2) |L_t - L_{t-W}| < tol, testable from t = W + 1;  (3) W consecutive increases;  (2) is tested first.
// Returns true (warp-uniform) when the spectrum goes on and update t is to be applied.  A spectrum that stops keeps
// its iterate: the group runs on until all its spectra have stopped (or max_iter), the stopped ones frozen.
// ------------------------------------------------------------------------------------------
__device__ __noinline__ bool v1_stop_test(int g, int t)
{
    const V1Args &a = v1_blk.A;
    if (v1_blk.stop_rule[g] != 0) return false;
    float chi2, ngood, cmin;
    v1_stats(g, chi2, ngood, cmin);
    const float Lt = sqrtf(chi2 / (float)v1_blk.M.P);
    int rule = 0;
    if (V1_LANE == 0) {
        const int W = a.stop_window, slot = t % W;
        float *h = V1SM + v1_blk.L.oHIST + g * W;
        const int rise = (t > 1 && Lt > v1_blk.lprev[g]) ? v1_blk.rise[g] + 1 : 0;
        if (t > W && fabsf(Lt - h[slot]) < a.stop_tol) rule = 2;      // h[slot] still holds L_(t-W)
        else if (rise >= W) rule = 3;
        h[slot] = Lt;
        v1_blk.rise[g] = rise;
        v1_blk.lprev[g] = Lt;
        if (rule) { v1_blk.stop_rule[g] = rule; v1_blk.nsteps[g] = t - 1; }
    }
    rule = __shfl_sync(FULL, rule, 0);
    return rule == 0;
}

// ------------------------------------------------------------------------------------------
// lasp_fit_batch: a1-a9 for groups of GS spectra, persistent CTAs
// ------------------------------------------------------------------------------------------
// The Clean-strategy mask updates (resident variant only) and the LM loop live in instantiations of their own: the default
// one carries none of that code (the step path is instruction-cache bound, profiles/r02_ncu.md).
// OPT 0: Adam;  1: Adam with the Clean-strategy mask updates;  2: Levenberg-Marquardt (n_iter LM iterations)
template <int MAXT, int MINB, bool STREAM, int OPT = 0>
__global__ void __launch_bounds__(MAXT, MINB)
lasp_v1_fit_kernel(const __grid_constant__ ModelDev M, const __grid_constant__ V1Lay L, const V1Args a)
{
    v1_init_block(M, L, a);
    const int NP = M.NP, g = V1_WARP;
    // groups are handed out by a global counter (the first gridDim.x statically): fits differ a little in length
    // (kernel supports, early cold steps), and the last wave would otherwise leave SMs idle
    for (int grp = blockIdx.x; grp < a.ngroups;) {
        __syncthreads();   // the previous group's last readers (output writers included) are done with the block state
        v1_set_group(grp);
        if (threadIdx.x == 0) v1_blk.next = a.queue ? (int)gridDim.x + (int)atomicAdd(a.queue, 1u) : grp + (int)gridDim.x;
        __syncthreads();
        const int grp_next = v1_blk.next;
        const bool valid = g < GS && (long long)grp * GS + g < a.B;
        if (g < GS) {
            for (int p = V1_LANE; p < NP; p += 32) {
                const float th = a.init[v1_blk.spec[g] * NP + p];
                SMV(L.oU, p, g) = 2.f * (th - M.lo[p]) / (M.hi[p] - M.lo[p]) - 1.f;   // not clipped: clipping follows updates (C.1)
                SMV(L.oM, p, g) = 0.f;
                SMV(L.oV, p, g) = 0.f;
            }
            __syncwarp();
            v1_param_setup(g);
        }
        const bool stopmode = a.stop_window > 0;
        if (threadIdx.x < GS) {
            v1_blk.stop_rule[threadIdx.x] = 0; v1_blk.nsteps[threadIdx.x] = a.n_iter;
            v1_blk.rise[threadIdx.x] = 0; v1_blk.lprev[threadIdx.x] = 0.f;
            v1_blk.force = 0; v1_blk.nclean = 0;
            SMV(L.oSC, SC_PB1, threadIdx.x) = 1.f; SMV(L.oSC, SC_PB2, threadIdx.x) = 1.f;
        }
        if constexpr (OPT == 2) {
            float *xj = a.XJ + (size_t)blockIdx.x * (2 + NP) * GS * M.Ppad;
            v1_evaluate<2, STREAM>(true, 1, xj + (size_t)(1 + NP) * GS * M.Ppad);   // rho at the initial guess
            if (g < GS) {
                float c2, ngood, cmin;
                v1_stats(g, c2, ngood, cmin);
                if (V1_LANE == 0) { v1_blk.lm_chi2[g] = c2; v1_blk.lm_lambda[g] = a.lm_lambda0; v1_blk.nsteps[g] = 0; }
            }
            for (;;) {
                __syncthreads();
                if (v1_blk.t >= a.n_iter) break;
                __syncthreads();
                if (V1_TID == 0) v1_blk.t += 1;
                v1_lm_iteration<STREAM>(xj);
            }
        } else
        // v1_blk.t was zeroed by v1_set_group; every evaluation below starts with a barrier, after which thread 0 advances
        // it, and ends with one, after which it is read again
        for (;;) {
            const int t = *(volatile int *)&v1_blk.t + 1;
            if (t > a.n_iter) break;
#ifdef LASP_PHASE_TIMING
            const long long te0 = a.dbg ? clock64() : 0;
#endif
            // fresh Gram factor on each of the first `warm` steps (the model moves fastest there), then every `refresh`-th
            // step, or (refresh == 0) when the drift monitor asks for it
            const int momsel = t <= a.warm ? 1 : (a.refresh >= 1 ? ((t - 1) % a.refresh == 0 ? 1 : 0) : 2);
            if (t > 1 && L.fastw && !a.CF) v1_step_hot<STREAM>(momsel);
            else v1_evaluate<0, STREAM>(t == 1, momsel, nullptr, t > 1 && L.fastw, stopmode, true);
#ifdef LASP_PHASE_TIMING
            if (a.dbg && V1_TID == 0) { atomicAdd(a.dbg + 14, (unsigned long long)(clock64() - te0)); atomicAdd(a.dbg + 15, 1ull); }
            const long long tu0 = a.dbg ? clock64() : 0;
#endif
            bool upd = V1_WARP < GS;
            if (stopmode && upd) upd = v1_stop_test(V1_WARP, *(volatile int *)&v1_blk.t);     // a stopped spectrum keeps its iterate
            if (upd) {
                const int g = V1_WARP;
                const float pb1 = SMV(L.oSC, SC_PB1, g) * a.b1, pb2 = SMV(L.oSC, SC_PB2, g) * a.b2;   // beta^t of this spectrum
                __syncwarp();
                if (V1_LANE == 0) { SMV(L.oSC, SC_PB1, g) = pb1; SMV(L.oSC, SC_PB2, g) = pb2; }
                const float ib1 = 1.f / (1.f - pb1), ib2 = 1.f / (1.f - pb2);   // bias corrections (C.2-20)
                if (L.fastupd) v1_update_fast(g, ib1, ib2);
                else {
                    const float gr = v1_gradient(g);
#ifdef LASP_PHASE_TIMING
                    if (a.dbg && V1_TID == 0) atomicAdd(a.dbg + 16, (unsigned long long)(clock64() - tu0));
#endif
                    // a8: Adam (C.2-20), then clip to the prior box (C.2-18); lane p owns parameter p
                    float du = 0.f;
                    for (int p0 = 0; p0 < NP; p0 += 32) {   // NP <= 32
                        const int p = p0 + V1_LANE;
                        if (p < NP) {
                            const float m = a.b1 * SMV(L.oM, p, g) + (1.f - a.b1) * gr;
                            const float v = a.b2 * SMV(L.oV, p, g) + (1.f - a.b2) * gr * gr;
                            SMV(L.oM, p, g) = m; SMV(L.oV, p, g) = v;
                            const float mh = m * ib1, vh = v * ib2;
                            const float u0 = SMV(L.oU, p, g);
                            float u = u0 - __fdividef(a.lr * mh, sqrtf(vh) + a.eps);
                            u = u < -1.f ? -1.f : (u > 1.f ? 1.f : u);   // clip (C.2-18); NaN stays NaN, as in the oracle
                            SMV(L.oU, p, g) = u;
                            du = fabsf(u - u0);
                        }
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) du = fmaxf(du, __shfl_xor_sync(FULL, du, o));
                    if (V1_LANE == 0) atomicMax(&v1_blk.stepmax, __float_as_int(du));   // re-factorisation monitor
                    __syncwarp();
#ifdef LASP_PHASE_TIMING
                    if (a.dbg && V1_TID == 0) atomicAdd(a.dbg + 17, (unsigned long long)(clock64() - tu0));
#endif
                    v1_param_setup(g);
                }
            }
#ifdef LASP_PHASE_TIMING
            if (a.dbg && V1_TID == 0) atomicAdd(a.dbg + 13, (unsigned long long)(clock64() - tu0));
#endif
            if constexpr (OPT == 1 && !STREAM) {
                if (a.clean_every > 0) {   // Clean: mask update after update t, t = every, 2 every, ...
                    __syncthreads();
                    if (v1_blk.t % a.clean_every == 0 && v1_blk.nclean < a.clean_max) {
                        v1_evaluate<4, false>(false, 1, nullptr, L.fastw != 0);   // residuals at the new iterate, re-solved
                        v1_clean_update(v1_blk.nclean == 0 ? 0.5f : 0.2f);       // f_shift
                    }
                }
            }
            if (stopmode) {   // the group ends when every spectrum of it has stopped
                __syncthreads();
                bool all = true;
#pragma unroll
                for (int q = 0; q < GS; ++q) all = all && v1_blk.stop_rule[q] != 0;
                if (all) break;
            }
        }
        if (a.stats && V1_TID == 0) { atomicAdd(a.stats, (unsigned long long)v1_blk.t); atomicAdd(a.stats + 1, (unsigned long long)v1_blk.nfresh); }
        // a9: one more evaluation at the final iterate (C.2-21)
        v1_evaluate<1, STREAM>(OPT != 2 && a.n_iter == 0, 1, nullptr);
        float chi2 = 0.f, ngood = 0.f, cmin = 0.f;
        if (g < GS) {
            v1_stats(g, chi2, ngood, cmin);
            int st = 0;
            bool fin = isfinite(chi2);
            bool bound = false;
            for (int p = V1_LANE; p < NP; p += 32) {
                const float u = SMV(L.oU, p, g);
                fin = fin && isfinite(u);
                bound = bound || (u <= -1.f || u >= 1.f);
            }
            for (int n = V1_LANE; n < M.nc; n += 32) fin = fin && isfinite(SMV(L.oB, n, g));
            fin = __all_sync(FULL, fin);
            bound = __any_sync(FULL, bound);
            const bool anyfail = __any_sync(FULL, V1_LANE < M.n_seg && V1SM[L.oSC + (SC_N + V1_LANE) * GS + g] != 0.f);
            if (anyfail) st |= LASP_ST_NOT_SPD;
            if (bound) st |= LASP_ST_ON_BOUND;
            if (!fin) st |= LASP_ST_NONFINITE;
            if (ngood > 0.f && cmin <= 0.f) st |= LASP_ST_NEG_CONT;
            if (v1_blk.stop_rule[g] == 2) st |= LASP_ST_STOP_TOL;
            if (v1_blk.stop_rule[g] == 3) st |= LASP_ST_STOP_RISE;
            if (valid) {
                const long long i = v1_blk.spec[g];
                for (int p = V1_LANE; p < NP; p += 32)
                    a.params[i * NP + p] = M.lo[p] + (SMV(L.oU, p, g) + 1.f) * (M.hi[p] - M.lo[p]) * 0.5f;
                if (V1_LANE == 0) {
                    a.chi2[i] = chi2;
                    if (a.status) a.status[i] = st;
                    if (a.nsteps) a.nsteps[i] = v1_blk.nsteps[g];
                }
                if (a.cont) v1_write_cont(g, a.cont + i * M.nc);
            }
        }
        if (a.err) v1_errors<STREAM>(chi2, ngood, valid);
        if (a.mask_out) {   // the final mask: the staged weights are zero at the edges, at ivar * mask = 0 and where Clean clipped
            for (int g2 = 0; g2 < GS; ++g2) {
                if ((long long)grp * GS + g2 >= a.B) break;
                const float *wrow = a.W + (size_t)v1_blk.spec[g2] * M.Ppad;
                unsigned char *mrow = a.mask_out + (size_t)v1_blk.spec[g2] * M.P;
                for (int s = 0; s < M.n_seg; ++s) {
                    const SegDev &sg = M.seg[s];
                    for (int r = V1_TID; r < sg.P; r += V1_NT) {
                        const int jp = sg.po + sg.halo + r;
                        const float w = __ldcg(wrow + ((jp & 4) ? (M.Ppad >> 1) : 0) + (jp >> 3) * 4 + (jp & 3));
                        mrow[sg.o + r] = w != 0.f ? 1 : 0;
                    }
                }
            }
        }
        grp = grp_next;
    }
}

// ------------------------------------------------------------------------------------------
// lasp_eval_grad: one cold evaluation of chi2 and d chi2/d u at given physical parameters
// ------------------------------------------------------------------------------------------
template <int MAXT, int MINB, bool STREAM>
__global__ void __launch_bounds__(MAXT, MINB)
lasp_v1_grad_kernel(const __grid_constant__ ModelDev M, const __grid_constant__ V1Lay L, const V1Args a)
{
    v1_init_block(M, L, a);
    const int NP = M.NP, g = V1_WARP;
    for (int grp = blockIdx.x; grp < a.ngroups; grp += gridDim.x) {
        __syncthreads();   // the previous group's last readers (output writers included) are done with the block state
        v1_set_group(grp);
        __syncthreads();
        const bool valid = g < GS && (long long)grp * GS + g < a.B;
        if (g < GS) {
            for (int p = V1_LANE; p < NP; p += 32)
                SMV(L.oU, p, g) = 2.f * (a.gparams[v1_blk.spec[g] * NP + p] - M.lo[p]) / (M.hi[p] - M.lo[p]) - 1.f;
            __syncwarp();
            v1_param_setup(g);
        }
        v1_evaluate<0, STREAM>(true, 1, nullptr);
        if (g < GS) {
            const float gr = v1_gradient(g);
            float chi2, ngood, cmin;
            v1_stats(g, chi2, ngood, cmin);
            const bool anyfail = __any_sync(FULL, V1_LANE < M.n_seg && V1SM[L.oSC + (SC_N + V1_LANE) * GS + g] != 0.f);
            if (valid) {
                const long long i = v1_blk.spec[g];
                if (V1_LANE < NP) a.grad_u[i * NP + V1_LANE] = gr;
                if (V1_LANE == 0) {
                    a.chi2[i] = chi2;
                    if (a.status) a.status[i] = anyfail ? LASP_ST_NOT_SPD : 0;
                }
                if (a.cont) v1_write_cont(g, a.cont + i * M.nc);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------
// lasp_eval_model: model_j = c_j S_j at given physical parameters and plain-Legendre continuum coefficients, on
// EVERY pixel of every segment (edge pixels included: there the stencil reads the replicated halo, C.2-16).  S comes
// from the same emulator, weight and stencil code as the fit (v1_param_setup, v1_setup_weights, v1_phase_emulator,
// v1_stencil_octet / v1_np_forward_octet); the continuum is evaluated in the paper's own basis, Legendre P_n at the
// nodes x^_j = -1 + 2 (j - o_s)/P_s, by Bonnet's recurrence shared by the GS spectra.
// ------------------------------------------------------------------------------------------
template <bool UNI, bool STREAM>
__device__ __noinline__ void v1_phase_model(int s, int grp)
{
    const SegDev &sg = v1_blk.M.seg[s];
    const V1Args &a = v1_blk.A;
    const V1Lay &L = v1_blk.L;
    const int *tap = (const int *)(V1SM + L.oTAP);
    const int RL = L.RL, NA = L.NA, nt8 = V1_NT * OCT, n1 = v1_blk.M.n1, P = v1_blk.M.P;
    const int seg_lo = sg.po + sg.halo, seg_hi = seg_lo + (sg.P + OCT - 1) / OCT * OCT;
    const float *rowT = v1_rowp(L.oT, sg.po);
    const float4 *gw4 = (const float4 *)(V1SM + L.oGW);
    const float *bco = V1SM + L.oB + s * n1 * GS;
    const float *ISg = a.IS + V1_TPAD, *SJg = a.SJ + V1_TPAD;
    for (int jb = seg_lo; jb < seg_hi; jb += nt8) {   // uniform trip count
        const int j0 = jb + V1_TID * OCT;
        if (STREAM) {
            __syncthreads();
            v1_window_load(v1_blk.tg, jb);
            __syncthreads();
            rowT = v1_rowp(L.oT, jb);
        }
        if (j0 >= seg_hi) continue;
        // The continuum factor is evaluated in fp64: near x^ = +-1 a degree-30 Legendre sum moves by ~n^2/2 per unit of
        // x^, so an fp32 node (6e-8) alone costs up to ~1e-5 of the flux there (measured 1.2e-5 on config-2 shapes),
        // the whole tolerance.  S, the part shared with the fit, stays in fp32.
        float isv[OCT], sjv[OCT];
        double xx[OCT];
#pragma unroll
        for (int i = 0; i < OCT; ++i) {
            xx[i] = (double)(2 * (j0 + i - seg_lo) - sg.P) / (double)sg.P;
            if (!UNI) { isv[i] = __ldg(ISg + j0 + i); sjv[i] = __ldg(SJg + j0 + i); }
        }
#pragma unroll 1
        for (int g = 0; g < GS; ++g) {   // one spectrum at a time (an inspection kernel: the basis recurrence is not shared)
            float S[OCT];
            if (UNI) {
                float acc[1][OCT];
                v1_stencil_octet<1>((const float4 *)(rowT + g * RL), j0, tap[2 * g], tap[2 * g + 1], gw4 + g * NA, 0, acc);
#pragma unroll
                for (int i = 0; i < OCT; ++i) S[i] = acc[0][i];
            } else {
                float DV[OCT], DG[OCT], EI[OCT];
                const V1Np np = ((const V1Np *)(V1SM + L.oNP))[g];
                v1_np_forward_octet((const float4 *)(rowT + g * RL), j0, np, isv, sjv, S, DV, DG, EI);
            }
            double cc[OCT], pp[OCT], pc[OCT];
#pragma unroll
            for (int i = 0; i < OCT; ++i) { cc[i] = 0.0; pp[i] = 0.0; pc[i] = 1.0; }
            for (int n = 0; n < n1; ++n) {
                const double bn_ = (double)bco[n * GS + g];
                const double an = (2.0 * n + 1.0) / (n + 1.0), bn = (double)n / (n + 1.0);   // (n+1) P_{n+1} = (2n+1) x P_n - n P_{n-1}
#pragma unroll
                for (int i = 0; i < OCT; ++i) {
                    cc[i] = fma(bn_, pc[i], cc[i]);
                    const double nx = fma(an * xx[i], pc[i], -bn * pp[i]);
                    pp[i] = pc[i]; pc[i] = nx;
                }
            }
            if ((long long)grp * GS + g >= a.B) continue;
            float *out = a.model + (size_t)v1_blk.spec[g] * P + sg.o + (j0 - seg_lo);
#pragma unroll
            for (int i = 0; i < OCT; ++i)
                if (j0 - seg_lo + i < sg.P) out[i] = (float)(cc[i] * (double)S[i]);
        }
    }
}

template <int MAXT, int MINB, bool STREAM>
__global__ void __launch_bounds__(MAXT, MINB)
lasp_v1_model_kernel(const __grid_constant__ ModelDev M, const __grid_constant__ V1Lay L, const V1Args a)
{
    v1_init_block(M, L, a);
    const int NP = M.NP, g = V1_WARP;
    for (int grp = blockIdx.x; grp < a.ngroups; grp += gridDim.x) {
        __syncthreads();
        v1_set_group(grp);
        __syncthreads();
        if (g < GS) {
            for (int p = V1_LANE; p < NP; p += 32)
                SMV(L.oU, p, g) = 2.f * (a.gparams[v1_blk.spec[g] * NP + p] - M.lo[p]) / (M.hi[p] - M.lo[p]) - 1.f;
            for (int n = V1_LANE; n < M.nc; n += 32) SMV(L.oB, n, g) = a.mcont[v1_blk.spec[g] * M.nc + n];
            __syncwarp();
            v1_param_setup(g);
        }
        for (int s = 0; s < M.n_seg; ++s) {
            const SegDev &sg = M.seg[s];
            if (g < GS) v1_setup_weights(sg, g);
            __syncthreads();
            // T over the whole segment plus the reach of the group's widest kernel (inside the halo: halo >= H + 18)
            if (!STREAM && a.CF) {
                const int ks = a.ksteps;
                if (ks <= 4) v1_phase_emulator_mma<1>(s, 1);
                else if (ks <= 8) v1_phase_emulator_mma<2>(s, 1);
                else v1_phase_emulator_mma<4>(s, 1);
            } else
                v1_phase_emulator<STREAM>(s, 1);
            __syncthreads();
            if (sg.uniform) v1_phase_model<true, STREAM>(s, grp); else v1_phase_model<false, STREAM>(s, grp);
            __syncthreads();
        }
    }
}
