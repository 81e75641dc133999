// lasp_common.cuh -- model description as the kernels see it (device-side mirror of lasp_model_desc).
//
// Paper / survey references: Eq. n and P:n are /root/reference/PAPER.md; C.2-n are the readings of
// SURVEY.md 8(c); a0..a9 are the steps of SURVEY.md 8(a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/lasp_gpu.h"

#define CH 8   // pixels per thread tile (octet); every padded offset below is a multiple of it
#define FULL 0xffffffffu
#define LASP_NPMAX (LASP_MAX_LABELS + 2)

struct SegDev {
    int po;       // first padded pixel of the segment (multiple of CH)
    int len;      // padded length = halo + roundup(P,CH) + halo
    int halo;     // replicated-edge columns on each side (multiple of CH, >= largest support H + 18)
    int P, o;     // real length and real offset
    int fit_lo, fit_hi;  // octet-aligned padded range containing every pixel that can have w != 0
    int uniform;  // 1: constant km/s per pixel (log grid) -> one kernel per spectrum per step
    float inv_s;  // 1/s (pixels per km/s) when uniform, else the LARGEST 1/s_j of the segment
    float sig_inst;
    float ta, tb; // ta = tm = 1/(fit_hi - fit_lo - 1): Chebyshev node t = tm (2 (jp - fit_lo) - (fit_hi - fit_lo - 1)); tb unused
};

struct ModelDev {
    int n_seg, L, K, NP, D, n1, nmom, Ppad, P, nc;
    SegDev seg[LASP_MAX_SEG];
    const uint8_t *exps;   // [K][L]
    const double *conv;    // [n_seg][n1][n1] internal Chebyshev(t) -> plain Legendre(x^) (C.2-8)
    float lo[LASP_NPMAX], hi[LASP_NPMAX];
    float emu_a[LASP_MAX_LABELS], emu_b[LASP_MAX_LABELS];
    uint8_t label_log10[LASP_MAX_LABELS];
    // piecewise emulator (lasp_model_desc.n_models > 1): model of every term, and per model the two ramps of its weight
    // in emulator-input units x_0: up = clamp((x_0 - bl_u0) bl_ui, 0, 1), down = clamp((bl_d1 - x_0) bl_di, 0, 1)
    // (bl_ui / bl_di = 0: no ramp on that side)
    int n_models;
    const uint8_t *term_model;
    float bl_u0[LASP_MAX_MODELS], bl_ui[LASP_MAX_MODELS], bl_d1[LASP_MAX_MODELS], bl_di[LASP_MAX_MODELS];
};

// a1: emulator input x_l = a_l tau_l(theta_l) + b_l (Eq. 1, C.2-19)
__device__ __forceinline__ float label_x(const ModelDev &M, int l, float theta)
{
    return M.emu_a[l] * (M.label_log10[l] ? log10f(theta) : theta) + M.emu_b[l];
}
