// lasp_resample.cuh -- flux-conserving resampling of an emulator coefficient table from the model's linear wavelength grid
// onto the observed grid (step 3 of the paper, Eq. 2-4).
//
// The paper resamples every model spectrum at every step: cumulative integral of the model over its integration nodes
// (Eq. 2), linear interpolation of that integral onto the observed integration nodes (Eq. 3), differences divided by the bin
// widths (Eq. 4).  The operation is linear and does not depend on the stellar parameters (Delta-4), so it is applied ONCE to
// the rows of the coefficient table; the fitting kernels then work on the observed grid.  Linear interpolation of a
// cumulative sum is the integral of the piecewise-constant model, so Eq. 2-4 equal, bin by bin,
//     T'_i = sum_m T_m |[node_i, node_(i+1)] intersected with model pixel m| / (node_(i+1) - node_i),
// which is what the kernel evaluates directly (5-7 model pixels per LAMOST bin): no prefix sum, and no cancellation between two
// large cumulative values.  Positions and overlaps are fp64 (wavelengths of ~5e3 A against a 0.2 A step), the sum too; the
// result is rounded once to float.  Bins (or parts of bins) beyond the model's nodes receive no flux (reading R-14).
#pragma once
#include <cstdint>

// one thread per (observed pixel i, term k); lo / hi: the two integration nodes of pixel i
__global__ void lasp_resample_kernel(int q, double node0, double dlam1, const float *__restrict__ coef_model, int n_pix,
                                     const double *__restrict__ lo, const double *__restrict__ hi, float *__restrict__ coef_obs)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    if (i >= n_pix) return;
    const double a = lo[i], b = hi[i];
    double ta = (a - node0) / dlam1, tb = (b - node0) / dlam1;   // positions in units of model pixels, node m at m
    ta = fmin(fmax(ta, 0.0), (double)q);
    tb = fmin(fmax(tb, 0.0), (double)q);
    const int ma = min((int)floor(ta), q - 1), mb = min((int)floor(tb), q - 1);
    const float *row = coef_model + (size_t)k * q;
    double acc = 0.0;
    for (int m = ma; m <= mb; ++m) {
        const double l = fmax(ta, (double)m), h = fmin(tb, (double)(m + 1));
        if (h > l) acc += (double)__ldg(row + m) * (h - l);
    }
    coef_obs[(size_t)k * n_pix + i] = (float)(acc * dlam1 / (b - a));
}
