// lasp_gpu.cu -- C-ABI host side of the LASP-Adam fitting library (include/lasp_gpu.h).
// Host work here is set-up only (validation, layout, basis tables, launches); every step of the hot path
// runs in the kernels of lasp_fit_v1.cuh.  No environment variable is read: every switch is a field of
// lasp_fit_opts.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "lasp_fit_v1.cuh"
#include "lasp_resample.cuh"

#define LASP_VERSION 200
static const double kC_KMS = 299792.458;

// kernel instantiations: index = launch variant
//   0: resident, 192 threads, 2 CTAs/SM   1: resident, up to 384 threads, 1 CTA/SM   2: streaming, 192 threads, 2 CTAs/SM
enum { KV_RES192 = 0, KV_RES384 = 1, KV_STREAM = 2, KV_N = 3 };
static const void *kFit[KV_N] = {(const void *)lasp_v1_fit_kernel<192, 2, false>, (const void *)lasp_v1_fit_kernel<384, 1, false>,
                                 (const void *)lasp_v1_fit_kernel<192, 2, true>};
static const void *kFitClean[KV_N] = {(const void *)lasp_v1_fit_kernel<192, 2, false, 1>,
                                        (const void *)lasp_v1_fit_kernel<384, 1, false, 1>, nullptr};
static const void *kFitLM[KV_N] = {(const void *)lasp_v1_fit_kernel<192, 2, false, 2>, (const void *)lasp_v1_fit_kernel<384, 1, false, 2>,
                                     (const void *)lasp_v1_fit_kernel<384, 1, true, 2>};
static const void *kGrad[KV_N] = {(const void *)lasp_v1_grad_kernel<192, 2, false>, (const void *)lasp_v1_grad_kernel<384, 1, false>,
                                  (const void *)lasp_v1_grad_kernel<192, 2, true>};
static const void *kModel[KV_N] = {(const void *)lasp_v1_model_kernel<192, 2, false>, (const void *)lasp_v1_model_kernel<384, 1, false>,
                                   (const void *)lasp_v1_model_kernel<192, 2, true>};

// Scratch of the allocation-free entry point lasp_eval_grad_static: one array per GPU that loads this library, held
// until the process exits.  In HOST code this name is only a stand-in for the symbol, not a device address: lasp_create
// asks the runtime for the address (cudaGetSymbolAddress, with the ctx's device current) and keeps it in the ctx.
static __device__ __align__(256) float lasp_static_scratch[LASP_STATIC_SCRATCH_BYTES / sizeof(float)];

struct Variant {          // one way of launching the kernels for this model
    bool ok = false;
    int kv = 0;           // kernel instantiation
    int nt = 0;           // threads per CTA
    int cta_per_sm = 1;
    V1Lay L;
};

struct lasp_ctx {
    ModelDev M;
    int device = 0, num_sms = 0;
    uint8_t *dexps = nullptr, *dtermmodel = nullptr;
    double *dconv = nullptr;
    int *dnedge = nullptr;
    long long launches = 0;
    bool nonuniform = false;
    float *dIS = nullptr, *dSJ = nullptr;
    Variant res, str;     // resident and streaming variants
    float *dC1 = nullptr;
    float4 *dCF = nullptr;   // coefficient table as tf32 [hi|lo] MMA fragments (emulator_path 2)
    int cf_ksteps = 0;
    // workspace shared by every call on this ctx: staged planes (per spectrum) and per-CTA scratch
    float *dY = nullptr, *dW = nullptr;
    size_t plane_rows = 0;
    float *dCP = nullptr, *dXJ = nullptr, *dDS = nullptr, *dTG = nullptr, *dAG = nullptr;
    size_t cp_ctas = 0, xj_ctas = 0, ds_ctas = 0, tg_ctas = 0;
    unsigned int *dqueue = nullptr;
    unsigned long long *dstats = nullptr;   // [0] group-steps of the Adam loops, [1] of them with a fresh Gram factor
    cudaEvent_t ws_event = nullptr;
    bool ws_pending = false;
    float *static_ws = nullptr;   // device address of lasp_static_scratch on this ctx's device
#ifdef LASP_PHASE_TIMING
    unsigned long long *ddbg = nullptr;
#endif
    // lasp_fit_batch_host: double-buffered device chunks, two copy streams and one compute stream
    struct HostPipe {
        int64_t cap = 0;
        float *flux[2] = {}, *ivar[2] = {}, *init[2] = {}, *params[2] = {}, *cont[2] = {}, *chi2[2] = {}, *err[2] = {};
        uint8_t *mask[2] = {};
        int32_t *status[2] = {}, *nsteps[2] = {};
        uint8_t *maskout[2] = {};
        cudaStream_t s_in = nullptr, s_out = nullptr, s_fit = nullptr;
        cudaEvent_t in_done[2] = {}, fit_done[2] = {}, out_done[2] = {};
    } hp;
    std::string err;
};

static std::string g_err;

static int fail(lasp_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg;
    g_err = msg;
    return code;
}

#define CUDA_TRY(c, call)                                                                     \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess)                                                                \
            return fail(c, e_ == cudaErrorMemoryAllocation ? LASP_ERR_NOMEM : LASP_ERR_CUDA,  \
                        std::string(#call) + ": " + cudaGetErrorString(e_));                  \
    } while (0)

// The entry points select the ctx's device and put the caller's current device back on return.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) != cudaSuccess) prev = -1; if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

static int roundup(int v, int m) { return (v + m - 1) / m * m; }

// Gauss-Legendre nodes and weights on [-1,1] (Newton on P_n), fp64
static void gauss_legendre(int n, std::vector<double> &x, std::vector<double> &w)
{
    x.resize(n); w.resize(n);
    for (int i = 0; i < n; ++i) {
        double z = cos(M_PI * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 100; ++it) {
            double p1 = 1.0, p2 = 0.0;
            for (int j = 0; j < n; ++j) {
                double p3 = p2;
                p2 = p1;
                p1 = ((2.0 * j + 1.0) * z * p2 - j * p3) / (j + 1.0);
            }
            pp = n * (z * p1 - p2) / (z * z - 1.0);
            double dz = p1 / pp;
            z -= dz;
            if (fabs(dz) < 1e-15) break;
        }
        x[i] = z;
        w[i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

static void hostpipe_free(lasp_ctx *c);

extern "C" int lasp_version(void) { return LASP_VERSION; }

extern "C" const char *lasp_last_error(const lasp_ctx *ctx) { return ctx ? ctx->err.c_str() : g_err.c_str(); }

// 1: the resident variant serves this model by default; 2: only the streaming variant does (rows too long for
// shared memory).  lasp_fit_opts.variant overrides the default per call.
extern "C" int lasp_kernel_variant(const lasp_ctx *ctx) { return !ctx ? 0 : (ctx->res.ok ? 1 : 2); }

extern "C" int lasp_launch_info(const lasp_ctx *c, int variant, int32_t *out4)
{
    if (!c || !out4 || variant < 1 || variant > 2) return LASP_ERR_INVALID_ARG;
    const Variant &v = variant == 1 ? c->res : c->str;
    out4[0] = v.ok; out4[1] = v.nt; out4[2] = v.cta_per_sm; out4[3] = v.L.oHIST * 4;
    return LASP_OK;
}

#ifdef LASP_PHASE_TIMING
// debug build only: per-phase cycle sums of the last fit (thread 0 of every CTA)
extern "C" int lasp_debug_phase_cycles(lasp_ctx *c, unsigned long long *out24)
{
    if (!c || !c->ddbg) return LASP_ERR_INVALID_ARG;
    return cudaMemcpy(out24, c->ddbg, 24 * sizeof(unsigned long long), cudaMemcpyDeviceToHost) == cudaSuccess ? LASP_OK : LASP_ERR_CUDA;
}
#endif

extern "C" int64_t lasp_launch_count(const lasp_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" int lasp_destroy(lasp_ctx *c)
{
    if (!c) return LASP_OK;
    DeviceGuard dg(c->device);
    cudaFree(c->dexps); cudaFree(c->dtermmodel); cudaFree(c->dconv); cudaFree(c->dnedge);
    cudaFree(c->dC1); cudaFree(c->dCF); cudaFree(c->dIS); cudaFree(c->dSJ); cudaFree(c->dDS); cudaFree(c->dY); cudaFree(c->dW);
    cudaFree(c->dCP); cudaFree(c->dXJ); cudaFree(c->dTG); cudaFree(c->dAG); cudaFree(c->dqueue); cudaFree(c->dstats);
#ifdef LASP_PHASE_TIMING
    cudaFree(c->ddbg);
#endif
    if (c->ws_event) cudaEventDestroy(c->ws_event);
    hostpipe_free(c);
    if (c->hp.s_in) {
        cudaStreamDestroy(c->hp.s_in); cudaStreamDestroy(c->hp.s_out); cudaStreamDestroy(c->hp.s_fit);
        for (int s = 0; s < 2; ++s) { cudaEventDestroy(c->hp.in_done[s]); cudaEventDestroy(c->hp.fit_done[s]); cudaEventDestroy(c->hp.out_done[s]); }
    }
    delete c;
    return LASP_OK;
}

static void setup_variant(lasp_ctx *c, const cudaDeviceProp &prop, int emax, bool stream, Variant &v);

extern "C" int lasp_create(const lasp_model_desc *d, int cuda_device, lasp_ctx **out)
{
    if (!d || !out) return fail(nullptr, LASP_ERR_INVALID_ARG, "null desc/out");
    *out = nullptr;
    if (!d->seg_offset || !d->loglam || !d->seg_sigma_inst || !d->term_exps || !d->coeffs || !d->lo ||
        !d->hi || !d->label_log10 || !d->emu_a || !d->emu_b || !d->seg_n_edge)
        return fail(nullptr, LASP_ERR_INVALID_ARG, "null pointer in lasp_model_desc");
    const int P = d->n_pix, nseg = d->n_seg, L = d->n_labels, K = d->n_terms, D = d->cont_degree;
    if (P < 2 || nseg < 1 || L < 1 || K < 1 || D < 0)
        return fail(nullptr, LASP_ERR_INVALID_ARG, "bad shape");
    if (nseg > LASP_MAX_SEG || L > LASP_MAX_LABELS || K > LASP_MAX_TERMS || D > LASP_MAX_DEGREE)
        return fail(nullptr, LASP_ERR_UNSUPPORTED, "shape exceeds LASP_MAX_* limits");
    if (d->seg_offset[0] != 0 || d->seg_offset[nseg] != P)
        return fail(nullptr, LASP_ERR_INVALID_ARG, "seg_offset must start at 0 and end at n_pix");
    const int NP = L + 2;
    if (d->n_models < 0 || d->n_models > LASP_MAX_MODELS)
        return fail(nullptr, d->n_models < 0 ? LASP_ERR_INVALID_ARG : LASP_ERR_UNSUPPORTED, "n_models must be in [0, LASP_MAX_MODELS]");
    if (d->n_models > 1) {
        if (!d->term_model || !d->model_blend) return fail(nullptr, LASP_ERR_INVALID_ARG, "n_models > 1 needs term_model and model_blend");
        for (int k = 0; k < K; ++k)
            if (d->term_model[k] >= d->n_models) return fail(nullptr, LASP_ERR_INVALID_ARG, "term_model entry >= n_models");
        for (int i = 0; i < 4 * d->n_models; ++i)
            if (!std::isfinite(d->model_blend[i]) || (d->label_log10[0] && d->model_blend[i] < 0.f))
                return fail(nullptr, LASP_ERR_INVALID_ARG, "model_blend must be finite (and >= 0 for a log10 label)");
    }
    for (int p = 0; p < NP; ++p)
        if (!(d->lo[p] < d->hi[p])) return fail(nullptr, LASP_ERR_INVALID_ARG, "lo >= hi");
    if (!(d->lo[L + 1] > 0.f)) return fail(nullptr, LASP_ERR_INVALID_ARG, "sigma lower bound must be > 0");
    for (int l = 0; l < L; ++l)
        if (d->label_log10[l] && !(d->lo[l] > 0.f))
            return fail(nullptr, LASP_ERR_INVALID_ARG, "log10 label needs lo > 0");
    for (int s = 0; s < nseg; ++s) {
        int o = d->seg_offset[s], e = d->seg_offset[s + 1];
        if (e - o < 2) return fail(nullptr, LASP_ERR_INVALID_ARG, "segment shorter than 2 pixels");
        if (d->seg_n_edge[s] < 0) return fail(nullptr, LASP_ERR_INVALID_ARG, "negative n_edge");
        if (!(d->seg_sigma_inst[s] >= 0.f)) return fail(nullptr, LASP_ERR_INVALID_ARG, "negative sigma_inst");
        for (int j = o + 1; j < e; ++j)
            if (!(d->loglam[j] > d->loglam[j - 1]))
                return fail(nullptr, LASP_ERR_INVALID_ARG, "loglam not strictly increasing inside a segment");
    }
    lasp_ctx *c = new (std::nothrow) lasp_ctx();
    if (!c) return fail(nullptr, LASP_ERR_NOMEM, "host allocation failed");
    c->device = cuda_device;
    int prev_dev = -1;
    cudaGetDevice(&prev_dev);
#define CUDA_TRY_C(call)                                                  \
    do {                                                                  \
        cudaError_t e_ = (call);                                          \
        if (e_ != cudaSuccess) {                                          \
            std::string m_ = std::string(#call) + ": " + cudaGetErrorString(e_); \
            lasp_destroy(c);                                              \
            if (prev_dev >= 0) cudaSetDevice(prev_dev);                   \
            return fail(nullptr, LASP_ERR_CUDA, m_);                      \
        }                                                                 \
    } while (0)
    CUDA_TRY_C(cudaSetDevice(cuda_device));
    cudaDeviceProp prop;
    CUDA_TRY_C(cudaGetDeviceProperties(&prop, cuda_device));
    c->num_sms = prop.multiProcessorCount;

    ModelDev &M = c->M;
    memset(&M, 0, sizeof(M));
    M.n_seg = nseg; M.L = L; M.K = K; M.NP = NP; M.D = D; M.n1 = D + 1; M.nmom = 2 * D + 1;
    M.P = P; M.nc = nseg * (D + 1);
    for (int p = 0; p < NP; ++p) { M.lo[p] = d->lo[p]; M.hi[p] = d->hi[p]; }
    for (int l = 0; l < L; ++l) {
        M.emu_a[l] = d->emu_a[l]; M.emu_b[l] = d->emu_b[l]; M.label_log10[l] = d->label_log10[l];
    }
    // per-pixel velocity scale s_j = c ln10 dloglam (C.1), fp64
    std::vector<double> s(P);
    const double vmax = fmax(fabs((double)d->lo[L]), fabs((double)d->hi[L]));
    const double smax = fmax(fabs((double)d->lo[L + 1]), fabs((double)d->hi[L + 1]));
    int po = 0;
    bool halo_ok = true;
    std::vector<double> conv((size_t)nseg * M.n1 * M.n1, 0.0);
    for (int sg = 0; sg < nseg; ++sg) {
        const int o = d->seg_offset[sg], e = d->seg_offset[sg + 1], Ps = e - o;
        double smin = 1e300, smx = 0, ssum = 0;
        for (int j = o; j < e; ++j) {
            double dl = (j == o) ? d->loglam[j + 1] - d->loglam[j]
                      : (j == e - 1) ? d->loglam[j] - d->loglam[j - 1]
                                     : 0.5 * (d->loglam[j + 1] - d->loglam[j - 1]);
            s[j] = kC_KMS * log(10.0) * dl;
            smin = fmin(smin, s[j]); smx = fmax(smx, s[j]); ssum += s[j];
        }
        SegDev &S = M.seg[sg];
        const double si = d->seg_sigma_inst[sg];
        const double hm = ceil((vmax + 5.0 * sqrt(smax * smax + si * si)) / smin) + 1.0;
        if (!(hm < (double)(V1_TPAD - 18))) { halo_ok = false; break; }
        const int Hm = (int)hm;
        S.halo = roundup(Hm + 18, CH);   // the kernels read up to 18 pixels past the largest support
        S.po = po; S.P = Ps; S.o = o;
        S.len = S.halo + roundup(Ps, CH) + S.halo;
        po += S.len;
        S.uniform = (smx - smin) <= 1e-6 * smin ? 1 : 0;
        if (!S.uniform) c->nonuniform = true;    // per-pixel kernels (linear grids, C.2-14)
        S.inv_s = (float)(S.uniform ? (double)Ps / ssum : 1.0 / smin);
        S.sig_inst = d->seg_sigma_inst[sg];
        const int ne = d->seg_n_edge[sg];
        const int jl = ne, jh = Ps - 1 - ne;
        if (jh >= jl) {
            // the pixels beside the first and the last one that can carry weight are included: the Clean mask update
            // takes the model's flux gradient across them (R-7)
            S.fit_lo = S.po + S.halo + (ne > 0 ? (ne - 1) / CH * CH : 0);
            S.fit_hi = S.po + S.halo + roundup(ne > 0 ? Ps - ne + 1 : Ps, CH);
            if (((S.fit_hi - S.fit_lo) / CH) & 1) S.fit_hi += CH;   // an even number of octets: they pair up about the centre
        } else {
            S.fit_lo = S.fit_hi = S.po + S.halo;
        }
        // Internal Chebyshev nodes, symmetric about the centre of the octet-aligned fitted range (lasp_fit_v1.cuh):
        // t_j = tm (2 (j - fit_lo) - (N - 1)), N = fit_hi - fit_lo, tm = 1/(N - 1): |t| <= 1 on every pixel with w != 0
        const int nfit = S.fit_hi - S.fit_lo;
        S.ta = nfit > 1 ? (float)(1.0 / (nfit - 1)) : 0.f;
        S.tb = 0.f;
        // conv[m][n] = (2m+1)/2 int P_m(x) T_n(alpha x + beta) dx, exact by Gauss-Legendre (D+2 nodes), with the
        // device's float tm so that the conversion matches the basis actually used; x^ = -1 + 2 j/Ps
        const double flo_rel = S.fit_lo - (S.po + S.halo);
        const double alpha = (double)S.ta * Ps, beta = (double)S.ta * (Ps - 2.0 * flo_rel - (nfit - 1));
        std::vector<double> gx, gw;
        gauss_legendre(M.n1 + 1, gx, gw);
        double *cv = conv.data() + (size_t)sg * M.n1 * M.n1;
        for (size_t q = 0; q < gx.size(); ++q) {
            std::vector<double> Pm(M.n1), Tn(M.n1);
            const double x = gx[q], t = alpha * x + beta;
            Pm[0] = 1.0; if (M.n1 > 1) Pm[1] = x;
            for (int n = 1; n + 1 < M.n1; ++n) Pm[n + 1] = ((2.0 * n + 1.0) * x * Pm[n] - n * Pm[n - 1]) / (n + 1.0);
            Tn[0] = 1.0; if (M.n1 > 1) Tn[1] = t;
            for (int n = 1; n + 1 < M.n1; ++n) Tn[n + 1] = 2.0 * t * Tn[n] - Tn[n - 1];
            for (int m = 0; m < M.n1; ++m)
                for (int n = 0; n < M.n1; ++n) cv[m * M.n1 + n] += 0.5 * (2.0 * m + 1.0) * gw[q] * Pm[m] * Tn[n];
        }
    }
    if (!halo_ok) {
        lasp_destroy(c);
        if (prev_dev >= 0) cudaSetDevice(prev_dev);
        return fail(nullptr, LASP_ERR_UNSUPPORTED, "largest kernel support over the prior box exceeds 238 pixels");
    }
    M.Ppad = po;
    // padded tables: halos replicate the segment's edge pixel (the clamp of C.2-16 for free)
    // K+2 rounded to 4 rows, plus 16 (prefetch overrun): zero past K, so the loops sweep whole batches without bounds tests
    const int Krows = roundup(K + 2, 4) + 16;
    std::vector<float> Cp((size_t)Krows * M.Ppad, 0.f), isp(M.Ppad);
    for (int sg = 0; sg < nseg; ++sg) {
        const SegDev &S = M.seg[sg];
        for (int q = 0; q < S.len; ++q) {
            int rel = q - S.halo;
            rel = rel < 0 ? 0 : (rel > S.P - 1 ? S.P - 1 : rel);
            isp[S.po + q] = (float)(1.0 / s[S.o + rel]);
            for (int k = 0; k < K; ++k) Cp[(size_t)k * M.Ppad + S.po + q] = d->coeffs[(size_t)k * P + S.o + rel];
        }
    }
    {   // the table in the split-octet layout (half h of octet o at h*Ppad/2 + 4 o)
        std::vector<float> C1(Cp.size());
        for (int k = 0; k < Krows; ++k)
            for (int jp = 0; jp < M.Ppad; ++jp)
                C1[(size_t)k * M.Ppad + ((jp >> 2) & 1) * (M.Ppad >> 1) + (jp >> 3) * 4 + (jp & 3)] = Cp[(size_t)k * M.Ppad + jp];
        CUDA_TRY_C(cudaMalloc(&c->dC1, C1.size() * sizeof(float)));
        CUDA_TRY_C(cudaMemcpy(c->dC1, C1.data(), C1.size() * sizeof(float), cudaMemcpyHostToDevice));
    }
    if (K <= 128) {
        // tensor-pipe copy: A fragments of mma.m16n8k8 (rows = pixels, columns = terms), one float4 per
        // (octet o, k-step s, lane l): {hi, hi', lo, lo'} of C[8s + l%4 (+4)][8o + l/4], hi = tf32(x), lo = tf32(x - hi)
        auto tf32 = [](float x) {
            uint32_t u; memcpy(&u, &x, 4);
            u = (u + 0x1000u) & 0xFFFFE000u;            // round to nearest, ties away (cvt.rna.tf32)
            float r; memcpy(&r, &u, 4); return r;
        };
        const int ks = (K + 7) / 8, noct = M.Ppad / 8 + 1;
        std::vector<float> CF((size_t)noct * ks * 32 * 4, 0.f);
        for (int o = 0; o + 1 < noct; ++o)
            for (int sidx = 0; sidx < ks; ++sidx)
                for (int l = 0; l < 32; ++l)
                    for (int h = 0; h < 2; ++h) {
                        const int k = 8 * sidx + (l & 3) + 4 * h, jp = 8 * o + (l >> 2);
                        const float x = k < K ? Cp[(size_t)k * M.Ppad + jp] : 0.f;
                        const float hi = tf32(x), lo = tf32(x - hi);
                        float *f = &CF[(((size_t)o * ks + sidx) * 32 + l) * 4];
                        f[h] = hi; f[2 + h] = lo;
                    }
        c->cf_ksteps = ks;
        CUDA_TRY_C(cudaMalloc(&c->dCF, CF.size() * sizeof(float)));
        CUDA_TRY_C(cudaMemcpy(c->dCF, CF.data(), CF.size() * sizeof(float), cudaMemcpyHostToDevice));
    }
    {   // 1/s_j and s_j for the per-pixel kernels, V1_TPAD replicated entries on both sides
        std::vector<float> is1(M.Ppad + 2 * V1_TPAD), sj1(M.Ppad + 2 * V1_TPAD);
        for (int q = 0; q < M.Ppad + 2 * V1_TPAD; ++q) {
            const int jp = std::min(std::max(q - V1_TPAD, 0), M.Ppad - 1);
            is1[q] = isp[jp];
            sj1[q] = (float)(1.0 / (double)isp[jp]);
        }
        CUDA_TRY_C(cudaMalloc(&c->dIS, is1.size() * sizeof(float)));
        CUDA_TRY_C(cudaMemcpy(c->dIS, is1.data(), is1.size() * sizeof(float), cudaMemcpyHostToDevice));
        CUDA_TRY_C(cudaMalloc(&c->dSJ, sj1.size() * sizeof(float)));
        CUDA_TRY_C(cudaMemcpy(c->dSJ, sj1.data(), sj1.size() * sizeof(float), cudaMemcpyHostToDevice));
    }
    CUDA_TRY_C(cudaMalloc(&c->dexps, (size_t)K * L));
    CUDA_TRY_C(cudaMemcpy(c->dexps, d->term_exps, (size_t)K * L, cudaMemcpyHostToDevice));
    CUDA_TRY_C(cudaMalloc(&c->dconv, conv.size() * sizeof(double)));
    CUDA_TRY_C(cudaMemcpy(c->dconv, conv.data(), conv.size() * sizeof(double), cudaMemcpyHostToDevice));
    CUDA_TRY_C(cudaMalloc(&c->dnedge, nseg * sizeof(int)));
    CUDA_TRY_C(cudaMemcpy(c->dnedge, d->seg_n_edge, nseg * sizeof(int), cudaMemcpyHostToDevice));
    CUDA_TRY_C(cudaMalloc(&c->dqueue, sizeof(unsigned int)));
    CUDA_TRY_C(cudaMalloc(&c->dstats, 2 * sizeof(unsigned long long)));
    CUDA_TRY_C(cudaMemset(c->dstats, 0, 2 * sizeof(unsigned long long)));
    CUDA_TRY_C(cudaEventCreateWithFlags(&c->ws_event, cudaEventDisableTiming));
    CUDA_TRY_C(cudaGetSymbolAddress((void **)&c->static_ws, lasp_static_scratch));   // this device's copy of the array
    M.exps = c->dexps; M.conv = c->dconv;
    M.n_models = d->n_models > 1 ? d->n_models : 0;
    if (M.n_models) {
        CUDA_TRY_C(cudaMalloc(&c->dtermmodel, (size_t)K));
        CUDA_TRY_C(cudaMemcpy(c->dtermmodel, d->term_model, (size_t)K, cudaMemcpyHostToDevice));
        M.term_model = c->dtermmodel;
        // the ramps in emulator-input units x_0 = emu_a tau_0(theta_0) + emu_b (fp64 here, floats on the device)
        auto X0 = [&](double th) { return (double)d->emu_a[0] * (d->label_log10[0] ? log10(th) : th) + (double)d->emu_b[0]; };
        for (int r = 0; r < M.n_models; ++r) {
            const float *bl = d->model_blend + 4 * r;
            M.bl_u0[r] = M.bl_ui[r] = M.bl_d1[r] = M.bl_di[r] = 0.f;
            if (bl[1] > bl[0]) { M.bl_u0[r] = (float)X0(bl[0]); M.bl_ui[r] = (float)(1.0 / (X0(bl[1]) - X0(bl[0]))); }
            if (bl[3] > bl[2]) { M.bl_d1[r] = (float)X0(bl[3]); M.bl_di[r] = (float)(1.0 / (X0(bl[3]) - X0(bl[2]))); }
        }
    }
    int emax = 0;
    for (int i = 0; i < K * L; ++i) emax = std::max(emax, (int)d->term_exps[i]);
    setup_variant(c, prop, emax, false, c->res);
    setup_variant(c, prop, emax, true, c->str);
    if (prev_dev >= 0) cudaSetDevice(prev_dev);
    if (!c->res.ok && !c->str.ok) {
        lasp_destroy(c);
        return fail(nullptr, LASP_ERR_UNSUPPORTED, "model state does not fit the kernels' shared memory");
    }
    *out = c;
    return LASP_OK;
}

// ------------------------------------------------------------------------------------------
// shared-memory layout and launch shape of one variant (lasp_fit_v1.cuh)
// ------------------------------------------------------------------------------------------
static void setup_variant(lasp_ctx *c, const cudaDeviceProp &prop, int emax, bool stream, Variant &v)
{
    const ModelDev &M = c->M;
    v.ok = false;
    int maxlen = 0, guard = 0, nfit = 0, hmax = 1;
    for (int s = 0; s < M.n_seg; ++s) {
        const SegDev &S = M.seg[s];
        maxlen = std::max(maxlen, S.len);
        guard = std::max(guard, S.halo);
        nfit = std::max(nfit, (S.fit_hi - S.fit_lo) / OCT);
        if (S.uniform) hmax = std::max(hmax, S.halo - 18);   // tap tables exist only for uniform segments
    }
    if (M.NP > 32 || M.n1 > 32) return;
    V1Lay &L = v.L;
    memset(&L, 0, sizeof(L));
    L.emax = emax;
    int nt = std::max(GS * 32, roundup(std::max(nfit, 1), 32));
    if (nt > 384) nt = 384;               // longer segments are swept in several passes
    if (stream) nt = 192;
    v.nt = nt;
    v.kv = stream ? KV_STREAM : (nt <= 192 ? KV_RES192 : KV_RES384);
    L.NW = nt / 32;
    L.nt8 = nt * OCT;
    L.GUARD = guard;
    L.RL = stream ? L.nt8 + 2 * guard : maxlen + 2 * guard;
    L.SL = maxlen;
    L.Hm = hmax;
    L.NA = (hmax + 3) / 4 + hmax / 4 + 2;
    L.n1r = roundup(M.n1, 8);
    L.nmomr = L.n1r + roundup(std::max(M.nmom - L.n1r, 0), 8);
    L.VR = L.nmomr + L.n1r + roundup(M.K + 2, 8) + 6;
    L.fastupd = (M.L >= 1 && M.L <= 4 && M.K + 2 <= 32 && L.NW <= 12 && M.n_models == 0) ? 1 : 0;
    L.fastw = (L.fastupd && M.n_seg == 1 && M.seg[0].uniform && M.seg[0].fit_hi > M.seg[0].fit_lo) ? 1 : 0;
    size_t bytes = 0;
    for (L.lfseg = 1; L.lfseg >= 0; --L.lfseg) {   // a factor slot per segment if shared memory allows it
        int o = 0;
        auto take = [&](int n) { int r = o; o += roundup(n, 4); return r; };
        L.oT = take(GS * L.RL);
        L.oA = stream ? L.oT : take(GS * L.RL);    // streaming: one window buffer serves both rows
        L.oU = take(GS * M.NP); L.oM = take(GS * M.NP); L.oV = take(GS * M.NP);
        L.Kq = roundup(M.K + 2, 4);
        L.oX = take(GS * M.L); L.oPHI = take(GS * L.Kq);
        L.oGW = take(GS * L.NA * 4); L.oGR = take(3 * GS * L.NA * 4); L.oTAP = take(2 * GS);
        L.oMOM = take(GS * L.nmomr); L.oRHS = take(GS * L.n1r); L.oB = take(GS * M.nc);
        L.oRED = take(L.NW * L.VR * GS);
        const int npair = M.NP * (M.NP + 1) / 2;
        L.oLF = take(std::max(GS * V1_LFS * (L.lfseg ? M.n_seg : 1), 2 * GS * npair + 4));
        L.oQ = take(GS * (M.K + 2)); L.oSC = take(GS * (SC_N + M.n_seg));
        L.oEXP = take(std::max((M.K * M.L + 3) / 4, M.K));   // bytes [K][L], or one packed word per term when L <= 4
        L.oXP = take(GS * M.L * (L.emax + 1)); L.oDPHI = take(GS * M.L * M.K); L.oGSC = take(GS * M.NP);
        L.oNP = take(GS * 8);
        L.oTM = take(M.n_models ? (M.K + 3) / 4 : 0);
        // LAST: the loss history of the stopping rules, GS rings of stop_window entries.  A launch asks for what its call
        // needs (launch(): oHIST + GS * stop_window floats), the layout is sized for the largest window.  Not cosmetic: with
        // two CTAs per SM the config-1 shape sits 0.1 % under a shared-memory carveout step -- 2 x (dynamic + static block
        // state + 1 KB reserved) <= 196 KB leaves 60 KB of L1, one byte more selects the 228 KB carveout and 28 KB of L1,
        // which costs 2 % (L1 hit rate of the table / plane loads 12.6 % -> 5.2 %, measured)
        L.oHIST = take(GS * V1_WMAX);
        L.total = o;
        bytes = (size_t)o * sizeof(float);
        if (bytes + 2048 <= prop.sharedMemPerBlockOptin) break;   // + the kernels' static block state
    }
    if (L.lfseg < 0) return;
    const void *fs[5] = {kFit[v.kv], kGrad[v.kv], kModel[v.kv], kFitClean[v.kv], kFitLM[v.kv]};
    // The limit is an attribute of the kernel function on this device, shared by every ctx: only ever raise it (a second
    // ctx with shorter rows must not take away what the launches of the first one need)
    for (const void *f : fs) {
        if (!f) continue;
        cudaFuncAttributes at;
        if (cudaFuncGetAttributes(&at, f) != cudaSuccess) { cudaGetLastError(); return; }
        if ((int)bytes > at.maxDynamicSharedSizeBytes &&
            cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) != cudaSuccess) { cudaGetLastError(); return; }
    }
    int per_sm = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kFit[v.kv], nt, bytes) != cudaSuccess || per_sm < 1) {
        cudaGetLastError();
        return;
    }
    v.cta_per_sm = per_sm;
    v.ok = true;
}

// ------------------------------------------------------------------------------------------
// options, workspace, launches
// ------------------------------------------------------------------------------------------
static const lasp_fit_opts kDefaultOpts = {0, 1e-2f, 0.9f, 0.999f, 1e-8f, 0, 0, 0, 0, 0, 0, 0.f, 0, 0, 0, 0.f};

// variant / emulator path of one call (opts may be null: defaults)
static int resolve(lasp_ctx *c, const lasp_fit_opts *o, const char *who, const Variant **v, bool *mma)
{
    if (!o) o = &kDefaultOpts;
    if (o->variant < 0 || o->variant > 2) return fail(c, LASP_ERR_INVALID_ARG, std::string(who) + ": variant must be 0, 1 or 2");
    if (o->emulator_path < 0 || o->emulator_path > 2)
        return fail(c, LASP_ERR_INVALID_ARG, std::string(who) + ": emulator_path must be 0, 1 or 2");
    if (o->refresh < 0 || o->warm < 0 || o->fd_fresh < 0 || o->fd_fresh > 1)
        return fail(c, LASP_ERR_INVALID_ARG, std::string(who) + ": refresh, warm must be >= 0 and fd_fresh 0 or 1");
    if (o->stop_window < 0 || o->stop_window > V1_WMAX || (o->stop_window > 0 && !(o->stop_tol >= 0.f)))
        return fail(c, LASP_ERR_INVALID_ARG, std::string(who) + ": stop_window must be in [0, 128] and stop_tol >= 0");
    if (o->clean_every < 0 || o->clean_max < 0)
        return fail(c, LASP_ERR_INVALID_ARG, std::string(who) + ": clean_every and clean_max must be >= 0");
    if (o->optimizer < 0 || o->optimizer > 1 || !(o->lm_lambda0 >= 0.f))
        return fail(c, LASP_ERR_INVALID_ARG, std::string(who) + ": optimizer must be 0 (Adam) or 1 (Levenberg-Marquardt), lm_lambda0 >= 0");
    const Variant *vv = nullptr;
    if (o->variant == 1) vv = c->res.ok ? &c->res : nullptr;
    else if (o->variant == 2) vv = c->str.ok ? &c->str : nullptr;
    else vv = c->res.ok ? &c->res : (c->str.ok ? &c->str : nullptr);
    if (!vv)
        return fail(c, LASP_ERR_UNSUPPORTED, std::string(who) + (o->variant == 1 ? ": the rows of this model do not fit shared memory (variant 1, resident)"
                                                                                   : ": variant not available for this model"));
    *mma = o->emulator_path == 2;
    if (*mma && !(vv == &c->res && c->dCF))
        return fail(c, LASP_ERR_UNSUPPORTED, std::string(who) + ": emulator_path 2 (tensor pipe) needs the resident variant and n_terms <= 128");
    *v = vv;
    return LASP_OK;
}

static int workspace(lasp_ctx *c, int64_t B, const Variant &v, bool need_planes, bool need_cp, bool need_xj)
{
    const ModelDev &M = c->M;
    if (need_planes && (size_t)B > c->plane_rows) {
        cudaFree(c->dY); cudaFree(c->dW);
        c->dY = c->dW = nullptr; c->plane_rows = 0;
        CUDA_TRY(c, cudaMalloc(&c->dY, (size_t)B * M.Ppad * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&c->dW, (size_t)B * M.Ppad * sizeof(float)));
        c->plane_rows = (size_t)B;
    }
    const size_t ctas = (size_t)c->num_sms * std::max(c->res.ok ? c->res.cta_per_sm : 1, c->str.ok ? c->str.cta_per_sm : 1);
    if (need_cp && ctas > c->cp_ctas) {
        cudaFree(c->dCP); c->dCP = nullptr; c->cp_ctas = 0;
        CUDA_TRY(c, cudaMalloc(&c->dCP, ctas * GS * M.Ppad * sizeof(float)));
        c->cp_ctas = ctas;
    }
    if (need_cp && c->nonuniform && ctas > c->ds_ctas) {
        cudaFree(c->dDS); c->dDS = nullptr; c->ds_ctas = 0;
        CUDA_TRY(c, cudaMalloc(&c->dDS, ctas * 3 * GS * v.L.SL * sizeof(float)));
        c->ds_ctas = ctas;
    }
    if (need_xj && ctas > c->xj_ctas) {
        cudaFree(c->dXJ); c->dXJ = nullptr; c->xj_ctas = 0;
        CUDA_TRY(c, cudaMalloc(&c->dXJ, ctas * (size_t)(2 + M.NP) * GS * M.Ppad * sizeof(float)));
        c->xj_ctas = ctas;
    }
    if (&v == &c->str && ctas > c->tg_ctas) {
        cudaFree(c->dTG); cudaFree(c->dAG); c->dTG = c->dAG = nullptr; c->tg_ctas = 0;
        CUDA_TRY(c, cudaMalloc(&c->dTG, ctas * GS * M.Ppad * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&c->dAG, ctas * GS * M.Ppad * sizeof(float)));
        c->tg_ctas = ctas;
    }
    return LASP_OK;
}

extern "C" int lasp_reserve(lasp_ctx *c, int64_t B)
{
    if (!c || B < 1) return fail(c, LASP_ERR_INVALID_ARG, "lasp_reserve: bad argument");
    DeviceGuard dg(c->device);
    return workspace(c, B, c->res.ok ? c->res : c->str, true, true, true);
}

// a0: w = mask*ivar, zero on the n_edge pixels at each end of each segment (Eq. 8); rows go to the
// padded layout (halos zero).  Exactly the oracle's rule: a pixel takes part iff w != 0, so y is zeroed where
// w == 0 (masked flux may hold anything) and nothing else is altered -- a non-finite flux or weight on a pixel
// that takes part propagates and ends in status bit LASP_ST_NONFINITE (reading R-1).
__global__ void lasp_v1_stage_kernel(const __grid_constant__ ModelDev M, const int *__restrict__ n_edge,
                                     const float *__restrict__ flux, const float *__restrict__ ivar,
                                     const uint8_t *__restrict__ mask, float *__restrict__ Y, float *__restrict__ W)
{
    const size_t row = blockIdx.x;
    for (int jp = threadIdx.x; jp < M.Ppad; jp += blockDim.x) {
        int s = 0;
        while (s + 1 < M.n_seg && jp >= M.seg[s + 1].po) ++s;
        const SegDev &sg = M.seg[s];
        const int rel = jp - sg.po - sg.halo;
        float y = 0.f, w = 0.f;
        if (rel >= 0 && rel < sg.P) {
            const size_t o = row * M.P + sg.o + rel;
            w = ivar[o];
            if (mask && mask[o] == 0) w = 0.f;
            const int ne = n_edge[s];
            if (rel < ne || rel >= sg.P - ne) w = 0.f;
            y = (w == 0.f) ? 0.f : flux[o];
        }
        // split-octet layout: half h of octet o at h*Ppad/2 + 4 o, so that a warp's 128-bit loads are contiguous
        const size_t q = row * M.Ppad + ((jp >> 2) & 1) * (M.Ppad >> 1) + (jp >> 3) * 4 + (jp & 3);
        Y[q] = y;
        W[q] = w;
    }
}

static int stage(lasp_ctx *c, int64_t B, const float *flux, const float *ivar, const uint8_t *mask, cudaStream_t st)
{
    lasp_v1_stage_kernel<<<(unsigned)B, 256, 0, st>>>(c->M, c->dnedge, flux, ivar, mask, c->dY, c->dW);
    c->launches += 1;
    CUDA_TRY(c, cudaGetLastError());
    return LASP_OK;
}

// every call waits, on ITS stream, for the ctx's previous call (possibly on another stream) before it touches the
// shared workspace, and records its own completion
static int ws_acquire(lasp_ctx *c, cudaStream_t st)
{
    if (c->ws_pending) CUDA_TRY(c, cudaStreamWaitEvent(st, c->ws_event, 0));
    return LASP_OK;
}

static int ws_release(lasp_ctx *c, cudaStream_t st)
{
    CUDA_TRY(c, cudaEventRecord(c->ws_event, st));
    c->ws_pending = true;
    return LASP_OK;
}

static void base_args(lasp_ctx *c, const Variant &v, bool mma, int64_t B, V1Args &a)
{
    memset(&a, 0, sizeof(a));
    a.Y = c->dY; a.W = c->dW; a.C1 = c->dC1; a.CP = c->dCP; a.B = B;
    a.IS = c->dIS; a.SJ = c->dSJ; a.DS = c->dDS;
    if (&v == &c->str) { a.TG = c->dTG; a.AG = c->dAG; }
    if (mma) { a.CF = c->dCF; a.ksteps = c->cf_ksteps; }
    a.ngroups = (int)((B + GS - 1) / GS);
}

static int launch(lasp_ctx *c, const void *const *table, const Variant &v, const V1Args &a, cudaStream_t st)
{
    const int grid = std::min(a.ngroups, c->num_sms * v.cta_per_sm);
    const size_t smem = (size_t)(v.L.oHIST + GS * a.stop_window) * sizeof(float);   // see setup_variant
    void *args[3] = {(void *)&c->M, (void *)&v.L, (void *)&a};
    CUDA_TRY(c, cudaLaunchKernel(table[v.kv], dim3(grid), dim3(v.nt), args, smem, st));
    c->launches += 1;
    return ws_release(c, st);
}

extern "C" int lasp_fit_batch(lasp_ctx *c, int64_t B, const float *flux, const float *ivar,
                              const uint8_t *mask, const float *init, const lasp_fit_opts *opts,
                              float *params, float *cont, float *chi2, float *err, int32_t *status,
                              int32_t *n_steps, uint8_t *mask_out, void *stream)
{
    if (!c) return fail(nullptr, LASP_ERR_INVALID_ARG, "null ctx");
    if (B < 1 || !flux || !ivar || !init || !opts || !params || !chi2)
        return fail(c, LASP_ERR_INVALID_ARG, "lasp_fit_batch: null pointer or B < 1");
    const bool lm = opts->optimizer == 1;
    if (opts->n_iter < 0 || (!lm && !(opts->lr > 0.f)) || !(opts->beta1 >= 0.f && opts->beta1 < 1.f) ||
        !(opts->beta2 >= 0.f && opts->beta2 < 1.f) || !(opts->eps >= 0.f))
        return fail(c, LASP_ERR_INVALID_ARG, "lasp_fit_batch: bad Adam hyper-parameters");
    if (B > (int64_t)1 << 30) return fail(c, LASP_ERR_UNSUPPORTED, "B too large");
    const Variant *v = nullptr;
    bool mma = false;
    int rc = resolve(c, opts, "lasp_fit_batch", &v, &mma);
    if (rc) return rc;
    if (opts->clean_every > 0) {
        // the mask update keeps one octet of the fitted range per thread and reads its neighbours from the resident rows
        const SegDev &S0 = c->M.seg[0];
        if (v != &c->res || c->M.n_seg != 1 || (S0.fit_hi - S0.fit_lo) / OCT > v->nt)
            return fail(c, LASP_ERR_UNSUPPORTED, "lasp_fit_batch: the Clean strategy needs the resident variant and one segment "
                                                 "whose fitted range is one sweep of the CTA");
    }
    if (lm && (opts->clean_every > 0 || opts->stop_window > 0))
        return fail(c, LASP_ERR_UNSUPPORTED, "lasp_fit_batch: the Levenberg-Marquardt optimiser runs n_iter iterations without the "
                                             "Clean strategy or the stopping rules");
    DeviceGuard dg(c->device);
    rc = workspace(c, B, *v, true, true, err != nullptr || lm);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ws_acquire(c, st);
    if (rc) return rc;
    rc = stage(c, B, flux, ivar, mask, st);
    if (rc) return rc;
    V1Args a;
    base_args(c, *v, mma, B, a);
    a.XJ = c->dXJ;
    a.init = init; a.n_iter = opts->n_iter; a.lr = opts->lr; a.b1 = opts->beta1; a.b2 = opts->beta2;
    a.eps = opts->eps; a.fd_h = 2e-3f;  // fp32 central-difference step in u (C.2-22)
    a.params = params; a.cont = cont; a.chi2 = chi2; a.err = err; a.status = status;
    a.warm = opts->warm > 0 ? opts->warm : 4;
    a.refresh = opts->refresh;
    a.fdfresh = opts->fd_fresh;
    a.drift_tol = 6.4e-3f;   // = 64 steps x (1e-2)^2: the fixed schedule the parity suite was tuned at
    a.stop_window = opts->stop_window; a.stop_tol = opts->stop_tol; a.nsteps = n_steps;
    a.clean_every = opts->clean_every; a.clean_max = opts->clean_max > 0 ? opts->clean_max : 11;
    a.mask_out = mask_out;
    a.lm_lambda0 = opts->lm_lambda0 > 0.f ? opts->lm_lambda0 : 1e-3f;
    CUDA_TRY(c, cudaMemsetAsync(c->dqueue, 0, sizeof(unsigned int), st));
    CUDA_TRY(c, cudaMemsetAsync(c->dstats, 0, 2 * sizeof(unsigned long long), st));
    a.queue = c->dqueue;
    a.stats = c->dstats;
#ifdef LASP_PHASE_TIMING
    if (!c->ddbg) { CUDA_TRY(c, cudaMalloc(&c->ddbg, 24 * sizeof(unsigned long long))); }
    CUDA_TRY(c, cudaMemsetAsync(c->ddbg, 0, 24 * sizeof(unsigned long long), st));
    a.dbg = c->ddbg;
#endif
    return launch(c, lm ? kFitLM : (opts->clean_every > 0 ? kFitClean : kFit), *v, a, st);
}

extern "C" int lasp_eval_grad(lasp_ctx *c, int64_t B, const float *flux, const float *ivar,
                              const uint8_t *mask, const float *params, const lasp_fit_opts *opts, float *chi2,
                              float *grad_u, float *cont, int32_t *status, void *stream)
{
    if (!c) return fail(nullptr, LASP_ERR_INVALID_ARG, "null ctx");
    if (B < 1 || !flux || !ivar || !params || !chi2 || !grad_u)
        return fail(c, LASP_ERR_INVALID_ARG, "lasp_eval_grad: null pointer or B < 1");
    const Variant *v = nullptr;
    bool mma = false;
    int rc = resolve(c, opts, "lasp_eval_grad", &v, &mma);
    if (rc) return rc;
    DeviceGuard dg(c->device);
    rc = workspace(c, B, *v, true, true, false);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ws_acquire(c, st);
    if (rc) return rc;
    rc = stage(c, B, flux, ivar, mask, st);
    if (rc) return rc;
    V1Args a;
    base_args(c, *v, mma, B, a);
    a.gparams = params; a.chi2 = chi2; a.grad_u = grad_u; a.cont = cont; a.status = status;
    return launch(c, kGrad, *v, a, st);
}

// lasp_eval_grad without any allocation: the staged planes and the per-CTA scratch are carved out of lasp_static_scratch.
// Calls nothing that allocates (no cudaMalloc / cudaFree, no library routine): two kernel launches, one memset, two event
// calls.  The array is shared by every ctx and every call on the device and keeps the last call's contents: the stage kernel
// rewrites every padded pixel of the planes it uses, the per-CTA part is cleared here, and calls that overlap on the GPU
// (different streams, different ctxs) race -- the caller serialises them.
extern "C" int lasp_eval_grad_static(lasp_ctx *c, int64_t B, const float *flux, const float *ivar,
                                     const uint8_t *mask, const float *params, const lasp_fit_opts *opts, float *chi2,
                                     float *grad_u, float *cont, int32_t *status, void *stream)
{
    if (!c) return fail(nullptr, LASP_ERR_INVALID_ARG, "null ctx");
    if (B < 1 || !flux || !ivar || !params || !chi2 || !grad_u)
        return fail(c, LASP_ERR_INVALID_ARG, "lasp_eval_grad_static: null pointer or B < 1");
    const Variant *v = nullptr;
    bool mma = false;
    int rc = resolve(c, opts, "lasp_eval_grad_static", &v, &mma);
    if (rc) return rc;
    if (!c->static_ws) return fail(c, LASP_ERR_CUDA, "lasp_eval_grad_static: the static scratch has no device address");
    const ModelDev &M = c->M;
    const size_t cap = LASP_STATIC_SCRATCH_BYTES / sizeof(float);
    const size_t ngroups = ((size_t)B + GS - 1) / GS;
    const size_t grid = std::min(ngroups, (size_t)c->num_sms * v->cta_per_sm);
    auto up = [](size_t n) { return (n + 63) / 64 * 64; };   // 256-byte steps
    const size_t n_plane = up((size_t)B * M.Ppad), n_cp = up(grid * GS * M.Ppad);
    const size_t n_ds = c->nonuniform ? up(grid * 3 * GS * v->L.SL) : 0;
    const size_t n_tg = v == &c->str ? n_cp : 0;
    const size_t need = 2 * n_plane + n_cp + n_ds + 2 * n_tg;
    if (B > (int64_t)1 << 30 || need > cap)
        return fail(c, LASP_ERR_UNSUPPORTED, "lasp_eval_grad_static: B = " + std::to_string(B) + " spectra of " +
                    std::to_string(M.Ppad) + " padded pixels need " + std::to_string(need * sizeof(float)) +
                    " bytes of scratch, the static array holds " + std::to_string((size_t)LASP_STATIC_SCRATCH_BYTES) +
                    " (use lasp_eval_grad, which allocates)");
    DeviceGuard dg(c->device);
    cudaStream_t st = (cudaStream_t)stream;
    rc = ws_acquire(c, st);
    if (rc) return rc;
    float *Y = c->static_ws, *W = Y + n_plane, *per_cta = W + n_plane;
    CUDA_TRY(c, cudaMemsetAsync(per_cta, 0, (n_cp + n_ds + 2 * n_tg) * sizeof(float), st));
    lasp_v1_stage_kernel<<<(unsigned)B, 256, 0, st>>>(M, c->dnedge, flux, ivar, mask, Y, W);
    c->launches += 1;
    CUDA_TRY(c, cudaGetLastError());
    V1Args a;
    memset(&a, 0, sizeof(a));
    a.Y = Y; a.W = W; a.C1 = c->dC1; a.B = B;
    a.CP = per_cta;
    a.IS = c->dIS; a.SJ = c->dSJ;
    if (n_ds) a.DS = per_cta + n_cp;
    if (n_tg) { a.TG = per_cta + n_cp + n_ds; a.AG = a.TG + n_tg; }
    if (mma) { a.CF = c->dCF; a.ksteps = c->cf_ksteps; }
    a.ngroups = (int)ngroups;
    a.gparams = params; a.chi2 = chi2; a.grad_u = grad_u; a.cont = cont; a.status = status;
    return launch(c, kGrad, *v, a, st);
}

extern "C" int lasp_eval_model(lasp_ctx *c, int64_t B, const float *params, const float *cont,
                               const lasp_fit_opts *opts, float *model, void *stream)
{
    if (!c) return fail(nullptr, LASP_ERR_INVALID_ARG, "null ctx");
    if (B < 1 || !params || !cont || !model)
        return fail(c, LASP_ERR_INVALID_ARG, "lasp_eval_model: null pointer or B < 1");
    const Variant *v = nullptr;
    bool mma = false;
    int rc = resolve(c, opts, "lasp_eval_model", &v, &mma);
    if (rc) return rc;
    DeviceGuard dg(c->device);
    rc = workspace(c, B, *v, false, false, false);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    rc = ws_acquire(c, st);
    if (rc) return rc;
    V1Args a;
    base_args(c, *v, mma, B, a);
    a.gparams = params; a.mcont = cont; a.model = model;
    return launch(c, kModel, *v, a, st);
}

// Algorithmic FMA of one Adam step of one spectrum: SURVEY.md 8(d) formula, moment route,
// given the mean number of stencil taps (2H+1 averaged over spectra and pixels).
extern "C" double lasp_fma_per_spectrum_step(const lasp_ctx *c, double mean_taps)
{
    if (!c) return 0.0;
    const ModelDev &M = c->M;
    const double P = M.P, K = M.K, n1 = M.n1, W = mean_taps;
    double G = (2.0 * M.D + 1.0) * P + M.n_seg * n1 * n1 * n1 / 6.0;
    return 2.0 * K * P + 4.0 * W * P + (c->nonuniform ? 2.0 * W * P : 0.0) + G + 4.0 * n1 * P +
           M.n_seg * (n1 * n1 * n1 / 6.0 + 4.0 * n1 * n1) + 8.0 * P;
}

// The same count for the algorithm AS BUILT: Gram moments and factorisation only on the
// fraction `fresh_frac` of the steps that re-factor, one right-hand side and one continuum evaluation per step
// (2 (D+1) P, the residual-form solve being warm-started), the explicit-inverse product (D+1)^2 per segment.
extern "C" double lasp_fma_executed_per_spectrum_step(const lasp_ctx *c, double mean_taps, double fresh_frac)
{
    if (!c) return 0.0;
    const ModelDev &M = c->M;
    const double P = M.P, K = M.K, n1 = M.n1, W = mean_taps;
    // resident variant: mirrored octet pairs share the basis values (T_n(-t) = (-1)^n T_n(t)), so a sum over the basis
    // costs (D+1) P / 2 FMAs; moments, Cholesky and explicit inverse only on fresh steps
    const double half = c->res.ok ? 0.5 : 1.0;
    const double G = half * (2.0 * M.D + 1.0) * P + M.n_seg * (n1 * n1 * n1 / 6.0 + n1 * n1 * n1);
    return 2.0 * K * P + 4.0 * W * P + (c->nonuniform ? 2.0 * W * P : 0.0) + fresh_frac * G + half * 2.0 * n1 * P +
           M.n_seg * n1 * n1 + 8.0 * P;
}

// Counters of the last lasp_fit_batch on this ctx (synchronises with the device): out[0] = group-steps of the Adam
// loops, out[1] = those that re-accumulated the Gram moments and re-factorised.
extern "C" int lasp_last_fit_stats(lasp_ctx *c, double *out2)
{
    if (!c || !out2) return fail(c, LASP_ERR_INVALID_ARG, "lasp_last_fit_stats: null argument");
    DeviceGuard dg(c->device);
    unsigned long long h[2] = {0, 0};
    if (c->ws_pending) CUDA_TRY(c, cudaEventSynchronize(c->ws_event));
    CUDA_TRY(c, cudaMemcpy(h, c->dstats, sizeof(h), cudaMemcpyDeviceToHost));
    out2[0] = (double)h[0]; out2[1] = (double)h[1];
    return LASP_OK;
}

// ------------------------------------------------------------------------------------------
// lasp_resample_coeffs: the flux-conserving resampler (Eq. 2-4) applied once to a coefficient table
// ------------------------------------------------------------------------------------------
extern "C" int lasp_resample_coeffs(int cuda_device, int32_t n_terms, int32_t q, double lam1, double dlam1,
                                    const float *coef_model, int32_t n_pix, int32_t n_seg, const int32_t *seg_offset,
                                    const double *loglam, float *coef_obs, void *stream)
{
    if (n_terms < 1 || q < 1 || !(dlam1 > 0.0) || !coef_model || n_pix < 1 || n_seg < 1 || !seg_offset || !loglam || !coef_obs)
        return fail(nullptr, LASP_ERR_INVALID_ARG, "lasp_resample_coeffs: null pointer or bad size");
    if (seg_offset[0] != 0 || seg_offset[n_seg] != n_pix)
        return fail(nullptr, LASP_ERR_INVALID_ARG, "lasp_resample_coeffs: seg_offset must run from 0 to n_pix");
    // observed integration nodes: per segment, midpoints in log-wavelength between neighbouring pixels and half a
    // step beyond the first and the last pixel; lo[i], hi[i] are the two nodes of pixel i
    std::vector<double> nodes(2 * (size_t)n_pix);
    double *lo = nodes.data(), *hi = nodes.data() + n_pix;
    for (int s = 0; s < n_seg; ++s) {
        const int o = seg_offset[s], e = seg_offset[s + 1];
        if (e <= o) return fail(nullptr, LASP_ERR_INVALID_ARG, "lasp_resample_coeffs: empty segment");
        for (int j = o; j < e; ++j) {
            const double left = j > o ? 0.5 * (loglam[j - 1] + loglam[j])
                                      : loglam[j] - 0.5 * (e - o > 1 ? loglam[j + 1] - loglam[j] : 1e-4);
            const double right = j + 1 < e ? 0.5 * (loglam[j] + loglam[j + 1])
                                           : loglam[j] + 0.5 * (e - o > 1 ? loglam[j] - loglam[j - 1] : 1e-4);
            if (!(right > left)) return fail(nullptr, LASP_ERR_INVALID_ARG, "lasp_resample_coeffs: loglam must increase within a segment");
            lo[j] = pow(10.0, left); hi[j] = pow(10.0, right);
        }
    }
    int prev_dev = -1;
    cudaGetDevice(&prev_dev);
    if (cudaSetDevice(cuda_device) != cudaSuccess) { cudaGetLastError(); return fail(nullptr, LASP_ERR_CUDA, "lasp_resample_coeffs: cudaSetDevice failed"); }
    cudaStream_t st = (cudaStream_t)stream;
    double *dn = nullptr;
    int rc = LASP_OK;
    cudaError_t e = cudaMalloc(&dn, nodes.size() * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpyAsync(dn, nodes.data(), nodes.size() * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) {
        const dim3 grid((n_pix + 127) / 128, n_terms);
        lasp_resample_kernel<<<grid, 128, 0, st>>>(q, lam1 - 0.5 * dlam1, dlam1, coef_model, n_pix, dn, dn + n_pix, coef_obs);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // the node table is freed below: a one-off precompute, blocking
    if (e != cudaSuccess) rc = fail(nullptr, LASP_ERR_CUDA, std::string("lasp_resample_coeffs: ") + cudaGetErrorString(e));
    cudaFree(dn);
    if (prev_dev >= 0) cudaSetDevice(prev_dev);
    return rc;
}

// ------------------------------------------------------------------------------------------
// lasp_fit_batch_host: chunked host->device->fit->host pipeline (config 3)
// ------------------------------------------------------------------------------------------
static void hostpipe_free(lasp_ctx *c)
{
    lasp_ctx::HostPipe &h = c->hp;
    for (int s = 0; s < 2; ++s) {
        cudaFree(h.flux[s]); cudaFree(h.ivar[s]); cudaFree(h.mask[s]); cudaFree(h.init[s]);
        cudaFree(h.params[s]); cudaFree(h.cont[s]); cudaFree(h.chi2[s]); cudaFree(h.err[s]); cudaFree(h.status[s]); cudaFree(h.nsteps[s]); cudaFree(h.maskout[s]);
        h.flux[s] = h.ivar[s] = h.init[s] = h.params[s] = h.cont[s] = h.chi2[s] = h.err[s] = nullptr;
        h.mask[s] = nullptr; h.status[s] = nullptr; h.nsteps[s] = nullptr; h.maskout[s] = nullptr;
    }
    h.cap = 0;
}

static int hostpipe_reserve(lasp_ctx *c, int64_t chunk)
{
    lasp_ctx::HostPipe &h = c->hp;
    const ModelDev &M = c->M;
    if (!h.s_in) {
        CUDA_TRY(c, cudaStreamCreateWithFlags(&h.s_in, cudaStreamNonBlocking));
        CUDA_TRY(c, cudaStreamCreateWithFlags(&h.s_out, cudaStreamNonBlocking));
        CUDA_TRY(c, cudaStreamCreateWithFlags(&h.s_fit, cudaStreamNonBlocking));
        for (int s = 0; s < 2; ++s) {
            CUDA_TRY(c, cudaEventCreateWithFlags(&h.in_done[s], cudaEventDisableTiming));
            CUDA_TRY(c, cudaEventCreateWithFlags(&h.fit_done[s], cudaEventDisableTiming));
            CUDA_TRY(c, cudaEventCreateWithFlags(&h.out_done[s], cudaEventDisableTiming));
        }
    }
    if (chunk <= h.cap) return LASP_OK;
    hostpipe_free(c);
    const size_t n = (size_t)chunk;
    for (int s = 0; s < 2; ++s) {
        CUDA_TRY(c, cudaMalloc(&h.flux[s], n * M.P * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.ivar[s], n * M.P * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.mask[s], n * M.P));
        CUDA_TRY(c, cudaMalloc(&h.init[s], n * M.NP * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.params[s], n * M.NP * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.cont[s], n * M.nc * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.chi2[s], n * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.err[s], n * M.NP * sizeof(float)));
        CUDA_TRY(c, cudaMalloc(&h.status[s], n * sizeof(int32_t)));
        CUDA_TRY(c, cudaMalloc(&h.nsteps[s], n * sizeof(int32_t)));
        CUDA_TRY(c, cudaMalloc(&h.maskout[s], n * M.P));
    }
    h.cap = chunk;
    return LASP_OK;
}

static int hostpipe_run(lasp_ctx *c, int64_t B, const float *flux, const float *ivar, const uint8_t *mask,
                        const float *init, const lasp_fit_opts *opts, float *params, float *cont, float *chi2,
                        float *err, int32_t *status, int32_t *n_steps, uint8_t *mask_out, int64_t first, int64_t chunk)
{
    // chunk 0 holds `first` spectra, every later one `chunk` (the last one what is left)
    lasp_ctx::HostPipe &h = c->hp;
    const ModelDev &M = c->M;
    const int64_t nchunk = 1 + (B - first + chunk - 1) / chunk;
    auto span = [&](int64_t i, int64_t &o, int64_t &n) {
        o = i == 0 ? 0 : first + (i - 1) * chunk;
        n = i == 0 ? first : std::min(chunk, B - o);
    };
    auto upload = [&](int64_t i) -> int {
        const int s = (int)(i & 1);
        int64_t o, n;
        span(i, o, n);
        // the slot's previous fit (chunk i-2) must be done reading its inputs
        if (i >= 2) CUDA_TRY(c, cudaStreamWaitEvent(h.s_in, h.fit_done[s], 0));
        CUDA_TRY(c, cudaMemcpyAsync(h.flux[s], flux + o * M.P, (size_t)n * M.P * sizeof(float), cudaMemcpyHostToDevice, h.s_in));
        CUDA_TRY(c, cudaMemcpyAsync(h.ivar[s], ivar + o * M.P, (size_t)n * M.P * sizeof(float), cudaMemcpyHostToDevice, h.s_in));
        if (mask) CUDA_TRY(c, cudaMemcpyAsync(h.mask[s], mask + o * M.P, (size_t)n * M.P, cudaMemcpyHostToDevice, h.s_in));
        CUDA_TRY(c, cudaMemcpyAsync(h.init[s], init + o * M.NP, (size_t)n * M.NP * sizeof(float), cudaMemcpyHostToDevice, h.s_in));
        CUDA_TRY(c, cudaEventRecord(h.in_done[s], h.s_in));
        return LASP_OK;
    };
    int rc = upload(0);
    if (rc) return rc;
    for (int64_t i = 0; i < nchunk; ++i) {
        const int s = (int)(i & 1);
        int64_t o, n;
        span(i, o, n);
        if (i + 1 < nchunk) { rc = upload(i + 1); if (rc) return rc; }
        CUDA_TRY(c, cudaStreamWaitEvent(h.s_fit, h.in_done[s], 0));
        if (i >= 2) CUDA_TRY(c, cudaStreamWaitEvent(h.s_fit, h.out_done[s], 0));   // slot's old results copied out
        rc = lasp_fit_batch(c, n, h.flux[s], h.ivar[s], mask ? h.mask[s] : nullptr, h.init[s], opts, h.params[s],
                            cont ? h.cont[s] : nullptr, h.chi2[s], err ? h.err[s] : nullptr,
                            status ? h.status[s] : nullptr, n_steps ? h.nsteps[s] : nullptr,
                            mask_out ? h.maskout[s] : nullptr, h.s_fit);
        if (rc) return rc;
        CUDA_TRY(c, cudaEventRecord(h.fit_done[s], h.s_fit));
        CUDA_TRY(c, cudaStreamWaitEvent(h.s_out, h.fit_done[s], 0));
        CUDA_TRY(c, cudaMemcpyAsync(params + o * M.NP, h.params[s], (size_t)n * M.NP * sizeof(float), cudaMemcpyDeviceToHost, h.s_out));
        CUDA_TRY(c, cudaMemcpyAsync(chi2 + o, h.chi2[s], (size_t)n * sizeof(float), cudaMemcpyDeviceToHost, h.s_out));
        if (cont) CUDA_TRY(c, cudaMemcpyAsync(cont + o * M.nc, h.cont[s], (size_t)n * M.nc * sizeof(float), cudaMemcpyDeviceToHost, h.s_out));
        if (err) CUDA_TRY(c, cudaMemcpyAsync(err + o * M.NP, h.err[s], (size_t)n * M.NP * sizeof(float), cudaMemcpyDeviceToHost, h.s_out));
        if (status) CUDA_TRY(c, cudaMemcpyAsync(status + o, h.status[s], (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToHost, h.s_out));
        if (n_steps) CUDA_TRY(c, cudaMemcpyAsync(n_steps + o, h.nsteps[s], (size_t)n * sizeof(int32_t), cudaMemcpyDeviceToHost, h.s_out));
        if (mask_out) CUDA_TRY(c, cudaMemcpyAsync(mask_out + o * M.P, h.maskout[s], (size_t)n * M.P, cudaMemcpyDeviceToHost, h.s_out));
        CUDA_TRY(c, cudaEventRecord(h.out_done[s], h.s_out));
    }
    return LASP_OK;
}

extern "C" int lasp_fit_batch_host(lasp_ctx *c, int64_t B, const float *flux, const float *ivar,
                                   const uint8_t *mask, const float *init, const lasp_fit_opts *opts,
                                   float *params, float *cont, float *chi2, float *err, int32_t *status,
                                   int32_t *n_steps, uint8_t *mask_out, int64_t chunk)
{
    if (!c) return fail(nullptr, LASP_ERR_INVALID_ARG, "null ctx");
    if (B < 1 || !flux || !ivar || !init || !opts || !params || !chi2 || chunk < 0)
        return fail(c, LASP_ERR_INVALID_ARG, "lasp_fit_batch_host: null pointer, B < 1 or chunk < 0");
    DeviceGuard dg(c->device);
    // 0 = automatic.  Every launch costs a ramp and a tail of partly idle SMs, and nothing overlaps the first upload, so: a
    // short first chunk -- four full rounds of the persistent grid (4 x SMs x CTAs per SM x GS spectra), whose fit hides the
    // next upload -- then chunks as large as the device buffers allow (131,072 spectra).  Measured on config 1, 65,536
    // spectra: 70.7 k spectra/s with 8 equal chunks, 73.0 k with 2, 73.4 k with 4,736 + 60,800 (the device-resident call:
    // 74.0 k in the same run).  All sizes are multiples of GS, so the CTA groups are those of one lasp_fit_batch call over the whole batch.
    int64_t first_n = 0;
    if (chunk == 0) {
        const Variant *v = nullptr;
        bool mma = false;
        int rc0 = resolve(c, opts, "lasp_fit_batch_host", &v, &mma);
        if (rc0) return rc0;
        first_n = 4 * (int64_t)c->num_sms * v->cta_per_sm * GS;
        if (B < 2 * first_n) first_n = B;                       // too small to overlap anything
        chunk = std::min<int64_t>(131072, std::max<int64_t>(GS, (B - first_n + GS - 1) / GS * GS));
    } else {
        chunk = std::min<int64_t>(chunk, B);
        first_n = chunk;
    }
    int rc = hostpipe_reserve(c, std::max(first_n, chunk));
    if (rc) return rc;
    rc = hostpipe_run(c, B, flux, ivar, mask, init, opts, params, cont, chi2, err, status, n_steps, mask_out, first_n, chunk);
    // success or not, nothing of this call may still be in flight on the private streams when it returns: the
    // copies read and write the caller's buffers
    const std::string first = c->err;
    cudaError_t e1 = cudaStreamSynchronize(c->hp.s_in), e2 = cudaStreamSynchronize(c->hp.s_fit), e3 = cudaStreamSynchronize(c->hp.s_out);
    if (rc) { c->err = first; g_err = first; return rc; }
    if (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess) {
        const cudaError_t e = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
        return fail(c, LASP_ERR_CUDA, std::string("lasp_fit_batch_host: ") + cudaGetErrorString(e));
    }
    return LASP_OK;
}
