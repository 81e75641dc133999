// pipe_probe.cu -- two micro-benchmarks behind DESIGN.md 6.4 ("why the table contractions stay on the FP32 pipe").
// Test infrastructure (tests/test_pipe_probe.py compiles and runs it on the GPU box); not part of the library.
//
//  probe_tcgen05: one CTA per SM issues `iters` tcgen05.mma.cta_group::1.kind::tf32 of shape M = 128, N = n_cols, K = 8
//      (A: 128 pixels x 8 terms and B: n_cols x 8 terms from shared memory, canonical K-major no-swizzle layout,
//      accumulator in TMEM), the A descriptor cycling over `n_tiles` different 4 KB tiles as a streamed coefficient
//      table would, and the MMAs rotating over `n_acc` independent accumulators.  Returns cycles per MMA (min over CTAs of clock64 around issue -> tcgen05.commit -> mbarrier wait)
//      and the accumulator of CTA 0 for a numerical check (inputs are small integers: exact in tf32).
//      This is the shape the fit kernel's table contractions would have on the tensor pipe: T[pixel][spectrum] =
//      sum_k C[k][pixel] phi_k[spectrum] with N = [phi_hi | phi_lo] of GS spectra (N = 8 for GS = 4, 16 for GS = 8).
//  probe_ffma: the FP32-pipe ceiling of the fit kernel's own inner block, acc[4][8] += p[g] * c[i] from registers,
//      `grid` x `threads` threads; returns TFLOP/s from CUDA-event time.
#include <cuda_runtime.h>
#include <stdint.h>

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// shared-memory matrix descriptor, K-major, SWIZZLE_NONE: core matrix = 8 rows x 16 bytes stored contiguously;
// LBO = byte distance between core matrices adjacent along K, SBO = between 8-row groups along M / N
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo)
{
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFF);
    d |= (uint64_t)((lbo >> 4) & 0x3FFF) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFF) << 32;
    d |= (uint64_t)1 << 46;   // descriptor version of sm_100
    return d;
}

// instruction descriptor, kind::tf32: D = F32, A = B = TF32, both K-major, dense
__host__ __device__ constexpr uint32_t umma_idesc_tf32(int M, int N)
{
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}

// element (r, k) of a [rows x 8] tf32 tile in the canonical layout used here: 8-row group mg = r / 8 at mg * 256 bytes,
// K core kc = k / 4 at kc * 128 bytes, row r % 8 at 16 bytes, element k % 4 at 4 bytes
__device__ __forceinline__ int tile_off(int r, int k) { return (r >> 3) * 64 + (k >> 2) * 32 + (r & 7) * 4 + (k & 3); }

extern __shared__ __align__(1024) float probe_smem[];

__global__ void __launch_bounds__(128, 1)
tcgen05_probe_kernel(int iters, int n_tiles, int n_cols, int n_acc, float *dout, unsigned long long *cycles, int *err)
{
    __shared__ uint64_t bar;
    __shared__ uint32_t tmem_base_s;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    float *As = probe_smem;                         // n_tiles tiles of 128 x 8 (4 KB each)
    float *Bs = probe_smem + n_tiles * 1024;        // one tile of n_cols x 8
    for (int i = tid; i < n_tiles * 1024 + n_cols * 8; i += 128) probe_smem[i] = 0.f;
    __syncthreads();
    for (int i = tid; i < n_tiles * 128 * 8; i += 128) {
        const int t = i / 1024, r = (i / 8) % 128, k = i % 8;
        As[t * 1024 + tile_off(r, k)] = (float)(((r + 3 * k + t) % 7) - 3);      // small integers: exact in tf32
    }
    for (int i = tid; i < n_cols * 8; i += 128) {
        const int n = i / 8, k = i % 8;
        Bs[tile_off(n, k)] = (float)(((2 * n + k) % 5) - 2);
    }
    uint32_t ncol_alloc = 32;
    while ((int)ncol_alloc < n_cols * n_acc) ncol_alloc <<= 1;       // power of two >= 32
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "r"(ncol_alloc));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
    }
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(&bar)));
        asm volatile("fence.mbarrier_init.release.cluster;");
    }
    // make the generic-proxy writes of the tiles visible to the async proxy (the tensor core reads shared memory)
    asm volatile("fence.proxy.async.shared::cta;");
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    const uint32_t tmem = tmem_base_s;
    long long t0 = 0, t1 = 0;
    bool ok = true;
    if (tid == 0) {
        const uint32_t a0 = smem_u32(As), b0 = smem_u32(Bs), idesc = umma_idesc_tf32(128, n_cols);
        const uint64_t bdesc = umma_desc(b0, 128, 256);
        // lean issue loop (one thread issues for the CTA): tile and accumulator indices by masks (powers of two), the
        // first n_acc MMAs overwrite their accumulators, the rest accumulate
        const uint64_t abase = umma_desc(a0, 128, 256);
        const int tmask = n_tiles - 1, amask = n_acc - 1;
        t0 = clock64();
        for (int i = 0; i < n_acc; ++i)
            asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                         "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                         ::"r"(tmem + (uint32_t)(i * n_cols)), "l"(abase + (uint64_t)((i & tmask) << 8)), "l"(bdesc), "r"(idesc), "r"(0u));
        for (int i = n_acc; i < iters; i += 8) {
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int ii = i + u;
                asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                             "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
                             ::"r"(tmem + (uint32_t)((ii & amask) * n_cols)), "l"(abase + (uint64_t)((ii & tmask) << 8)), "l"(bdesc),
                               "r"(idesc), "r"(1u));
            }
        }
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(&bar)));
        uint32_t done = 0;
        for (int spin = 0; spin < (1 << 20) && !done; ++spin)
            asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                         : "=r"(done) : "r"(smem_u32(&bar)), "r"(0u));
        t1 = clock64();
        ok = done != 0;
        if (!ok) atomicExch(err, 1);
        cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
    }
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;");
    if (blockIdx.x == 0 && *((volatile int *)err) == 0) {
        // accumulator row = TMEM lane = 32 * warp + lane; 16 columns per load; the n_acc accumulators are summed
        for (int c0 = 0; c0 < n_cols; c0 += 16) {
          float sum[16];
          for (int j = 0; j < 16; ++j) sum[j] = 0.f;
          for (int q = 0; q < n_acc; ++q) {
            uint32_t r[16];
            const uint32_t taddr = tmem + ((uint32_t)(32 * warp) << 16) + (uint32_t)(q * n_cols + c0);
            asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                         : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
                           "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                         : "r"(taddr));
            asm volatile("tcgen05.wait::ld.sync.aligned;");
            for (int j = 0; j < 16; ++j) sum[j] += __uint_as_float(r[j]);
          }
          for (int j = 0; j < 16 && c0 + j < n_cols; ++j) dout[(32 * warp + lane) * n_cols + c0 + j] = sum[j];
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(ncol_alloc));
}

// out: dout [128 * n_cols] accumulator of CTA 0; returns min cycles per MMA over the CTAs, or < 0 on error
extern "C" double probe_tcgen05(int iters, int n_tiles, int n_cols, int n_acc, float *dout_host)
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (n_cols < 16 || n_cols > 256 || n_cols % 16 || n_tiles < 1 || n_tiles > 32 || (n_tiles & (n_tiles - 1)) || n_acc < 1 ||
        (n_acc & (n_acc - 1)) || n_cols * n_acc > 512 || iters < n_acc + 8 || (iters - n_acc) % 8) return -1.0;
    float *dout = nullptr; unsigned long long *cyc = nullptr; int *err = nullptr;
    cudaMalloc(&dout, 128 * n_cols * sizeof(float));
    cudaMalloc(&cyc, sms * sizeof(unsigned long long));
    cudaMalloc(&err, sizeof(int));
    cudaMemset(err, 0, sizeof(int));
    const size_t smem = (size_t)(n_tiles * 1024 + n_cols * 8) * sizeof(float);
    if (cudaFuncSetAttribute(tcgen05_probe_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return -2.0;
    tcgen05_probe_kernel<<<sms, 128, smem>>>(iters, n_tiles, n_cols, n_acc, dout, cyc, err);
    if (cudaDeviceSynchronize() != cudaSuccess) return -3.0;
    int herr = 0;
    cudaMemcpy(&herr, err, sizeof(int), cudaMemcpyDeviceToHost);
    unsigned long long hc[256];
    cudaMemcpy(hc, cyc, sms * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
    cudaMemcpy(dout_host, dout, 128 * n_cols * sizeof(float), cudaMemcpyDeviceToHost);
    cudaFree(dout); cudaFree(cyc); cudaFree(err);
    if (herr) return -4.0;
    unsigned long long best = ~0ull;
    for (int i = 0; i < sms; ++i) best = hc[i] < best ? hc[i] : best;
    return (double)best / iters;
}

// ---------------------------------------------------------------------------------------------------------------------
__global__ void ffma_probe_kernel(int iters, float *out, const float *in)
{
    float acc[4][8], p[4], c[8];
#pragma unroll
    for (int g = 0; g < 4; ++g) { p[g] = in[g] + threadIdx.x * 1e-9f; }
#pragma unroll
    for (int i = 0; i < 8; ++i) c[i] = in[4 + i];
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[g][i] = 0.f;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
                for (int i = 0; i < 8; ++i) acc[g][i] = fmaf(p[g], c[i], acc[g][i]);
#pragma unroll
            for (int i = 0; i < 8; ++i) c[i] += 1e-7f;     // keeps the block from being folded; 8 FADD per 256 FFMA
        }
    }
    float s = 0.f;
#pragma unroll
    for (int g = 0; g < 4; ++g)
#pragma unroll
        for (int i = 0; i < 8; ++i) s += acc[g][i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// the same block with packed FP32 (fma.rn.f32x2 -> FFMA2): half the instructions for the same FMAs
__device__ __forceinline__ void ffma2(unsigned long long &d, unsigned long long a, unsigned long long b)
{
    asm volatile("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
}
__device__ __forceinline__ unsigned long long pack2(float x, float y)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(x), "f"(y));
    return r;
}
__global__ void ffma2_probe_kernel(int iters, float *out, const float *in)
{
    unsigned long long acc[4][4], p[4], c[4];
    for (int g = 0; g < 4; ++g) { float v = in[g] + threadIdx.x * 1e-9f; p[g] = pack2(v, v); }
    for (int i = 0; i < 4; ++i) c[i] = pack2(in[4 + 2 * i], in[5 + 2 * i]);
    for (int g = 0; g < 4; ++g) for (int i = 0; i < 4; ++i) acc[g][i] = 0ull;
    const unsigned long long inc = pack2(1e-7f, 1e-7f), one = pack2(1.f, 1.f);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
#pragma unroll
            for (int g = 0; g < 4; ++g)
#pragma unroll
                for (int i = 0; i < 4; ++i) ffma2(acc[g][i], p[g], c[i]);
#pragma unroll
            for (int i = 0; i < 4; ++i) ffma2(c[i], inc, one);
        }
    }
    float s = 0.f;
    for (int g = 0; g < 4; ++g) for (int i = 0; i < 4; ++i) { float2 f = *(float2 *)&acc[g][i]; s += f.x + f.y; }
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
static double ffma_run(int grid, int threads, int iters, bool packed)
{
    float *out = nullptr, *in = nullptr;
    cudaMalloc(&out, (size_t)grid * threads * sizeof(float));
    cudaMalloc(&in, 12 * sizeof(float));
    float h[12];
    for (int i = 0; i < 12; ++i) h[i] = 1.f + 0.01f * i;
    cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice);
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    if (packed) ffma2_probe_kernel<<<grid, threads>>>(iters / 10 + 1, out, in); else ffma_probe_kernel<<<grid, threads>>>(iters / 10 + 1, out, in);
    cudaEventRecord(e0);
    if (packed) ffma2_probe_kernel<<<grid, threads>>>(iters, out, in); else ffma_probe_kernel<<<grid, threads>>>(iters, out, in);
    cudaEventRecord(e1);
    if (cudaDeviceSynchronize() != cudaSuccess) return -1.0;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    cudaFree(out); cudaFree(in);
    const double flop = 2.0 * 256.0 * iters * (double)grid * threads;
    return flop / (ms * 1e-3) / 1e12;
}

extern "C" double probe_ffma(int grid, int threads, int iters) { return ffma_run(grid, threads, iters, false); }
extern "C" double probe_ffma2(int grid, int threads, int iters) { return ffma_run(grid, threads, iters, true); }
