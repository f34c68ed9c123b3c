// FP32 issue-rate probe: the denominator of the "alu" roofline of the pair kernels.
// Not a step of the path: it measures what this GPU sustains on dependent-free fused multiply-adds, scalar
// (FFMA) and packed (FFMA2, sm_100), so that bench.py can quote the pair loops against a measured peak
// instead of the nominal 148 SM x 128 lanes x 2 flop x clock.
#include "sph_ctx.cuh"

#define PROBE_ACC 16
template <int PACKED>
__global__ void __launch_bounds__(256)
k_fp32_probe(float* __restrict__ out, int iters, float a, float b) {
    float acc[PROBE_ACC];
#pragma unroll
    for (int k = 0; k < PROBE_ACC; ++k) acc[k] = (float)(threadIdx.x + k);
    if (PACKED) {
        const float2 a2 = make_float2(a, a), b2 = make_float2(b, b);
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < PROBE_ACC; k += 2) {
                float2 v = __ffma2_rn(make_float2(acc[k], acc[k + 1]), a2, b2);
                acc[k] = v.x; acc[k + 1] = v.y;
            }
        }
    } else {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int k = 0; k < PROBE_ACC; ++k) acc[k] = fmaf(acc[k], a, b);
        }
    }
    float s = 0.0f;
#pragma unroll
    for (int k = 0; k < PROBE_ACC; ++k) s += acc[k];
    if (s == 12345.678f) out[0] = s;           // never true in practice: keeps the loop alive
}

extern "C" int sph_fp32_probe(sph_ctx* c, int packed, int iters, double* tflops, double* ms_out) {
    if (!c || !tflops) return SPH_ERR_NULL;
    if (iters < 1) return sph_fail(c, SPH_ERR_BAD_ARG, "iters must be positive");
    const int blocks = c->sm_count * 8, threads = 256;
    cudaEvent_t e0, e1;
    SPH_CUDA_OK(c, cudaEventCreate(&e0)); SPH_CUDA_OK(c, cudaEventCreate(&e1));
    float best = 1.0e30f;
    for (int rep = 0; rep < 4; ++rep) {        // first repetition warms up
        SPH_CUDA_OK(c, cudaEventRecord(e0, c->stream));
        if (packed) k_fp32_probe<1><<<blocks, threads, 0, c->stream>>>((float*)c->hminmax, iters, 0.999f, 0.001f);
        else        k_fp32_probe<0><<<blocks, threads, 0, c->stream>>>((float*)c->hminmax, iters, 0.999f, 0.001f);
        SPH_CUDA_OK(c, cudaEventRecord(e1, c->stream));
        SPH_CUDA_OK(c, cudaEventSynchronize(e1));
        float ms = 0.0f; SPH_CUDA_OK(c, cudaEventElapsedTime(&ms, e0, e1));
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    const double flop = 2.0 * PROBE_ACC * (double)iters * (double)blocks * threads;
    *tflops = flop / ((double)best * 1.0e-3) * 1.0e-12;
    if (ms_out) *ms_out = best;
    return SPH_OK;
}
