// bench_probe.cu — a register-resident FP32 FMA loop used by bench.py to MEASURE the FMA-pipe
// peak of the device the solver runs on (the denominator context for the "alu" roofline; SURVEY.md
// 8(d)).  Built as its own helper library (libpinmpc_benchprobe.so); not part of libpinmpc.so or its ABI.
#include <cuda_runtime.h>

__global__ void __launch_bounds__(256) k_probe_fma(int iters, float a, float b, float *out)
{
    float v0 = threadIdx.x * 1e-3f, v1 = v0 + 1.0f, v2 = v0 + 2.0f, v3 = v0 + 3.0f;
    float v4 = v0 + 4.0f, v5 = v0 + 5.0f, v6 = v0 + 6.0f, v7 = v0 + 7.0f;
#pragma unroll 1
    for (int i = 0; i < iters; i++) {
#pragma unroll
        for (int r = 0; r < 16; r++) {
            v0 = fmaf(v0, a, b); v1 = fmaf(v1, a, b); v2 = fmaf(v2, a, b); v3 = fmaf(v3, a, b);
            v4 = fmaf(v4, a, b); v5 = fmaf(v5, a, b); v6 = fmaf(v6, a, b); v7 = fmaf(v7, a, b);
        }
    }
    float s = ((v0 + v1) + (v2 + v3)) + ((v4 + v5) + (v6 + v7));
    if (s == 123.456f) out[0] = s;      // keep the loop alive
}

// Enqueue the probe: `blocks` CTAs of 256 threads, each thread 128 * iters FMAs.
// Returns the number of FLOPs the launch performs (2 per FMA), or 0 on a launch error.
extern "C" double bench_probe_fma(int blocks, int iters, float *d_out, void *stream)
{
    k_probe_fma<<<blocks, 256, 0, (cudaStream_t)stream>>>(iters, 0.999f, 0.001f, d_out);
    if (cudaGetLastError() != cudaSuccess) return 0.0;
    return 2.0 * 128.0 * (double)iters * 256.0 * (double)blocks;
}
