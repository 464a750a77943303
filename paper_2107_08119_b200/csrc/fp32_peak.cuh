// fp32_peak.cuh -- register-resident FMA-chain microbenchmark: the measured FP32 (non-tensor) peak that
// bench.py reports beside the derived 148 x 128 x 2 x f figure.
// Included by nep_b200.cu; exported as nep_measure_fp32_peak().
#pragma once

template <bool PACKED>
__global__ void __launch_bounds__(256) k_fma_chain(float* out, int iters, float a, float b) {
    float acc[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) acc[k] = (float)(threadIdx.x + k);
    for (int it = 0; it < iters; ++it) {
        if (PACKED) {
#pragma unroll
            for (int k = 0; k < 16; k += 2) {
                // fma.rn.f32x2 (sm_100+): two FP32 FMAs per lane per instruction
                unsigned long long v, aa, bb;
                asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(acc[k]), "f"(acc[k + 1]));
                asm("mov.b64 %0, {%1, %1};" : "=l"(aa) : "f"(a));
                asm("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
                asm("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(v) : "l"(aa), "l"(bb));
                asm("mov.b64 {%0, %1}, %2;" : "=f"(acc[k]), "=f"(acc[k + 1]) : "l"(v));
            }
        } else {
#pragma unroll
            for (int k = 0; k < 16; ++k) acc[k] = fmaf(acc[k], a, b);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += acc[k];
    if (s == 123.456f) out[0] = s;      // keeps the chain alive
}
