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

// Three further register-resident patterns, launched like k_main (64-thread blocks, 4 per SM):
//   MODE 0  FFMA whose three source registers all differ (no operand reuse): the register-file read limit
//   MODE 1  the descriptor contraction of k_main:  s2[n][mm] += {g_n, g_n} * {b_2mm, b_2mm+1}   (48 FFMA2)
//   MODE 2  the force contraction of k_main:  Sp[mm] += A[n][mm] * {g'_n, g'_n};  St[mm] += A[n][mm] * {g_n, g_n}   (96 FFMA2)
// They bound what the packed-FMA inner loops of k_main can reach with 8 warps per SM.
template <int MODE>
__global__ void __launch_bounds__(64) k_fma_pattern(float* out, int iters, float a, float b) {
    typedef unsigned long long u64;
    auto pk = [](float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; };
    auto f2 = [](u64 x, u64 y, u64 z) { u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(x), "l"(y), "l"(z)); return d; };
    float acc = 0.f;
    if (MODE == 0) {
        float x[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = threadIdx.x * 0.001f + i * a;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < 16; ++i) x[i] = fmaf(x[i], x[(i + 5) & 15], x[(i + 9) & 15]);
        }
#pragma unroll
        for (int i = 0; i < 16; ++i) acc += x[i];
    } else {
        u64 s2[8][6], Sp[6], St[6];
        float g[8], bb[12];
#pragma unroll
        for (int n = 0; n < 8; ++n)
#pragma unroll
            for (int m = 0; m < 6; ++m) s2[n][m] = pk(threadIdx.x + n, m + b);
#pragma unroll
        for (int m = 0; m < 6; ++m) { Sp[m] = pk(0.f, 0.f); St[m] = pk(0.f, 0.f); }
#pragma unroll
        for (int n = 0; n < 8; ++n) g[n] = a + n;
#pragma unroll
        for (int m = 0; m < 12; ++m) bb[m] = b + m;
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int n = 0; n < 8; ++n) g[n] *= a;                 // the operands change every iteration
            if (MODE == 1) {
                u64 bp[6];
#pragma unroll
                for (int m = 0; m < 6; ++m) bp[m] = pk(bb[2 * m], bb[2 * m + 1]);
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const u64 gp = pk(g[n], g[n]);
#pragma unroll
                    for (int m = 0; m < 6; ++m) s2[n][m] = f2(gp, bp[m], s2[n][m]);
                }
            } else {
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const u64 dp = pk(g[n], g[n]), gp = pk(bb[n], bb[n]);
#pragma unroll
                    for (int m = 0; m < 6; ++m) { Sp[m] = f2(s2[n][m], dp, Sp[m]); St[m] = f2(s2[n][m], gp, St[m]); }
                }
            }
        }
#pragma unroll
        for (int n = 0; n < 8; ++n)
#pragma unroll
            for (int m = 0; m < 6; ++m) acc += (float)(s2[n][m] & 0xffff);
#pragma unroll
        for (int m = 0; m < 6; ++m) acc += (float)((Sp[m] ^ St[m]) & 0xffff);
    }
    if (acc == 123.456f) out[0] = acc;      // keeps the chains alive
}
