// nep_desc64.cuh -- k_desc64: descriptor and network in fp64 for multi-species models (included by
// nep_b200.cu after nep_main.cuh).
//
// Eq. 19 multiplies every radial function by sqrt(Z_i Z_j).  With Z = 82 / 52 the
// descriptor reaches ~4e3 while the network's pre-activations cancel to O(1): fp32 cannot hold the
// 1e-5 eV / 1e-4 RMS-force bars there -- not even the fp32 rounding of r_ij is admissible
// (dq/dr ~ 4e3 / A).  So for n_types > 1 this kernel evaluates, per atom and in double, straight from
// the fp64 positions:  q_n (Eq. 12), s[n][lm] and q_nl (Eq. 17-18 route to Eq. 13), the network
// (Eq. 21-22) and Fp = dU/dq, and hands U_i, Fp and s (rounded to fp32, relative error 6e-8) to k_main,
// which then runs only its force phases P4 / P5 (their terms do not cancel).
// One thread per atom in k_order's window-sorted order (the column k_main uses); s lives in local
// memory: this is the accuracy path, not the throughput path.
#pragma once

template <int NR, int NA>
__global__ void __launch_bounds__(64) k_desc64(SysDev d, Box b, const __grid_constant__ Desc64Params P,
                                               const double* __restrict__ par /* w1[H][D] | b1[H] | w2[H] | b2 */) {
    constexpr int D = NR + 4 * NA;
    constexpr int NP = kHalfLM / 2;
    constexpr double C[kNumLM] = {NEP_CLM_LIST};
    constexpr int LOF[kNumLM] = {NEP_LOF_LIST};
    const size_t gcol = (size_t)blockIdx.x * 64 + threadIdx.x;
    const size_t npad = (size_t)gridDim.x * 64;
    const int i = d.order[gcol];
    if (i < 0) return;
    const int N = P.N;
    const int nR = d.nnR[i], nA = d.nnA[i];
    const double4 pi = d.xs4[i];
    const double* zrow = P.zz + (int)__double_as_longlong(pi.w) * kMaxTypes;

    double q[D];
#pragma unroll
    for (int v = 0; v < D; ++v) q[v] = 0.0;
    double s[NA][kNumLM];
    for (int n = 0; n < NA; ++n)
        for (int m = 0; m < kNumLM; ++m) s[n][m] = 0.0;

    for (int k = 0; k < nR; ++k) {
        const int slot = k < nA ? k : P.capR - 1 - (k - nA);
        const int j = d.jrev[(size_t)slot * N + i] & kJMask;
        const double4 pj = d.xs4[j];
        const double dx = min_image(pj.x - pi.x, b.L[0], b.invL[0]);
        const double dy = min_image(pj.y - pi.y, b.L[1], b.invL[1]);
        const double dz = min_image(pj.z - pi.z, b.L[2], b.invL[2]);
        const double r = sqrt(dx * dx + dy * dy + dz * dz);
        const double om = zrow[(int)__double_as_longlong(pj.w) & (kMaxTypes - 1)];
        double g[NR > NA ? NR : NA];
        radial_g64<NR>(r, P.rcR, om, g);
#pragma unroll
        for (int n = 0; n < NR; ++n) q[n] += g[n];                       // Eq. 12
        if (k < nA) {
            radial_g64<NA>(r, P.rcA, om, g);
            double bb[kNumLM];
            const double rinv = 1.0 / r;
            ylm_basis64(dx * rinv, dy * rinv, dz * rinv, bb);
            for (int n = 0; n < NA; ++n)
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) s[n][m] += g[n] * bb[m];   // Eq. 18 in real form
        }
    }
    for (int n = 0; n < NA; ++n) {
        double ql[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
        for (int m = 0; m < kNumLM; ++m) ql[LOF[m] - 1] += C[m] * s[n][m] * s[n][m];   // Eq. 17 with n' = n
#pragma unroll
        for (int l = 0; l < 4; ++l) q[NR + 4 * n + l] = ql[l];
    }

    // network, Eq. 21-22 with the minus biases, and Fp = dU/dq
    const int H = P.H;
    const double* b1 = par + (size_t)H * D;
    const double* w2 = b1 + H;
    double U = -w2[H];
    double Fp[D];
#pragma unroll
    for (int v = 0; v < D; ++v) Fp[v] = 0.0;
    for (int mu = 0; mu < H; ++mu) {
        const double* w = par + (size_t)mu * D;
        double a0 = -b1[mu], a1 = 0.0;
#pragma unroll
        for (int v = 0; v + 1 < D; v += 2) { a0 += w[v] * q[v]; a1 += w[v + 1] * q[v + 1]; }
        if (D & 1) a0 += w[D - 1] * q[D - 1];
        const double a = a0 + a1;
        const double e = exp(-2.0 * fabs(a));
        const double inv = 1.0 / (1.0 + e);
        const double t = copysign((1.0 - e) * inv, a);                   // tanh(a)
        const double gm = w2[mu] * 4.0 * e * inv * inv;                  // w2 (1 - tanh^2 a), no cancellation
        U += w2[mu] * t;
#pragma unroll
        for (int v = 0; v < D; ++v) Fp[v] += gm * w[v];
    }
    d.Us[i] = (float)U;
#pragma unroll
    for (int v = 0; v < D; ++v) d.FpG[(size_t)v * npad + gcol] = (float)Fp[v];
    // s in k_main's parked layout: half h, pair mm of radial index n
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) {
            d.spark0[(size_t)(n * NP + mm) * npad + gcol] =
                make_float2((float)s[n][half_m<0>(2 * mm)], (float)s[n][half_m<0>(2 * mm + 1)]);
            d.spark1[(size_t)(n * NP + mm) * npad + gcol] =
                make_float2((float)s[n][half_m<1>(2 * mm)], (float)s[n][half_m<1>(2 * mm + 1)]);
        }
}
