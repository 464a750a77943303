// nep_highl.cuh -- k_highl: descriptor + network + partial forces for l_max = 5..8 ("l_max > 4";
// included by nep_b200.cu after nep_gen.cuh).  The paper uses l_max = 4 throughout, for which
// k_main / k_gen carry the 24 real harmonics written out; this kernel is the general form: the harmonics and their
// gradients come from recurrences, one thread per atom, per-atom arrays in local memory.  It is a correctness path
// (parity-tested against the oracle's literal Legendre double sum), not a tuned one.
//
//   b_{l,m,c}(u) = Pi_l^m(z) c_m,  b_{l,m,s}(u) = Pi_l^m(z) s_m,   Pi_l^m = d^m P_l / dz^m,
//   c_m + i s_m = (x + i y)^m,     P_l(u1 . u2) = sum_m C_lm [b_lmc b'_lmc + b_lms b'_lms],  C_lm = (2 - delta_m0)(l-m)!/(l+m)!
// (the addition theorem, Eq. 17-18 route to Eq. 13 with n' = n).  With B_lm the homogeneous form of b_lm,
//   grad(g(r) b_lm(u)) = g' b_lm u + (g / r)(grad B_lm(u) - l b_lm u)      (the same identity k_gen uses),
//   B = r^(l-m) Pi_l^m(z/r) C_m(x, y):  grad B = C_m [h_r u + (0, 0, Pi_l^{m+1})] + Pi_l^m grad C_m  at r = 1,
//   h_r = (l - m) Pi_l^m - z Pi_l^{m+1},  grad c_m = m (c_{m-1}, -s_{m-1}, 0),  grad s_m = m (s_{m-1}, c_{m-1}, 0).
#pragma once

constexpr int kHLMaxL = 8;
constexpr int kHLMaxLM = 80;          // sum_{l=1..8} (2l+1)
constexpr int kHLMaxN = 16;
constexpr int kHLMaxD = kHLMaxN + kHLMaxN * kHLMaxL;

struct HighLParams {
    float rcR_inv, rcA_inv;
    int NR, NA, LMAX, H, D, Dp, N, capR;
    const float* params;              // staged fp32 layout w1[H][Dp] | b1[H] | w2[H] | b2
    float* q_out;                     // nullable parity hooks, [D][N] caller order
    float* fp_out;
};

// b[k], grad B[k] (k runs over l = 1..L, then m = 0, 1c, 1s, 2c, 2s, ...) and the l and C_lm of each component
__device__ __forceinline__ int highl_basis(float x, float y, float z, int L, float* b, float* gx, float* gy, float* gz,
                                           int* lof, float* clm) {
    float c[kHLMaxL + 1], s[kHLMaxL + 1];
    c[0] = 1.f; s[0] = 0.f;
    for (int m = 1; m <= L; ++m) { c[m] = x * c[m - 1] - y * s[m - 1]; s[m] = x * s[m - 1] + y * c[m - 1]; }
    float Pi[kHLMaxL + 1][kHLMaxL + 2];                   // Pi[l][m], zero for m > l
    for (int l = 0; l <= L; ++l)
        for (int m = 0; m <= L + 1; ++m) Pi[l][m] = 0.f;
    float dfact = 1.f;                                      // (2m - 1)!!
    for (int m = 0; m <= L; ++m) {
        if (m > 0) dfact *= (float)(2 * m - 1);
        Pi[m][m] = dfact;
        if (m + 1 <= L) Pi[m + 1][m] = (float)(2 * m + 1) * z * dfact;
        for (int l = m + 2; l <= L; ++l)
            Pi[l][m] = ((float)(2 * l - 1) * z * Pi[l - 1][m] - (float)(l + m - 1) * Pi[l - 2][m]) / (float)(l - m);
    }
    int k = 0;
    for (int l = 1; l <= L; ++l) {
        float ratio = 1.f;                                  // (l - m)! / (l + m)!
        for (int m = 0; m <= l; ++m) {
            if (m > 0) ratio /= (float)((l + m) * (l - m + 1));
            const float H = Pi[l][m], Hz = Pi[l][m + 1], Hr = (float)(l - m) * H - z * Hz;
            for (int cs = 0; cs < (m == 0 ? 1 : 2); ++cs) {
                const float C = cs == 0 ? c[m] : s[m];
                float dCx = 0.f, dCy = 0.f;
                if (m > 0) {
                    dCx = (float)m * (cs == 0 ? c[m - 1] : s[m - 1]);
                    dCy = (float)m * (cs == 0 ? -s[m - 1] : c[m - 1]);
                }
                b[k] = H * C;
                gx[k] = C * Hr * x + H * dCx;
                gy[k] = C * Hr * y + H * dCy;
                gz[k] = C * (Hr * z + Hz);
                lof[k] = l;
                clm[k] = (m == 0 ? 1.f : 2.f) * ratio;
                ++k;
            }
        }
    }
    return k;
}

__global__ void __launch_bounds__(64) k_highl(SysDev d, const __grid_constant__ HighLParams P) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int N = P.N;
    if (i >= N) return;
    const int NR = P.NR, NA = P.NA, L = P.LMAX, D = P.D, Dp = P.Dp, H = P.H, capR = P.capR;
    const int nR = d.nnR[i], nA = d.nnA[i];
    float q[kHLMaxD], Fp[kHLMaxD];
    float sums[kHLMaxN][kHLMaxLM];                          // s[n][lm] = sum_j g_n(r_ij) b_lm(r^_ij)
    float b[kHLMaxLM], gx[kHLMaxLM], gy[kHLMaxLM], gz[kHLMaxLM], clm[kHLMaxLM];
    int lof[kHLMaxLM];
    int nlm = 0;
    for (int v = 0; v < D; ++v) q[v] = 0.f;
    for (int n = 0; n < NA; ++n)
        for (int m = 0; m < kHLMaxLM; ++m) sums[n][m] = 0.f;
    auto slot_of = [&](int k) { return k < nA ? k : capR - 1 - (k - nA); };
    // ---- descriptor, Eq. 12 and Eq. 13 (through Eq. 17-18) ----
    for (int k = 0; k < nR; ++k) {
        const float4 e = d.rec[rix(slot_of(k), i, N)];
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        const float rinv = inv_norm(r2), r = r2 * rinv;
        float g[kHLMaxN], dg[kHLMaxN];
        radial_gd<kHLMaxN>(r, P.rcR_inv, 1.f, 1.f, g, dg);
        for (int n = 0; n < NR; ++n) q[n] += g[n];
        if (k < nA) {
            radial_gd<kHLMaxN>(r, P.rcA_inv, 1.f, 1.f, g, dg);
            nlm = highl_basis(e.x * rinv, e.y * rinv, e.z * rinv, L, b, gx, gy, gz, lof, clm);
            for (int n = 0; n < NA; ++n)
                for (int m = 0; m < nlm; ++m) sums[n][m] = fmaf(g[n], b[m], sums[n][m]);
        }
    }
    if (nA == 0) nlm = highl_basis(0.f, 0.f, 1.f, L, b, gx, gy, gz, lof, clm);     // lof / clm for the loops below
    for (int n = 0; n < NA; ++n)
        for (int m = 0; m < nlm; ++m) q[NR + n * L + lof[m] - 1] = fmaf(clm[m] * sums[n][m], sums[n][m], q[NR + n * L + lof[m] - 1]);
    // ---- network, Eq. 21-22 (minus biases), and Fp = dU/dq ----
    const float* b1 = P.params + (size_t)H * Dp;
    const float* w2 = b1 + H;
    float U = -w2[H];
    for (int v = 0; v < D; ++v) Fp[v] = 0.f;
    for (int mu = 0; mu < H; ++mu) {
        const float* w = P.params + (size_t)mu * Dp;
        float a = -b1[mu];
        for (int v = 0; v < D; ++v) a = fmaf(w[v], q[v], a);
        float t, dd;
        tanh_sech2(a, &t, &dd);
        U = fmaf(w2[mu], t, U);
        const float gm = w2[mu] * dd;
        for (int v = 0; v < D; ++v) Fp[v] = fmaf(gm, w[v], Fp[v]);
    }
    d.Us[i] = U;
    if (P.q_out || P.fp_out) {
        const int row = d.perm[i];
        for (int v = 0; v < D; ++v) {
            if (P.q_out) P.q_out[(size_t)v * N + row] = q[v];
            if (P.fp_out) P.fp_out[(size_t)v * N + row] = Fp[v];
        }
    }
    // ---- partial forces, Eq. 24 and Eq. 25: A[n][lm] = 2 Fp_nl C_lm s_nlm in place of s ----
    for (int n = 0; n < NA; ++n)
        for (int m = 0; m < nlm; ++m) sums[n][m] *= 2.f * clm[m] * Fp[NR + n * L + lof[m] - 1];
    float fsx = 0.f, fsy = 0.f, fsz = 0.f;
    for (int k = 0; k < nR; ++k) {
        const int slot = slot_of(k);
        const float4 e = d.rec[rix(slot, i, N)];
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        const float rinv = inv_norm(r2), r = r2 * rinv;
        const float x = e.x * rinv, y = e.y * rinv, z = e.z * rinv;
        float g[kHLMaxN], dg[kHLMaxN];
        radial_gd<kHLMaxN>(r, P.rcR_inv, 1.f, 1.f, g, dg);
        float cr = 0.f;
        for (int n = 0; n < NR; ++n) cr = fmaf(Fp[n], dg[n], cr);
        float px = cr * x, py = cr * y, pz = cr * z;
        if (k < nA) {
            radial_gd<kHLMaxN>(r, P.rcA_inv, 1.f, rinv, g, dg);            // g <- g_n / r
            highl_basis(x, y, z, L, b, gx, gy, gz, lof, clm);
            float R = 0.f, vx = 0.f, vy = 0.f, vz = 0.f;
            for (int m = 0; m < nlm; ++m) {
                float Sp = 0.f, St = 0.f;                                  // S'_m = sum_n A g_n',  S_m / r = sum_n A g_n / r
                for (int n = 0; n < NA; ++n) { Sp = fmaf(sums[n][m], dg[n], Sp); St = fmaf(sums[n][m], g[n], St); }
                R = fmaf(b[m], Sp - (float)lof[m] * St, R);
                vx = fmaf(St, gx[m], vx); vy = fmaf(St, gy[m], vy); vz = fmaf(St, gz[m], vz);
            }
            px += fmaf(R, x, vx); py += fmaf(R, y, vy); pz += fmaf(R, z, vz);
        }
        fsx += px; fsy += py; fsz += pz;
        d.p[(size_t)i * capR + slot] = make_float4(px, py, pz, 0.f);
    }
    d.Fself[i] = make_float4(fsx, fsy, fsz, 0.f);
}
