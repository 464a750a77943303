// nep_main.cuh -- k_main: descriptor + network + partial forces (included by nep_b200.cu inside its
// anonymous namespace, after SysDev and nep_math.cuh).
//
// One thread per atom, one warp per block.  k_order sorts every window of 256 atoms by neighbour
// count, so the 32 atoms of a warp have (nearly) equal trip counts and the hardware block scheduler
// balances the windows' light and heavy warps.  Per atom, in order:
//   P1  radial descriptor q_n (Eq. 12) over all r < r_c^R neighbours, read once from global memory;
//       the angular neighbours are left in shared memory as {r^_ij, r_ij}
//   P2  angular sums s[n][lm] = sum_j g_n(r_ij) b_lm(r^_ij) (Eq. 17-18 route to Eq. 13) in two halves of
//       12 lm (96 register accumulators each); half 0 is parked in shared memory
//   P3  network (Eq. 21-22) and Fp = dU/dq, weights read from the kernel-parameter constant bank
//   P4  partial forces of the radial-only neighbours (Eq. 24)
//   P5  partial forces of the angular neighbours (Eq. 24 + Eq. 25), half 1 then half 0
// Nothing but U_i, sum_j p_ij and the partial forces p_ij leaves the chip.
#pragma once

constexpr int kRowsS = 24;          // angular neighbour rows staged in shared memory (more: read from global)
constexpr int kWin = 256;           // k_order's sort window (atoms)
struct MainParams {
    float rcR_inv, rcA_inv;
    int H, N, capR;
};

// Packed FP32x2 arithmetic (sm_100+: FFMA2 issues two FMAs per lane in one instruction slot).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 ffma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

__device__ __forceinline__ float inv_norm(float r2) {
    float rinv;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(r2));       // MUFU.RSQ, no denormal fix-up (r2 >> 0)
    return rinv * fmaf(-0.5f * r2 * rinv, rinv, 1.5f);      // one Newton step: < 1 ulp
}
__device__ __forceinline__ float fast_rcp(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));            // MUFU.RCP, 1 ulp
    return r;
}

// ------------------------------------------------------------------------------------------------
// k_order: order[w*256 + t] = the atom of window w with the t-th largest key (nA, then nR - nA).
// Entries past N are -1.  One block of 256 threads per window; rank by counting.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kWin) k_order(SysDev d, int N) {
    __shared__ int key[kWin];
    const int t = threadIdx.x;
    const int i = blockIdx.x * kWin + t;
    int k = -1;
    if (i < N) {
        const int nA = d.nnA[i], nR = d.nnR[i];
        k = (nA << 8) | (nR - nA);
    }
    key[t] = k;
    __syncthreads();
    int rank = 0;
#pragma unroll 8
    for (int j = 0; j < kWin; ++j) {
        const int kj = key[j];
        rank += (kj > k) || (kj == k && j < t);
    }
    d.order[blockIdx.x * kWin + rank] = i < N ? i : -1;
}

// ------------------------------------------------------------------------------------------------
// k_main
// ------------------------------------------------------------------------------------------------
// angular sums of one half: s2[n][mm] = {s[n][2mm], s[n][2mm+1]} over the half's 12 lm, and the
// half's share of q_nl = sum_m C_lm s_nlm^2 (Eq. 17 with n' = n)
template <int HALF, int NR, int NA, class LoadNbr>
__device__ __forceinline__ void desc_half(int nA, float rcA_inv, const LoadNbr& load_nbr, f32x2 (&s2)[NA][kHalfLM / 2],
                                          float* q) {
    constexpr int NP = kHalfLM / 2;
    constexpr float C[kNumLM] = {NEP_CLM_LIST};
#pragma unroll
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) s2[n][mm] = pack2(0.f, 0.f);
    for (int k = 0; k < nA; ++k) {
        float x, y, z, r, om;
        load_nbr(k, x, y, z, r, om);
        float g[NA];
        radial_g<NA>(r, rcA_inv, om, g);
        float b[kHalfLM];
        ylm_basis_half<HALF>(x, y, z, b);
        f32x2 bp[NP];
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) bp[mm] = pack2(b[2 * mm], b[2 * mm + 1]);
#pragma unroll
        for (int n = 0; n < NA; ++n) {
            const f32x2 gp = pack2(g[n], g[n]);
#pragma unroll
            for (int mm = 0; mm < NP; ++mm) s2[n][mm] = ffma2(gp, bp[mm], s2[n][mm]);
        }
    }
#pragma unroll
    for (int n = 0; n < NA; ++n) {
        float ql[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) {
            float s0, s1;
            unpack2(s2[n][mm], s0, s1);
            ql[half_l<HALF>(2 * mm) - 1] = fmaf(C[half_m<HALF>(2 * mm)] * s0, s0, ql[half_l<HALF>(2 * mm) - 1]);
            ql[half_l<HALF>(2 * mm + 1) - 1] = fmaf(C[half_m<HALF>(2 * mm + 1)] * s1, s1, ql[half_l<HALF>(2 * mm + 1) - 1]);
        }
        if (HALF == 0) { q[NR + 4 * n + 0] = ql[0]; q[NR + 4 * n + 3] = ql[3]; }
        else           { q[NR + 4 * n + 1] = ql[1]; q[NR + 4 * n + 2] = ql[2]; }
    }
}

// s -> A[n][lm] = 2 Fp_nl C_lm s_nlm, in place
template <int HALF, int NR, int NA>
__device__ __forceinline__ void scale_half(f32x2 (&s2)[NA][kHalfLM / 2], const float* Fp) {
    constexpr float C[kNumLM] = {NEP_CLM_LIST};
#pragma unroll
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int mm = 0; mm < kHalfLM / 2; ++mm) {
            float s0, s1;
            unpack2(s2[n][mm], s0, s1);
            s0 *= (2.f * C[half_m<HALF>(2 * mm)]) * Fp[NR + 4 * n + half_l<HALF>(2 * mm) - 1];
            s1 *= (2.f * C[half_m<HALF>(2 * mm + 1)]) * Fp[NR + 4 * n + half_l<HALF>(2 * mm + 1) - 1];
            s2[n][mm] = pack2(s0, s1);
        }
}

// Angular partial force (Eq. 25 through the addition theorem) of neighbour (x, y, z, r) from one half:
//   p = R r^ + V,  R = sum_m b_m (S'_m - l_m S_m / r),  V = sum_m (S_m / r) grad B_m(r^)
//   S'_m = sum_n A[n][m] g_n'(r),   S_m / r = sum_n A[n][m] g_n(r) / r
template <int HALF, int NA>
__device__ __forceinline__ void force_half(const f32x2 (&A2)[NA][kHalfLM / 2], float x, float y, float z,
                                           const float* gs, const float* dg, float& px, float& py, float& pz) {
    constexpr int NP = kHalfLM / 2;
    f32x2 Sp2[NP], St2[NP];
    {
        const f32x2 dp = pack2(dg[0], dg[0]), gp = pack2(gs[0], gs[0]);
        const f32x2 zero = pack2(0.f, 0.f);
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) { Sp2[mm] = ffma2(A2[0][mm], dp, zero); St2[mm] = ffma2(A2[0][mm], gp, zero); }
    }
#pragma unroll
    for (int n = 1; n < NA; ++n) {
        const f32x2 dp = pack2(dg[n], dg[n]), gp = pack2(gs[n], gs[n]);
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) {
            Sp2[mm] = ffma2(A2[n][mm], dp, Sp2[mm]);
            St2[mm] = ffma2(A2[n][mm], gp, St2[mm]);
        }
    }
    float Sq[kHalfLM], St[kHalfLM];
#pragma unroll
    for (int mm = 0; mm < NP; ++mm) {
        unpack2(Sp2[mm], Sq[2 * mm], Sq[2 * mm + 1]);
        unpack2(St2[mm], St[2 * mm], St[2 * mm + 1]);
    }
    float b[kHalfLM];
    ylm_basis_half<HALF>(x, y, z, b);
    float R0 = 0.f, R1 = 0.f;
#pragma unroll
    for (int k = 0; k < kHalfLM; k += 2) {
        R0 = fmaf(b[k], fmaf(-(float)half_l<HALF>(k), St[k], Sq[k]), R0);
        R1 = fmaf(b[k + 1], fmaf(-(float)half_l<HALF>(k + 1), St[k + 1], Sq[k + 1]), R1);
    }
    const float R = R0 + R1;
    float vx, vy, vz;
    ylm_grad_half<HALF>(x, y, z, St, &vx, &vy, &vz);
    px = fmaf(R, x, vx); py = fmaf(R, y, vy); pz = fmaf(R, z, vz);
}

template <int NR, int NA, bool MULTI>
__global__ void __launch_bounds__(32, NEP_MAIN_MIN_BLOCKS) k_main(SysDev d, MainParams P,
                                                                 const __grid_constant__ NetParams W) {
    constexpr int D = NR + 4 * NA;
    constexpr int NP = kHalfLM / 2;
    extern __shared__ __align__(16) float sm[];
    float4* srec = reinterpret_cast<float4*>(sm);                      // [kRowsS][32] {r^_ij, r_ij} of angular neighbours
    float2* spark = reinterpret_cast<float2*>(sm + kRowsS * 32 * 4);   // [NA*6][32] parked s (half 0)
    float* som = sm + kRowsS * 32 * 4 + NA * kHalfLM * 32;            // [kRowsS][32] omega_ij (MULTI only)

    const int lane = threadIdx.x;
    const int N = P.N;
    const int i_ord = d.order[blockIdx.x * 32 + lane];
    const bool active = i_ord >= 0;
    const int i = active ? i_ord : 0;
    const int nR = active ? d.nnR[i] : 0, nA = active ? d.nnA[i] : 0;
    const int nO = nR - nA;
    const float4* grec = d.rec + i;                  // record of slot s: grec[(size_t)s * N]
    const float* zrow = W.zz + (MULTI ? d.type_s[i] * kMaxTypes : 0);
    auto omega_of = [&](const float4& e) { return MULTI ? zrow[__float_as_int(e.w) & (kMaxTypes - 1)] : 1.f; };

    // neighbour k (an angular one) as unit vector, distance and Eq. 19 weight
    auto load_nbr = [&](int k, float& x, float& y, float& z, float& r, float& om) {
        if (k < kRowsS) {
            const float4 e = srec[k * 32 + lane];
            x = e.x; y = e.y; z = e.z; r = e.w;
            om = MULTI ? som[k * 32 + lane] : 1.f;
        } else {
            const float4 e = grec[(size_t)k * N];
            const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
            const float rinv = inv_norm(r2);
            x = e.x * rinv; y = e.y * rinv; z = e.z * rinv; r = r2 * rinv;
            om = omega_of(e);
        }
    };

    // ---- P1: radial descriptor, Eq. 12; stages the angular neighbours ----
    float q[D];
#pragma unroll
    for (int v = 0; v < D; ++v) q[v] = 0.f;
    for (int k0 = 0; k0 < nR; k0 += 4) {
        float4 e[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int kk = min(k0 + u, nR - 1);
            const int slot = kk < nA ? kk : P.capR - 1 - (kk - nA);
            e[u] = __ldg(&grec[(size_t)slot * N]);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int kk = k0 + u;
            if (kk < nR) {
                const float r2 = e[u].x * e[u].x + e[u].y * e[u].y + e[u].z * e[u].z;
                const float rinv = inv_norm(r2);
                const float r = r2 * rinv;
                const float om = omega_of(e[u]);
                float g[NR];
                radial_g<NR>(r, P.rcR_inv, om, g);
#pragma unroll
                for (int n = 0; n < NR; ++n) q[n] += g[n];
                if (kk < nA && kk < kRowsS) {
                    srec[kk * 32 + lane] = make_float4(e[u].x * rinv, e[u].y * rinv, e[u].z * rinv, r);
                    if (MULTI) som[kk * 32 + lane] = om;
                }
            }
        }
    }

    // ---- P2: angular sums, half 0 (parked in shared memory) then half 1 (stays in registers) ----
    f32x2 s2[NA][NP];
    desc_half<0, NR, NA>(nA, P.rcA_inv, load_nbr, s2, q);
#pragma unroll
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) {
            float s0, s1;
            unpack2(s2[n][mm], s0, s1);
            spark[(n * NP + mm) * 32 + lane] = make_float2(s0, s1);
        }
    desc_half<1, NR, NA>(nA, P.rcA_inv, load_nbr, s2, q);

    // ---- P3: network Eq. 21-22 (minus biases) and Fp = dU/dq; two neurons per iteration ----
    float Fp[D];
#pragma unroll
    for (int v = 0; v < D; ++v) Fp[v] = 0.f;
    const int H = P.H;
    const float* b1 = W.w + H * D;
    const float* w2 = b1 + H;
    float U = -w2[H];                                                   // - b2
    for (int mu = 0; mu < H; mu += 2) {
        const bool two = mu + 1 < H;
        const int mu1 = two ? mu + 1 : mu;
        const float* r0 = W.w + mu * D;
        const float* r1 = W.w + mu1 * D;
        float a0 = -b1[mu], a1 = 0.f, c0 = -b1[mu1], c1 = 0.f;
#pragma unroll
        for (int v = 0; v + 1 < D; v += 2) {
            a0 = fmaf(r0[v], q[v], a0); a1 = fmaf(r0[v + 1], q[v + 1], a1);
            c0 = fmaf(r1[v], q[v], c0); c1 = fmaf(r1[v + 1], q[v + 1], c1);
        }
        if (D & 1) { a0 = fmaf(r0[D - 1], q[D - 1], a0); c0 = fmaf(r1[D - 1], q[D - 1], c0); }
        float t0, d0, t1, d1;
        tanh_sech2(a0 + a1, &t0, &d0);
        tanh_sech2(c0 + c1, &t1, &d1);
        const float g0 = w2[mu] * d0, g1 = two ? w2[mu1] * d1 : 0.f;
        U = fmaf(w2[mu], t0, U);
        if (two) U = fmaf(w2[mu1], t1, U);
#pragma unroll
        for (int v = 0; v < D; ++v) Fp[v] = fmaf(g0, r0[v], fmaf(g1, r1[v], Fp[v]));
    }
    if (active) d.Us[i] = U;

    // ---- P4: radial-only neighbours, Eq. 24 ----
    float fsx = 0.f, fsy = 0.f, fsz = 0.f;
    float4* prow = d.p + (size_t)i * P.capR;         // p_ij lives at the record's own slot
    for (int k0 = 0; k0 < nO; k0 += 4) {
        float4 e[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) e[u] = __ldg(&grec[(size_t)(P.capR - 1 - min(k0 + u, nO - 1)) * N]);
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (k0 + u < nO) {
                const float r2 = e[u].x * e[u].x + e[u].y * e[u].y + e[u].z * e[u].z;
                const float rinv = inv_norm(r2);
                float gs[NR], dg[NR];
                radial_gd<NR>(r2 * rinv, P.rcR_inv, omega_of(e[u]), 1.f, gs, dg);
                float c0 = 0.f, c1 = 0.f;
#pragma unroll
                for (int n = 0; n + 1 < NR; n += 2) { c0 = fmaf(Fp[n], dg[n], c0); c1 = fmaf(Fp[n + 1], dg[n + 1], c1); }
                if (NR & 1) c0 = fmaf(Fp[NR - 1], dg[NR - 1], c0);
                const float c = (c0 + c1) * rinv;
                const float px = c * e[u].x, py = c * e[u].y, pz = c * e[u].z;
                fsx += px; fsy += py; fsz += pz;
                prow[P.capR - 1 - (k0 + u)] = make_float4(px, py, pz, 0.f);
            }
        }
    }

    // ---- P5: angular neighbours, Eq. 24 + Eq. 25: half 1 (with the radial family), then half 0 ----
    scale_half<1, NR, NA>(s2, Fp);
    for (int k = 0; k < nA; ++k) {
        float x, y, z, r, om;
        load_nbr(k, x, y, z, r, om);
        const float rinv = fast_rcp(r);
        float gs[NA], dg[NA];
        radial_gd<NA>(r, P.rcA_inv, om, rinv, gs, dg);
        float px, py, pz;
        force_half<1, NA>(s2, x, y, z, gs, dg, px, py, pz);
        float gR[NR], dR[NR];
        radial_gd<NR>(r, P.rcR_inv, om, 1.f, gR, dR);
        float c0 = 0.f, c1 = 0.f;
#pragma unroll
        for (int n = 0; n + 1 < NR; n += 2) { c0 = fmaf(Fp[n], dR[n], c0); c1 = fmaf(Fp[n + 1], dR[n + 1], c1); }
        if (NR & 1) c0 = fmaf(Fp[NR - 1], dR[NR - 1], c0);
        const float c = c0 + c1;
        prow[k] = make_float4(fmaf(c, x, px), fmaf(c, y, py), fmaf(c, z, pz), 0.f);
    }
#pragma unroll
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) {
            const float2 v = spark[(n * NP + mm) * 32 + lane];
            s2[n][mm] = pack2(v.x, v.y);
        }
    scale_half<0, NR, NA>(s2, Fp);
    for (int k = 0; k < nA; ++k) {
        const float4 pold = prow[k];                 // half 1's share (this thread wrote it above)
        float x, y, z, r, om;
        load_nbr(k, x, y, z, r, om);
        const float rinv = fast_rcp(r);
        float gs[NA], dg[NA];
        radial_gd<NA>(r, P.rcA_inv, om, rinv, gs, dg);
        float px, py, pz;
        force_half<0, NA>(s2, x, y, z, gs, dg, px, py, pz);
        px += pold.x; py += pold.y; pz += pold.z;
        fsx += px; fsy += py; fsz += pz;
        prow[k] = make_float4(px, py, pz, 0.f);
    }
    if (active) d.Fself[i] = make_float4(fsx, fsy, fsz, 0.f);
}
