// nep_main.cuh -- k_main: descriptor + network + partial forces (included by nep_b200.cu inside its
// anonymous namespace, after SysDev and nep_math.cuh).
//
// Block = 128 threads = 64 atoms x 2 lanes.  Lane h of an atom's pair owns the angular radial
// indices n = h*NH .. h*NH+NH-1 (all 24 lm of each) and every second hidden neuron, so both lanes run
// one instruction stream; q, dU/dq and the per-neighbour partial force cross the pair with __shfl_xor.
//
// Neighbour records of the block's 64 atoms are staged once into shared memory with cp.async
// (16 B per thread, rows of 64 records = 1 KB contiguous in the [slot][atom] layout), so the three
// passes over the neighbours read shared memory instead of stalling on global loads.
#pragma once

struct MainParams {
    float rcR_inv, rcA_inv;
    int H, N, capR, capMD;
};

constexpr int kMainThreads = 128;
constexpr int kMainAtoms = kMainThreads / 2;

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

__device__ __forceinline__ float inv_norm(float r2) {
    float rinv;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(rinv) : "f"(r2));       // MUFU.RSQ, no denormal fix-up (r2 >> 0)
    return rinv * fmaf(-0.5f * r2 * rinv, rinv, 1.5f);      // one Newton step: < 1 ulp
}

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

template <int NR, int NA, bool MULTI>
__global__ void __launch_bounds__(kMainThreads, NEP_MAIN_MIN_BLOCKS) k_main(SysDev d, MainParams P,
                                                                          const float* __restrict__ params,
                                                                          const float* __restrict__ sqrtzz) {
    constexpr int NH = (NA + 1) / 2;
    constexpr int D = NR + 4 * NA;
    constexpr int Dp = (D + 3) & ~3;
    constexpr float C[kNumLM] = {NEP_CLM_LIST};
    constexpr int LOF[kNumLM] = {NEP_LOF_LIST};
    extern __shared__ __align__(16) float sm[];
    __shared__ int s_max[2];
    const int H = P.H, N = P.N;
    const int nfl = H * Dp + 2 * H + 1;
    float* szz = sm + ((nfl + 3) & ~3);
    float4* srec = reinterpret_cast<float4*>(szz + kMaxTypes * kMaxTypes);     // [rows][64] neighbour records
    float* scr = reinterpret_cast<float*>(srec + P.capR * kMainAtoms);         // [rows][64] radial-family scalars

    const int tid = threadIdx.x;
    const int a_loc = tid >> 1;                       // atom within the block
    const int i0 = blockIdx.x * kMainAtoms;
    const bool active = i0 + a_loc < N;
    const int i = active ? i0 + a_loc : N - 1;
    const int h = tid & 1;
    const unsigned PAIR = 3u << (tid & 30);           // the atom's lane pair (trip counts differ across pairs)
    const int nR = d.nnR[i], nA = d.nnA[i];
    const int nO = nR - nA;

    // ---- stage weights and this block's neighbour records ----
    if (tid < 2) s_max[tid] = 0;
    __syncthreads();
    {
        int mA = nA, mO = nO;
        mA = __reduce_max_sync(0xffffffffu, mA);
        mO = __reduce_max_sync(0xffffffffu, mO);
        if ((tid & 31) == 0) { atomicMax(&s_max[0], mA); atomicMax(&s_max[1], mO); }
    }
    for (int k = tid; k < nfl; k += kMainThreads) sm[k] = params[k];
    if (MULTI) for (int k = tid; k < kMaxTypes * kMaxTypes; k += kMainThreads) szz[k] = sqrtzz[k];
    __syncthreads();
    const int maxA = s_max[0], maxO = s_max[1];
    {
        // smem row r < maxA holds global slot r; row maxA + o holds global slot capR-1-o
        const int rows = maxA + maxO;
        const int col = tid & (kMainAtoms - 1);
        const int src_atom = min(i0 + col, N - 1);
        for (int r = tid >> 6; r < rows; r += 2) {
            const int slot = r < maxA ? r : P.capR - 1 - (r - maxA);
            cp_async16(&srec[r * kMainAtoms + col], &d.rec[(size_t)slot * N + src_atom]);
        }
        cp_async_wait_all();
        if (MULTI) {        // Eq. 19: replace the neighbour's type by omega_ij = sqrt(Z_i Z_j), once
            const float* zr = szz + d.type_s[src_atom] * kMaxTypes;
            for (int r = tid >> 6; r < rows; r += 2) {
                float* w = &srec[r * kMainAtoms + col].w;
                *w = zr[__float_as_int(*w) & 7];
            }
        }
    }
    __syncthreads();
    const float4* myrec = srec + a_loc;
    float* mycr = scr + a_loc;
    auto omega = [&](const float4& e) { return MULTI ? e.w : 1.f; };

    // ---- radial descriptor, Eq. 12: neighbours split between the two lanes ----
    float q[Dp];
#pragma unroll
    for (int v = 0; v < Dp; ++v) q[v] = 0.f;
    for (int k = h; k < nR; k += 2) {
        const float4 e = myrec[(k < nA ? k : maxA + (k - nA)) * kMainAtoms];
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        const float rinv = inv_norm(r2);
        float g[NR];
        radial_fn<NR, false>(r2 * rinv, P.rcR_inv, omega(e), g, nullptr);
#pragma unroll
        for (int n = 0; n < NR; ++n) q[n] += g[n];
    }
#pragma unroll
    for (int n = 0; n < NR; ++n) q[n] += __shfl_xor_sync(PAIR, q[n], 1);

    // ---- angular sums s[n][lm] = sum_j g_n(r_ij) b_lm(r^_ij)  (Eq. 18 in real form) ----
    constexpr int NP = kNumLM / 2;           // lm pairs: s2[a][mm] = {s[a][2mm], s[a][2mm+1]}
    f32x2 s2[NH][NP];
#pragma unroll
    for (int k = 0; k < NH; ++k)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) s2[k][mm] = pack2(0.f, 0.f);
    for (int k = 0; k < nA; ++k) {
        const float4 e = myrec[k * kMainAtoms];
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        const float rinv = inv_norm(r2);
        float g[NA];
        radial_fn<NA, false>(r2 * rinv, P.rcA_inv, omega(e), g, nullptr);
        float b[kNumLM];
        ylm_basis(e.x * rinv, e.y * rinv, e.z * rinv, b);
        f32x2 bp[NP];
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) bp[mm] = pack2(b[2 * mm], b[2 * mm + 1]);
#pragma unroll
        for (int a = 0; a < NH; ++a) {
            const float go = h ? (a + NH < NA ? g[a + NH < NA ? a + NH : 0] : 0.f) : g[a];
            const f32x2 gp = pack2(go, go);
#pragma unroll
            for (int mm = 0; mm < NP; ++mm) s2[a][mm] = ffma2(gp, bp[mm], s2[a][mm]);
        }
    }
    float s[NH][kNumLM];
#pragma unroll
    for (int a = 0; a < NH; ++a)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) unpack2(s2[a][mm], s[a][2 * mm], s[a][2 * mm + 1]);

    // ---- q_nl = sum_m C_lm s_nlm^2 (Eq. 17 with n' = n), exchanged across the pair ----
    {
        float qa[NH][4];
#pragma unroll
        for (int a = 0; a < NH; ++a) {
#pragma unroll
            for (int l = 0; l < 4; ++l) qa[a][l] = 0.f;
#pragma unroll
            for (int m = 0; m < kNumLM; ++m) qa[a][LOF[m] - 1] = fmaf(C[m] * s[a][m], s[a][m], qa[a][LOF[m] - 1]);
        }
#pragma unroll
        for (int a = 0; a < NH; ++a)
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                const float mine = qa[a][l];
                const float other = __shfl_xor_sync(PAIR, mine, 1);
                q[NR + 4 * a + l] = h ? other : mine;                           // n = a       (lane 0's)
                if (a + NH < NA) q[NR + 4 * (a + NH) + l] = h ? mine : other;   // n = a + NH  (lane 1's)
            }
    }

    // ---- network Eq. 21-22 and Fp = dU/dq.  Lane h evaluates neurons mu = h, h+2, ... (two per
    //      iteration for ILP); the partial U and Fp are summed across the pair. ----
    float Fp[Dp];
    const float* b1 = sm + H * Dp;
    const float* w2 = b1 + H;
    float U = h ? 0.f : -w2[H];                                              // - b2 (once)
    {
        f32x2 qp[Dp / 2], Fpp[Dp / 2];
#pragma unroll
        for (int v = 0; v < Dp / 2; ++v) { qp[v] = pack2(q[2 * v], q[2 * v + 1]); Fpp[v] = pack2(0.f, 0.f); }
        for (int mu = h; mu < H; mu += 4) {
            const bool two = mu + 2 < H;
            const int mu1 = two ? mu + 2 : mu;
            const ulonglong2* r0 = reinterpret_cast<const ulonglong2*>(sm + mu * Dp);
            const ulonglong2* r1 = reinterpret_cast<const ulonglong2*>(sm + mu1 * Dp);
            f32x2 a0 = pack2(-b1[mu], 0.f), a1 = pack2(-b1[mu1], 0.f), a2 = pack2(0.f, 0.f), a3 = pack2(0.f, 0.f);
#pragma unroll
            for (int v = 0; v < Dp / 4; ++v) {
                const ulonglong2 w0 = r0[v], w1 = r1[v];
                a0 = ffma2(w0.x, qp[2 * v], a0); a2 = ffma2(w0.y, qp[2 * v + 1], a2);
                a1 = ffma2(w1.x, qp[2 * v], a1); a3 = ffma2(w1.y, qp[2 * v + 1], a3);
            }
            float x0, x1, x2, x3, y0, y1, y2, y3;
            unpack2(a0, x0, x1); unpack2(a2, x2, x3); unpack2(a1, y0, y1); unpack2(a3, y2, y3);
            float t0, d0, t1, d1;
            tanh_sech2((x0 + x1) + (x2 + x3), &t0, &d0);
            tanh_sech2((y0 + y1) + (y2 + y3), &t1, &d1);
            const float g0 = w2[mu] * d0, g1 = two ? w2[mu1] * d1 : 0.f;
            U = fmaf(w2[mu], t0, U);
            if (two) U = fmaf(w2[mu1], t1, U);
            const f32x2 g0p = pack2(g0, g0), g1p = pack2(g1, g1);
#pragma unroll
            for (int v = 0; v < Dp / 4; ++v) {
                const ulonglong2 w0 = r0[v], w1 = r1[v];
                Fpp[2 * v] = ffma2(g0p, w0.x, ffma2(g1p, w1.x, Fpp[2 * v]));
                Fpp[2 * v + 1] = ffma2(g0p, w0.y, ffma2(g1p, w1.y, Fpp[2 * v + 1]));
            }
        }
#pragma unroll
        for (int v = 0; v < Dp / 2; ++v) unpack2(Fpp[v], Fp[2 * v], Fp[2 * v + 1]);
    }
    U += __shfl_xor_sync(PAIR, U, 1);
#pragma unroll
    for (int v = 0; v < D; ++v) Fp[v] += __shfl_xor_sync(PAIR, Fp[v], 1);
    if (active && h == 0) d.Us[i] = U;

    // ---- A[n][lm] = 2 Fp_nl C_lm s_nlm, in place ----
#pragma unroll
    for (int a = 0; a < NH; ++a)
#pragma unroll
        for (int m = 0; m < kNumLM; ++m) {
            const float f0 = Fp[NR + 4 * a + LOF[m] - 1];
            const float f1 = (a + NH < NA) ? Fp[NR + 4 * (a + NH < NA ? a + NH : 0) + LOF[m] - 1] : 0.f;
            s[a][m] *= 2.f * C[m] * (h ? f1 : f0);
        }
#pragma unroll
    for (int a = 0; a < NH; ++a)
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) s2[a][mm] = pack2(s[a][2 * mm], s[a][2 * mm + 1]);
    // ---- partial forces, Eq. 23-25 ----
    float fsx = 0.f, fsy = 0.f, fsz = 0.f;
    float4* prow = d.p + (size_t)i * P.capR;       // p_ij lives at the record's own slot
    // radial family (Eq. 24), neighbours split between the lanes: radial-only neighbours are finished
    // here; for angular neighbours the scalar c = sum_n Fp_n g_n'(r)/r is parked in shared memory
    for (int k = h; k < nR; k += 2) {
        const int row = k < nA ? k : maxA + (k - nA);
        const float4 e = myrec[row * kMainAtoms];
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        const float rinv = inv_norm(r2);
        float gr[NR], dgr[NR];
        radial_fn<NR, true>(r2 * rinv, P.rcR_inv, omega(e), gr, dgr);
        float c0 = 0.f, c1 = 0.f;
#pragma unroll
        for (int n = 0; n + 1 < NR; n += 2) { c0 = fmaf(Fp[n], dgr[n], c0); c1 = fmaf(Fp[n + 1], dgr[n + 1], c1); }
        if (NR & 1) c0 = fmaf(Fp[NR - 1], dgr[NR - 1], c0);
        const float c = (c0 + c1) * rinv;
        if (k < nA) {
            mycr[row * kMainAtoms] = c;
        } else {
            const float px = c * e.x, py = c * e.y, pz = c * e.z;
            fsx += px; fsy += py; fsz += pz;
            if (active) prow[P.capR - 1 - (k - nA)] = make_float4(px, py, pz, 0.f);
        }
    }
    __syncwarp(PAIR);
    for (int k = 0; k < nA; ++k) {          // angular family (Eq. 25): both lanes, own half of n
        const float4 e = myrec[k * kMainAtoms];
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        const float rinv = inv_norm(r2);
        const float x = e.x * rinv, y = e.y * rinv, z = e.z * rinv;
        float g[NA], dg[NA];
        radial_fn<NA, true>(r2 * rinv, P.rcA_inv, omega(e), g, dg);
        f32x2 Sp2[NP], St2[NP];
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) { Sp2[mm] = pack2(0.f, 0.f); St2[mm] = pack2(0.f, 0.f); }
#pragma unroll
        for (int a = 0; a < NH; ++a) {
            const int a1 = a + NH < NA ? a + NH : 0;
            const float ga = (h ? (a + NH < NA ? g[a1] : 0.f) : g[a]) * rinv;       // g_n / r
            const float da = h ? (a + NH < NA ? dg[a1] : 0.f) : dg[a];              // g_n'
            const f32x2 gp = pack2(ga, ga), dp = pack2(da, da);
#pragma unroll
            for (int mm = 0; mm < NP; ++mm) {
                Sp2[mm] = ffma2(s2[a][mm], dp, Sp2[mm]);
                St2[mm] = ffma2(s2[a][mm], gp, St2[mm]);
            }
        }
        float Sq[kNumLM], St[kNumLM];
#pragma unroll
        for (int mm = 0; mm < NP; ++mm) {
            unpack2(Sp2[mm], Sq[2 * mm], Sq[2 * mm + 1]);
            unpack2(St2[mm], St[2 * mm], St[2 * mm + 1]);
        }
#pragma unroll
        for (int m = 0; m < kNumLM; ++m) Sq[m] = fmaf(-(float)LOF[m], St[m], Sq[m]);   // S' - l S/r
        float px, py, pz;
        ylm_force(x, y, z, Sq, St, &px, &py, &pz);
        px += __shfl_xor_sync(PAIR, px, 1);
        py += __shfl_xor_sync(PAIR, py, 1);
        pz += __shfl_xor_sync(PAIR, pz, 1);
        if (h == 0) {
            const float c = mycr[k * kMainAtoms];
            px = fmaf(c, e.x, px); py = fmaf(c, e.y, py); pz = fmaf(c, e.z, pz);
            fsx += px; fsy += py; fsz += pz;
            if (active) prow[k] = make_float4(px, py, pz, 0.f);
        }
    }
    fsx += __shfl_xor_sync(PAIR, fsx, 1);
    fsy += __shfl_xor_sync(PAIR, fsy, 1);
    fsz += __shfl_xor_sync(PAIR, fsz, 1);
    if (active && h == 0) d.Fself[i] = make_float4(fsx, fsy, fsz, 0.f);
}
