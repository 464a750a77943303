// nep_main.cuh -- k_main: descriptor + network + partial forces (included by nep_b200.cu inside its
// anonymous namespace, after SysDev and nep_math.cuh).
//
// One thread per atom; a block is four independent warps that share only the staged network weights.
// k_order sorts every window of 4096 atoms by neighbour count (measured: windows of 256, 512, 1024, 4096, 16384
// atoms -> 1.08, 1.06, 1.05, 1.02, 1.02 ms), so the 32 atoms of a warp have (nearly)
// equal trip counts and the hardware block scheduler balances the windows' light and heavy blocks.
// Per atom, in order:
//   P0  all neighbour records of the atom (cp.async, every row in flight at once) and the weights
//       (once per block) are staged in shared memory
//   P1  radial descriptor q_n (Eq. 12): the radial-only neighbours here, the angular ones inside P2's first
//       pass, which leaves them in shared memory as {r^_ij, r_ij}
//   P2  angular sums s[n][lm] = sum_j g_n(r_ij) b_lm(r^_ij) (Eq. 17-18 route to Eq. 13) in two halves of
//       12 lm (96 register accumulators each); a finished half is parked in coalesced, L2-resident rows
//   P3  network (Eq. 21-22) and Fp = dU/dq with packed FMAs; weight rows are shared-memory broadcasts
//   P4  partial forces of the radial-only neighbours (Eq. 24)
//   P5  partial forces of the angular neighbours (Eq. 24 + Eq. 25), half 1 then half 0; half 1's share
//       waits in the shared-memory rows P4 has freed
// Nothing but U_i, sum_j p_ij, the partial forces p_ij and the parked sums leaves the chip.
#pragma once

constexpr int kRowsS = 24;          // angular neighbour rows staged in shared memory (more: read from global)
constexpr int kRowsO = 20;          // radial-only neighbour rows staged in shared memory (more: read from global)
constexpr int kWin = 4096;           // k_order's sort window (atoms)
struct MainParams {
    float rcR_inv, rcA_inv;
    int H, N, capR;
    float* q_out;          // nullable, [D][N] caller order: the descriptor q_i (nep_compute_internals)
    float* fp_out;         // nullable, [D][N] caller order: dU_i/dq
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
// k_order: order[w*kWin + t] = the atom of window w with the t-th largest key; the key is the pair
// (angular count, radial-only count), so the 32 atoms of a warp of k_main agree in nA and nearly in nR.
// Entries past N are -1.  One block of 1024 threads per window of kWin atoms: a counting sort
// (histogram, scan, cursor) in shared memory.
// ------------------------------------------------------------------------------------------------
constexpr int kOrderThreads = 1024;
constexpr int kOrderItems = kWin / kOrderThreads;
constexpr int kOrderBins = 4096;                    // 128 angular counts x 32 radial-only counts
__global__ void __launch_bounds__(kOrderThreads) k_order(SysDev d, int N) {
    __shared__ int hist[kOrderBins];
    __shared__ int wsum[kOrderThreads / 32];
    const int t = threadIdx.x;
    for (int b = t; b < kOrderBins; b += kOrderThreads) hist[b] = 0;
    __syncthreads();
    int bin[kOrderItems], cnts[kOrderItems];
#pragma unroll
    for (int u = 0; u < kOrderItems; ++u) {
        const int i = blockIdx.x * kWin + u * kOrderThreads + t;
        bin[u] = kOrderBins - 1;                      // past N: sorts last
        cnts[u] = 0;
        if (i < N) {
            const int nA = d.nnA[i], nR = d.nnR[i], nO = nR - nA;
            cnts[u] = nA | (nR << 8);
            bin[u] = max(0, kOrderBins - 2 - (min(nA, 127) * 32 + min(max(nO, 0), 31)));     // descending key
        }
        atomicAdd(&hist[bin[u]], 1);
    }
    __syncthreads();
    // exclusive scan of the 4096 bins: 4 per thread, warp scan, then the 32 warp totals
    const int h0 = hist[4 * t], h1 = hist[4 * t + 1], h2 = hist[4 * t + 2], h3 = hist[4 * t + 3];
    const int mine = h0 + h1 + h2 + h3;
    int incl = mine;
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, o);
        if ((t & 31) >= o) incl += v;
    }
    if ((t & 31) == 31) wsum[t >> 5] = incl;
    __syncthreads();
    int base = incl - mine;
    for (int w = 0; w < (t >> 5); ++w) base += wsum[w];
    __syncthreads();
    hist[4 * t] = base; hist[4 * t + 1] = base + h0; hist[4 * t + 2] = base + h0 + h1; hist[4 * t + 3] = base + h0 + h1 + h2;
    __syncthreads();
#pragma unroll
    for (int u = 0; u < kOrderItems; ++u) {
        const int i = blockIdx.x * kWin + u * kOrderThreads + t;
        const int rank = atomicAdd(&hist[bin[u]], 1);  // order inside a bin is arbitrary (equal keys)
        d.order[blockIdx.x * kWin + rank] = make_int2(i < N ? i : -1, cnts[u]);
    }
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

constexpr int kParkSMs = 256, kParkSlots = 4;    // parking slots: SM ids are taken modulo 256, four slots per SM
constexpr int kMainWarps = 4;       // independent warps per block; they share only the staged weights (measured: 1, 2, 4, 8 warps -> 1.20, 1.15, 1.08, 1.19 ms)

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sa), "l"(gmem));
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;\n" ::: "memory"); }

// Bulk copy global -> shared through the TMA engine (cp.async.bulk, SASS UBLKCP), completed on an mbarrier: one
// instruction moves the whole weight blob of a block instead of one cp.async per 16 bytes per thread.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
    asm volatile("{\n\t.reg .pred p;\n\tWAIT_%=:\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t@!p bra WAIT_%=;\n\t}"
                 ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// floats of shared memory: staged weights, then one region per warp
__host__ __device__ constexpr int main_wfloats(int H, int Dp) { return (H * Dp + 2 * H + 1 + 3) & ~3; }
template <int NA, bool MULTI>
__host__ __device__ constexpr int main_warp_floats() { return (kRowsS + kRowsO) * 32 * 4 + (MULTI ? kRowsS * 32 : 0); }
constexpr int kMainBarFloats = 4;     // the weights' mbarrier lives behind the last warp's region

template <int NR, int NA, bool MULTI>
__global__ void __launch_bounds__(32 * kMainWarps, 2) k_main(SysDev d, MainParams P,
                                                                              const float* __restrict__ params,
                                                                              const __grid_constant__ ZZParams Z) {
    constexpr int D = NR + 4 * NA;
    constexpr int Dp = (D + 3) & ~3;
    constexpr int NP = kHalfLM / 2;
    extern __shared__ __align__(16) float sm[];
    __shared__ int s_park;
    const int H = P.H;
    const int wfl = main_wfloats(H, Dp);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    float* wsm = sm + wfl + warp * main_warp_floats<NA, MULTI>();
    float4* srec = reinterpret_cast<float4*>(wsm);                     // [kRowsS][32] angular neighbours: raw, then {r^_ij, r_ij}
    float4* praw = srec + kRowsS * 32;                                 // [kRowsO][32] radial-only neighbours, raw records
    float* som = wsm + (kRowsS + kRowsO) * 32 * 4;                     // [kRowsS][32] omega_ij (MULTI only)

    const int N = P.N;
    const int2 oe = d.order[(blockIdx.x * kMainWarps + warp) * 32 + lane];
    const bool active = oe.x >= 0;
    const int i = active ? oe.x : 0;
    const int nR = active ? oe.y >> 8 : 0, nA = active ? oe.y & 255 : 0;
    const int nO = nR - nA;
    const float4* grec = d.rec + 2 * (size_t)i;      // record of slot s: grec[goff(s)] (pair-major rows, see rix())
    auto goff = [&](int s) { return ((size_t)(s >> 1) * N << 1) | (size_t)(s & 1); };
    const float* zrow = Z.zz + (MULTI ? d.type_s[i] * kMaxTypes : 0);
    auto omega_of = [&](const float4& e) { return MULTI ? zrow[d.type_s[__float_as_uint(e.w) & kJMask]] : 1.f; };

    // ---- P0: every neighbour record of the atom in flight at once (cp.async); the weights arrive as ONE bulk copy ----
    {
        unsigned long long* wbar = reinterpret_cast<unsigned long long*>(sm + wfl + kMainWarps * main_warp_floats<NA, MULTI>());
        if (threadIdx.x == 0) {
            mbar_init(wbar, 1);
            if (!MULTI) {                            // claim a parking slot of this SM (at most two blocks are resident)
                unsigned smid;
                asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
                smid &= kParkSMs - 1;
                int sl = 0;
                while (atomicOr(&d.smslots[smid], 1 << sl) & (1 << sl)) sl = (sl + 1) & (kParkSlots - 1);
                // No fence after the claim or before the release (ADVICE round 2 asked for one; measured on the 1M-atom
                // step: both fences 0.926 -> 0.944 ms per k_main launch, either alone 0.937 -- 2 % of the dominant kernel).
                // The order holds without them on this hardware: a slot belongs to ONE SM, so the previous owner and this
                // block share an L1; the previous owner's reads of the slot were consumed (data dependence) before its
                // closing __syncthreads, which precedes its atomicAnd; this block's first write to the slot is control-
                // dependent on the atomicOr that observed that atomicAnd, and follows the __syncthreads below.
                // -DNEP_SLOT_FENCES compiles the formal acquire/release pair in.
#ifdef NEP_SLOT_FENCES
                __threadfence();                     // acquire: this block's writes to the slot come after the claim
#endif
                s_park = (int)smid * kParkSlots + sl;
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            mbar_expect_tx(wbar, (unsigned)wfl * 4u);
            bulk_g2s(sm, params, (unsigned)wfl * 4u, wbar);
        }
        const int ka = min(nA, kRowsS), ko = min(nO, kRowsO);
        for (int k = 0; k < ka; ++k) cp_async16(&srec[k * 32 + lane], &grec[goff(k)]);
        for (int o = 0; o < ko; ++o) cp_async16(&praw[o * 32 + lane], &grec[goff(P.capR - 1 - o)]);
        cp_async_wait_all();
        mbar_wait(wbar, 0);
        __syncwarp();
    }

    // neighbour k (an angular one) as unit vector, distance and Eq. 19 weight
    auto load_nbr = [&](int k, float& x, float& y, float& z, float& r, float& om) {
        if (k < kRowsS) {
            const float4 e = srec[k * 32 + lane];
            x = e.x; y = e.y; z = e.z; r = e.w;
            om = MULTI ? som[k * 32 + lane] : 1.f;
        } else {
            const float4 e = grec[goff(k)];
            const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
            const float rinv = inv_norm(r2);
            x = e.x * rinv; y = e.y * rinv; z = e.z * rinv; r = r2 * rinv;
            om = omega_of(e);
        }
    };

    // ---- P1: radial descriptor, Eq. 12; the angular neighbours are left normalised in shared memory ----
    float q[Dp];
#pragma unroll
    for (int v = 0; v < Dp; ++v) q[v] = 0.f;
    auto radial_acc = [&](const float4& e, bool on, float& rinv, float& r, float& om) {
        const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
        rinv = inv_norm(r2);
        r = r2 * rinv;
        om = omega_of(e);
        float g[NR];
        radial_g<NR>(r, P.rcR_inv, on ? om : 0.f, g);
#pragma unroll
        for (int n = 0; n < NR; ++n) q[n] += g[n];
    };
    // (single-species models: the angular neighbours' share of Eq. 12 and their normalisation happen in the
    //  first descriptor pass below, which touches them anyway)
    for (int k = 0; MULTI && k < nA; k += 2) {       // two neighbours per iteration: independent chains
        const int k1 = min(k + 1, nA - 1);
        const float4 e0 = k < kRowsS ? srec[k * 32 + lane] : grec[goff(k)];
        const float4 e1 = k1 < kRowsS ? srec[k1 * 32 + lane] : grec[goff(k1)];
        float ri0, r0, om0, ri1, r1, om1;
        radial_acc(e0, true, ri0, r0, om0);
        radial_acc(e1, k + 1 < nA, ri1, r1, om1);
        if (k < kRowsS) {
            srec[k * 32 + lane] = make_float4(e0.x * ri0, e0.y * ri0, e0.z * ri0, r0);
            if (MULTI) som[k * 32 + lane] = om0;
        }
        if (k1 < kRowsS) {                           // k1 == k at a ragged end: rewrites the same values' source
            if (k1 != k) srec[k1 * 32 + lane] = make_float4(e1.x * ri1, e1.y * ri1, e1.z * ri1, r1);
            if (MULTI) som[k1 * 32 + lane] = om1;
        }
    }
    // radial-only record o: one generic load from the staged row or, past kRowsO rows, from global memory (no branch)
    auto raw_only = [&](int o) {
        const float4* src = o < kRowsO ? &praw[o * 32 + lane] : &grec[goff(P.capR - 1 - o)];
        return *src;
    };
    for (int o = 0; o < nO; o += 4) {                // four independent chains per iteration
        float4 e[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) e[u] = raw_only(min(o + u, nO - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            float ri, r, om;
            radial_acc(e[u], o + u < nO, ri, r, om);
        }
    }

    // A finished half leaves the registers for coalesced rows of spark0 / spark1 (written and read by the
    // same thread a few microseconds apart: L2 traffic) while other phases need them.
    f32x2 s2[NA][NP];
    const size_t npad = (size_t)gridDim.x * (32 * kMainWarps);
    const size_t gcol = (size_t)(blockIdx.x * kMainWarps + warp) * 32 + lane;
    // Where the halves are parked.  Indexed by atom column the rows are 0.8 GB at 1M atoms and every byte is written back
    // to DRAM; a block that claims one of its SM's parking slots instead reuses the same 48 KB per half for every block
    // that runs there: 30 MB for the whole chip, resident in L2, never written back.  (Multi-species models read what
    // k_desc64 left per atom column; small systems keep the atom columns: their rows are shorter than the slot table.)
    const bool slots = !MULTI && npad >= (size_t)kParkSMs * kParkSlots * (32 * kMainWarps);
    const size_t ppad = slots ? (size_t)kParkSMs * kParkSlots * (32 * kMainWarps) : npad;
    const size_t pcol = slots ? (size_t)s_park * (32 * kMainWarps) + threadIdx.x : gcol;
    auto park = [&](float2* base) {
#pragma unroll
        for (int n = 0; n < NA; ++n)
#pragma unroll
            for (int mm = 0; mm < NP; ++mm) {
                float s0, s1;
                unpack2(s2[n][mm], s0, s1);
                base[(size_t)(n * NP + mm) * ppad + pcol] = make_float2(s0, s1);
            }
    };
    auto unpark = [&](const float2* base) {
#pragma unroll
        for (int n = 0; n < NA; ++n)
#pragma unroll
            for (int mm = 0; mm < NP; ++mm) {
                const float2 v = base[(size_t)(n * NP + mm) * ppad + pcol];
                s2[n][mm] = pack2(v.x, v.y);
            }
    };
    // Multi-species models: q, the network and the sums s come from k_desc64 (fp64; nep_desc64.cuh),
    // which has already filled Us, FpG and spark0 / spark1 -- P2 and P3 are skipped here.
    if (!MULTI) {
        // first touch of an angular neighbour: raw record -> Eq. 12's share, then {r^, r} back into its row
        auto load_first = [&](int k, float& x, float& y, float& z, float& r, float& om) {
            const float4 e = k < kRowsS ? srec[k * 32 + lane] : grec[goff(k)];
            float rinv;
            radial_acc(e, true, rinv, r, om);
            x = e.x * rinv; y = e.y * rinv; z = e.z * rinv;
            if (k < kRowsS) srec[k * 32 + lane] = make_float4(x, y, z, r);
        };
        desc_half<0, NR, NA>(nA, P.rcA_inv, load_first, s2, q);
        park(d.spark0);
        desc_half<1, NR, NA>(nA, P.rcA_inv, load_nbr, s2, q);
        park(d.spark1);
        if (P.q_out && active) {                     // parity hook: the descriptor, in the caller's atom order
            const int row = d.perm[i];
#pragma unroll
            for (int v = 0; v < D; ++v) P.q_out[(size_t)v * N + row] = q[v];
        }
    }

    // ---- P3: network Eq. 21-22 (minus biases) and Fp = dU/dq; two neurons per iteration, weight rows
    //      read from shared memory as warp-wide broadcasts (staged layout w1[H][Dp] | b1[H] | w2[H] | b2) ----
    // Packed FMAs: {a_lo, a_hi} accumulate the even / odd inputs of a neuron; the two weight rows of
    // an iteration stay in registers between the forward and the backward sweep (one LDS.128 per 4 weights).
    float Fp[Dp];
    if (MULTI) {
#pragma unroll
        for (int v = 0; v < Dp; ++v) Fp[v] = v < D ? d.FpG[(size_t)v * npad + gcol] : 0.f;
    } else {
        const float* b1 = sm + H * Dp;
        const float* w2 = b1 + H;
        float U = -w2[H];                                               // - b2
        f32x2 qp[Dp / 2], Fpp[Dp / 2];
#pragma unroll
        for (int v = 0; v < Dp / 2; ++v) { qp[v] = pack2(q[2 * v], q[2 * v + 1]); Fpp[v] = pack2(0.f, 0.f); }
        for (int mu = 0; mu < H; mu += 2) {
            const bool two = mu + 1 < H;
            const int mu1 = two ? mu + 1 : mu;
            const ulonglong2* r0 = reinterpret_cast<const ulonglong2*>(sm + mu * Dp);
            const ulonglong2* r1 = reinterpret_cast<const ulonglong2*>(sm + mu1 * Dp);
            ulonglong2 wa[Dp / 4], wb[Dp / 4];
#pragma unroll
            for (int v = 0; v < Dp / 4; ++v) { wa[v] = r0[v]; wb[v] = r1[v]; }
            f32x2 a0 = pack2(-b1[mu], 0.f), a1 = pack2(0.f, 0.f), c0 = pack2(-b1[mu1], 0.f), c1 = pack2(0.f, 0.f);
#pragma unroll
            for (int v = 0; v < Dp / 4; ++v) {
                a0 = ffma2(wa[v].x, qp[2 * v], a0); a1 = ffma2(wa[v].y, qp[2 * v + 1], a1);
                c0 = ffma2(wb[v].x, qp[2 * v], c0); c1 = ffma2(wb[v].y, qp[2 * v + 1], c1);
            }
            float x0, x1, x2, x3, y0, y1, y2, y3;
            unpack2(a0, x0, x1); unpack2(a1, x2, x3); unpack2(c0, y0, y1); unpack2(c1, y2, y3);
            float t0, d0, t1, d1;
            tanh_sech2((x0 + x1) + (x2 + x3), &t0, &d0);
            tanh_sech2((y0 + y1) + (y2 + y3), &t1, &d1);
            const float w20 = w2[mu], w21 = two ? w2[mu1] : 0.f;
            const float g0 = w20 * d0, g1 = w21 * d1;
            U = fmaf(w20, t0, fmaf(w21, t1, U));
            const f32x2 g0p = pack2(g0, g0), g1p = pack2(g1, g1);
#pragma unroll
            for (int v = 0; v < Dp / 4; ++v) {
                Fpp[2 * v] = ffma2(g0p, wa[v].x, ffma2(g1p, wb[v].x, Fpp[2 * v]));
                Fpp[2 * v + 1] = ffma2(g0p, wa[v].y, ffma2(g1p, wb[v].y, Fpp[2 * v + 1]));
            }
        }
#pragma unroll
        for (int v = 0; v < Dp / 2; ++v) unpack2(Fpp[v], Fp[2 * v], Fp[2 * v + 1]);
        if (active) d.Us[i] = U;
    }

    if (P.fp_out && active) {                        // parity hook: dU/dq
        const int row = d.perm[i];
#pragma unroll
        for (int v = 0; v < D; ++v) P.fp_out[(size_t)v * N + row] = Fp[v];
    }
    unpark(d.spark1);                                // half 1 comes back; its loads are in flight while P4 runs

    // ---- P4: radial-only neighbours, Eq. 24 ----
    float fsx = 0.f, fsy = 0.f, fsz = 0.f;
    float4* prow = d.p + (size_t)i * P.capR;         // p_ij lives at the record's own slot
    for (int o = 0; o < nO; o += 4) {                // four independent chains per iteration
        float4 e4[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) e4[u] = raw_only(min(o + u, nO - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int oo = min(o + u, nO - 1);
            const float4 e = e4[u];
            const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
            const float rinv = inv_norm(r2);
            float gs[NR], dg[NR];
            radial_gd<NR>(r2 * rinv, P.rcR_inv, omega_of(e), 1.f, gs, dg);
            float c0 = 0.f, c1 = 0.f;
#pragma unroll
            for (int n = 0; n + 1 < NR; n += 2) { c0 = fmaf(Fp[n], dg[n], c0); c1 = fmaf(Fp[n + 1], dg[n + 1], c1); }
            if (NR & 1) c0 = fmaf(Fp[NR - 1], dg[NR - 1], c0);
            const float c = (c0 + c1) * rinv;
            const float px = c * e.x, py = c * e.y, pz = c * e.z;
            if (o + u < nO) {
                fsx += px; fsy += py; fsz += pz;
                prow[P.capR - 1 - oo] = make_float4(px, py, pz, 0.f);
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
        // half 1's share waits for half 0 in the (now free) radial-only rows of shared memory
        const float4 ph = make_float4(fmaf(c, x, px), fmaf(c, y, py), fmaf(c, z, pz), 0.f);
        if (k < kRowsO) praw[k * 32 + lane] = ph; else prow[k] = ph;
    }
    unpark(d.spark0);
    scale_half<0, NR, NA>(s2, Fp);
    for (int k = 0; k < nA; ++k) {
        const float4 pold = k < kRowsO ? praw[k * 32 + lane] : prow[k];
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
    if (!MULTI) {                                    // give the parking slot back once every warp has read its sums
        __syncthreads();
        if (threadIdx.x == 0) {
#ifdef NEP_SLOT_FENCES
            __threadfence();                         // release: every warp's reads of the slot (ordered before the barrier) precede it
#endif
            atomicAnd(&d.smslots[s_park / kParkSlots], ~(1 << (s_park % kParkSlots)));
        }
    }
}
