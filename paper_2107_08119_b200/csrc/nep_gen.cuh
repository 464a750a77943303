// nep_gen.cuh -- k_gen: descriptor + network + partial forces for ANY model shape, eight lanes per atom
// (included by nep_b200.cu inside its anonymous namespace, after nep_main.cuh and nep_desc64.cuh).
//
// k_main (nep_main.cuh) is one thread per atom with everything in registers: the fastest form once a few
// hundred thousand atoms fill the machine, but instantiated only for 8 or 9 radial functions per family and
// serial in the atom (one warp = 32 atoms, ~35 us of dependent instructions).  k_gen is the cooperative form:
// a group of 8 lanes owns one atom (4 atoms per warp), the runtime shape is free -- n_max^R, n_max^A up to
// NMAX-1 (NMAX = 8 or 16), l_max = 1..4, any N_neu, Table I's models included -- and an
// atom's work is spread over its lanes, so small systems (C0-C2, the paper's 8000-atom protocol,
// PAPER.md:395) finish in a fraction of k_main's latency.  Per atom:
//   R   q_n = sum_j g_n(r_ij), Eq. 12: lane = neighbour, partial sums in registers, shuffle reduction
//   D   s[n][lm] = sum_j g_n(r_ij) b_lm(r^_ij) (Eq. 17-18 route to Eq. 13): a chunk of 8 neighbours leaves
//       g_n and b_lm in shared memory (lane = neighbour), then lane = three lm columns accumulates
//       its s[.][lm] in registers (no shuffles, no atomics); q_nl = sum_m C_lm s_nlm^2
//   N   network Eq. 21-22 with the minus biases: lane = neuron for the forward sweep, lane = four
//       descriptor components for dU/dq; weights come through L1 (ld.global.nc), never staged
//   F   A[n][lm] = 2 Fp_nl C_lm s_nlm in shared memory; lane = neighbour contracts it with g_n'(r_ij) and
//       g_n(r_ij)/r_ij (broadcast reads) and applies the harmonic gradients: Eq. 23-25, p_ij to global memory
// TD = float: everything in fp32.  TD = double (multi-species models): R, D and N in fp64 straight from the
// fp64 positions, exactly as k_desc64 does and for the same reason (Eq. 19's sqrt(Z_i Z_j) weights make the
// pre-activations cancel); F stays fp32.
#pragma once

constexpr int kGenLanes = 8;                 // lanes per atom
constexpr int kGenWarps = 4;                 // warps per block
constexpr int kGenAtomsPerBlock = kGenWarps * (32 / kGenLanes);
constexpr int kMaxHGen = 128;                // hidden neurons (the paper's largest model has 50)

struct GenParams {
    double rcR, rcA;
    double zz64[kMaxTypes * kMaxTypes];      // sqrt(Z_a Z_b), Eq. 19
    float zz[kMaxTypes * kMaxTypes];
    float rcR_inv, rcA_inv;
    int NR, NA, LMAX, H, D, Dp, N, capR;
    Box box;
    const float* params;                     // staged fp32 layout w1[H][Dp] | b1[H] | w2[H] | b2
    const double* params64;                  // fp64 layout w1[H][D] | b1[H] | w2[H] | b2 (TD = double)
    float* q_out;                            // nullable parity hooks, [D][N] caller order
    float* fp_out;
};

template <int NMAX, typename TD>
struct alignas(16) GenSmem {                 // per 8-lane group
    TD S[NMAX][kNumLM];                      // s[n][lm], later (TD = float) A[n][lm] in place
    TD Gs[kGenLanes][NMAX];                  // chunk: g_n of 8 neighbours
    TD Bs[kGenLanes][kNumLM];                // chunk: b_lm of 8 neighbours
    TD q[NMAX * 5];                          // descriptor
    float Fp[NMAX * 5];                      // dU/dq
    TD hid[kMaxHGen];                        // w2 (1 - tanh^2) per neuron
    float A[sizeof(TD) == 8 ? NMAX * kNumLM : 1];    // TD = double: fp32 copy of A for the force phase
};

template <typename TD> struct GenMath;
template <> struct GenMath<float> {
    template <int N> static __device__ __forceinline__ void radial(float r, float rc_inv, double, float om, float* g) {
        radial_g<N>(r, rc_inv, om, g);
    }
    static __device__ __forceinline__ void basis(float x, float y, float z, float* b) { ylm_basis(x, y, z, b); }
    static __device__ __forceinline__ void act(float a, float* t, float* dd) { tanh_sech2(a, t, dd); }
};
template <> struct GenMath<double> {
    template <int N> static __device__ __forceinline__ void radial(double r, float, double rc, double om, double* g) {
        radial_g64<N>(r, rc, om, g);
    }
    static __device__ __forceinline__ void basis(double x, double y, double z, double* b) { ylm_basis64(x, y, z, b); }
    static __device__ __forceinline__ void act(double a, double* t, double* dd) {
        const double e = exp(-2.0 * fabs(a));
        const double inv = 1.0 / (1.0 + e);
        *t = copysign((1.0 - e) * inv, a);
        *dd = 4.0 * e * inv * inv;
    }
};

// record slot of neighbour k: angular ones from the front, radial-only ones from the back
__device__ __forceinline__ int gen_slot(int k, int nA, int capR) { return k < nA ? k : capR - 1 - (k - nA); }

template <int NMAX, typename TD>
__global__ void __launch_bounds__(32 * kGenWarps) k_gen(SysDev d, const __grid_constant__ GenParams P) {
    constexpr bool F64 = sizeof(TD) == 8;
    constexpr float C[kNumLM] = {NEP_CLM_LIST};
    constexpr int LOF[kNumLM] = {NEP_LOF_LIST};
    extern __shared__ __align__(16) unsigned char gsm_raw[];
    using SM = GenSmem<NMAX, TD>;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int grp = lane >> 3, gl = lane & 7;
    SM& sm = reinterpret_cast<SM*>(gsm_raw)[warp * 4 + grp];
    const int N = P.N, NR = P.NR, NA = P.NA, LMAX = P.LMAX, H = P.H, D = P.D, Dp = P.Dp, capR = P.capR;
    const int nlm = LMAX * (LMAX + 2);                       // 3, 8, 15, 24 harmonics for l_max = 1..4
    const float* b1f = P.params + (size_t)H * Dp;
    const float* w2f = b1f + H;

    for (int base = (blockIdx.x * kGenWarps + warp) * 4; base < N; base += gridDim.x * kGenAtomsPerBlock) {
        const int ia = base + grp;
        const bool valid = ia < N;
        const int i = valid ? ia : N - 1;
        const int nR = valid ? d.nnR[i] : 0, nA = valid ? d.nnA[i] : 0;
        // warp-uniform trip counts: the four groups of a warp stay converged
        const int chR = (__reduce_max_sync(0xffffffffu, nR) + kGenLanes - 1) / kGenLanes;
        const int chA = (__reduce_max_sync(0xffffffffu, nA) + kGenLanes - 1) / kGenLanes;
        const int ti = d.type_s[i];
        double4 pi = make_double4(0.0, 0.0, 0.0, 0.0);
        if (F64) pi = d.xs4[i];

        // neighbour k of the atom in the descriptor precision: unit vector, distance, Eq. 19 weight
        auto nbr = [&](int k, TD& x, TD& y, TD& z, TD& r, TD& om) {
            const int slot = gen_slot(k, nA, capR);
            if (F64) {
                const int j = (int)(d.jrev[(size_t)slot * N + i] & kJMask);
                const double4 pj = d.xs4[j];
                const double dx = min_image(pj.x - pi.x, P.box.L[0], P.box.invL[0]);
                const double dy = min_image(pj.y - pi.y, P.box.L[1], P.box.invL[1]);
                const double dz = min_image(pj.z - pi.z, P.box.L[2], P.box.invL[2]);
                const double rr = sqrt(dx * dx + dy * dy + dz * dz), ri = 1.0 / rr;
                x = (TD)(dx * ri); y = (TD)(dy * ri); z = (TD)(dz * ri); r = (TD)rr;
                om = (TD)P.zz64[ti * kMaxTypes + ((int)__double_as_longlong(pj.w) & (kMaxTypes - 1))];
            } else {
                const float4 e = d.rec[(size_t)slot * N + i];
                const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
                const float ri = inv_norm(r2);
                x = (TD)(e.x * ri); y = (TD)(e.y * ri); z = (TD)(e.z * ri); r = (TD)(r2 * ri);
                om = (TD)P.zz[ti * kMaxTypes + (__float_as_int(e.w) & (kMaxTypes - 1))];
            }
        };

        // ---- R: radial descriptor, Eq. 12 ----
        {
            TD qa[NMAX];
#pragma unroll
            for (int n = 0; n < NMAX; ++n) qa[n] = (TD)0;
            for (int c = 0; c < chR; ++c) {
                const int k = c * kGenLanes + gl;
                if (k < nR) {
                    TD x, y, z, r, om, g[NMAX];
                    nbr(k, x, y, z, r, om);
                    GenMath<TD>::template radial<NMAX>(r, P.rcR_inv, P.rcR, om, g);
#pragma unroll
                    for (int n = 0; n < NMAX; ++n) qa[n] += g[n];
                }
            }
#pragma unroll
            for (int n = 0; n < NMAX; ++n) {
                TD v = qa[n];
                v += __shfl_xor_sync(0xffffffffu, v, 1);
                v += __shfl_xor_sync(0xffffffffu, v, 2);
                v += __shfl_xor_sync(0xffffffffu, v, 4);
                if (gl == (n & 7) && n < NR) sm.q[n] = v;
            }
        }

        // ---- D: angular sums s[n][lm] and q_nl (Eq. 13 through Eq. 17-18 with n' = n) ----
        {
            TD acc[NMAX][3];
#pragma unroll
            for (int n = 0; n < NMAX; ++n) { acc[n][0] = acc[n][1] = acc[n][2] = (TD)0; }
            for (int c = 0; c < chA; ++c) {
                const int k = c * kGenLanes + gl;
                TD g[NMAX], bb[kNumLM];
                if (k < nA) {
                    TD x, y, z, r, om;
                    nbr(k, x, y, z, r, om);
                    GenMath<TD>::template radial<NMAX>(r, P.rcA_inv, P.rcA, om, g);
                    GenMath<TD>::basis(x, y, z, bb);
                } else {
#pragma unroll
                    for (int n = 0; n < NMAX; ++n) g[n] = (TD)0;
#pragma unroll
                    for (int m = 0; m < kNumLM; ++m) bb[m] = (TD)0;
                }
#pragma unroll
                for (int n = 0; n < NMAX; ++n) sm.Gs[gl][n] = g[n];
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) sm.Bs[gl][m] = bb[m];
                __syncwarp();
#pragma unroll
                for (int kk = 0; kk < kGenLanes; ++kk) {
                    const TD b0 = sm.Bs[kk][3 * gl], b1 = sm.Bs[kk][3 * gl + 1], b2 = sm.Bs[kk][3 * gl + 2];
#pragma unroll
                    for (int n = 0; n < NMAX; ++n) {
                        const TD gn = sm.Gs[kk][n];
                        acc[n][0] += gn * b0; acc[n][1] += gn * b1; acc[n][2] += gn * b2;
                    }
                }
                __syncwarp();
            }
#pragma unroll
            for (int n = 0; n < NMAX; ++n) {
                sm.S[n][3 * gl] = acc[n][0]; sm.S[n][3 * gl + 1] = acc[n][1]; sm.S[n][3 * gl + 2] = acc[n][2];
            }
            __syncwarp();
            for (int o = gl; o < NA * LMAX; o += kGenLanes) {            // q_nl, descriptor order n-major, l = 1..l_max
                const int n = o / LMAX, l = o - n * LMAX + 1;
                TD v = (TD)0;
#pragma unroll
                for (int m = 0; m < kNumLM; ++m)
                    if (LOF[m] == l) v += (TD)C[m] * sm.S[n][m] * sm.S[n][m];
                sm.q[NR + o] = v;
            }
            __syncwarp();
        }
        if (P.q_out && valid) {
            const int row = d.perm[i];
            for (int v = gl; v < D; v += kGenLanes) P.q_out[(size_t)v * N + row] = (float)sm.q[v];
        }

        // ---- N: network, Eq. 21-22 (minus biases), and Fp = dU/dq ----
        {
            if (gl < Dp - D) sm.q[D + gl] = (TD)0;                        // the padded tail of q (w1's padded columns are zero too)
            __syncwarp();
            TD Upart = (TD)0;
            for (int mu = gl; mu < H; mu += kGenLanes) {
                TD a, w2;
                if (F64) {
                    const double* w = P.params64 + (size_t)mu * D;
                    double a0 = -P.params64[(size_t)H * D + mu], a1 = 0.0;
                    int v = 0;
                    for (; v + 1 < D; v += 2) { a0 += w[v] * (double)sm.q[v]; a1 += w[v + 1] * (double)sm.q[v + 1]; }
                    if (v < D) a0 += w[v] * (double)sm.q[v];
                    a = (TD)(a0 + a1);
                    w2 = (TD)P.params64[(size_t)H * D + H + mu];
                } else {
                    const float4* w = reinterpret_cast<const float4*>(P.params + (size_t)mu * Dp);
                    float a0 = -__ldg(&b1f[mu]), a1 = 0.f, a2 = 0.f, a3 = 0.f;
                    for (int v = 0; v < Dp / 4; ++v) {                  // padded columns of w1 are zero; q is padded with zeros below
                        const float4 ww = __ldg(&w[v]);
                        a0 = fmaf(ww.x, (float)sm.q[4 * v], a0); a1 = fmaf(ww.y, (float)sm.q[4 * v + 1], a1);
                        a2 = fmaf(ww.z, (float)sm.q[4 * v + 2], a2); a3 = fmaf(ww.w, (float)sm.q[4 * v + 3], a3);
                    }
                    a = (TD)((a0 + a1) + (a2 + a3));
                    w2 = (TD)__ldg(&w2f[mu]);
                }
                TD t, dd;
                GenMath<TD>::act(a, &t, &dd);
                Upart += w2 * t;
                sm.hid[mu] = w2 * dd;
            }
            Upart += __shfl_xor_sync(0xffffffffu, Upart, 1);
            Upart += __shfl_xor_sync(0xffffffffu, Upart, 2);
            Upart += __shfl_xor_sync(0xffffffffu, Upart, 4);
            __syncwarp();
            if (gl == 0 && valid) {
                const TD b2 = F64 ? (TD)P.params64[(size_t)H * D + 2 * H] : (TD)__ldg(&w2f[H]);
                d.Us[i] = (float)(Upart - b2);
            }
            for (int v4 = gl; v4 < Dp / 4; v4 += kGenLanes) {              // four descriptor components per lane
                TD f0 = (TD)0, f1 = (TD)0, f2 = (TD)0, f3 = (TD)0;
                for (int mu = 0; mu < H; ++mu) {
                    const TD gm = sm.hid[mu];
                    if (F64) {
                        const double* w = P.params64 + (size_t)mu * D + 4 * v4;
                        f0 += gm * (TD)w[0];
                        if (4 * v4 + 1 < D) f1 += gm * (TD)w[1];
                        if (4 * v4 + 2 < D) f2 += gm * (TD)w[2];
                        if (4 * v4 + 3 < D) f3 += gm * (TD)w[3];
                    } else {
                        const float4 ww = __ldg(reinterpret_cast<const float4*>(P.params + (size_t)mu * Dp) + v4);
                        f0 += gm * (TD)ww.x; f1 += gm * (TD)ww.y; f2 += gm * (TD)ww.z; f3 += gm * (TD)ww.w;
                    }
                }
                sm.Fp[4 * v4] = (float)f0; sm.Fp[4 * v4 + 1] = (float)f1; sm.Fp[4 * v4 + 2] = (float)f2; sm.Fp[4 * v4 + 3] = (float)f3;
            }
            __syncwarp();
        }
        if (P.fp_out && valid) {
            const int row = d.perm[i];
            for (int v = gl; v < D; v += kGenLanes) P.fp_out[(size_t)v * N + row] = sm.Fp[v];
        }

        // ---- F: partial forces, Eq. 23-25 ----
        float* A = F64 ? sm.A : reinterpret_cast<float*>(&sm.S[0][0]);     // A[n][lm] = 2 Fp_nl C_lm s_nlm (0 beyond l_max)
        for (int e = gl; e < NMAX * kNumLM; e += kGenLanes) {
            const int n = e / kNumLM, m = e - n * kNumLM;
            float v = 0.f;
            if (n < NA && m < nlm) v = 2.f * C[m] * sm.Fp[NR + n * LMAX + LOF[m] - 1] * (float)sm.S[n][m];
            A[e] = v;                                                    // in place when TD = float: same element, same lane
        }
        __syncwarp();
        float fsx = 0.f, fsy = 0.f, fsz = 0.f;
        float4* prow = d.p + (size_t)i * capR;
        for (int c = 0; c < chR; ++c) {
            const int k = c * kGenLanes + gl;
            const bool on = k < nR;
            const int slot = gen_slot(on ? k : 0, nA, capR);
            float4 e = make_float4(1.f, 0.f, 0.f, 0.f);
            if (on) e = d.rec[(size_t)slot * N + i];
            const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
            const float rinv = inv_norm(r2), r = r2 * rinv;
            const float x = e.x * rinv, y = e.y * rinv, z = e.z * rinv;
            const float om = P.zz[ti * kMaxTypes + (__float_as_int(e.w) & (kMaxTypes - 1))];
            // radial family, Eq. 24
            float gR[NMAX], dR[NMAX];
            radial_gd<NMAX>(r, P.rcR_inv, om, 1.f, gR, dR);
            float cr = 0.f;
#pragma unroll
            for (int n = 0; n < NMAX; ++n)
                if (n < NR) cr = fmaf(sm.Fp[n], dR[n], cr);
            float px = cr * x, py = cr * y, pz = cr * z;
            if (c < chA && __any_sync(0xffffffffu, on && k < nA)) {      // angular family, Eq. 25 (warp-uniform branch)
                float gs[NMAX], dg[NMAX];
                radial_gd<NMAX>(r, P.rcA_inv, om, rinv, gs, dg);
                float Sq[kNumLM], St[kNumLM];
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) { Sq[m] = 0.f; St[m] = 0.f; }
#pragma unroll
                for (int n = 0; n < NMAX; ++n) {
                    if (n < NA) {                                        // uniform
                        const float4* An = reinterpret_cast<const float4*>(A + n * kNumLM);
#pragma unroll
                        for (int m4 = 0; m4 < kNumLM / 4; ++m4) {
                            const float4 a = An[m4];
                            Sq[4 * m4] = fmaf(a.x, dg[n], Sq[4 * m4]); St[4 * m4] = fmaf(a.x, gs[n], St[4 * m4]);
                            Sq[4 * m4 + 1] = fmaf(a.y, dg[n], Sq[4 * m4 + 1]); St[4 * m4 + 1] = fmaf(a.y, gs[n], St[4 * m4 + 1]);
                            Sq[4 * m4 + 2] = fmaf(a.z, dg[n], Sq[4 * m4 + 2]); St[4 * m4 + 2] = fmaf(a.z, gs[n], St[4 * m4 + 2]);
                            Sq[4 * m4 + 3] = fmaf(a.w, dg[n], Sq[4 * m4 + 3]); St[4 * m4 + 3] = fmaf(a.w, gs[n], St[4 * m4 + 3]);
                        }
                    }
                }
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) Sq[m] = fmaf(-(float)LOF[m], St[m], Sq[m]);      // S'_m - l_m S_m / r
                float ax, ay, az;
                ylm_force(x, y, z, Sq, St, &ax, &ay, &az);
                if (k < nA) { px += ax; py += ay; pz += az; }
            }
            if (on) {
                fsx += px; fsy += py; fsz += pz;
                prow[slot] = make_float4(px, py, pz, 0.f);
            }
        }
#pragma unroll
        for (int o = 1; o < kGenLanes; o <<= 1) {
            fsx += __shfl_xor_sync(0xffffffffu, fsx, o);
            fsy += __shfl_xor_sync(0xffffffffu, fsy, o);
            fsz += __shfl_xor_sync(0xffffffffu, fsz, o);
        }
        if (gl == 0 && valid) d.Fself[i] = make_float4(fsx, fsy, fsz, 0.f);
        __syncwarp();
    }
}
