// nep_gen.cuh -- k_gen: descriptor + network + partial forces for ANY model shape, a group of lanes per atom
// (included by nep_b200.cu inside its anonymous namespace, after nep_main.cuh and nep_desc64.cuh).
//
// k_main (nep_main.cuh) is one thread per atom with everything in registers: the fastest form once a few
// hundred thousand atoms fill the machine, but instantiated only for 8/8, 9/9 or 13/7 radial/angular functions,
// l_max = 4, N_neu <= 64, and serial in the atom (one warp = 32 atoms, ~35 us of dependent instructions).  k_gen is the cooperative form:
// a group of G = 16 lanes owns one atom (2 atoms per warp), the runtime shape is free -- n_max^R, n_max^A up to
// NMAX-1 (NMAX = 8 or 16), l_max = 1..4, any N_neu, Table I's models included -- and an
// atom's work is spread over its lanes, so small systems (C0-C2, the paper's 8000-atom protocol,
// PAPER.md:395) finish in a fraction of k_main's latency.  Per atom:
//   R   q_n = sum_j g_n(r_ij), Eq. 12: lane = neighbour, partial sums in registers, shuffle reduction
//   D   s[n][lm] = sum_j g_n(r_ij) b_lm(r^_ij) (Eq. 17-18 route to Eq. 13): a chunk of G neighbours leaves
//       g_n and b_lm in shared memory (lane = neighbour), then lane = (three lm columns, a slice of n)
//       accumulates its s[n][lm] in registers (no shuffles, no atomics); q_nl = sum_m C_lm s_nlm^2
//   N   network Eq. 21-22 with the minus biases: lane = neuron for the forward sweep, lane = four
//       descriptor components for dU/dq; the weights are staged in shared memory once per (persistent) block
//   F   A[n][lm] = 2 Fp_nl C_lm s_nlm in shared memory; lane = neighbour contracts it with g_n'(r_ij) and
//       g_n(r_ij)/r_ij (broadcast reads) and applies the harmonic gradients: Eq. 23-25, p_ij to global memory
// TD = float: everything in fp32.  TD = double (multi-species models): R, D and N in fp64 straight from the
// fp64 positions, exactly as k_desc64 does and for the same reason (Eq. 19's sqrt(Z_i Z_j) weights make the
// pre-activations cancel); F stays fp32.
#pragma once

constexpr int kGenLanes = 16;                // lanes per atom (8: 27 us per C1 evaluation, 16: see DESIGN.md section 6)
constexpr int kGenGroups = 32 / kGenLanes;   // atoms per warp
constexpr int kGenSplit = kGenLanes / 8;     // the 8 lm triples x kGenSplit slices of n = the lanes of phase D
constexpr int kGenWarps = 4;                 // warps per block
constexpr int kGenAtomsPerBlock = kGenWarps * kGenGroups;
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
    // variants: the SOAP-like descriptor q_nn'l of Eq. 17 and two or three hidden layers
    int kind;                                // 0: q_nl (Eq. 13), 1: q_nn'l for the pairs n <= n' (Eq. 17)
    int nlayers;                             // hidden layers; > 1: the padded blob below replaces params / params64
    int lw[3], lin_p[3];                     // width of hidden layer k and the padded length of its input rows
    int off_w[3], off_b[3], off_out;         // element offsets of W_k, b_k and of w_out | b_out in the blob
    int blob_elems;
    const float* blob;                       // W1[H1][in_p] | b1 | W2[H2][H1_p] | b2 | ... | w_out | b_out, sections 4-aligned
    const double* blob64;
    const double* boxes;                     // nullable: concatenated structures (training side), [S][6] = L[3], 1/L[3]
    const int* sid;                          //   structure of (sorted) atom i
    float* q_out;                            // nullable parity hooks, [D][N] caller order
    float* fp_out;
};

template <int NMAX, typename TD>
struct alignas(16) GenSmem {                 // per group of lanes
    TD S[NMAX][kNumLM];                      // s[n][lm], later (TD = float) A[n][lm] in place
    TD Gs[kGenLanes][NMAX + 1];              // chunk: g_n of G neighbours (odd row stride: conflict-free stores)
    TD Bs[kGenLanes][kNumLM + 1];            // chunk: b_lm of G neighbours
    TD q[NMAX == 8 ? 152 : NMAX * 5];        // descriptor (NMAX = 8 also holds the 8 + 36 x 4 components of q_nn'l)
    float Fp[NMAX == 8 ? 152 : NMAX * 5];    // dU/dq
    TD hid[kMaxHGen];                        // w2 (1 - tanh^2) per neuron; deep networks: layer 1
    TD act[2][kMaxHGen];                     // deep networks: layers 2 and 3
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
    const int grp = lane / kGenLanes, gl = lane % kGenLanes;
    SM& sm = reinterpret_cast<SM*>(gsm_raw)[warp * kGenGroups + grp];
    const int N = P.N, NR = P.NR, NA = P.NA, LMAX = P.LMAX, H = P.H, D = P.D, Dp = P.Dp, capR = P.capR;
    // weights: staged once per block (the grid-stride loop below reuses them), rows padded by 4 floats so that
    // the forward sweep's per-lane rows fall into distinct bank groups
    const int Dps = F64 ? (Dp | 1) : Dp + 4;             // odd stride in 8-byte units for doubles
    TD* wsm = reinterpret_cast<TD*>(gsm_raw + (size_t)kGenAtomsPerBlock * sizeof(SM));       // w1[H][Dps] | b1[H] | w2[H] | b2
    if (P.nlayers > 1) {                                                  // deep network: the host-padded blob as it is
        for (int e = threadIdx.x; e < P.blob_elems; e += blockDim.x) wsm[e] = F64 ? (TD)P.blob64[e] : (TD)P.blob[e];
        __syncthreads();
    } else {
        for (int mu = warp; mu < H; mu += kGenWarps) {                    // one row per warp: every load in flight at once
            TD* dst = wsm + mu * Dps;
            if (F64) {
                for (int v = lane; v < Dps; v += 32) dst[v] = v < D ? (TD)P.params64[(size_t)mu * D + v] : (TD)0;
            } else {
                for (int c = lane; c < Dp / 4; c += 32) cp_async16(dst + 4 * c, P.params + (size_t)mu * Dp + 4 * c);
                if (lane < 4) dst[Dp + lane] = (TD)0;
            }
        }
        for (int e = threadIdx.x; e < 2 * H + 1; e += blockDim.x)
            wsm[H * Dps + e] = F64 ? (TD)P.params64[(size_t)H * D + e] : (TD)P.params[(size_t)H * Dp + e];
        cp_async_wait_all();
        __syncthreads();
    }
    const TD* b1s = wsm + H * Dps;
    const TD* w2s = b1s + H;

    for (int base = (blockIdx.x * kGenWarps + warp) * kGenGroups; base < N; base += gridDim.x * kGenAtomsPerBlock) {
        const int ia = base + grp;
        const bool valid = ia < N;
        const int i = valid ? ia : N - 1;
        const int nR = valid ? d.nnR[i] : 0, nA = valid ? d.nnA[i] : 0;
        // warp-uniform trip counts: the four groups of a warp stay converged
        const int chR = (__reduce_max_sync(0xffffffffu, nR) + kGenLanes - 1) / kGenLanes;
        const int chA = (__reduce_max_sync(0xffffffffu, nA) + kGenLanes - 1) / kGenLanes;
        const int ti = d.type_s[i];
        double4 pi = make_double4(0.0, 0.0, 0.0, 0.0);
        double bL[3] = {P.box.L[0], P.box.L[1], P.box.L[2]}, bI[3] = {P.box.invL[0], P.box.invL[1], P.box.invL[2]};
        if (F64) {
            pi = d.xs4[i];
            if (P.boxes) {                                                // every structure of a concatenated set has its own box
                const double* bx = P.boxes + 6 * (size_t)P.sid[i];
#pragma unroll
                for (int a = 0; a < 3; ++a) { bL[a] = bx[a]; bI[a] = bx[3 + a]; }
            }
        }

        // neighbour k of the atom in the descriptor precision: unit vector, distance, Eq. 19 weight
        auto nbr = [&](int k, TD& x, TD& y, TD& z, TD& r, TD& om) {
            const int slot = gen_slot(k, nA, capR);
            if (F64) {
                const int j = (int)(__float_as_uint(d.rec[rix(slot, i, N)].w) & kJMask);
                const double4 pj = d.xs4[j];
                const double dx = min_image(pj.x - pi.x, bL[0], bI[0]);
                const double dy = min_image(pj.y - pi.y, bL[1], bI[1]);
                const double dz = min_image(pj.z - pi.z, bL[2], bI[2]);
                const double rr = sqrt(dx * dx + dy * dy + dz * dz), ri = 1.0 / rr;
                x = (TD)(dx * ri); y = (TD)(dy * ri); z = (TD)(dz * ri); r = (TD)rr;
                om = (TD)P.zz64[ti * kMaxTypes + ((int)__double_as_longlong(pj.w) & (kMaxTypes - 1))];
            } else {
                const float4 e = d.rec[rix(slot, i, N)];
                const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
                const float ri = inv_norm(r2);
                x = (TD)(e.x * ri); y = (TD)(e.y * ri); z = (TD)(e.z * ri); r = (TD)(r2 * ri);
                om = (TD)P.zz[ti * kMaxTypes + d.type_s[__float_as_uint(e.w) & kJMask]];
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
#pragma unroll
                for (int o = 1; o < kGenLanes; o <<= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (gl == (n % kGenLanes) && n < NR) sm.q[n] = v;
            }
        }

        // ---- D: angular sums s[n][lm] and q_nl (Eq. 13 through Eq. 17-18 with n' = n) ----
        {
            constexpr int NH = NMAX / kGenSplit;                          // n slice of a lane
            const int tl = gl & 7, hn = (gl >> 3) * NH;                   // lm triple 3 tl .. 3 tl + 2, n in hn .. hn + NH - 1
            TD acc[NH][3];
#pragma unroll
            for (int n = 0; n < NH; ++n) { acc[n][0] = acc[n][1] = acc[n][2] = (TD)0; }
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
                const int kend = min(kGenLanes, __reduce_max_sync(0xffffffffu, nA) - c * kGenLanes);     // warp-uniform
#pragma unroll
                for (int kk = 0; kk < kGenLanes; ++kk) {
                    if (kk >= kend) break;                                // warp-uniform
                    const TD b0 = sm.Bs[kk][3 * tl], b1 = sm.Bs[kk][3 * tl + 1], b2 = sm.Bs[kk][3 * tl + 2];
#pragma unroll
                    for (int n = 0; n < NH; ++n) {
                        const TD gn = sm.Gs[kk][hn + n];
                        acc[n][0] += gn * b0; acc[n][1] += gn * b1; acc[n][2] += gn * b2;
                    }
                }
                __syncwarp();
            }
#pragma unroll
            for (int n = 0; n < NH; ++n) {
                sm.S[hn + n][3 * tl] = acc[n][0]; sm.S[hn + n][3 * tl + 1] = acc[n][1]; sm.S[hn + n][3 * tl + 2] = acc[n][2];
            }
            __syncwarp();
            if (P.kind == 1) {                                           // q_nn'l = (2l+1)/(4 pi) sum_m C_lm s_nlm s_n'lm, n <= n'
                for (int pi2 = gl; pi2 < NA * (NA + 1) / 2; pi2 += kGenLanes) {
                    int n = 0, rem = pi2;
                    while (rem >= NA - n) { rem -= NA - n; ++n; }
                    const int n2 = n + rem;
                    TD v[4] = {(TD)0, (TD)0, (TD)0, (TD)0};
#pragma unroll
                    for (int m = 0; m < kNumLM; ++m) v[LOF[m] - 1] += (TD)C[m] * sm.S[n][m] * sm.S[n2][m];
#pragma unroll
                    for (int l = 0; l < 4; ++l)
                        if (l < LMAX) sm.q[NR + pi2 * LMAX + l] = v[l] * (TD)((2 * l + 3) * 0.07957747154594767);    // (2l+1)/(4 pi), l = index + 1
                }
            } else
            for (int n = gl; n < NA; n += kGenLanes) {                   // q_nl, descriptor order n-major, l = 1..l_max
                TD v[4] = {(TD)0, (TD)0, (TD)0, (TD)0};
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) { const TD sv = sm.S[n][m]; v[LOF[m] - 1] += (TD)C[m] * sv * sv; }
#pragma unroll
                for (int l = 0; l < 4; ++l)
                    if (l < LMAX) sm.q[NR + n * LMAX + l] = v[l];
            }
            __syncwarp();
        }
        if (P.q_out && valid) {
            const int row = d.perm[i];
            for (int v = gl; v < D; v += kGenLanes) P.q_out[(size_t)v * N + row] = (float)sm.q[v];
        }

        // ---- N: network, Eq. 21-22 (minus biases), and Fp = dU/dq ----
        if (P.nlayers > 1) {                  // more hidden layers: x^(k) = tanh(W^(k) x^(k-1) - b^(k))
            if (gl < Dp - D) sm.q[D + gl] = (TD)0;
            __syncwarp();
            const int L = P.nlayers;
            TD* bufs[3] = {sm.hid, sm.act[0], sm.act[1]};
            const TD* xin = sm.q;
            for (int k = 0; k < L; ++k) {
                const int wk = P.lw[k], inp = P.lin_p[k];
                const TD* W = wsm + P.off_w[k];
                const TD* bk = wsm + P.off_b[k];
                TD* xout = bufs[k];
                for (int mu = gl; mu < wk; mu += kGenLanes) {
                    const TD* w = W + mu * inp;
                    TD a0 = -bk[mu], a1 = (TD)0;
                    for (int v = 0; v < inp; v += 2) { a0 += w[v] * xin[v]; a1 += w[v + 1] * xin[v + 1]; }
                    TD t, dd;
                    GenMath<TD>::act(a0 + a1, &t, &dd);
                    xout[mu] = t;
                }
                if (gl < 4 && wk + gl < kMaxHGen) xout[wk + gl] = (TD)0;  // zero tail up to the next layer's padded row length
                __syncwarp();
                xin = xout;
            }
            const int HL = P.lw[L - 1];
            const TD* wout = wsm + P.off_out;
            TD* xl = bufs[L - 1];
            TD Upart = (TD)0;
            for (int m = gl; m < HL; m += kGenLanes) {
                const TD t = xl[m];
                Upart += wout[m] * t;
                xl[m] = wout[m] * ((TD)1 - t) * ((TD)1 + t);              // delta^(L)
            }
#pragma unroll
            for (int o = 1; o < kGenLanes; o <<= 1) Upart += __shfl_xor_sync(0xffffffffu, Upart, o);
            if (gl == 0 && valid) d.Us[i] = (float)(Upart - wout[HL]);
            __syncwarp();
            for (int k = L - 1; k >= 0; --k) {                            // delta^(k-1) = (W^(k))^T delta^(k) (1 - x^(k-1)^2)
                const int wk = P.lw[k], inp = P.lin_p[k], nin = k == 0 ? D : P.lw[k - 1];
                const TD* W = wsm + P.off_w[k];
                const TD* dk = bufs[k];
                for (int v = gl; v < nin; v += kGenLanes) {
                    TD sacc = (TD)0;
                    for (int m = 0; m < wk; ++m) sacc += dk[m] * W[m * inp + v];
                    if (k == 0) sm.Fp[v] = (float)sacc;
                    else { const TD t = bufs[k - 1][v]; bufs[k - 1][v] = sacc * ((TD)1 - t) * ((TD)1 + t); }
                }
                __syncwarp();
            }
        } else {
            if (gl < Dp - D) sm.q[D + gl] = (TD)0;                        // the padded tail of q (w1's padded columns are zero too)
            __syncwarp();
            TD Upart = (TD)0;
            for (int mu = gl; mu < H; mu += kGenLanes) {
                const TD* w = wsm + mu * Dps;
                TD a0 = -b1s[mu], a1 = (TD)0, a2 = (TD)0, a3 = (TD)0;
                if (F64) {
#pragma unroll 4
                    for (int v = 0; v < Dp; v += 4) {                   // padded columns of w1 and the padded tail of q are zero
                        a0 += w[v] * sm.q[v]; a1 += w[v + 1] * sm.q[v + 1]; a2 += w[v + 2] * sm.q[v + 2]; a3 += w[v + 3] * sm.q[v + 3];
                    }
                } else {                                                // one LDS.128 of weights and one of q per four FMAs
                    const float4* w4 = reinterpret_cast<const float4*>(w);
                    const float4* q4 = reinterpret_cast<const float4*>(&sm.q[0]);
#pragma unroll 5
                    for (int v = 0; v < Dp / 4; ++v) {
                        const float4 ww = w4[v], qq = q4[v];
                        a0 += (TD)ww.x * (TD)qq.x; a1 += (TD)ww.y * (TD)qq.y; a2 += (TD)ww.z * (TD)qq.z; a3 += (TD)ww.w * (TD)qq.w;
                    }
                }
                const TD a = (a0 + a1) + (a2 + a3);
                const TD w2 = w2s[mu];
                TD t, dd;
                GenMath<TD>::act(a, &t, &dd);
                Upart += w2 * t;
                sm.hid[mu] = w2 * dd;
            }
#pragma unroll
            for (int o = 1; o < kGenLanes; o <<= 1) Upart += __shfl_xor_sync(0xffffffffu, Upart, o);
            __syncwarp();
            if (gl == 0 && valid) {
                d.Us[i] = (float)(Upart - w2s[H]);                        // - b2
            }
            for (int v4 = gl; v4 < Dp / 4; v4 += kGenLanes) {              // four descriptor components per lane
                TD f0 = (TD)0, f1 = (TD)0, f2 = (TD)0, f3 = (TD)0;
                if (F64) {
#pragma unroll 4
                    for (int mu = 0; mu < H; ++mu) {
                        const TD gm = sm.hid[mu];
                        const TD* w = wsm + mu * Dps + 4 * v4;
                        f0 += gm * w[0]; f1 += gm * w[1]; f2 += gm * w[2]; f3 += gm * w[3];
                    }
                } else {
#pragma unroll 5
                    for (int mu = 0; mu < H; ++mu) {
                        const TD gm = sm.hid[mu];
                        const float4 ww = *reinterpret_cast<const float4*>(wsm + mu * Dps + 4 * v4);
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
        if (P.kind == 1) {
            // A[n][m] = (2l+1)/(4 pi) C_m [ 2 Fp_nn s_n + sum_{b>n} Fp_nb s_b + sum_{a<n} Fp_an s_a ]: needs every row of s,
            // so it is built beside s (TD = float: in the chunk buffers, free by now)
            if (!F64) A = reinterpret_cast<float*>(&sm.Gs[0][0]);
            for (int e = gl; e < NMAX * kNumLM; e += kGenLanes) {
                const int n = e / kNumLM, m = e - n * kNumLM;
                float acc = 0.f;
                if (n < NA) {
                    int lm1 = 0;                                          // l - 1 of component m
                    lm1 = m < 3 ? 0 : (m < 8 ? 1 : (m < 15 ? 2 : 3));
                    if (lm1 < LMAX) {
                        for (int b = 0; b < NA; ++b) {
                            const int lo = min(n, b), hi = max(n, b);
                            const int pidx = lo * NA - lo * (lo - 1) / 2 + (hi - lo);
                            const float f = sm.Fp[NR + pidx * LMAX + lm1] * (b == n ? 2.f : 1.f);
                            acc = fmaf(f, (float)sm.S[b][m], acc);
                        }
                        acc *= clm(m) * (float)((2 * lm1 + 3) * 0.07957747154594767);
                    }
                }
                A[e] = acc;
            }
        } else
        for (int n = gl; n < NMAX; n += kGenLanes) {                     // row n: in place when TD = float (same lane reads and writes it)
            float fl[4];
#pragma unroll
            for (int l = 0; l < 4; ++l) fl[l] = (n < NA && l < LMAX) ? 2.f * sm.Fp[NR + n * LMAX + l] : 0.f;
#pragma unroll
            for (int m = 0; m < kNumLM; ++m) A[n * kNumLM + m] = C[m] * fl[LOF[m] - 1] * (float)sm.S[n][m];
        }
        __syncwarp();
        float fsx = 0.f, fsy = 0.f, fsz = 0.f;
        float4* prow = d.p + (size_t)i * capR;
        for (int c = 0; c < chR; ++c) {
            const int k = c * kGenLanes + gl;
            const bool on = k < nR;
            const int slot = gen_slot(on ? k : 0, nA, capR);
            float4 e = make_float4(1.f, 0.f, 0.f, __uint_as_float((unsigned)i));
            if (on) e = d.rec[rix(slot, i, N)];
            const float r2 = e.x * e.x + e.y * e.y + e.z * e.z;
            const float rinv = inv_norm(r2), r = r2 * rinv;
            const float x = e.x * rinv, y = e.y * rinv, z = e.z * rinv;
            const float om = P.zz[ti * kMaxTypes + d.type_s[__float_as_uint(e.w) & kJMask]];
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
                f32x2 acc2[kNumLM];                                      // {S'_m, S_m / r} packed: one FFMA2 per (n, m)
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) acc2[m] = pack2(0.f, 0.f);
#pragma unroll
                for (int n = 0; n < NMAX; ++n) {                         // rows n >= NA of A are zero: no branch (a uniform
                    const float4* An = reinterpret_cast<const float4*>(A + n * kNumLM);      // `if (n < NA)` cost a MOV per FFMA2)
                    const f32x2 dgs = pack2(dg[n], gs[n]);
#pragma unroll
                    for (int m4 = 0; m4 < kNumLM / 4; ++m4) {
                        const float4 a = An[m4];
                        acc2[4 * m4] = ffma2(pack2(a.x, a.x), dgs, acc2[4 * m4]);
                        acc2[4 * m4 + 1] = ffma2(pack2(a.y, a.y), dgs, acc2[4 * m4 + 1]);
                        acc2[4 * m4 + 2] = ffma2(pack2(a.z, a.z), dgs, acc2[4 * m4 + 2]);
                        acc2[4 * m4 + 3] = ffma2(pack2(a.w, a.w), dgs, acc2[4 * m4 + 3]);
                    }
                }
                float Sq[kNumLM], St[kNumLM];
#pragma unroll
                for (int m = 0; m < kNumLM; ++m) unpack2(acc2[m], Sq[m], St[m]);
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
