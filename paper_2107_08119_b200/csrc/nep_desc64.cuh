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
// One thread per atom in k_order's window-sorted order (the column k_main uses); the 24 lm components are
// swept in three passes of 8 so that the 8 x 8 double accumulators stay in registers.
#pragma once

// fp64 geometry of neighbour `slot` of atom i: minimum-image r_ij from the fp64 positions, and Eq. 19's weight
struct Nbr64 { double x, y, z, r, om; };
__device__ __forceinline__ Nbr64 nbr64(const SysDev& d, const Box& b, const double4& pi, const double* zrow, int slot, int N, int i) {
    const int j = (int)(__float_as_uint(d.rec[rix(slot, i, N)].w) & kJMask);
    const double4 pj = d.xs4[j];
    Nbr64 o;
    o.x = min_image(pj.x - pi.x, b.L[0], b.invL[0]);
    o.y = min_image(pj.y - pi.y, b.L[1], b.invL[1]);
    o.z = min_image(pj.z - pi.z, b.L[2], b.invL[2]);
    o.r = sqrt(o.x * o.x + o.y * o.y + o.z * o.z);
    o.om = zrow[(int)__double_as_longlong(pj.w) & (kMaxTypes - 1)];
    return o;
}

constexpr int kD64Rows = 16;          // angular neighbours whose geometry is kept in shared memory between the sweeps (48 KB per block)

// One third of the angular sums (lm components 8 T .. 8 T + 7; 64 register accumulators): s, its share of
// q_nl, and s rounded to fp32 into k_main's parked layout.  The first third also does Eq. 12 for the
// angular neighbours.
template <int T, int NR, int NA>
__device__ __forceinline__ void desc64_third(const SysDev& d, const Box& b, const Desc64Params& P, const double4& pi,
                                             const double* zrow, int i, int nA, size_t npad, size_t gcol, double* q) {
    constexpr double C[kNumLM] = {NEP_CLM_LIST};
    constexpr int LOF[kNumLM] = {NEP_LOF_LIST};
    constexpr int NP = kHalfLM / 2;
    const int N = P.N;
    double s[NA][8];
#pragma unroll
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int m = 0; m < 8; ++m) s[n][m] = 0.0;
    extern __shared__ double sgeo[];                                     // [kD64Rows][6][64]: x, y, z, r, omega, cos(pi r / r_c^A)
    for (int k = 0; k < nA; ++k) {
        // the first sweep leaves the neighbour's geometry and its cutoff cosine in shared memory: the other two read
        // them instead of repeating the gather, the minimum image, the square root and the fp64 cosine
        Nbr64 e;
        double cosA;
        double* row = sgeo + (size_t)(k * 6) * 64 + threadIdx.x;
        if (T == 0 || k >= kD64Rows) {
            e = nbr64(d, b, pi, zrow, k, N, i);
            cosA = cos(3.14159265358979323846 * (e.r / P.rcA));
            if (T == 0 && k < kD64Rows) { row[0] = e.x; row[64] = e.y; row[128] = e.z; row[192] = e.r; row[256] = e.om; row[320] = cosA; }
        } else {
            e.x = row[0]; e.y = row[64]; e.z = row[128]; e.r = row[192]; e.om = row[256]; cosA = row[320];
        }
        double g[NR > NA ? NR : NA];
        if (T == 0) {
            radial_g64<NR>(e.r, P.rcR, e.om, g);
#pragma unroll
            for (int n = 0; n < NR; ++n) q[n] += g[n];                   // Eq. 12
        }
        radial_g64c<NA>(e.r, P.rcA, e.om, cosA, g);
        double bb[kNumLM];
        const double rinv = 1.0 / e.r;
        ylm_basis64(e.x * rinv, e.y * rinv, e.z * rinv, bb);             // the unused components are dead code
#pragma unroll
        for (int n = 0; n < NA; ++n)
#pragma unroll
            for (int m = 0; m < 8; ++m) s[n][m] += g[n] * bb[8 * T + m];   // Eq. 18 in real form
    }
#pragma unroll
    for (int n = 0; n < NA; ++n)
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            constexpr int dummy = 0; (void)dummy;
            const int gm = 8 * T + m;                                    // global lm index (compile-time after unrolling)
            q[NR + 4 * n + LOF[gm] - 1] += C[gm] * s[n][m] * s[n][m];   // Eq. 17 with n' = n
            // k_main's parked layout: half 0 holds m 0..2 and 15..23, half 1 holds m 3..14
            const bool h0 = gm < 3 || gm >= 15;
            const int kk = h0 ? (gm < 3 ? gm : gm - 12) : gm - 3;
            float* base = reinterpret_cast<float*>(h0 ? d.spark0 : d.spark1);
            base[((size_t)(n * NP + (kk >> 1)) * npad + gcol) * 2 + (kk & 1)] = (float)s[n][m];
        }
}

template <int NR, int NA>
__global__ void __launch_bounds__(64) k_desc64(SysDev d, Box b, const __grid_constant__ Desc64Params P,
                                               const double* __restrict__ par /* w1[H][D] | b1[H] | w2[H] | b2 */) {
    constexpr int D = NR + 4 * NA;
    constexpr int NP = kHalfLM / 2;
    constexpr double C[kNumLM] = {NEP_CLM_LIST};
    constexpr int LOF[kNumLM] = {NEP_LOF_LIST};
    const size_t gcol = (size_t)blockIdx.x * 64 + threadIdx.x;
    const size_t npad = (size_t)gridDim.x * 64;
    const int i = d.order[gcol].x;
    if (i < 0) return;
    const int N = P.N;
    const int nR = d.nnR[i], nA = d.nnA[i];
    const double4 pi = d.xs4[i];
    const double* zrow = P.zz + (int)__double_as_longlong(pi.w) * kMaxTypes;

    double q[D];
#pragma unroll
    for (int v = 0; v < D; ++v) q[v] = 0.0;
    for (int k = nA; k < nR; ++k) {                                      // Eq. 12, radial-only neighbours
        const Nbr64 e = nbr64(d, b, pi, zrow, P.capR - 1 - (k - nA), N, i);
        double g[NR];
        radial_g64<NR>(e.r, P.rcR, e.om, g);
#pragma unroll
        for (int n = 0; n < NR; ++n) q[n] += g[n];
    }
    desc64_third<0, NR, NA>(d, b, P, pi, zrow, i, nA, npad, gcol, q);
    desc64_third<1, NR, NA>(d, b, P, pi, zrow, i, nA, npad, gcol, q);
    desc64_third<2, NR, NA>(d, b, P, pi, zrow, i, nA, npad, gcol, q);

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
    if (P.q_out) {                                                       // parity hook (nep_compute_internals)
        const int row = d.perm[i];
#pragma unroll
        for (int v = 0; v < D; ++v) P.q_out[(size_t)v * N + row] = (float)q[v];
    }
#pragma unroll
    for (int v = 0; v < D; ++v) d.FpG[(size_t)v * npad + gcol] = (float)Fp[v];
}
