// nep_b200.cu -- libnep_b200.so: NEP force evaluation for one B200 (sm_100a).  C ABI: include/nep_b200.h.
//
// Data flow of one evaluation (all in the cell-sorted atom order):
//   k_filter    Verlet list -> per-step radial/angular lists as records {r_ij (fp32 from an fp64
//               minimum-image difference), j | rev << 24}; predicate |d|^2 < r_c^2 in fp64; two records of an
//               atom leave as one full 32-byte sector
//   k_main      one thread per atom: radial descriptor (Eq. 12), angular sums s[n][lm] (Eq. 17-18 route
//               to Eq. 13), network (Eq. 21-22) and dU/dq, partial forces (Eq. 23-25) -> p_ij
//   k_assemble  F_i = sum_j (p_ij - p_ji), W_i = sum_j r_ij (x) p_ji (Eq. 4-6), second half-kick,
//               J_i = W_i . v_i (Eq. 7), thermo sums; outputs in the caller's atom order; then the NEXT
//               step's first half-kick and drift (not after the last step of a call)
// Neighbour build (rare): k_bin -> k_scan -> k_fill -> k_sort_cells -> k_gather -> k_build_md -> k_rev.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>
#include <math.h>
#include <new>
#include <math_constants.h>

#include "../../include/nep_b200.h"
#include "../../include/nep_b200_measure.h"
#include "nep_math.cuh"

using namespace nepk;

namespace {

constexpr int kMaxTypes = 8;
constexpr unsigned kJMask = 0x00FFFFFFu;       // sorted index of the neighbour (N < 2^24)
constexpr int kMaxCapMD = 124;                // Verlet slots per atom: the accepted-slot masks hold 128 bits
constexpr double kAmuConv = 103.642697;       // 1 amu A^2/fs^2 in eV

// device status / counter words (int32 each)
enum { F_STATUS = 0, F_REBUILD = 1, F_STEP = 2, F_NREBUILD = 3, F_MAXR = 4, F_MAXA = 5, F_MAXMD = 6, F_BUILT = 7, F_NSTEPS = 8,
       F_COUNT = 16 };
enum { ST_OVERFLOW = 1, ST_STALE = 2, ST_BADTYPE = 4, ST_NAN = 8 };

struct Box {
    double L[3], invL[3];
    int nc[3];
    int ncell;
};

struct SysDev {                 // device pointers into the caller's workspace
    int* flags;
    int* type_in;               // [N] caller order
    int* perm;                  // [N] sorted -> caller index
    int* perm_tmp;              // [N]
    int* cell_of;               // [N] cell id in the order of the build input
    int* cell_cnt;              // [max_cells + 1]
    int* cell_start;            // [max_cells + 1]
    int* cell_fill;             // [max_cells]
    int* type_s;                // [N] sorted
    double* xs;                 // [3][N] sorted positions (unwrapped)
    double4* xs4;               // [N] the same as {x, y, z, bits(type)}: one 32-B sector per gathered neighbour
    double* vs;                 // [3][N] sorted velocities
    double* xref;               // [3][N] sorted positions at the last build
    double* tmp3;               // [3][N]
    float* Fs;                  // [3][N] sorted forces
    float* Us;                  // [N] sorted site energies
    float4* Fself;              // [N] sum_j p_ij
    int* md_cnt;                // [N]
    unsigned* md_idx;           // [ceil(cap_md/8)][N][8]  j | rev << 24   (rev: slot of i in j's Verlet row, < 128): eight
                                //   consecutive slots of an atom are one 32-byte sector, written and read as such; element (slot, i) at mix()
    int capMD;                  // slots per Verlet row
    int* nnR;                   // [N]
    int* nnA;                   // [N]
    float4* rec;                // [ceil(cap_R/2)][N][2]  {dx, dy, dz, bits(j | rev << 24)}: slots 2k and 2k+1 of an atom share one
                                //   32-byte sector (k_filter stores them as ONE full sector: partial-sector stores run at a
                                //   quarter of the rate); element (slot, i) at rix(slot, i, N)      (read by k_main, k_assemble)
    uint4* masks;               // [N][2] bit s set: Verlet slot s is inside r_c^R ([0]) / r_c^A ([1])
    float4* p;                  // [N][cap_R] partial forces dU_i/dr_ij at the record slots
    float2* spark0;             // [NA*6][ceil(N/kWin)*kWin] angular sums s[n][lm] of lm half 0 / half 1: parked here by k_main
    float2* spark1;             //   (coalesced rows, L2-resident between write and read) while the registers hold other phases
    float* FpG;                 // [D][ceil(N/kWin)*kWin] dU/dq from k_desc64 (multi-species models only)
    int* smslots;               // [256] per SM: which of its parking slots (k_main) are taken
    int2* order;                // [ceil(N/kWin)*kWin] atoms of each kWin-atom window sorted by neighbour count: {atom (-1: none),
                                //   nA | nR << 8}, so that k_main needs ONE load before it can fetch its records
};

constexpr int kMaxH = 64;           // hidden neurons k_main supports (it stages the weights in shared memory)
constexpr int64_t kThreadPathMinAtoms = 12000;    // nep_system_create: from here on k_main (one thread per atom) is chosen (crossover measured at ~8-10k atoms)

// sqrt(Z_a Z_b) of Eq. 19, passed to k_main by value (kernel-parameter constant bank)
struct ZZParams {
    float zz[kMaxTypes * kMaxTypes];
};

// parameters of k_desc64 (nep_desc64.cuh), passed by value
struct Desc64Params {
    double rcR, rcA;
    double zz[kMaxTypes * kMaxTypes];     // sqrt(Z_a Z_b) in double
    int H, N, capR;
    float* q_out;                         // nullable parity hook, [D][N] caller order
};

// element (slot, i) of the octet-major Verlet array
// (N < 2^24 and at most 128 slots: the element index fits 32 bits)
__host__ __device__ __forceinline__ unsigned mix(int slot, int i, int N) { return ((((unsigned)(slot >> 3)) * (unsigned)N + (unsigned)i) << 3) | (unsigned)(slot & 7); }
// element (slot, i) of the pair-major record array
__host__ __device__ __forceinline__ unsigned rix(int slot, int i, int N) { return ((((unsigned)(slot >> 1)) * (unsigned)N + (unsigned)i) << 1) | (unsigned)(slot & 1); }

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

}  // namespace

constexpr int kProfMaxEvents = 2048;
enum { PH_KICK = 0, PH_BUILD = 1, PH_FILTER = 2, PH_MAIN = 3, PH_ASSEMBLE = 4, PH_STATE = 5, NEP_PHASES = 8 };

struct nep_model {
    nep_hyper h;
    int D, NR, NA, H, npar;
    int Z[kMaxTypes];
    float* params_dev;          // staged fp32 layout: w1[H][Dp] (rows zero-padded) | b1[H] | w2[H] | b2 | pad
    int params_floats;
    ZZParams zz;
    double* params64_dev;       // multi-species models: the Eq. 26 vector in double, caller order (k_desc64, k_gen<double>)
    Desc64Params p64;
    bool thread_path_ok;        // k_main / k_desc64 are instantiated for this shape
    // variants (nep_create_ex): SOAP-like descriptor, two or three hidden layers
    int kind, nlayers, lw[3], lin_p[3], off_w[3], off_b[3], off_out, blob_elems;
    float* blob_dev; double* blob64_dev;
};

struct nep_system {
    const nep_model* model;
    int64_t N;
    int capR, capA, capMD, max_cells;
    double skin;
    SysDev d;
    Box box;
    bool built, have_forces;
    const double* batch_boxes; const int* batch_sid;     // set by nep_trainer: concatenated structures, one box each
    bool last_driven; float last_fe[3];    // equations of motion of the last nep_md_step (its kick force is reused)
    int path;                              // NEP_PATH_THREAD or NEP_PATH_GROUP: which kernel evaluates Eq. 12-25
    float* dump_q; float* dump_fp;        // set only inside nep_compute_internals
    cudaStream_t last_stream;
    // one MD step captured as a CUDA graph (replayed n_steps times; re-captured when its arguments change)
    cudaGraphExec_t step_graph;
    cudaStream_t cap_stream;               // library-owned stream used only for capture
    unsigned char g_key[512];              // AsmParams + dt of the captured step
    int64_t g_launches;                    // kernels per replay
    int64_t host_stats[4];
    int64_t launches;                      // kernels launched since creation
    // optional per-phase event timing (nep_profile)
    bool prof_on;
    int prof_n;                            // events recorded
    cudaEvent_t prof_ev[kProfMaxEvents];
    int prof_phase[kProfMaxEvents];        // phase that STARTS at event k (-1: end marker)
    double prof_ms[NEP_PHASES];
    int64_t prof_cnt[NEP_PHASES];
};

namespace {

// ------------------------------------------------------------------------------------------------
// neighbour build
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ int cell_coord(double x, double L, double invL, int nc) {
    double f = x * invL;
    f -= floor(f);
    int c = (int)(f * nc);
    return c >= nc ? nc - 1 : (c < 0 ? 0 : c);
}

__device__ __forceinline__ bool gate_closed(const int* flags, int gated) { return gated && flags[F_REBUILD] == 0; }

// Each phase of the build is a device function over a flat thread index (tid of nth): the same bodies serve
// the multi-kernel chain (large systems: one kernel per phase, all SMs) and k_build_cluster (small systems:
// one launch, the phases separated by cluster barriers).
__device__ __forceinline__ void ph_clear(const SysDev& d, int ncell, int tid, int nth) {
    for (int c = tid; c <= ncell; c += nth) d.cell_cnt[c] = 0;
}

// cell id of every atom of the build input `x` ([3][N]) and the per-cell population
__device__ __forceinline__ void ph_bin(const SysDev& d, const double* __restrict__ x, int N, const Box& b, int tid, int nth) {
    for (int i = tid; i < N; i += nth) {
        const int cx = cell_coord(x[i], b.L[0], b.invL[0], b.nc[0]);
        const int cy = cell_coord(x[N + i], b.L[1], b.invL[1], b.nc[1]);
        const int cz = cell_coord(x[2 * N + i], b.L[2], b.invL[2], b.nc[2]);
        const int c = (cx * b.nc[1] + cy) * b.nc[2] + cz;
        d.cell_of[i] = c;
        atomicAdd(&d.cell_cnt[c], 1);
    }
}

// exclusive scan of cell_cnt[0..ncell) -> cell_start[0..ncell]; one block of 1024 threads
// exclusive scan of the cell counts by ONE block of 1024 threads, in tiles of 4096 cells: coalesced loads, a shuffle scan
// per warp and one over the 32 warp totals (a contiguous chunk per thread cost 156 us for the 91k cells of the 1M-atom box)
__device__ __forceinline__ void ph_scan(const SysDev& d, int ncell, int* part /* shared, [1024] */) {
    const int t = threadIdx.x, lane = t & 31, wid = t >> 5;
    int carry = 0;                                   // atoms in the cells before this tile
    for (int base = 0; base < ncell; base += 4096) {
        const int c0 = base + 4 * t;
        int v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = c0 + u < ncell ? d.cell_cnt[c0 + u] : 0;
        const int mine = (v[0] + v[1]) + (v[2] + v[3]);
        int incl = mine;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int x = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += x;
        }
        if (lane == 31) part[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            const int w = part[lane];
            int wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int x = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += x;
            }
            part[32 + lane] = wi - w;                // warps before this one
            if (lane == 31) part[64] = wi;           // the tile's total
        }
        __syncthreads();
        int run = carry + part[32 + wid] + incl - mine;
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (c0 + u < ncell) { d.cell_start[c0 + u] = run; d.cell_fill[c0 + u] = run; run += v[u]; }
        carry += part[64];
        __syncthreads();
    }
    if (t == 0) d.cell_start[ncell] = carry;
}

__device__ __forceinline__ void ph_fill(const SysDev& d, int N, int tid, int nth) {
    for (int i = tid; i < N; i += nth) {
        const int slot = atomicAdd(&d.cell_fill[d.cell_of[i]], 1);
        d.perm_tmp[slot] = i;
    }
}

// deterministic order inside a cell: ascending build-input index (insertion sort, cells are small)
__device__ __forceinline__ void ph_sort_cells(const SysDev& d, int ncell, int tid, int nth) {
    for (int c = tid; c < ncell; c += nth) {
        const int lo = d.cell_start[c], hi = d.cell_start[c + 1];
        for (int a = lo + 1; a < hi; ++a) {
            const int v = d.perm_tmp[a];
            int k = a - 1;
            while (k >= lo && d.perm_tmp[k] > v) { d.perm_tmp[k + 1] = d.perm_tmp[k]; --k; }
            d.perm_tmp[k + 1] = v;
        }
    }
}

// Gather the build input into the new sorted order.  first != 0: input is the caller's arrays
// (perm := perm_tmp).  first == 0 (in-loop rebuild): input is the current sorted state, so
// perm := perm[perm_tmp]; velocities move too.  Two-phase through tmp buffers (gather_a / gather_b).
__device__ __forceinline__ void ph_gather_a(const SysDev& d, const double* __restrict__ xin, const double* __restrict__ vin,
                                            int N, int first, int tid, int nth) {
    for (int k = tid; k < N; k += nth) {
        const int src = d.perm_tmp[k];
#pragma unroll
        for (int a = 0; a < 3; ++a) d.xref[a * N + k] = xin[a * N + src];
        if (vin) {
#pragma unroll
            for (int a = 0; a < 3; ++a) d.tmp3[a * N + k] = vin[a * N + src];
        }
        d.cell_of[k] = first ? src : d.perm[src];      // cell_of is free now: reuse as the new perm
    }
}

__device__ __forceinline__ void ph_gather_b(const SysDev& d, int N, int have_v, int n_types, int tid, int nth) {
    for (int k = tid; k < N; k += nth) {
#pragma unroll
        for (int a = 0; a < 3; ++a) d.xs[a * N + k] = d.xref[a * N + k];
        if (have_v) {
#pragma unroll
            for (int a = 0; a < 3; ++a) d.vs[a * N + k] = d.tmp3[a * N + k];
        }
        const int p = d.cell_of[k];
        d.perm[k] = p;
        int ty = d.type_in[p];
        if (ty < 0 || ty >= n_types) { atomicOr(&d.flags[F_STATUS], ST_BADTYPE); ty = 0; }    // reported by nep_status as NEP_EINVAL
        d.type_s[k] = ty;
        d.xs4[k] = make_double4(d.xref[k], d.xref[N + k], d.xref[2 * N + k], __longlong_as_double((long long)ty));
    }
}

// gated == 2: the chain opens an MD step -- its first kernel also advances the step counter (nothing else runs then)
__global__ void k_clear_cells(SysDev d, int ncell, int gated) {
    if (gated == 2 && blockIdx.x == 0 && threadIdx.x == 0) d.flags[F_STEP] += 1;
    if (gate_closed(d.flags, gated)) return;
    ph_clear(d, ncell, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}
__global__ void k_bin(SysDev d, const double* __restrict__ x, int N, Box b, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_bin(d, x, N, b, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}
__global__ void __launch_bounds__(1024) k_scan(SysDev d, int ncell, int gated) {
    if (gate_closed(d.flags, gated)) return;
    __shared__ int part[1024];
    ph_scan(d, ncell, part);
}
__global__ void k_fill(SysDev d, int N, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_fill(d, N, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}
__global__ void k_sort_cells(SysDev d, int ncell, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_sort_cells(d, ncell, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}
__global__ void k_gather_a(SysDev d, const double* __restrict__ xin, const double* __restrict__ vin, int N,
                           int first, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_gather_a(d, xin, vin, N, first, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}
__global__ void k_gather_b(SysDev d, int N, int have_v, int n_types, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_gather_b(d, N, have_v, n_types, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

// 256-bit read-only loads (sm_100: LDG.E.256): one request per gathered 32-byte sector instead of two
__device__ __forceinline__ double4 ldg256(const double4* p) {
    double4 v;
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
    return v;
}
__device__ __forceinline__ void ldg256(const uint4* p, uint4& a, uint4& b) {      // p[0], p[1]
    unsigned long long x, y, z, w;
    asm volatile("ld.global.nc.v4.b64 {%0,%1,%2,%3}, [%4];" : "=l"(x), "=l"(y), "=l"(z), "=l"(w) : "l"(p));
    a = make_uint4((unsigned)x, (unsigned)(x >> 32), (unsigned)y, (unsigned)(y >> 32));
    b = make_uint4((unsigned)z, (unsigned)(z >> 32), (unsigned)w, (unsigned)(w >> 32));
}

// eight 32-bit words (one sector) as one load / one store
__device__ __forceinline__ void ld_octet(const unsigned* p, unsigned (&v)[8]) {
    asm volatile("ld.global.v8.u32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];" : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]),
                 "=r"(v[5]), "=r"(v[6]), "=r"(v[7]) : "l"(p));
}
__device__ __forceinline__ void st_octet(unsigned* p, const unsigned (&v)[8]) {
    asm volatile("st.global.v8.u32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]),
                 "r"(v[5]), "r"(v[6]), "r"(v[7]) : "memory");
}
// one 32-byte sector as one store (STG.E.256): {a, b} to a 32-byte aligned address
__device__ __forceinline__ void stg256(float4* p, const float4& a, const float4& b) {
    asm volatile("st.global.v8.f32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "f"(a.x), "f"(a.y), "f"(a.z), "f"(a.w),
                 "f"(b.x), "f"(b.y), "f"(b.z), "f"(b.w) : "memory");
}

__device__ __forceinline__ double min_image(double t, double L, double invL) { return t - L * rint(t * invL); }

// Verlet list: all j != i with |r_ij|^2 < (r_c^R + skin)^2, rows ascending in the sorted index j
// (neighbour cells are visited in ascending cell id; a cell's atoms are contiguous and ascending).
// NC: read positions through the non-coherent path (valid when an earlier KERNEL wrote them).
// the wrapped coordinates {c-1, c, c+1} of one axis in ascending order (one value when the axis has a single cell)
__device__ __forceinline__ int sorted_axis(int c, int nc, int (&a)[3]) {
    if (nc == 1) { a[0] = a[1] = a[2] = 0; return 1; }
    const int m = c == 0 ? nc - 1 : c - 1, p = c == nc - 1 ? 0 : c + 1;     // nc >= 3: three distinct values
    if (m > c) { a[0] = c; a[1] = p; a[2] = m; }          // c == 0:      {0, 1, nc-1}
    else if (p < c) { a[0] = p; a[1] = m; a[2] = c; }     // c == nc-1:   {0, nc-2, nc-1}
    else { a[0] = m; a[1] = c; a[2] = p; }
    return 3;
}

// LANES (1, 2 or 4 adjacent lanes of a warp) share an atom: each lane takes a contiguous part of the sorted cell
// list, keeps the neighbours it accepts in a small local buffer, and the parts are concatenated through a shuffle
// prefix -- the row stays ascending.  Small systems use it to spread one atom's ~310 candidate tests (a serial
// chain of FP64 latencies) over the otherwise idle threads of the cluster.
constexpr int kBuildBuf = 48;       // accepted neighbours a lane can buffer (a whole row when LANES = 1: else it re-scans)
template <bool NC, int LANES>
__device__ __forceinline__ void ph_build_md(const SysDev& d, int N, const Box& b, double rc2, int capMD, int tid, int nth) {
    const int l = tid % LANES;
    const int natoms_pad = ((N + 31) / 32) * 32;                     // whole warps stay in the loop (shuffles below)
    for (int i0 = tid / LANES; i0 < natoms_pad; i0 += nth / LANES) {
        const bool valid = i0 < N;
        const int i = valid ? i0 : N - 1;
        const double xi = d.xs[i], yi = d.xs[N + i], zi = d.xs[2 * N + i];
        const int cx = cell_coord(xi, b.L[0], b.invL[0], b.nc[0]);
        const int cy = cell_coord(yi, b.L[1], b.invL[1], b.nc[1]);
        const int cz = cell_coord(zi, b.L[2], b.invL[2], b.nc[2]);
        // The 27 neighbour cells in ascending cell id = lexicographic order of (X, Y, Z) with each axis' three wrapped
        // coordinates sorted; a (X, Y) column's Z cells are adjacent in memory, so an unwrapped column is ONE index range.
        int ax[3], ay[3], az[3];
        const int nx = sorted_axis(cx, b.nc[0], ax), ny = sorted_axis(cy, b.nc[1], ay), nz = sorted_axis(cz, b.nc[2], az);
        const bool zrun = nz == 1 || (az[2] - az[0] == 2);               // the column's Z cells are contiguous
        const int ncols = nx * ny;
        const int q0 = valid ? (l * ncols) / LANES : 0, q1 = valid ? ((l + 1) * ncols) / LANES : 0;
        int base = 0;                // slot of this lane's first neighbour (known after the first sweep when LANES > 1)
        int cnt = 0;
        unsigned buf[LANES > 1 ? kBuildBuf : 1];
        // sweep 0 counts (and buffers); with LANES == 1 it writes directly.  Sweep 1 (only if a buffer overflowed) re-scans.
        for (int sweep = 0; sweep < (LANES > 1 ? 2 : 1); ++sweep) {
            const bool direct = LANES == 1 || sweep == 1;
            cnt = 0;
            for (int qq = q0 * (zrun ? 1 : nz); qq < q1 * (zrun ? 1 : nz); ++qq) {
                const int q = zrun ? qq : qq / nz, zi0 = zrun ? 0 : qq % nz;
                const int col = (ax[q / ny] * b.nc[1] + ay[q % ny]) * b.nc[2];
                const int lo = d.cell_start[col + az[zi0]], hi = d.cell_start[col + az[zrun ? nz - 1 : zi0] + 1];
                for (int j0 = lo; j0 < hi; j0 += 4) {                // four candidates in flight (the loads are L2 round trips)
                    double4 pc[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = min(j0 + u, hi - 1);
                        pc[u] = NC ? ldg256(&d.xs4[j]) : d.xs4[j];
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int j = j0 + u;
                        if (j >= hi || j == i) continue;
                        const double4 pj = pc[u];
                        const double dx = min_image(pj.x - xi, b.L[0], b.invL[0]);
                        const double dy = min_image(pj.y - yi, b.L[1], b.invL[1]);
                        const double dz = min_image(pj.z - zi, b.L[2], b.invL[2]);
                        const double r2 = dx * dx + dy * dy + dz * dz;
                        if (r2 < rc2) {
                            if (direct) { if (base + cnt < capMD) d.md_idx[mix(base + cnt, i, N)] = j; }
                            else if (cnt < kBuildBuf) buf[cnt] = (unsigned)j;
                            ++cnt;
                        }
                    }
                }
            }
            if (LANES == 1) break;
            if (sweep == 0) {
                int incl = cnt;                                          // prefix over the lanes of the atom
#pragma unroll
                for (int o = 1; o < LANES; o <<= 1) {
                    const int v = __shfl_up_sync(0xffffffffu, incl, o, LANES);
                    if (l >= o) incl += v;
                }
                base = incl - cnt;
                const bool fits = cnt <= kBuildBuf;
                if (fits) {
                    for (int k = 0; k < cnt; ++k)
                        if (base + k < capMD) d.md_idx[mix(base + k, i, N)] = buf[k];
                }
                if (fits) break;                                         // (a lane whose buffer overflowed re-scans and writes directly)
            }
        }
        int total = cnt;
        if (LANES > 1) {
#pragma unroll
            for (int o = 1; o < LANES; o <<= 1) total += __shfl_xor_sync(0xffffffffu, total, o, LANES);
        }
        if (valid && l == 0) {
            d.md_cnt[i] = min(total, capMD);
            if (total > capMD) atomicOr(&d.flags[F_STATUS], ST_OVERFLOW);
            atomicMax(&d.flags[F_MAXMD], total);
        }
    }
}

// reverse slot: position of i in j's (ascending) row, by binary search -- eight searches at a time, so that the
// dependent probes of one search overlap those of seven others (the probes are L2 round trips)
__device__ __forceinline__ void ph_rev(const SysDev& d, int N, int tid, int nth) {
    constexpr int B = 8;
    // one task per (octet of a row, atom), atoms fastest: a row's octets are searched by different threads
    const int noct = (d.capMD + 7) >> 3;
    for (long long t = tid; t < (long long)noct * N; t += nth) {
        const int i = (int)(t % N), s0 = (int)(t / N) * B;
        const int cnt = d.md_cnt[i];
        if (s0 >= cnt) continue;
        int j[B], lo[B], hi[B];
        unsigned oct[8];
        ld_octet(&d.md_idx[mix(s0, i, N)], oct);
#pragma unroll
        for (int u = 0; u < B; ++u) {
            j[u] = s0 + u < cnt ? (int)(oct[u] & kJMask) : (int)(oct[0] & kJMask);     // past the row: repeat a valid entry
            lo[u] = 0;
        }
        int cj[B];
#pragma unroll
        for (int u = 0; u < B; ++u) { cj[u] = d.md_cnt[j[u]]; hi[u] = ((cj[u] + 7) >> 3) - 1; }
        // first the octet of j's row that holds i (rows ascend; at most 16 octets: four halvings over the octets' first
        // entries), then that octet as one sector: i's slot = 8 * octet + the number of its entries below i
#pragma unroll 1
        for (int it = 0; it < 4; ++it) {
            int v[B];
#pragma unroll
            for (int u = 0; u < B; ++u) v[u] = (int)(d.md_idx[mix(((lo[u] + hi[u] + 1) >> 1) << 3, j[u], N)] & kJMask);
#pragma unroll
            for (int u = 0; u < B; ++u) {
                const int mid = (lo[u] + hi[u] + 1) >> 1;
                if (v[u] <= i) lo[u] = mid; else hi[u] = mid - 1;          // last octet whose first entry is <= i
            }
        }
#pragma unroll
        for (int h = 0; h < B; h += 4) {
            unsigned oc[4][8];
#pragma unroll
            for (int u = 0; u < 4; ++u) ld_octet(&d.md_idx[mix(lo[h + u] << 3, j[h + u], N)], oc[u]);
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                int below = 0;
#pragma unroll
                for (int t = 0; t < 8; ++t)
                    below += ((lo[h + u] << 3) + t < cj[h + u] && (int)(oc[u][t] & kJMask) < i) ? 1 : 0;
                lo[h + u] = (lo[h + u] << 3) + below;
            }
        }
#pragma unroll
        for (int u = 0; u < B; ++u) oct[u] = (unsigned)j[u] | ((unsigned)lo[u] << 24);
        st_octet(&d.md_idx[mix(s0, i, N)], oct);
    }
}

__device__ __forceinline__ void ph_done(const SysDev& d) {
    d.flags[F_REBUILD] = 0;
    d.flags[F_NREBUILD] += 1;
    d.flags[F_BUILT] = 1;
}

__global__ void __launch_bounds__(128) k_build_md(SysDev d, int N, Box b, double rc2, int capMD, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_build_md<true, 1>(d, N, b, rc2, capMD, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}
__global__ void __launch_bounds__(128) k_rev(SysDev d, int N, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_rev(d, N, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

// The whole build in ONE launch for small systems: a cluster of 8 CTAs x 1024 threads, phases separated by
// cluster barriers (hardware barrier across the cluster's SMs, release/acquire at cluster scope).  A step
// without rebuild then costs one early-exit launch instead of ten.
constexpr int kClusterCTAs = 16;               // non-portable cluster size (opt-in attribute, set at the first launch)
constexpr int64_t kClusterBuildMaxAtoms = 16384;
// Up to here the cheap phases (cells, sort, gather) still run as ONE cluster launch and only the Verlet build and the
// reverse slots are separate full-chip kernels: 4 gated launches per step instead of 10.
constexpr int64_t kClusterPreMaxAtoms = 65536;
__device__ __forceinline__ void cluster_barrier() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__global__ void __cluster_dims__(kClusterCTAs, 1, 1) __launch_bounds__(1024, 1)
k_build_cluster(SysDev d, const double* xin, const double* vin, int N, Box b, double rc2,
                int capMD, int first, int n_types, int gated, int upto_gather) {
    if (gated == 2 && blockIdx.x == 0 && threadIdx.x == 0) d.flags[F_STEP] += 1;
    if (gate_closed(d.flags, gated)) return;               // uniform over the cluster: nobody reaches a barrier
    __shared__ int part[1024];
    // warps are dealt round-robin over the CTAs: with tid = blockIdx * 1024 + threadIdx a 4096-atom system would keep
    // 4 of the 16 SMs busy (measured: its Verlet build was bound by the FP64 pipes of those four SMs, 107 of 185 us)
    const int nth = gridDim.x * blockDim.x;
    const int tid = ((threadIdx.x >> 5) * gridDim.x + blockIdx.x) * 32 + (threadIdx.x & 31);
    ph_clear(d, b.ncell, tid, nth);
    cluster_barrier();
    ph_bin(d, xin, N, b, tid, nth);
    cluster_barrier();
    if (blockIdx.x == 0) ph_scan(d, b.ncell, part);
    cluster_barrier();
    ph_fill(d, N, tid, nth);
    cluster_barrier();
    ph_sort_cells(d, b.ncell, tid, nth);
    cluster_barrier();
    ph_gather_a(d, xin, vin, N, first, tid, nth);
    cluster_barrier();
    ph_gather_b(d, N, vin != nullptr, n_types, tid, nth);
    if (upto_gather) return;                               // mid-size systems: the Verlet build runs on the whole chip
    cluster_barrier();
    if (4 * N <= nth) ph_build_md<false, 4>(d, N, b, rc2, capMD, tid, nth);          // as many lanes per atom as the cluster has threads for
    else if (2 * N <= nth) ph_build_md<false, 2>(d, N, b, rc2, capMD, tid, nth);
    else ph_build_md<false, 1>(d, N, b, rc2, capMD, tid, nth);
    cluster_barrier();
    ph_rev(d, N, tid, nth);
    cluster_barrier();
    if (tid == 0) ph_done(d);
}

__global__ void k_build_done(SysDev d, int gated) {
    if (gate_closed(d.flags, gated)) return;
    ph_done(d);
}

// ------------------------------------------------------------------------------------------------
// per-step list filter (the paper's "multiple levels of neighbor list")
// ------------------------------------------------------------------------------------------------
// One thread per sorted atom i walks its Verlet row.  The predicate is the oracle's plain IEEE expression
//   d = (x_j - x_i) - L rint((x_j - x_i)/L);  (dx*dx + dy*dy) + dz*dz < rc*rc     (no FMA contraction)
// so the sets agree bit for bit (reading Q9).  Angular neighbours (r < r_c^A) are packed
// from slot 0 upwards, radial-only ones (r_c^A <= r < r_c^R) from slot capR-1 downwards.  Records,
// the slot masks and the counts go to global memory (k_main and k_assemble read them).  A record is
// {r_ij (fp32 from the fp64 difference), j | rev << 24}; two records of an atom leave as ONE 32-byte store.
struct FilterParams {
    Box b;
    double rcR2, rcA2;
    int capR, capA;
    const double* boxes;        // nullable: concatenated structures (training side), [S][6] = L[3], 1/L[3] of structure sid[i]
    const int* sid;
};

// 4 blocks per SM (128 registers; 5 / 6 blocks per SM spill: 0.62 -> 0.71 / 0.81 ms at 1M atoms)
__global__ void __launch_bounds__(128, 4) k_filter(SysDev d, int N, const __grid_constant__ FilterParams F) {
    const int capR = F.capR;
    const int gi = blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = gi < N;
    const int i = min(gi, N - 1);                // a lane without atom only takes part in the warp statistics
    Box b = F.b;
    if (F.boxes) {                               // every structure of a concatenated set has its own box
        const double* bx = F.boxes + 6 * (size_t)F.sid[i];
#pragma unroll
        for (int a = 0; a < 3; ++a) { b.L[a] = bx[a]; b.invL[a] = bx[3 + a]; }
    }
    const int lane = threadIdx.x & 31;
    const double4 pi = d.xs4[i];
    const int cnt = valid ? d.md_cnt[i] : 0;
    int nA = 0, nO = 0, kA = 0, kO = 0;          // accepted / stored (<= capR in total) angular and radial-only neighbours
    float4 hA = make_float4(0.f, 0.f, 0.f, 0.f), hO = hA;       // the record of a pair that arrived first
    unsigned mR[4] = {0u, 0u, 0u, 0u}, mA[4] = {0u, 0u, 0u, 0u};
    constexpr int B = 8;                 // batch: B list entries, then B position gathers, in flight together
    static_assert(B == 8, "a batch is one octet of the Verlet row");
    unsigned en[B];                      // list entries of the NEXT batch: their load (one sector) overlaps this batch's gathers
#pragma unroll
    for (int u = 0; u < B; ++u) en[u] = (unsigned)i;
    if (cnt > 0) ld_octet(&d.md_idx[mix(0, i, N)], en);
    for (int s0 = 0; s0 < cnt; s0 += B) {
        unsigned eb[B];
        double4 pb[B];
#pragma unroll
        for (int u = 0; u < B; ++u) eb[u] = s0 + u < cnt ? en[u] : (unsigned)i;       // past the row: a harmless gather
#pragma unroll
        for (int u = 0; u < B; ++u) pb[u] = ldg256(&d.xs4[eb[u] & kJMask]);
        if (s0 + B < cnt) ld_octet(&d.md_idx[mix(s0 + B, i, N)], en);
        unsigned bR = 0u, bA = 0u;
#pragma unroll
        for (int u = 0; u < B; ++u) {
            const int s = s0 + u;
            if (s >= cnt) break;
            const unsigned e = eb[u];
            const double4 pj = pb[u];
            const double dx = min_image(pj.x - pi.x, b.L[0], b.invL[0]);
            const double dy = min_image(pj.y - pi.y, b.L[1], b.invL[1]);
            const double dz = min_image(pj.z - pi.z, b.L[2], b.invL[2]);
            const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            if (r2 < F.rcR2) {
                const bool ang = r2 < F.rcA2;
                if (nA + nO < capR) {
                    const float4 rv = make_float4((float)dx, (float)dy, (float)dz, __uint_as_float(e));
                    // angular slots ascend: an even slot waits for its odd partner; radial-only slots descend: an odd
                    // slot waits for the even one below it.  One store site, selects instead of branches.
                    const int slot = ang ? nA : capR - 1 - nO;
                    const bool odd = slot & 1;
                    const bool pair = ang ? odd : (!odd && nO > 0);
                    const float4 lo = ang ? hA : rv, hi = ang ? rv : hO;     // (two store sites instead of the selects: 0.36 -> 0.39 ms)
                    float4* dst = &d.rec[rix(slot & ~1, i, N)];
                    if (pair) stg256(dst, lo, hi);
                    else if (!ang && !odd) *dst = rv;                        // the top slot of an odd capacity has no partner
                    if (ang) { hA = rv; kA = nA + 1; } else { hO = rv; kO = nO + 1; }
                }
                bR |= 1u << u;
                if (ang) bA |= 1u << u;
                if (ang) ++nA; else ++nO;
            }
        }
        // the batch's 8 bits go into byte (s0 >> 3) & 3 of word s0 >> 5
#pragma unroll
        for (int wq = 0; wq < 4; ++wq)
            if ((s0 >> 5) == wq) { mR[wq] |= bR << (s0 & 31); mA[wq] |= bA << (s0 & 31); }
    }
    // records still waiting for a partner leave as single 16-byte stores
    if (kA & 1) d.rec[rix(kA - 1, i, N)] = hA;
    if (kO > 0 && ((capR - kO) & 1)) d.rec[rix(capR - kO, i, N)] = hO;
    const int nR = nA + nO;
    const bool over = nR > capR || nA > F.capA;
    if (valid) {
        d.nnA[i] = over ? 0 : nA;          // an overflowing atom is dropped (and reported), never truncated
        d.nnR[i] = over ? 0 : nR;
        if (over) atomicOr(&d.flags[F_STATUS], ST_OVERFLOW);
        const unsigned mm[8] = {mR[0], mR[1], mR[2], mR[3], mA[0], mA[1], mA[2], mA[3]};
        st_octet(reinterpret_cast<unsigned*>(&d.masks[2 * (size_t)i]), mm);        // both masks: one full sector
    }
    // warp-aggregated statistics
    int xR = nR, xA = nA;
    for (int o = 16; o > 0; o >>= 1) {
        xR = max(xR, __shfl_xor_sync(0xffffffffu, xR, o));
        xA = max(xA, __shfl_xor_sync(0xffffffffu, xA, o));
    }
    if (lane == 0) {
        if (xR > d.flags[F_MAXR]) atomicMax(&d.flags[F_MAXR], xR);
        if (xA > d.flags[F_MAXA]) atomicMax(&d.flags[F_MAXA], xA);
    }
}

// The same filter with eight lanes per atom (small systems): lane l of the group takes Verlet entries l, l + 8, ...;
// the entries of a chunk of eight are judged at once, their record slots follow from the chunk's ballots (order of
// the Verlet row preserved, so rows, masks and counts are bit-identical to k_filter's).  Indices are fetched two
// chunks ahead and positions one chunk ahead: a row of 48 entries costs ~6 short rounds instead of 6 batches in series.
__global__ void __launch_bounds__(128) k_filter_group(SysDev d, int N, const __grid_constant__ FilterParams F) {
    const int capR = F.capR;
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int ia = gt >> 3, gl = threadIdx.x & 7, lane = threadIdx.x & 31, gsh = lane & 24;       // gsh: first lane of the group
    const bool valid = ia < N;
    const int i = valid ? ia : N - 1;
    Box b = F.b;
    if (F.boxes) {
        const double* bx = F.boxes + 6 * (size_t)F.sid[i];
#pragma unroll
        for (int a = 0; a < 3; ++a) { b.L[a] = bx[a]; b.invL[a] = bx[3 + a]; }
    }
    const double4 pi = d.xs4[i];
    const int cnt = valid ? d.md_cnt[i] : 0;
    const int nch = (__reduce_max_sync(0xffffffffu, cnt) + 7) >> 3;       // warp-uniform trip count
    int nA = 0, nO = 0;
    unsigned mR[4] = {0u, 0u, 0u, 0u}, mA[4] = {0u, 0u, 0u, 0u};
    auto entry = [&](int c) { const int s = c * 8 + gl; return s < cnt ? d.md_idx[mix(s, i, N)] : (unsigned)i; };
    unsigned e1 = entry(0), e2 = entry(1);
    double4 p1 = ldg256(&d.xs4[e1 & kJMask]);
    for (int c = 0; c < nch; ++c) {
        const unsigned e = e1;
        const double4 pj = p1;
        e1 = e2; e2 = entry(c + 2);
        p1 = ldg256(&d.xs4[e1 & kJMask]);
        const int s = c * 8 + gl;
        const double dx = min_image(pj.x - pi.x, b.L[0], b.invL[0]);
        const double dy = min_image(pj.y - pi.y, b.L[1], b.invL[1]);
        const double dz = min_image(pj.z - pi.z, b.L[2], b.invL[2]);
        const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        const bool inR = s < cnt && r2 < F.rcR2, inA = inR && r2 < F.rcA2;
        const unsigned bR = (__ballot_sync(0xffffffffu, inR) >> gsh) & 0xffu, bA = (__ballot_sync(0xffffffffu, inA) >> gsh) & 0xffu;
        const unsigned below = (1u << gl) - 1u, bO = bR & ~bA;
        if (inR && nA + nO + __popc(bR & below) < capR) {
            const int slot = inA ? nA + __popc(bA & below) : capR - 1 - (nO + __popc(bO & below));
            d.rec[rix(slot, i, N)] = make_float4((float)dx, (float)dy, (float)dz, __uint_as_float(e));
        }
        nA += __popc(bA); nO += __popc(bO);
#pragma unroll
        for (int wq = 0; wq < 4; ++wq)
            if ((c >> 2) == wq) { mR[wq] |= bR << ((c & 3) * 8); mA[wq] |= bA << ((c & 3) * 8); }
    }
    const int nR = nA + nO;
    const bool over = nR > capR || nA > F.capA;
    if (valid && gl == 0) {
        d.nnA[i] = over ? 0 : nA;
        d.nnR[i] = over ? 0 : nR;
        if (over) atomicOr(&d.flags[F_STATUS], ST_OVERFLOW);
        d.masks[2 * (size_t)i] = make_uint4(mR[0], mR[1], mR[2], mR[3]);
        d.masks[2 * (size_t)i + 1] = make_uint4(mA[0], mA[1], mA[2], mA[3]);
    }
    int xR = nR, xA = nA;
    for (int o = 16; o > 0; o >>= 1) {
        xR = max(xR, __shfl_xor_sync(0xffffffffu, xR, o));
        xA = max(xA, __shfl_xor_sync(0xffffffffu, xA, o));
    }
    if (lane == 0) {
        if (xR > d.flags[F_MAXR]) atomicMax(&d.flags[F_MAXR], xR);
        if (xA > d.flags[F_MAXA]) atomicMax(&d.flags[F_MAXA], xA);
    }
}

// lists in the caller's numbering for nep_get_neighbors
__global__ void k_export_lists(SysDev d, int N, int which, int capR, int cap_out, int* count, int* index) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int nA = d.nnA[i], nR = d.nnR[i];
    const int n = which ? nA : nR;
    const int row = d.perm[i];
    count[row] = n;
    for (int k = 0; k < cap_out; ++k) {
        int v = -1;
        if (k < n) {
            const int slot = k < nA ? k : capR - 1 - (k - nA);
            v = d.perm[__float_as_uint(d.rec[rix(slot, i, N)].w) & kJMask];
        }
        index[(size_t)row * cap_out + k] = v;
    }
}

// partial forces dU_i/dr_ij in the caller's numbering, neighbour order of k_export_lists(which = 0)
__global__ void k_export_p(SysDev d, int N, int capR, float* p_out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int nA = d.nnA[i], nR = d.nnR[i];
    const int row = d.perm[i];
    for (int k = 0; k < capR; ++k) {
        float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
        if (k < nR) v = d.p[(size_t)i * capR + (k < nA ? k : capR - 1 - (k - nA))];
        float* o = p_out + ((size_t)row * capR + k) * 3;
        o[0] = v.x; o[1] = v.y; o[2] = v.z;
    }
}

#include "nep_main.cuh"
#include "nep_desc64.cuh"
#include "nep_gen.cuh"
#include "nep_highl.cuh"
#include "fp32_peak.cuh"

// ------------------------------------------------------------------------------------------------
// assembly (Eq. 4-7) + second half-kick + thermo, and the integrator's first half
// ------------------------------------------------------------------------------------------------
struct AsmParams {
    int N, capR, capMD;
    int md;                       // 0: nep_compute; 1: MD step (kick, J from vs, thermo); 2: F(t0) of nep_md_step
    double half_dt;               // dt/2
    double dt, half_skin2;        // MD step: the NEXT step's half-kick + drift happen here too (not after the call's last step)
    double inv_mass[kMaxTypes];   // 1 / (m * 103.642697)
    double ke_mass[kMaxTypes];    // 0.5 * m * 103.642697
    const double* vel_in;         // nep_compute: caller-order velocities (nullable)
    float* energy; float* force; float* virial; float* heat;   // caller-order outputs (virial/heat nullable)
    double* heat_sum; double* thermo;
    int driven;                   // HNEMD: F_i += F_e . W_i (Eq. 9) in both half-kicks
    float fe[3];                  // F_e, 1/A
    const float* w0;              // [9][N] caller order, nullable: W_i(0) of Eq. 11
    double* kt;                   // [n_steps][3], nullable: K(t) = sum_i W_i(0) . v_i(t)
};

__device__ __forceinline__ int rank_below(const uint4& m, int t) {      // number of set bits at positions < t
    const unsigned w[4] = {m.x, m.y, m.z, m.w};
    int r = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int lo = t - 32 * q;                                      // bits of word q below t
        const unsigned msk = lo >= 32 ? 0xffffffffu : (lo <= 0 ? 0u : ((1u << lo) - 1u));
        r += __popc(w[q] & msk);
    }
    return r;
}
__device__ __forceinline__ bool bit_set(const uint4& m, int t) {
    const unsigned w[4] = {m.x, m.y, m.z, m.w};
    unsigned v = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) if ((t >> 5) == q) v = w[q];
    return (v >> (t & 31)) & 1u;
}

// LANES = 1: one thread per atom (large systems: fewest instructions).  LANES = 8: eight lanes share an atom's
// neighbours (small systems: the three dependent loads of ~28 neighbours become one or two rounds instead of four
// batches in series), partial sums reduced by shuffles, lane 0 of the group finishes the atom.
template <int LANES>
// 4 blocks per SM = at most 128 registers (measured at 1M atoms: 3 / 4 / 5 / 6 blocks per SM -> 0.45 / 0.39 / 0.47 / 0.57 ms)
__global__ void __launch_bounds__(128, 4) k_assemble(SysDev d, AsmParams P) {
    const int N = P.N;
    const int gt = blockIdx.x * blockDim.x + threadIdx.x;
    const int ia = gt / LANES, gl = gt % LANES;
    const bool has_atom = ia < N;
    const int i = has_atom ? ia : N - 1;
    double tU = 0.0, tK = 0.0, tJ[3] = {0.0, 0.0, 0.0}, tKt[3] = {0.0, 0.0, 0.0};
    float fx = 0.f, fy = 0.f, fz = 0.f;
    float w[9] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    const int nR = has_atom ? d.nnR[i] : 0, nA = has_atom ? d.nnA[i] : 0;
    {
        constexpr int B = LANES == 1 ? 8 : 4;    // batch the three dependent loads (record -> masks -> p) for MLP
        for (int k0 = 0; k0 < nR; k0 += B * LANES) {
            unsigned jr[B];
            float4 eb[B], pb[B];
            uint4 mrb[B], mab[B];
#pragma unroll
            for (int u = 0; u < B; ++u) {
                const int k = min(k0 + u * LANES + gl, nR - 1);
                const int slot = k < nA ? k : P.capR - 1 - (k - nA);
                eb[u] = d.rec[rix(slot, i, N)];
                jr[u] = __float_as_uint(eb[u].w);
            }
#pragma unroll
            for (int u = 0; u < B; ++u) ldg256(&d.masks[2 * (size_t)(jr[u] & kJMask)], mrb[u], mab[u]);
#pragma unroll
            for (int u = 0; u < B; ++u) {
                const int rev = (int)(jr[u] >> 24);                   // rev: Verlet slot of i in j's row
                // record slot of i in j's row = rank of Verlet slot rev among j's accepted slots
                const int cs = rank_below(mab[u], rev);
                const int cslot = bit_set(mab[u], rev) ? cs : P.capR - 1 - (rank_below(mrb[u], rev) - cs);
                pb[u] = d.p[(size_t)(jr[u] & kJMask) * P.capR + cslot];      // dU_j/dr_ji
            }
#pragma unroll
            for (int u = 0; u < B; ++u) {
                if (k0 + u * LANES + gl >= nR) continue;
                const float4 e = eb[u], pj = pb[u];
                fx += pj.x; fy += pj.y; fz += pj.z;
                w[0] = fmaf(e.x, pj.x, w[0]); w[1] = fmaf(e.x, pj.y, w[1]); w[2] = fmaf(e.x, pj.z, w[2]);
                w[3] = fmaf(e.y, pj.x, w[3]); w[4] = fmaf(e.y, pj.y, w[4]); w[5] = fmaf(e.y, pj.z, w[5]);
                w[6] = fmaf(e.z, pj.x, w[6]); w[7] = fmaf(e.z, pj.y, w[7]); w[8] = fmaf(e.z, pj.z, w[8]);
            }
        }
    }
    if (LANES > 1) {
#pragma unroll
        for (int o = 1; o < LANES; o <<= 1) {
            fx += __shfl_xor_sync(0xffffffffu, fx, o); fy += __shfl_xor_sync(0xffffffffu, fy, o); fz += __shfl_xor_sync(0xffffffffu, fz, o);
#pragma unroll
            for (int c = 0; c < 9; ++c) w[c] += __shfl_xor_sync(0xffffffffu, w[c], o);
        }
    }
    if (has_atom && gl == 0) {
        const float4 fs = d.Fself[i];
        fx = fs.x - fx; fy = fs.y - fy; fz = fs.z - fz;               // Eq. 4-5
        const int row = d.perm[i];
        const float u = d.Us[i];
        if (!(isfinite(u) && isfinite(fx + fy + fz))) atomicOr(&d.flags[F_STATUS], ST_NAN);      // reported, never silent: NEP_ENAN
        P.energy[row] = u;
        P.force[row] = fx; P.force[N + row] = fy; P.force[2 * N + row] = fz;      // the potential force of Eq. 4
        if (P.driven) {                                                // Eq. 9: (F^ext)^b = sum_a F_e^a W^{ab}
            fx = fmaf(P.fe[0], w[0], fmaf(P.fe[1], w[3], fmaf(P.fe[2], w[6], fx)));
            fy = fmaf(P.fe[0], w[1], fmaf(P.fe[1], w[4], fmaf(P.fe[2], w[7], fy)));
            fz = fmaf(P.fe[0], w[2], fmaf(P.fe[1], w[5], fmaf(P.fe[2], w[8], fz)));
        }
        d.Fs[i] = fx; d.Fs[N + i] = fy; d.Fs[2 * N + i] = fz;         // what the integrator kicks with
        if (P.virial) {
#pragma unroll
            for (int c = 0; c < 9; ++c) P.virial[(size_t)c * N + row] = w[c];
        }
        double vx = 0.0, vy = 0.0, vz = 0.0;
        bool have_v = false;
        if (P.md) {
            const int ty = d.type_s[i];
            const double im = P.md == 1 ? P.inv_mass[ty] * P.half_dt : 0.0;   // md == 2: F(t0) only, no kick
            vx = d.vs[i] + im * (double)fx; vy = d.vs[N + i] + im * (double)fy; vz = d.vs[2 * N + i] + im * (double)fz;
            tK = P.ke_mass[ty] * (vx * vx + vy * vy + vz * vz);
            tU = (double)u;
            have_v = true;
            if (P.md == 1 && d.flags[F_STEP] < d.flags[F_NSTEPS]) {
                // not the call's last step: the next step's first half-kick and drift, while v and F are in registers
                // (nothing in this kernel reads positions; K, J and K(t) below use the velocity at t + dt)
                const double wx = vx + im * (double)fx, wy = vy + im * (double)fy, wz = vz + im * (double)fz;
                const double xn = d.xs[i] + P.dt * wx, yn = d.xs[N + i] + P.dt * wy, zn = d.xs[2 * N + i] + P.dt * wz;
                d.vs[i] = wx; d.vs[N + i] = wy; d.vs[2 * N + i] = wz;
                d.xs[i] = xn; d.xs[N + i] = yn; d.xs[2 * N + i] = zn;
                d.xs4[i] = make_double4(xn, yn, zn, __longlong_as_double((long long)ty));
                const double ax = xn - d.xref[i], ay = yn - d.xref[N + i], az = zn - d.xref[2 * N + i];
                if (ax * ax + ay * ay + az * az > P.half_skin2) d.flags[F_REBUILD] = 1;
            } else { d.vs[i] = vx; d.vs[N + i] = vy; d.vs[2 * N + i] = vz; }
        } else if (P.vel_in) {
            vx = P.vel_in[row]; vy = P.vel_in[N + row]; vz = P.vel_in[2 * N + row];
            have_v = true;
        }
        if (have_v) {                                                // Eq. 7: J^a = sum_b W^{ab} v^b
            const float fvx = (float)vx, fvy = (float)vy, fvz = (float)vz;
            const float jx = w[0] * fvx + w[1] * fvy + w[2] * fvz;
            const float jy = w[3] * fvx + w[4] * fvy + w[5] * fvz;
            const float jz = w[6] * fvx + w[7] * fvy + w[8] * fvz;
            if (P.heat) { P.heat[row] = jx; P.heat[N + row] = jy; P.heat[2 * N + row] = jz; }
            if (P.md == 1 && P.heat_sum) {
                P.heat_sum[row] += (double)jx; P.heat_sum[N + row] += (double)jy; P.heat_sum[2 * N + row] += (double)jz;
            }
            tJ[0] = jx; tJ[1] = jy; tJ[2] = jz;
            if (P.md == 1 && P.kt) {                                   // Eq. 11 with the caller's W_i(0)
#pragma unroll
                for (int a = 0; a < 3; ++a)
                    tKt[a] = (double)P.w0[(size_t)(3 * a) * N + row] * vx + (double)P.w0[(size_t)(3 * a + 1) * N + row] * vy +
                             (double)P.w0[(size_t)(3 * a + 2) * N + row] * vz;
            }
        }
    }
    if (P.md == 1 && (P.thermo || P.kt)) {
        __shared__ double red[8][4];
        double v[8] = {tU, tK, tJ[0], tJ[1], tJ[2], tKt[0], tKt[1], tKt[2]};
#pragma unroll
        for (int c = 0; c < 8; ++c)
            for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
        const int wid = threadIdx.x >> 5;
        if ((threadIdx.x & 31) == 0)
            for (int c = 0; c < 8; ++c) red[c][wid] = v[c];
        __syncthreads();
        if (threadIdx.x < 8) {
            const double t = red[threadIdx.x][0] + red[threadIdx.x][1] + red[threadIdx.x][2] + red[threadIdx.x][3];
            const size_t step = (size_t)(d.flags[F_STEP] - 1);
            if (threadIdx.x < 5) { if (P.thermo) atomicAdd(&P.thermo[step * 5 + threadIdx.x], t); }
            else if (P.kt) atomicAdd(&P.kt[step * 3 + (threadIdx.x - 5)], t);
        }
    }
}

// v += dt/2 F/m;  r += dt v;  raise the rebuild flag when an atom has moved > skin/2 since the build
__global__ void k_kick_drift(SysDev d, int N, double dt, double half_skin2, AsmParams P) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int ty = d.type_s[i];
    const double im = P.inv_mass[ty] * P.half_dt;
    double disp2 = 0.0, xn[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double v = d.vs[a * N + i] + im * (double)d.Fs[a * N + i];
        const double x = d.xs[a * N + i] + dt * v;
        d.vs[a * N + i] = v;
        d.xs[a * N + i] = x;
        xn[a] = x;
        const double dd = x - d.xref[a * N + i];
        disp2 += dd * dd;
    }
    d.xs4[i] = make_double4(xn[0], xn[1], xn[2], __longlong_as_double((long long)ty));
    if (disp2 > half_skin2) d.flags[F_REBUILD] = 1;
}

// caller arrays -> sorted state.  mode 0 (nep_compute): a displacement > skin/2 is an error (stale
// list); mode 1 (nep_md_step): it requests a rebuild.
__global__ void k_load_state(SysDev d, int N, const double* __restrict__ pos, const double* __restrict__ vel,
                             double half_skin2, int mode, int n_steps) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k == 0 && mode == 1) { d.flags[F_STEP] = 0; d.flags[F_NSTEPS] = n_steps; }
    if (k >= N) return;
    const int src = d.perm[k];
    double disp2 = 0.0, xn[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const double x = pos[a * N + src];
        d.xs[a * N + k] = x;
        xn[a] = x;
        const double dd = x - d.xref[a * N + k];
        disp2 += dd * dd;
        if (vel) d.vs[a * N + k] = vel[a * N + src];
    }
    d.xs4[k] = make_double4(xn[0], xn[1], xn[2], __longlong_as_double((long long)d.type_s[k]));
    if (disp2 > half_skin2) {
        if (mode == 0) atomicOr(&d.flags[F_STATUS], ST_STALE); else d.flags[F_REBUILD] = 1;
    }
}

__global__ void k_store_state(SysDev d, int N, double* __restrict__ pos, double* __restrict__ vel) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= N) return;
    const int dst = d.perm[k];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        pos[a * N + dst] = d.xs[a * N + k];
        vel[a * N + dst] = d.vs[a * N + k];
    }
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// host side: C ABI
// ------------------------------------------------------------------------------------------------
namespace {

#define NEP_CUDA_OK(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { set_cuda_error(e_, #expr); return NEP_ECUDA; } } while (0)

thread_local char g_cuda_msg[256] = "CUDA error";
void set_cuda_error(cudaError_t e, const char* what) {
    snprintf(g_cuda_msg, sizeof(g_cuda_msg), "CUDA error: %s (%s)", cudaGetErrorString(e), what);
}

int cap_md_of(const nep_model* m, int capR, double skin) {
    const double f = (m->h.rc_radial + skin) / m->h.rc_radial;
    int c = (int)ceil(capR * f * f * f);
    c = (c + 3) & ~3;
    return c > kMaxCapMD ? kMaxCapMD : c;
}

struct Layout {
    size_t off[32];
    size_t total;
};

// carve the workspace; the same routine sizes it (base == nullptr)
Layout carve(int64_t N, int capR, int capMD, int max_cells, int NA, int D64, SysDev* d, char* base) {
    Layout L; size_t o = 0; int k = 0;
    auto take = [&](size_t bytes) { size_t at = o; o = align256(o + bytes); L.off[k++] = at; return base ? base + at : nullptr; };
    const size_t n = (size_t)N;
    SysDev t;
    t.flags = (int*)take(F_COUNT * sizeof(int));
    t.smslots = (int*)take(256 * sizeof(int));
    t.type_in = (int*)take(n * 4);
    t.perm = (int*)take(n * 4);
    t.perm_tmp = (int*)take(n * 4);
    t.cell_of = (int*)take(n * 4);
    t.cell_cnt = (int*)take(((size_t)max_cells + 1) * 4);
    t.cell_start = (int*)take(((size_t)max_cells + 1) * 4);
    t.cell_fill = (int*)take(((size_t)max_cells + 1) * 4);
    t.type_s = (int*)take(n * 4);
    t.xs = (double*)take(3 * n * 8);
    t.vs = (double*)take(3 * n * 8);
    t.xref = (double*)take(3 * n * 8);
    t.tmp3 = (double*)take(3 * n * 8);
    t.Fs = (float*)take(3 * n * 4);
    t.Us = (float*)take(n * 4);
    t.Fself = (float4*)take(n * 16);
    t.md_cnt = (int*)take(n * 4);
    t.md_idx = (unsigned*)take(n * 32 * (size_t)((capMD + 7) / 8));
    t.capMD = capMD;
    t.nnR = (int*)take(n * 4);
    t.nnA = (int*)take(n * 4);
    t.rec = (float4*)take(n * 32 * (size_t)((capR + 1) / 2));
    t.masks = (uint4*)take(n * 32);
    t.xs4 = (double4*)take(n * 32);
    t.p = (float4*)take(n * 16 * capR);
    t.order = (int2*)take(((n + kWin - 1) / kWin) * kWin * 8);
    t.FpG = (float*)take(((n + kWin - 1) / kWin) * kWin * 4 * (size_t)D64 + 16);
    t.spark0 = (float2*)take(((n + kWin - 1) / kWin) * kWin * 8 * (size_t)(NA * kHalfLM / 2));
    t.spark1 = (float2*)take(((n + kWin - 1) / kWin) * kWin * 8 * (size_t)(NA * kHalfLM / 2));
    L.total = o;
    if (d) *d = t;
    return L;
}

int max_cells_of(int64_t N) { return (int)(2 * N + 64); }

int grid_for(int64_t n, int block) { return (int)((n + block - 1) / block); }
int grid_stride(int64_t n) { int g = grid_for(n, 256); return g > 148 * 8 ? 148 * 8 : (g < 1 ? 1 : g); }

// the neighbour build as a fixed launch sequence; gated != 0: every kernel exits unless F_REBUILD is set
void launch_build(nep_system* s, const double* xin, const double* vin, int first, int gated, cudaStream_t st) {
    const int N = (int)s->N;
    const SysDev& d = s->d;
    const Box& b = s->box;
    const double rc = s->model->h.rc_radial + s->skin;
    if (s->N <= kClusterPreMaxAtoms) {
        static bool np_done[64] = {};
        int dev = 0;
        cudaGetDevice(&dev);
        if (dev < 0 || dev >= 64 || !np_done[dev]) {
            if (cudaFuncSetAttribute(k_build_cluster, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess && dev >= 0 && dev < 64)
                np_done[dev] = true;
        }
        k_build_cluster<<<kClusterCTAs, 1024, 0, st>>>(d, xin, vin, N, b, rc * rc, s->capMD, first, s->model->h.n_types, gated, s->N > kClusterBuildMaxAtoms);
        s->launches += 1;
        if (s->N <= kClusterBuildMaxAtoms) return;
        const int gbm = grid_for(N, 128) > 148 * 16 ? 148 * 16 : grid_for(N, 128);
        k_build_md<<<gbm, 128, 0, st>>>(d, N, b, rc * rc, s->capMD, gated ? 1 : 0);
        k_rev<<<gbm, 128, 0, st>>>(d, N, gated ? 1 : 0);
        k_build_done<<<1, 1, 0, st>>>(d, gated ? 1 : 0);
        s->launches += 3;
        return;
    }
    k_clear_cells<<<grid_stride(b.ncell + 1), 256, 0, st>>>(d, b.ncell, gated);
    k_bin<<<grid_stride(N), 256, 0, st>>>(d, xin, N, b, gated);
    k_scan<<<1, 1024, 0, st>>>(d, b.ncell, gated);
    k_fill<<<grid_stride(N), 256, 0, st>>>(d, N, gated);
    k_sort_cells<<<grid_stride(b.ncell), 256, 0, st>>>(d, b.ncell, gated);
    k_gather_a<<<grid_stride(N), 256, 0, st>>>(d, xin, vin, N, first, gated);
    k_gather_b<<<grid_stride(N), 256, 0, st>>>(d, N, vin != nullptr, s->model->h.n_types, gated);
    const int gb = grid_for(N, 128) > 148 * 16 ? 148 * 16 : grid_for(N, 128);      // grid-stride: a closed gate costs few blocks
    k_build_md<<<gb, 128, 0, st>>>(d, N, b, rc * rc, s->capMD, gated);
    k_rev<<<gb, 128, 0, st>>>(d, N, gated);
    k_build_done<<<1, 1, 0, st>>>(d, gated);
    s->launches += 10;
}

constexpr int kMainSmemLimit = 112 * 1024;          // two blocks of k_main per SM
template <int NA, bool MULTI>
size_t main_smem_bytes(int params_floats) {
    return ((size_t)params_floats + kMainWarps * main_warp_floats<NA, MULTI>() + kMainBarFloats) * sizeof(float);
}

template <int NR, int NA, bool MULTI>
void launch_main_t(nep_system* s, cudaStream_t st) {
    const nep_model* m = s->model;
    MainParams P;
    P.rcR_inv = (float)(1.0 / m->h.rc_radial); P.rcA_inv = (float)(1.0 / m->h.rc_angular);
    P.H = m->H; P.N = (int)s->N; P.capR = s->capR;
    P.q_out = MULTI ? nullptr : s->dump_q; P.fp_out = s->dump_fp;
    const size_t smem = main_smem_bytes<NA, MULTI>(m->params_floats);
    static bool attr_done[64] = {};                // per device: the attribute belongs to the (device, function) pair
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || !attr_done[dev]) {
        cudaError_t e = cudaFuncSetAttribute(k_main<NR, NA, MULTI>, cudaFuncAttributeMaxDynamicSharedMemorySize, kMainSmemLimit);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_main<NR, NA, MULTI>, cudaFuncAttributePreferredSharedMemoryCarveout,
                                                        cudaSharedmemCarveoutMaxShared);
        if (e == cudaSuccess && dev >= 0 && dev < 64) attr_done[dev] = true;      // on failure the launch below reports it
    }
    const int windows = (int)((s->N + kWin - 1) / kWin);
    if (MULTI) {
        Desc64Params p64 = m->p64;
        p64.N = (int)s->N; p64.capR = s->capR; p64.q_out = s->dump_q;
        static bool d64_attr[64] = {};
        if (dev < 0 || dev >= 64 || !d64_attr[dev]) {
            if (cudaFuncSetAttribute(k_desc64<NR, NA>, cudaFuncAttributeMaxDynamicSharedMemorySize, kD64Rows * 6 * 64 * 8) == cudaSuccess &&
                dev >= 0 && dev < 64) d64_attr[dev] = true;
        }
        k_desc64<NR, NA><<<windows * (kWin / 64), 64, kD64Rows * 6 * 64 * 8, st>>>(s->d, s->box, p64, m->params64_dev);
        s->launches += 1;
    }
    k_main<NR, NA, MULTI><<<windows * (kWin / (32 * kMainWarps)), 32 * kMainWarps, smem, st>>>(s->d, P, m->params_dev, m->zz);
    s->launches += 1;
}

bool main_supported(const nep_model* m) {
    // instantiated shapes: the BASELINE.json models (8/8, 9/9 radial functions) and Table I's PbTe model (13/7)
    if (!((m->NR == 8 && m->NA == 8) || (m->NR == 9 && m->NA == 9) || (m->NR == 13 && m->NA == 7)) || m->H > kMaxH || m->h.l_max != 4) return false;
    // the staged weights must fit beside the per-warp record rows (H = 64 with D = 45 and Eq. 19 does not)
    const size_t smem = m->h.n_types > 1 ? main_smem_bytes<8, true>(m->params_floats) : main_smem_bytes<8, false>(m->params_floats);
    return smem <= (size_t)kMainSmemLimit;
}

// dynamic shared memory of k_gen<NMAX, TD> for a model: the per-atom blocks of one CTA plus the staged weights of every layer
template <int NMAX, typename TD>
size_t gen_smem_bytes_t(const nep_model* m) {
    const int Dp = (m->D + 3) & ~3;
    const size_t wbytes = m->nlayers > 1 ? (size_t)m->blob_elems * sizeof(TD)
                                         : ((size_t)m->H * (sizeof(TD) == 8 ? (Dp | 1) : Dp + 4) + 2 * m->H + 1) * sizeof(TD);
    return (size_t)kGenAtomsPerBlock * sizeof(GenSmem<NMAX, TD>) + ((wbytes + 15) & ~(size_t)15);
}

// Does the k_gen instantiation this model runs on fit the opt-in shared memory of the current device?  Every model can
// be put on the group path (small systems, nep_system_set_path, the trainer), so nep_create_ex refuses what does not
// fit instead of handing out a model whose every later launch fails.  l_max > 4 runs on k_highl (no weights in smem).
template <int NMAX, typename TD>
bool gen_fits_t(const nep_model* m, size_t* need, size_t* limit) {
    cudaFuncAttributes fa;
    int dev = 0, optin = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaFuncGetAttributes(&fa, k_gen<NMAX, TD>) != cudaSuccess ||
        cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) { cudaGetLastError(); return false; }
    *need = gen_smem_bytes_t<NMAX, TD>(m) + fa.sharedSizeBytes;
    *limit = (size_t)optin;
    return *need <= *limit;
}
bool gen_fits(const nep_model* m, size_t* need, size_t* limit) {
    *need = 0; *limit = 0;
    if (m->h.l_max > 4) return true;
    const bool multi = m->h.n_types > 1, small = m->NR <= 8 && m->NA <= 8;
    if (small) return multi ? gen_fits_t<8, double>(m, need, limit) : gen_fits_t<8, float>(m, need, limit);
    return multi ? gen_fits_t<16, double>(m, need, limit) : gen_fits_t<16, float>(m, need, limit);
}

template <int NMAX, typename TD>
void launch_gen_t(nep_system* s, cudaStream_t st) {
    const nep_model* m = s->model;
    GenParams P;
    memset(&P, 0, sizeof(P));
    P.rcR = m->h.rc_radial; P.rcA = m->h.rc_angular;
    P.rcR_inv = (float)(1.0 / m->h.rc_radial); P.rcA_inv = (float)(1.0 / m->h.rc_angular);
    for (int k = 0; k < kMaxTypes * kMaxTypes; ++k) { P.zz[k] = m->zz.zz[k]; P.zz64[k] = m->p64.zz[k]; }
    P.NR = m->NR; P.NA = m->NA; P.LMAX = m->h.l_max; P.H = m->H; P.D = m->D; P.Dp = (m->D + 3) & ~3;
    P.N = (int)s->N; P.capR = s->capR; P.box = s->box;
    P.params = m->params_dev; P.params64 = m->params64_dev;
    P.q_out = s->dump_q; P.fp_out = s->dump_fp;
    P.boxes = s->batch_boxes; P.sid = s->batch_sid;
    P.kind = m->kind; P.nlayers = m->nlayers; P.off_out = m->off_out; P.blob_elems = m->blob_elems;
    for (int k = 0; k < 3; ++k) { P.lw[k] = m->lw[k]; P.lin_p[k] = m->lin_p[k]; P.off_w[k] = m->off_w[k]; P.off_b[k] = m->off_b[k]; }
    P.blob = m->blob_dev; P.blob64 = m->blob64_dev;
    const size_t smem = gen_smem_bytes_t<NMAX, TD>(m);             // per-atom blocks + the staged weights (checked in nep_create_ex)
    static size_t attr_smem[64] = {};              // per device: the largest dynamic size this instantiation was opted in for
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= 64 || smem > attr_smem[dev]) {
        cudaError_t e = cudaFuncSetAttribute(k_gen<NMAX, TD>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e == cudaSuccess && dev >= 0 && dev < 64) attr_smem[dev] = smem;          // on failure the launch below reports it
    }
    const int64_t need = (s->N + kGenAtomsPerBlock - 1) / kGenAtomsPerBlock;
    const int64_t cap = 148 * 16;
    k_gen<NMAX, TD><<<(int)(need < cap ? need : cap), 32 * kGenWarps, smem, st>>>(s->d, P);
    s->launches += 1;
}

void launch_highl(nep_system* s, cudaStream_t st) {
    const nep_model* m = s->model;
    HighLParams P;
    memset(&P, 0, sizeof(P));
    P.rcR_inv = (float)(1.0 / m->h.rc_radial); P.rcA_inv = (float)(1.0 / m->h.rc_angular);
    P.NR = m->NR; P.NA = m->NA; P.LMAX = m->h.l_max; P.H = m->H; P.D = m->D; P.Dp = (m->D + 3) & ~3;
    P.N = (int)s->N; P.capR = s->capR;
    P.params = m->params_dev;
    P.q_out = s->dump_q; P.fp_out = s->dump_fp;
    k_highl<<<grid_for(s->N, 64), 64, 0, st>>>(s->d, P);
    s->launches += 1;
}

void launch_gen(nep_system* s, cudaStream_t st) {
    const nep_model* m = s->model;
    if (m->h.l_max > 4) { launch_highl(s, st); return; }           // the harmonics of k_gen / k_main are written out for l <= 4
    const bool multi = m->h.n_types > 1;
    const bool small = m->NR <= 8 && m->NA <= 8;
    if (small) { if (multi) launch_gen_t<8, double>(s, st); else launch_gen_t<8, float>(s, st); }
    else       { if (multi) launch_gen_t<16, double>(s, st); else launch_gen_t<16, float>(s, st); }
}

void launch_main(nep_system* s, cudaStream_t st) {
    const nep_model* m = s->model;
    const bool multi = m->h.n_types > 1;
    if (s->path == NEP_PATH_GROUP) { launch_gen(s, st); return; }
    if (m->NR == 8 && m->NA == 8) { if (multi) launch_main_t<8, 8, true>(s, st); else launch_main_t<8, 8, false>(s, st); }
    else if (m->NR == 9 && m->NA == 9) { if (multi) launch_main_t<9, 9, true>(s, st); else launch_main_t<9, 9, false>(s, st); }
    else if (m->NR == 13 && m->NA == 7) { if (multi) launch_main_t<13, 7, true>(s, st); else launch_main_t<13, 7, false>(s, st); }
}

FilterParams filter_params(const nep_system* s) {
    const nep_hyper& h = s->model->h;
    FilterParams F;
    F.b = s->box;
    F.rcR2 = h.rc_radial * h.rc_radial; F.rcA2 = h.rc_angular * h.rc_angular;
    F.capR = s->capR; F.capA = s->capA;
    F.boxes = s->batch_boxes; F.sid = s->batch_sid;
    return F;
}

void launch_order(nep_system* s, cudaStream_t st) {
    k_order<<<(int)((s->N + kWin - 1) / kWin), kOrderThreads, 0, st>>>(s->d, (int)s->N);
    s->launches += 1;
}

// small systems: the gather kernels spread an atom's neighbours over eight lanes (latency, not throughput, is what
// a 4096-atom step waits for)
constexpr int64_t kGroupGatherMaxAtoms = 16384;
bool group_gather(const nep_system* s) { return s->N <= kGroupGatherMaxAtoms; }

void launch_assemble(nep_system* s, const AsmParams& P, cudaStream_t st) {
    if (group_gather(s)) k_assemble<8><<<grid_for(s->N * 8, 128), 128, 0, st>>>(s->d, P);
    else k_assemble<1><<<grid_for(s->N, 128), 128, 0, st>>>(s->d, P);
    s->launches += 1;
}

void launch_filter(nep_system* s, cudaStream_t st) {
    if (group_gather(s)) k_filter_group<<<grid_for(s->N * 8, 128), 128, 0, st>>>(s->d, (int)s->N, filter_params(s));
    else k_filter<<<grid_for(s->N, 128), 128, 0, st>>>(s->d, (int)s->N, filter_params(s));
    s->launches += 1;
    if (s->path == NEP_PATH_THREAD) launch_order(s, st);         // k_gen takes the atoms in sorted order as they are
}

void fill_masses(AsmParams* P, const nep_model* m, const double* mass_by_type) {
    for (int t = 0; t < kMaxTypes; ++t) {
        const double mm = (mass_by_type && t < m->h.n_types) ? mass_by_type[t] : 1.0;
        P->inv_mass[t] = 1.0 / (mm * kAmuConv);
        P->ke_mass[t] = 0.5 * mm * kAmuConv;
    }
}

// marks the start of a phase on the stream (only when nep_profile is on)
void phase(nep_system* s, int ph, cudaStream_t st) {
    if (!s->prof_on || s->prof_n >= kProfMaxEvents) return;
    cudaEventRecord(s->prof_ev[s->prof_n], st);
    s->prof_phase[s->prof_n++] = ph;
}

void prof_resolve(nep_system* s) {
    for (int k = 0; k + 1 < s->prof_n; ++k) {
        if (s->prof_phase[k] < 0) continue;
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, s->prof_ev[k], s->prof_ev[k + 1]) == cudaSuccess) {
            s->prof_ms[s->prof_phase[k]] += ms;
            s->prof_cnt[s->prof_phase[k]] += 1;
        }
    }
    s->prof_n = 0;
}

bool device_ok() {
    int n = 0;
    return cudaGetDeviceCount(&n) == cudaSuccess && n > 0;
}

// one velocity-Verlet step: half-kick + drift, device-gated rebuild, filter, k_main, assembly + second half-kick
// (the half-kick + drift of every step but the call's first happen inside the previous step's assembly)
void launch_step(nep_system* s, const AsmParams& P, cudaStream_t st) {
    phase(s, PH_BUILD, st);
    launch_build(s, s->d.xs, s->d.vs, 0, 2, st);
    phase(s, PH_FILTER, st);
    launch_filter(s, st);
    phase(s, PH_MAIN, st);
    launch_main(s, st);
    phase(s, PH_ASSEMBLE, st);
    launch_assemble(s, P, st);
}

// The step as a CUDA graph, captured on a library-owned stream (the caller's may be the legacy default
// stream, which cannot capture) and launched into the caller's stream.  Keyed on every argument baked in.
int ensure_step_graph(nep_system* s, const AsmParams& P, double dt_fs, double hs2) {
    static_assert(sizeof(AsmParams) + sizeof(double) <= sizeof(s->g_key), "g_key too small");
    unsigned char key[sizeof(s->g_key)];
    memset(key, 0, sizeof(key));
    memcpy(key, &P, sizeof(P));
    memcpy(key + sizeof(P), &dt_fs, sizeof(double));
    if (s->step_graph && memcmp(key, s->g_key, sizeof(key)) == 0) return NEP_OK;
    if (s->step_graph) { cudaGraphExecDestroy(s->step_graph); s->step_graph = nullptr; }
    if (!s->cap_stream) NEP_CUDA_OK(cudaStreamCreateWithFlags(&s->cap_stream, cudaStreamNonBlocking));
    cudaGraph_t g = nullptr;
    NEP_CUDA_OK(cudaStreamBeginCapture(s->cap_stream, cudaStreamCaptureModeThreadLocal));
    const int64_t l0 = s->launches;
    launch_step(s, P, s->cap_stream);
    s->g_launches = s->launches - l0;
    s->launches = l0;
    NEP_CUDA_OK(cudaStreamEndCapture(s->cap_stream, &g));
    cudaError_t e = cudaGraphInstantiate(&s->step_graph, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { s->step_graph = nullptr; set_cuda_error(e, "cudaGraphInstantiate"); return NEP_ECUDA; }
    memcpy(s->g_key, key, sizeof(key));
    return NEP_OK;
}

}  // namespace

extern "C" {

const char* nep_strerror(int code) {
    switch (code) {
        case NEP_OK: return "ok";
        case NEP_EINVAL: return "invalid argument (hyper-parameters, parameter count, null pointer, or a shape whose staged "
                                "weights exceed the shared memory of the lanes-per-atom kernel: see nep_create_ex in nep_b200.h)";
        case NEP_EBOX: return "box length <= 2 (r_c^R + skin): minimum image ambiguous";
        case NEP_ENOMEM: return "workspace too small";
        case NEP_ECUDA: return g_cuda_msg;
        case NEP_EOVERFLOW: return "neighbour capacity exceeded (cap_radial / cap_angular / Verlet cap)";
        case NEP_ESTALE: return "positions moved more than skin/2 since nep_neighbors";
        case NEP_ESTATE: return "nep_neighbors must be called first";
        case NEP_ENAN: return "a site energy or force is not finite";
        default: return "unknown error";
    }
}

int nep_create(const nep_hyper* hy, const int* atomic_number, const double* params, size_t n_params, nep_model** out) {
    if (!hy) return NEP_EINVAL;
    nep_hyper_ex hx;
    memset(&hx, 0, sizeof(hx));
    hx.base = *hy; hx.n_hidden_layers = 1; hx.angular_kind = NEP_ANGULAR_QNL;
    return nep_create_ex(&hx, atomic_number, params, n_params, out);
}

int nep_create_ex(const nep_hyper_ex* hx, const int* atomic_number, const double* params, size_t n_params, nep_model** out) {
    if (!hx || !params || !out) return NEP_EINVAL;
    const nep_hyper* hy = &hx->base;
    *out = nullptr;
    if (!(hy->rc_radial > 0.0) || !(hy->rc_angular > 0.0) || hy->rc_angular > hy->rc_radial) return NEP_EINVAL;
    if (hy->n_max_radial < 0 || hy->n_max_radial > 15 || hy->n_max_angular < 0 || hy->n_max_angular > 15) return NEP_EINVAL;
    if (hy->l_max < 1 || hy->l_max > kHLMaxL) return NEP_EINVAL;
    if (hy->n_neurons < 1 || hy->n_neurons > kMaxHGen) return NEP_EINVAL;
    if (hy->n_types < 1 || hy->n_types > kMaxTypes) return NEP_EINVAL;
    if (hy->n_types > 1 && !atomic_number) return NEP_EINVAL;
    const int L = hx->n_hidden_layers;
    if (L < 1 || L > 3) return NEP_EINVAL;
    if (L >= 2 && (hx->n_neurons_2 < 1 || hx->n_neurons_2 > kMaxHGen)) return NEP_EINVAL;
    if (L >= 3 && (hx->n_neurons_3 < 1 || hx->n_neurons_3 > kMaxHGen)) return NEP_EINVAL;
    if (hx->angular_kind != NEP_ANGULAR_QNL && hx->angular_kind != NEP_ANGULAR_QNNL) return NEP_EINVAL;
    if (hx->angular_kind == NEP_ANGULAR_QNNL && (hy->n_max_radial > 7 || hy->n_max_angular > 7)) return NEP_EINVAL;
    // l_max = 5..8 (k_highl, the general-l kernel): one species, one hidden layer, the q_nl descriptor
    if (hy->l_max > 4 && (hy->n_types > 1 || L != 1 || hx->angular_kind != NEP_ANGULAR_QNL)) return NEP_EINVAL;
    nep_model* m = new (std::nothrow) nep_model();
    if (!m) return NEP_ENOMEM;
    m->h = *hy;
    m->kind = hx->angular_kind; m->nlayers = L;
    m->blob_dev = nullptr; m->blob64_dev = nullptr; m->params_dev = nullptr; m->params64_dev = nullptr;
    m->NR = hy->n_max_radial + 1; m->NA = hy->n_max_angular + 1; m->H = hy->n_neurons;
    m->D = m->NR + (m->kind == NEP_ANGULAR_QNNL ? m->NA * (m->NA + 1) / 2 : m->NA) * hy->l_max;     // Eq. 16 (pairs n <= n' for Eq. 17)
    m->lw[0] = hy->n_neurons; m->lw[1] = L >= 2 ? hx->n_neurons_2 : 0; m->lw[2] = L >= 3 ? hx->n_neurons_3 : 0;
    {
        int in = m->D, np = 0;
        for (int k = 0; k < L; ++k) { np += (in + 1) * m->lw[k]; in = m->lw[k]; }
        m->npar = np + in + 1;                           // Eq. 26 for L = 1: (D + 2) H + 1
    }
    // staged fp32 layout: w1[H][Dp] (rows zero-padded to a multiple of 4) | b1[H] | w2[H] | b2
    const int H = m->H, D = m->D, Dp = (D + 3) & ~3;
    m->params_floats = (H * Dp + 2 * H + 1 + 3) & ~3;
    if (n_params != (size_t)m->npar) { delete m; return NEP_EINVAL; }
    m->thread_path_ok = L == 1 && m->kind == NEP_ANGULAR_QNL && main_supported(m);
    if (!device_ok()) { delete m; set_cuda_error(cudaErrorNoDevice, "nep_create"); return NEP_ECUDA; }
    for (int t = 0; t < kMaxTypes; ++t) m->Z[t] = (hy->n_types > 1 && t < hy->n_types) ? atomic_number[t] : 1;
    for (int a = 0; a < kMaxTypes; ++a)
        for (int b = 0; b < kMaxTypes; ++b) m->zz.zz[a * kMaxTypes + b] = (float)sqrt((double)m->Z[a] * (double)m->Z[b]);   // Eq. 19
    m->p64.rcR = hy->rc_radial; m->p64.rcA = hy->rc_angular; m->p64.H = H;
    for (int a = 0; a < kMaxTypes; ++a)
        for (int b = 0; b < kMaxTypes; ++b) m->p64.zz[a * kMaxTypes + b] = sqrt((double)m->Z[a] * (double)m->Z[b]);   // Eq. 19
    cudaError_t e = cudaSuccess;
    if (L == 1) {
        float* stage = new float[(size_t)m->params_floats]();
        for (int mu = 0; mu < H; ++mu)
            for (int v = 0; v < D; ++v) stage[mu * Dp + v] = (float)params[(size_t)mu * D + v];
        for (int k = 0; k < 2 * H + 1; ++k) stage[H * Dp + k] = (float)params[(size_t)H * D + k];
        e = cudaMalloc(&m->params_dev, (size_t)m->params_floats * sizeof(float));
        if (e == cudaSuccess) e = cudaMemcpy(m->params_dev, stage, (size_t)m->params_floats * sizeof(float), cudaMemcpyHostToDevice);
        delete[] stage;
        if (e == cudaSuccess && hy->n_types > 1) {
            e = cudaMalloc(&m->params64_dev, (size_t)m->npar * sizeof(double));
            if (e == cudaSuccess) e = cudaMemcpy(m->params64_dev, params, (size_t)m->npar * sizeof(double), cudaMemcpyHostToDevice);
        }
    } else {
        // deep network: one padded blob  W1[H1][in_p] | b1 | W2[H2][H1_p] | b2 | ... | w_out | b_out  (sections 4-aligned)
        int off = 0, in = D;
        for (int k = 0; k < L; ++k) {
            m->lin_p[k] = (in + 3) & ~3;
            m->off_w[k] = off; off += m->lw[k] * m->lin_p[k];
            m->off_b[k] = off; off += (m->lw[k] + 3) & ~3;
            in = m->lw[k];
        }
        m->off_out = off; off += (in + 1 + 3) & ~3;
        m->blob_elems = off;
        double* blob = new double[(size_t)off]();
        const double* p = params;
        in = D;
        for (int k = 0; k < L; ++k) {
            for (int mu = 0; mu < m->lw[k]; ++mu)
                for (int v = 0; v < in; ++v) blob[m->off_w[k] + mu * m->lin_p[k] + v] = p[(size_t)mu * in + v];
            p += (size_t)m->lw[k] * in;
            for (int mu = 0; mu < m->lw[k]; ++mu) blob[m->off_b[k] + mu] = p[mu];
            p += m->lw[k];
            in = m->lw[k];
        }
        for (int mu = 0; mu <= in; ++mu) blob[m->off_out + mu] = p[mu];
        if (hy->n_types > 1) {
            e = cudaMalloc(&m->blob64_dev, (size_t)off * sizeof(double));
            if (e == cudaSuccess) e = cudaMemcpy(m->blob64_dev, blob, (size_t)off * sizeof(double), cudaMemcpyHostToDevice);
        } else {
            float* bf = new float[(size_t)off];
            for (int k = 0; k < off; ++k) bf[k] = (float)blob[k];
            e = cudaMalloc(&m->blob_dev, (size_t)off * sizeof(float));
            if (e == cudaSuccess) e = cudaMemcpy(m->blob_dev, bf, (size_t)off * sizeof(float), cudaMemcpyHostToDevice);
            delete[] bf;
        }
        delete[] blob;
    }
    if (e != cudaSuccess) { set_cuda_error(e, "nep_create"); nep_destroy(m); return NEP_ECUDA; }
    {
        size_t need = 0, limit = 0;
        if (!gen_fits(m, &need, &limit)) {
            nep_destroy(m);
            return NEP_EINVAL;
        }
    }
    *out = m;
    return NEP_OK;
}

int nep_descriptor_dim(const nep_model* m) { return m ? m->D : NEP_EINVAL; }
int nep_num_params(const nep_model* m) { return m ? m->npar : NEP_EINVAL; }

void nep_destroy(nep_model* m) {
    if (!m) return;
    if (m->params_dev) cudaFree(m->params_dev);
    if (m->params64_dev) cudaFree(m->params64_dev);
    if (m->blob_dev) cudaFree(m->blob_dev);
    if (m->blob64_dev) cudaFree(m->blob64_dev);
    delete m;
}

size_t nep_workspace_bytes(const nep_model* m, int64_t n_atoms, int cap_radial, int cap_angular, double skin) {
    if (!m || n_atoms < 1 || n_atoms >= (1 << 24) || cap_radial < 1 || cap_radial > kMaxCapMD || cap_angular < 1 ||
        cap_angular > cap_radial || !(skin >= 0.0))
        return 0;
    return carve(n_atoms, cap_radial, cap_md_of(m, cap_radial, skin), max_cells_of(n_atoms), m->NA, m->h.n_types > 1 ? m->D : 0, nullptr, nullptr).total;
}

int nep_system_create(const nep_model* m, int64_t n_atoms, const int* type_dev, int cap_radial, int cap_angular,
                      double skin, void* workspace_dev, size_t workspace_bytes, nep_system** out) {
    if (!out) return NEP_EINVAL;
    *out = nullptr;
    const size_t need = nep_workspace_bytes(m, n_atoms, cap_radial, cap_angular, skin);
    if (need == 0 || !type_dev || !workspace_dev || ((uintptr_t)workspace_dev & 255)) return NEP_EINVAL;
    if (workspace_bytes < need) return NEP_ENOMEM;
    nep_system* s = new (std::nothrow) nep_system();
    if (!s) return NEP_ENOMEM;
    s->model = m; s->N = n_atoms; s->capR = cap_radial; s->capA = cap_angular; s->skin = skin;
    s->capMD = cap_md_of(m, cap_radial, skin);
    s->max_cells = max_cells_of(n_atoms);
    // one thread per atom pays once the machine is full; below that (and for every shape k_main is not
    // instantiated for) 16 lanes share an atom (k_gen)
    s->path = (m->thread_path_ok && n_atoms >= kThreadPathMinAtoms) ? NEP_PATH_THREAD : NEP_PATH_GROUP;
    carve(n_atoms, s->capR, s->capMD, s->max_cells, m->NA, m->h.n_types > 1 ? m->D : 0, &s->d, (char*)workspace_dev);
    s->last_driven = false; s->last_fe[0] = s->last_fe[1] = s->last_fe[2] = 0.f;
    s->batch_boxes = nullptr; s->batch_sid = nullptr;
    s->built = false; s->have_forces = false; s->dump_q = nullptr; s->dump_fp = nullptr; s->last_stream = nullptr; s->step_graph = nullptr; s->cap_stream = nullptr; s->g_launches = 0;
    s->launches = 0; s->prof_on = false; s->prof_n = 0;
    for (int k = 0; k < NEP_PHASES; ++k) { s->prof_ms[k] = 0.0; s->prof_cnt[k] = 0; }
    for (int k = 0; k < kProfMaxEvents; ++k) s->prof_ev[k] = nullptr;
    // Set-up call: the whole device is synchronised on both sides of the clear and the copy.  They are issued on the
    // legacy default stream, which orders itself against blocking streams only; a cudaStreamNonBlocking stream (any
    // PyTorch side stream) that produced type_dev, or that runs nep_neighbors next, would otherwise overlap them.
    cudaError_t e = cudaDeviceSynchronize();
    if (e == cudaSuccess) e = cudaMemset(workspace_dev, 0, need);
    if (e == cudaSuccess) e = cudaMemcpy(s->d.type_in, type_dev, (size_t)n_atoms * sizeof(int), cudaMemcpyDeviceToDevice);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) { set_cuda_error(e, "nep_system_create"); delete s; return NEP_ECUDA; }
    *out = s;
    return NEP_OK;
}

void nep_system_destroy(nep_system* s) {
    if (!s) return;
    if (s->step_graph) cudaGraphExecDestroy(s->step_graph);
    if (s->cap_stream) cudaStreamDestroy(s->cap_stream);
    for (int k = 0; k < kProfMaxEvents; ++k) if (s->prof_ev[k]) cudaEventDestroy(s->prof_ev[k]);
    delete s;
}

int nep_system_set_path(nep_system* s, int path) {
    if (!s || (path != NEP_PATH_AUTO && path != NEP_PATH_THREAD && path != NEP_PATH_GROUP)) return NEP_EINVAL;
    if (path == NEP_PATH_THREAD && !s->model->thread_path_ok) return NEP_EINVAL;
    if (path == NEP_PATH_AUTO)
        path = (s->model->thread_path_ok && s->N >= kThreadPathMinAtoms) ? NEP_PATH_THREAD : NEP_PATH_GROUP;
    if (path != s->path) {
        s->path = path;
        s->built = false; s->have_forces = false;                      // k_order's output belongs to the thread path
        if (s->step_graph) { cudaGraphExecDestroy(s->step_graph); s->step_graph = nullptr; }
    }
    return NEP_OK;
}

int nep_system_path(const nep_system* s) { return s ? s->path : NEP_EINVAL; }

int nep_neighbors(nep_system* s, const double* pos_dev, const double box[3], void* cuda_stream) {
    if (!s || !pos_dev || !box) return NEP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const double rc = s->model->h.rc_radial + s->skin;
    Box b;
    for (int a = 0; a < 3; ++a) {
        if (!(box[a] > 2.0 * rc)) return NEP_EBOX;
        b.L[a] = box[a]; b.invL[a] = 1.0 / box[a];
        int nc = (int)floor(box[a] / rc);
        b.nc[a] = nc < 3 ? 1 : nc;
    }
    while ((int64_t)b.nc[0] * b.nc[1] * b.nc[2] > s->max_cells) {     // sparse systems: coarser cells
        int a = b.nc[0] >= b.nc[1] ? (b.nc[0] >= b.nc[2] ? 0 : 2) : (b.nc[1] >= b.nc[2] ? 1 : 2);
        b.nc[a] = b.nc[a] > 3 ? b.nc[a] - 1 : 1;
    }
    b.ncell = b.nc[0] * b.nc[1] * b.nc[2];
    s->box = b;
    s->last_stream = st;
    if (s->step_graph) { cudaGraphExecDestroy(s->step_graph); s->step_graph = nullptr; }   // the box is baked into it
    phase(s, PH_BUILD, st);
    launch_build(s, pos_dev, nullptr, 1, 0, st);
    phase(s, PH_FILTER, st);
    launch_filter(s, st);
    phase(s, -1, st);
    NEP_CUDA_OK(cudaGetLastError());
    s->built = true; s->have_forces = false;
    return NEP_OK;
}

int nep_get_neighbors(nep_system* s, int which, int* count_dev, int* index_dev, void* cuda_stream) {
    if (!s || !count_dev || !index_dev || (which != 0 && which != 1)) return NEP_EINVAL;
    if (!s->built) return NEP_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->last_stream = st;
    k_export_lists<<<grid_for(s->N, 128), 128, 0, st>>>(s->d, (int)s->N, which, s->capR, which ? s->capA : s->capR,
                                                       count_dev, index_dev);
    s->launches += 1;
    NEP_CUDA_OK(cudaGetLastError());
    return NEP_OK;
}

int nep_compute(nep_system* s, const double* pos_dev, const double* vel_dev, float* energy_dev, float* force_dev,
                float* virial_dev, float* heat_dev, void* cuda_stream) {
    if (!s || !pos_dev || !energy_dev || !force_dev) return NEP_EINVAL;
    if (!s->built) return NEP_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->last_stream = st;
    const int N = (int)s->N;
    const double hs = 0.5 * s->skin;
    phase(s, PH_STATE, st);
    k_load_state<<<grid_for(N, 256), 256, 0, st>>>(s->d, N, pos_dev, nullptr, hs * hs * (1.0 + 1e-12) + 1e-24, 0, 0);
    phase(s, PH_FILTER, st);
    launch_filter(s, st);
    phase(s, PH_MAIN, st);
    launch_main(s, st);
    AsmParams P;
    memset(&P, 0, sizeof(P));
    P.N = N; P.capR = s->capR; P.capMD = s->capMD; P.md = 0;
    fill_masses(&P, s->model, nullptr);
    P.vel_in = vel_dev; P.energy = energy_dev; P.force = force_dev; P.virial = virial_dev;
    P.heat = vel_dev ? heat_dev : nullptr;
    phase(s, PH_ASSEMBLE, st);
    launch_assemble(s, P, st);
    phase(s, -1, st);
    s->launches += 1;
    NEP_CUDA_OK(cudaGetLastError());
    s->have_forces = false;
    return NEP_OK;
}

int nep_compute_internals(nep_system* s, const double* pos_dev, float* q_dev, float* fp_dev, float* p_dev, void* cuda_stream) {
    if (!s || !pos_dev) return NEP_EINVAL;
    if (!s->built) return NEP_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->last_stream = st;
    const int N = (int)s->N;
    const double hs = 0.5 * s->skin;
    k_load_state<<<grid_for(N, 256), 256, 0, st>>>(s->d, N, pos_dev, nullptr, hs * hs * (1.0 + 1e-12) + 1e-24, 0, 0);
    launch_filter(s, st);
    s->dump_q = q_dev; s->dump_fp = fp_dev;
    launch_main(s, st);
    s->dump_q = nullptr; s->dump_fp = nullptr;
    if (p_dev) { k_export_p<<<grid_for(N, 128), 128, 0, st>>>(s->d, N, s->capR, p_dev); s->launches += 1; }
    s->launches += 1;
    NEP_CUDA_OK(cudaGetLastError());
    s->have_forces = false;
    return NEP_OK;
}

int nep_md_step(nep_system* s, double* pos_dev, double* vel_dev, const double* mass_by_type, double dt_fs, int n_steps,
                float* energy_dev, float* force_dev, float* virial_dev, float* heat_dev, double* heat_sum_dev,
                double* thermo_dev, void* cuda_stream) {
    return nep_md_step_driven(s, pos_dev, vel_dev, mass_by_type, dt_fs, n_steps, nullptr, energy_dev, force_dev, virial_dev,
                              heat_dev, heat_sum_dev, thermo_dev, nullptr, nullptr, cuda_stream);
}

int nep_md_step_driven(nep_system* s, double* pos_dev, double* vel_dev, const double* mass_by_type, double dt_fs, int n_steps,
                       const double* driving_force, float* energy_dev, float* force_dev, float* virial_dev, float* heat_dev,
                       double* heat_sum_dev, double* thermo_dev, const float* w0_dev, double* kt_dev, void* cuda_stream) {
    if (!s || !pos_dev || !vel_dev || !mass_by_type || !energy_dev || !force_dev || n_steps < 0 || !(dt_fs > 0.0))
        return NEP_EINVAL;
    if (kt_dev && !w0_dev) return NEP_EINVAL;
    if (!s->built) return NEP_ESTATE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    s->last_stream = st;
    const int N = (int)s->N;
    const double hs = 0.5 * s->skin;
    const double hs2 = hs * hs;
    AsmParams P;
    memset(&P, 0, sizeof(P));
    P.N = N; P.capR = s->capR; P.capMD = s->capMD;
    P.half_dt = 0.5 * dt_fs; P.dt = dt_fs; P.half_skin2 = hs2;
    fill_masses(&P, s->model, mass_by_type);
    P.energy = energy_dev; P.force = force_dev; P.virial = virial_dev; P.heat = heat_dev;
    P.heat_sum = heat_sum_dev; P.thermo = thermo_dev;
    if (driving_force) {
        P.driven = 1;
        for (int a = 0; a < 3; ++a) P.fe[a] = (float)driving_force[a];
        if (!s->have_forces || !s->last_driven || memcmp(s->last_fe, P.fe, sizeof(P.fe)) != 0) s->have_forces = false;
    } else if (s->last_driven) s->have_forces = false;        // the stored kick force must match this call's equations of motion
    s->last_driven = driving_force != nullptr;
    memcpy(s->last_fe, P.fe, sizeof(P.fe));
    P.w0 = kt_dev ? w0_dev : nullptr; P.kt = kt_dev;
    if (thermo_dev && n_steps > 0) NEP_CUDA_OK(cudaMemsetAsync(thermo_dev, 0, (size_t)n_steps * 5 * sizeof(double), st));
    if (kt_dev && n_steps > 0) NEP_CUDA_OK(cudaMemsetAsync(kt_dev, 0, (size_t)n_steps * 3 * sizeof(double), st));
    // caller arrays -> sorted state
    phase(s, PH_STATE, st);
    k_load_state<<<grid_for(N, 256), 256, 0, st>>>(s->d, N, pos_dev, vel_dev, hs2, 1, n_steps);
    s->launches += 1;
    if (!s->have_forces) {       // F(t0); a call that directly follows nep_md_step continues from its forces
        phase(s, PH_BUILD, st);
        launch_build(s, s->d.xs, s->d.vs, 0, 1, st);
        phase(s, PH_FILTER, st);
        launch_filter(s, st);
        phase(s, PH_MAIN, st);
        launch_main(s, st);
        P.md = 2;
        phase(s, PH_ASSEMBLE, st);
        launch_assemble(s, P, st);
    }
    P.md = 1;
    if (n_steps > 0) {           // the first step's half-kick + drift; the later ones are fused into the assembly before them
        phase(s, PH_KICK, st);
        k_kick_drift<<<grid_for(N, 256), 256, 0, st>>>(s->d, N, dt_fs, hs2, P);
        s->launches += 1;
    }
    if (s->prof_on || n_steps < 2) {
        for (int step = 0; step < n_steps; ++step) launch_step(s, P, st);
    } else {
        // the step's launch sequence is fixed (rebuilds are device-gated): capture it once, replay it
        const int rc = ensure_step_graph(s, P, dt_fs, hs2);
        if (rc != NEP_OK) return rc;
        for (int step = 0; step < n_steps; ++step) NEP_CUDA_OK(cudaGraphLaunch(s->step_graph, st));
        s->launches += s->g_launches * n_steps;
    }
    phase(s, PH_STATE, st);
    k_store_state<<<grid_for(N, 256), 256, 0, st>>>(s->d, N, pos_dev, vel_dev);
    phase(s, -1, st);
    s->launches += 1;
    NEP_CUDA_OK(cudaGetLastError());
    s->have_forces = true;
    return NEP_OK;
}

int nep_status(nep_system* s) {
    if (!s) return NEP_EINVAL;
    NEP_CUDA_OK(cudaStreamSynchronize(s->last_stream));
    int flags[F_COUNT];
    NEP_CUDA_OK(cudaMemcpy(flags, s->d.flags, sizeof(flags), cudaMemcpyDeviceToHost));
    s->host_stats[0] = flags[F_NREBUILD]; s->host_stats[1] = flags[F_MAXR];
    s->host_stats[2] = flags[F_MAXA]; s->host_stats[3] = flags[F_MAXMD];
    if (flags[F_STATUS]) NEP_CUDA_OK(cudaMemset(s->d.flags + F_STATUS, 0, sizeof(int)));
    if (flags[F_STATUS] & ST_BADTYPE) return NEP_EINVAL;
    if (flags[F_STATUS] & ST_OVERFLOW) return NEP_EOVERFLOW;
    if (flags[F_STATUS] & ST_STALE) return NEP_ESTALE;
    if (flags[F_STATUS] & ST_NAN) return NEP_ENAN;
    return NEP_OK;
}

int nep_stats(nep_system* s, int64_t out[4]) {
    if (!s || !out) return NEP_EINVAL;
    NEP_CUDA_OK(cudaStreamSynchronize(s->last_stream));
    int flags[F_COUNT];
    NEP_CUDA_OK(cudaMemcpy(flags, s->d.flags, sizeof(flags), cudaMemcpyDeviceToHost));
    out[0] = flags[F_NREBUILD]; out[1] = flags[F_MAXR]; out[2] = flags[F_MAXA]; out[3] = flags[F_MAXMD];
    return NEP_OK;
}

int64_t nep_launch_count(const nep_system* s) { return s ? s->launches : 0; }

int nep_measure_fp32_peak(double* tflops_ffma, double* tflops_ffma2, void* cuda_stream) {
    if (!tflops_ffma || !tflops_ffma2) return NEP_EINVAL;
    if (!device_ok()) { set_cuda_error(cudaErrorNoDevice, "nep_measure_fp32_peak"); return NEP_ECUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    { int dev_ = 0; NEP_CUDA_OK(cudaGetDevice(&dev_)); NEP_CUDA_OK(cudaGetDeviceProperties(&prop, dev_)); }
    float* out = nullptr;
    NEP_CUDA_OK(cudaMalloc(&out, 16));
    cudaEvent_t e0, e1;
    NEP_CUDA_OK(cudaEventCreate(&e0)); NEP_CUDA_OK(cudaEventCreate(&e1));
    const int blocks = prop.multiProcessorCount * 8, iters = 1 << 15;
    double* res[2] = {tflops_ffma, tflops_ffma2};
    for (int v = 0; v < 2; ++v) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            NEP_CUDA_OK(cudaEventRecord(e0, st));
            if (v == 0) k_fma_chain<false><<<blocks, 256, 0, st>>>(out, iters, 0.999f, 0.001f);
            else k_fma_chain<true><<<blocks, 256, 0, st>>>(out, iters, 0.999f, 0.001f);
            NEP_CUDA_OK(cudaEventRecord(e1, st));
            NEP_CUDA_OK(cudaEventSynchronize(e1));
            float ms = 0.f;
            NEP_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0 && ms < best) best = ms;
        }
        *res[v] = 2.0 * 16.0 * iters * 256.0 * blocks / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    return NEP_OK;
}

int nep_measure_fp32_patterns(double tflops[3], void* cuda_stream) {
    if (!tflops) return NEP_EINVAL;
    if (!device_ok()) { set_cuda_error(cudaErrorNoDevice, "nep_measure_fp32_patterns"); return NEP_ECUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaDeviceProp prop;
    { int dev_ = 0; NEP_CUDA_OK(cudaGetDevice(&dev_)); NEP_CUDA_OK(cudaGetDeviceProperties(&prop, dev_)); }
    float* out = nullptr;
    NEP_CUDA_OK(cudaMalloc(&out, 16));
    cudaEvent_t e0, e1;
    NEP_CUDA_OK(cudaEventCreate(&e0)); NEP_CUDA_OK(cudaEventCreate(&e1));
    const int blocks = prop.multiProcessorCount * 4, iters = 1 << 13;        // k_main's residency: 4 x 64 threads per SM
    const double fma_per_iter[3] = {16.0, 96.0, 192.0};
    for (int v = 0; v < 3; ++v) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {
            NEP_CUDA_OK(cudaEventRecord(e0, st));
            if (v == 0) k_fma_pattern<0><<<blocks, 64, 0, st>>>(out, iters * 8, 0.999f, 0.001f);
            else if (v == 1) k_fma_pattern<1><<<blocks, 64, 0, st>>>(out, iters, 0.999f, 0.001f);
            else k_fma_pattern<2><<<blocks, 64, 0, st>>>(out, iters, 0.999f, 0.001f);
            NEP_CUDA_OK(cudaEventRecord(e1, st));
            NEP_CUDA_OK(cudaEventSynchronize(e1));
            float ms = 0.f;
            NEP_CUDA_OK(cudaEventElapsedTime(&ms, e0, e1));
            if (rep > 0 && ms < best) best = ms;
        }
        tflops[v] = 2.0 * fma_per_iter[v] * iters * (v == 0 ? 8 : 1) * 64.0 * blocks / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(out);
    return NEP_OK;
}

int nep_profile(nep_system* s, int enable) {
    if (!s) return NEP_EINVAL;
    NEP_CUDA_OK(cudaStreamSynchronize(s->last_stream));
    s->prof_n = 0;
    for (int k = 0; k < NEP_PHASES; ++k) { s->prof_ms[k] = 0.0; s->prof_cnt[k] = 0; }
    if (enable)
        for (int k = 0; k < kProfMaxEvents; ++k)
            if (!s->prof_ev[k]) NEP_CUDA_OK(cudaEventCreate(&s->prof_ev[k]));
    s->prof_on = enable != 0;
    return NEP_OK;
}

int nep_get_profile(nep_system* s, double ms[8], int64_t count[8]) {
    if (!s || !ms || !count) return NEP_EINVAL;
    NEP_CUDA_OK(cudaStreamSynchronize(s->last_stream));
    prof_resolve(s);
    for (int k = 0; k < NEP_PHASES; ++k) { ms[k] = s->prof_ms[k]; count[k] = s->prof_cnt[k]; }
    return NEP_OK;
}

}  // extern "C"

#include "nep_train.cuh"
