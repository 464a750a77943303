/*
 * nep_noalloc.cu -- nep_loss_noalloc: the loss terms of Eq. 29-34 from predictions that are already
 * on the device, for callers that are not in a position to allocate device memory.
 *
 * Who that is.  Every other compute call of this library works in a workspace the caller allocates
 * (nep_workspace_bytes / nep_trainer_workspace_bytes).  That presumes the caller owns an allocator.  Some do not:
 *   - a force or loss callback that another program (an MD engine, an optimiser loop) invokes with nothing but the
 *     device arrays of this step -- it has no place to keep a workspace between invocations and may be called at a
 *     point where cudaMalloc is off limits (cudaMalloc synchronises the whole device and is refused while a stream
 *     of the process is being captured);
 *   - a process whose device memory has been handed over entirely to one pool (PyTorch's caching allocator, a job
 *     scheduler's arena): a raw cudaMalloc there either fails or takes memory away from the pool behind its back;
 *   - code on a latency budget (a control loop, an in-situ analysis hook) that may not take the milliseconds and the
 *     device-wide synchronisation an allocation can cost.
 * For them this file holds its scratch in the library image itself: g_loss_scratch below, a file-scope __device__
 * array of kScratchBytes = 524,544 bytes (0.5 MiB + 256 B).  Every GPU on which the library gets loaded carries that
 * array from the moment its code is loaded on the device until the process exits, whether or not this entry point
 * is ever called: that is the price, and the reason the size is modest and fixed.
 *
 * What follows from one shared, fixed array:
 *   - a problem that needs more partial rows than the array has is REJECTED (NEP_ENOMEM plus a message), never
 *     truncated: the limit is 3 n_atoms + 7 n_structures + n_par <= 16,777,216 (about 5.5 million atoms);
 *   - the array keeps whatever the previous call left.  The only part that has to start at zero is the ticket
 *     counter in its first 256 bytes; every call clears it on its own stream before the kernel.  The partial rows
 *     are fully overwritten before they are read;
 *   - two calls that can overlap on the GPU (different streams without an event between them, or two host threads
 *     on two streams) use the same rows and the same ticket and RACE.  Serialise them: one stream, or an event;
 *   - the first call on each device looks up the array's device address (cudaGetSymbolAddress, which may also make
 *     the CUDA runtime load this library's device code on that GPU).  Make that first call during start-up, outside
 *     any stream capture, with the device you mean to use current.  Later calls on that device do no set-up.
 *
 * This file is self-contained: it shares no kernel with nep_b200.cu and changes nothing there.  The existing path
 * for the same numbers is nep_trainer_predict -> nep_trainer_losses (k_train_reduce + k_train_loss, whose
 * squared-error accumulators sit in the trainer's caller-allocated workspace).
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include <mutex>

#include "../../include/nep_b200.h"

namespace {

constexpr int kLossThreads = 256;
constexpr int kLossPerThread = 8;
constexpr int kLossChunk = kLossThreads * kLossPerThread;      // elements of the concatenated index space per block
constexpr int kRowDoubles = 8;                                 // one partial row: 5 sums, padded to 64 bytes
constexpr int kHeaderDoubles = 32;                             // 256 bytes: the ticket counter lives in the first 4
constexpr int kMaxRows = 8192;                                 // blocks one call may use
constexpr size_t kScratchDoubles = (size_t)kHeaderDoubles + (size_t)kMaxRows * kRowDoubles;
constexpr size_t kScratchBytes = kScratchDoubles * sizeof(double);   // 524,544 bytes
constexpr int64_t kMaxElements = (int64_t)kMaxRows * kLossChunk;     // 16,777,216

// The scratch.  In HOST code this name is only a handle for the runtime (cudaGetSymbolAddress below), not an address a
// kernel could use; kernels get the device address as an argument.
static __device__ __align__(256) double g_loss_scratch[kScratchDoubles];

// sums over the concatenated index space  [ 3N force components | S energies | 6S virial components | n_par weights ]
//   acc 0: (e - e_tar)^2   1: (f - f_tar)^2   2: (v - v_tar)^2   3: |z|   4: z^2
// Each block owns one fixed chunk, writes its five sums to its row, takes a ticket; the block that draws the last
// ticket adds the rows in a fixed order and writes the six losses.
__global__ void __launch_bounds__(kLossThreads)
k_loss_static(double* __restrict__ scratch, int64_t N, int64_t S, int64_t npar,
              const float* __restrict__ e, const float* __restrict__ f, const float* __restrict__ v,
              const float* __restrict__ e_tar, const float* __restrict__ f_tar, const float* __restrict__ v_tar,
              const double* __restrict__ z, double le, double lf, double lv, double l1w, double l2w, double* __restrict__ out) {
    const int64_t nF = 3 * N, nE = S, nV = 6 * S;
    const int64_t total = nF + nE + nV + npar;
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    const int64_t base = (int64_t)blockIdx.x * kLossChunk;
#pragma unroll
    for (int k = 0; k < kLossPerThread; ++k) {
        int64_t i = base + (int64_t)k * kLossThreads + threadIdx.x;
        if (i >= total) break;
        if (i < nF) { const double d = (double)f[i] - (double)f_tar[i]; acc[1] += d * d; continue; }
        i -= nF;
        if (i < nE) { const double d = (double)e[i] - (double)e_tar[i]; acc[0] += d * d; continue; }
        i -= nE;
        if (i < nV) { const double d = (double)v[i] - (double)v_tar[i]; acc[2] += d * d; continue; }
        i -= nV;
        const double zi = z[i];
        acc[3] += fabs(zi); acc[4] += zi * zi;
    }
    __shared__ double red[5][kLossThreads / 32];
    __shared__ int s_last;
#pragma unroll
    for (int c = 0; c < 5; ++c)
        for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    if ((threadIdx.x & 31) == 0)
        for (int c = 0; c < 5; ++c) red[c][threadIdx.x >> 5] = acc[c];
    __syncthreads();
    double* rows = scratch + kHeaderDoubles;
    if (threadIdx.x == 0) {
        for (int c = 0; c < 5; ++c) {
            double t = 0.0;
            for (int w = 0; w < kLossThreads / 32; ++w) t += red[c][w];
            rows[(size_t)blockIdx.x * kRowDoubles + c] = t;
        }
        __threadfence();                                        // the row is visible before the ticket is taken
        const unsigned ticket = atomicAdd((unsigned*)scratch, 1u);
        s_last = (ticket == gridDim.x - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // the last block: rows in a fixed order (thread t takes rows t, t + 256, ...), then the same block reduction
#pragma unroll
    for (int c = 0; c < 5; ++c) acc[c] = 0.0;
    for (unsigned r = threadIdx.x; r < gridDim.x; r += kLossThreads)
#pragma unroll
        for (int c = 0; c < 5; ++c) acc[c] += __ldcg(&rows[(size_t)r * kRowDoubles + c]);
#pragma unroll
    for (int c = 0; c < 5; ++c)
        for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    __syncthreads();
    if ((threadIdx.x & 31) == 0)
        for (int c = 0; c < 5; ++c) red[c][threadIdx.x >> 5] = acc[c];
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[5];
        for (int c = 0; c < 5; ++c) { t[c] = 0.0; for (int w = 0; w < kLossThreads / 32; ++w) t[c] += red[c][w]; }
        out[0] = sqrt(t[0] / (double)S);                        // Eq. 30, per-atom energies (reading Q23)
        out[1] = sqrt(t[1] / (3.0 * (double)N));                // Eq. 31
        out[2] = sqrt(t[2] / (6.0 * (double)S));                // Eq. 32, six components xx yy zz xy yz zx (reading Q24)
        out[3] = t[3] / (double)npar;                           // Eq. 33
        out[4] = sqrt(t[4] / (double)npar);                     // Eq. 34
        out[5] = le * out[0] + lf * out[1] + lv * out[2] + l1w * out[3] + l2w * out[4];     // Eq. 29
    }
}

// per-device set-up: the device address of g_loss_scratch on each GPU, looked up once with that GPU current
constexpr int kMaxDevices = 64;
std::mutex g_setup_mutex;
double* g_scratch_addr[kMaxDevices] = {nullptr};

void say(char* buf, size_t len, const char* fmt, long long a = 0, long long b = 0, long long c = 0) {
    if (buf && len) snprintf(buf, len, fmt, a, b, c);
}

int scratch_on_current_device(double** out, char* errbuf, size_t errlen) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        if (errbuf && errlen) snprintf(errbuf, errlen, "nep_loss_noalloc: no usable current CUDA device (%s)",
                                       e != cudaSuccess ? cudaGetErrorString(e) : "device ordinal out of range");
        return NEP_ECUDA;
    }
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_scratch_addr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_loss_scratch);           // NOT &g_loss_scratch: that would be a host address
        if (e != cudaSuccess || !p) {
            if (errbuf && errlen) snprintf(errbuf, errlen, "nep_loss_noalloc: cudaGetSymbolAddress failed on device %d (%s)",
                                           dev, cudaGetErrorString(e));
            return NEP_ECUDA;
        }
        g_scratch_addr[dev] = (double*)p;
    }
    *out = g_scratch_addr[dev];
    return NEP_OK;
}

}  // namespace

extern "C" int nep_loss_noalloc(int64_t n_structures, int64_t n_atoms, int64_t n_par, const float* e_dev, const float* f_dev,
                                const float* v_dev, const float* e_tar_dev, const float* f_tar_dev, const float* v_tar_dev,
                                const double* z_dev, const double* lambda, double* loss_dev, void* cuda_stream, char* errbuf,
                                size_t errbuf_len) {
    if (errbuf && errbuf_len) errbuf[0] = 0;
    if (!e_dev || !f_dev || !v_dev || !e_tar_dev || !f_tar_dev || !v_tar_dev || !z_dev || !lambda || !loss_dev ||
        n_structures < 1 || n_atoms < 1 || n_par < 1) {
        say(errbuf, errbuf_len, "nep_loss_noalloc: null pointer or a size < 1");
        return NEP_EINVAL;
    }
    // sizes first (no CUDA call yet): what does not fit the fixed array is refused, never truncated
    if (n_atoms > kMaxElements || n_structures > kMaxElements || n_par > kMaxElements ||
        3 * n_atoms + 7 * n_structures + n_par > kMaxElements) {
        say(errbuf, errbuf_len,
            "nep_loss_noalloc: 3*n_atoms + 7*n_structures + n_par = %lld exceeds the fixed scratch (limit %lld elements, "
            "%lld bytes held in the library image); use nep_trainer_losses with a workspace of your own",
            (long long)(3 * n_atoms + 7 * n_structures + n_par), (long long)kMaxElements, (long long)kScratchBytes);
        return NEP_ENOMEM;
    }
    double* scratch = nullptr;
    const int rc = scratch_on_current_device(&scratch, errbuf, errbuf_len);
    if (rc != NEP_OK) return rc;
    const int64_t total = 3 * n_atoms + 7 * n_structures + n_par;
    const unsigned blocks = (unsigned)((total + kLossChunk - 1) / kLossChunk);          // <= kMaxRows by the test above
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemsetAsync(scratch, 0, kHeaderDoubles * sizeof(double), st);     // the ticket starts at zero
    if (e == cudaSuccess) {
        k_loss_static<<<blocks, kLossThreads, 0, st>>>(scratch, n_atoms, n_structures, n_par, e_dev, f_dev, v_dev, e_tar_dev,
                                                       f_tar_dev, v_tar_dev, z_dev, lambda[0], lambda[1], lambda[2], lambda[3],
                                                       lambda[4], loss_dev);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) {
        if (errbuf && errbuf_len) snprintf(errbuf, errbuf_len, "nep_loss_noalloc: CUDA error: %s", cudaGetErrorString(e));
        return NEP_ECUDA;
    }
    return NEP_OK;
}
