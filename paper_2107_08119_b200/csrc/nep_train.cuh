// nep_train.cuh -- training side of the NEP hot path (included at the end of nep_b200.cu): the loss of Eq. 29-34
// for a whole population of parameter vectors over a set of small structures concatenated into one system
// (PAPER.md:306), and one generation of the separable natural evolution strategy, Eq. 35-39.
//
// The structures are static, so the neighbour lists and the per-step records are built ONCE (nep_trainer_create);
// a population member then costs: stage its weights, k_gen (descriptor + network + partial forces over all atoms of
// all structures), k_assemble (F, W), one reduction per structure.  Readings Q23-Q25: energy and virial per
// atom, the six components xx yy zz xy yz zx, the standard NES rank utilities.  Multi-species sets (Eq. 19): k_gen<double>.
#pragma once

struct nep_trainer {
    nep_model* model;
    nep_system* sys;
    int S, npar, stage_n;
    int64_t N;
    int* sid;                   // [N] structure of atom i
    int* first;                 // [S + 1]
    double* boxes;              // [S][6]: L[3], 1/L[3]
    int* types;                 // [N] (a copy of the caller's, or zeros)
    int* stage_map;             // [stage_n] index into z of every staged weight (-1: padding)
    float *U, *F, *W;           // [N], [3][N], [9][N] outputs of the member being evaluated
    double* sse;                // [3] squared-error sums of the member being evaluated
    const float *e_tar, *f_tar, *v_tar;      // caller-owned targets: [S] per atom, [3][N], [S][6] per atom
};

namespace {

// Verlet list of a concatenated set: thread i scans the atoms of its own structure (small: O(100) atoms), ascending j
__global__ void k_build_batch(SysDev d, int N, const double* __restrict__ pos, const int* __restrict__ type, int n_types,
                              const int* __restrict__ sid, const int* __restrict__ first, const double* __restrict__ boxes,
                              double rc2, int capMD) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int n = sid[i];
    const double* bx = boxes + 6 * (size_t)n;
    const double xi = pos[i], yi = pos[N + i], zi = pos[2 * (size_t)N + i];
    int ty = type[i];
    if (ty < 0 || ty >= n_types) { atomicOr(&d.flags[F_STATUS], ST_BADTYPE); ty = 0; }
    d.perm[i] = i; d.type_s[i] = ty;
    d.xs[i] = xi; d.xs[N + i] = yi; d.xs[2 * (size_t)N + i] = zi;
    d.xref[i] = xi; d.xref[N + i] = yi; d.xref[2 * (size_t)N + i] = zi;
    d.xs4[i] = make_double4(xi, yi, zi, __longlong_as_double((long long)ty));
    int cnt = 0;
    for (int j = first[n]; j < first[n + 1]; ++j) {
        if (j == i) continue;
        const double dx = min_image(pos[j] - xi, bx[0], bx[3]);
        const double dy = min_image(pos[N + j] - yi, bx[1], bx[4]);
        const double dz = min_image(pos[2 * (size_t)N + j] - zi, bx[2], bx[5]);
        if (dx * dx + dy * dy + dz * dz < rc2) {
            if (cnt < capMD) d.md_idx[mix(cnt, i, N)] = (unsigned)j;
            ++cnt;
        }
    }
    d.md_cnt[i] = min(cnt, capMD);
    if (cnt > capMD) atomicOr(&d.flags[F_STATUS], ST_OVERFLOW);
    atomicMax(&d.flags[F_MAXMD], cnt);
}

// z (fp64, Eq. 26 order or the deep-network order) -> the staged layout the kernels read (fp32, or fp64 for Eq. 19)
template <typename T>
__global__ void k_stage_params(const double* __restrict__ z, const int* __restrict__ map, T* __restrict__ dst, int n) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < n) dst[e] = map[e] >= 0 ? (T)z[map[e]] : (T)0;
}

// one block per structure: per-atom energy and virial of the structure, squared errors of Eq. 30-32
__global__ void __launch_bounds__(128) k_train_reduce(int N, const int* __restrict__ first, const float* __restrict__ U,
                                                      const float* __restrict__ F, const float* __restrict__ W,
                                                      const float* __restrict__ e_tar, const float* __restrict__ f_tar,
                                                      const float* __restrict__ v_tar, double* sse, float* e_out, float* v_out) {
    const int n = blockIdx.x;
    const int a0 = first[n], a1 = first[n + 1];
    const int comp[6] = {0, 4, 8, 1, 5, 6};                       // xx yy zz xy yz zx (reading Q24)
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};                     // energy, six virial components, force squared error
    for (int i = a0 + threadIdx.x; i < a1; i += blockDim.x) {
        acc[0] += (double)U[i];
#pragma unroll
        for (int c = 0; c < 6; ++c) acc[1 + c] += (double)W[(size_t)comp[c] * N + i];
        if (f_tar) {
#pragma unroll
            for (int a = 0; a < 3; ++a) { const double df = (double)F[(size_t)a * N + i] - (double)f_tar[(size_t)a * N + i]; acc[7] += df * df; }
        }
    }
    __shared__ double red[8][4];
#pragma unroll
    for (int c = 0; c < 8; ++c)
        for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    if ((threadIdx.x & 31) == 0)
        for (int c = 0; c < 8; ++c) red[c][threadIdx.x >> 5] = acc[c];
    __syncthreads();
    if (threadIdx.x == 0) {
        double t[8];
        for (int c = 0; c < 8; ++c) t[c] = red[c][0] + red[c][1] + red[c][2] + red[c][3];
        const double nat = (double)(a1 - a0);
        const double e = t[0] / nat;                               // reading Q23: per atom
        if (e_out) e_out[n] = (float)e;
        double sv = 0.0;
        for (int c = 0; c < 6; ++c) {
            const double w = t[1 + c] / nat;
            if (v_out) v_out[6 * (size_t)n + c] = (float)w;
            if (v_tar) { const double dv = w - (double)v_tar[6 * (size_t)n + c]; sv += dv * dv; }
        }
        if (sse) {
            if (e_tar) atomicAdd(&sse[0], (e - (double)e_tar[n]) * (e - (double)e_tar[n]));
            atomicAdd(&sse[1], t[7]);
            atomicAdd(&sse[2], sv);
        }
    }
}

// one block: L_e, L_f, L_v from the squared-error sums, L_1, L_2 from z, and the weighted total (Eq. 29-34)
__global__ void __launch_bounds__(256) k_train_loss(const double* __restrict__ z, int npar, const double* sse, int S, int64_t N,
                                                    double le, double lf, double lv, double l1w, double l2w, double* out) {
    double a1 = 0.0, a2 = 0.0;
    for (int k = threadIdx.x; k < npar; k += blockDim.x) { a1 += fabs(z[k]); a2 += z[k] * z[k]; }
    __shared__ double r1[8], r2[8];
    for (int o = 16; o > 0; o >>= 1) { a1 += __shfl_xor_sync(0xffffffffu, a1, o); a2 += __shfl_xor_sync(0xffffffffu, a2, o); }
    if ((threadIdx.x & 31) == 0) { r1[threadIdx.x >> 5] = a1; r2[threadIdx.x >> 5] = a2; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double s1 = 0.0, s2 = 0.0;
        for (int w = 0; w < 8; ++w) { s1 += r1[w]; s2 += r2[w]; }
        out[0] = sqrt(sse[0] / S); out[1] = sqrt(sse[1] / (3.0 * (double)N)); out[2] = sqrt(sse[2] / (6.0 * S));
        out[3] = s1 / npar; out[4] = sqrt(s2 / npar);
        out[5] = le * out[0] + lf * out[1] + lv * out[2] + l1w * out[3] + l2w * out[4];
    }
}

// Eq. 35
__global__ void k_snes_sample(const double* __restrict__ m, const double* __restrict__ s, const double* __restrict__ r,
                              int npop, int npar, double* __restrict__ z) {
    const size_t e = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e < (size_t)npop * npar) { const int n = (int)(e % npar); z[e] = m[n] + s[n] * r[e]; }
}

// Eq. 36-39 with the rank utilities of reading Q25; npop <= 1024 (the paper uses 50)
__global__ void __launch_bounds__(256) k_snes_update(double* m, double* s, const double* __restrict__ r, const double* __restrict__ loss,
                                                     int loss_stride, int npop, int npar, double eta_m, double eta_s) {
    __shared__ double util[1024];
    double norm = 0.0;
    for (int j = 1; j <= npop; ++j) norm += fmax(0.0, log(npop / 2.0 + 1.0) - log((double)j));
    for (int k = threadIdx.x; k < npop; k += blockDim.x) {
        // a loss that is not finite counts as +inf: the member ranks last, not first (reading Q25)
        const double lk0 = loss[(size_t)k * loss_stride], lk = isfinite(lk0) ? lk0 : CUDART_INF;
        int rank = 1;                                   // 1 = smallest loss, ties by index
        for (int j = 0; j < npop; ++j) {
            const double lj0 = loss[(size_t)j * loss_stride], lj = isfinite(lj0) ? lj0 : CUDART_INF;
            if (lj < lk || (lj == lk && j < k)) ++rank;
        }
        util[k] = fmax(0.0, log(npop / 2.0 + 1.0) - log((double)rank)) / norm - 1.0 / npop;
    }
    __syncthreads();
    // m[n], s[n] are read and written by exactly one thread (n is owned by one thread of the grid-stride loop): no atomics
    for (int n = blockIdx.x * blockDim.x + threadIdx.x; n < npar; n += gridDim.x * blockDim.x) {
        double gm = 0.0, gs = 0.0;
        for (int k = 0; k < npop; ++k) {
            const double rk = r[(size_t)k * npar + n];
            gm += util[k] * rk;                         // Eq. 36
            gs += util[k] * (rk * rk - 1.0);            // Eq. 37
        }
        m[n] += eta_m * (s[n] * gm);                    // Eq. 38
        s[n] *= exp(0.5 * eta_s * gs);                  // Eq. 39
    }
}

struct TrainLayout { size_t sys, sid, first, boxes, tz, map, U, F, W, sse, total; };
TrainLayout train_layout(size_t sys_bytes, int S, int64_t N, int stage_n) {
    TrainLayout L; size_t o = align256(sys_bytes);
    auto take = [&](size_t b) { size_t at = o; o = align256(o + b); return at; };
    L.sys = 0;
    L.sid = take((size_t)N * 4); L.first = take(((size_t)S + 1) * 4); L.boxes = take((size_t)S * 6 * 8); L.tz = take((size_t)N * 4);
    L.map = take((size_t)stage_n * 4); L.U = take((size_t)N * 4); L.F = take((size_t)N * 12); L.W = take((size_t)N * 36); L.sse = take(64);
    L.total = o;
    return L;
}

// elements of the staged weight buffer: the padded blob (deep), the raw Eq. 26 vector (fp64 path) or the padded fp32 layout
int train_stage_n(const nep_model* m) { return m->nlayers > 1 ? m->blob_elems : (m->h.n_types > 1 ? m->npar : m->params_floats); }

}  // namespace

extern "C" {

size_t nep_trainer_workspace_bytes(const nep_hyper_ex* hx, int n_structures, int64_t n_atoms, int cap_radial, int cap_angular) {
    if (!hx || n_structures < 1 || n_atoms < 1 || hx->base.n_types < 1 || hx->base.n_types > kMaxTypes) return 0;
    // the system part is sized by a model of this shape; only NA, D and n_types enter carve()
    nep_model tmp;
    tmp.h = hx->base;
    tmp.NA = hx->base.n_max_angular + 1; tmp.NR = hx->base.n_max_radial + 1;
    tmp.D = tmp.NR + (hx->angular_kind == NEP_ANGULAR_QNNL ? tmp.NA * (tmp.NA + 1) / 2 : tmp.NA) * hx->base.l_max;
    const size_t sys = nep_workspace_bytes(&tmp, n_atoms, cap_radial, cap_angular, 0.0);
    if (sys == 0) return 0;
    // staged weights: at most the padded blob of three 128-wide layers over a 152-component descriptor
    const int stage_max = 4 * (kMaxHGen * 160 + 2 * kMaxHGen * kMaxHGen + 4 * kMaxHGen + 8);
    return train_layout(sys, n_structures, n_atoms, stage_max).total;
}

int nep_trainer_create(const nep_hyper_ex* hx, const int* atomic_number, int n_structures, const int64_t* first, const double* boxes,
                       const double* pos_dev, const int* type_dev, const float* e_tar_dev, const float* f_tar_dev,
                       const float* v_tar_dev, int cap_radial, int cap_angular, void* workspace_dev, size_t workspace_bytes,
                       void* cuda_stream, nep_trainer** out) {
    if (!out) return NEP_EINVAL;
    *out = nullptr;
    if (!hx || !first || !boxes || !pos_dev || !workspace_dev || n_structures < 1) return NEP_EINVAL;
    if (hx->base.n_types > 1 && (!atomic_number || !type_dev)) return NEP_EINVAL;
    const int S = n_structures;
    const int64_t N = first[S];
    if (first[0] != 0 || N < 1) return NEP_EINVAL;
    for (int n = 0; n < S; ++n) {
        if (first[n + 1] <= first[n]) return NEP_EINVAL;
        for (int a = 0; a < 3; ++a)
            if (!(boxes[3 * n + a] > 2.0 * hx->base.rc_radial)) return NEP_EBOX;        // minimum image inside every structure
    }
    const size_t need = nep_trainer_workspace_bytes(hx, S, N, cap_radial, cap_angular);
    if (need == 0 || ((uintptr_t)workspace_dev & 255)) return NEP_EINVAL;
    if (workspace_bytes < need) return NEP_ENOMEM;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    // a model of this shape with zero weights: every member's weights are staged into its buffers
    nep_trainer* t = new (std::nothrow) nep_trainer();
    if (!t) return NEP_ENOMEM;
    int npar;
    {
        const int NR = hx->base.n_max_radial + 1, NA = hx->base.n_max_angular + 1;
        const int D = NR + (hx->angular_kind == NEP_ANGULAR_QNNL ? NA * (NA + 1) / 2 : NA) * hx->base.l_max;
        const int L = hx->n_hidden_layers, w[3] = {hx->base.n_neurons, hx->n_neurons_2, hx->n_neurons_3};
        int in = D; npar = 0;
        for (int k = 0; k < L && k < 3; ++k) { npar += (in + 1) * w[k]; in = w[k]; }
        npar += in + 1;
    }
    double* zeros = new double[(size_t)(npar > 0 ? npar : 1)]();
    int rc = nep_create_ex(hx, atomic_number, zeros, (size_t)npar, &t->model);
    delete[] zeros;
    if (rc != NEP_OK) { delete t; return rc; }
    nep_model* m = t->model;
    t->S = S; t->N = N; t->npar = m->npar; t->stage_n = train_stage_n(m);
    const size_t sys_bytes = nep_workspace_bytes(m, N, cap_radial, cap_angular, 0.0);
    const TrainLayout Lay = train_layout(sys_bytes, S, N, t->stage_n);
    char* base = (char*)workspace_dev;
    t->sid = (int*)(base + Lay.sid); t->first = (int*)(base + Lay.first); t->boxes = (double*)(base + Lay.boxes);
    t->types = (int*)(base + Lay.tz); t->stage_map = (int*)(base + Lay.map);
    t->U = (float*)(base + Lay.U); t->F = (float*)(base + Lay.F); t->W = (float*)(base + Lay.W); t->sse = (double*)(base + Lay.sse);
    t->e_tar = e_tar_dev; t->f_tar = f_tar_dev; t->v_tar = v_tar_dev;
    // host tables -> device
    int* h_sid = new int[(size_t)N]; int* h_first = new int[(size_t)S + 1]; double* h_box = new double[(size_t)S * 6];
    for (int n = 0; n < S; ++n) {
        for (int64_t i = first[n]; i < first[n + 1]; ++i) h_sid[i] = n;
        for (int a = 0; a < 3; ++a) { h_box[6 * n + a] = boxes[3 * n + a]; h_box[6 * n + 3 + a] = 1.0 / boxes[3 * n + a]; }
    }
    for (int n = 0; n <= S; ++n) h_first[n] = (int)first[n];
    int* h_map = new int[(size_t)t->stage_n];
    for (int e = 0; e < t->stage_n; ++e) h_map[e] = -1;
    if (m->nlayers == 1 && m->h.n_types > 1) {
        for (int e = 0; e < t->stage_n; ++e) h_map[e] = e;                 // k_gen<double> reads the Eq. 26 vector as it is
    } else if (m->nlayers == 1) {
        const int H = m->H, D = m->D, Dp = (D + 3) & ~3;
        for (int mu = 0; mu < H; ++mu) for (int v = 0; v < D; ++v) h_map[mu * Dp + v] = mu * D + v;
        for (int k = 0; k < 2 * H + 1; ++k) h_map[H * Dp + k] = H * D + k;
    } else {
        int in = m->D, src = 0;
        for (int k = 0; k < m->nlayers; ++k) {
            for (int mu = 0; mu < m->lw[k]; ++mu) for (int v = 0; v < in; ++v) h_map[m->off_w[k] + mu * m->lin_p[k] + v] = src + mu * in + v;
            src += m->lw[k] * in;
            for (int mu = 0; mu < m->lw[k]; ++mu) h_map[m->off_b[k] + mu] = src + mu;
            src += m->lw[k];
            in = m->lw[k];
        }
        for (int mu = 0; mu <= in; ++mu) h_map[m->off_out + mu] = src + mu;
    }
    cudaError_t e = cudaMemsetAsync(base + Lay.sid, 0, Lay.total - Lay.sid, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->sid, h_sid, (size_t)N * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->first, h_first, ((size_t)S + 1) * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->boxes, h_box, (size_t)S * 48, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(t->stage_map, h_map, (size_t)t->stage_n * 4, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess && type_dev) e = cudaMemcpyAsync(t->types, type_dev, (size_t)N * 4, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    delete[] h_sid; delete[] h_first; delete[] h_box; delete[] h_map;
    if (e != cudaSuccess) { set_cuda_error(e, "nep_trainer_create"); nep_destroy(t->model); delete t; return NEP_ECUDA; }
    rc = nep_system_create(m, N, t->types, cap_radial, cap_angular, 0.0, workspace_dev, sys_bytes, &t->sys);
    if (rc != NEP_OK) { nep_destroy(t->model); delete t; return rc; }
    nep_system* s = t->sys;
    s->path = NEP_PATH_GROUP;
    s->batch_boxes = t->boxes; s->batch_sid = t->sid;
    for (int a = 0; a < 3; ++a) { s->box.L[a] = 1.0; s->box.invL[a] = 1.0; s->box.nc[a] = 1; }
    s->box.ncell = 1;
    s->last_stream = st;
    // lists and records once: the structures do not move
    const int Ni = (int)N;
    const double rc2 = hx->base.rc_radial * hx->base.rc_radial;
    k_build_batch<<<grid_for(N, 128), 128, 0, st>>>(s->d, Ni, pos_dev, t->types, m->h.n_types, t->sid, t->first, t->boxes, rc2, s->capMD);
    k_rev<<<grid_for(N, 128), 128, 0, st>>>(s->d, Ni, 0);
    k_build_done<<<1, 1, 0, st>>>(s->d, 0);
    s->launches += 3;
    launch_filter(s, st);
    e = cudaGetLastError();
    if (e != cudaSuccess) { set_cuda_error(e, "nep_trainer_create"); nep_system_destroy(s); nep_destroy(t->model); delete t; return NEP_ECUDA; }
    s->built = true;
    *out = t;
    return NEP_OK;
}

void nep_trainer_destroy(nep_trainer* t) {
    if (!t) return;
    nep_system_destroy(t->sys);
    nep_destroy(t->model);
    delete t;
}

int nep_trainer_num_params(const nep_trainer* t) { return t ? t->npar : NEP_EINVAL; }
int nep_trainer_status(nep_trainer* t) { return t ? nep_status(t->sys) : NEP_EINVAL; }

}  // extern "C"

namespace {
// one member: stage its weights, evaluate all atoms of all structures, assemble F and W
void train_eval_member(nep_trainer* t, const double* z_dev, cudaStream_t st) {
    nep_model* m = t->model; nep_system* s = t->sys;
    if (m->h.n_types > 1)
        k_stage_params<double><<<grid_for(t->stage_n, 256), 256, 0, st>>>(z_dev, t->stage_map, m->nlayers > 1 ? m->blob64_dev : m->params64_dev, t->stage_n);
    else
        k_stage_params<float><<<grid_for(t->stage_n, 256), 256, 0, st>>>(z_dev, t->stage_map, m->nlayers > 1 ? m->blob_dev : m->params_dev, t->stage_n);
    s->launches += 1;
    launch_main(s, st);
    AsmParams P;
    memset(&P, 0, sizeof(P));
    P.N = (int)t->N; P.capR = s->capR; P.capMD = s->capMD; P.md = 0;
    fill_masses(&P, m, nullptr);
    P.energy = t->U; P.force = t->F; P.virial = t->W;
    launch_assemble(s, P, st);
}
}  // namespace

extern "C" {

int nep_trainer_losses(nep_trainer* t, const double* z_dev, int n_pop, const double* lambda, double* loss_dev, void* cuda_stream) {
    if (!t || !z_dev || !lambda || !loss_dev || n_pop < 1 || !t->e_tar || !t->f_tar || !t->v_tar) return NEP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    t->sys->last_stream = st;
    for (int k = 0; k < n_pop; ++k) {
        const double* zk = z_dev + (size_t)k * t->npar;
        NEP_CUDA_OK(cudaMemsetAsync(t->sse, 0, 3 * sizeof(double), st));
        train_eval_member(t, zk, st);
        k_train_reduce<<<t->S, 128, 0, st>>>((int)t->N, t->first, t->U, t->F, t->W, t->e_tar, t->f_tar, t->v_tar, t->sse, nullptr, nullptr);
        k_train_loss<<<1, 256, 0, st>>>(zk, t->npar, t->sse, t->S, t->N, lambda[0], lambda[1], lambda[2], lambda[3], lambda[4],
                                        loss_dev + (size_t)k * 6);
        t->sys->launches += 2;
    }
    NEP_CUDA_OK(cudaGetLastError());
    return NEP_OK;
}

int nep_trainer_predict(nep_trainer* t, const double* z_dev, float* e_dev, float* f_dev, float* v_dev, void* cuda_stream) {
    if (!t || !z_dev) return NEP_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    t->sys->last_stream = st;
    train_eval_member(t, z_dev, st);
    k_train_reduce<<<t->S, 128, 0, st>>>((int)t->N, t->first, t->U, t->F, t->W, nullptr, nullptr, nullptr, nullptr, e_dev, v_dev);
    t->sys->launches += 1;
    if (f_dev) NEP_CUDA_OK(cudaMemcpyAsync(f_dev, t->F, (size_t)t->N * 12, cudaMemcpyDeviceToDevice, st));
    NEP_CUDA_OK(cudaGetLastError());
    return NEP_OK;
}

int nep_snes_sample(const double* m_dev, const double* s_dev, const double* r_dev, int n_pop, int n_par, double* z_dev, void* cuda_stream) {
    if (!m_dev || !s_dev || !r_dev || !z_dev || n_pop < 1 || n_par < 1) return NEP_EINVAL;
    const size_t n = (size_t)n_pop * n_par;
    k_snes_sample<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(m_dev, s_dev, r_dev, n_pop, n_par, z_dev);
    NEP_CUDA_OK(cudaGetLastError());
    return NEP_OK;
}

int nep_snes_update(double* m_dev, double* s_dev, const double* r_dev, const double* loss_dev, int loss_stride, int n_pop, int n_par,
                    double eta_m, double eta_s, void* cuda_stream) {
    if (!m_dev || !s_dev || !r_dev || !loss_dev || n_pop < 1 || n_pop > 1024 || n_par < 1 || loss_stride < 1) return NEP_EINVAL;
    int g = (n_par + 255) / 256; if (g > 148 * 4) g = 148 * 4;
    k_snes_update<<<g, 256, 0, (cudaStream_t)cuda_stream>>>(m_dev, s_dev, r_dev, loss_dev, loss_stride, n_pop, n_par, eta_m, eta_s);
    NEP_CUDA_OK(cudaGetLastError());
    return NEP_OK;
}

}  // extern "C"
