/*
 * nep_b200.h -- C ABI of libnep_b200.so: the NEP (neuroevolution potential, arXiv 2107.08119)
 * per-step force evaluation on one NVIDIA B200 (sm_100a).
 *
 * The calls follow the paper's statement of the problem (PAPER.md = /root/reference/PAPER.md):
 *   inputs  {r_i}, species, periodic box                      PAPER.md:54-66   (Sec. II A, Eq. 1-3)
 *   hyper-parameters r_c^R, r_c^A, n_max^R, n_max^A, l_max,
 *                    N_neu                                    PAPER.md:334-347 (Table I)
 *   parameter vector z of dimension N_par                     PAPER.md:221-224 (Eq. 26)
 *   outputs U_i, F_i, W_i (3x3), J_i                          PAPER.md:68-92   (Eq. 4-7)
 *
 * General rules
 *   - Every `*_dev` pointer is a DEVICE pointer owned by the caller (e.g. torch tensor.data_ptr());
 *     every other pointer is a HOST pointer.  The library never allocates in nep_compute /
 *     nep_md_step; all scratch lives in the caller-provided workspace.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  All compute
 *     calls are asynchronous on that stream.
 *   - Per-atom vectors are SoA: x[N] | y[N] | z[N].  The virial is [9][N], row-major components
 *     xx,xy,xz,yx,yy,yz,zx,zy,zz with  W_i^{ab} = sum_j r_ij^a (dU_j/dr_ji)^b  (Eq. 6).
 *   - Units: eV, Angstrom, amu, fs.  Force eV/A, virial eV, heat current eV*A/fs.
 *   - Outputs are in the caller's atom order although the library sorts atoms by cell internally.
 *   - Return value: NEP_OK (0) or a negative nep_error.  Device-side conditions (neighbour
 *     capacity overflow, stale list) are recorded in a sticky status word read by nep_status().
 *     Nothing is ever silently truncated.
 *   - There is no CPU fallback: without a CUDA device every compute entry point returns NEP_ECUDA.
 */
#ifndef NEP_B200_H
#define NEP_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    NEP_OK        = 0,
    NEP_EINVAL    = -1,  /* bad hyper-parameters, n_params mismatch, null pointer, unsupported shape   */
    NEP_EBOX      = -2,  /* a box length <= 2 (r_c^R + skin): minimum image ambiguous                   */
    NEP_ENOMEM    = -3,  /* workspace too small                                                         */
    NEP_ECUDA     = -4,  /* CUDA runtime / launch failure (or no device)                                */
    NEP_EOVERFLOW = -5,  /* some atom has more neighbours than cap_radial / cap_angular / the MD cap    */
    NEP_ESTALE    = -6,  /* nep_compute called with positions that moved > skin/2 since nep_neighbors   */
    NEP_ESTATE    = -7,  /* call order: nep_compute / nep_md_step before nep_neighbors                  */
    NEP_ENAN      = -8   /* a site energy or force came out non-finite (e.g. two atoms at one position)    */
} nep_error;

typedef struct nep_model  nep_model;   /* opaque, library-owned, immutable after nep_create           */
typedef struct nep_system nep_system;  /* opaque, library-owned: lists, scratch layout, permutation   */

/* Table I.  n_max follows the PAPER's convention: n = 0..n_max inclusive, so a
 * family has n_max+1 radial functions and N_des = (n_max_R+1) + (n_max_A+1) l_max  (Eq. 16). */
typedef struct {
    double rc_radial;       /* r_c^R, Angstrom                                                        */
    double rc_angular;      /* r_c^A, Angstrom, <= rc_radial                                          */
    int    n_max_radial;    /* 0..15                                                                  */
    int    n_max_angular;   /* 0..15                                                                  */
    int    l_max;           /* 1..8; 5..8 (general-l kernel): one species, one hidden layer, q_nl only    */
    int    n_neurons;       /* N_neu, single hidden layer (Eq. 21-22), 1..128                         */
    int    n_types;         /* 1..8; >1 switches on the sqrt(Z_i Z_j) weighting of Eq. 19             */
} nep_hyper;

/* ---- model -------------------------------------------------------------------------------------- */

/* Validates the hyper-parameters and uploads the network.
 *   atomic_number [n_types] host: Z of each type (Eq. 19); ignored when n_types == 1.
 *   params [n_params] host, fp64, order  w1[H][D] row-major | b1[H] | w2[H] | b2   with
 *          x_mu = tanh(sum_nu w1[mu][nu] q_nu - b1[mu]),  U_i = sum_mu w2[mu] x_mu - b2  (Eq. 21-22;
 *          note the MINUS biases).  Descriptor order q = [q_0..q_{n_max_R} | (n=0: l=1..l_max) |
 *          (n=1: l=1..l_max) | ...].  n_params must equal (D+2)H+1 (Eq. 26) else NEP_EINVAL. */
int  nep_create(const nep_hyper* hyper, const int* atomic_number, const double* params, size_t n_params,
                nep_model** out);
/* Variants the paper mentions without using them; evaluated by the 16-lanes-per-atom
 * kernel (NEP_PATH_GROUP) only:
 *   n_hidden_layers 1..3 ("generalization to more hidden layers is straightforward"):
 *     x^(k) = tanh(W^(k) x^(k-1) - b^(k)), x^(0) = q, U = w_out . x^(L) - b_out, every bias with the minus sign of
 *     Eq. 21-22; params order  W1[H1][D] | b1[H1] | W2[H2][H1] | b2[H2] | ... | w_out[H_L] | b_out; widths
 *     base.n_neurons, n_neurons_2, n_neurons_3 (each 1..128); n_params = sum_k (in_k + 1) H_k + H_L + 1.
 *   angular_kind NEP_ANGULAR_QNNL: the SOAP-like q_nn'l of Eq. 17-18,
 *     q_nn'l = (2l+1)/(4 pi) sum_jk g_n(r_ij) g_n'(r_ik) P_l(cos theta_ijk) = sum_m c_nlm c*_n'lm, for the pairs n <= n'
 *     (q_nn'l = q_n'nl), ordered n, then n' >= n, then l; N_des = (n_max_R+1) + (n_max_A+1)(n_max_A+2)/2 l_max;
 *     needs n_max_radial, n_max_angular <= 7.
 * Size limit: the lanes-per-atom kernel keeps the weights of ALL layers in shared memory beside its per-atom blocks, so
 * the padded weight count  sum_k H_k (in_k rounded up to 4) + the biases  is bounded by what a block may opt in to
 * (227 KB on B200): about 46,400 fp32 values for n_max <= 7 and 45,000 above; for n_types > 1 (fp64 weights) 17,300 /
 * 14,900 values.  nep_create_ex checks this on the current device and returns NEP_EINVAL for a shape that does not
 * fit, instead of a model whose launches fail.  Every one-species single-layer shape fits, and so do 3 x 128 at
 * D = 80 and 2 x 128 over q_nn'l; NOT: 3 x 128 over q_nn'l (D = 152); with n_types > 1: 2 x 128 at D = 80, or one
 * layer of 128 over q_nn'l (one layer of 128 at D = 80 and one of 100 over q_nn'l fit).
 * nep_create(h, ...) is nep_create_ex with one hidden layer and NEP_ANGULAR_QNL. */
enum { NEP_ANGULAR_QNL = 0, NEP_ANGULAR_QNNL = 1 };
typedef struct {
    nep_hyper base;
    int n_hidden_layers;    /* 1..3 */
    int n_neurons_2;        /* width of hidden layer 2 (n_hidden_layers >= 2) */
    int n_neurons_3;        /* width of hidden layer 3 (n_hidden_layers == 3) */
    int angular_kind;       /* NEP_ANGULAR_QNL or NEP_ANGULAR_QNNL */
} nep_hyper_ex;
int  nep_create_ex(const nep_hyper_ex* hyper, const int* atomic_number, const double* params, size_t n_params,
                   nep_model** out);
int  nep_descriptor_dim(const nep_model*);          /* Eq. 16 */
int  nep_num_params(const nep_model*);              /* Eq. 26 */
void nep_destroy(nep_model*);

/* ---- system ------------------------------------------------------------------------------------- */

/* Bytes of device workspace nep_system_create needs (0 on invalid arguments).  cap_radial /
 * cap_angular bound the neighbours per atom inside r_c^R / r_c^A (the paper's "M");
 * the internal Verlet list with skin is sized from them. */
size_t nep_workspace_bytes(const nep_model*, int64_t n_atoms, int cap_radial, int cap_angular, double skin);

/* type_dev [N] device int32 in 0..n_types-1 (copied).  workspace_dev: caller-owned device memory,
 * 256-byte aligned, >= nep_workspace_bytes(); must outlive the system.  skin >= 0 (Angstrom) is the
 * Verlet skin: lists stay valid while no atom has moved more than skin/2 since the last build.
 * A set-up call: it clears the workspace and copies the types, and synchronises the WHOLE DEVICE before and after doing
 * so -- whatever stream produced type_dev has finished, and any stream may be used for nep_neighbors afterwards. */
int  nep_system_create(const nep_model*, int64_t n_atoms, const int* type_dev, int cap_radial,
                       int cap_angular, double skin, void* workspace_dev, size_t workspace_bytes,
                       nep_system** out);
void nep_system_destroy(nep_system*);

/* Which kernel evaluates Eq. 12-25 (the descriptor, the network and the partial forces):
 *   NEP_PATH_THREAD  one thread per atom (k_main): every per-atom quantity in registers; instantiated for
 *                    n_max_radial / n_max_angular = 7/7, 8/8 or 12/6, l_max == 4, n_neurons <= 64 -- the BASELINE.json
 *                    shapes (D = 40 / 45); the faster form from ~1e4 atoms (nep_system_create switches at 12000)
 *   NEP_PATH_GROUP   16 lanes per atom (k_gen): any shape nep_create accepts, Table I's 80-50-1, 65-40-1 and
 *                    41-40-1 models included; the form for small systems
 * nep_system_create picks one from the shape and n_atoms (NEP_PATH_AUTO); nep_system_set_path overrides it
 * (NEP_EINVAL if the thread path is not instantiated for the model).  Changing the path invalidates the
 * lists: call nep_neighbors again.  Both paths produce the same quantities from the same lists. */
enum { NEP_PATH_AUTO = 0, NEP_PATH_THREAD = 1, NEP_PATH_GROUP = 2 };
int  nep_system_set_path(nep_system*, int path);
int  nep_system_path(const nep_system*);

/* Cell binning, cell sort and the Verlet list (cutoff r_c^R + skin) with reverse slots
 * ("smaller than r_c", "three neighbor lists").
 *   pos_dev [3][N] fp64 device, any real values (wrapped internally).
 *   box [3] host: orthorhombic periodic lengths; each must exceed 2 (r_c^R + skin) else NEP_EBOX. */
int  nep_neighbors(nep_system*, const double* pos_dev, const double box[3], void* cuda_stream);

/* The radial (which = 0, r < r_c^R) or angular (which = 1, r < r_c^A) list the force kernels use,
 * filtered from the Verlet list at the positions of the last nep_neighbors / nep_compute /
 * nep_md_step, with the predicate |d|^2 < r_c^2 evaluated in fp64 on minimum-image differences.
 *   count_dev [N], index_dev [N][cap] (cap = cap_radial or cap_angular) device int32, caller's atom
 *   numbering, row order unspecified (compare as sorted sets); unused entries are -1. */
int  nep_get_neighbors(nep_system*, int which, int* count_dev, int* index_dev, void* cuda_stream);

/* One evaluation of Eq. 12-15, 19, 21-25 and 4-7 at pos_dev with the lists of the last
 * nep_neighbors (positions may have moved by up to skin/2 per atom; more sets NEP_ESTALE).
 *   vel_dev [3][N] fp64, nullable (then heat_dev is not written).
 *   energy_dev [N], force_dev [3][N], virial_dev [9][N] (nullable), heat_dev [3][N] (nullable): fp32. */
int  nep_compute(nep_system*, const double* pos_dev, const double* vel_dev, float* energy_dev,
                 float* force_dev, float* virial_dev, float* heat_dev, void* cuda_stream);

/* Parity hook for the intermediate rows of the path: runs the same kernels as
 * nep_compute up to the partial forces and copies out, in the caller's atom order,
 *   q_dev  [D][N]  the descriptor q_i (Eq. 12-13; fp32, from the fp64 kernel for multi-species models)
 *   fp_dev [D][N]  dU_i/dq (Eq. 21-23)
 *   p_dev  [N][cap_radial][3]  dU_i/dr_ij (Eq. 23-25); neighbour k of atom i is entry k of
 *          nep_get_neighbors(which = 0) called after this function
 * Each pointer may be NULL.  Same preconditions and errors as nep_compute. */
int  nep_compute_internals(nep_system* system, const double* pos_dev, float* q_dev, float* fp_dev, float* p_dev,
                           void* cuda_stream);

/* n_steps velocity-Verlet NVE steps (BASELINE.json north_star; the paper's own timing used NVT,
 * PAPER.md:395):  v += dt/2 F/m;  r += dt v;  [rebuild lists on device when an atom moved > skin/2];
 * evaluate;  v += dt/2 F/m;  J_i = W_i . v_i (Eq. 7, both at t+dt).  a = F / (m * 103.642697) A/fs^2.
 * Requires nep_neighbors at the current positions first.  The first nep_md_step after nep_neighbors /
 * nep_compute evaluates F(t0) itself; a nep_md_step that directly follows another nep_md_step on the
 * same system CONTINUES the trajectory from the forces of that call: the caller must pass back the
 * positions it returned (velocities may be changed, e.g. rescaled).  Call nep_neighbors to restart.
 *   pos_dev, vel_dev [3][N] fp64: updated in place (positions are not wrapped).
 *   mass_by_type [n_types] host, amu.
 *   energy/force/virial/heat_dev: state after the last step (virial/heat nullable).
 *   heat_sum_dev [3][N] fp64 nullable: J_i added once per step (per-atom heat current accumulation).
 *   thermo_dev [n_steps][5] fp64 nullable: U_tot, K_tot, Jx, Jy, Jz after each step.
 * No host synchronisation happens inside; the whole call is a fixed launch sequence. */
int  nep_md_step(nep_system*, double* pos_dev, double* vel_dev, const double* mass_by_type, double dt_fs,
                 int n_steps, float* energy_dev, float* force_dev, float* virial_dev, float* heat_dev,
                 double* heat_sum_dev, double* thermo_dev, void* cuda_stream);

/* nep_md_step with the equations of motion of the homogeneous nonequilibrium MD method:
 *   driving_force [3] host, 1/Angstrom, nullable (NULL: identical to nep_md_step).  Eq. 9: the external force
 *     F_i^ext = F_e . W_i, read as (F_i^ext)^b = sum_a F_e^a W_i^{ab} -- the reading for which the power of the
 *     driving force is F_e . J with J = sum_i W_i . v_i (Eq. 7-8) -- is added to F_i in both half-kicks.
 *     force_dev still receives the potential force of Eq. 4.  No thermostat and no total-force correction are
 *     applied (the paper specifies neither); thermo_dev's J columns give <J(t)> of Eq. 8.
 *   w0_dev [9][N] fp32 device, nullable; kt_dev [n_steps][3] fp64 device, nullable (needs w0_dev).  Eq. 11: the
 *     virial-velocity correlation K(t) = sum_i W_i(0) . v_i(t) after each step, W_i(0) being the per-atom virial
 *     the caller kept from an earlier nep_compute / nep_md_step (same layout as virial_dev).
 * Everything else as nep_md_step. */
int  nep_md_step_driven(nep_system*, double* pos_dev, double* vel_dev, const double* mass_by_type, double dt_fs,
                        int n_steps, const double* driving_force, float* energy_dev, float* force_dev,
                        float* virial_dev, float* heat_dev, double* heat_sum_dev, double* thermo_dev,
                        const float* w0_dev, double* kt_dev, void* cuda_stream);

/* Synchronises the stream last used by this system and returns the sticky device status
 * (NEP_OK, NEP_EINVAL for an atom type outside the model, NEP_EOVERFLOW, NEP_ESTALE, NEP_ENAN) or NEP_ECUDA.
 * Clears the sticky word. */
int  nep_status(nep_system*);

/* Counters since nep_system_create (host values; synchronises like nep_status):
 * out[0] = list rebuilds, out[1] = max radial count seen, out[2] = max angular count seen,
 * out[3] = max Verlet-list count seen. */
int  nep_stats(nep_system*, int64_t out[4]);

/* ---- training side (Sec. II E-F) ------------------------------------------------ */

/* The loss of Eq. 29-34 for a population of parameter vectors over a training set of small periodic structures
 * "combined into a single one", and the separable natural evolution strategy of Eq. 35-39.
 * Structure n owns atoms first[n] .. first[n+1]-1 of the concatenated arrays and its own orthorhombic box
 * boxes[n][3] (every edge > 2 r_c^R: minimum image inside the structure).  Readings (Q23-Q25): U(n) and
 * W(n) of Eq. 30 / 32 are per atom ("eV/atom for energy and virial"); the six virial components are
 * xx, yy, zz, xy, yz, zx; the rank utilities u_k of Eq. 36-37, which the paper defers to its Ref. 44, are
 * max(0, ln(N_pop/2+1) - ln k) normalised to sum 1, minus 1/N_pop (k = 1 the smallest loss, ties by member index).
 * The structures do not move, so lists and records are built once in nep_trainer_create.
 *   atomic_number [n_types] HOST (Eq. 19; NULL when n_types == 1).  first [S+1], boxes [S][3]: HOST.
 *   pos_dev [3][N] fp64 (N = first[S]); type_dev [N] int32 device, 0..n_types-1 (NULL: all zero; copied).
 *   e_tar_dev [S] (per atom), f_tar_dev [3][N], v_tar_dev [S][6] (per atom): fp32 DEVICE targets, caller-owned, must
 *   outlive the trainer; all three nullable if only nep_trainer_predict is used. */
typedef struct nep_trainer nep_trainer;
size_t nep_trainer_workspace_bytes(const nep_hyper_ex*, int n_structures, int64_t n_atoms, int cap_radial, int cap_angular);
int  nep_trainer_create(const nep_hyper_ex*, const int* atomic_number, int n_structures, const int64_t* first,
                        const double* boxes, const double* pos_dev, const int* type_dev, const float* e_tar_dev,
                        const float* f_tar_dev, const float* v_tar_dev, int cap_radial, int cap_angular,
                        void* workspace_dev, size_t workspace_bytes, void* cuda_stream, nep_trainer** out);
void nep_trainer_destroy(nep_trainer*);
int  nep_trainer_num_params(const nep_trainer*);
int  nep_trainer_status(nep_trainer*);      /* as nep_status (capacity overflow) */

/* Eq. 29-34 for n_pop parameter vectors z_dev [n_pop][N_par] (fp64 device, the order of nep_create / nep_create_ex):
 * loss_dev [n_pop][6] = L_e, L_f, L_v, L_1, L_2 and the weighted total L; lambda [5] HOST = lambda_e, _f, _v, _1, _2. */
int  nep_trainer_losses(nep_trainer*, const double* z_dev, int n_pop, const double* lambda, double* loss_dev, void* cuda_stream);

/* One parameter vector: per-atom energy e_dev [S], forces f_dev [3][N], per-atom virial v_dev [S][6] (each nullable). */
int  nep_trainer_predict(nep_trainer*, const double* z_dev, float* e_dev, float* f_dev, float* v_dev, void* cuda_stream);

/* Eq. 35: z_k = m + s (.) r_k; r_dev [n_pop][n_par] standard normals supplied by the caller. */
int  nep_snes_sample(const double* m_dev, const double* s_dev, const double* r_dev, int n_pop, int n_par, double* z_dev,
                     void* cuda_stream);
/* Eq. 36-39: natural gradients from the ranks of loss_dev[k * loss_stride], then m and s in place (n_pop <= 1024). */
int  nep_snes_update(double* m_dev, double* s_dev, const double* r_dev, const double* loss_dev, int loss_stride, int n_pop,
                     int n_par, double eta_m, double eta_s, void* cuda_stream);

/* ---- for callers that cannot allocate device memory ------------------------------------------------ */

/* The loss of Eq. 29-34 for ONE parameter vector from predictions already on the device -- the
 * numbers nep_trainer_predict returns -- computed without any workspace from the caller and without a single
 * allocation inside the library (no cudaMalloc / cudaFree, no allocating library routine).
 *
 * Meant for code that has device arrays in its hands but no allocator: a callback invoked by another program with
 * just this step's arrays; a process whose device memory belongs wholly to one pool (PyTorch's caching allocator, a
 * scheduler's arena), where a raw cudaMalloc fails or robs the pool; a loop that cannot afford the device-wide
 * synchronisation of cudaMalloc, or runs while a stream of the process is being captured, when cudaMalloc is refused.
 * Everyone else should use nep_trainer_losses, which evaluates the model too and has no size limit.
 *
 * The partial sums live in a fixed 524,544-byte (0.5 MiB + 256 B) __device__ array inside libnep_b200.so; each GPU
 * that loads the library's device code holds that array until the process exits, used or not.  Consequences:
 *   - LIMIT: 3 n_atoms + 7 n_structures + n_par <= 16,777,216.  Beyond it the call returns NEP_ENOMEM, writes the
 *     reason to errbuf and touches nothing.
 *   - FIRST CALL PER DEVICE does a one-time set-up (looks up the array's address on the current device with
 *     cudaGetSymbolAddress; the runtime may load the library's device code at that moment).  Make it at start-up with
 *     the intended device current and BEFORE any stream capture begins.  Later calls on that device do none.
 *   - The array is shared by every call in the process and keeps the previous call's contents; the call clears the
 *     one counter that must start at zero itself (a memset on cuda_stream ahead of the kernel).  Calls that may
 *     OVERLAP on the GPU -- two streams with no event between them, two host threads -- race on it and give wrong
 *     losses: keep all calls on a device in one stream order.
 *
 *   e_dev [S] per-atom energy of each structure, f_dev [3][N] forces, v_dev [S][6] per-atom virial (xx yy zz xy yz zx):
 *     fp32 DEVICE, the layout of nep_trainer_predict; e_tar_dev, f_tar_dev, v_tar_dev: the targets, same layouts.
 *   z_dev [n_par] fp64 DEVICE: the parameter vector (L_1, L_2 of Eq. 33-34).  lambda [5] HOST: lambda_e, _f, _v, _1, _2.
 *   loss_dev [6] fp64 DEVICE, caller-owned: L_e, L_f, L_v, L_1, L_2 and the weighted total (Eq. 29).
 *   errbuf [errbuf_len] HOST, nullable: a plain-text reason whenever the return value is not NEP_OK.
 * Asynchronous on cuda_stream like every compute call.  Returns NEP_OK, NEP_EINVAL (null pointer, size < 1),
 * NEP_ENOMEM (beyond the limit above) or NEP_ECUDA. */
int  nep_loss_noalloc(int64_t n_structures, int64_t n_atoms, int64_t n_par, const float* e_dev, const float* f_dev,
                      const float* v_dev, const float* e_tar_dev, const float* f_tar_dev, const float* v_tar_dev,
                      const double* z_dev, const double* lambda, double* loss_dev, void* cuda_stream, char* errbuf,
                      size_t errbuf_len);

const char* nep_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* NEP_B200_H */
