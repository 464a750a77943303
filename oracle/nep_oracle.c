/*
 * nep_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the NEP hot path computes, written
 * from the paper (arXiv 2107.08119, /root/reference/PAPER.md) equation by
 * equation, in the paper's order and notation.  It shares no code, header,
 * table or constant with paper_2107_08119_b200/csrc/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.
 *
 * What is literal here (no blocking, fusion or reordering):
 *   - neighbours: every ordered pair, minimum image, strict r < r_c
 *   - radial functions g_n, Eq. 14-15, Chebyshev by Eq. A1-A3
 *   - multi-component weighting f_c -> f_c sqrt(Z_i Z_j), Eq. 19
 *   - radial descriptor Eq. 12, angular descriptor Eq. 13 as the literal
 *     double sum over j and k (j = k included), Legendre by recurrence
 *   - network Eq. 21-22 with MINUS biases
 *   - partial forces Eq. 23-25
 *   - force Eq. 4-5, per-atom virial Eq. 6, heat current Eq. 7
 *   - velocity-Verlet NVE step (BASELINE.json; not in the paper), lists rebuilt
 *     from scratch every step.
 *
 * Pins (tests/test_oracle_*.py): Chebyshev/Legendre closed forms, g_n special
 * values, N_des/N_par printed by the paper, dimer/trimer closed forms, the
 * addition-theorem identity Eq. 17-18 via scipy's complex Y_lm, invariances,
 * F = -grad U and W = -dU/d(strain) by central differences, the heat-current
 * identity on an open cluster, brute-force vs cell-list neighbours, NVE; the PER-ATOM
 * split of W_i and J_i = W_i . v_i through dU_j/dr_ji == dU_j/dr_i, i.e. central
 * differences of the per-atom energies U_j as atom i moves (open cluster and periodic C0),
 * with the transposed index order and p_ij-for-p_ji as failing negative controls.
 *
 * Layout: positions/velocities/forces SoA  x[N] | y[N] | z[N];  virial [9][N]
 * row-major (xx,xy,xz,yx,...), W^{ab} = sum_j r_ij^a (dU_j/dr_ji)^b.
 * Descriptor order: q_0..q_{nmaxR}, then for n = 0..nmaxA: l = 1..lmax.
 * Parameter order: w1[H][D] | b1[H] | w2[H] | b2.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAX_N 32   /* radial functions per family */
#define ORC_MAX_L 8
#define ORC_MAX_D 1200 /* descriptor components (variants included) */
#define ORC_MAX_H 256  /* neurons per hidden layer */

typedef struct {
    double rc_r, rc_a;          /* r_c^R, r_c^A (Table I)                    */
    int nmax_r, nmax_a;         /* inclusive n_max (Eq. 16)                  */
    int lmax;                   /* l = 1..lmax                               */
    int nneu;                   /* N_neu                                     */
    int ntypes;                 /* 1 => omega_ij = 1; >1 => Eq. 19           */
    /* variants the paper mentions but does not use (0 = the paper's own form): */
    int nlayers;                /* hidden layers, 0 or 1 = the single layer of Eq. 21-22; 2, 3: "generalization to
                                   more hidden layers is straightforward"                         */
    int nneu2, nneu3;           /* widths of hidden layers 2 and 3                                              */
    int kind;                   /* 0: q_nl of Eq. 13; 1: the SOAP-like q_nn'l of Eq. 17      */
} orc_hyper;

static int orc_layers(const orc_hyper *h, int *width) {  /* hidden-layer widths; returns their number */
    int L = h->nlayers < 1 ? 1 : h->nlayers;
    width[0] = h->nneu; width[1] = h->nneu2; width[2] = h->nneu3;
    return L;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

int orc_descriptor_dim(const orc_hyper *h) {              /* Eq. 16 */
    if (h->kind == 1)                                     /* q_nn'l = q_n'nl: the pairs n <= n' */
        return (h->nmax_r + 1) + ((h->nmax_a + 1) * (h->nmax_a + 2) / 2) * h->lmax;
    return (h->nmax_r + 1) + (h->nmax_a + 1) * h->lmax;
}
int orc_num_params(const orc_hyper *h) {                  /* Eq. 26 */
    if (h->nlayers > 1) {                                 /* every layer: weights + biases; output: weights + bias */
        int w[3], L = orc_layers(h, w), in = orc_descriptor_dim(h), np = 0;
        for (int k = 0; k < L; ++k) { np += (in + 1) * w[k]; in = w[k]; }
        return np + in + 1;
    }
    return (orc_descriptor_dim(h) + 2) * h->nneu + 1;
}

/* Eq. A1, A3: T_0..T_nmax and U_0..U_nmax at x. */
void orc_chebyshev(double x, int nmax, double *T, double *U) {
    T[0] = 1.0; U[0] = 1.0;
    if (nmax >= 1) { T[1] = x; U[1] = 2.0 * x; }
    for (int n = 2; n <= nmax; ++n) {
        T[n] = 2.0 * x * T[n - 1] - T[n - 2];
        U[n] = 2.0 * x * U[n - 1] - U[n - 2];
    }
}

/* Eq. 15 and its derivative; strict zero at and beyond r_c. */
void orc_cutoff(double r, double rc, double *fc, double *dfc) {
    if (r < rc) {
        *fc = 0.5 * (1.0 + cos(M_PI * r / rc));
        *dfc = -0.5 * (M_PI / rc) * sin(M_PI * r / rc);
    } else { *fc = 0.0; *dfc = 0.0; }
}

/* Eq. 14 (+ Eq. 19 weight omega): g_n(r) = (T_n(x)+1)/2 * f_c(r) * omega,
 * x = 2 (r/r_c - 1)^2 - 1; dg_n/dr by the product rule with Eq. A2. */
void orc_radial(double r, double rc, int nmax, double omega, double *g, double *dg) {
    double T[ORC_MAX_N + 1], U[ORC_MAX_N + 1], fc, dfc;
    double x = 2.0 * (r / rc - 1.0) * (r / rc - 1.0) - 1.0;
    double dx = 4.0 * (r / rc - 1.0) / rc;
    orc_chebyshev(x, nmax, T, U);
    orc_cutoff(r, rc, &fc, &dfc);
    for (int n = 0; n <= nmax; ++n) {
        double dT = (n == 0) ? 0.0 : n * U[n - 1];            /* Eq. A2 */
        g[n] = 0.5 * (T[n] + 1.0) * fc * omega;
        dg[n] = 0.5 * (dT * dx * fc + (T[n] + 1.0) * dfc) * omega;
    }
}

/* Legendre P_0..P_lmax and derivatives: (l+1)P_{l+1} = (2l+1) c P_l - l P_{l-1},
 * P'_{l+1} = P'_{l-1} + (2l+1) P_l. */
void orc_legendre(double c, int lmax, double *P, double *dP) {
    P[0] = 1.0; dP[0] = 0.0;
    if (lmax >= 1) { P[1] = c; dP[1] = 1.0; }
    for (int l = 1; l < lmax; ++l) {
        P[l + 1] = ((2 * l + 1) * c * P[l] - l * P[l - 1]) / (l + 1);
        dP[l + 1] = dP[l - 1] + (2 * l + 1) * P[l];
    }
}

static inline void min_image(const double *pos, int64_t n, const double *box, int64_t i, int64_t j, double d[3]) {
    for (int a = 0; a < 3; ++a) {
        double t = pos[a * n + j] - pos[a * n + i];           /* Eq. 3: r_ij = r_j - r_i */
        t -= box[a] * nearbyint(t / box[a]);
        d[a] = t;
    }
}

/* All j != i with |r_ij|^2 < rc^2 (strict), ascending j.  O(N^2).
 * Returns the largest count found (may exceed cap: rows are then truncated and
 * the caller must treat it as an error).  borderline: number of ordered pairs
 * with | |d|^2 - rc^2 | <= 1e-9 A^2 (reading Q9). */
int orc_neighbors_brute(int64_t n, const double *pos, const double *box, double rc, int cap,
                        int *count, int *index, int64_t *borderline) {
    int maxc = 0; int64_t nb = 0;
    #pragma omp parallel for schedule(dynamic, 64) reduction(max:maxc) reduction(+:nb)
    for (int64_t i = 0; i < n; ++i) {
        int c = 0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double d[3]; min_image(pos, n, box, i, j, d);
            double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
            if (fabs(r2 - rc * rc) <= 1e-9) ++nb;
            if (r2 < rc * rc) { if (c < cap) index[i * (int64_t)cap + c] = (int)j; ++c; }
        }
        count[i] = c;
        if (c > maxc) maxc = c;
    }
    if (borderline) *borderline = nb;
    return maxc;
}

/* Same result through the oracle's own cell list (for N > 8000).  Cells of edge
 * >= rc; an axis with fewer than 3 cells is treated as one cell. */
int orc_neighbors_cell(int64_t n, const double *pos, const double *box, double rc, int cap,
                       int *count, int *index, int64_t *borderline) {
    int nc[3];
    for (int a = 0; a < 3; ++a) { nc[a] = (int)floor(box[a] / rc); if (nc[a] < 3) nc[a] = 1; }
    int64_t ncell = (int64_t)nc[0] * nc[1] * nc[2];
    int *cell_of = (int *)malloc(sizeof(int) * n);
    int64_t *start = (int64_t *)calloc(ncell + 1, sizeof(int64_t));
    int *members = (int *)malloc(sizeof(int) * n);
    for (int64_t i = 0; i < n; ++i) {
        int c[3];
        for (int a = 0; a < 3; ++a) {
            double f = pos[a * n + i] / box[a]; f -= floor(f);
            c[a] = (int)(f * nc[a]); if (c[a] >= nc[a]) c[a] = nc[a] - 1;
        }
        cell_of[i] = (c[0] * nc[1] + c[1]) * nc[2] + c[2];
        start[cell_of[i] + 1]++;
    }
    for (int64_t c = 0; c < ncell; ++c) start[c + 1] += start[c];
    int64_t *fill = (int64_t *)malloc(sizeof(int64_t) * ncell);
    memcpy(fill, start, sizeof(int64_t) * ncell);
    for (int64_t i = 0; i < n; ++i) members[fill[cell_of[i]]++] = (int)i;   /* ascending i inside a cell */
    int maxc = 0; int64_t nb = 0;
    #pragma omp parallel for schedule(dynamic, 64) reduction(max:maxc) reduction(+:nb)
    for (int64_t i = 0; i < n; ++i) {
        int ci = cell_of[i];
        int cz = ci % nc[2], cy = (ci / nc[2]) % nc[1], cx = ci / (nc[2] * nc[1]);
        int c = 0;
        int *row = index + i * (int64_t)cap;
        for (int ox = (nc[0] > 1 ? -1 : 0); ox <= (nc[0] > 1 ? 1 : 0); ++ox)
        for (int oy = (nc[1] > 1 ? -1 : 0); oy <= (nc[1] > 1 ? 1 : 0); ++oy)
        for (int oz = (nc[2] > 1 ? -1 : 0); oz <= (nc[2] > 1 ? 1 : 0); ++oz) {
            int64_t cj = (((cx + ox + nc[0]) % nc[0]) * (int64_t)nc[1] + (cy + oy + nc[1]) % nc[1]) * nc[2]
                         + (cz + oz + nc[2]) % nc[2];
            for (int64_t s = start[cj]; s < start[cj + 1]; ++s) {
                int64_t j = members[s];
                if (j == i) continue;
                double d[3]; min_image(pos, n, box, i, j, d);
                double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                if (fabs(r2 - rc * rc) <= 1e-9) ++nb;
                if (r2 < rc * rc) { if (c < cap) row[c] = (int)j; ++c; }
            }
        }
        /* ascending j (insertion sort; rows are short) */
        int m = c < cap ? c : cap;
        for (int a = 1; a < m; ++a) { int v = row[a], b = a - 1; while (b >= 0 && row[b] > v) { row[b + 1] = row[b]; --b; } row[b + 1] = v; }
        count[i] = c;
        if (c > maxc) maxc = c;
    }
    free(cell_of); free(start); free(members); free(fill);
    if (borderline) *borderline = nb;
    return maxc;
}

static inline double omega_ij(const orc_hyper *h, const int *znum, const int *type, int64_t i, int64_t j) {
    if (h->ntypes <= 1) return 1.0;
    return sqrt((double)znum[type[i]] * (double)znum[type[j]]);            /* Eq. 19 */
}

/* Eq. 21-22 and dU/dq (chain rule through tanh).  params: w1[H][D] | b1[H] | w2[H] | b2. */
/* More hidden layers: x^(k) = tanh(W^(k) x^(k-1) - b^(k)), x^(0) = q, U = w_out . x^(L) - b_out, every
 * bias with the minus sign of Eq. 21-22.  params: W1[H1][D] | b1[H1] | W2[H2][H1] | b2[H2] | ... | w_out[H_L] | b_out.
 * dU/dq by back-propagation: delta^(L) = w_out (1 - x^(L)^2), delta^(k-1) = (W^(k))^T delta^(k) (1 - x^(k-1)^2). */
static void orc_network_deep(const orc_hyper *h, const double *params, const double *q, double *U, double *Fp) {
    int w[3], L = orc_layers(h, w), D = orc_descriptor_dim(h);
    double x[4][ORC_MAX_D > ORC_MAX_H ? ORC_MAX_D : ORC_MAX_H], delta[ORC_MAX_D > ORC_MAX_H ? ORC_MAX_D : ORC_MAX_H], prev[ORC_MAX_D > ORC_MAX_H ? ORC_MAX_D : ORC_MAX_H];
    const double *W[3], *b[3];
    int in = D; const double *p = params;
    for (int v = 0; v < D; ++v) x[0][v] = q[v];
    for (int k = 0; k < L; ++k) {
        W[k] = p; b[k] = p + (size_t)w[k] * in; p = b[k] + w[k];
        for (int m = 0; m < w[k]; ++m) {
            double a = 0.0;
            for (int v = 0; v < in; ++v) a += W[k][m * in + v] * x[k][v];
            x[k + 1][m] = tanh(a - b[k][m]);
        }
        in = w[k];
    }
    double u = 0.0;
    for (int m = 0; m < in; ++m) { u += p[m] * x[L][m]; delta[m] = p[m] * (1.0 - x[L][m] * x[L][m]); }
    *U = u - p[in];
    for (int k = L - 1; k >= 0; --k) {
        int nin = k == 0 ? D : w[k - 1];
        for (int v = 0; v < nin; ++v) {
            double s = 0.0;
            for (int m = 0; m < w[k]; ++m) s += delta[m] * W[k][m * nin + v];
            prev[v] = k == 0 ? s : s * (1.0 - x[k][v] * x[k][v]);
        }
        for (int v = 0; v < nin; ++v) delta[v] = prev[v];
    }
    for (int v = 0; v < D; ++v) Fp[v] = delta[v];
}

void orc_network(const orc_hyper *h, const double *params, const double *q, double *U, double *Fp) {
    if (h->nlayers > 1) { orc_network_deep(h, params, q, U, Fp); return; }
    int D = orc_descriptor_dim(h), H = h->nneu;
    const double *w1 = params, *b1 = params + (size_t)H * D, *w2 = b1 + H, *b2 = w2 + H;
    double u = 0.0;
    for (int v = 0; v < D; ++v) Fp[v] = 0.0;
    for (int m = 0; m < H; ++m) {
        double a = 0.0;
        for (int v = 0; v < D; ++v) a += w1[m * D + v] * q[v];
        a -= b1[m];                                                        /* Eq. 21: minus bias */
        double x = tanh(a);
        u += w2[m] * x;
        for (int v = 0; v < D; ++v) Fp[v] += w2[m] * (1.0 - x * x) * w1[m * D + v];
    }
    *U = u - b2[0];                                                        /* Eq. 22: minus bias */
}

/* Descriptor of atom i from its two lists: Eq. 12 and the literal double sum of Eq. 13. */
void orc_descriptor_atom(const orc_hyper *h, const int *znum, const int *type, int64_t n, const double *pos,
                         const double *box, int64_t i, int nR, const int *listR, int nA, const int *listA,
                         double *q) {
    int D = orc_descriptor_dim(h);
    for (int v = 0; v < D; ++v) q[v] = 0.0;
    double g[ORC_MAX_N + 1], dg[ORC_MAX_N + 1];
    for (int a = 0; a < nR; ++a) {                                         /* Eq. 12 */
        int64_t j = listR[a]; double d[3]; min_image(pos, n, box, i, j, d);
        double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
        orc_radial(r, h->rc_r, h->nmax_r, omega_ij(h, znum, type, i, j), g, dg);
        for (int k = 0; k <= h->nmax_r; ++k) q[k] += g[k];
    }
    double gk[ORC_MAX_N + 1], P[ORC_MAX_L + 1], dP[ORC_MAX_L + 1];
    for (int a = 0; a < nA; ++a) {                                         /* Eq. 13: sum over j ... */
        int64_t j = listA[a]; double dj[3]; min_image(pos, n, box, i, j, dj);
        double rj = sqrt(dj[0] * dj[0] + dj[1] * dj[1] + dj[2] * dj[2]);
        orc_radial(rj, h->rc_a, h->nmax_a, omega_ij(h, znum, type, i, j), g, dg);
        for (int b = 0; b < nA; ++b) {                                     /* ... and over k, k = j included */
            int64_t k = listA[b]; double dk[3]; min_image(pos, n, box, i, k, dk);
            double rk = sqrt(dk[0] * dk[0] + dk[1] * dk[1] + dk[2] * dk[2]);
            orc_radial(rk, h->rc_a, h->nmax_a, omega_ij(h, znum, type, i, k), gk, dg);
            double c = (dj[0] * dk[0] + dj[1] * dk[1] + dj[2] * dk[2]) / (rj * rk);
            orc_legendre(c, h->lmax, P, dP);
            if (h->kind == 1) {                /* Eq. 17 written as the double sum it came from:
                                                  g_n(r_ij) g_n'(r_ik) (2l+1)/(4 pi) P_l, for the pairs n <= n' */
                int v = h->nmax_r + 1;
                for (int m = 0; m <= h->nmax_a; ++m)
                    for (int m2 = m; m2 <= h->nmax_a; ++m2)
                        for (int l = 1; l <= h->lmax; ++l)
                            q[v++] += g[m] * gk[m2] * ((2 * l + 1) / (4.0 * M_PI)) * P[l];
                continue;
            }
            for (int m = 0; m <= h->nmax_a; ++m)
                for (int l = 1; l <= h->lmax; ++l)
                    q[(h->nmax_r + 1) + m * h->lmax + (l - 1)] += g[m] * gk[m] * P[l];
        }
    }
}

static int find_slot(const int *row, int cnt, int target) {
    for (int a = 0; a < cnt; ++a) if (row[a] == target) return a;
    return -1;
}

/*
 * One full evaluation given the two neighbour lists (rows ascending, capR/capA wide).
 * Outputs (any may be NULL): U[N]; F[3][N]; W[9][N]; J[3][N] (needs vel);
 * q[N][D]; Fp[N][D]; p[N][capR][3] (partial forces dU_i/dr_ij in radial-list slots).
 * Returns 0, or -1 if a list is asymmetric (j in R(i) but i not in R(j)).
 */
int orc_compute(int64_t n, const double *pos, const double *vel, const int *type, const double *box,
                const orc_hyper *h, const int *znum, const double *params,
                int capR, const int *cntR, const int *idxR, int capA, const int *cntA, const int *idxA,
                double *U, double *F, double *W, double *J, double *q_out, double *Fp_out, double *p_out) {
    int D = orc_descriptor_dim(h);
    double *p = p_out ? p_out : (double *)malloc(sizeof(double) * 3 * (size_t)n * capR);
    memset(p, 0, sizeof(double) * 3 * (size_t)n * capR);
    int bad = 0;

    #pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < n; ++i) {
        double q[ORC_MAX_D], Fp[ORC_MAX_D], Ui;
        const int *LR = idxR + i * (int64_t)capR, *LA = idxA + i * (int64_t)capA;
        int nR = cntR[i], nA = cntA[i];
        orc_descriptor_atom(h, znum, type, n, pos, box, i, nR, LR, nA, LA, q);
        orc_network(h, params, q, &Ui, Fp);
        if (U) U[i] = Ui;
        if (q_out) memcpy(q_out + i * (int64_t)D, q, sizeof(double) * D);
        if (Fp_out) memcpy(Fp_out + i * (int64_t)D, Fp, sizeof(double) * D);

        double g[ORC_MAX_N + 1], dg[ORC_MAX_N + 1], gk[ORC_MAX_N + 1], dgk[ORC_MAX_N + 1];
        double P[ORC_MAX_L + 1], dP[ORC_MAX_L + 1];
        double *pi = p + 3 * i * (int64_t)capR;
        /* radial part: Eq. 23 with Eq. 24 */
        for (int a = 0; a < nR; ++a) {
            int64_t j = LR[a]; double d[3]; min_image(pos, n, box, i, j, d);
            double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
            orc_radial(r, h->rc_r, h->nmax_r, omega_ij(h, znum, type, i, j), g, dg);
            double s = 0.0;
            for (int k = 0; k <= h->nmax_r; ++k) s += Fp[k] * dg[k];
            for (int c = 0; c < 3; ++c) pi[3 * a + c] += s * d[c] / r;
        }
        /* angular part: Eq. 23 with Eq. 25 */
        for (int a = 0; a < nA; ++a) {
            int64_t j = LA[a]; double dj[3]; min_image(pos, n, box, i, j, dj);
            double rj = sqrt(dj[0] * dj[0] + dj[1] * dj[1] + dj[2] * dj[2]);
            orc_radial(rj, h->rc_a, h->nmax_a, omega_ij(h, znum, type, i, j), g, dg);
            int slot = find_slot(LR, nR, (int)j);          /* A(i) is a subset of R(i) since r_c^A <= r_c^R */
            if (slot < 0) { bad = 1; continue; }
            double acc[3] = {0.0, 0.0, 0.0};
            for (int b = 0; b < nA; ++b) {
                int64_t k = LA[b]; double dk[3]; min_image(pos, n, box, i, k, dk);
                double rk = sqrt(dk[0] * dk[0] + dk[1] * dk[1] + dk[2] * dk[2]);
                orc_radial(rk, h->rc_a, h->nmax_a, omega_ij(h, znum, type, i, k), gk, dgk);
                double c = (dj[0] * dk[0] + dj[1] * dk[1] + dj[2] * dk[2]) / (rj * rk);
                orc_legendre(c, h->lmax, P, dP);
                if (h->kind == 1) {            /* d q_nn'l / d r_ij: atom j enters the double sum once as the first
                                                  factor (radial index n) and once as the second (n') */
                    int v = h->nmax_r + 1;
                    for (int m = 0; m <= h->nmax_a; ++m)
                        for (int m2 = m; m2 <= h->nmax_a; ++m2)
                            for (int l = 1; l <= h->lmax; ++l) {
                                double fp = Fp[v++] * ((2 * l + 1) / (4.0 * M_PI));
                                for (int x = 0; x < 3; ++x) {
                                    double rhat_j = dj[x] / rj, rhat_k = dk[x] / rk;
                                    double ang = dP[l] * (1.0 / rj) * (rhat_k - rhat_j * c);
                                    double first = dg[m] * gk[m2] * rhat_j * P[l] + g[m] * gk[m2] * ang;
                                    double second = gk[m] * dg[m2] * rhat_j * P[l] + gk[m] * g[m2] * ang;
                                    acc[x] += fp * (first + second);
                                }
                            }
                    continue;
                }
                for (int m = 0; m <= h->nmax_a; ++m)
                    for (int l = 1; l <= h->lmax; ++l) {
                        double fp = Fp[(h->nmax_r + 1) + m * h->lmax + (l - 1)];
                        for (int x = 0; x < 3; ++x) {
                            double rhat_j = dj[x] / rj, rhat_k = dk[x] / rk;
                            double t1 = 2.0 * dg[m] * gk[m] * rhat_j * P[l];
                            double t2 = 2.0 * g[m] * gk[m] * dP[l] * (1.0 / rj) * (rhat_k - rhat_j * c);
                            acc[x] += fp * (t1 + t2);
                        }
                    }
            }
            for (int x = 0; x < 3; ++x) pi[3 * slot + x] += acc[x];
        }
    }
    if (bad) { if (!p_out) free(p); return -1; }

    /* Eq. 4-7 */
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        const int *LR = idxR + i * (int64_t)capR;
        double f[3] = {0, 0, 0}, w[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
        for (int a = 0; a < cntR[i]; ++a) {
            int64_t j = LR[a];
            int back = find_slot(idxR + j * (int64_t)capR, cntR[j], (int)i);
            if (back < 0) { bad = 1; continue; }
            const double *pij = p + 3 * (i * (int64_t)capR + a);
            const double *pji = p + 3 * (j * (int64_t)capR + back);
            double d[3]; min_image(pos, n, box, i, j, d);
            for (int x = 0; x < 3; ++x) f[x] += pij[x] - pji[x];                    /* Eq. 4-5 */
            for (int x = 0; x < 3; ++x) for (int y = 0; y < 3; ++y) w[3 * x + y] += d[x] * pji[y];   /* Eq. 6 */
        }
        if (F) for (int x = 0; x < 3; ++x) F[x * n + i] = f[x];
        if (W) for (int c = 0; c < 9; ++c) W[c * n + i] = w[c];
        if (J && vel) for (int x = 0; x < 3; ++x)                                   /* Eq. 7 */
            J[x * n + i] = w[3 * x + 0] * vel[0 * n + i] + w[3 * x + 1] * vel[1 * n + i] + w[3 * x + 2] * vel[2 * n + i];
    }
    if (!p_out) free(p);
    return bad ? -1 : 0;
}

/* Lists (brute force up to 8000 atoms, the oracle's cell list above) + orc_compute.
 * Returns 0; -1 asymmetric list; -2 capacity exceeded. */
int orc_evaluate(int64_t n, const double *pos, const double *vel, const int *type, const double *box,
                 const orc_hyper *h, const int *znum, const double *params, int capR, int capA,
                 double *U, double *F, double *W, double *J) {
    int *cR = (int *)malloc(sizeof(int) * n), *cA = (int *)malloc(sizeof(int) * n);
    int *iR = (int *)malloc(sizeof(int) * (size_t)n * capR), *iA = (int *)malloc(sizeof(int) * (size_t)n * capA);
    int mR, mA;
    if (n <= 8000) {
        mR = orc_neighbors_brute(n, pos, box, h->rc_r, capR, cR, iR, NULL);
        mA = orc_neighbors_brute(n, pos, box, h->rc_a, capA, cA, iA, NULL);
    } else {
        mR = orc_neighbors_cell(n, pos, box, h->rc_r, capR, cR, iR, NULL);
        mA = orc_neighbors_cell(n, pos, box, h->rc_a, capA, cA, iA, NULL);
    }
    int rc = (mR > capR || mA > capA) ? -2
           : orc_compute(n, pos, vel, type, box, h, znum, params, capR, cR, iR, capA, cA, iA, U, F, W, J, NULL, NULL, NULL);
    free(cR); free(cA); free(iR); free(iA);
    return rc;
}

/*
 * Velocity-Verlet step of the HNEMD method's equations of motion:
 *   Eq. 9   F_i^ext = F_e . W_i, read as (F_i^ext)^b = sum_a F_e^a W_i^{ab}, added to F_i in both half-kicks
 *           (the only reading for which the power of the driving force is F_e . J with J = sum_i W_i . v_i of
 *           Eq. 7 -- pinned by tests/test_oracle_hnemd.py through the energy balance);
 *   Eq. 11  K(t) = sum_i W_i(0) . v_i(t), the virial-velocity correlation with a single time origin:
 *           K^a(t) = sum_i sum_b W0_i^{ab} v_i^b(t), W0 = the per-atom virial at step 0 (or the array given).
 * With Fe == NULL (or zero) this is plain NVE (BASELINE.json north_star; the paper times NVT).
 * a = F / (m * 103.642697) A/fs^2 with F in eV/A, m in amu.  Lists from scratch every step.
 * thermo[n_steps+1][5] = U_tot, K_tot, Jx, Jy, Jz at steps 0..n_steps (J with W and v at the same time level,
 * reading Q12).  pos/vel are updated in place; U,F,W,J hold the state after the last step (F = the potential
 * force of Eq. 4, without the driving force).  Jsum (nullable, [3][N]) accumulates J_i over steps 1..n_steps.
 * Kt (nullable, [n_steps+1][3]) receives K(t) at steps 0..n_steps; W0 (nullable, [9][N]) is W_i(0), default:
 * the virial of this run's step 0.  No thermostat and no total-force correction: the paper gives neither.
 */
int orc_md_driven(int64_t n, double *pos, double *vel, const int *type, const double *box,
                  const orc_hyper *h, const int *znum, const double *params, const double *mass_by_type,
                  double dt, int n_steps, int capR, int capA, const double *Fe, const double *W0, double *Kt,
                  double *U, double *F, double *W, double *J, double *Jsum, double *thermo) {
    const double conv = 103.642697;
    int rc = orc_evaluate(n, pos, vel, type, box, h, znum, params, capR, capA, U, F, W, J);
    if (rc) return rc;
    double *W0own = NULL;
    if (Kt && !W0) {
        W0own = (double *)malloc(sizeof(double) * 9 * (size_t)n);
        memcpy(W0own, W, sizeof(double) * 9 * (size_t)n);
        W0 = W0own;
    }
    double *Ft = (double *)malloc(sizeof(double) * 3 * (size_t)n);        /* F_i + F_e . W_i */
    for (int step = 0; step <= n_steps; ++step) {
        for (int64_t i = 0; i < n; ++i)
            for (int b = 0; b < 3; ++b) {
                double f = F[b * n + i];
                if (Fe) for (int a = 0; a < 3; ++a) f += Fe[a] * W[(3 * a + b) * n + i];     /* Eq. 9 */
                Ft[b * n + i] = f;
            }
        if (thermo) {
            double u = 0, k = 0, jx = 0, jy = 0, jz = 0;
            for (int64_t i = 0; i < n; ++i) {
                u += U[i];
                k += 0.5 * conv * mass_by_type[type[i]] * (vel[i] * vel[i] + vel[n + i] * vel[n + i] + vel[2 * n + i] * vel[2 * n + i]);
                jx += J[i]; jy += J[n + i]; jz += J[2 * n + i];
            }
            double *t = thermo + 5 * step; t[0] = u; t[1] = k; t[2] = jx; t[3] = jy; t[4] = jz;
        }
        if (Kt) {
            for (int a = 0; a < 3; ++a) {
                double s = 0;
                for (int64_t i = 0; i < n; ++i)
                    for (int b = 0; b < 3; ++b) s += W0[(3 * a + b) * n + i] * vel[b * n + i];   /* Eq. 11 */
                Kt[3 * step + a] = s;
            }
        }
        if (step == n_steps) break;
        for (int64_t i = 0; i < n; ++i) {
            double im = 1.0 / (mass_by_type[type[i]] * conv);
            for (int a = 0; a < 3; ++a) {
                vel[a * n + i] += 0.5 * dt * Ft[a * n + i] * im;
                pos[a * n + i] += dt * vel[a * n + i];
            }
        }
        rc = orc_evaluate(n, pos, NULL, type, box, h, znum, params, capR, capA, U, F, W, NULL);
        if (rc) break;
        for (int64_t i = 0; i < n; ++i) {
            double im = 1.0 / (mass_by_type[type[i]] * conv);
            for (int b = 0; b < 3; ++b) {
                double f = F[b * n + i];
                if (Fe) for (int a = 0; a < 3; ++a) f += Fe[a] * W[(3 * a + b) * n + i];     /* Eq. 9 */
                vel[b * n + i] += 0.5 * dt * f * im;
            }
            for (int x = 0; x < 3; ++x) {
                J[x * n + i] = W[(3 * x + 0) * n + i] * vel[i] + W[(3 * x + 1) * n + i] * vel[n + i] + W[(3 * x + 2) * n + i] * vel[2 * n + i];
                if (Jsum) Jsum[x * n + i] += J[x * n + i];
            }
        }
    }
    free(Ft); free(W0own);
    return rc;
}

/* Plain NVE: orc_md_driven without driving force (kept as the entry point the round-1 pins use). */
int orc_md(int64_t n, double *pos, double *vel, const int *type, const double *box,
           const orc_hyper *h, const int *znum, const double *params, const double *mass_by_type,
           double dt, int n_steps, int capR, int capA,
           double *U, double *F, double *W, double *J, double *Jsum, double *thermo) {
    return orc_md_driven(n, pos, vel, type, box, h, znum, params, mass_by_type, dt, n_steps, capR, capA,
                         NULL, NULL, NULL, U, F, W, J, Jsum, thermo);
}

/* ------------------------------------------------------------------------------------------------
 * Training side (Sec. II E): the loss of Eq. 29-34 over a set of structures and one
 * generation of the separable natural evolution strategy, Eq. 35-39.  Plain loops, one structure and
 * one population member at a time; "all structures concatenated" is only the layout of
 * the inputs: positions / types / forces of structure n occupy atoms first[n] .. first[n+1]-1.
 *
 * Readings (the paper is silent; Q23-Q25):
 *   Q23  "eV/atom for energy and virial": U(n) and W(n) of Eq. 30 / 32 are the structure's
 *        total energy and total virial divided by its number of atoms.
 *   Q24  the six independent components mu nu of Eq. 32 are xx, yy, zz, xy, yz, zx of the total virial.
 *   Q25  the rank-based utilities u_k are not printed ("see Ref. 44"): the standard NES choice
 *        u_k = max(0, ln(N_pop/2 + 1) - ln k) / sum_j max(0, ln(N_pop/2 + 1) - ln j) - 1/N_pop  for the member of
 *        rank k (k = 1 the smallest loss), which sums to zero.  Ties are broken by member index.
 * ------------------------------------------------------------------------------------------------ */

/* Eq. 30-34 and 29 for ONE parameter vector z.  box[S][3]; first[S+1]; pos/F_tar [3][N] concatenated; e_tar[S] per
 * atom; v_tar[S][6] per atom; lambda[5] = lambda_e, lambda_f, lambda_v, lambda_1, lambda_2.
 * out[6] = L_e, L_f, L_v, L_1, L_2, L.  Returns 0 or orc_evaluate's error. */
int orc_loss(int S, const int64_t *first, const double *pos, const int *type, const double *box,
             const orc_hyper *h, const int *znum, const double *z, int capR, int capA,
             const double *e_tar, const double *f_tar, const double *v_tar, const double *lambda, double *out) {
    const int64_t N = first[S];
    const int npar = orc_num_params(h);
    double sse_e = 0.0, sse_f = 0.0, sse_v = 0.0;
    static const int comp[6] = {0, 4, 8, 1, 5, 6};            /* xx yy zz xy yz zx of the row-major 3x3 */
    for (int n = 0; n < S; ++n) {
        const int64_t a0 = first[n], nat = first[n + 1] - a0;
        double *p = (double *)malloc(sizeof(double) * 3 * nat);
        double *U = (double *)malloc(sizeof(double) * nat), *F = (double *)malloc(sizeof(double) * 3 * nat);
        double *W = (double *)malloc(sizeof(double) * 9 * nat);
        for (int a = 0; a < 3; ++a) for (int64_t i = 0; i < nat; ++i) p[a * nat + i] = pos[a * N + a0 + i];
        int rc = orc_evaluate(nat, p, NULL, type + a0, box + 3 * n, h, znum, z, capR, capA, U, F, W, NULL);
        if (rc) { free(p); free(U); free(F); free(W); return rc; }
        double e = 0.0, w[6] = {0, 0, 0, 0, 0, 0};
        for (int64_t i = 0; i < nat; ++i) {
            e += U[i];
            for (int c = 0; c < 6; ++c) w[c] += W[comp[c] * nat + i];
            for (int a = 0; a < 3; ++a) { double df = F[a * nat + i] - f_tar[a * N + a0 + i]; sse_f += df * df; }   /* Eq. 31 */
        }
        e /= (double)nat;                                                                   /* Q23 */
        sse_e += (e - e_tar[n]) * (e - e_tar[n]);                                           /* Eq. 30 */
        for (int c = 0; c < 6; ++c) { double dv = w[c] / (double)nat - v_tar[6 * n + c]; sse_v += dv * dv; }   /* Eq. 32 */
        free(p); free(U); free(F); free(W);
    }
    double l1 = 0.0, l2 = 0.0;
    for (int k = 0; k < npar; ++k) { l1 += fabs(z[k]); l2 += z[k] * z[k]; }
    out[0] = sqrt(sse_e / S); out[1] = sqrt(sse_f / (3.0 * N)); out[2] = sqrt(sse_v / (6.0 * S));
    out[3] = l1 / npar; out[4] = sqrt(l2 / npar);                                           /* Eq. 33-34 */
    out[5] = lambda[0] * out[0] + lambda[1] * out[1] + lambda[2] * out[2] + lambda[3] * out[3] + lambda[4] * out[4];   /* Eq. 29 */
    return 0;
}

/* Eq. 35: z_k = m + s (.) r_k for the whole population; z, r [npop][npar]. */
void orc_snes_sample(int npop, int npar, const double *m, const double *s, const double *r, double *z) {
    for (int k = 0; k < npop; ++k)
        for (int n = 0; n < npar; ++n) z[(size_t)k * npar + n] = m[n] + s[n] * r[(size_t)k * npar + n];
}

/* Rank-based utilities of reading Q25: util[k] for member k given the losses.  A loss that is not finite (NaN from
 * coincident atoms, overflowing weights) counts as +infinity, so the member ranks last instead of first (Q25). */
static double orc_rank_key(double l) { return isfinite(l) ? l : INFINITY; }
void orc_snes_utilities(int npop, const double *loss, double *util) {
    double norm = 0.0;
    for (int j = 1; j <= npop; ++j) { double v = log(npop / 2.0 + 1.0) - log((double)j); norm += v > 0 ? v : 0; }
    for (int k = 0; k < npop; ++k) {
        int rank = 1;                                   /* 1 = smallest loss; ties by index */
        const double lk = orc_rank_key(loss[k]);
        for (int j = 0; j < npop; ++j) { const double lj = orc_rank_key(loss[j]); if (lj < lk || (lj == lk && j < k)) ++rank; }
        double v = log(npop / 2.0 + 1.0) - log((double)rank);
        util[k] = (v > 0 ? v : 0) / norm - 1.0 / npop;
    }
}

/* Eq. 36-39: one update of (m, s) from the population's random vectors and losses. */
void orc_snes_update(int npop, int npar, const double *r, const double *loss, double eta_m, double eta_s,
                     double *m, double *s) {
    double *u = (double *)malloc(sizeof(double) * npop);
    orc_snes_utilities(npop, loss, u);
    for (int n = 0; n < npar; ++n) {
        double gm = 0.0, gs = 0.0;
        for (int k = 0; k < npop; ++k) {
            double rk = r[(size_t)k * npar + n];
            gm += u[k] * rk;                            /* Eq. 36 */
            gs += u[k] * (rk * rk - 1.0);               /* Eq. 37 */
        }
        m[n] += eta_m * (s[n] * gm);                    /* Eq. 38 */
        s[n] *= exp(0.5 * eta_s * gs);                  /* Eq. 39 */
    }
    free(u);
}
