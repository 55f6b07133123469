/*
 * oracle/ani_oracle.c — fp64 CPU ORACLE for the ANI-2x-style potential of Deep-HP (arXiv 2207.14276).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code with the CUDA
 * path under paper_2207_14276_b200/csrc/ and neither includes the other.
 *
 * It evaluates the DEFINITION directly (the method is not an approximation of anything cheaper):
 *   pairs    : brute-force O(N^2) minimum-image search           PAPER.md L134 (§2.2.2), Eq. 3 "R <= Rc" (L70)
 *   f_c      : cosine cutoff                                     PAPER.md L68-73, Eq. 3
 *   radial   : sum_j exp(-eta (R_ij - R_s)^2) f_c(R_ij)           PAPER.md L75-80, Eq. 4, per neighbour species (L85)
 *   angular  : 2^(1-zeta) sum_{j<k} (1+cos(theta-theta_s))^zeta
 *              exp(-eta ((R_ij+R_ik)/2 - R_s)^2) f_c f_c          PAPER.md L82-85, Eq. 5, per species pair (L85)
 *   energy   : E = (1/M) sum_e sum_i NN_{s_i}^{(e)}(G_i)          PAPER.md L58-64, Eq. 2; ensemble L159
 *   forces   : F = -dE/dr, exact chain rule through the above
 * Readings of the points the paper leaves open are those of SURVEY.md §8(c) Q1-Q22 (listed in DESIGN.md).
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): closed-form dimer / trimer values, f_c
 * special values, 1008 feature count, scipy cKDTree pair sets, torch-autograd MLP, central finite
 * differences of E, translation / rotation / permutation invariance, sum F = 0, zero torque.
 * Parity unpinned: energies of the real (trained) ANI-2x model — no trained weights, no printed
 * energy for any structure in the paper.
 *
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (oracle/build.py).  -ffp-contract=off keeps
 * the pair predicate free of FMA contraction.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NSP 7            /* H C N O S F Cl */
#define NR 16            /* radial shifts                          */
#define NAZ 32           /* entries of one angular sub-AEV = n_a radial shifts x n_z sections: 8 x 4 for the ANI-2x shape
                            (BASELINE.json configs[0]), 4 x 8 for the ANI-1x shape (reading R4) */
#define NAMAX 8
#define NZMAX 8
#define NPAIR (NSP * (NSP + 1) / 2)
#define AEV_RAD (NSP * NR)                    /* 112 */
#define AEV_DIM (AEV_RAD + NPAIR * NAZ)       /* 1008  (N radial + N(N+1)/2 angular sub-AEVs) */
#define L0 AEV_DIM
#define L1 256
#define L2 192
#define L3 160
#define NET_PARAMS (L0 * L1 + L1 + L1 * L2 + L2 + L2 * L3 + L3 + L3 + 1)   /* 338689 */

typedef struct {
    double rcr, rca, eta_r, eta_a, zeta, alpha;
    double shf_r[NR], shf_a[NAMAX], shf_z[NZMAX];
    int n_a, n_z;            /* n_a * n_z == NAZ; layout of a sub-AEV: [a][z], index n_z * a + z */
} ora_params;

static const double ORA_PI = 3.14159265358979323846;

int ora_aev_dim(void) { return AEV_DIM; }
int ora_net_params(void) { return NET_PARAMS; }
int ora_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* upper-triangle, row-major index of the unordered species pair {u,v} */
static int pairidx(int a, int b)
{
    int u = a < b ? a : b, v = a < b ? b : a;
    return NSP * u - u * (u - 1) / 2 + (v - u);
}

/* Canonical pair predicate: fp32 inputs converted exactly to fp64,
 * minimum image by d -= L*rint(d/L), R^2 = (dx*dx + dy*dy) + dz*dz without FMA contraction. */
static double pair_r2(const float *pos, const float *box, int64_t i, int64_t j, double d[3])
{
    for (int c = 0; c < 3; ++c) {
        double x = (double)pos[3 * j + c] - (double)pos[3 * i + c];
        if (box) {
            double L = (double)box[c];
            x -= L * rint(x / L);
        }
        d[c] = x;
    }
    double xx = d[0] * d[0], yy = d[1] * d[1], zz = d[2] * d[2];
    double s = xx + yy;
    return s + zz;
}

/* Brute-force full pair list (both directions), CSR, columns ascending.  mol_id may be NULL.
 * Pass col == NULL to get the row pointer / count only.  Returns nnz, or -1 if cap is too small. */
int64_t ora_pairs(const float *pos, int64_t n, const float *box, const int32_t *mol_id, double rc,
                  int64_t *row_ptr, int32_t *col, int64_t cap)
{
    const double rc2 = rc * rc;
    int64_t *cnt = (int64_t *)calloc((size_t)n + 1, sizeof(int64_t));
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t c = 0;
        double d[3];
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            if (mol_id && mol_id[j] != mol_id[i]) continue;
            if (pair_r2(pos, box, i, j, d) <= rc2) ++c;
        }
        cnt[i] = c;
    }
    row_ptr[0] = 0;
    for (int64_t i = 0; i < n; ++i) row_ptr[i + 1] = row_ptr[i] + cnt[i];
    free(cnt);
    int64_t nnz = row_ptr[n];
    if (!col) return nnz;
    if (nnz > cap) return -1;
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t p = row_ptr[i];
        double d[3];
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            if (mol_id && mol_id[j] != mol_id[i]) continue;
            if (pair_r2(pos, box, i, j, d) <= rc2) col[p++] = (int32_t)j;
        }
    }
    return nnz;
}

/* Eq. 3: f_c(R) = 1/2 cos(pi R / Rc) + 1/2 for R <= Rc, else 0; and its derivative. */
static double fcut(double R, double Rc) { return R <= Rc ? 0.5 * cos(ORA_PI * R / Rc) + 0.5 : 0.0; }
static double dfcut(double R, double Rc) { return R <= Rc ? -0.5 * (ORA_PI / Rc) * sin(ORA_PI * R / Rc) : 0.0; }

typedef struct {
    int64_t j;
    int sp;
    double R, u[3]; /* distance and unit vector r_hat_ij = (r_j - r_i)/R */
} nbr_t;

/* All neighbours of centre i within rc (brute force over all atoms). Returns count. */
static int64_t gather_neighbours(const float *pos, const int32_t *species, int64_t n, const float *box,
                                 const int32_t *mol_id, int64_t i, double rc, nbr_t *out)
{
    const double rc2 = rc * rc;
    int64_t m = 0;
    for (int64_t j = 0; j < n; ++j) {
        if (j == i) continue;
        if (mol_id && mol_id[j] != mol_id[i]) continue;
        double d[3];
        double r2 = pair_r2(pos, box, i, j, d);
        if (r2 <= rc2) {
            double R = sqrt(r2);
            out[m].j = j;
            out[m].sp = species[j];
            out[m].R = R;
            out[m].u[0] = d[0] / R; out[m].u[1] = d[1] / R; out[m].u[2] = d[2] / R;
            ++m;
        }
    }
    return m;
}

/* G_i (Eqs. 4 and 5).  Layout (Q9): radial [s_j][m], then angular [pairidx][a][z]. */
static void aev_of(const ora_params *P, const nbr_t *nb, int64_t m, double *G)
{
    memset(G, 0, sizeof(double) * AEV_DIM);
    /* radial, Eq. 4: one sum per neighbour species */
    for (int64_t a = 0; a < m; ++a) {
        double R = nb[a].R, fc = fcut(R, P->rcr);
        for (int q = 0; q < NR; ++q) {
            double dr = R - P->shf_r[q];
            G[NR * nb[a].sp + q] += exp(-P->eta_r * dr * dr) * fc;
        }
    }
    /* angular, Eq. 5: unordered pairs {j,k}, j != k, both within Rca (Q6) */
    for (int64_t a = 0; a < m; ++a) {
        if (nb[a].R > P->rca) continue;
        for (int64_t b = a + 1; b < m; ++b) {
            if (nb[b].R > P->rca) continue;
            const double *uj = nb[a].u, *uk = nb[b].u;
            double c = uj[0] * uk[0] + uj[1] * uk[1] + uj[2] * uk[2];
            double cx = uj[1] * uk[2] - uj[2] * uk[1];
            double cy = uj[2] * uk[0] - uj[0] * uk[2];
            double cz = uj[0] * uk[1] - uj[1] * uk[0];
            double s = sqrt(cx * cx + cy * cy + cz * cz);            /* sin(theta) >= 0 */
            double fj = fcut(nb[a].R, P->rca), fk = fcut(nb[b].R, P->rca);
            double *blk = G + AEV_RAD + NAZ * pairidx(nb[a].sp, nb[b].sp);
            const int NA = P->n_a, NZ = P->n_z;
            for (int q = 0; q < NA; ++q) {
                double mm = 0.5 * (nb[a].R + nb[b].R) - P->shf_a[q];
                double B = exp(-P->eta_a * mm * mm);
                for (int z = 0; z < NZ; ++z) {
                    /* 2^(1-zeta) (1 + cos(theta - theta_z))^zeta = 2 ((1 + cos(theta-theta_z))/2)^zeta */
                    double u = 0.5 * (1.0 + c * cos(P->shf_z[z]) + s * sin(P->shf_z[z]));
                    blk[NZ * q + z] += 2.0 * pow(u, P->zeta) * B * fj * fk;
                }
            }
        }
    }
}

static double celu(double x, double a) { return x > 0.0 ? x : a * (exp(x / a) - 1.0); }
static double dcelu(double x, double a) { return x > 0.0 ? 1.0 : exp(x / a); }

/* One network (fp64 copy of the blob slice): forward, then input gradient.  Returns E_i; g = dE_i/dG. */
static double net_forward_backward(const double *w, double alpha, const double *G, double *g)
{
    const double *W1 = w, *b1 = W1 + L0 * L1, *W2 = b1 + L1, *b2 = W2 + L1 * L2, *W3 = b2 + L2,
                 *b3 = W3 + L2 * L3, *W4 = b3 + L3, *b4 = W4 + L3;
    double z1[L1], h1[L1], z2[L2], h2[L2], z3[L3], h3[L3];
    for (int o = 0; o < L1; ++o) {
        double s = b1[o];
        for (int k = 0; k < L0; ++k) s += W1[(size_t)o * L0 + k] * G[k];
        z1[o] = s; h1[o] = celu(s, alpha);
    }
    for (int o = 0; o < L2; ++o) {
        double s = b2[o];
        for (int k = 0; k < L1; ++k) s += W2[o * L1 + k] * h1[k];
        z2[o] = s; h2[o] = celu(s, alpha);
    }
    for (int o = 0; o < L3; ++o) {
        double s = b3[o];
        for (int k = 0; k < L2; ++k) s += W3[o * L2 + k] * h2[k];
        z3[o] = s; h3[o] = celu(s, alpha);
    }
    double E = b4[0];
    for (int k = 0; k < L3; ++k) E += W4[k] * h3[k];
    if (!g) return E;
    /* back-substitution: delta3 = W4^T . CELU'(z3); delta2 = (W3^T delta3) . CELU'(z2); ... g = W1^T delta1 */
    double d3[L3], d2[L2], d1[L1];
    for (int o = 0; o < L3; ++o) d3[o] = W4[o] * dcelu(z3[o], alpha);
    for (int k = 0; k < L2; ++k) {
        double s = 0.0;
        for (int o = 0; o < L3; ++o) s += W3[o * L2 + k] * d3[o];
        d2[k] = s * dcelu(z2[k], alpha);
    }
    for (int k = 0; k < L1; ++k) {
        double s = 0.0;
        for (int o = 0; o < L2; ++o) s += W2[o * L1 + k] * d2[o];
        d1[k] = s * dcelu(z1[k], alpha);
    }
    for (int k = 0; k < L0; ++k) g[k] = 0.0;
    for (int o = 0; o < L1; ++o) {           /* g[k] = sum_o W1[o][k] d1[o], o ascending */
        double d = d1[o];
        const double *row = W1 + (size_t)o * L0;
        for (int k = 0; k < L0; ++k) g[k] += row[k] * d;
    }
    return E;
}

/* AEV rows for a list of centres.  aev: [n_centres][1008]. */
void ora_aev(const float *pos, const int32_t *species, int64_t n, const float *box, const int32_t *mol_id,
             const ora_params *P, const int32_t *centres, int64_t n_centres, double *aev)
{
#pragma omp parallel
    {
        nbr_t *nb = (nbr_t *)malloc(sizeof(nbr_t) * (size_t)(n > 0 ? n : 1));
#pragma omp for schedule(dynamic, 8)
        for (int64_t c = 0; c < n_centres; ++c) {
            int64_t m = gather_neighbours(pos, species, n, box, mol_id, centres[c], P->rcr, nb);
            aev_of(P, nb, m, aev + (size_t)c * AEV_DIM);
        }
        free(nb);
    }
}

/* Network on given AEV rows (used by the MLP pins): E[c], g[c][1008] (g may be NULL); ensemble mean. */
void ora_mlp(const double *aev, const int32_t *sp, int64_t n_rows, const float *weights, int n_models,
             double alpha, double *E, double *g)
{
    size_t nw = (size_t)n_models * NSP * NET_PARAMS;
    double *w = (double *)malloc(sizeof(double) * nw);
    for (size_t t = 0; t < nw; ++t) w[t] = (double)weights[t];
#pragma omp parallel
    {
        double *ge = (double *)malloc(sizeof(double) * AEV_DIM);
#pragma omp for schedule(dynamic, 4)
        for (int64_t c = 0; c < n_rows; ++c) {
            double Ei = 0.0;
            if (g) for (int k = 0; k < AEV_DIM; ++k) g[(size_t)c * AEV_DIM + k] = 0.0;
            for (int e = 0; e < n_models; ++e) {
                const double *net = w + ((size_t)e * NSP + sp[c]) * NET_PARAMS;
                Ei += net_forward_backward(net, alpha, aev + (size_t)c * AEV_DIM, g ? ge : NULL);
                if (g) for (int k = 0; k < AEV_DIM; ++k) g[(size_t)c * AEV_DIM + k] += ge[k];
            }
            E[c] = Ei / n_models;
            if (g) for (int k = 0; k < AEV_DIM; ++k) g[(size_t)c * AEV_DIM + k] /= n_models;
        }
        free(ge);
    }
    free(w);
}

/* Forces from one centre: F_x -= g[idx] * dG[idx]/dr_x for x in {i, j, k}. */
static void centre_forces(const ora_params *P, int64_t i, const nbr_t *nb, int64_t m, const double *g, double *F)
{
    /* radial: dG/dR = t (-2 eta (R - Rs) f_c + f_c'), direction r_hat_ij */
    for (int64_t a = 0; a < m; ++a) {
        double R = nb[a].R, fc = fcut(R, P->rcr), dfc = dfcut(R, P->rcr), coef = 0.0;
        for (int q = 0; q < NR; ++q) {
            double dr = R - P->shf_r[q];
            double t = exp(-P->eta_r * dr * dr);
            coef += g[NR * nb[a].sp + q] * t * (-2.0 * P->eta_r * dr * fc + dfc);
        }
        for (int c = 0; c < 3; ++c) {
            double v = coef * nb[a].u[c];
            F[3 * nb[a].j + c] -= v;
            F[3 * i + c] += v;
        }
    }
    /* angular */
    for (int64_t a = 0; a < m; ++a) {
        if (nb[a].R > P->rca) continue;
        for (int64_t b = a + 1; b < m; ++b) {
            if (nb[b].R > P->rca) continue;
            const double *uj = nb[a].u, *uk = nb[b].u;
            double Rj = nb[a].R, Rk = nb[b].R;
            double c = uj[0] * uk[0] + uj[1] * uk[1] + uj[2] * uk[2];
            double cx = uj[1] * uk[2] - uj[2] * uk[1];
            double cy = uj[2] * uk[0] - uj[0] * uk[2];
            double cz = uj[0] * uk[1] - uj[1] * uk[0];
            double s = sqrt(cx * cx + cy * cy + cz * cz);
            double ej[3], ek[3];
            for (int q = 0; q < 3; ++q) {          /* unit vectors; d theta/d r_j = -e_j / R_ij (Q7: 0 if collinear) */
                ej[q] = s < 1e-300 ? 0.0 : (uk[q] - c * uj[q]) / s;
                ek[q] = s < 1e-300 ? 0.0 : (uj[q] - c * uk[q]) / s;
            }
            double fj = fcut(Rj, P->rca), fk = fcut(Rk, P->rca);
            double dfj = dfcut(Rj, P->rca), dfk = dfcut(Rk, P->rca);
            const double *gb = g + AEV_RAD + NAZ * pairidx(nb[a].sp, nb[b].sp);
            const int NA = P->n_a, NZ = P->n_z;
            double gj[3] = {0, 0, 0}, gk[3] = {0, 0, 0};   /* sum over (a,z) of g * grad_j, g * grad_k */
            for (int q = 0; q < NA; ++q) {
                double mm = 0.5 * (Rj + Rk) - P->shf_a[q];
                double B = exp(-P->eta_a * mm * mm);
                double dB = -P->eta_a * mm * B;      /* dB/dR_ij = dB/dR_ik */
                for (int z = 0; z < NZ; ++z) {
                    double cz_ = cos(P->shf_z[z]), sz_ = sin(P->shf_z[z]);
                    double u = 0.5 * (1.0 + c * cz_ + s * sz_);
                    double A = 2.0 * pow(u, P->zeta);
                    double At = -P->zeta * pow(u, P->zeta - 1.0) * (s * cz_ - c * sz_);   /* dA/dtheta */
                    double gg = gb[NZ * q + z];
                    double tj = -At * B * fj * fk / Rj, rj = A * (dB * fj + B * dfj) * fk;
                    double tk = -At * B * fj * fk / Rk, rk = A * (dB * fk + B * dfk) * fj;
                    for (int x = 0; x < 3; ++x) {
                        gj[x] += gg * (tj * ej[x] + rj * uj[x]);
                        gk[x] += gg * (tk * ek[x] + rk * uk[x]);
                    }
                }
            }
            for (int x = 0; x < 3; ++x) {
                F[3 * nb[a].j + x] -= gj[x];
                F[3 * nb[b].j + x] -= gk[x];
                F[3 * i + x] += gj[x] + gk[x];
            }
        }
    }
}

/* Energies of the listed centres and the forces THEY exert on every atom.
 *   E_atom [n_centres]   ensemble-mean atomic energies (Eq. 2 summands)
 *   F      [n][3]        F = -sum_{c in centres} dE_c/dr   (zeroed here)
 *   dEdG   [n_centres][1008] or NULL
 * With centres = all atoms, sum(E_atom) and F are the total energy and the forces. */
void ora_energy_forces(const float *pos, const int32_t *species, int64_t n, const float *box,
                       const int32_t *mol_id, const ora_params *P, const float *weights, int n_models,
                       const int32_t *centres, int64_t n_centres, double *E_atom, double *F, double *dEdG)
{
    size_t nw = (size_t)n_models * NSP * NET_PARAMS;
    double *w = (double *)malloc(sizeof(double) * nw);
    for (size_t t = 0; t < nw; ++t) w[t] = (double)weights[t];
    for (int64_t t = 0; t < 3 * n; ++t) F[t] = 0.0;
#pragma omp parallel
    {
        nbr_t *nb = (nbr_t *)malloc(sizeof(nbr_t) * (size_t)(n > 0 ? n : 1));
        double *Fp = (double *)calloc((size_t)(3 * n + 1), sizeof(double));
        double G[AEV_DIM], g[AEV_DIM], ge[AEV_DIM];
#pragma omp for schedule(dynamic, 4)
        for (int64_t c = 0; c < n_centres; ++c) {
            int64_t i = centres[c];
            int64_t m = gather_neighbours(pos, species, n, box, mol_id, i, P->rcr, nb);
            aev_of(P, nb, m, G);
            double Ei = 0.0;
            for (int k = 0; k < AEV_DIM; ++k) g[k] = 0.0;
            for (int e = 0; e < n_models; ++e) {
                const double *net = w + ((size_t)e * NSP + species[i]) * NET_PARAMS;
                Ei += net_forward_backward(net, P->alpha, G, ge);
                for (int k = 0; k < AEV_DIM; ++k) g[k] += ge[k];
            }
            for (int k = 0; k < AEV_DIM; ++k) g[k] /= n_models;
            E_atom[c] = Ei / n_models;
            if (dEdG) memcpy(dEdG + (size_t)c * AEV_DIM, g, sizeof(double) * AEV_DIM);
            centre_forces(P, i, nb, m, g, Fp);
        }
#pragma omp critical
        for (int64_t t = 0; t < 3 * n; ++t) F[t] += Fp[t];
        free(Fp);
        free(nb);
    }
    free(w);
}
