/*
 * tc_oracle.c -- CPU ORACLE for the closed-shell (T) energy.  TEST INFRASTRUCTURE ONLY.
 * See tc_oracle.h for the equations, citations and layouts.
 *
 * Everything here is the plain definition written out: one loop per index,
 * one statement per term of eqs. (1)-(5) of PAPER.md:33-53, FP64 throughout.
 * OpenMP is used only to run independent (a) rows / independent triplets on
 * several cores; no blocking, fusion or reordering of the arithmetic of an
 * element.  No code is shared with the CUDA path.
 */
#include "tc_oracle.h"

#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

int tco_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---- triplet index: idx = i(i+1)(i+2)/6 + j(j+1)/2 + k ---- */

long long tco_triplet_count(int o) {
    long long n = o;
    return n * (n + 1) * (n + 2) / 6;
}

int tco_triplet_decode(int o, long long idx, int* pi, int* pj, int* pk, double* weight) {
    if (o < 1 || idx < 0 || idx >= tco_triplet_count(o)) return 1;
    /* plain search: largest i with i(i+1)(i+2)/6 <= idx, then largest j with j(j+1)/2 <= rest */
    int i = 0;
    while ((long long)(i + 1) * (i + 2) * (i + 3) / 6 <= idx) i++;
    long long rest = idx - (long long)i * (i + 1) * (i + 2) / 6;
    int j = 0;
    while ((long long)(j + 1) * (j + 2) / 2 <= rest) j++;
    int k = (int)(rest - (long long)j * (j + 1) / 2);
    *pi = i; *pj = j; *pk = k;
    if (weight) *weight = 2.0 - (i == j ? 1.0 : 0.0) - (j == k ? 1.0 : 0.0);   /* eq. (1): 2 - d_ij - d_jk */
    return 0;
}

/* ---- element accessors: one per array, spelling out the layout ---- */

static inline double T2(const double* t2, int o, int v, int i, int j, int a, int b) {
    return t2[(((size_t)i * o + j) * v + a) * v + b];                    /* t_ij^ab */
}
/* (bd|cx) from slice I_x[d][b][c] */
static inline double VVVO(const double* I_x, int v, int b, int d, int c) {
    return I_x[((size_t)d * v + b) * v + c];
}
/* (lj|kc) = ovoo[j][k][l][c] */
static inline double OVOO(const double* ovoo, int o, int v, int l, int j, int k, int c) {
    return ovoo[(((size_t)j * o + k) * o + l) * v + c];
}
/* (jb|kc) = ovov[j][k][b][c] */
static inline double OVOV(const double* ovov, int o, int v, int j, int b, int k, int c) {
    return ovov[(((size_t)j * o + k) * v + b) * v + c];
}

/* ---- W_ijk^abc, eq. (2)+(5) in the north_star index pattern ---- */

void tco_W_triplet(int o, int v, int i, int j, int k,
                   const double* t2, const double* I_i, const double* I_j, const double* I_k,
                   const double* ovoo, double* W) {
    /* One loop nest per row of the table in SURVEY.md section 8(c) step 2; every nest
     * adds its term into W[a][b][c].  The summed index (d or l) sits between a and (b,c)
     * only so that the innermost accesses are mostly contiguous; each element still
     * receives its terms in table order with d (l) ascending. */
#pragma omp parallel for schedule(static)
    for (int a = 0; a < v; a++) {
        double* Wa = W + (size_t)a * v * v;
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] = 0.0;

        /* ijk/abc:  + sum_d t_ij^ad (bd|ck) */
        for (int d = 0; d < v; d++) {
            const double t = T2(t2, o, v, i, j, a, d);
            for (int b = 0; b < v; b++)
                for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] += t * VVVO(I_k, v, b, d, c);
        }
        /* ikj/acb:  + sum_d t_ik^ad (cd|bj) */
        for (int d = 0; d < v; d++) {
            const double t = T2(t2, o, v, i, k, a, d);
            for (int b = 0; b < v; b++)
                for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] += t * VVVO(I_j, v, c, d, b);
        }
        /* jik/bac:  + sum_d t_ji^bd (ad|ck) */
        for (int d = 0; d < v; d++)
            for (int b = 0; b < v; b++) {
                const double t = T2(t2, o, v, j, i, b, d);
                for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] += t * VVVO(I_k, v, a, d, c);
            }
        /* jki/bca:  + sum_d t_jk^bd (cd|ai) */
        for (int d = 0; d < v; d++)
            for (int b = 0; b < v; b++) {
                const double t = T2(t2, o, v, j, k, b, d);
                for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] += t * VVVO(I_i, v, c, d, a);
            }
        /* kij/cab:  + sum_d t_ki^cd (ad|bj) */
        for (int d = 0; d < v; d++)
            for (int b = 0; b < v; b++) {
                const double g = VVVO(I_j, v, a, d, b);
                for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] += T2(t2, o, v, k, i, c, d) * g;
            }
        /* kji/cba:  + sum_d t_kj^cd (bd|ai) */
        for (int d = 0; d < v; d++)
            for (int b = 0; b < v; b++) {
                const double g = VVVO(I_i, v, b, d, a);
                for (int c = 0; c < v; c++) Wa[(size_t)b * v + c] += T2(t2, o, v, k, j, c, d) * g;
            }

        /* hole terms:  - sum_l t_xl^{pq} (ly|zr) */
        for (int l = 0; l < o; l++)
            for (int b = 0; b < v; b++)
                for (int c = 0; c < v; c++) {
                    double h = 0.0;
                    h += T2(t2, o, v, i, l, a, b) * OVOO(ovoo, o, v, l, j, k, c);   /* t_il^ab (lj|kc) */
                    h += T2(t2, o, v, i, l, a, c) * OVOO(ovoo, o, v, l, k, j, b);   /* t_il^ac (lk|jb) */
                    h += T2(t2, o, v, j, l, b, a) * OVOO(ovoo, o, v, l, i, k, c);   /* t_jl^ba (li|kc) */
                    h += T2(t2, o, v, j, l, b, c) * OVOO(ovoo, o, v, l, k, i, a);   /* t_jl^bc (lk|ia) */
                    h += T2(t2, o, v, k, l, c, a) * OVOO(ovoo, o, v, l, i, j, b);   /* t_kl^ca (li|jb) */
                    h += T2(t2, o, v, k, l, c, b) * OVOO(ovoo, o, v, l, j, i, a);   /* t_kl^cb (lj|ia) */
                    Wa[(size_t)b * v + c] -= h;
                }
    }
}

/* ---- S_ijk = sum_abc Y R / D  (eqs. (1), (3), (4)) ---- */

double tco_S_from_W(int o, int v, int i, int j, int k,
                    const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* ovov, const double* W, double* Y_out) {
    double S = 0.0;
    const double eo = eps_occ[i] + eps_occ[j] + eps_occ[k];
#define W_(a, b, c) W[((size_t)(a) * v + (b)) * v + (c)]
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++) {
                /* eq. (3): Vd = t_i^a (jb|kc) + t_j^b (ia|kc) + t_k^c (ia|jb) */
                double Vd = t1[(size_t)i * v + a] * OVOV(ovov, o, v, j, b, k, c)
                          + t1[(size_t)j * v + b] * OVOV(ovov, o, v, i, a, k, c)
                          + t1[(size_t)k * v + c] * OVOV(ovov, o, v, i, a, j, b);
                double Y = W_(a, b, c) + Vd;
                /* D = e_i + e_j + e_k - e_a - e_b - e_c (Fig. 4 line 23) */
                double D = eo - eps_vir[a] - eps_vir[b] - eps_vir[c];
                /* eq. (1) weights, virtual-index form */
                double R = 4.0 * W_(a, b, c) + W_(b, c, a) + W_(c, a, b)
                         - 2.0 * W_(a, c, b) - 2.0 * W_(c, b, a) - 2.0 * W_(b, a, c);
                S += Y * R / D;
                if (Y_out) Y_out[((size_t)a * v + b) * v + c] = Y;
            }
#undef W_
    return S;
}

/* ---- the same sum restricted to one orbit of virtual tiles (the paper's abcijk scheme loops over tiles of the virtual
 *      indices, Fig. 1): only the points (a,b,c) whose tile indices (a/T, b/T, c/T), sorted in descending order,
 *      equal (A,B,C).  The orbits partition the abc cube, so the restricted sums add up to tco_S_from_W. ---- */

double tco_S_from_W_tile_orbit(int o, int v, int i, int j, int k,
                               const double* eps_occ, const double* eps_vir,
                               const double* t1, const double* ovov, const double* W,
                               int T, int A, int B, int C) {
    double S = 0.0;
    const double eo = eps_occ[i] + eps_occ[j] + eps_occ[k];
#define W_(a, b, c) W[((size_t)(a) * v + (b)) * v + (c)]
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++) {
                int hi = a / T, mid = b / T, lo = c / T, tmp;       /* sort the three tile indices, descending */
                if (hi < mid) { tmp = hi; hi = mid; mid = tmp; }
                if (mid < lo) { tmp = mid; mid = lo; lo = tmp; }
                if (hi < mid) { tmp = hi; hi = mid; mid = tmp; }
                if (hi != A || mid != B || lo != C) continue;
                double Vd = t1[(size_t)i * v + a] * OVOV(ovov, o, v, j, b, k, c)
                          + t1[(size_t)j * v + b] * OVOV(ovov, o, v, i, a, k, c)
                          + t1[(size_t)k * v + c] * OVOV(ovov, o, v, i, a, j, b);
                double Y = W_(a, b, c) + Vd;
                double D = eo - eps_vir[a] - eps_vir[b] - eps_vir[c];
                double R = 4.0 * W_(a, b, c) + W_(b, c, a) + W_(c, a, b)
                         - 2.0 * W_(a, c, b) - 2.0 * W_(c, b, a) - 2.0 * W_(b, a, c);
                S += Y * R / D;
            }
#undef W_
    return S;
}

/* ---- energy over a range of the linear triplet index ---- */

int tco_triples_energy_slices(int o, int v,
                              const double* eps_occ, const double* eps_vir,
                              const double* t1, const double* t2,
                              const double* const* slices, const double* ovoo, const double* ovov,
                              long long first, long long count,
                              double* S_out, double* E_out) {
    if (o < 1 || v < 1 || first < 0 || count < 0 || first + count > tco_triplet_count(o)) return 1;
    double* W = (double*)malloc(sizeof(double) * (size_t)v * v * v);
    if (!W) return 2;
    double E = 0.0;
    for (long long n = 0; n < count; n++) {
        int i, j, k; double w;
        tco_triplet_decode(o, first + n, &i, &j, &k, &w);
        if (!slices[i] || !slices[j] || !slices[k]) { free(W); return 3; }
        tco_W_triplet(o, v, i, j, k, t2, slices[i], slices[j], slices[k], ovoo, W);
        double S = tco_S_from_W(o, v, i, j, k, eps_occ, eps_vir, t1, ovov, W, NULL);
        if (S_out) S_out[n] = S;
        E += w * S;
    }
    free(W);
    if (E_out) *E_out = E;
    return 0;
}

int tco_triples_energy_blocks(int o, int v,
                              const double* eps_occ, const double* eps_vir,
                              const double* t1, const double* t2,
                              const double* vvvo, const double* ovoo, const double* ovov,
                              long long first, long long count,
                              double* S_out, double* E_out) {
    if (o < 1 || v < 1) return 1;
    const double** slices = (const double**)malloc(sizeof(double*) * (size_t)o);
    if (!slices) return 2;
    for (int x = 0; x < o; x++) slices[x] = vvvo + (size_t)x * v * v * v;
    int rc = tco_triples_energy_slices(o, v, eps_occ, eps_vir, t1, t2, slices, ovoo, ovov,
                                       first, count, S_out, E_out);
    free((void*)slices);
    return rc;
}

/* ---- unrestricted brute force: (1/3) sum over all o^3 ordered (i,j,k) ---- */

int tco_triples_energy_bruteforce(int o, int v,
                                  const double* eps_occ, const double* eps_vir,
                                  const double* t1, const double* t2,
                                  const double* vvvo, const double* ovoo, const double* ovov,
                                  double* E_out) {
    if (o < 1 || v < 1) return 1;
    const size_t v3 = (size_t)v * v * v;
    double* W = (double*)malloc(sizeof(double) * v3);
    if (!W) return 2;
    double E = 0.0;
    for (int i = 0; i < o; i++)
        for (int j = 0; j < o; j++)
            for (int k = 0; k < o; k++) {
                tco_W_triplet(o, v, i, j, k, t2, vvvo + i * v3, vvvo + j * v3, vvvo + k * v3, ovoo, W);
                E += tco_S_from_W(o, v, i, j, k, eps_occ, eps_vir, t1, ovov, W, NULL);
            }
    free(W);
    *E_out = E / 3.0;
    return 0;
}

/* ---- integrals from DF factors, eq. (6): (pq|rs) = sum_Q B^Q_pq B^Q_rs ---- */

void tco_build_vvvo_slice(int o, int v, int naux, int x,
                          const double* Bov, const double* Bvv, double* I_x) {
#pragma omp parallel for schedule(static)
    for (int d = 0; d < v; d++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++) {
                double s = 0.0;
                for (int Q = 0; Q < naux; Q++)        /* (bd|cx) = sum_Q B^Q_bd B^Q_xc */
                    s += Bvv[((size_t)Q * v + b) * v + d] * Bov[((size_t)Q * o + x) * v + c];
                I_x[((size_t)d * v + b) * v + c] = s;
            }
}

void tco_build_ovoo(int o, int v, int naux, const double* Boo, const double* Bov, double* ovoo) {
    for (int j = 0; j < o; j++)
        for (int k = 0; k < o; k++)
            for (int l = 0; l < o; l++)
                for (int c = 0; c < v; c++) {
                    double s = 0.0;
                    for (int Q = 0; Q < naux; Q++)    /* (lj|kc) = sum_Q B^Q_lj B^Q_kc */
                        s += Boo[((size_t)Q * o + l) * o + j] * Bov[((size_t)Q * o + k) * v + c];
                    ovoo[(((size_t)j * o + k) * o + l) * v + c] = s;
                }
}

void tco_build_ovov(int o, int v, int naux, const double* Bov, double* ovov) {
    for (int j = 0; j < o; j++)
        for (int k = 0; k < o; k++)
            for (int b = 0; b < v; b++)
                for (int c = 0; c < v; c++) {
                    double s = 0.0;
                    for (int Q = 0; Q < naux; Q++)    /* (jb|kc) = sum_Q B^Q_jb B^Q_kc */
                        s += Bov[((size_t)Q * o + j) * v + b] * Bov[((size_t)Q * o + k) * v + c];
                    ovov[(((size_t)j * o + k) * v + b) * v + c] = s;
                }
}
