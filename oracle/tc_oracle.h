/*
 * tc_oracle.h -- CPU ORACLE for the closed-shell (T) energy.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, obviously-correct restatement of eqs. (1)-(5) of
 * arxiv 2512.01055 as explicit nested loops in FP64.
 * It shares no code with the CUDA path (paper_2512_01055_b200/csrc) and is
 * imported only by tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs.
 *
 * Index pattern (BASELINE.json north_star):
 *   A_ijk^abc = sum_d t_ij^ad (bd|ck) - sum_l t_il^ab (lj|kc)
 *   W_ijk^abc = A_ijk^abc + A_ikj^acb + A_jik^bac + A_jki^bca + A_kij^cab + A_kji^cba   (eq. (5))
 *   Vd        = t_i^a (jb|kc) + t_j^b (ia|kc) + t_k^c (ia|jb)                             (eq. (3))
 *   Y = W + Vd,   D = e_i+e_j+e_k-e_a-e_b-e_c   (Fig. 4 line 23; reading 1 of DESIGN.md)
 *   R_abc = 4W_abc + W_bca + W_cab - 2W_acb - 2W_cba - 2W_bac                             (eq. (1))
 *   S_ijk = sum_abc Y_abc R_abc / D_abc
 *   E = sum_{i>=j>=k} (2 - d_ij - d_jk) S_ijk      =  (1/3) sum_{ijk} S_ijk
 *
 * Parity pins (tests/test_oracle_pins.py): P1-P10 of SURVEY.md section 8(c).  Every
 * function below is pinned by at least one of them; none is "parity unpinned".
 *
 * Array layouts (C order, doubles):
 *   t1[i][a]; t2[i][j][a][b] = t_ij^ab
 *   vvvo[x][d][b][c] = (bd|cx);  ovoo[j][k][l][c] = (lj|kc);  ovov[j][k][b][c] = (jb|kc)
 *   Boo[Q][i][j], Bov[Q][i][a], Bvv[Q][a][b]   with (pq|rs) = sum_Q B^Q_pq B^Q_rs (eq. (6))
 */
#ifndef TC_ORACLE_H
#define TC_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* Linear triplet index idx(i,j,k) = i(i+1)(i+2)/6 + j(j+1)/2 + k, i>=j>=k>=0. */
long long tco_triplet_count(int o);
int tco_triplet_decode(int o, long long idx, int* i, int* j, int* k, double* weight);

/* W_ijk^abc for one (i,j,k), any order of i,j,k.  W[a][b][c], v^3 doubles.
 * I_i, I_j, I_k: the three slices vvvo[x] (each v^3). */
void tco_W_triplet(int o, int v, int i, int j, int k,
                   const double* t2, const double* I_i, const double* I_j, const double* I_k,
                   const double* ovoo, double* W);

/* S_ijk from a finished W (adds Vd, divides by D, applies the eq. (1) weights).
 * If Y_out != NULL it receives Y = W + Vd (v^3). */
double tco_S_from_W(int o, int v, int i, int j, int k,
                    const double* eps_occ, const double* eps_vir,
                    const double* t1, const double* ovov, const double* W, double* Y_out);

/* The same sum restricted to the points (a,b,c) of one orbit of virtual tiles: tile indices (a/T, b/T, c/T) sorted in
 * descending order equal to (A,B,C) (the abcijk scheme of the paper tiles the virtual indices, Fig. 1).
 * Pinned by: the restricted sums over all orbits A>=B>=C add up to tco_S_from_W; a numpy mask over Y R / D on tiny inputs. */
double tco_S_from_W_tile_orbit(int o, int v, int i, int j, int k,
                               const double* eps_occ, const double* eps_vir,
                               const double* t1, const double* ovov, const double* W,
                               int T, int A, int B, int C);

/* S_ijk for the triplets first..first+count-1 of the linear index (i>=j>=k),
 * and E_partial = sum w_ijk S_ijk over that range.  S_out may be NULL. */
int tco_triples_energy_blocks(int o, int v,
                              const double* eps_occ, const double* eps_vir,
                              const double* t1, const double* t2,
                              const double* vvvo, const double* ovoo, const double* ovov,
                              long long first, long long count,
                              double* S_out, double* E_out);

/* Same, with the three (vv|v.) slices of each triplet supplied through a callback-free
 * interface: slices[x] may be NULL for occupied indices not touched by the range. */
int tco_triples_energy_slices(int o, int v,
                              const double* eps_occ, const double* eps_vir,
                              const double* t1, const double* t2,
                              const double* const* slices, const double* ovoo, const double* ovov,
                              long long first, long long count,
                              double* S_out, double* E_out);

/* Unrestricted brute force: E = (1/3) sum over ALL ordered (i,j,k) of S_ijk. */
int tco_triples_energy_bruteforce(int o, int v,
                                  const double* eps_occ, const double* eps_vir,
                                  const double* t1, const double* t2,
                                  const double* vvvo, const double* ovoo, const double* ovov,
                                  double* E_out);

/* Integral blocks from DF factors by plain loops (eq. (6)). */
void tco_build_vvvo_slice(int o, int v, int naux, int x,
                          const double* Bov, const double* Bvv, double* I_x);
void tco_build_ovoo(int o, int v, int naux, const double* Boo, const double* Bov, double* ovoo);
void tco_build_ovov(int o, int v, int naux, const double* Bov, double* ovov);

/* Number of OpenMP threads the loops will use. */
int tco_num_threads(void);

#ifdef __cplusplus
}
#endif
#endif
