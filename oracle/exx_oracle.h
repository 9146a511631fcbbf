/*
 * exx_oracle.h -- CPU oracle for the exact-exchange hot path of arXiv:1712.07973.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call anything in this directory.  The CUDA library
 * (paper_1712_07973_b200/csrc) shares no code, header, table or constant generator with it.
 *
 * What it computes (plain definition, fp64, the slow obvious way -- SURVEY.md 8(c)):
 *   for every ORDERED pair (i,j):   rho_ij(r) = psi_i(r) psi_j(r)                       PAPER.md:101 Eq. 8
 *                                   V_ij = Poisson solve of rho_ij by convolution with
 *                                          the Green's function on the (padded) grid     PAPER.md:73-75 Eq. 4, :125-127
 *                                   Kpsi_i(r) -= f_j V_ij(r) psi_j(r)                   PAPER.md:67-69 Eq. 3 (sum over j)
 *                                   e_ij = dV sum_r rho_ij(r) V_ij(r);  E_x -= 1/2 f_i f_j e_ij   PAPER.md:81-82 Eq. 5
 * No i<=j shortcut, no two-in-one complex packing, no pruning of the padded transform: those are the GPU's
 * optimisations and the oracle has to be able to catch a mistake in them.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 FFT vs direct DFT; P2/P3 brute-force O(M^2) real-space
 * convolution on tiny grids (free / periodic); P4/P5 plane-wave closed forms; P6 Gaussian -> erf(r/(sqrt2 s))/r;
 * P7 symmetry invariants; P8 energy/operator consistency incl. finite differences; P9 N=1 Hartree, index-n plane;
 * P10 Table 1 pair counts; P11 apply_to (coincident sets, two-cosine closed form, linearity, symmetry); P12 apply_block
 * (union of two sets = parts + block); P13 masked apply (all-ones mask, block-diagonal mask = independent subsystems);
 * P14 periodic filter table (Coulomb table = analytic kernel, screened plane-wave closed form); P15 mixed boundary
 * conditions (direct sum with wrap-around = the FREE path with a periodic-even table; all axes periodic = the periodic
 * solver); P16 general periodic cells (full-grid filter = the folded filter for an even table; triclinic plane-wave closed
 * form; brute-force convolution with the real-space image of the table).  Parity unpinned: none.
 *
 * All pointers are HOST pointers.  Arrays are C order, psi[i][a][b][c], last index fastest.
 * Return value: 0 on success, non-zero on invalid arguments / allocation failure.
 */
#ifndef EXX_ORACLE_H
#define EXX_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct exx_oracle exx_oracle;

enum { EXX_ORACLE_PERIODIC = 0, EXX_ORACLE_FREE = 1 };

/* kernel_host: PERIODIC -> ignored (analytic 4 pi/|G|^2, G=0 -> 0); FREE -> table g[a][b][c] of n1*n2*n3 doubles,
 * Green's function at displacement (a h1, b h2, c h3); copied. */
int exx_oracle_create(exx_oracle **o, const int dims[3], const double spacing[3], int bc,
                      const double *kernel_host);
void exx_oracle_destroy(exx_oracle *o);

/* Unnormalised 1-D DFT of n interleaved complex values, in place. sign=-1: forward e^{-i..}; +1: inverse e^{+i..}. */
int exx_oracle_fft1d(int n, double *data_interleaved, int sign);

/* Transform-grid dims (n for periodic, 2n for free). */
void exx_oracle_transform_dims(const exx_oracle *o, int tdims[3]);
/* Fourier-space kernel K^ on the transform grid, interleaved complex, T1*T2*T3 values. */
int exx_oracle_get_khat(const exx_oracle *o, double *khat_interleaved);

/* One Poisson solve: V = Re IDFT3( DFT3(embed(rho)) * K^ ) / T_tot restricted to the n-grid. */
int exx_oracle_poisson(const exx_oracle *o, const double *rho, double *v);

/* Full apply.  kpsi (N*M) is OVERWRITTEN, *ex receives E_x, e_pair (N*N, may be NULL) receives e_ij.
 * symmetric=0: all N^2 ordered pairs (the definition).  symmetric=1: i<=j only, each V used for both orbitals --
 * exists to make long runs affordable and is itself validated against symmetric=0 in the tests. */
int exx_oracle_apply(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                     double *kpsi, double *ex, double *e_pair, int symmetric);

/* As exx_oracle_apply (symmetric=0) with the ordered pairs (i,j) whose mask[i*n_orb+j] == 0 left out of every sum
 * (localised orbitals, Eq. 6-7). */
int exx_oracle_apply_masked(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                            const unsigned char *mask, double *kpsi, double *ex, double *e_pair);

/* K of the occupied set (psi, occ) applied to another set: kphi[t] = - sum_j f_j V[phi_t psi_j] psi_j
 * (PAPER.md:67-69 Eq. 3; :210, :244 unoccupied states / second spin channel).  kphi (n_tgt*M) is OVERWRITTEN. */
int exx_oracle_apply_to(const exx_oracle *o, int n_occ, const double *psi, const double *occ,
                        int n_tgt, const double *phi, double *kphi);

/* All pairs between two disjoint blocks A and B (the round-robin unit of work): ka[a] = -sum_b f_b
 * V_ab psi_b, kb[b] = -sum_a f_a V_ba psi_a (both OVERWRITTEN), e_block[a][b] = e_ab (may be NULL),
 * *ex = -sum_ab f_a f_b e_ab. */
int exx_oracle_apply_block(const exx_oracle *o, int n_a, const double *psi_a, const double *occ_a, double *ka,
                           int n_b, const double *psi_b, const double *occ_b, double *kb, double *ex, double *e_block);

/* PERIODIC only: use the host table K^[s0][s1][s2] (symmetric index range s = 0..t/2 per axis, even in every index)
 * instead of 4 pi/|G|^2 (screened hybrids change only this filter). */
int exx_oracle_set_periodic_filter(exx_oracle *o, const double *table);

/* PERIODIC only, general (non-orthorhombic) cells: K^[m0][m1][m2] on the FULL transform grid (FFT index order), used as
 * is; dV is the product of the spacings given at creation (pass three equal nominal spacings cbrt(cell volume / M)). */
int exx_oracle_set_periodic_filter_full(exx_oracle *o, const double *table_full);

/* Complete rows: for each listed i, Kpsi_i (all j) into kpsi_rows[row][M] and e_ij into e_rows[row][N] (may be NULL). */
int exx_oracle_rows(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                    int n_rows, const int *rows, double *kpsi_rows, double *e_rows);

/* Sampled pair energies e_ij for listed (i,j). */
int exx_oracle_pair_energies(const exx_oracle *o, int n_orb, const double *psi,
                             int n_pairs, const int *pi, const int *pj, double *e_out);

/* Real-space kernel on the n-grid used by the direct sums below: FREE -> dV * g(|a-a'|,..) (the host table);
 * PERIODIC -> g_per(r) = (1/M) sum_G K^(G) e^{iG.r}.  n1*n2*n3 doubles. */
int exx_oracle_realspace_kernel(const exx_oracle *o, double *g_out);

/* Brute force, no FFT in the convolution: V(r) = sum_r' g(r - r') rho(r') by the O(M^2) double loop. */
int exx_oracle_poisson_direct(const exx_oracle *o, const double *rho, double *v);

/* Mixed boundary conditions (slab: two periodic axes, wire: one), the definition as an O(M^2) double loop
 * with no FFT and no handle: V(r) = dV sum_r' g(d(r,r')) rho(r'), d_a = (r_a - r'_a) mod n_a on a periodic axis (the
 * table holds one full period of the Green's function there), |r_a - r'_a| on an isolated one.  periodic[a] != 0 marks
 * a periodic axis.  The claim the product relies on -- a FREE plan given a table that is even under d -> n - d along the
 * periodic axes computes exactly this -- is pinned in tests/test_oracle_pins_ext.py (P15). */
int exx_oracle_poisson_direct_mixed(const int dims[3], const double spacing[3], const int periodic[3],
                                    const double *table, const double *rho, double *v);

/* Sampled entries of K psi by direct real-space summation, O(N*M) each:
 * out[s] = - sum_j f_j psi_j(r_s) sum_r' g(r_s - r') psi_i(r') psi_j(r'),  i = orb[s], r_s = flat index point[s]. */
int exx_oracle_kpsi_points(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                           int n_samples, const int *orb, const long long *point, double *out);

/* Threads the last parallel call used (OpenMP), for the bench's "cores" field. */
int exx_oracle_threads(void);

#ifdef __cplusplus
}
#endif
#endif
