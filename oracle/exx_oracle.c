/*
 * exx_oracle.c -- plain fp64 CPU oracle for the exact-exchange hot path (see exx_oracle.h for scope and pins).
 *
 * TEST INFRASTRUCTURE: never linked into, imported by, or called from the CUDA product path.
 * Every function cites the passage of /root/reference/PAPER.md (arXiv:1712.07973) or the SURVEY.md 8(c)
 * reading it follows.  Deliberately un-clever: own recursive mixed-radix FFT, N^2 ordered pairs, full
 * padded transforms, one real co-density per complex transform.
 */
#include "exx_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double re, im; } cplx;

struct exx_oracle {
    int n[3];          /* orbital grid                                             */
    int t[3];          /* transform grid: n (periodic) or 2n (free)  */
    double h[3];
    double dV;
    int bc;
    long long M, T;    /* points of the n-grid / transform grid                    */
    cplx *khat;        /* Fourier-space kernel on the transform grid               */
    double *gtab;      /* FREE: copy of the host table g[a][b][c]; PERIODIC: NULL  */
    cplx *roots[3];    /* roots[ax][j] = exp(-2 pi i j / t[ax])                    */
};

static int g_threads_used = 1;

/* ---------------------------------------------------------------------------------------------------
 * 1-D FFT: recursive mixed radix, split on the smallest prime factor, O(n^2) direct DFT for prime n,
 * twiddles from long double sin/cos.  Unnormalised; sign=-1 forward e^{-i...}.
 * ------------------------------------------------------------------------------------------------- */
static cplx *make_roots(int n)
{
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!w) return NULL;
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int j = 0; j < n; ++j) {
        long double ang = two_pi * (long double)j / (long double)n;
        w[j].re = (double)cosl(ang);
        w[j].im = (double)(-sinl(ang));
    }
    return w;
}

static int smallest_prime_factor(int n)
{
    for (int p = 2; (long long)p * p <= n; ++p)
        if (n % p == 0) return p;
    return n;
}

/* W_n^x with roots of the root length n0 (n divides n0); sign=+1 conjugates. */
static inline cplx root_pow(const cplx *roots, int n0, int n, long long x, int sign)
{
    long long idx = (x % n) * (n0 / n);
    cplx w = roots[idx];
    if (sign > 0) w.im = -w.im;
    return w;
}

static inline cplx cmul(cplx a, cplx b)
{
    cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re };
    return r;
}

static void fft_rec(int n, const cplx *in, long long is, cplx *out, const cplx *roots, int n0, int sign,
                    cplx *tmp /* at least n entries, only used at this level */)
{
    if (n == 1) { out[0] = in[0]; return; }
    int p = smallest_prime_factor(n);
    if (p == n) {                                  /* prime length: X[k] = sum_j x[j] W_n^{jk} */
        for (int k = 0; k < n; ++k) {
            double sr = 0.0, si = 0.0;
            for (int j = 0; j < n; ++j) {
                cplx w = root_pow(roots, n0, n, (long long)j * k, sign);
                cplx v = cmul(in[j * is], w);
                sr += v.re; si += v.im;
            }
            out[k].re = sr; out[k].im = si;
        }
        return;
    }
    int m = n / p;
    /* p sub-transforms of the decimated sequences x[p j + r] */
    for (int r = 0; r < p; ++r)
        fft_rec(m, in + r * is, is * p, out + (long long)r * m, roots, n0, sign, tmp);
    /* combine: X[k + q m] = sum_r W_n^{r (k + q m)} Y_r[k] */
    for (int k = 0; k < m; ++k) {
        for (int r = 0; r < p; ++r) tmp[r] = out[(long long)r * m + k];
        for (int q = 0; q < p; ++q) {
            double sr = 0.0, si = 0.0;
            for (int r = 0; r < p; ++r) {
                cplx w = root_pow(roots, n0, n, (long long)r * (k + (long long)q * m), sign);
                cplx v = cmul(tmp[r], w);
                sr += v.re; si += v.im;
            }
            out[k + (long long)q * m].re = sr;
            out[k + (long long)q * m].im = si;
        }
    }
}

int exx_oracle_fft1d(int n, double *data, int sign)
{
    if (n <= 0 || !data || (sign != 1 && sign != -1)) return 1;
    cplx *roots = make_roots(n);
    cplx *out = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!roots || !out || !tmp) { free(roots); free(out); free(tmp); return 2; }
    fft_rec(n, (const cplx *)data, 1, out, roots, n, sign, tmp);
    memcpy(data, out, sizeof(cplx) * (size_t)n);
    free(roots); free(out); free(tmp);
    return 0;
}

/* 3-D DFT on the transform grid: three nested passes of the 1-D FFT, one axis at a time. */
static int dft3(const exx_oracle *o, cplx *f, int sign)
{
    const int t0 = o->t[0], t1 = o->t[1], t2 = o->t[2];
    int tmax = t0 > t1 ? t0 : t1; if (t2 > tmax) tmax = t2;
    cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)tmax * 3);
    if (!line) return 2;
    cplx *res = line + tmax, *tmp = line + 2 * tmax;
    /* axis 2 (contiguous) */
    for (long long ab = 0; ab < (long long)t0 * t1; ++ab) {
        cplx *p = f + ab * t2;
        fft_rec(t2, p, 1, res, o->roots[2], t2, sign, tmp);
        memcpy(p, res, sizeof(cplx) * (size_t)t2);
    }
    /* axis 1 */
    for (int a = 0; a < t0; ++a)
        for (int c = 0; c < t2; ++c) {
            cplx *p = f + (long long)a * t1 * t2 + c;
            for (int b = 0; b < t1; ++b) line[b] = p[(long long)b * t2];
            fft_rec(t1, line, 1, res, o->roots[1], t1, sign, tmp);
            for (int b = 0; b < t1; ++b) p[(long long)b * t2] = res[b];
        }
    /* axis 0 */
    for (long long bc = 0; bc < (long long)t1 * t2; ++bc) {
        cplx *p = f + bc;
        for (int a = 0; a < t0; ++a) line[a] = p[(long long)a * t1 * t2];
        fft_rec(t0, line, 1, res, o->roots[0], t0, sign, tmp);
        for (int a = 0; a < t0; ++a) p[(long long)a * t1 * t2] = res[a];
    }
    free(line);
    return 0;
}

/* ---------------------------------------------------------------------------------------------------
 * Fourier-space kernel ("Green's function ... free ... and periodic").
 * ------------------------------------------------------------------------------------------------- */
static int build_khat(exx_oracle *o, const double *g)
{
    const int t0 = o->t[0], t1 = o->t[1], t2 = o->t[2];
    const double pi = 3.14159265358979323846;
    if (o->bc == EXX_ORACLE_PERIODIC) {
        /* index a -> m = a if 2a <= t else a - t;  G = 2 pi m / (t h);  K^ = 4 pi / |G|^2;  K^(0) = 0 (A6, A19) */
        for (int a = 0; a < t0; ++a) {
            int ma = (2 * a <= t0) ? a : a - t0;
            double ga = 2.0 * pi * ma / (t0 * o->h[0]);
            for (int b = 0; b < t1; ++b) {
                int mb = (2 * b <= t1) ? b : b - t1;
                double gb = 2.0 * pi * mb / (t1 * o->h[1]);
                for (int c = 0; c < t2; ++c) {
                    int mc = (2 * c <= t2) ? c : c - t2;
                    double gc = 2.0 * pi * mc / (t2 * o->h[2]);
                    double g2 = ga * ga + gb * gb + gc * gc;
                    cplx *k = &o->khat[((long long)a * t1 + b) * t2 + c];
                    k->re = (a == 0 && b == 0 && c == 0) ? 0.0 : 4.0 * pi / g2;
                    k->im = 0.0;
                }
            }
        }
        return 0;
    }
    /* FREE: g_ext[a][b][c] = g[min(a,2n1-a)][min(b,2n2-b)][min(c,2n3-c)], any index equal to n -> 0 (A8);
     * K^ = dV * DFT3(g_ext), kept complex (its imaginary part is rounding noise). */
    const int n0 = o->n[0], n1 = o->n[1], n2 = o->n[2];
    for (int a = 0; a < t0; ++a) {
        int ia = a < t0 - a ? a : t0 - a;
        for (int b = 0; b < t1; ++b) {
            int ib = b < t1 - b ? b : t1 - b;
            for (int c = 0; c < t2; ++c) {
                int ic = c < t2 - c ? c : t2 - c;
                cplx *k = &o->khat[((long long)a * t1 + b) * t2 + c];
                k->im = 0.0;
                if (ia == n0 || ib == n1 || ic == n2) k->re = 0.0;
                else k->re = g[((long long)ia * n1 + ib) * n2 + ic];
            }
        }
    }
    int rc = dft3(o, o->khat, -1);
    if (rc) return rc;
    for (long long x = 0; x < o->T; ++x) { o->khat[x].re *= o->dV; o->khat[x].im *= o->dV; }
    return 0;
}

int exx_oracle_create(exx_oracle **out, const int dims[3], const double spacing[3], int bc, const double *kernel_host)
{
    if (!out || !dims || !spacing) return 1;
    if (bc != EXX_ORACLE_PERIODIC && bc != EXX_ORACLE_FREE) return 1;
    if (bc == EXX_ORACLE_FREE && !kernel_host) return 1;
    for (int ax = 0; ax < 3; ++ax) if (dims[ax] <= 0 || !(spacing[ax] > 0.0)) return 1;
    exx_oracle *o = (exx_oracle *)calloc(1, sizeof(*o));
    if (!o) return 2;
    o->bc = bc;
    o->dV = 1.0; o->M = 1; o->T = 1;
    for (int ax = 0; ax < 3; ++ax) {
        o->n[ax] = dims[ax];
        o->t[ax] = (bc == EXX_ORACLE_FREE) ? 2 * dims[ax] : dims[ax];
        o->h[ax] = spacing[ax];
        o->dV *= spacing[ax];
        o->M *= o->n[ax];
        o->T *= o->t[ax];
        o->roots[ax] = make_roots(o->t[ax]);
        if (!o->roots[ax]) { exx_oracle_destroy(o); return 2; }
    }
    o->khat = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
    if (!o->khat) { exx_oracle_destroy(o); return 2; }
    if (bc == EXX_ORACLE_FREE) {
        o->gtab = (double *)malloc(sizeof(double) * (size_t)o->M);
        if (!o->gtab) { exx_oracle_destroy(o); return 2; }
        memcpy(o->gtab, kernel_host, sizeof(double) * (size_t)o->M);
    }
    int rc = build_khat(o, o->gtab);
    if (rc) { exx_oracle_destroy(o); return rc; }
    *out = o;
    return 0;
}

/* PERIODIC only: replace the analytic Coulomb kernel by a host-supplied Fourier-space filter ("only the filter F of
 * kernel 2 would be different", PAPER.md:236 -- screened hybrids): table[s0][s1][s2] on the symmetric index range
 * s_ax = 0..t_ax/2, frequency index m = a if 2a <= t else a - t, K^(a,b,c) = table[|ma|][|mb|][|mc|]. */
int exx_oracle_set_periodic_filter(exx_oracle *o, const double *table)
{
    if (!o || !table || o->bc != EXX_ORACLE_PERIODIC) return 1;
    const int t0 = o->t[0], t1 = o->t[1], t2 = o->t[2];
    const int s1 = t1 / 2 + 1, s2 = t2 / 2 + 1;
    for (int a = 0; a < t0; ++a) {
        int ma = (2 * a <= t0) ? a : t0 - a;
        for (int b = 0; b < t1; ++b) {
            int mb = (2 * b <= t1) ? b : t1 - b;
            for (int c = 0; c < t2; ++c) {
                int mc = (2 * c <= t2) ? c : t2 - c;
                cplx *k = &o->khat[((long long)a * t1 + b) * t2 + c];
                k->re = table[((long long)ma * s1 + mb) * s2 + mc];
                k->im = 0.0;
            }
        }
    }
    return 0;
}

/* General periodic cell (non-orthorhombic lattice; reading A25): K^ given on the FULL transform grid, used as is. */
int exx_oracle_set_periodic_filter_full(exx_oracle *o, const double *table_full)
{
    if (!o || !table_full || o->bc != EXX_ORACLE_PERIODIC) return 1;
    for (long long x = 0; x < o->T; ++x) {
        o->khat[x].re = table_full[x];
        o->khat[x].im = 0.0;
    }
    return 0;
}

void exx_oracle_destroy(exx_oracle *o)
{
    if (!o) return;
    for (int ax = 0; ax < 3; ++ax) free(o->roots[ax]);
    free(o->khat);
    free(o->gtab);
    free(o);
}

void exx_oracle_transform_dims(const exx_oracle *o, int tdims[3])
{
    for (int ax = 0; ax < 3; ++ax) tdims[ax] = o->t[ax];
}

int exx_oracle_get_khat(const exx_oracle *o, double *khat)
{
    if (!o || !khat) return 1;
    memcpy(khat, o->khat, sizeof(cplx) * (size_t)o->T);
    return 0;
}

/* ---------------------------------------------------------------------------------------------------
 * One Poisson solve (SURVEY.md 8(c) step 3; PAPER.md:73-75 Eq. 4, :125-127):
 * rho -> embed in T with zeros -> R = DFT3(rho) -> R *= K^ -> V = Re IDFT3(R) / T_tot on the n-grid.
 * `work` holds T complex values.
 * ------------------------------------------------------------------------------------------------- */
static int poisson_work(const exx_oracle *o, const double *rho, double *v, cplx *work)
{
    const int n0 = o->n[0], n1 = o->n[1], n2 = o->n[2];
    const int t1 = o->t[1], t2 = o->t[2];
    memset(work, 0, sizeof(cplx) * (size_t)o->T);
    for (int a = 0; a < n0; ++a)
        for (int b = 0; b < n1; ++b)
            for (int c = 0; c < n2; ++c)
                work[((long long)a * t1 + b) * t2 + c].re = rho[((long long)a * n1 + b) * n2 + c];
    int rc = dft3(o, work, -1);
    if (rc) return rc;
    for (long long x = 0; x < o->T; ++x) work[x] = cmul(work[x], o->khat[x]);
    rc = dft3(o, work, +1);
    if (rc) return rc;
    const double inv = 1.0 / (double)o->T;
    for (int a = 0; a < n0; ++a)
        for (int b = 0; b < n1; ++b)
            for (int c = 0; c < n2; ++c)
                v[((long long)a * n1 + b) * n2 + c] = work[((long long)a * t1 + b) * t2 + c].re * inv;
    return 0;
}

int exx_oracle_poisson(const exx_oracle *o, const double *rho, double *v)
{
    if (!o || !rho || !v) return 1;
    cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
    if (!work) return 2;
    int rc = poisson_work(o, rho, v, work);
    free(work);
    return rc;
}

/* Neumaier-compensated accumulation ("sums over r pairwise or compensated"). */
typedef struct { double s, c; } ksum;
static inline void ksum_add(ksum *k, double x)
{
    double t = k->s + x;
    if (fabs(k->s) >= fabs(x)) k->c += (k->s - t) + x; else k->c += (x - t) + k->s;
    k->s = t;
}
static inline double ksum_get(const ksum *k) { return k->s + k->c; }

/* e_ij = dV sum_r rho_ij(r) V_ij(r)   (Eq. 5, integral -> dV sum, A10) */
static double pair_energy(const exx_oracle *o, const double *rho, const double *v)
{
    ksum k = { 0.0, 0.0 };
    for (long long r = 0; r < o->M; ++r) ksum_add(&k, rho[r] * v[r]);
    return o->dV * ksum_get(&k);
}

/* ---------------------------------------------------------------------------------------------------
 * Full apply.  symmetric=0 is the definition: every ordered pair (i,j):
 *   Kpsi_i -= f_j V_ij psi_j   (Eq. 3, reading A1: sum over j)
 *   E_x    -= 1/2 f_i f_j e_ij (Eq. 2 / :81-82 Eq. 5, reading A4: one channel, f as passed)
 * OpenMP over the target orbital i: the owner computes Kpsi_i, no shared writes.
 * ------------------------------------------------------------------------------------------------- */
static int apply_pairs(const exx_oracle *o, int n_orb, const double *psi, const double *occ, const unsigned char *mask,
                       double *kpsi, double *ex, double *e_pair, int symmetric)
{
    /* mask (optional, [n_orb][n_orb]): the ordered pair (i,j) is left out of every sum when mask[i][j] == 0
     * (localised orbitals: co-densities of orbitals that do not overlap vanish). */
    if (!o || n_orb <= 0 || !psi || !occ || !kpsi || !ex) return 1;
    const long long M = o->M;
    memset(kpsi, 0, sizeof(double) * (size_t)M * n_orb);
    double *e_mat = (double *)calloc((size_t)n_orb * n_orb, sizeof(double));
    if (!e_mat) return 2;
    int fail = 0;
#ifdef _OPENMP
    g_threads_used = omp_get_max_threads();
#endif
    if (!symmetric) {
#pragma omp parallel
        {
            cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
            double *rho = (double *)malloc(sizeof(double) * (size_t)M);
            double *v = (double *)malloc(sizeof(double) * (size_t)M);
            if (!work || !rho || !v) {
#pragma omp atomic write
                fail = 1;
            }
#pragma omp barrier
            if (!fail) {
#pragma omp for schedule(dynamic, 1)
                for (int i = 0; i < n_orb; ++i) {
                    const double *pi = psi + (long long)i * M;
                    double *ki = kpsi + (long long)i * M;
                    for (int j = 0; j < n_orb; ++j) {
                        const double *pj = psi + (long long)j * M;
                        if (mask && !mask[(long long)i * n_orb + j]) continue;
                        for (long long r = 0; r < M; ++r) rho[r] = pi[r] * pj[r];          /* Eq. 8 */
                        if (poisson_work(o, rho, v, work)) {                              /* Eq. 4 */
#pragma omp atomic write
                            fail = 1;
                            continue;
                        }
                        const double fj = occ[j];
                        for (long long r = 0; r < M; ++r) ki[r] -= fj * v[r] * pj[r];      /* Eq. 3 */
                        e_mat[(long long)i * n_orb + j] = pair_energy(o, rho, v);          /* Eq. 5 */
                    }
                }
            }
            free(work); free(rho); free(v);
        }
    } else {
        /* i <= j only; V_ij = V_ji used for both orbitals.  For each i the loop over j is
         * parallel: Kpsi_j (distinct j) is written by one thread, the Kpsi_i contributions go to a private
         * buffer that is reduced afterwards in thread order. */
        int nthreads = 1;
#ifdef _OPENMP
        nthreads = omp_get_max_threads();
#endif
        double *priv = (double *)malloc(sizeof(double) * (size_t)M * nthreads);
        if (!priv) { free(e_mat); return 2; }
#pragma omp parallel
        {
            int tid = 0;
#ifdef _OPENMP
            tid = omp_get_thread_num();
#endif
            cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
            double *rho = (double *)malloc(sizeof(double) * (size_t)M);
            double *v = (double *)malloc(sizeof(double) * (size_t)M);
            double *mine = priv + (long long)tid * M;
            if (!work || !rho || !v) {
#pragma omp atomic write
                fail = 1;
            }
#pragma omp barrier
            if (!fail) {
                for (int i = 0; i < n_orb; ++i) {
                    const double *pi = psi + (long long)i * M;
                    const double fi = occ[i];
                    memset(mine, 0, sizeof(double) * (size_t)M);
#pragma omp for schedule(dynamic, 1)
                    for (int j = i; j < n_orb; ++j) {
                        const double *pj = psi + (long long)j * M;
                        const double fj = occ[j];
                        if (fi == 0.0 && fj == 0.0) continue;                             /* A15 */
                        if (mask && !mask[(long long)i * n_orb + j]) continue;
                        for (long long r = 0; r < M; ++r) rho[r] = pi[r] * pj[r];
                        if (poisson_work(o, rho, v, work)) {
#pragma omp atomic write
                            fail = 1;
                            continue;
                        }
                        for (long long r = 0; r < M; ++r) mine[r] -= fj * v[r] * pj[r];
                        if (j != i) {
                            double *kj = kpsi + (long long)j * M;
                            for (long long r = 0; r < M; ++r) kj[r] -= fi * v[r] * pi[r];
                        }
                        double e = pair_energy(o, rho, v);
                        e_mat[(long long)i * n_orb + j] = e;
                        e_mat[(long long)j * n_orb + i] = e;
                    }
                    /* implicit barrier of the omp for; reduce private buffers into Kpsi_i */
#pragma omp for schedule(static)
                    for (long long r = 0; r < M; ++r) {
                        double s = 0.0;
                        for (int t = 0; t < nthreads; ++t) s += priv[(long long)t * M + r];
                        kpsi[(long long)i * M + r] += s;
                    }
                }
            }
            free(work); free(rho); free(v);
        }
        free(priv);
    }
    if (fail) { free(e_mat); return 2; }
    /* E_x = -1/2 sum_{ij} f_i f_j e_ij over ORDERED pairs, compensated (Eq. 2 / Eq. 5). */
    ksum k = { 0.0, 0.0 };
    for (int i = 0; i < n_orb; ++i)
        for (int j = 0; j < n_orb; ++j)
            ksum_add(&k, -0.5 * occ[i] * occ[j] * e_mat[(long long)i * n_orb + j]);
    *ex = ksum_get(&k);
    if (e_pair) memcpy(e_pair, e_mat, sizeof(double) * (size_t)n_orb * n_orb);
    free(e_mat);
    return 0;
}

int exx_oracle_apply(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                     double *kpsi, double *ex, double *e_pair, int symmetric)
{
    return apply_pairs(o, n_orb, psi, occ, NULL, kpsi, ex, e_pair, symmetric);
}

int exx_oracle_apply_masked(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                            const unsigned char *mask, double *kpsi, double *ex, double *e_pair)
{
    if (!mask) return 1;
    return apply_pairs(o, n_orb, psi, occ, mask, kpsi, ex, e_pair, 0);
}

/* ---------------------------------------------------------------------------------------------------
 * The exchange operator built from the occupied set (psi_j, f_j) applied to another orbital set phi_t
 * (Eq. 3 with phi_t in the place of psi_i; unoccupied states and the second spin channel of the
 * paper's runs):   Kphi_t = - sum_j f_j V[phi_t psi_j] psi_j.   OpenMP over t.
 * ------------------------------------------------------------------------------------------------- */
int exx_oracle_apply_to(const exx_oracle *o, int n_occ, const double *psi, const double *occ,
                        int n_tgt, const double *phi, double *kphi)
{
    if (!o || n_occ <= 0 || n_tgt <= 0 || !psi || !occ || !phi || !kphi) return 1;
    const long long M = o->M;
    memset(kphi, 0, sizeof(double) * (size_t)M * n_tgt);
    int fail = 0;
#ifdef _OPENMP
    g_threads_used = omp_get_max_threads();
#endif
#pragma omp parallel
    {
        cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
        double *rho = (double *)malloc(sizeof(double) * (size_t)M);
        double *v = (double *)malloc(sizeof(double) * (size_t)M);
        if (!work || !rho || !v) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int t = 0; t < n_tgt; ++t) {
                const double *pt = phi + (long long)t * M;
                double *kt = kphi + (long long)t * M;
                for (int j = 0; j < n_occ; ++j) {
                    const double *pj = psi + (long long)j * M;
                    for (long long r = 0; r < M; ++r) rho[r] = pt[r] * pj[r];             /* Eq. 8 */
                    if (poisson_work(o, rho, v, work)) {                                  /* Eq. 4 */
#pragma omp atomic write
                        fail = 1;
                        continue;
                    }
                    const double fj = occ[j];
                    for (long long r = 0; r < M; ++r) kt[r] -= fj * v[r] * pj[r];          /* Eq. 3 */
                }
            }
        }
        free(work); free(rho); free(v);
    }
    return fail ? 2 : 0;
}

/* ---------------------------------------------------------------------------------------------------
 * All pairs between two DISJOINT orbital blocks A (n_a orbitals) and B (n_b): the unit of work of the paper's
 * round-robin distribution (Fig. 1).  Written from each owner's point of view, every potential
 * solved separately for the two sides (no reuse of V_ab for V_ba):
 *   ka[a] = - sum_b f_b V_ab psi_b      kb[b] = - sum_a f_a V_ba psi_a      e[a][b] = dV sum_r rho_ab V_ab
 *   ex    = - sum_{a,b} f_a f_b e_ab    (Eq. 5 counts the ordered pairs (a,b) and (b,a): 2 * (-1/2))
 * ka, kb are OVERWRITTEN.
 * ------------------------------------------------------------------------------------------------- */
int exx_oracle_apply_block(const exx_oracle *o, int n_a, const double *psi_a, const double *occ_a, double *ka,
                           int n_b, const double *psi_b, const double *occ_b, double *kb, double *ex, double *e_block)
{
    if (!o || n_a <= 0 || n_b <= 0 || !psi_a || !occ_a || !ka || !psi_b || !occ_b || !kb || !ex) return 1;
    const long long M = o->M;
    memset(ka, 0, sizeof(double) * (size_t)M * n_a);
    memset(kb, 0, sizeof(double) * (size_t)M * n_b);
    double *e_mat = (double *)calloc((size_t)n_a * n_b, sizeof(double));
    if (!e_mat) return 2;
    int fail = 0;
#ifdef _OPENMP
    g_threads_used = omp_get_max_threads();
#endif
#pragma omp parallel
    {
        cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
        double *rho = (double *)malloc(sizeof(double) * (size_t)M);
        double *v = (double *)malloc(sizeof(double) * (size_t)M);
        if (!work || !rho || !v) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int a = 0; a < n_a; ++a) {                              /* side A receives from every b */
                const double *pa = psi_a + (long long)a * M;
                double *k = ka + (long long)a * M;
                for (int b = 0; b < n_b; ++b) {
                    const double *pb = psi_b + (long long)b * M;
                    for (long long r = 0; r < M; ++r) rho[r] = pa[r] * pb[r];
                    if (poisson_work(o, rho, v, work)) {
#pragma omp atomic write
                        fail = 1;
                        continue;
                    }
                    const double fb = occ_b[b];
                    for (long long r = 0; r < M; ++r) k[r] -= fb * v[r] * pb[r];
                    e_mat[(long long)a * n_b + b] = pair_energy(o, rho, v);
                }
            }
#pragma omp for schedule(dynamic, 1)
            for (int b = 0; b < n_b; ++b) {                              /* side B receives from every a */
                const double *pb = psi_b + (long long)b * M;
                double *k = kb + (long long)b * M;
                for (int a = 0; a < n_a; ++a) {
                    const double *pa = psi_a + (long long)a * M;
                    for (long long r = 0; r < M; ++r) rho[r] = pb[r] * pa[r];
                    if (poisson_work(o, rho, v, work)) {
#pragma omp atomic write
                        fail = 1;
                        continue;
                    }
                    const double fa = occ_a[a];
                    for (long long r = 0; r < M; ++r) k[r] -= fa * v[r] * pa[r];
                }
            }
        }
        free(work); free(rho); free(v);
    }
    if (fail) { free(e_mat); return 2; }
    ksum k = { 0.0, 0.0 };
    for (int a = 0; a < n_a; ++a)
        for (int b = 0; b < n_b; ++b) ksum_add(&k, -occ_a[a] * occ_b[b] * e_mat[(long long)a * n_b + b]);
    *ex = ksum_get(&k);
    if (e_block) memcpy(e_block, e_mat, sizeof(double) * (size_t)n_a * n_b);
    free(e_mat);
    return 0;
}

/* Complete rows Kpsi_i = -sum_j f_j V_ij psi_j for listed i (same arithmetic as the N^2 mode). */
int exx_oracle_rows(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                    int n_rows, const int *rows, double *kpsi_rows, double *e_rows)
{
    if (!o || n_orb <= 0 || !psi || !occ || n_rows <= 0 || !rows || !kpsi_rows) return 1;
    for (int s = 0; s < n_rows; ++s) if (rows[s] < 0 || rows[s] >= n_orb) return 1;
    const long long M = o->M;
    memset(kpsi_rows, 0, sizeof(double) * (size_t)M * n_rows);
    int fail = 0;
    int nthreads = 1;
#ifdef _OPENMP
    nthreads = omp_get_max_threads();
    g_threads_used = nthreads;
#endif
    double *priv = (double *)malloc(sizeof(double) * (size_t)M * nthreads);
    if (!priv) return 2;
#pragma omp parallel
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
        double *rho = (double *)malloc(sizeof(double) * (size_t)M);
        double *v = (double *)malloc(sizeof(double) * (size_t)M);
        double *mine = priv + (long long)tid * M;
        if (!work || !rho || !v) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
            for (int s = 0; s < n_rows; ++s) {
                const int i = rows[s];
                const double *pi = psi + (long long)i * M;
                memset(mine, 0, sizeof(double) * (size_t)M);
#pragma omp for schedule(dynamic, 1)
                for (int j = 0; j < n_orb; ++j) {
                    const double *pj = psi + (long long)j * M;
                    for (long long r = 0; r < M; ++r) rho[r] = pi[r] * pj[r];
                    if (poisson_work(o, rho, v, work)) {
#pragma omp atomic write
                        fail = 1;
                        continue;
                    }
                    const double fj = occ[j];
                    for (long long r = 0; r < M; ++r) mine[r] -= fj * v[r] * pj[r];
                    if (e_rows) e_rows[(long long)s * n_orb + j] = pair_energy(o, rho, v);
                }
#pragma omp for schedule(static)
                for (long long r = 0; r < M; ++r) {
                    double acc = 0.0;
                    for (int t = 0; t < nthreads; ++t) acc += priv[(long long)t * M + r];
                    kpsi_rows[(long long)s * M + r] = acc;
                }
            }
        }
        free(work); free(rho); free(v);
    }
    free(priv);
    return fail ? 2 : 0;
}

int exx_oracle_pair_energies(const exx_oracle *o, int n_orb, const double *psi,
                             int n_pairs, const int *pi_idx, const int *pj_idx, double *e_out)
{
    if (!o || n_orb <= 0 || !psi || n_pairs <= 0 || !pi_idx || !pj_idx || !e_out) return 1;
    for (int s = 0; s < n_pairs; ++s)
        if (pi_idx[s] < 0 || pi_idx[s] >= n_orb || pj_idx[s] < 0 || pj_idx[s] >= n_orb) return 1;
    const long long M = o->M;
    int fail = 0;
#ifdef _OPENMP
    g_threads_used = omp_get_max_threads();
#endif
#pragma omp parallel
    {
        cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
        double *rho = (double *)malloc(sizeof(double) * (size_t)M);
        double *v = (double *)malloc(sizeof(double) * (size_t)M);
        if (!work || !rho || !v) {
#pragma omp atomic write
            fail = 1;
        }
#pragma omp barrier
        if (!fail) {
#pragma omp for schedule(dynamic, 1)
            for (int s = 0; s < n_pairs; ++s) {
                const double *pa = psi + (long long)pi_idx[s] * M;
                const double *pb = psi + (long long)pj_idx[s] * M;
                for (long long r = 0; r < M; ++r) rho[r] = pa[r] * pb[r];
                if (poisson_work(o, rho, v, work)) {
#pragma omp atomic write
                    fail = 1;
                    continue;
                }
                e_out[s] = pair_energy(o, rho, v);
            }
        }
        free(work); free(rho); free(v);
    }
    return fail ? 2 : 0;
}

/* ---------------------------------------------------------------------------------------------------
 * Direct real-space route (no FFT inside the convolution) -- used by the pins P2/P3 and by sampled parity.
 * FREE:     V(r) = dV sum_r' g(|a-a'|,|b-b'|,|c-c'|) rho(r')        (Eq. 4 discretised; A5, A10)
 * PERIODIC: V(r) = sum_r' g_per((r - r') mod n) rho(r'),  g_per = (1/M) sum_G K^(G) e^{iG.r}
 * ------------------------------------------------------------------------------------------------- */
int exx_oracle_realspace_kernel(const exx_oracle *o, double *g_out)
{
    if (!o || !g_out) return 1;
    if (o->bc == EXX_ORACLE_FREE) {
        for (long long r = 0; r < o->M; ++r) g_out[r] = o->dV * o->gtab[r];
        return 0;
    }
    cplx *work = (cplx *)malloc(sizeof(cplx) * (size_t)o->T);
    if (!work) return 2;
    memcpy(work, o->khat, sizeof(cplx) * (size_t)o->T);
    int rc = dft3(o, work, +1);
    if (!rc) {
        const double inv = 1.0 / (double)o->T;
        for (long long r = 0; r < o->M; ++r) g_out[r] = work[r].re * inv;
    }
    free(work);
    return rc;
}

static inline long long disp_index(const exx_oracle *o, int a, int b, int c, int a2, int b2, int c2)
{
    int da, db, dc;
    if (o->bc == EXX_ORACLE_FREE) {
        da = abs(a - a2); db = abs(b - b2); dc = abs(c - c2);
    } else {
        da = (a - a2) % o->n[0]; if (da < 0) da += o->n[0];
        db = (b - b2) % o->n[1]; if (db < 0) db += o->n[1];
        dc = (c - c2) % o->n[2]; if (dc < 0) dc += o->n[2];
    }
    return ((long long)da * o->n[1] + db) * o->n[2] + dc;
}

int exx_oracle_poisson_direct(const exx_oracle *o, const double *rho, double *v)
{
    if (!o || !rho || !v) return 1;
    double *g = (double *)malloc(sizeof(double) * (size_t)o->M);
    if (!g) return 2;
    int rc = exx_oracle_realspace_kernel(o, g);
    if (rc) { free(g); return rc; }
    const int n0 = o->n[0], n1 = o->n[1], n2 = o->n[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int a = 0; a < n0; ++a)
        for (int b = 0; b < n1; ++b)
            for (int c = 0; c < n2; ++c) {
                ksum k = { 0.0, 0.0 };
                for (int a2 = 0; a2 < n0; ++a2)
                    for (int b2 = 0; b2 < n1; ++b2)
                        for (int c2 = 0; c2 < n2; ++c2)
                            ksum_add(&k, g[disp_index(o, a, b, c, a2, b2, c2)] *
                                         rho[((long long)a2 * n1 + b2) * n2 + c2]);
                v[((long long)a * n1 + b) * n2 + c] = ksum_get(&k);
            }
    free(g);
    return 0;
}

/* Mixed boundary conditions (slab / wire, "free, wire, slab and periodic"), the plain definition:
 *   V(r) = dV * sum_{r'} g(d(r, r')) rho(r'),   d_a = (r_a - r'_a) mod n_a  on a periodic axis (displacement to the
 *   nearest-or-any image: g holds one full period there), d_a = |r_a - r'_a| on an isolated axis (g even).
 * O(M^2) double loop, no FFT, no handle: everything is an argument.  DESIGN.md reading A24. */
int exx_oracle_poisson_direct_mixed(const int dims[3], const double spacing[3], const int periodic[3],
                                    const double *table, const double *rho, double *v)
{
    if (!dims || !spacing || !periodic || !table || !rho || !v) return 1;
    const int n0 = dims[0], n1 = dims[1], n2 = dims[2];
    if (n0 < 1 || n1 < 1 || n2 < 1) return 1;
    const double dV = spacing[0] * spacing[1] * spacing[2];
#pragma omp parallel for collapse(2) schedule(static)
    for (int a = 0; a < n0; ++a)
        for (int b = 0; b < n1; ++b)
            for (int c = 0; c < n2; ++c) {
                ksum k = { 0.0, 0.0 };
                for (int a2 = 0; a2 < n0; ++a2) {
                    const int da = periodic[0] ? ((a - a2) % n0 + n0) % n0 : (a >= a2 ? a - a2 : a2 - a);
                    for (int b2 = 0; b2 < n1; ++b2) {
                        const int db = periodic[1] ? ((b - b2) % n1 + n1) % n1 : (b >= b2 ? b - b2 : b2 - b);
                        for (int c2 = 0; c2 < n2; ++c2) {
                            const int dc = periodic[2] ? ((c - c2) % n2 + n2) % n2 : (c >= c2 ? c - c2 : c2 - c);
                            ksum_add(&k, table[((long long)da * n1 + db) * n2 + dc] *
                                         rho[((long long)a2 * n1 + b2) * n2 + c2]);
                        }
                    }
                }
                v[((long long)a * n1 + b) * n2 + c] = dV * ksum_get(&k);
            }
    return 0;
}

int exx_oracle_kpsi_points(const exx_oracle *o, int n_orb, const double *psi, const double *occ,
                           int n_samples, const int *orb, const long long *point, double *out)
{
    if (!o || n_orb <= 0 || !psi || !occ || n_samples <= 0 || !orb || !point || !out) return 1;
    const long long M = o->M;
    for (int s = 0; s < n_samples; ++s)
        if (orb[s] < 0 || orb[s] >= n_orb || point[s] < 0 || point[s] >= M) return 1;
    double *g = (double *)malloc(sizeof(double) * (size_t)M);
    if (!g) return 2;
    int rc = exx_oracle_realspace_kernel(o, g);
    if (rc) { free(g); return rc; }
    const int n1 = o->n[1], n2 = o->n[2];
#ifdef _OPENMP
    g_threads_used = omp_get_max_threads();
#endif
    for (int s = 0; s < n_samples; ++s) {
        const int i = orb[s];
        const long long p = point[s];
        const int a = (int)(p / ((long long)n1 * n2)), b = (int)((p / n2) % n1), c = (int)(p % n2);
        const double *pi = psi + (long long)i * M;
        double total = 0.0, comp = 0.0;
#pragma omp parallel for schedule(dynamic, 1)
        for (int j = 0; j < n_orb; ++j) {
            const double *pj = psi + (long long)j * M;
            ksum k = { 0.0, 0.0 };
            for (int a2 = 0; a2 < o->n[0]; ++a2)
                for (int b2 = 0; b2 < n1; ++b2) {
                    const long long base = ((long long)a2 * n1 + b2) * n2;
                    for (int c2 = 0; c2 < n2; ++c2)
                        ksum_add(&k, g[disp_index(o, a, b, c, a2, b2, c2)] * pi[base + c2] * pj[base + c2]);
                }
            const double term = -occ[j] * pj[p] * ksum_get(&k);
#pragma omp critical
            {
                ksum kk = { total, comp };
                ksum_add(&kk, term);
                total = kk.s; comp = kk.c;
            }
        }
        out[s] = total + comp;
    }
    free(g);
    return 0;
}

int exx_oracle_threads(void) { return g_threads_used; }
