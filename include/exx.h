/*
 * exx.h -- C ABI of libexx_b200: exact-exchange operator application on one B200 (sm_100a).
 *
 * Implements the data-parallel hot path of arXiv:1712.07973 (citations are /root/reference/PAPER.md lines):
 * "for a given set of psi_i(r), the value of E_X as well as the action of the corresponding Fock operator D_X
 * on the entire set of occupied orbitals", as a "stand-alone library" for codes with "orbitals on
 * a Cartesian real space grid".  For every unordered orbital pair i <= j (PAPER.md:77-79,
 * "all the N(N+1)/2 charge densities"):
 *
 *   Kernel 1   rho_ij(r) = psi_i(r) psi_j(r)                                            PAPER.md:101 Eq. 8, :115
 *   Kernel 2   V_ij = solution of  laplace V_ij = -4 pi rho_ij  by FFT convolution with
 *              the Green's function, "appropriate padding" for isolated systems         PAPER.md:73-75 Eq. 4, :116, :125-127
 *   Kernel 3   K psi_i += -f_j V_ij psi_j ;  K psi_j += -f_i V_ij psi_i  (i != j)       PAPER.md:67-69 Eq. 3, :111, :117
 *              e_ij = dV sum_r rho_ij V_ij ;  E_x = -1/2 sum_{i,j} f_i f_j e_ij         PAPER.md:81-82 Eq. 5, :117
 *
 * Everything runs in hand-written CUDA kernels (fp64): two real co-densities are packed into one complex 3-D
 * FFT; co-density + zero padding are fused into the first FFT pass, the Green's-function multiply between the
 * forward and the inverse transform, and the K psi accumulation + energy reduction into the last inverse pass.
 * There is no CPU fallback: every entry point that computes fails with EXX_ERR_CUDA if no device is usable.
 *
 * Conventions: real orbitals; one spin channel, occupations used as
 * passed (no spin-degeneracy factor, no hybrid mixing fraction); integrals are dV * sum over grid points;
 * periodic kernel 4 pi/|G|^2 with the G=0 term set to 0; free kernel = host table, Hockney padding to 2n.
 *
 * Memory order: psi[i][a][b][c], C order, c fastest: index = ((i*n1 + a)*n2 + b)*n3 + c.
 * Threading: a plan is not re-entrant; distinct plans are independent.  All device work is enqueued on the
 * plan's stream.  No entry point throws, aborts or exits; errors are status codes plus exx_last_error text.
 */
#ifndef EXX_B200_H
#define EXX_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct exx_plan exx_plan;                 /* opaque, owned by the library */

typedef enum {
    EXX_OK = 0,
    EXX_ERR_INVALID_ARG = 1,        /* NULL where not allowed, n_orb out of range, bad enum, spacing <= 0      */
    EXX_ERR_UNSUPPORTED_SIZE = 2,   /* a grid length the FFT does not cover (see exx_plan_create)              */
    EXX_ERR_BAD_POINTER = 3,        /* host pointer where a device pointer is required, or the reverse         */
    EXX_ERR_ALLOC = 4,              /* device or host allocation failed                                        */
    EXX_ERR_CUDA = 5,               /* CUDA runtime / launch failure, or no usable device                      */
    EXX_ERR_INTERNAL = 6
} exx_status;

typedef enum { EXX_BC_PERIODIC = 0, EXX_BC_FREE = 1 } exx_bc;

/*
 * exx_plan_create -- one-time setup for a grid, boundary condition and Green's function (PAPER.md:125:
 * "The Green's function can be discretized for ... free ... and periodic" boundary conditions).
 *   dims        HOST, n1,n2,n3.  Transform length per axis T = n (periodic) or 2n (free); T must be one of
 *               {16, 32, 64, 96, 128, 192, 256} (radix-2/3 only), else EXX_ERR_UNSUPPORTED_SIZE.
 *   spacing     HOST, h1,h2,h3 in bohr (> 0).
 *   bc          EXX_BC_PERIODIC or EXX_BC_FREE.
 *   kernel_host HOST.  PERIODIC: NULL => analytic 4 pi/|G|^2, G = 0 -> 0.  (A non-NULL pointer is rejected.)
 *               FREE: table g[a][b][c] of n1*n2*n3 doubles = Green's function at displacement
 *               (a h1, b h2, c h3), units 1/bohr; copied during the call, caller may free it afterwards.
 *   max_orbitals  upper bound for n_orb of later exx_apply calls (sizes the pair-energy buffers).
 *   cuda_stream cudaStream_t as void* (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream.
 * On success *plan receives a handle that the caller must release with exx_plan_destroy.
 */
exx_status exx_plan_create(exx_plan **plan, const int dims[3], const double spacing[3], exx_bc bc,
                           const double *kernel_host, int max_orbitals, void *cuda_stream);

/*
 * exx_apply -- the hot path: K psi for all orbitals and E_x (PAPER.md:67-69 Eq. 3, :81-82 Eq. 5).
 *   psi_dev   DEVICE, [n_orb][n1][n2][n3] doubles, contiguous, read-only, 16-byte aligned.
 *   occ_host  HOST, [n_orb] occupations f_i.  A pair with f_i = f_j = 0 is skipped.
 *   kpsi_dev  DEVICE, same shape as psi; OVERWRITTEN with K psi_i = -sum_j f_j V_ij psi_j.  Must not alias psi.
 *   ex_host   HOST, one double; written after the plan's stream has been synchronised.
 * exx_apply_async is the same without the synchronisation: E_x lands in DEVICE memory (ex_dev).
 */
exx_status exx_apply(exx_plan *plan, int n_orb, const double *psi_dev, const double *occ_host,
                     double *kpsi_dev, double *ex_host);
exx_status exx_apply_async(exx_plan *plan, int n_orb, const double *psi_dev, const double *occ_host,
                           double *kpsi_dev, double *ex_dev);

/*
 * exx_apply_host -- end-to-end convenience: psi_host / kpsi_host are HOST buffers (pinned or pageable); the
 * library stages them through device memory it owns (host->device copy of psi on the plan's stream; each K psi
 * row is copied device->host on an internal copy stream as soon as its block-row has finished, overlapping the
 * remaining pair solves when kpsi_host is pinned), and synchronises.  Same arithmetic as exx_apply.
 */
exx_status exx_apply_host(exx_plan *plan, int n_orb, const double *psi_host, const double *occ_host,
                          double *kpsi_host, double *ex_host);

/*
 * exx_get_pair_energies -- e_ij = dV sum_r rho_ij(r) V_ij(r) of the most recent apply, HOST [n_orb*n_orb],
 * symmetric (Eq. 5 integrand).  Pairs skipped for zero occupations read 0.  Synchronises.
 */
exx_status exx_get_pair_energies(exx_plan *plan, double *e_host);

/*
 * exx_schedule_pairs -- HOST-only view of the pair scheduler (no GPU needed): the number of Poisson solves
 * (unordered pairs i <= j, pairs with f_i = f_j = 0 skipped) and of packed complex transforms an apply with
 * these occupations performs.  PAPER.md:77-79; Table 1: N(N+1)/2.
 */
exx_status exx_schedule_pairs(int n_orb, const double *occ_host, long long *n_pairs, long long *n_transforms);

/*
 * exx_schedule_list -- HOST-only listing of the same schedule, cut into batches of at most max_batch transforms
 * (max_batch < 1: unlimited).  Row t of xforms_host [capacity][5] receives {j, l, i, flags, batch}: the transform
 * carries the pairs (j,i) in its real part (flags bit 0) and (l,i) in its imaginary part (flags bit 1) of the
 * co-density z = psi_i psi_j + i psi_i psi_l (Eq. 8); j, l are the two resident orbitals of batch
 * `batch` (l = -1: none).  *n_transforms receives the total; at most `capacity` rows are written (xforms_host may
 * be NULL when capacity is 0).  Every unordered pair that is not doubly empty appears exactly once.
 */
exx_status exx_schedule_list(int n_orb, const double *occ_host, int max_batch, int *xforms_host, long long capacity,
                             long long *n_transforms);

/* Transform-grid lengths (n or 2n) of a plan and the bytes of device workspace it owns. */
exx_status exx_plan_transform_dims(const exx_plan *plan, int tdims[3]);
size_t     exx_plan_workspace_bytes(const exx_plan *plan);

/* Name of the kernel this plan's geometry dispatches to for pass 0 (A), 1 (B) or 2 (C); "" for anything else.  The
 * string is static, owned by the library. */
const char *exx_plan_kernel_name(const exx_plan *plan, int pass);

/* Number of kernel launches the library has enqueued for this plan since creation (for bench "gpu_launches"). */
long long  exx_plan_launch_count(const exx_plan *plan);

/*
 * Per-pass device timing (CUDA events on the plan's stream around every pass launch).  Off by default.
 * exx_plan_get_profile synchronises and returns, for the most recent apply, the summed milliseconds and the
 * launch counts of  [0] pass A, [1] pass B, [2] pass C, [3] energy reduction.
 */
exx_status exx_plan_set_profiling(exx_plan *plan, int enable);
exx_status exx_plan_get_profile(exx_plan *plan, double pass_ms[4], long long pass_launches[4]);

/* Tuning knob: maximum packed transforms per batch (same-i group); <= 0 restores the default. */
exx_status exx_plan_set_batch(exx_plan *plan, int max_transforms_per_batch);

exx_status  exx_plan_destroy(exx_plan *plan);       /* NULL is allowed */
const char *exx_status_string(exx_status s);
const char *exx_last_error(const exx_plan *plan);   /* detail text incl. CUDA error name; plan may be NULL for
                                                       the last exx_plan_create failure on this thread */
const char *exx_version(void);

#ifdef __cplusplus
}
#endif
#endif
