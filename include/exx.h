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
 * Threading: a plan is not re-entrant; distinct plans (also on different devices) are independent.  All device work
 * is enqueued on the plan's stream.  No entry point throws, aborts or exits; errors are status codes plus
 * exx_last_error text.  The apply calls perform no host or device allocation (the one exception: exx_apply_host grows
 * its device staging buffers when n_orb exceeds every earlier call's).
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
 *   dims        HOST, n1,n2,n3.  Transform length per axis T = n (periodic) or 2n (free); every T must be one of
 *               {16, 32, 48, 64, 96, 128, 144, 192, 256} (any mix over the three axes), or the transform grid is cubic
 *               with T = 24 or 72 (radix-2/3 only, reading A9); else EXX_ERR_UNSUPPORTED_SIZE.
 *   spacing     HOST, h1,h2,h3 in bohr (> 0).
 *   bc          EXX_BC_PERIODIC or EXX_BC_FREE.
 *   kernel_host HOST.  PERIODIC: NULL => analytic 4 pi/|G|^2, G = 0 -> 0.  Non-NULL => Fourier-space filter table
 *               K^[s1][s2][s3] of (n1/2+1)*(n2/2+1)*(n3/2+1) doubles on the symmetric index range (frequency index
 *               m_a = +-s_a, G_a = 2 pi m_a / (n_a h_a); K^ is taken even in every index), WITHOUT the 1/(n1 n2 n3)
 *               of the inverse transform -- e.g. the screened kernel of HSE06-type hybrids, "only the filter F of
 *               kernel 2 would be different".
 *               FREE: table g[a][b][c] of n1*n2*n3 doubles = Green's function at displacement
 *               (a h1, b h2, c h3), units 1/bohr (an interpolating-scaling-function table can be passed as is).
 *               SLAB / WIRE boundary conditions ("free, wire, slab and periodic") are FREE plans whose
 *               table holds ONE FULL PERIOD of the mixed Green's function along each periodic axis (index d <->
 *               displacement d*h, even under d -> n-d) and displacements 0..n-1 along each isolated axis: zero-padded
 *               convolution with g[|d|] equals wrap-around convolution on every axis on which g is even-periodic
 *               (reading A24).
 *               Either table is copied during the call; the caller may free it afterwards.
 *   max_orbitals  upper bound for n_orb of later exx_apply calls (sizes the pair-energy buffers).
 *   cuda_stream cudaStream_t as void* (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream.
 * On success *plan receives a handle that the caller must release with exx_plan_destroy.
 */
exx_status exx_plan_create(exx_plan **plan, const int dims[3], const double spacing[3], exx_bc bc,
                           const double *kernel_host, int max_orbitals, void *cuda_stream);

/*
 * exx_plan_create_general -- periodic cell of ANY shape (non-orthorhombic lattice vectors a1, a2, a3; the
 * solver is "completely general").  The grid points are r = (i1/n1) a1 + (i2/n2) a2 + (i3/n3) a3, so the transforms are the
 * same as for an orthorhombic cell; what differs is the Fourier-space kernel, which is no longer even in every index:
 *   khat_full_host  HOST, K^[m1][m2][m3], n1*n2*n3 doubles on the FULL FFT index grid (index m_a <-> frequency m_a for
 *                   m_a <= n_a/2, m_a - n_a above), e.g. 4 pi / |m1 b1 + m2 b2 + m3 b3|^2 with the reciprocal vectors b_a
 *                   and K^(0) = 0; must satisfy K^(-m) = K^(m) for real potentials; WITHOUT the 1/(n1 n2 n3) of the inverse
 *                   transform.  Copied during the call.
 *   cell_volume     |a1 . (a2 x a3)| in bohr^3: only dV = cell_volume / (n1 n2 n3) enters (energies, A10).
 * dims, max_orbitals, cuda_stream as exx_plan_create.  DESIGN.md reading A25.
 */
exx_status exx_plan_create_general(exx_plan **plan, const int dims[3], double cell_volume, const double *khat_full_host,
                                   int max_orbitals, void *cuda_stream);

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
 * exx_plan_release_staging -- frees the device staging buffers exx_apply_host keeps between calls (2 * n_orb * n1*n2*n3
 * doubles: the algorithm needs every orbital and every K psi row resident; they count in exx_plan_workspace_bytes).
 */
exx_status exx_plan_release_staging(exx_plan *plan);

/*
 * exx_get_pair_energies -- e_ij = dV sum_r rho_ij(r) V_ij(r) of the most recent exx_apply / _async / _host / _pairs,
 * HOST [n_orb*n_orb], symmetric (Eq. 5 integrand).  n_orb must equal that apply's orbital count
 * (EXX_ERR_INVALID_ARG otherwise: the buffer size is the caller's statement, never guessed).  Pairs skipped for zero
 * occupations or by a pair mask read 0.  Synchronises.
 */
exx_status exx_get_pair_energies(exx_plan *plan, int n_orb, double *e_host);

/*
 * exx_apply_pairs -- exx_apply restricted to a caller-supplied list of pairs: localised orbitals, for which "the
 * matrix K^{alpha beta} is sparse" (Eq. 6-7) because co-densities of non-overlapping orbitals vanish.
 *   pair_mask_host  HOST, [n_orb*n_orb] bytes, symmetric; pair (a,b) is solved iff mask[a*n_orb+b] != 0 (and not both
 *                   occupations are zero).  Excluded pairs contribute nothing to K psi, E_x and read 0 in e_ij.
 * Other arguments as exx_apply.  EXX_ERR_INVALID_ARG for an asymmetric mask.
 */
exx_status exx_apply_pairs(exx_plan *plan, int n_orb, const double *psi_dev, const double *occ_host,
                           const unsigned char *pair_mask_host, double *kpsi_dev, double *ex_host);

/*
 * exx_apply_to -- the exchange operator built from the occupied set applied to ANOTHER set of orbitals (unoccupied /
 * virtual states, a trial subspace; the second spin channel is a second call with that channel's occupied set --
 * PAPER.md:210, Table 3 caption :244; Eq. 3 :67-69 with phi_t in place of psi_i):
 *      K phi_t (r) = - sum_j f_j  V[phi_t psi_j](r)  psi_j(r),      j over the n_occ occupied orbitals.
 *   psi_dev   DEVICE [n_occ][n1][n2][n3], occ_host HOST [n_occ] (orbitals with f_j = 0 are skipped);
 *   phi_dev   DEVICE [n_tgt][n1][n2][n3];  kphi_dev DEVICE, same shape as phi, OVERWRITTEN.
 * n_occ, n_tgt <= max_orbitals; all arrays 16-byte aligned; kphi must not overlap psi or phi (phi may be psi).  No
 * energy is produced.  Synchronises the plan's stream before returning.
 */
exx_status exx_apply_to(exx_plan *plan, int n_occ, const double *psi_dev, const double *occ_host, int n_tgt,
                        const double *phi_dev, double *kphi_dev);

/*
 * exx_apply_to_cross -- exx_apply_to with a partner set: the potential of the co-density (phi_t, psi_j) is multiplied by
 * chi_j instead of psi_j,
 *      K phi_t (r) = - sum_j f_j  V[phi_t psi_j](r)  chi_j(r),
 * the building block that the real and imaginary parts of complex orbitals need (below).  chi_dev DEVICE
 * [n_occ][n1][n2][n3]; everything else as exx_apply_to.
 *
 * exx_apply_complex -- the hot path for COMPLEX orbitals psi = u + i v (Eq. 8 keeps the conjugate; the
 * paper's own runs are real, Gamma point, :159):  rho_ij = conj(psi_j) psi_i,  K psi_i = - sum_j f_j V_ij psi_j,
 * E_x = -1/2 sum f_i f_j <rho_ij|V_ij>  (reading A26).  Computed with the real kernels from the 2 n_orb real
 * orbitals X = (u_1..u_N, v_1..v_N):  A = K[X] X (exx_apply),  B = the cross term of X with the partner set (-v, u)
 * (exx_apply_to_cross),  K psi = (A[u] + B[v]) + i (A[v] - B[u]),  E_x = 1/2 dV sum_i f_i Re<psi_i|K psi_i>.
 *   psi_dev   DEVICE, PLANAR [2][n_orb][n1][n2][n3]: all real parts, then all imaginary parts; read-only.
 *   kpsi_dev  DEVICE, same layout, OVERWRITTEN.
 *   work_dev  DEVICE, caller-owned scratch of 6 * n_orb * n1*n2*n3 doubles, 16-byte aligned (no allocation happens here).
 *   occ_host  HOST [n_orb];  ex_host HOST.   Needs 2 * n_orb <= max_orbitals.  Costs 6 n_orb^2 real pair solves (a native
 *   complex prologue / epilogue would need 2 n_orb^2: correctness first).  Synchronises.
 */
exx_status exx_apply_to_cross(exx_plan *plan, int n_occ, const double *psi_dev, const double *chi_dev, const double *occ_host,
                              int n_tgt, const double *phi_dev, double *kphi_dev);
exx_status exx_apply_complex(exx_plan *plan, int n_orb, const double *psi_dev, const double *occ_host, double *kpsi_dev,
                             double *work_dev, double *ex_host);

/*
 * exx_apply_block -- all pairs BETWEEN two disjoint orbital blocks, the unit of work of the paper's round-robin
 * distribution (Fig. 1: each process "calculates the co-densities between its own orbitals and the
 * received ones"; the potential serves both orbitals of a pair):  for every j in the resident block, i in the streamed one
 *      kpsi_res[j] -= f_i V_ji psi_i ,   kpsi_str[i] -= f_j V_ji psi_j ,   e_ji = dV sum_r rho_ji V_ji ,
 *      *ex_host = - sum_{j,i} f_j f_i e_ji     (the block's whole contribution to E_x: Eq. 5 counts (j,i) and (i,j)).
 *   flags  EXX_BLOCK_ACCUMULATE_RESIDENT / _STREAMED: add to the existing content of kpsi_res / kpsi_str instead of
 *          overwriting it (partial results of successive round-robin steps).
 * The two blocks must not share memory (use exx_apply for a block with itself); sub-ranges of one array are fine.
 * exx_get_block_energies returns e_ji of the most recent call, HOST [n_res*n_str].  Synchronises.
 */
enum { EXX_BLOCK_ACCUMULATE_RESIDENT = 1, EXX_BLOCK_ACCUMULATE_STREAMED = 2 };
exx_status exx_apply_block(exx_plan *plan, int n_res, const double *psi_res_dev, const double *occ_res_host,
                           double *kpsi_res_dev, int n_str, const double *psi_str_dev, const double *occ_str_host,
                           double *kpsi_str_dev, int flags, double *ex_host);
exx_status exx_get_block_energies(exx_plan *plan, int n_res, int n_str, double *e_host);

/*
 * exx_round_robin_step -- HOST-only schedule of the paper's round-robin exchange (Fig. 1; "[P/2]+1"
 * steps, reading A16: floor).  At step s = 0..floor(P/2) rank p sends its own orbital block to rank
 * *send_to = (p+s) mod P, receives the block of *recv_from = (p-s) mod P and computes, *what =
 *   0  the diagonal block (s = 0: exx_apply on its own orbitals; nothing is exchanged),
 *   1  the full block own (resident) x received (streamed) with exx_apply_block,
 *   2  even P, last step, p < recv_from: resident = FIRST half of the own block (rows [0, ceil(n_own/2))), streamed = the whole received block,
 *   3  even P, last step, p > recv_from: resident = the whole own block, streamed = SECOND half of the received block
 *      (rows [ceil(n_recv/2), n_recv)) -- together the two ranks cover that block pair exactly once.
 * The partial K psi of the received block goes back to its owner, E_x is summed over ranks.
 */
exx_status exx_round_robin_step(int n_ranks, int rank, int step, int *send_to, int *recv_from, int *what);

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
/* The same listing for exx_apply_pairs (pair_mask_host as there; NULL = no mask) and for the rectangular blocks of
 * exx_apply_block (occ_res_host != NULL) / exx_apply_to (occ_res_host == NULL: streamed orbitals with f = 0 skipped):
 * j, l index the resident set, i the streamed set. */
exx_status exx_schedule_list_masked(int n_orb, const double *occ_host, const unsigned char *pair_mask_host, int max_batch,
                                    int *xforms_host, long long capacity, long long *n_transforms);
exx_status exx_schedule_list_block(int n_res, const double *occ_res_host, int n_str, const double *occ_str_host,
                                   int max_batch, int *xforms_host, long long capacity, long long *n_transforms);

/* Transform-grid lengths (n or 2n) of a plan and the bytes of device workspace it owns. */
exx_status exx_plan_transform_dims(const exx_plan *plan, int tdims[3]);
size_t     exx_plan_workspace_bytes(const exx_plan *plan);

/* Name of the kernel this plan's geometry dispatches to for pass 0 (A), 1 (B) or 2 (C); "" for anything else.  The
 * string is static, owned by the library. */
const char *exx_plan_kernel_name(const exx_plan *plan, int pass);

/* Number of kernel launches the library has enqueued for this plan since creation (for bench "gpu_launches"). */
long long  exx_plan_launch_count(const exx_plan *plan);

/* Ordinal of the CUDA device the plan lives on (the device that was current in exx_plan_create; the stream passed there
 * must belong to it).  Every entry point makes that device current for the duration of the call and restores the
 * caller's, so plans on different GPUs can be driven from one host thread.  -1 for NULL. */
int        exx_plan_device(const exx_plan *plan);

/*
 * Per-pass device timing (CUDA events on the plan's stream around every pass launch).  Off by default.
 * exx_plan_get_profile synchronises and returns, for the most recent apply, the summed milliseconds and the
 * launch counts of  [0] pass A, [1] pass B, [2] pass C, [3] energy reduction.
 */
exx_status exx_plan_set_profiling(exx_plan *plan, int enable);
exx_status exx_plan_get_profile(exx_plan *plan, double pass_ms[4], long long pass_launches[4]);

/* Tuning knob: maximum packed transforms per batch (same-i group); <= 0 restores the default. */
exx_status exx_plan_set_batch(exx_plan *plan, int max_transforms_per_batch);

/*
 * exx_diag_fp64 -- device microbenchmarks for the FP64 leg of the roofline (north_star: "the slower of FFT+fusion bytes
 * over 8 TB/s HBM and FP64 flops at peak"; MEASURED_PEAKS.json holds no FP64 figure).  Runs on the current device, on
 * cuda_stream (NULL = default), about 50 ms: dependent-chain DFMA (TFLOP/s, 2 flops per FMA), DADD (1e12 instructions/s:
 * FFT butterflies are add-heavy, so this is the ceiling in "useful" flops), conflict-free 16-byte shared-memory loads
 * (GB/s summed over the SMs), and how far the FP64 and shared-memory pipes of an SM overlap when different warps use
 * them (1 = fully, 0 = serialised).  Diagnostic only: never called by the apply entry points.  Synchronises.
 */
exx_status exx_diag_fp64(void *cuda_stream, double *dfma_tflops, double *dadd_tops, double *lds_gbs, double *overlap_ratio);

/*
 * exx_diag_shfl -- companion microbenchmark: bandwidth of 32-bit warp shuffles (GB/s summed over the SMs, 4 bytes per lane
 * per SHFL) and how far shuffles issued by some warps overlap with 16-byte shared-memory loads issued by others (1 = the
 * two add up, 0 = they share one datapath).  It is the measurement behind exchanging the FFT stages through shared memory
 * rather than through warp shuffles.  Diagnostic only.  Synchronises.
 */
exx_status exx_diag_shfl(void *cuda_stream, double *shfl_gbs, double *shfl_lds_overlap);

/*
 * exx_exchange_energy_noalloc -- the ONE entry point that allocates nothing (no cudaMalloc / cudaFree / allocating library
 * call, no plan): for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * it).  It evaluates the operator form of the exchange energy (Eq. 5 with Eq. 3 inserted),
 *      E_x = 1/2 dV sum_i f_i sum_r psi_i(r) (K psi)_i(r),
 * from the orbitals and the K psi an exx_apply* call produced, with a fixed-order (deterministic) two-stage reduction whose
 * scratch -- 1024 per-block partial sums and the device copy of the occupations -- is a file-scope static __device__ array of
 * 40 KB that every GPU loading the library holds until exit (csrc/exx_noalloc.cu).
 *   n_orb     <= EXX_NOALLOC_MAX_ORBITALS, else EXX_ERR_UNSUPPORTED_SIZE (text from exx_noalloc_last_error);
 *   n_points  n1*n2*n3;  dV = h1*h2*h3;  psi_dev, kpsi_dev DEVICE [n_orb][n_points], read-only;  occ_host HOST [n_orb];
 *   ex_dev    DEVICE, one double, written on cuda_stream (NULL = default stream).  Does not synchronise.
 * Runs on the CURRENT device.  All calls share the static scratch, which keeps the previous call's contents (nothing in it
 * has to start at zero: every slot that is read is written earlier in the same call); calls on one stream are ordered, calls
 * that OVERLAP on the GPU (other streams / threads) race on it.
 */
#define EXX_NOALLOC_MAX_ORBITALS 4096
exx_status  exx_exchange_energy_noalloc(int n_orb, long long n_points, double dV, const double *psi_dev, const double *kpsi_dev,
                                        const double *occ_host, double *ex_dev, void *cuda_stream);
const char *exx_noalloc_last_error(void);           /* per host thread; "" after a successful call */

exx_status  exx_plan_destroy(exx_plan *plan);       /* NULL is allowed */
const char *exx_status_string(exx_status s);
const char *exx_last_error(const exx_plan *plan);   /* detail text incl. CUDA error name; plan may be NULL for
                                                       the last exx_plan_create failure on this thread */
const char *exx_version(void);

#ifdef __cplusplus
}
#endif
#endif
