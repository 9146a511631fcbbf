// exx_api.cu -- plan, tables, pair scheduling and the C ABI of libexx_b200 (include/exx.h).
//
// Hot path per same-(j,l) batch (PAPER.md:113-117 kernels 1-3, fused): pass A -> pass B -> pass C -> energy reduce,
// all enqueued on the plan's stream; the host only schedules.  No CPU fallback exists anywhere in this file:
// without a usable CUDA device every computing entry point returns EXX_ERR_CUDA.
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda.h>               // CUtensorMap + the prototype of cuTensorMapEncodeTiled (resolved at run time, libcuda is not linked)
#include <nvtx3/nvToolsExt.h>   // header-only; the ranges cost nothing unless a tool (nsys, ncu --nvtx) attaches

#include "../../include/exx.h"
#include "exx_launch.h"
#include "exx_sched.hpp"

using namespace exx;

namespace {

thread_local std::string g_create_error;

constexpr double kPi = 3.14159265358979323846264338327950288;

// ------------------------------------------------------------------------------------------ small kernels

// Periodic Fourier-space kernel on the symmetric index range s = 0..T/2 per axis (m = s):
// K^ = 4 pi / |G|^2, G = 2 pi (m1/(t1 h1), m2/(t2 h2), m3/(t3 h3)), K^(0) = 0; times 1/T_tot (inverse FFT norm).
__global__ void ks_periodic_kernel(double* ks, int na, int nb, int nc, double ga, double gb, double gc, double scale) {
    const long long total = static_cast<long long>(na) * nb * nc;
    for (long long x = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; x < total;
         x += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int sc = static_cast<int>(x % nc);
        const int sb = static_cast<int>((x / nc) % nb);
        const int sa = static_cast<int>(x / (static_cast<long long>(nc) * nb));
        const double g1 = ga * sa, g2 = gb * sb, g3 = gc * sc;
        const double gg = g1 * g1 + g2 * g2 + g3 * g3;
        ks[x] = (x == 0) ? 0.0 : scale * 4.0 * kPi / gg;
    }
}

// g'[a][b][c] = g[a][b][c] * (1/2 per zero index): folds the even mirror extension of the Hockney kernel.
__global__ void halve_origin_planes_kernel(double* g, int na, int nb, int nc) {
    const long long total = static_cast<long long>(na) * nb * nc;
    for (long long x = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; x < total;
         x += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int c = static_cast<int>(x % nc);
        const int b = static_cast<int>((x / nc) % nb);
        const int a = static_cast<int>(x / (static_cast<long long>(nc) * nb));
        double f = 1.0;
        if (a == 0) f *= 0.5;
        if (b == 0) f *= 0.5;
        if (c == 0) f *= 0.5;
        g[x] *= f;
    }
}

// out[o][k][i] = scale * sum_a 2 cos(2 pi a k / T) in[o][a][i],  k = 0..n_out-1  (one axis of the DFT of the
// even extension g_ext of the free-BC table; the index-n plane of g_ext is zero, reading A8).
__global__ void cos_transform_kernel(const double* in, double* out, long long outer, int n_in, int n_out, long long inner,
                                     int T, double scale) {
    const long long total = outer * n_out * inner;
    for (long long x = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; x < total;
         x += static_cast<long long>(gridDim.x) * blockDim.x) {
        const long long i = x % inner;
        const int k = static_cast<int>((x / inner) % n_out);
        const long long o = x / (inner * n_out);
        const double* src = in + o * n_in * inner + i;
        double s = 0.0, comp = 0.0;
        for (int a = 0; a < n_in; ++a) {
            const int m = static_cast<int>((static_cast<long long>(a) * k) % T);
            const double term = 2.0 * cospi(2.0 * m / T) * src[a * inner];
            const double y = term - comp;                 // Kahan
            const double t = s + y;
            comp = (t - s) - y;
            s = t;
        }
        out[x] = scale * s;
    }
}

// ks_perm[sb][p][sa] = ks_sym[sa][sb][sc(p)]: the c index in the digit-scrambled order of the in-tile FFT
// (position p = k1*QC + k2 holds frequency kc = k1 + PC*k2) and the symmetric a index fastest, so that the lanes of a
// pass-B warp (consecutive k1 of one column) read K^ contiguously.
__global__ void permute_kernel_axes(const double* ks_sym, double* ks_perm, int nah, int nbh, int tc, int pc, int qc) {
    const int nch = tc / 2 + 1;
    const long long total = static_cast<long long>(nbh) * tc * nah;
    for (long long x = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; x < total;
         x += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int sa = static_cast<int>(x % nah);
        const int p = static_cast<int>((x / nah) % tc);
        const int sb = static_cast<int>(x / (static_cast<long long>(nah) * tc));
        const int kc = (p / qc) + pc * (p % qc);
        const int sc = kc <= tc - kc ? kc : tc - kc;
        ks_perm[x] = ks_sym[(static_cast<long long>(sa) * nbh + sb) * nch + sc];
    }
}

// General periodic cells: ks_perm[kb][p][ka] = scale * table[ka][kb][kc(p)], every frequency index along a and b, the c
// index in the digit-scrambled order of the in-tile FFT (position p = k1*QC + k2 holds frequency kc = k1 + PC*k2).
__global__ void permute_full_kernel(const double* table, double* ks_perm, int ta, int tb, int tc, int pc, int qc, double scale) {
    const long long total = static_cast<long long>(tb) * tc * ta;
    for (long long x = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; x < total;
         x += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int ka = static_cast<int>(x % ta);
        const int p = static_cast<int>((x / ta) % tc);
        const int kb = static_cast<int>(x / (static_cast<long long>(ta) * tc));
        const int kc = (p / qc) + pc * (p % qc);
        ks_perm[x] = scale * table[(static_cast<long long>(ka) * tb + kb) * tc + kc];
    }
}

// ks[x] *= scale  (host-supplied periodic Fourier table: fold in the 1/T_tot of the inverse transform)
__global__ void scale_kernel(double* ks, long long total, double scale) {
    for (long long x = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; x < total;
         x += static_cast<long long>(gridDim.x) * blockDim.x)
        ks[x] *= scale;
}

// e_ij = dV * sum over tiles of the per-CTA partial sums of pass C, fixed order (deterministic).
// square (rect = 0): e_mat is [n][n], ld = n, written symmetrically; rect = 1: e_mat is [n_res][n_str], ld = n_str, entry (j,i).
__global__ void reduce_energy_kernel(const double* epart, int tiles, const XformDesc* desc, int j, int l, int n_orb, int rect, double dV,
                                     double* e_mat) {
    __shared__ double sh[2][256];
    const int t = blockIdx.x;
    const double* ep = epart + static_cast<size_t>(t) * tiles * 2;
    double s1 = 0.0, s2 = 0.0;
    for (int k = threadIdx.x; k < tiles; k += blockDim.x) { s1 += ep[2 * k]; s2 += ep[2 * k + 1]; }
    sh[0][threadIdx.x] = s1; sh[1][threadIdx.x] = s2;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) { sh[0][threadIdx.x] += sh[0][threadIdx.x + o]; sh[1][threadIdx.x] += sh[1][threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const XformDesc d = desc[t];
        if (d.flags & 1) {
            const double e1 = dV * sh[0][0];
            e_mat[static_cast<size_t>(j) * n_orb + d.i] = e1;
            if (!rect) e_mat[static_cast<size_t>(d.i) * n_orb + j] = e1;
        }
        if (d.flags & 2) {
            const double e2 = dV * sh[1][0];
            e_mat[static_cast<size_t>(l) * n_orb + d.i] = e2;
            if (!rect) e_mat[static_cast<size_t>(d.i) * n_orb + l] = e2;
        }
    }
}

// E_x = -1/2 sum_{i,j} f_i f_j e_ij over ordered pairs (Eq. 5), fixed-order tree.  e_mat is
// [n_rows][n_cols] with row occupations occ_r and column occupations occ_c; the square apply passes the same set twice
// and scale = -1/2; a rectangular block between two disjoint sets holds each of its pairs once but Eq. 5 counts both
// orders, so scale = -1.
__global__ void exchange_energy_kernel(const double* e_mat, const double* occ_r, const double* occ_c, int n_rows, int n_cols, double scale,
                                       double* ex) {
    __shared__ double sh[1024];
    const long long total = static_cast<long long>(n_rows) * n_cols;
    double s = 0.0;
    for (long long x = threadIdx.x; x < total; x += blockDim.x) {
        const int i = static_cast<int>(x / n_cols), j = static_cast<int>(x % n_cols);
        s += occ_r[i] * occ_c[j] * e_mat[x];
    }
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *ex = scale * sh[0];
}

// Complex orbitals psi = u + i v by real building blocks (exx_apply_complex).  X = (u_1..u_N, v_1..v_N) is the caller's
// planar array; jx = (-v_1..-v_N, u_1..u_N) is the partner set of the cross term.
__global__ void complex_partner_kernel(const double* x, double* jx, long long nm) {      // nm = N * M
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < nm;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        jx[k] = -x[nm + k];
        jx[nm + k] = x[k];
    }
}
// K psi = (A[u] + B[v]) + i (A[v] - B[u]) written over out = [2][N][M]; per-block partial sums of
// sum_i f_i Re <psi_i | K psi_i> = sum_i f_i sum_r (u_i Kre_i + v_i Kim_i) in a fixed order (deterministic).
__global__ void complex_combine_kernel(const double* x, const double* a, const double* b, const double* occ, double* out,
                                       long long m_points, int n_orb, double* partial) {
    __shared__ double sh[256];
    const long long nm = m_points * n_orb;
    double s = 0.0;
    for (long long k = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; k < nm;
         k += static_cast<long long>(gridDim.x) * blockDim.x) {
        const double kre = a[k] + b[nm + k], kim = a[nm + k] - b[k];
        out[k] = kre;
        out[nm + k] = kim;
        s += occ[k / m_points] * (x[k] * kre + x[nm + k] * kim);
    }
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) partial[blockIdx.x] = sh[0];
}
__global__ void complex_energy_kernel(const double* partial, int n, double scale, double* ex) {
    __shared__ double sh[256];
    double s = 0.0;
    for (int k = threadIdx.x; k < n; k += blockDim.x) s += partial[k];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = blockDim.x / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *ex = scale * sh[0];
}

}  // namespace

// ------------------------------------------------------------------------------------------ plan
struct exx_plan {
    int n[3], t[3];
    double h[3];
    double dV;
    int bc;
    long long M;
    Geometry geo;
    int max_orb;
    int max_batch;
    cudaStream_t stream;
    double2* tw[3];
    double2* twb;           // [b2*R1 + q] = W_TB^{b2 q}
    double2* twc_rot;       // [n2*NCLS + cls] = W_TC^{n2 (k1 + PC r)}: the rotated c-axis twiddles of pass C's TMA-gather variant
    double* ks;             // [TB/2+1][TC][TA/2+1], c index in scrambled order (see permute_kernel_axes)
    double2* w1;
    size_t w1_elems_per_xform;
    double* epart;
    double* e_mat;
    double* occ_dev;
    XformDesc* desc_dev;
    size_t desc_cap;
    XformDesc* desc_pinned;
    double* occ_pinned;
    double* ex_dev;
    double* ex_pinned;
    cudaEvent_t upload_done;
    cudaStream_t copy_stream;   // exx_apply_host: finished K psi rows leave while later block-rows compute
    cudaEvent_t row_done, copy_done;
    double* psi_stage;
    double* kpsi_stage;
    size_t stage_elems;
    KernelInfo info_a, info_b, info_c;
    alignas(64) unsigned char w1_map[128];   // CUtensorMap of W1 for pass C's TMA tile gather (info_c.needs_w1_map)
    long long launches;
    int device;             // ordinal of the device the plan was created on; every entry point switches to it
    int last_rows, last_cols;   // shape of the energy matrix the most recent apply left in e_mat (0: none)
    int last_rect;          // 1: that matrix is a rectangular block [n_res][n_str], 0: the symmetric [n][n] one
    int custom_kernel;      // periodic BC with a host-supplied Fourier table
    int fullk;              // that table covers every frequency index (general cell, exx_plan_create_general): ks is [TB][TC][TA]
    int profiling;
    std::vector<cudaEvent_t> events;   // 5 per batch when profiling (pool grown by exx_plan_set_profiling / set_batch)
    size_t events_used;
    Schedule sched;         // reserved for the largest apply at creation: exx_apply* allocate nothing
    std::vector<char> copied;   // exx_apply_host: rows of K psi already on their way to the host
    std::vector<double> occ2;   // exx_apply_complex: occupations (f, f) of the 2N real orbitals (reserved at creation)
    size_t ws_bytes;        // batch workspace (W1 + energy partials)
    size_t fixed_bytes;     // tables, descriptors, pair-energy matrix
    std::string err;
};

namespace {

exx_status fail(exx_plan* p, exx_status s, const std::string& msg) {
    if (p) p->err = msg; else g_create_error = msg;
    return s;
}

exx_status cuda_fail(exx_plan* p, cudaError_t e, const char* what) {
    std::string msg = std::string(what) + ": " + cudaGetErrorName(e) + " (" + cudaGetErrorString(e) + ")";
    cudaGetLastError();
    return fail(p, EXX_ERR_CUDA, msg);
}

#define EXX_CUDA(plan, call)                                             \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return cuda_fail(plan, e__, #call);      \
    } while (0)

bool is_device_pointer(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// [k1*Q + n2] = W_T^{n2 k1};  roots[m] = W_T^m.  long double trigonometry, rounded once (no recurrences).
void host_tables(int T, std::vector<double2>& tw, std::vector<double2>& roots) {
    const int P = split_p(T), Q = split_q(T);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    roots.resize(T);
    for (int m = 0; m < T; ++m) {
        const long double ang = two_pi * m / T;
        roots[m] = make_double2(static_cast<double>(cosl(ang)), static_cast<double>(-sinl(ang)));
    }
    tw.resize(T);
    for (int k1 = 0; k1 < P; ++k1)
        for (int n2 = 0; n2 < Q; ++n2) tw[k1 * Q + n2] = roots[(k1 * n2) % T];
}

void split_of(int T, int* P, int* Q) { *P = split_p(T); *Q = split_q(T); }

void bsplit_of(int T, int* R1, int* R2) { *R1 = r1_of(T); *R2 = r2_of(T); }

struct DeviceGuard {                                        // makes the plan's device current for the scope of an entry point
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev) {
        if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; ok = false; return; }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) { cudaGetLastError(); ok = false; }
    }
    ~DeviceGuard() {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};
#define EXX_ENTER(plan)                                                                       \
    DeviceGuard guard__((plan)->device);                                                      \
    if (!guard__.ok) return fail(plan, EXX_ERR_CUDA, "cannot switch to the plan's CUDA device")

void free_workspace(exx_plan* p) {
    if (p->w1) cudaFree(p->w1);
    if (p->epart) cudaFree(p->epart);
    p->w1 = nullptr;
    p->epart = nullptr;
}

// upper bound of the number of batches of any apply of this plan with batches of max_batch transforms
size_t max_batches(const exx_plan* p, int max_batch) {
    const size_t n = static_cast<size_t>(p->max_orb), rows = (n + 1) / 2;
    return rows * ((n + max_batch - 1) / max_batch);
}

// event pool for per-pass profiling: 5 events per batch of the largest apply
exx_status grow_event_pool(exx_plan* p) {
    const size_t need = max_batches(p, p->max_batch) * 5;
    try {
        p->events.reserve(need);
    } catch (const std::bad_alloc&) {
        return fail(p, EXX_ERR_ALLOC, "out of host memory (event pool)");
    }
    while (p->events.size() < need) {
        cudaEvent_t ev;
        EXX_CUDA(p, cudaEventCreate(&ev));
        p->events.push_back(ev);
    }
    return EXX_OK;
}

// 5-D tensor map of W1 [t][q][pch][a][b2][pin] for pass C's tile gather: dimensions fastest first
// (2 CHUNK doubles, R2, na, NPCH, R1 * max_batch), box = (2 CHUNK, 1, 1, NPCH, R1) = the whole tile of one transform, landing
// dense (the layout the *_tg phase functions of exx_passes.cuh read).
exx_status encode_w1_map(exx_plan* p, double2* w1, int max_batch, unsigned char out[128]) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*, const cuuint32_t*,
                                 const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static_assert(sizeof(CUtensorMap) == 128, "CUtensorMap size");
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn || qr != cudaDriverEntryPointSuccess) {
        cudaGetLastError();
        return fail(p, EXX_ERR_CUDA, "the driver does not provide cuTensorMapEncodeTiled");
    }
    int r1 = 0, r2 = 0;
    bsplit_of(p->t[1], &r1, &r2);
    const cuuint64_t chunk = static_cast<cuuint64_t>(p->geo.chunk), npch = static_cast<cuuint64_t>(p->t[2]) / chunk, na = static_cast<cuuint64_t>(p->n[0]);
    const cuuint64_t dims[5] = {2 * chunk, static_cast<cuuint64_t>(r2), na, npch, static_cast<cuuint64_t>(r1) * max_batch};
    const cuuint64_t strides[4] = {chunk * 16, r2 * chunk * 16, na * r2 * chunk * 16, npch * na * r2 * chunk * 16};
    const cuuint32_t box[5] = {static_cast<cuuint32_t>(2 * chunk), 1, 1, static_cast<cuuint32_t>(npch), static_cast<cuuint32_t>(r1)};
    const cuuint32_t estr[5] = {1, 1, 1, 1, 1};
    CUtensorMap map;
    const CUresult r = reinterpret_cast<EncodeFn>(fn)(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 5, w1, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                                      CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(p, EXX_ERR_CUDA, "cuTensorMapEncodeTiled failed (" + std::to_string(static_cast<int>(r)) + ")");
    std::memcpy(out, &map, 128);
    return EXX_OK;
}

// The new buffers are allocated BEFORE the old ones are released: a failed request (e.g. an absurd batch size) leaves
// the plan exactly as it was, with its previous workspace and batch size.
exx_status alloc_workspace(exx_plan* p, int max_batch) {
    const size_t w1_bytes = p->w1_elems_per_xform * sizeof(double2) * static_cast<size_t>(max_batch);
    const size_t ep_bytes = static_cast<size_t>(max_batch) * p->info_c.tiles * 2 * sizeof(double);
    double2* w1 = nullptr;
    double* epart = nullptr;
    if (cudaMalloc(&w1, w1_bytes) != cudaSuccess) {
        cudaGetLastError();
        return fail(p, EXX_ERR_ALLOC, "cudaMalloc(workspace W1) failed; the previous workspace is kept");
    }
    if (cudaMalloc(&epart, ep_bytes) != cudaSuccess) {
        cudaGetLastError();
        cudaFree(w1);
        return fail(p, EXX_ERR_ALLOC, "cudaMalloc(energy partials) failed; the previous workspace is kept");
    }
    if (p->info_a.needs_w1_map || p->info_c.needs_w1_map) {
        unsigned char map[128];
        const exx_status st = encode_w1_map(p, w1, max_batch, map);
        if (st != EXX_OK) { cudaFree(w1); cudaFree(epart); return st; }
        std::memcpy(p->w1_map, map, 128);
    }
    free_workspace(p);
    p->w1 = w1;
    p->epart = epart;
    p->max_batch = max_batch;
    p->ws_bytes = w1_bytes + ep_bytes;
    return p->profiling ? grow_event_pool(p) : EXX_OK;
}

// Transforms per batch: as many as fit a 4 GiB intermediate, at most 128.  Measured on B200: a larger intermediate
// makes the scattered W1 stores of pass A miss the TLB (256^3 free BC, 8 GiB: pass A 1.6x slower), while longer
// batches than that gain nothing.
int default_batch(const exx_plan* p) {
    const double per = static_cast<double>(p->w1_elems_per_xform) * sizeof(double2);
    long long b = static_cast<long long>(4.0 * 1024 * 1024 * 1024 / per);
    if (b < 1) b = 1;
    if (b > 128) b = 128;
    return static_cast<int>(b);
}

// general periodic cell: the host table K^[m1][m2][m3] on the full FFT index grid, 1/T_tot folded in here
exx_status build_full_fourier_kernel(exx_plan* p, const double* khat_full_host) {
    const size_t total = static_cast<size_t>(p->t[0]) * p->t[1] * p->t[2];
    double* tmp = nullptr;
    if (cudaMalloc(&p->ks, total * sizeof(double)) != cudaSuccess || cudaMalloc(&tmp, total * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        if (tmp) cudaFree(tmp);
        return fail(p, EXX_ERR_ALLOC, "cudaMalloc(Fourier kernel) failed");
    }
    int pc = 0, qc = 0;
    split_of(p->t[2], &pc, &qc);
    cudaError_t e = cudaMemcpyAsync(tmp, khat_full_host, total * sizeof(double), cudaMemcpyHostToDevice, p->stream);
    if (e == cudaSuccess) {
        permute_full_kernel<<<4096, 256, 0, p->stream>>>(tmp, p->ks, p->t[0], p->t[1], p->t[2], pc, qc, 1.0 / static_cast<double>(total));
        ++p->launches;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaStreamSynchronize(p->stream);
    cudaFree(tmp);
    if (e != cudaSuccess) return cuda_fail(p, e, "building the full Fourier kernel");
    return EXX_OK;
}

exx_status build_fourier_kernel(exx_plan* p, const double* kernel_host) {
    if (p->fullk) return build_full_fourier_kernel(p, kernel_host);
    const int na = p->t[0] / 2 + 1, nb = p->t[1] / 2 + 1, nc = p->t[2] / 2 + 1;
    const size_t total = static_cast<size_t>(na) * nb * nc;
    const size_t total_perm = static_cast<size_t>(na) * nb * p->t[2];
    double* ks_sym = nullptr;
    if (cudaMalloc(&p->ks, total_perm * sizeof(double)) != cudaSuccess || cudaMalloc(&ks_sym, total * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        if (ks_sym) cudaFree(ks_sym);
        return fail(p, EXX_ERR_ALLOC, "cudaMalloc(Fourier kernel) failed");
    }
    struct Guard { double* q; ~Guard() { if (q) cudaFree(q); } } guard{ks_sym};
    auto permute = [&]() -> cudaError_t {
        int pc = 0, qc = 0;
        split_of(p->t[2], &pc, &qc);
        permute_kernel_axes<<<2048, 256, 0, p->stream>>>(ks_sym, p->ks, na, nb, p->t[2], pc, qc);
        ++p->launches;
        cudaError_t e = cudaGetLastError();
        return e != cudaSuccess ? e : cudaStreamSynchronize(p->stream);
    };
    const double t_tot = static_cast<double>(p->t[0]) * p->t[1] * p->t[2];
    const int threads = 256;
    if (p->bc == EXX_BC_PERIODIC) {
        const int blocks = static_cast<int>((total + threads - 1) / threads < 4096 ? (total + threads - 1) / threads : 4096);
        if (kernel_host) {
            // host-supplied Fourier-space filter on the symmetric index range ("only the filter F of kernel 2 would be
            // different"): K^(s1,s2,s3), s_a = 0..n_a/2, even in every index; 1/T_tot folded in here
            EXX_CUDA(p, cudaMemcpyAsync(ks_sym, kernel_host, total * sizeof(double), cudaMemcpyHostToDevice, p->stream));
            scale_kernel<<<blocks, threads, 0, p->stream>>>(ks_sym, static_cast<long long>(total), 1.0 / t_tot);
        } else {
            ks_periodic_kernel<<<blocks, threads, 0, p->stream>>>(ks_sym, na, nb, nc, 2.0 * kPi / (p->t[0] * p->h[0]),
                                                                  2.0 * kPi / (p->t[1] * p->h[1]),
                                                                  2.0 * kPi / (p->t[2] * p->h[2]), 1.0 / t_tot);
        }
        EXX_CUDA(p, cudaGetLastError());
        ++p->launches;
        EXX_CUDA(p, permute());
        return EXX_OK;
    }
    // FREE: K^ = dV * DFT3(g_ext) restricted to the symmetric index range, computed as three cosine transforms of
    // g' (even extension folded); 1/T_tot of the inverse transform folded in.
    const int n0 = p->n[0], n1 = p->n[1], n2 = p->n[2];
    double *g = nullptr, *t1 = nullptr, *t2 = nullptr;
    const size_t gsz = static_cast<size_t>(n0) * n1 * n2;
    const size_t t1sz = static_cast<size_t>(na) * n1 * n2;
    const size_t t2sz = static_cast<size_t>(na) * nb * n2;
    if (cudaMalloc(&g, gsz * sizeof(double)) != cudaSuccess || cudaMalloc(&t1, t1sz * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&t2, t2sz * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        if (g) cudaFree(g);
        if (t1) cudaFree(t1);
        if (t2) cudaFree(t2);
        return fail(p, EXX_ERR_ALLOC, "cudaMalloc(kernel table scratch) failed");
    }
    cudaError_t e = cudaMemcpyAsync(g, kernel_host, gsz * sizeof(double), cudaMemcpyHostToDevice, p->stream);
    auto blocks_for = [&](size_t n) { size_t b = (n + threads - 1) / threads; return static_cast<int>(b < 8192 ? b : 8192); };
    if (e == cudaSuccess) {
        halve_origin_planes_kernel<<<blocks_for(gsz), threads, 0, p->stream>>>(g, n0, n1, n2);
        cos_transform_kernel<<<blocks_for(t1sz), threads, 0, p->stream>>>(g, t1, 1, n0, na, static_cast<long long>(n1) * n2,
                                                                          p->t[0], 1.0);
        cos_transform_kernel<<<blocks_for(t2sz), threads, 0, p->stream>>>(t1, t2, na, n1, nb, n2, p->t[1], 1.0);
        cos_transform_kernel<<<blocks_for(total), threads, 0, p->stream>>>(t2, ks_sym, static_cast<long long>(na) * nb, n2, nc, 1,
                                                                           p->t[2], p->dV / t_tot);
        p->launches += 4;
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = permute();
    cudaFree(g); cudaFree(t1); cudaFree(t2);
    if (e != cudaSuccess) return cuda_fail(p, e, "building the free-BC Fourier kernel");
    return EXX_OK;
}

// One application of the pair machinery.  SQUARE: one orbital set on both sides (i <= j triangle, diagonal pairs,
// symmetric energy matrix).  RECTANGULAR: every pair between a resident set and a disjoint streamed set.
struct Job {
    bool square;
    int n_res, n_str;               // square: both = n_orb
    const double* psi_res;
    const double* psi_str;
    const double* psi_str_epi;      // nullptr, or the set pass C multiplies the potentials with instead of psi_str (exx_apply_to_cross)
    double* kpsi_res;               // nullptr: the resident side receives nothing
    double* kpsi_str;               // nullptr: the streamed side receives nothing
    const double* occ_res;          // host; nullptr: all zero (exx_apply_to)
    const double* occ_str;          // host
    const unsigned char* mask;      // square only, optional
    bool zero_res, zero_str;        // overwrite (true) or accumulate into (false) the outputs
    bool skip_empty_streamed;
    bool energy;                    // pair energies + E_x contribution
    double* kpsi_host;              // square host path: finished rows are copied out on the copy stream
};

// kpsi_host != nullptr (exx_apply_host): K psi_j and K psi_l are final once the last batch of block-row {j,l} has run
// (later block-rows only stream orbitals i > l), so their device-to-host copies overlap the remaining block-rows.
exx_status run_job_unguarded(exx_plan* p, const Job& job) {
    if (!p->w1 || !p->epart) return fail(p, EXX_ERR_ALLOC, "the plan has no batch workspace");
    // wait until the previous apply's descriptor upload has left the pinned staging buffers
    EXX_CUDA(p, cudaEventSynchronize(p->upload_done));
    Schedule& sched = p->sched;
    if (job.square) build_schedule(sched, job.n_str, job.occ_str, p->max_batch, job.mask);
    else build_schedule_rect(sched, job.n_res, job.occ_res, job.n_str, job.occ_str, job.skip_empty_streamed, p->max_batch);
    if (sched.xforms.size() > p->desc_cap) return fail(p, EXX_ERR_INTERNAL, "descriptor capacity exceeded");
    if (!sched.xforms.empty()) std::memcpy(p->desc_pinned, sched.xforms.data(), sched.xforms.size() * sizeof(XformDesc));
    // occupations on the device: [0, max_orb) the rows of the energy matrix (resident set), [max_orb, 2 max_orb) the columns
    double* occ_r_pinned = p->occ_pinned;
    double* occ_c_pinned = p->occ_pinned + p->max_orb;
    for (int k = 0; k < job.n_res; ++k) occ_r_pinned[k] = job.square ? job.occ_str[k] : (job.occ_res ? job.occ_res[k] : 0.0);
    for (int k = 0; k < job.n_str; ++k) occ_c_pinned[k] = job.occ_str[k];
    cudaStream_t s = p->stream;
    if (!sched.xforms.empty())
        EXX_CUDA(p, cudaMemcpyAsync(p->desc_dev, p->desc_pinned, sched.xforms.size() * sizeof(XformDesc), cudaMemcpyHostToDevice, s));
    EXX_CUDA(p, cudaMemcpyAsync(p->occ_dev, p->occ_pinned, sizeof(double) * 2 * p->max_orb, cudaMemcpyHostToDevice, s));
    EXX_CUDA(p, cudaEventRecord(p->upload_done, s));
    if (job.kpsi_res && job.zero_res)
        EXX_CUDA(p, cudaMemsetAsync(job.kpsi_res, 0, sizeof(double) * static_cast<size_t>(job.n_res) * p->M, s));
    if (job.kpsi_str && job.zero_str && !(job.square && job.zero_res))
        EXX_CUDA(p, cudaMemsetAsync(job.kpsi_str, 0, sizeof(double) * static_cast<size_t>(job.n_str) * p->M, s));
    const int e_ld = job.n_str;
    if (job.energy)
        EXX_CUDA(p, cudaMemsetAsync(p->e_mat, 0, sizeof(double) * static_cast<size_t>(job.n_res) * job.n_str, s));

    ArgsAC ac{};
    ac.psi = job.psi_str; ac.psi_r = job.psi_res; ac.kpsi = job.kpsi_str; ac.kpsi_r = job.kpsi_res;
    ac.w1 = p->w1; ac.twc = p->tw[2]; ac.twb = p->twb; ac.epart = p->epart;
    ArgsCX cx{};
    std::memcpy(cx.w1_map, p->w1_map, 128);
    cx.twc_rot = p->twc_rot;
    ac.m_points = p->M; ac.na = p->n[0];
    ArgsB ab{};
    ab.w1 = p->w1; ab.twa = p->tw[0]; ab.ks = p->ks; ab.fullk = p->fullk; ab.tc = p->t[2];
    ab.npch = p->t[2] / p->geo.chunk;

    p->events_used = 0;
    const bool prof = p->profiling && sched.batches.size() * 5 <= p->events.size();
    auto mark = [&]() -> cudaError_t {
        if (!prof) return cudaSuccess;
        return cudaEventRecord(p->events[p->events_used++], s);
    };
    if (job.kpsi_host) std::fill(p->copied.begin(), p->copied.begin() + job.n_str, 0);
    for (const Batch& b : sched.batches) {
        ac.desc = p->desc_dev + b.first;
        ac.j = b.j; ac.l = b.l; ac.fj = b.fj; ac.fl = b.fl; ac.count = b.count;
        ac.jd = job.square ? b.j : -1;
        ac.ld = job.square ? b.l : -2;
        EXX_CUDA(p, mark());
        EXX_CUDA(p, launch_pass_a(p->geo, ac, cx, s, nullptr));
        EXX_CUDA(p, mark());
        EXX_CUDA(p, launch_pass_b(p->geo, ab, b.count, s, nullptr));
        EXX_CUDA(p, mark());
        if (job.psi_str_epi) {                             // Kernel 3 multiplies V[phi psi_i] with chi_i instead of psi_i
            ArgsAC acc = ac;
            acc.psi = job.psi_str_epi;
            EXX_CUDA(p, launch_pass_c(p->geo, acc, cx, s, nullptr));
        } else {
            EXX_CUDA(p, launch_pass_c(p->geo, ac, cx, s, nullptr));
        }
        EXX_CUDA(p, mark());
        p->launches += 3;
        if (job.energy) {
            reduce_energy_kernel<<<b.count, 256, 0, s>>>(p->epart, p->info_c.tiles, ac.desc, b.j, b.l, e_ld, job.square ? 0 : 1, p->dV, p->e_mat);
            EXX_CUDA(p, cudaGetLastError());
            ++p->launches;
        }
        EXX_CUDA(p, mark());
        const bool row_ends = (&b == &sched.batches.back()) || ((&b)[1].j != b.j);
        if (job.kpsi_host && row_ends) {
            const size_t rows = b.l >= 0 ? 2 : 1, off = static_cast<size_t>(b.j) * p->M;
            EXX_CUDA(p, cudaEventRecord(p->row_done, s));
            EXX_CUDA(p, cudaStreamWaitEvent(p->copy_stream, p->row_done, 0));
            EXX_CUDA(p, cudaMemcpyAsync(job.kpsi_host + off, job.kpsi_res + off, rows * p->M * sizeof(double), cudaMemcpyDeviceToHost, p->copy_stream));
            for (size_t r = 0; r < rows; ++r) p->copied[b.j + r] = 1;
        }
    }
    if (job.kpsi_host) {                                   // rows of block-rows without any pair (all occupations zero)
        EXX_CUDA(p, cudaEventRecord(p->row_done, s));
        EXX_CUDA(p, cudaStreamWaitEvent(p->copy_stream, p->row_done, 0));
        for (int r = 0; r < job.n_str; ++r)
            if (!p->copied[r])
                EXX_CUDA(p, cudaMemcpyAsync(job.kpsi_host + static_cast<size_t>(r) * p->M, job.kpsi_res + static_cast<size_t>(r) * p->M,
                                            p->M * sizeof(double), cudaMemcpyDeviceToHost, p->copy_stream));
        EXX_CUDA(p, cudaEventRecord(p->copy_done, p->copy_stream));
        EXX_CUDA(p, cudaStreamWaitEvent(s, p->copy_done, 0));
    }
    if (job.energy) {
        exchange_energy_kernel<<<1, 1024, 0, s>>>(p->e_mat, p->occ_dev, p->occ_dev + p->max_orb, job.n_res, job.n_str,
                                                  job.square ? -0.5 : -1.0, p->ex_dev);
        EXX_CUDA(p, cudaGetLastError());
        ++p->launches;
        p->last_rows = job.n_res; p->last_cols = job.n_str; p->last_rect = job.square ? 0 : 1;
    } else {
        p->last_rows = p->last_cols = 0;
    }
    return EXX_OK;
}

// No exception crosses the C ABI: the schedule vectors are reserved at plan creation, so nothing in the hot path
// allocates, and anything that throws all the same is turned into a status code here.
struct NvtxRange {                                          // one named range per apply on the tools' timeline
    explicit NvtxRange(const char* name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

exx_status run_job(exx_plan* p, const Job& job) {
    NvtxRange range(job.square ? (job.mask ? "exx_apply_pairs" : (job.kpsi_host ? "exx_apply_host" : "exx_apply"))
                               : (job.kpsi_str ? "exx_apply_block" : "exx_apply_to"));
    exx_status st;
    try {
        st = run_job_unguarded(p, job);
    } catch (const std::bad_alloc&) {
        st = fail(p, EXX_ERR_ALLOC, "out of host memory in exx_apply");
    } catch (...) {
        st = fail(p, EXX_ERR_INTERNAL, "unexpected exception in exx_apply");
    }
    if (st != EXX_OK && job.kpsi_host && p->copy_stream) {
        // device-to-host copies of finished rows may still be in flight into the caller's buffer
        cudaStreamSynchronize(p->copy_stream);
        cudaStreamSynchronize(p->stream);
        cudaGetLastError();
    }
    return st;
}

bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

bool ranges_overlap(const double* a, size_t na, const double* b, size_t nb) {
    const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), a1 = a0 + na * sizeof(double);
    const uintptr_t b0 = reinterpret_cast<uintptr_t>(b), b1 = b0 + nb * sizeof(double);
    return a0 < b1 && b0 < a1;
}

// common checks of the device-pointer entry points: psi-like arrays must be 16-byte aligned device memory (the TMA
// bulk copies and bulk reduce-adds of passes A / C move 16-byte units), outputs must not overlap any input
exx_status check_set(exx_plan* p, int n, const double* psi, const double* kpsi, const char* what) {
    if (n < 1 || n > p->max_orb) return fail(p, EXX_ERR_INVALID_ARG, std::string(what) + ": orbital count outside [1, max_orbitals]");
    if (!psi) return fail(p, EXX_ERR_INVALID_ARG, std::string(what) + ": NULL orbital array");
    if (!is_device_pointer(psi) || (kpsi && !is_device_pointer(kpsi)))
        return fail(p, EXX_ERR_BAD_POINTER, std::string(what) + ": orbital arrays must be device pointers");
    if (!aligned16(psi) || (kpsi && !aligned16(kpsi)))
        return fail(p, EXX_ERR_INVALID_ARG, std::string(what) + ": orbital arrays must be 16-byte aligned");
    if ((p->M & 1) != 0) return fail(p, EXX_ERR_INTERNAL, "odd grid size");
    return EXX_OK;
}

exx_status check_apply_args(exx_plan* p, int n_orb, const void* psi, const double* occ, const void* kpsi, const void* ex) {
    if (!p) return EXX_ERR_INVALID_ARG;
    if (!psi || !occ || !kpsi || !ex) return fail(p, EXX_ERR_INVALID_ARG, "NULL argument");
    if (n_orb < 1 || n_orb > p->max_orb) return fail(p, EXX_ERR_INVALID_ARG, "n_orb outside [1, max_orbitals]");
    return EXX_OK;
}

exx_status square_device_apply(exx_plan* p, int n_orb, const double* psi_dev, const double* occ_host, const unsigned char* mask,
                               double* kpsi_dev) {
    exx_status st = check_set(p, n_orb, psi_dev, kpsi_dev, "exx_apply");
    if (st != EXX_OK) return st;
    if (is_device_pointer(occ_host)) return fail(p, EXX_ERR_BAD_POINTER, "occ_host must be a host pointer");
    const size_t elems = static_cast<size_t>(n_orb) * p->M;
    if (ranges_overlap(psi_dev, elems, kpsi_dev, elems)) return fail(p, EXX_ERR_INVALID_ARG, "kpsi must not overlap psi");
    Job job{};
    job.square = true;
    job.n_res = job.n_str = n_orb;
    job.psi_res = job.psi_str = psi_dev;
    job.kpsi_res = job.kpsi_str = kpsi_dev;
    job.occ_res = job.occ_str = occ_host;
    job.mask = mask;
    job.zero_res = job.zero_str = true;
    job.energy = true;
    return run_job(p, job);
}

exx_status finish_sync(exx_plan* p, double* ex_host) {
    EXX_CUDA(p, cudaMemcpyAsync(p->ex_pinned, p->ex_dev, sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    *ex_host = *p->ex_pinned;
    return EXX_OK;
}

}  // namespace

// ------------------------------------------------------------------------------------------ C ABI
extern "C" {

const char* exx_version(void) { return "exx-b200 0.2 (sm_100a)"; }

const char* exx_status_string(exx_status s) {
    switch (s) {
        case EXX_OK: return "EXX_OK";
        case EXX_ERR_INVALID_ARG: return "EXX_ERR_INVALID_ARG";
        case EXX_ERR_UNSUPPORTED_SIZE: return "EXX_ERR_UNSUPPORTED_SIZE";
        case EXX_ERR_BAD_POINTER: return "EXX_ERR_BAD_POINTER";
        case EXX_ERR_ALLOC: return "EXX_ERR_ALLOC";
        case EXX_ERR_CUDA: return "EXX_ERR_CUDA";
        case EXX_ERR_INTERNAL: return "EXX_ERR_INTERNAL";
    }
    return "EXX_ERR_UNKNOWN";
}

const char* exx_last_error(const exx_plan* plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

exx_status exx_schedule_pairs(int n_orb, const double* occ_host, long long* n_pairs, long long* n_transforms) {
    if (n_orb < 1 || !occ_host || !n_pairs || !n_transforms) return EXX_ERR_INVALID_ARG;
    try {
        Schedule s;
        build_schedule(s, n_orb, occ_host, 1 << 30);
        *n_pairs = s.n_pairs;
        *n_transforms = static_cast<long long>(s.xforms.size());
    } catch (const std::bad_alloc&) {
        return EXX_ERR_ALLOC;
    }
    return EXX_OK;
}

static exx_status list_schedule(const Schedule& s, int* xforms_host, long long capacity, long long* n_transforms) {
    *n_transforms = static_cast<long long>(s.xforms.size());
    for (size_t b = 0; b < s.batches.size(); ++b) {
        const Batch& bt = s.batches[b];
        for (int t = bt.first; t < bt.first + bt.count && t < capacity; ++t) {
            int* row = xforms_host + static_cast<size_t>(t) * 5;
            row[0] = bt.j; row[1] = bt.l; row[2] = s.xforms[t].i; row[3] = s.xforms[t].flags; row[4] = static_cast<int>(b);
        }
    }
    return EXX_OK;
}

exx_status exx_schedule_list(int n_orb, const double* occ_host, int max_batch, int* xforms_host, long long capacity,
                             long long* n_transforms) {
    return exx_schedule_list_masked(n_orb, occ_host, nullptr, max_batch, xforms_host, capacity, n_transforms);
}

exx_status exx_schedule_list_masked(int n_orb, const double* occ_host, const unsigned char* pair_mask_host, int max_batch,
                                    int* xforms_host, long long capacity, long long* n_transforms) {
    if (n_orb < 1 || !occ_host || !n_transforms || capacity < 0 || (capacity > 0 && !xforms_host)) return EXX_ERR_INVALID_ARG;
    try {
        Schedule s;
        build_schedule(s, n_orb, occ_host, max_batch < 1 ? 1 << 30 : max_batch, pair_mask_host);
        return list_schedule(s, xforms_host, capacity, n_transforms);
    } catch (const std::bad_alloc&) {
        return EXX_ERR_ALLOC;
    }
}

exx_status exx_schedule_list_block(int n_res, const double* occ_res_host, int n_str, const double* occ_str_host, int max_batch,
                                   int* xforms_host, long long capacity, long long* n_transforms) {
    if (n_res < 1 || n_str < 1 || !occ_str_host || !n_transforms || capacity < 0 || (capacity > 0 && !xforms_host))
        return EXX_ERR_INVALID_ARG;
    try {
        Schedule s;
        build_schedule_rect(s, n_res, occ_res_host, n_str, occ_str_host, occ_res_host == nullptr, max_batch < 1 ? 1 << 30 : max_batch);
        return list_schedule(s, xforms_host, capacity, n_transforms);
    } catch (const std::bad_alloc&) {
        return EXX_ERR_ALLOC;
    }
}

/* Round-robin exchange of orbital blocks between n_ranks owners (Fig. 1): at step s rank p works on
 * its own block and the block of rank (p - s) mod P, which it receives from that rank, and sends its own block to
 * rank (p + s) mod P.  floor(P/2) + 1 steps (s = 0: the diagonal block) cover every unordered block pair exactly once,
 * except that for even P the last step s = P/2 pairs p with p + P/2 on BOTH ranks: each of the two then takes one half
 * of the resident rows (what = 2: the rank owning the lower block takes the first half of ITS block as resident rows
 * against the whole visiting block; what = 3: the other rank takes the visiting block's second half, streamed, against
 * its whole own block as resident rows). */
exx_status exx_round_robin_step(int n_ranks, int rank, int step, int* send_to, int* recv_from, int* what) {
    if (n_ranks < 1 || rank < 0 || rank >= n_ranks || step < 0 || step > n_ranks / 2 || !send_to || !recv_from || !what)
        return EXX_ERR_INVALID_ARG;
    if (step == 0) {
        *send_to = *recv_from = rank;
        *what = 0;                                         // diagonal block: the square apply of the own orbitals
        return EXX_OK;
    }
    *send_to = (rank + step) % n_ranks;
    *recv_from = ((rank - step) % n_ranks + n_ranks) % n_ranks;
    if (n_ranks % 2 == 0 && step == n_ranks / 2) *what = rank < *recv_from ? 2 : 3;
    else *what = 1;                                        // full rectangular block own x visiting
    return EXX_OK;
}

static exx_status create_impl(exx_plan** plan, const int dims[3], const double spacing[3], exx_bc bc, const double* kernel_host,
                              int fullk, int max_orbitals, void* cuda_stream) {
    g_create_error.clear();
    if (!plan || !dims || !spacing) return fail(nullptr, EXX_ERR_INVALID_ARG, "NULL argument");
    *plan = nullptr;
    if (bc != EXX_BC_PERIODIC && bc != EXX_BC_FREE) return fail(nullptr, EXX_ERR_INVALID_ARG, "unknown boundary condition");
    if (bc == EXX_BC_FREE && !kernel_host) return fail(nullptr, EXX_ERR_INVALID_ARG, "free BC needs a kernel table");
    if (max_orbitals < 1) return fail(nullptr, EXX_ERR_INVALID_ARG, "max_orbitals < 1");
    for (int ax = 0; ax < 3; ++ax) {
        if (dims[ax] < 1) return fail(nullptr, EXX_ERR_UNSUPPORTED_SIZE, "non-positive grid length");
        if (!(spacing[ax] > 0.0) || !std::isfinite(spacing[ax])) return fail(nullptr, EXX_ERR_INVALID_ARG, "spacing must be > 0");
    }
    Geometry geo{};
    geo.free_bc = bc == EXX_BC_FREE ? 1 : 0;
    geo.ta = geo.free_bc ? 2 * dims[0] : dims[0];
    geo.tb = geo.free_bc ? 2 * dims[1] : dims[1];
    geo.tc = geo.free_bc ? 2 * dims[2] : dims[2];
    if (!geometry_supported(geo)) return fail(nullptr, EXX_ERR_UNSUPPORTED_SIZE, unsupported_geometry_text());
    geo.chunk = chunk_of(geo);

    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, EXX_ERR_CUDA, std::string("no usable CUDA device: ") + (ce != cudaSuccess ? cudaGetErrorName(ce) : "device count 0"));
    }
    if (kernel_host && is_device_pointer(kernel_host))
        return fail(nullptr, EXX_ERR_BAD_POINTER, "kernel_host must be a host pointer");

    exx_plan* p = new (std::nothrow) exx_plan();
    if (!p) return fail(nullptr, EXX_ERR_ALLOC, "out of host memory");
    if (cudaGetDevice(&p->device) != cudaSuccess || p->device < 0 || p->device >= kMaxDevices) {
        cudaGetLastError();
        delete p;
        return fail(nullptr, EXX_ERR_CUDA, "cannot identify the current CUDA device");
    }
    p->bc = bc;
    p->geo = geo;
    p->dV = 1.0;
    p->M = 1;
    for (int ax = 0; ax < 3; ++ax) {
        p->n[ax] = dims[ax];
        p->h[ax] = spacing[ax];
        p->dV *= spacing[ax];
        p->M *= dims[ax];
    }
    p->t[0] = geo.ta; p->t[1] = geo.tb; p->t[2] = geo.tc;
    p->max_orb = max_orbitals;
    p->stream = static_cast<cudaStream_t>(cuda_stream);
    p->custom_kernel = (bc == EXX_BC_PERIODIC && kernel_host) ? 1 : 0;
    p->fullk = fullk;

    auto bail = [&](exx_status st) {
        g_create_error = p->err;
        exx_plan_destroy(p);
        return st;
    };
    if (query_pass_a(geo, &p->info_a) != cudaSuccess || query_pass_b(geo, &p->info_b) != cudaSuccess ||
        query_pass_c(geo, &p->info_c) != cudaSuccess)
        return bail(fail(p, EXX_ERR_INTERNAL, "no kernel instantiation for this geometry"));
    try {
        reserve_schedule(p->sched, static_cast<size_t>(max_orbitals), static_cast<size_t>(max_orbitals));
        p->copied.assign(static_cast<size_t>(max_orbitals), 0);
        p->occ2.reserve(static_cast<size_t>(max_orbitals));
    } catch (const std::bad_alloc&) {
        return bail(fail(p, EXX_ERR_ALLOC, "out of host memory (schedule storage)"));
    }

    for (int ax = 0; ax < 3; ++ax) {
        std::vector<double2> tw, roots;
        host_tables(p->t[ax], tw, roots);
        const size_t bytes = sizeof(double2) * p->t[ax];
        if (cudaMalloc(&p->tw[ax], bytes) != cudaSuccess) {
            cudaGetLastError();
            return bail(fail(p, EXX_ERR_ALLOC, "cudaMalloc(twiddles) failed"));
        }
        if (cudaMemcpy(p->tw[ax], tw.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError();
            return bail(fail(p, EXX_ERR_CUDA, "twiddle upload failed"));
        }
    }
    {   // twb[b2*R1 + q] = W_TB^{b2 q}: twiddle between the two stages of the b-axis FFT (passes A and C)
        int r1 = 0, r2 = 0;
        bsplit_of(p->t[1], &r1, &r2);
        std::vector<double2> tw, roots, twb(static_cast<size_t>(r1) * r2);
        host_tables(p->t[1], tw, roots);
        for (int b2 = 0; b2 < r2; ++b2)
            for (int q = 0; q < r1; ++q) twb[static_cast<size_t>(b2) * r1 + q] = roots[(b2 * q) % p->t[1]];
        if (cudaMalloc(&p->twb, twb.size() * sizeof(double2)) != cudaSuccess) {
            cudaGetLastError();
            return bail(fail(p, EXX_ERR_ALLOC, "cudaMalloc(twiddles) failed"));
        }
        if (cudaMemcpy(p->twb, twb.data(), twb.size() * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError();
            return bail(fail(p, EXX_ERR_CUDA, "twiddle upload failed"));
        }
    }
    {   // rotated c-axis twiddles (c1_compute_tg): class cls = (k1 = cls % PC, r = cls & 7), entry [n2*NCLS + cls] = W_TC^{n2 (k1 + PC r)}
        int pc = 0, qc = 0;
        split_of(p->t[2], &pc, &qc);
        const int ncls = tg_classes(pc);
        std::vector<double2> tw, roots, rot(static_cast<size_t>(qc) * ncls);
        host_tables(p->t[2], tw, roots);
        for (int n2 = 0; n2 < qc; ++n2)
            for (int cls = 0; cls < ncls; ++cls) {
                const long long m = static_cast<long long>(n2) * ((cls % pc) + pc * (cls & 7));
                rot[static_cast<size_t>(n2) * ncls + cls] = roots[m % p->t[2]];
            }
        if (cudaMalloc(&p->twc_rot, rot.size() * sizeof(double2)) != cudaSuccess) {
            cudaGetLastError();
            return bail(fail(p, EXX_ERR_ALLOC, "cudaMalloc(twiddles) failed"));
        }
        if (cudaMemcpy(p->twc_rot, rot.data(), rot.size() * sizeof(double2), cudaMemcpyHostToDevice) != cudaSuccess) {
            cudaGetLastError();
            return bail(fail(p, EXX_ERR_CUDA, "twiddle upload failed"));
        }
    }

    exx_status st = build_fourier_kernel(p, kernel_host);
    if (st != EXX_OK) return bail(st);

    p->w1_elems_per_xform = static_cast<size_t>(p->n[0]) * p->t[1] * p->t[2];
    st = alloc_workspace(p, default_batch(p));
    if (st != EXX_OK) return bail(st);
    const size_t n = static_cast<size_t>(max_orbitals);
    p->desc_cap = max_transforms(n, n);
    bool ok = cudaMalloc(&p->e_mat, n * n * sizeof(double)) == cudaSuccess &&
              cudaMalloc(&p->occ_dev, 2 * n * sizeof(double)) == cudaSuccess &&
              cudaMalloc(&p->desc_dev, p->desc_cap * sizeof(XformDesc)) == cudaSuccess &&
              cudaMalloc(&p->ex_dev, sizeof(double)) == cudaSuccess &&
              cudaMallocHost(&p->desc_pinned, p->desc_cap * sizeof(XformDesc)) == cudaSuccess &&
              cudaMallocHost(&p->occ_pinned, 2 * n * sizeof(double)) == cudaSuccess &&
              cudaMallocHost(&p->ex_pinned, sizeof(double)) == cudaSuccess &&
              cudaEventCreateWithFlags(&p->upload_done, cudaEventDisableTiming) == cudaSuccess &&
              cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking) == cudaSuccess &&
              cudaEventCreateWithFlags(&p->row_done, cudaEventDisableTiming) == cudaSuccess &&
              cudaEventCreateWithFlags(&p->copy_done, cudaEventDisableTiming) == cudaSuccess;
    if (!ok) {
        cudaGetLastError();
        return bail(fail(p, EXX_ERR_ALLOC, "allocation of plan buffers failed"));
    }
    std::memset(p->occ_pinned, 0, 2 * n * sizeof(double));
    p->fixed_bytes = n * n * sizeof(double) + 2 * n * sizeof(double) + p->desc_cap * sizeof(XformDesc) +
                     sizeof(double) * (fullk ? static_cast<size_t>(p->t[0]) * p->t[1] * p->t[2]
                                             : static_cast<size_t>(p->t[0] / 2 + 1) * (p->t[1] / 2 + 1) * p->t[2]);
    if (cudaMemset(p->e_mat, 0, n * n * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        return bail(fail(p, EXX_ERR_CUDA, "cudaMemset failed"));
    }
    *plan = p;
    return EXX_OK;
}

exx_status exx_plan_create(exx_plan** plan, const int dims[3], const double spacing[3], exx_bc bc, const double* kernel_host,
                           int max_orbitals, void* cuda_stream) {
    return create_impl(plan, dims, spacing, bc, kernel_host, 0, max_orbitals, cuda_stream);
}

exx_status exx_plan_create_general(exx_plan** plan, const int dims[3], double cell_volume, const double* khat_full_host,
                                   int max_orbitals, void* cuda_stream) {
    g_create_error.clear();
    if (!plan || !dims) return fail(nullptr, EXX_ERR_INVALID_ARG, "NULL argument");
    *plan = nullptr;
    if (!khat_full_host) return fail(nullptr, EXX_ERR_INVALID_ARG, "a general periodic cell needs its Fourier-space table");
    if (!(cell_volume > 0.0) || !std::isfinite(cell_volume)) return fail(nullptr, EXX_ERR_INVALID_ARG, "cell_volume must be > 0");
    for (int ax = 0; ax < 3; ++ax)
        if (dims[ax] < 1) return fail(nullptr, EXX_ERR_UNSUPPORTED_SIZE, "non-positive grid length");
    // only dV = cell_volume / (n1 n2 n3) enters the path (energies); it is carried as three equal nominal spacings
    const double h = std::cbrt(cell_volume / (static_cast<double>(dims[0]) * dims[1] * dims[2]));
    const double spacing[3] = {h, h, h};
    return create_impl(plan, dims, spacing, EXX_BC_PERIODIC, khat_full_host, 1, max_orbitals, cuda_stream);
}

exx_status exx_plan_destroy(exx_plan* p) {
    if (!p) return EXX_OK;
    DeviceGuard guard(p->device);
    if (p->stream || p->w1) cudaStreamSynchronize(p->stream);
    if (p->copy_stream) cudaStreamSynchronize(p->copy_stream);
    for (int ax = 0; ax < 3; ++ax) {
        if (p->tw[ax]) cudaFree(p->tw[ax]);
    }
    if (p->ks) cudaFree(p->ks);
    if (p->twb) cudaFree(p->twb);
    if (p->twc_rot) cudaFree(p->twc_rot);
    free_workspace(p);
    if (p->e_mat) cudaFree(p->e_mat);
    if (p->occ_dev) cudaFree(p->occ_dev);
    if (p->desc_dev) cudaFree(p->desc_dev);
    if (p->ex_dev) cudaFree(p->ex_dev);
    if (p->desc_pinned) cudaFreeHost(p->desc_pinned);
    if (p->occ_pinned) cudaFreeHost(p->occ_pinned);
    if (p->ex_pinned) cudaFreeHost(p->ex_pinned);
    if (p->upload_done) cudaEventDestroy(p->upload_done);
    if (p->row_done) cudaEventDestroy(p->row_done);
    if (p->copy_done) cudaEventDestroy(p->copy_done);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (cudaEvent_t ev : p->events) cudaEventDestroy(ev);
    if (p->psi_stage) cudaFree(p->psi_stage);
    if (p->kpsi_stage) cudaFree(p->kpsi_stage);
    cudaGetLastError();
    delete p;
    return EXX_OK;
}

exx_status exx_plan_transform_dims(const exx_plan* p, int tdims[3]) {
    if (!p || !tdims) return EXX_ERR_INVALID_ARG;
    for (int ax = 0; ax < 3; ++ax) tdims[ax] = p->t[ax];
    return EXX_OK;
}

size_t exx_plan_workspace_bytes(const exx_plan* p) { return p ? p->ws_bytes + p->fixed_bytes + 2 * p->stage_elems * sizeof(double) : 0; }

long long exx_plan_launch_count(const exx_plan* p) { return p ? p->launches : 0; }

int exx_plan_device(const exx_plan* p) { return p ? p->device : -1; }

const char* exx_plan_kernel_name(const exx_plan* p, int pass) {
    if (!p) return "";
    const KernelInfo& k = pass == 0 ? p->info_a : pass == 1 ? p->info_b : p->info_c;
    return (pass >= 0 && pass <= 2 && k.name) ? k.name : "";
}

exx_status exx_plan_set_profiling(exx_plan* p, int enable) {
    if (!p) return EXX_ERR_INVALID_ARG;
    EXX_ENTER(p);
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    p->events_used = 0;
    if (enable) {
        exx_status st = grow_event_pool(p);
        if (st != EXX_OK) return st;
    }
    p->profiling = enable ? 1 : 0;
    return EXX_OK;
}

exx_status exx_plan_get_profile(exx_plan* p, double pass_ms[4], long long pass_launches[4]) {
    if (!p || !pass_ms || !pass_launches) return EXX_ERR_INVALID_ARG;
    EXX_ENTER(p);
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    for (int k = 0; k < 4; ++k) { pass_ms[k] = 0.0; pass_launches[k] = 0; }
    for (size_t b = 0; b + 5 <= p->events_used; b += 5) {
        for (int k = 0; k < 4; ++k) {
            float ms = 0.f;
            EXX_CUDA(p, cudaEventElapsedTime(&ms, p->events[b + k], p->events[b + k + 1]));
            pass_ms[k] += ms;
            pass_launches[k] += 1;
        }
    }
    return EXX_OK;
}

exx_status exx_plan_set_batch(exx_plan* p, int max_transforms_per_batch) {
    if (!p) return EXX_ERR_INVALID_ARG;
    EXX_ENTER(p);
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    int b = max_transforms_per_batch > 0 ? max_transforms_per_batch : default_batch(p);
    if (b > 4096) b = 4096;
    return alloc_workspace(p, b);
}

exx_status exx_apply_async(exx_plan* p, int n_orb, const double* psi_dev, const double* occ_host, double* kpsi_dev, double* ex_dev) {
    exx_status st = check_apply_args(p, n_orb, psi_dev, occ_host, kpsi_dev, ex_dev);
    if (st != EXX_OK) return st;
    EXX_ENTER(p);
    if (!is_device_pointer(ex_dev)) return fail(p, EXX_ERR_BAD_POINTER, "psi_dev, kpsi_dev and ex_dev must be device pointers");
    st = square_device_apply(p, n_orb, psi_dev, occ_host, nullptr, kpsi_dev);
    if (st != EXX_OK) return st;
    EXX_CUDA(p, cudaMemcpyAsync(ex_dev, p->ex_dev, sizeof(double), cudaMemcpyDeviceToDevice, p->stream));
    return EXX_OK;
}

exx_status exx_apply(exx_plan* p, int n_orb, const double* psi_dev, const double* occ_host, double* kpsi_dev, double* ex_host) {
    exx_status st = check_apply_args(p, n_orb, psi_dev, occ_host, kpsi_dev, ex_host);
    if (st != EXX_OK) return st;
    EXX_ENTER(p);
    if (is_device_pointer(ex_host)) return fail(p, EXX_ERR_BAD_POINTER, "occ_host and ex_host must be host pointers");
    st = square_device_apply(p, n_orb, psi_dev, occ_host, nullptr, kpsi_dev);
    if (st != EXX_OK) return st;
    return finish_sync(p, ex_host);
}

exx_status exx_apply_pairs(exx_plan* p, int n_orb, const double* psi_dev, const double* occ_host, const unsigned char* pair_mask_host,
                           double* kpsi_dev, double* ex_host) {
    exx_status st = check_apply_args(p, n_orb, psi_dev, occ_host, kpsi_dev, ex_host);
    if (st != EXX_OK) return st;
    EXX_ENTER(p);
    if (!pair_mask_host) return fail(p, EXX_ERR_INVALID_ARG, "NULL pair mask");
    if (is_device_pointer(ex_host) || is_device_pointer(pair_mask_host))
        return fail(p, EXX_ERR_BAD_POINTER, "occ_host, pair_mask_host and ex_host must be host pointers");
    for (int a = 0; a < n_orb; ++a)
        for (int b = a + 1; b < n_orb; ++b)
            if ((pair_mask_host[static_cast<size_t>(a) * n_orb + b] != 0) != (pair_mask_host[static_cast<size_t>(b) * n_orb + a] != 0))
                return fail(p, EXX_ERR_INVALID_ARG, "the pair mask must be symmetric");
    st = square_device_apply(p, n_orb, psi_dev, occ_host, pair_mask_host, kpsi_dev);
    if (st != EXX_OK) return st;
    return finish_sync(p, ex_host);
}

static exx_status apply_to_impl(exx_plan* p, int n_occ, const double* psi_dev, const double* chi_dev, const double* occ_host, int n_tgt,
                                const double* phi_dev, double* kphi_dev, bool sync) {
    exx_status st = check_set(p, n_occ, psi_dev, nullptr, "exx_apply_to (occupied set)");
    if (st != EXX_OK) return st;
    if (chi_dev) {
        st = check_set(p, n_occ, chi_dev, nullptr, "exx_apply_to_cross (partner set)");
        if (st != EXX_OK) return st;
    }
    st = check_set(p, n_tgt, phi_dev, kphi_dev, "exx_apply_to (target set)");
    if (st != EXX_OK) return st;
    if (is_device_pointer(occ_host)) return fail(p, EXX_ERR_BAD_POINTER, "occ_host must be a host pointer");
    const size_t e_occ = static_cast<size_t>(n_occ) * p->M, e_tgt = static_cast<size_t>(n_tgt) * p->M;
    if (ranges_overlap(kphi_dev, e_tgt, psi_dev, e_occ) || ranges_overlap(kphi_dev, e_tgt, phi_dev, e_tgt) ||
        (chi_dev && ranges_overlap(kphi_dev, e_tgt, chi_dev, e_occ)))
        return fail(p, EXX_ERR_INVALID_ARG, "kphi must not overlap psi, chi or phi");
    Job job{};
    job.square = false;
    job.n_res = n_tgt; job.n_str = n_occ;
    job.psi_res = phi_dev; job.psi_str = psi_dev; job.psi_str_epi = chi_dev;
    job.kpsi_res = kphi_dev; job.kpsi_str = nullptr;
    job.occ_res = nullptr; job.occ_str = occ_host;
    job.zero_res = true;
    job.skip_empty_streamed = true;
    job.energy = false;
    st = run_job(p, job);
    if (st != EXX_OK) return st;
    if (sync) EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    return EXX_OK;
}

exx_status exx_apply_to(exx_plan* p, int n_occ, const double* psi_dev, const double* occ_host, int n_tgt, const double* phi_dev,
                        double* kphi_dev) {
    if (!p) return EXX_ERR_INVALID_ARG;
    if (!psi_dev || !occ_host || !phi_dev || !kphi_dev) return fail(p, EXX_ERR_INVALID_ARG, "NULL argument");
    EXX_ENTER(p);
    return apply_to_impl(p, n_occ, psi_dev, nullptr, occ_host, n_tgt, phi_dev, kphi_dev, true);
}

exx_status exx_apply_to_cross(exx_plan* p, int n_occ, const double* psi_dev, const double* chi_dev, const double* occ_host, int n_tgt,
                              const double* phi_dev, double* kphi_dev) {
    if (!p) return EXX_ERR_INVALID_ARG;
    if (!psi_dev || !chi_dev || !occ_host || !phi_dev || !kphi_dev) return fail(p, EXX_ERR_INVALID_ARG, "NULL argument");
    EXX_ENTER(p);
    return apply_to_impl(p, n_occ, psi_dev, chi_dev, occ_host, n_tgt, phi_dev, kphi_dev, true);
}

exx_status exx_apply_complex(exx_plan* p, int n_orb, const double* psi_dev, const double* occ_host, double* kpsi_dev, double* work_dev,
                             double* ex_host) {
    if (!p) return EXX_ERR_INVALID_ARG;
    if (!psi_dev || !occ_host || !kpsi_dev || !work_dev || !ex_host) return fail(p, EXX_ERR_INVALID_ARG, "NULL argument");
    if (n_orb < 1 || 2 * static_cast<long long>(n_orb) > p->max_orb)
        return fail(p, EXX_ERR_INVALID_ARG, "exx_apply_complex needs 2 * n_orb <= max_orbitals");
    EXX_ENTER(p);
    if (!is_device_pointer(work_dev) || !aligned16(work_dev)) return fail(p, EXX_ERR_BAD_POINTER, "work_dev must be 16-byte aligned device memory");
    if (is_device_pointer(occ_host) || is_device_pointer(ex_host)) return fail(p, EXX_ERR_BAD_POINTER, "occ_host and ex_host must be host pointers");
    const int n2 = 2 * n_orb;
    const size_t nm = static_cast<size_t>(n_orb) * p->M, set = 2 * nm;
    exx_status st = check_set(p, n2, psi_dev, kpsi_dev, "exx_apply_complex");
    if (st != EXX_OK) return st;
    if (ranges_overlap(work_dev, 3 * set, psi_dev, set) || ranges_overlap(work_dev, 3 * set, kpsi_dev, set) ||
        ranges_overlap(psi_dev, set, kpsi_dev, set))
        return fail(p, EXX_ERR_INVALID_ARG, "psi, kpsi and work must not overlap");
    double* jx = work_dev;                                 // partner set (-v, u)
    double* ka = work_dev + set;                           // A = K[X] X      (square apply of the 2N real orbitals)
    double* kb = work_dev + 2 * set;                       // B = T(X, JX) X  (cross term)
    // the 2N real orbitals carry the occupations (f, f); the pinned occupation staging doubles as the host copy
    try {
        p->occ2.assign(static_cast<size_t>(n2), 0.0);
    } catch (const std::bad_alloc&) {
        return fail(p, EXX_ERR_ALLOC, "out of host memory");
    }
    for (int k = 0; k < n_orb; ++k) p->occ2[k] = p->occ2[n_orb + k] = occ_host[k];
    cudaStream_t s = p->stream;
    complex_partner_kernel<<<2048, 256, 0, s>>>(psi_dev, jx, static_cast<long long>(nm));
    EXX_CUDA(p, cudaGetLastError());
    ++p->launches;
    st = square_device_apply(p, n2, psi_dev, p->occ2.data(), nullptr, ka);
    if (st != EXX_OK) return st;
    st = apply_to_impl(p, n2, psi_dev, jx, p->occ2.data(), n2, psi_dev, kb, false);
    if (st != EXX_OK) return st;
    // occupations of the orbitals on the device: run_job left (f, f) in occ_dev + max_orb (the streamed set's columns)
    const long long ep_cap = static_cast<long long>(p->max_batch) * p->info_c.tiles * 2;   // doubles in the partial-sum buffer
    const int nblk = static_cast<int>(ep_cap < 1024 ? (ep_cap < 1 ? 1 : ep_cap) : 1024);
    complex_combine_kernel<<<nblk, 256, 0, s>>>(psi_dev, ka, kb, p->occ_dev + p->max_orb, kpsi_dev, p->M, n_orb, p->epart);
    complex_energy_kernel<<<1, 256, 0, s>>>(p->epart, nblk, 0.5 * p->dV, p->ex_dev);
    EXX_CUDA(p, cudaGetLastError());
    p->launches += 2;
    p->last_rows = p->last_cols = 0;
    return finish_sync(p, ex_host);
}

exx_status exx_apply_block(exx_plan* p, int n_res, const double* psi_res_dev, const double* occ_res_host, double* kpsi_res_dev, int n_str,
                           const double* psi_str_dev, const double* occ_str_host, double* kpsi_str_dev, int flags, double* ex_host) {
    if (!p) return EXX_ERR_INVALID_ARG;
    if (!psi_res_dev || !occ_res_host || !kpsi_res_dev || !psi_str_dev || !occ_str_host || !kpsi_str_dev || !ex_host)
        return fail(p, EXX_ERR_INVALID_ARG, "NULL argument");
    if (flags & ~(EXX_BLOCK_ACCUMULATE_RESIDENT | EXX_BLOCK_ACCUMULATE_STREAMED)) return fail(p, EXX_ERR_INVALID_ARG, "unknown flag");
    EXX_ENTER(p);
    exx_status st = check_set(p, n_res, psi_res_dev, kpsi_res_dev, "exx_apply_block (resident set)");
    if (st != EXX_OK) return st;
    st = check_set(p, n_str, psi_str_dev, kpsi_str_dev, "exx_apply_block (streamed set)");
    if (st != EXX_OK) return st;
    if (is_device_pointer(occ_res_host) || is_device_pointer(occ_str_host) || is_device_pointer(ex_host))
        return fail(p, EXX_ERR_BAD_POINTER, "occupations and ex_host must be host pointers");
    const size_t e_res = static_cast<size_t>(n_res) * p->M, e_str = static_cast<size_t>(n_str) * p->M;
    if (ranges_overlap(psi_res_dev, e_res, psi_str_dev, e_str))
        return fail(p, EXX_ERR_INVALID_ARG, "the two orbital sets must be disjoint (use exx_apply for a set with itself)");
    if (ranges_overlap(kpsi_res_dev, e_res, kpsi_str_dev, e_str) || ranges_overlap(kpsi_res_dev, e_res, psi_res_dev, e_res) ||
        ranges_overlap(kpsi_res_dev, e_res, psi_str_dev, e_str) || ranges_overlap(kpsi_str_dev, e_str, psi_res_dev, e_res) ||
        ranges_overlap(kpsi_str_dev, e_str, psi_str_dev, e_str))
        return fail(p, EXX_ERR_INVALID_ARG, "outputs must not overlap each other or the inputs");
    Job job{};
    job.square = false;
    job.n_res = n_res; job.n_str = n_str;
    job.psi_res = psi_res_dev; job.psi_str = psi_str_dev;
    job.kpsi_res = kpsi_res_dev; job.kpsi_str = kpsi_str_dev;
    job.occ_res = occ_res_host; job.occ_str = occ_str_host;
    job.zero_res = !(flags & EXX_BLOCK_ACCUMULATE_RESIDENT);
    job.zero_str = !(flags & EXX_BLOCK_ACCUMULATE_STREAMED);
    job.energy = true;
    st = run_job(p, job);
    if (st != EXX_OK) return st;
    return finish_sync(p, ex_host);
}

exx_status exx_apply_host(exx_plan* p, int n_orb, const double* psi_host, const double* occ_host, double* kpsi_host, double* ex_host) {
    exx_status st = check_apply_args(p, n_orb, psi_host, occ_host, kpsi_host, ex_host);
    if (st != EXX_OK) return st;
    EXX_ENTER(p);
    if (is_device_pointer(psi_host) || is_device_pointer(kpsi_host) || is_device_pointer(occ_host) || is_device_pointer(ex_host))
        return fail(p, EXX_ERR_BAD_POINTER, "exx_apply_host takes host pointers");
    const size_t elems = static_cast<size_t>(n_orb) * p->M;
    if (ranges_overlap(psi_host, elems, kpsi_host, elems)) return fail(p, EXX_ERR_INVALID_ARG, "kpsi must not overlap psi");
    if (elems > p->stage_elems) {
        // grow the staging pair; the old pair is released first (psi + K psi of C5 are 2 x 58 GB: no room for two pairs)
        EXX_CUDA(p, cudaStreamSynchronize(p->stream));
        if (p->psi_stage) cudaFree(p->psi_stage);
        if (p->kpsi_stage) cudaFree(p->kpsi_stage);
        p->psi_stage = p->kpsi_stage = nullptr;
        p->stage_elems = 0;
        if (cudaMalloc(&p->psi_stage, elems * sizeof(double)) != cudaSuccess || cudaMalloc(&p->kpsi_stage, elems * sizeof(double)) != cudaSuccess) {
            cudaGetLastError();
            if (p->psi_stage) cudaFree(p->psi_stage);
            p->psi_stage = p->kpsi_stage = nullptr;
            return fail(p, EXX_ERR_ALLOC, "cudaMalloc(device staging for exx_apply_host) failed");
        }
        p->stage_elems = elems;
    }
    EXX_CUDA(p, cudaMemcpyAsync(p->psi_stage, psi_host, elems * sizeof(double), cudaMemcpyHostToDevice, p->stream));
    Job job{};
    job.square = true;
    job.n_res = job.n_str = n_orb;
    job.psi_res = job.psi_str = p->psi_stage;
    job.kpsi_res = job.kpsi_str = p->kpsi_stage;
    job.occ_res = job.occ_str = occ_host;
    job.zero_res = job.zero_str = true;
    job.energy = true;
    job.kpsi_host = kpsi_host;
    st = run_job(p, job);
    if (st != EXX_OK) return st;
    return finish_sync(p, ex_host);
}

exx_status exx_plan_release_staging(exx_plan* p) {
    if (!p) return EXX_ERR_INVALID_ARG;
    EXX_ENTER(p);
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    if (p->psi_stage) cudaFree(p->psi_stage);
    if (p->kpsi_stage) cudaFree(p->kpsi_stage);
    p->psi_stage = p->kpsi_stage = nullptr;
    p->stage_elems = 0;
    return EXX_OK;
}

exx_status exx_get_pair_energies(exx_plan* p, int n_orb, double* e_host) {
    if (!p || !e_host) return EXX_ERR_INVALID_ARG;
    EXX_ENTER(p);
    if (p->last_rows < 1 || p->last_rect) return fail(p, EXX_ERR_INVALID_ARG, "the most recent apply left no symmetric pair-energy matrix");
    if (n_orb != p->last_rows) return fail(p, EXX_ERR_INVALID_ARG, "n_orb differs from the orbital count of the most recent apply");
    const size_t n = static_cast<size_t>(n_orb);
    EXX_CUDA(p, cudaMemcpyAsync(e_host, p->e_mat, n * n * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    return EXX_OK;
}

exx_status exx_get_block_energies(exx_plan* p, int n_res, int n_str, double* e_host) {
    if (!p || !e_host) return EXX_ERR_INVALID_ARG;
    EXX_ENTER(p);
    if (p->last_rows < 1 || !p->last_rect) return fail(p, EXX_ERR_INVALID_ARG, "the most recent apply was not exx_apply_block");
    if (n_res != p->last_rows || n_str != p->last_cols) return fail(p, EXX_ERR_INVALID_ARG, "block shape differs from the most recent exx_apply_block");
    EXX_CUDA(p, cudaMemcpyAsync(e_host, p->e_mat, static_cast<size_t>(n_res) * n_str * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
    EXX_CUDA(p, cudaStreamSynchronize(p->stream));
    return EXX_OK;
}

}  // extern "C"
