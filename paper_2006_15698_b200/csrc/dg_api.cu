// dg_api.cu -- the C-ABI boundary (include/dg_b200.h): argument checking, workspace carving, operator
// tables and kernel launches.  No arithmetic of the method runs here; it all runs in dg_kernels.cu.
// Shares nothing with oracle/ (the operator construction below is written independently).
#include "../../include/dg_b200.h"
#include "../../include/dg_b200_test.h"
#include "dg_internal.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

namespace {

// ------------------------------------------------------------------------------------------------
// 1-D operators of the N-point Gauss-Legendre collocation basis, long double.
// ------------------------------------------------------------------------------------------------
struct HostOps {
    long double xi[DG_NMAX], w[DG_NMAX];
    long double D[DG_NMAX][DG_NMAX];   // D[q][i] = l_i'(xi_q)
    long double lp[DG_NMAX], lm[DG_NMAX];
};

// Legendre polynomial by Bonnet's recurrence; derivative from P_N' = N (P_{N-1} - x P_N) / (1 - x^2).
void legendre_pair(int N, long double x, long double &PN, long double &dPN) {
    long double Pm = 1.0L, P = x;
    if (N == 0) { PN = 1.0L; dPN = 0.0L; return; }
    for (int k = 2; k <= N; ++k) {
        const long double Pk = ((2 * k - 1) * x * P - (k - 1) * Pm) / k;
        Pm = P;
        P = Pk;
    }
    PN = P;
    dPN = N * (Pm - x * P) / (1.0L - x * x);
}

void build_host_ops(int N, HostOps &o) {
    const long double pi = acosl(-1.0L);
    // nodes: Newton from the Chebyshev-like guess, left half then mirrored (ascending order)
    for (int i = 0; i < (N + 1) / 2; ++i) {
        long double x = -cosl(pi * (4 * i + 3) / (4 * N + 2));
        for (int it = 0; it < 60; ++it) {
            long double P, dP;
            legendre_pair(N, x, P, dP);
            const long double step = P / dP;
            x -= step;
            if (fabsl(step) <= 4e-20L) break;
        }
        if (2 * i + 1 == N) x = 0.0L;
        long double P, dP;
        legendre_pair(N, x, P, dP);
        const long double wi = 2.0L / ((1.0L - x * x) * dP * dP);
        o.xi[i] = x;          o.w[i] = wi;
        o.xi[N - 1 - i] = -x; o.w[N - 1 - i] = wi;
    }
    // l_i'(xi_q) by the product formula: q != i: prod_{m != i,q} (xi_q - xi_m) / prod_{m != i} (xi_i - xi_m);
    // q == i: sum_{m != i} 1 / (xi_i - xi_m).  l_i(+-1) = prod_{m != i} (+-1 - xi_m) / (xi_i - xi_m).
    for (int i = 0; i < N; ++i) {
        long double den = 1.0L, ep = 1.0L, em = 1.0L;
        for (int m = 0; m < N; ++m) {
            if (m == i) continue;
            den *= (o.xi[i] - o.xi[m]);
            ep *= (1.0L - o.xi[m]);
            em *= (-1.0L - o.xi[m]);
        }
        o.lp[i] = ep / den;
        o.lm[i] = em / den;
        for (int q = 0; q < N; ++q) {
            if (q == i) {
                long double s = 0.0L;
                for (int m = 0; m < N; ++m)
                    if (m != i) s += 1.0L / (o.xi[i] - o.xi[m]);
                o.D[q][i] = s;
            } else {
                long double num = 1.0L;
                for (int m = 0; m < N; ++m)
                    if (m != i && m != q) num *= (o.xi[q] - o.xi[m]);
                o.D[q][i] = num / den;
            }
        }
    }
}

// Device tables on the reference element: the weak-form volume operator and the lift weights with the
// inverse (diagonal) mass folded in; the constant geometric factor 2/h_a of each axis
// travels separately (DgStageArgs::scale).
void build_ref_ops(int N, DgRefOps &d) {
    HostOps o;
    build_host_ops(N, o);
    std::memset(&d, 0, sizeof(d));
    for (int i = 0; i < N; ++i) {
        d.lp[i] = (double)o.lp[i];
        d.lq[i] = (double)(0.5L * o.lp[i] / o.w[i]);   // 1/2: the kernel's interface flux is 2 F*
        for (int q = 0; q < N; ++q) d.D[q][i] = (double)(o.w[q] * o.D[q][i] / o.w[i]);
    }
    // even-odd form (see DgRefOps): Dhat[i][q] = w_q D[q][i] / w_i in long double, then the half sums / differences
    const int H = N / 2, mid = N / 2;
    auto Dhat = [&](int i, int q) { return o.w[q] * o.D[q][i] / o.w[i]; };
    auto lq = [&](int i) { return 0.5L * o.lp[i] / o.w[i]; };
    for (int q = 0; q < H; ++q) {
        for (int i = 0; i < H; ++i) d.Pe[q][i] = (double)(0.5L * (Dhat(i, q) + Dhat(i, N - 1 - q)));
        for (int i = 0; i < H + (N & 1); ++i) d.Po[q][i] = (double)(0.5L * (Dhat(i, q) - Dhat(i, N - 1 - q)));
    }
    for (int i = 0; i < H; ++i) {
        d.Dm[i] = (N & 1) ? (double)Dhat(i, mid) : 0.0;
        d.ls[i] = (double)(0.5L * (lq(i) + lq(N - 1 - i)));
        d.la[i] = (double)(0.5L * (lq(N - 1 - i) - lq(i)));
    }
    if (N & 1) d.ls[mid] = (double)lq(mid);
}

// Carpenter-Kennedy (5,4) 2N-storage Runge-Kutta, "LSERK45" (reading R9).
const long double kRkA[5] = {0.0L, -567301805773.0L / 1357537059087.0L, -2404267990393.0L / 2016746695238.0L,
                             -3550918686646.0L / 2091501179385.0L, -1275806237668.0L / 842570457699.0L};
const long double kRkB[5] = {1432997174477.0L / 9575080441755.0L, 5161836677717.0L / 13612068292357.0L,
                             1720146321549.0L / 2090206949498.0L, 3134564353537.0L / 4481467310338.0L,
                             2277821191437.0L / 14882151754819.0L};

const DgKernelTable *variants_for(int N, int *count) {
    switch (N) {
        case 2: return dg_variants_N2(count);
        case 3: return dg_variants_N3(count);
        case 4: return dg_variants_N4(count);
        case 5: return dg_variants_N5(count);
        case 6: return dg_variants_N6(count);
        case 7: return dg_variants_N7(count);
        case 8: return dg_variants_N8(count);
    }
    *count = 0;
    return nullptr;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

}  // namespace

// FP64 peak microbenchmark (test/bench entry dg_fp64_peak): 8 independent DFMA chains per thread, 4096 deep.
__global__ void __launch_bounds__(256) dg_fp64_peak_kernel(double *out, int iters, double a, double b) {
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 16; ++j) {
            x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
            x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
        }
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// "Update" half of the paper's update-project kernel: K = A K + dt R, Q = Q + B K over the internal
// vectors (padding included: it stays zero); the "project" half is the face-trace kernel launched right after.
__global__ void __launch_bounds__(256) dg_split_update_kernel(double *Q, double *K, const double *R, size_t n, double rkA,
                                                              double rkB, double dt) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double k = (rkA == 0.0) ? dt * R[i] : fma(rkA, K[i], dt * R[i]);
        K[i] = k;
        Q[i] = fma(rkB, k, Q[i]);
    }
}

// Gathers the runs src[o * outer_stride + i * inner_stride + 0 .. run) into a dense buffer (dg_halo_export).
__global__ void __launch_bounds__(256) dg_pack_kernel(double *dst, const double *src, long long n_outer, long long outer_stride,
                                                      long long n_inner, long long inner_stride, int run) {
    const long long total = n_outer * n_inner * run;
    for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (long long)gridDim.x * blockDim.x) {
        const long long blk = idx / run, r = idx - blk * run;
        const long long o = blk / n_inner, i = blk - o * n_inner;
        dst[idx] = src[o * outer_stride + i * inner_stride + r];
    }
}

__global__ void dg_fastmath_kernel(const double *x, double *r, double *q, size_t n) {
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        r[i] = rcp_pos(x[i]);
        q[i] = sqrt_pos(x[i]);
    }
}

struct dg_ctx {
    int nx, ny, nz, p, N;
    double gamma;
    double extent[3];
    double h[3];        // element size per axis (extent / n unless dg_set_spacing gave it)
    const DgKernelTable *kt;
    int variant;
    int nbx, nby;       // columns of bx x by elements
    int lz, nchunks;    // layers per chunk (one thread block marches through one chunk of one column)
    int lz_user;        // 0 = heuristic
    size_t nslots;      // layer slots = nbx * nby * nz
    size_t state_len;   // canonical doubles
    size_t int_len;     // internal (column-padded) doubles
    size_t txy_len;     // doubles per x/y trace buffer
    size_t tz_len;      // doubles per z trace buffer
    // borrowed workspace
    double *Q, *K, *S, *Txy[2], *Tz[2];
    double *V[3];       // viscous terms enabled (dg_set_viscosity): gradient / viscous-flux vectors, internal layout
    double mu, prandtl; // dynamic viscosity (0 = inviscid, no V vectors) and Prandtl number (reading R20)
    unsigned long long *scal;
    int tcur;           // Txy[tcur], Tz[tcur] hold the traces of the current Q
    bool lam_valid;     // scal[lcur] holds the max wavespeed of the current Q (reduced by the last stage)
    int lcur;           // scal[0..1]: two wavespeed slots (one read, one written by a CFL step); scal[2..3]: time advanced, last dt
    int sms, blocks_per_sm;
    double g[3];        // 2/h_a per axis
    int bc[6];          // boundary condition per domain face (dg_set_boundary), 0 = periodic
    const double *halo[6];   // DG_BC_HALO faces: the caller's device buffer with the neighbour context's traces
    const double *halo2[6][2];   // ... or a PAIR of buffers read alternately (dg_set_halo_pair; parity = tcur)
    double *push[6][2];      // push mode: the neighbour context's pair for its opposite face (dg_set_halo_push)
    double qinf[DG_NV];
    bool bound, has_state;
    cudaStream_t stream;
    unsigned long long launches;
    char err[256];
};

namespace {

int fail(dg_ctx *c, int code, const char *fmt, ...) {
    if (c) {
        va_list ap;
        va_start(ap, fmt);
        vsnprintf(c->err, sizeof(c->err), fmt, ap);
        va_end(ap);
    }
    return code;
}

int cuda_fail(dg_ctx *c, cudaError_t e, const char *what) {
    return fail(c, DG_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

// Layers per chunk: enough blocks to fill the GPU several times over with a small tail, chunks long enough
// that the extra work at their two ends (pipeline fill, one more interface flux, z traces through HBM)
// stays small.  `resident` = thread blocks the whole GPU holds at once.
int pick_lz(int columns, int nz, long long resident) {
    int best = 1;
    double best_score = -1.0;
    for (int lz = 1; lz <= nz && lz <= 64; ++lz) {
        const long long blocks = (long long)columns * ((nz + lz - 1) / lz);
        const double waves = (double)blocks / (double)resident;
        const double fill = waves / std::ceil(waves);
        const double score = fill * (double)lz / ((double)lz + 0.6);
        if (score > best_score + 1e-12) {
            best_score = score;
            best = lz;
        }
    }
    return best;
}

void set_layout(dg_ctx *c, int variant, const DgKernelTable *kt) {
    c->kt = kt;
    c->variant = variant;
    c->nbx = (c->nx + kt->bx - 1) / kt->bx;
    c->nby = (c->ny + kt->by - 1) / kt->by;
    const int sms = c->sms > 0 ? c->sms : 148;
    c->lz = c->lz_user > 0 ? (c->lz_user < c->nz ? c->lz_user : c->nz)
                           : pick_lz(c->nbx * c->nby, c->nz, (long long)sms * (kt->minb > 0 ? kt->minb : 1));
    c->nchunks = (c->nz + c->lz - 1) / c->lz;
    c->nslots = (size_t)c->nbx * c->nby * c->nz;
    c->int_len = c->nslots * (size_t)kt->slot;
    c->txy_len = c->nslots * (size_t)kt->txy;
    c->tz_len = (size_t)c->nbx * c->nby * c->nchunks * (size_t)kt->tz;
}

struct Carve {
    size_t q, k, s, txy0, txy1, tz0, tz1, scal, v[3], total;
};
Carve carve(const dg_ctx *c) {
    Carve v;
    size_t off = 0;
    v.q = off;    off += align_up(c->int_len * 8 + 16, 256);   // +16: the L2 prefetch rounds out to 16-byte granules
    v.k = off;    off += align_up(c->int_len * 8 + 16, 256);
    v.s = off;    off += align_up((c->int_len > c->state_len ? c->int_len : c->state_len) * 8, 256);   // staging / split-mode R
    v.txy0 = off; off += align_up(c->txy_len * 8 + 16, 256);
    v.txy1 = off; off += align_up(c->txy_len * 8 + 16, 256);
    v.tz0 = off;  off += align_up(c->tz_len * 8, 256);
    v.tz1 = off;  off += align_up(c->tz_len * 8, 256);
    v.scal = off; off += 256;
    for (int a = 0; a < 3; ++a) {
        v.v[a] = off;
        if (c->mu > 0.0) off += align_up(c->int_len * 8, 256);
    }
    v.total = off;
    return v;
}

DgStageArgs stage_args(const dg_ctx *c, int mode) {
    DgStageArgs a;
    std::memset(&a, 0, sizeof(a));
    a.Q = c->Q;
    a.K = c->K;   // residual mode: the Runge-Kutta register is dead between steps, the residual lands there
    a.Txy_old = c->Txy[c->tcur];
    a.Txy_new = c->Txy[1 - c->tcur];
    a.Tz_old = c->Tz[c->tcur];
    a.Tz_new = c->Tz[1 - c->tcur];
    a.lam_bits = c->scal;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nbx = c->nbx; a.nby = c->nby;
    a.lz = c->lz; a.nchunks = c->nchunks;
    a.gamma = c->gamma;
    a.gm1 = c->gamma - 1.0;
    a.mode = mode;
    for (int i = 0; i < 3; ++i) a.scale[i] = c->g[i];
    for (int i = 0; i < 6; ++i) {
        a.bc[i] = (c->bc[i] == DG_BC_HALO) ? 0 : c->bc[i];
        a.halo_ext[i] = (c->bc[i] == DG_BC_HALO) ? (c->halo2[i][0] ? c->halo2[i][c->tcur] : c->halo[i]) : nullptr;
        // the updated state's traces go where the neighbour reads in the NEXT stage (its parity will be 1 - tcur)
        a.halo_push[i] = (mode == DG_MODE_STAGE && c->bc[i] == DG_BC_HALO) ? c->push[i][1 - c->tcur] : nullptr;
    }
    for (int i = 0; i < DG_NV; ++i) a.qinf[i] = c->qinf[i];
    return a;
}

int launch_layout(dg_ctx *c, double *internal, double *canonical, int to_internal) {
    DgLayoutArgs a;
    a.internal = internal;
    a.canonical = canonical;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nbx = c->nbx; a.nby = c->nby;
    a.to_internal = to_internal;
    cudaError_t e = c->kt->launch_layout(a, c->sms, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "layout kernel");
    c->launches++;
    return DG_OK;
}

// internal vector -> caller's canonical array (device: directly; host: through the staging vector)
int export_vector(dg_ctx *c, double *internal, double *out, int on_device, const char *what) {
    if (on_device) return launch_layout(c, internal, out, 0);
    int rc = launch_layout(c, internal, c->S, 0);
    if (rc != DG_OK) return rc;
    cudaError_t e = cudaMemcpyAsync(out, c->S, c->state_len * 8, cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, what);
    e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, what);
    return DG_OK;
}

// One LSERK45 step = 5 launches of the fused stage kernel.  cfl_factor > 0: the time step is formed on the device from
// the wavespeed in scal[lcur] and the last stage reduces the wavespeed of the state it produces into the other slot
// (a9 fused: no extra sweep over the state, no host round trip).
int check_halos(dg_ctx *c) {
    for (int f = 0; f < 6; ++f)
        if (c->bc[f] == DG_BC_HALO && !c->halo[f] && !c->halo2[f][0]) return fail(c, DG_ESTATE, "face %d is a halo face but dg_set_halo was not called", f);
    return DG_OK;
}

int enqueue_stage(dg_ctx *c, int s, double dt, double cfl_factor) {
    const bool cfl = cfl_factor > 0.0;
    DgStageArgs a = stage_args(c, DG_MODE_STAGE);
    for (int i = 0; i < 3; ++i) a.scale[i] = cfl ? c->g[i] : dt * c->g[i];
    a.rkA = (double)kRkA[s];
    a.rkB = (double)kRkB[s];
    a.want_lam = (cfl && s == 4) ? 1 : 0;
    a.store_k = (s == 4) ? 0 : 1;
    a.lam_in = cfl ? c->scal + c->lcur : nullptr;
    a.cfl_factor = cfl_factor;
    a.t_acc = (cfl && s == 0) ? reinterpret_cast<double *>(c->scal + 2) : nullptr;
    a.lam_bits = c->scal + (1 - c->lcur);
    cudaError_t e = c->kt->launch_stage(a, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "stage kernel");
    c->launches++;
    c->tcur = 1 - c->tcur;
    return DG_OK;
}

int enqueue_step(dg_ctx *c, double dt, double cfl_factor) {
    const bool cfl = cfl_factor > 0.0;
    int rc = check_halos(c);
    if (rc != DG_OK) return rc;
    if (cfl) {
        cudaError_t e = cudaMemsetAsync(c->scal + (1 - c->lcur), 0, 8, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "memset");
    }
    for (int s = 0; s < 5; ++s) {
        rc = enqueue_stage(c, s, dt, cfl_factor);
        if (rc != DG_OK) return rc;
    }
    if (cfl) c->lcur = 1 - c->lcur;
    c->lam_valid = cfl;
    return DG_OK;
}

// face traces of the current Q into buffer 0 (after dg_set_state and after a split-mode update)
int refresh_traces(dg_ctx *c) {
    c->tcur = 0;
    DgTraceArgs a;
    std::memset(&a, 0, sizeof(a));
    a.Q = c->Q;
    a.Txy = c->Txy[0];
    a.Tz = c->Tz[0];
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nbx = c->nbx; a.nby = c->nby;
    a.lz = c->lz; a.nchunks = c->nchunks;
    cudaError_t e = c->kt->launch_traces(a, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "trace kernel");
    c->launches++;
    return DG_OK;
}

DgSplitArgs split_args(const dg_ctx *c) {
    DgSplitArgs a;
    std::memset(&a, 0, sizeof(a));
    a.Q = c->Q;
    a.R = c->S;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nbx = c->nbx; a.nby = c->nby;
    a.gamma = c->gamma;
    a.gm1 = c->gamma - 1.0;
    for (int i = 0; i < 3; ++i) a.scale[i] = c->g[i];
    return a;
}

// Push mode: make sure kernels of the current device can store to `ptr`.  Memory of the current device, host-registered
// memory and pointers the runtime does not know (no GPU in this process: the CPU-side tests) pass unchanged.
int enable_peer_access_to(dg_ctx *c, const void *ptr) {
    cudaPointerAttributes attr;
    int cur = -1;
    if (cudaPointerGetAttributes(&attr, ptr) != cudaSuccess || cudaGetDevice(&cur) != cudaSuccess) {
        (void)cudaGetLastError();   // not fatal: nothing known about the pointer
        return DG_OK;
    }
    if (attr.type != cudaMemoryTypeDevice || attr.device == cur) return DG_OK;
    int can = 0;
    cudaError_t e = cudaDeviceCanAccessPeer(&can, cur, attr.device);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaDeviceCanAccessPeer");
    if (!can) return fail(c, DG_EUNSUPPORTED, "device %d cannot access the memory of device %d: push mode needs peer access, use dg_halo_export + a copy", cur, attr.device);
    e = cudaDeviceEnablePeerAccess(attr.device, 0);
    if (e == cudaErrorPeerAccessAlreadyEnabled) {
        (void)cudaGetLastError();
        e = cudaSuccess;
    }
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaDeviceEnablePeerAccess");
    return DG_OK;
}

// the max wavespeed of the current state is in scal[lcur] (enqueued; reduction kernel only if no stage left it there)
int ensure_lam(dg_ctx *c) {
    if (c->lam_valid) return DG_OK;
    cudaError_t e = cudaMemsetAsync(c->scal + c->lcur, 0, 8, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "memset");
    DgWaveArgs a;
    a.Q = c->Q;
    a.lam_bits = c->scal + c->lcur;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nbx = c->nbx; a.nby = c->nby;
    a.gamma = c->gamma;
    a.gm1 = c->gamma - 1.0;
    e = c->kt->launch_wavespeed(a, c->sms, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "wavespeed kernel");
    c->launches++;
    c->lam_valid = true;
    return DG_OK;
}

int read_lam(dg_ctx *c, double *lam_host) {
    const int rc = ensure_lam(c);
    if (rc != DG_OK) return rc;
    cudaError_t e = cudaMemcpyAsync(lam_host, c->scal + c->lcur, 8, cudaMemcpyDeviceToHost, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "device->host copy");
    e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "synchronise");
    return DG_OK;
}

}  // namespace

extern "C" {

int dg_create(dg_ctx **out, int nx, int ny, int nz, int p, double gamma, const double extent[3]) {
    if (!out || !extent) return DG_EINVAL;
    if (nx < 1 || ny < 1 || nz < 1) return DG_EINVAL;
    if (!(gamma > 1.0) || !std::isfinite(gamma)) return DG_EINVAL;
    for (int a = 0; a < 3; ++a)
        if (!(extent[a] > 0.0) || !std::isfinite(extent[a])) return DG_EINVAL;
    if (p < 1 || p > 7) return DG_EUNSUPPORTED;
    int count = 0;
    const DgKernelTable *kt = variants_for(p + 1, &count);
    if (!kt || count < 1) return DG_EUNSUPPORTED;
    dg_ctx *c = new (std::nothrow) dg_ctx;
    if (!c) return DG_ENOMEM;
    std::memset(c, 0, sizeof(*c));
    c->nx = nx; c->ny = ny; c->nz = nz; c->p = p; c->N = p + 1;
    c->gamma = gamma;
    for (int a = 0; a < 3; ++a) c->extent[a] = extent[a];
    c->h[0] = extent[0] / nx;
    c->h[1] = extent[1] / ny;
    c->h[2] = extent[2] / nz;
    c->state_len = (size_t)nx * ny * nz * (size_t)(c->N * c->N * c->N) * DG_NV;
    // default variant: the first compiled column shape that wastes < 4 % of its nodes on padding of ragged
    // columns (they are listed fastest first), else the one that wastes least
    int pick = 0;
    double best_waste = 1e30;
    for (int v = 0; v < count; ++v) {
        const double padded = (double)((nx + kt[v].bx - 1) / kt[v].bx * kt[v].bx) * ((ny + kt[v].by - 1) / kt[v].by * kt[v].by);
        const double waste = padded / ((double)nx * ny) - 1.0;
        if (waste < 0.04) {
            pick = v;
            break;
        }
        if (waste < best_waste) {
            best_waste = waste;
            pick = v;
        }
    }
    set_layout(c, pick, &kt[pick]);
    *out = c;
    return DG_OK;
}

int dg_set_brick(dg_ctx *c, int bx, int by, int lz) {
    if (!c) return DG_EINVAL;
    if (c->bound) return fail(c, DG_ESTATE, "dg_set_brick after dg_bind");
    if (bx < 0 || by < 0 || lz < 0) return fail(c, DG_EINVAL, "negative brick size");
    int count = 0;
    const DgKernelTable *kt = variants_for(c->N, &count);
    if (bx == 0 && by == 0) {
        c->lz_user = lz;
        set_layout(c, c->variant, c->kt);
        return DG_OK;
    }
    for (int v = 0; v < count; ++v)
        if (kt[v].bx == bx && kt[v].by == by) {
            c->lz_user = lz;
            set_layout(c, v, &kt[v]);
            return DG_OK;
        }
    return fail(c, DG_EUNSUPPORTED, "column %dx%d is not compiled for p=%d", bx, by, c->p);
}

int dg_set_boundary(dg_ctx *c, const int bc[6], const double q_inf[5]) {
    if (!c || !bc) return c ? fail(c, DG_EINVAL, "null boundary array") : DG_EINVAL;
    bool far = false;
    for (int a = 0; a < 3; ++a) {
        const int lo = bc[2 * a], hi = bc[2 * a + 1];
        if (lo < 0 || lo > 3 || hi < 0 || hi > 3) return fail(c, DG_EINVAL, "boundary condition outside 0..3");
        if ((lo == DG_BC_PERIODIC) != (hi == DG_BC_PERIODIC))
            return fail(c, DG_EINVAL, "an axis is periodic on both of its faces or on neither");
        far = far || lo == DG_BC_FARFIELD || hi == DG_BC_FARFIELD;
    }
    if (far) {
        if (!q_inf) return fail(c, DG_EINVAL, "a far-field face needs the far-field state");
        for (int n = 0; n < DG_NV; ++n)
            if (!std::isfinite(q_inf[n])) return fail(c, DG_EINVAL, "far-field state is not finite");
    }
    for (int f = 0; f < 6; ++f) c->bc[f] = bc[f];
    for (int n = 0; n < DG_NV; ++n) c->qinf[n] = q_inf ? q_inf[n] : 0.0;
    return DG_OK;
}

int dg_variant_count(int p) {
    int count = 0;
    if (p < 1 || p > 7) return 0;
    variants_for(p + 1, &count);
    return count;
}

int dg_set_variant(dg_ctx *c, int index) {
    if (!c) return DG_EINVAL;
    if (c->bound) return fail(c, DG_ESTATE, "dg_set_variant after dg_bind");
    int count = 0;
    const DgKernelTable *kt = variants_for(c->N, &count);
    if (index < 0 || index >= count) return fail(c, DG_EINVAL, "variant %d outside 0..%d", index, count - 1);
    set_layout(c, index, &kt[index]);
    return DG_OK;
}

size_t dg_state_len(const dg_ctx *c) { return c ? c->state_len : 0; }

size_t dg_workspace_bytes(const dg_ctx *c) { return c ? carve(c).total : 0; }

int dg_bind(dg_ctx *c, void *ws, size_t bytes, void *stream) {
    if (!c) return DG_EINVAL;
    if (!ws || ((size_t)ws & 255u)) return fail(c, DG_EINVAL, "workspace must be a 256-byte aligned device pointer");
    const Carve v = carve(c);
    if (bytes < v.total) return fail(c, DG_ENOMEM, "workspace %zu bytes < required %zu", bytes, v.total);
    if (c->nby > 65535 || c->nchunks > 65535) return fail(c, DG_EUNSUPPORTED, "more than 65535 columns along y or chunks");
    char *base = (char *)ws;
    c->Q = (double *)(base + v.q);
    c->K = (double *)(base + v.k);
    c->S = (double *)(base + v.s);
    c->Txy[0] = (double *)(base + v.txy0);
    c->Txy[1] = (double *)(base + v.txy1);
    c->Tz[0] = (double *)(base + v.tz0);
    c->Tz[1] = (double *)(base + v.tz1);
    c->scal = (unsigned long long *)(base + v.scal);
    for (int a = 0; a < 3; ++a) c->V[a] = (c->mu > 0.0) ? (double *)(base + v.v[a]) : nullptr;
    c->stream = (cudaStream_t)stream;
    c->tcur = 0;
    c->has_state = false;
    c->lam_valid = false;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return cuda_fail(c, e, "device query");
    // The nodes that pad ragged columns (and the even-pitch pad of every plane) travel with the bulk copies but are
    // never used: give them a defined value.  Only Q and K have such nodes; a mesh the columns tile exactly
    // with even planes has none.
    const bool padded = (c->nx % c->kt->bx) || (c->ny % c->kt->by) ||
                        ((size_t)c->kt->slot != (size_t)DG_NV * c->N * c->N * c->N * c->kt->bx * c->kt->by);
    if (padded) {
        e = cudaMemsetAsync(c->Q, 0, c->int_len * 8, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->K, 0, c->int_len * 8, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "workspace memset");
    }
    e = cudaMemsetAsync(c->scal, 0, 256, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "workspace memset");
    for (int a = 0; a < 3; ++a) c->g[a] = 2.0 / c->h[a];
    DgRefOps ref;
    build_ref_ops(c->N, ref);
    e = c->kt->prepare(ref, &c->blocks_per_sm);
    if (e != cudaSuccess) return cuda_fail(c, e, "stage kernel setup");
    if (c->blocks_per_sm < 1) return fail(c, DG_ECUDA, "stage kernel does not fit on the GPU");
    c->bound = true;
    c->err[0] = 0;
    return DG_OK;
}

int dg_set_state(dg_ctx *c, const double *q, int on_device) {
    if (!c || !q) return c ? fail(c, DG_EINVAL, "null state pointer") : DG_EINVAL;
    if (!c->bound) return fail(c, DG_ESTATE, "dg_set_state before dg_bind");
    const double *src = q;
    if (!on_device) {
        cudaError_t e = cudaMemcpyAsync(c->S, q, c->state_len * 8, cudaMemcpyHostToDevice, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "host->device copy of the state");
        src = c->S;
    }
    int rc = launch_layout(c, c->Q, const_cast<double *>(src), 1);
    if (rc != DG_OK) return rc;
    rc = refresh_traces(c);
    if (rc != DG_OK) return rc;
    c->has_state = true;
    c->lam_valid = false;
    return DG_OK;
}

int dg_residual(dg_ctx *c, double *r_out, int on_device) {
    if (!c || !r_out) return c ? fail(c, DG_EINVAL, "null residual pointer") : DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_residual needs dg_bind and dg_set_state first");
    const int hrc = check_halos(c);
    if (hrc != DG_OK) return hrc;
    DgStageArgs a = stage_args(c, DG_MODE_RESIDUAL);
    cudaError_t e = c->kt->launch_stage(a, c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "residual kernel");
    c->launches++;
    return export_vector(c, c->K, r_out, on_device, "device->host copy of the residual");
}

int dg_max_wavespeed(dg_ctx *c, double *lam_host) {
    if (!c || !lam_host) return c ? fail(c, DG_EINVAL, "null pointer") : DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_max_wavespeed needs dg_bind and dg_set_state first");
    return read_lam(c, lam_host);
}

int dg_rk_step(dg_ctx *c, double dt, int nsteps) {
    if (!c) return DG_EINVAL;
    if (nsteps < 0 || !std::isfinite(dt)) return fail(c, DG_EINVAL, "nsteps < 0 or dt not finite");
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_rk_step needs dg_bind and dg_set_state first");
    // five stages back to back would read the neighbours' traces of the FIRST stage in all five (and, in push mode, store
    // into their buffers out of step): with halo faces the caller exchanges between stages
    for (int f = 0; f < 6; ++f)
        if (c->bc[f] == DG_BC_HALO)
            return fail(c, DG_EUNSUPPORTED, "face %d is a halo face: the faces must be exchanged after every stage, use dg_rk_stage", f);
    for (int step = 0; step < nsteps; ++step) {
        const int rc = enqueue_step(c, dt, 0.0);
        if (rc != DG_OK) return rc;
    }
    return DG_OK;
}

int dg_rk_stage(dg_ctx *c, double dt, int stage) {
    if (!c) return DG_EINVAL;
    if (stage < 0 || stage > 4 || !std::isfinite(dt)) return fail(c, DG_EINVAL, "stage outside 0..4 or dt not finite");
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_rk_stage needs dg_bind and dg_set_state first");
    int rc = check_halos(c);
    if (rc != DG_OK) return rc;
    c->lam_valid = false;
    return enqueue_stage(c, stage, dt, 0.0);
}

int dg_set_spacing(dg_ctx *c, const double h[3]) {
    if (!c || !h) return c ? fail(c, DG_EINVAL, "null spacing") : DG_EINVAL;
    if (c->bound) return fail(c, DG_ESTATE, "dg_set_spacing after dg_bind");
    for (int a = 0; a < 3; ++a)
        if (!(h[a] > 0.0) || !std::isfinite(h[a])) return fail(c, DG_EINVAL, "element size must be positive and finite");
    const int n[3] = {c->nx, c->ny, c->nz};
    for (int a = 0; a < 3; ++a) {
        c->h[a] = h[a];
        c->extent[a] = h[a] * n[a];
    }
    return DG_OK;
}

int dg_set_halo(dg_ctx *c, int face, const double *halo_dev) {
    if (!c || face < 0 || face > 5) return c ? fail(c, DG_EINVAL, "face outside 0..5") : DG_EINVAL;
    c->halo[face] = halo_dev;
    return DG_OK;
}

int dg_set_halo_pair(dg_ctx *c, int face, const double *halo0_dev, const double *halo1_dev) {
    if (!c || face < 0 || face > 5) return c ? fail(c, DG_EINVAL, "face outside 0..5") : DG_EINVAL;
    if ((halo0_dev == nullptr) != (halo1_dev == nullptr)) return fail(c, DG_EINVAL, "both buffers or none");
    c->halo2[face][0] = halo0_dev;
    c->halo2[face][1] = halo1_dev;
    return DG_OK;
}

int dg_set_halo_push(dg_ctx *c, int face, double *peer0_dev, double *peer1_dev) {
    if (!c || face < 0 || face > 5) return c ? fail(c, DG_EINVAL, "face outside 0..5") : DG_EINVAL;
    if ((peer0_dev == nullptr) != (peer1_dev == nullptr)) return fail(c, DG_EINVAL, "both buffers or none");
    // The stage kernel of THIS context's device stores into these buffers.  When they live on another GPU (peer
    // allocation or CUDA IPC mapping) the current device needs peer access to that GPU; opening an IPC handle enables
    // it only for the device that was current at the time, which need not be this one.
    double *const peers[2] = {peer0_dev, peer1_dev};
    for (int i = 0; i < 2 && peers[i]; ++i) {
        int rc = enable_peer_access_to(c, peers[i]);
        if (rc != DG_OK) return rc;
    }
    c->push[face][0] = peer0_dev;
    c->push[face][1] = peer1_dev;
    return DG_OK;
}

size_t dg_halo_len(const dg_ctx *c, int face) {
    if (!c || face < 0 || face > 5) return 0;
    if (face < 2) return (size_t)c->nz * c->nby * DG_NV * c->kt->cx;
    if (face < 4) return (size_t)c->nz * c->nbx * DG_NV * c->kt->cy;
    return (size_t)c->nby * c->nbx * DG_NV * c->kt->cz;
}

int dg_halo_export(dg_ctx *c, int face, double *dst_dev) {
    if (!c || !dst_dev || face < 0 || face > 5) return c ? fail(c, DG_EINVAL, "bad face or null buffer") : DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_halo_export needs dg_bind and dg_set_state first");
    const long long txy = c->kt->txy, tz = c->kt->tz, cx = c->kt->cx, cy = c->kt->cy, cz = c->kt->cz;
    const long long nbx = c->nbx, nby = c->nby, nz = c->nz;
    const double *src;
    long long n_outer, outer_stride, n_inner, inner_stride;
    int run;
    if (face < 2) {          // T- of the first / T+ of the last column along x, every (ez, by)
        src = c->Txy[c->tcur] + (face == 0 ? 0 : (nbx - 1) * txy + DG_NV * cx);
        n_outer = 1; outer_stride = 0; n_inner = nz * nby; inner_stride = nbx * txy; run = (int)(DG_NV * cx);
    } else if (face < 4) {   // ... along y, every (ez, bx)
        src = c->Txy[c->tcur] + 2 * DG_NV * cx + (face == 2 ? 0 : (nby - 1) * nbx * txy + DG_NV * cy);
        n_outer = nz; outer_stride = nby * nbx * txy; n_inner = nbx; inner_stride = txy; run = (int)(DG_NV * cy);
    } else {                 // T- of the first / T+ of the last layer, every column
        src = c->Tz[c->tcur] + (face == 4 ? 0 : ((long long)c->nchunks - 1) * nby * nbx * tz + DG_NV * cz);
        n_outer = 1; outer_stride = 0; n_inner = nby * nbx; inner_stride = tz; run = (int)(DG_NV * cz);
    }
    const long long total = n_outer * n_inner * run;
    const long long want = (total + 255) / 256, cap = (long long)(c->sms > 0 ? c->sms : 1) * 16;
    dg_pack_kernel<<<(unsigned)(want < cap ? (want ? want : 1) : cap), 256, 0, c->stream>>>(dst_dev, src, n_outer, outer_stride,
                                                                                       n_inner, inner_stride, run);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "pack kernel");
    c->launches++;
    return DG_OK;
}

int dg_rk_step_cfl(dg_ctx *c, double cfl, int nsteps, double *t_advanced, double *dt_last) {
    if (!c) return DG_EINVAL;
    if (nsteps < 0 || !(cfl > 0.0) || !std::isfinite(cfl)) return fail(c, DG_EINVAL, "nsteps < 0 or cfl not positive");
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_rk_step_cfl needs dg_bind and dg_set_state first");
    for (int f = 0; f < 6; ++f)
        if (c->bc[f] == DG_BC_HALO)
            return fail(c, DG_EUNSUPPORTED, "with halo faces the wavespeed is a maximum over all contexts: use dg_max_wavespeed + dg_rk_stage");
    double hmin = c->h[0];
    if (c->h[1] < hmin) hmin = c->h[1];
    if (c->h[2] < hmin) hmin = c->h[2];
    // the wavespeed of the state the call starts from is checked on the host (one read-back per call) ...
    double lam = 0.0;
    int rc = read_lam(c, &lam);
    if (rc != DG_OK) return rc;
    if (!(lam > 0.0) || !std::isfinite(lam)) return fail(c, DG_ENONPHYSICAL, "max wavespeed %g is not positive and finite: the state is non-physical, nothing stepped", lam);
    double out[2] = {0.0, 0.0};
    if (nsteps > 0) {
        // ... every step then forms its dt on the device from the wavespeed the step before reduced
        const double cfl_factor = cfl * hmin / (2.0 * c->p + 1.0);
        cudaError_t e = cudaMemsetAsync(c->scal + 2, 0, 16, c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "memset");
        for (int step = 0; step < nsteps; ++step) {
            rc = enqueue_step(c, 0.0, cfl_factor);
            if (rc != DG_OK) return rc;
        }
        e = cudaMemcpyAsync(out, c->scal + 2, 16, cudaMemcpyDeviceToHost, c->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
        if (e != cudaSuccess) return cuda_fail(c, e, "read-back of the time advanced");
    }
    if (t_advanced) *t_advanced = out[0];
    if (dt_last) *dt_last = out[1];
    if (!std::isfinite(out[0])) return fail(c, DG_ENONPHYSICAL, "the state became non-physical during the steps (time advanced %g)", out[0]);
    return DG_OK;
}

int dg_cfl_dt(const dg_ctx *c, double cfl, double lam_max, double *dt) {
    if (!c || !dt) return DG_EINVAL;
    if (!(cfl > 0.0) || !std::isfinite(cfl) || !(lam_max > 0.0) || !std::isfinite(lam_max)) return DG_EINVAL;
    double hmin = c->h[0];
    if (c->h[1] < hmin) hmin = c->h[1];
    if (c->h[2] < hmin) hmin = c->h[2];
    *dt = (cfl * hmin / (2.0 * c->p + 1.0)) / lam_max;   // the same operations, in the same order, as dg_rk_step_cfl's device-side dt
    return DG_OK;
}

int dg_split_volume(dg_ctx *c) {
    if (!c) return DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_split_volume needs dg_bind and dg_set_state first");
    cudaError_t e = c->kt->launch_split_volume(split_args(c), c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "volume kernel");
    c->launches++;
    return DG_OK;
}

int dg_split_surface(dg_ctx *c) {
    if (!c) return DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_split_surface needs dg_bind and dg_set_state first");
    for (int f = 0; f < 6; ++f)
        if (c->bc[f]) return fail(c, DG_EUNSUPPORTED, "the per-kernel mode is periodic only");
    cudaError_t e = c->kt->launch_split_surface(split_args(c), c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "surface kernel");
    c->launches++;
    return DG_OK;
}

int dg_split_update(dg_ctx *c, double dt, int stage) {
    if (!c) return DG_EINVAL;
    if (stage < 0 || stage > 4 || !std::isfinite(dt)) return fail(c, DG_EINVAL, "stage outside 0..4 or dt not finite");
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_split_update needs dg_bind and dg_set_state first");
    const size_t want = (c->int_len + 255) / 256, cap = (size_t)(c->sms > 0 ? c->sms : 1) * 16u;
    dg_split_update_kernel<<<(unsigned)(want < cap ? want : cap), 256, 0, c->stream>>>(
        c->Q, c->K, c->S, c->int_len, (double)kRkA[stage], (double)kRkB[stage], dt);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "update kernel");
    c->launches++;
    c->lam_valid = false;
    return refresh_traces(c);   // "project": face traces of the updated state, so that the fused path can go on
}

// Viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4 (reading R20; the paper names them only).
int dg_set_viscosity(dg_ctx *c, double mu, double prandtl) {
    if (!c) return DG_EINVAL;
    if (c->bound) return fail(c, DG_ESTATE, "dg_set_viscosity after dg_bind (it changes the workspace size)");
    if (!(mu >= 0.0) || !std::isfinite(mu) || !(prandtl > 0.0) || !std::isfinite(prandtl))
        return fail(c, DG_EINVAL, "need mu >= 0 and Prandtl number > 0");
    c->mu = mu;
    c->prandtl = prandtl;
    return DG_OK;
}

int dg_split_viscous(dg_ctx *c) {
    if (!c) return DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_split_viscous needs dg_bind and dg_set_state first");
    if (!(c->mu > 0.0)) return fail(c, DG_ESTATE, "no viscosity set (dg_set_viscosity before dg_bind)");
    for (int f = 0; f < 6; ++f)
        if (c->bc[f]) return fail(c, DG_EUNSUPPORTED, "the viscous terms are periodic only");
    DgViscArgs a;
    std::memset(&a, 0, sizeof(a));
    a.Q = c->Q;
    a.nx = c->nx; a.ny = c->ny; a.nz = c->nz;
    a.nbx = c->nbx; a.nby = c->nby;
    a.gm1 = c->gamma - 1.0;
    a.mu = c->mu;
    a.kappa = c->mu * c->gamma / (c->prandtl * (c->gamma - 1.0));
    for (int d = 0; d < 3; ++d) {
        a.S[d] = c->V[d];
        a.scale3[d] = c->g[d];
    }
    a.out = c->S;
    cudaError_t e = c->kt->launch_visc_gradflux(a, c->stream);   // steps v1 + v2: gradients, then Fv_a at the nodes
    c->launches++;
    if (e == cudaSuccess) {
        e = c->kt->launch_visc_div(a, c->stream);                // step v3: R += div Fv
        c->launches++;
    }
    if (e != cudaSuccess) return cuda_fail(c, e, "viscous kernels");
    return DG_OK;
}

int dg_rk_step_ns(dg_ctx *c, double dt, int nsteps) {
    if (!c) return DG_EINVAL;
    if (nsteps < 0 || !std::isfinite(dt)) return fail(c, DG_EINVAL, "nsteps < 0 or dt not finite");
    for (int step = 0; step < nsteps; ++step)
        for (int s = 0; s < 5; ++s) {
            int rc = dg_split_volume(c);
            if (rc == DG_OK) rc = dg_split_surface(c);
            if (rc == DG_OK) rc = dg_split_viscous(c);
            if (rc == DG_OK) rc = dg_split_update(c, dt, s);
            if (rc != DG_OK) return rc;
        }
    return DG_OK;
}

int dg_split_get_r(dg_ctx *c, double *r_out, int on_device) {
    if (!c || !r_out) return c ? fail(c, DG_EINVAL, "null pointer") : DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_split_get_r needs dg_bind and dg_set_state first");
    if (on_device) return launch_layout(c, c->S, r_out, 0);
    // host: R lives in the staging vector itself, so the canonical copy goes through the K array (dead between steps)
    int rc = launch_layout(c, c->S, c->K, 0);
    if (rc != DG_OK) return rc;
    cudaError_t e = cudaMemcpyAsync(r_out, c->K, c->state_len * 8, cudaMemcpyDeviceToHost, c->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) return cuda_fail(c, e, "device->host copy of the residual");
    return DG_OK;
}

int dg_get_state(dg_ctx *c, double *q_out, int on_device) {
    if (!c || !q_out) return c ? fail(c, DG_EINVAL, "null state pointer") : DG_EINVAL;
    if (!c->bound || !c->has_state) return fail(c, DG_ESTATE, "dg_get_state needs dg_bind and dg_set_state first");
    return export_vector(c, c->Q, q_out, on_device, "device->host copy of the state");
}

int dg_nodes(const dg_ctx *c, double *xi, double *w) {
    if (!c || !xi || !w) return DG_EINVAL;
    HostOps o;
    build_host_ops(c->N, o);
    for (int i = 0; i < c->N; ++i) {
        xi[i] = (double)o.xi[i];
        w[i] = (double)o.w[i];
    }
    return DG_OK;
}

unsigned long long dg_launch_count(const dg_ctx *c) { return c ? c->launches : 0; }

int dg_kernel_info(const dg_ctx *c, long long out[8]) {
    if (!c || !out) return DG_EINVAL;
    out[0] = c->kt->bx; out[1] = c->kt->by; out[2] = c->lz;
    out[3] = c->kt->threads;
    out[4] = c->kt->smem_bytes;
    out[5] = c->bound ? (long long)c->blocks_per_sm * c->sms : (long long)c->nbx * c->nby * c->nchunks;
    out[6] = (long long)((c->int_len + (1u << 20) - 1) >> 20);
    out[7] = c->variant;
    return DG_OK;
}

int dg_selftest_fastmath(const double *x, double *r, double *q, size_t n, void *stream) {
    if (!x || !r || !q) return DG_EINVAL;
    if (n == 0) return DG_OK;
    dg_fastmath_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(x, r, q, n);
    return cudaGetLastError() == cudaSuccess ? DG_OK : DG_ECUDA;
}

int dg_fp64_peak(double *out, int blocks, int iters, void *stream, unsigned long long *fma_count) {
    if (!out || blocks < 1 || iters < 1) return DG_EINVAL;
    dg_fp64_peak_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(out, iters, 0.999999, 1e-6);
    if (fma_count) *fma_count = (unsigned long long)blocks * 256ull * (unsigned long long)iters * 128ull;
    return cudaGetLastError() == cudaSuccess ? DG_OK : DG_ECUDA;
}

int dg_destroy(dg_ctx *c) {
    delete c;
    return DG_OK;
}

const char *dg_last_error(const dg_ctx *c) { return c ? c->err : "null context"; }

}  // extern "C"
