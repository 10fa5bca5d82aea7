// dg_internal.h -- shared between the C-ABI translation unit (dg_api.cu) and the per-degree
// kernel translation units (dg_kernels.cu compiled once per N = p+1 with -DDG_N=<N>).
// Not part of the public boundary (include/dg_b200.h is).
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>

#define DG_NV 5      // rho, rho u, rho v, rho w, rho E       (eq (2))
#define DG_NMAX 8    // largest N = p+1 compiled

// 1-D operators of the collocated Gauss-Legendre Lagrange basis on the reference element [-1,1]
// (PAPER.md:72-80), built on the host in long double (dg_api.cu), rounded to double once.  They depend on
// N = p+1 only, so every kernel translation unit keeps ONE copy in __constant__ memory (uploaded by
// prepare()); the constant geometric factor 2/h_a of each axis and the time step travel
// in DgStageArgs::scale and are applied when an axis' contribution is added to the Runge-Kutta register.
// The nodes are symmetric: l_i(-1) = l_{N-1-i}(+1), so the "-" tables are the "+" tables read backwards.
struct DgRefOps {
    double D[DG_NMAX][DG_NMAX];   // D[q][i] = w_q l_i'(xi_q) / w_i        (eq (5) 2nd term / mass)
    double lq[DG_NMAX];           // 1/2 l_i(+1) / w_i                     (lift / mass; the kernel forms 2 F*)
    double lp[DG_NMAX];           // l_i(+1)                               (face traces)
    // Even-odd form of the same operators (symmetric nodes: Dhat is centro-antisymmetric, Dhat[N-1-i][N-1-q] = -Dhat[i][q]),
    // H = N/2, q' = N-1-q, i' = N-1-i; the kernels use it for N >= 5 (N^2/2 + 2N instead of N^2 + 2N operations per line
    // and variable for derivative + lift):
    //   r_i = a_i + s_i, r_i' = s_i - a_i,  a_i = sum_{q<H} Pe[q][i] (F_q + F_q') (+ Dm[i] F_mid),  s_i = sum_{q<H} Po[q][i] (F_q - F_q')
    double Pe[DG_NMAX / 2][DG_NMAX / 2];       // 1/2 (Dhat[i][q] + Dhat[i][q'])
    double Po[DG_NMAX / 2][DG_NMAX / 2 + 1];   // 1/2 (Dhat[i][q] - Dhat[i][q']), i up to the middle node
    double Dm[DG_NMAX / 2];                    // Dhat[i][mid] (odd N)
    double ls[DG_NMAX / 2 + 1];                // lift, even part: 1/2 (lq[i] + lq[i']) (middle node: lq[mid]); multiplies (F*_- - F*_+)
    double la[DG_NMAX / 2];                    // lift, odd part:  1/2 (lq[i'] - lq[i]);                        multiplies (F*_- + F*_+)
};

#ifdef __CUDACC__
// Branch-free reciprocal and square root for positive, normal arguments (densities, gamma p / rho):
// hardware seed (MUFU.RCP64H / MUFU.RSQ64H, good to about 2^-20) and ONE cubic correction; measured error
// <= 1 ulp (reciprocal) and <= 2 ulp (square root) over 14 decades (dg_selftest_fastmath in dg_b200_test.h
// exposes them; tests/test_gpu_parity.py::test_fast_math), with none of the slow-path branches of the
// IEEE-rounded library routines and about half their operations.
__device__ __forceinline__ double rcp_pos(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    const double e = fma(-x, r, 1.0);
    return fma(r, fma(e, e, e), r);                    // r (1 + e + e^2)
}
__device__ __forceinline__ double sqrt_pos(double x) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e = fma(-(x * y), y, 1.0);         // 1 - x y^2
    y = fma(y, e * fma(0.375, e, 0.5), y);          // y (1 + e/2 + 3 e^2/8)
    return x * y;
}
#endif

enum DgMode {
    DG_MODE_STAGE = 0,     // full Runge-Kutta stage: residual + K,Q update + new traces
    DG_MODE_RESIDUAL = 1   // residual only, written to the K array (internal layout)
};

// Arguments of the fused stage kernel (passed by value, lives in the constant bank).
//
// Internal layout: the mesh is cut into COLUMNS of BX x BY elements; one "layer" of a column
// (BX x BY x 1 elements) is one contiguous slot [n][k][HP] of Q and K, HP = the (gy,gx) node plane padded to
// an even number of doubles; slot index = (ez * nby + by) * nbx + bx.
struct DgStageArgs {
    double *Q;            // state
    double *K;            // Runge-Kutta register (RESIDUAL mode: the residual lands here)
    const double *Txy_old;  // x and y face traces of the current Q on the column boundaries, per layer slot
    double *Txy_new;        // ... of the updated Q
    const double *Tz_old;   // z face traces of the current Q at the ends of every chunk of lz layers, per chunk slot
    double *Tz_new;
    unsigned long long *lam_bits;   // LAM kernels: max wavespeed of the updated state (bit pattern, atomicMax)
    int nx, ny, nz;       // elements per axis
    int nbx, nby;         // columns per axis
    int lz, nchunks;      // layers per chunk (the unit of work of one thread block), chunks per column
    double gamma, gm1;
    double rkA, rkB;      // stage coefficients; rkA == 0 means "do not read K" (stage 1)
    int mode;
    int want_lam;
    int store_k;          // 0 in the last stage of a step: K is dead then (the next stage 1 has A = 0) and is not written
    double scale[3];      // 2/h_a per axis, times dt in stage mode: K accumulates dt * L(Q)
    // CFL stepping (dg_rk_step_cfl): when lam_in is set the time step is formed ON THE DEVICE, dt = cfl_factor / lam
    // with lam the max wavespeed the previous step's last stage left in *lam_in, and multiplies `scale`; the first
    // block of a step's first stage adds dt to t_acc[0] and stores it in t_acc[1].  No host round trip per step.
    const unsigned long long *lam_in;
    double cfl_factor;    // cfl * min(h) / (2p + 1)
    double *t_acc;
    // Faces whose neighbour lives in ANOTHER context (block decomposition over GPUs): the traces of
    // the elements beyond domain face f come from the caller's buffer halo_ext[f] (null: none), laid out like the
    // neighbour's export (dg_halo_export): x faces [ez][by][5][CX], y faces [ez][bx][5][CY], z faces [by][bx][5][CZ]
    const double *halo_ext[6];
    // "push" mode: the stage kernel ALSO stores the traces of the UPDATED state on domain face f into halo_push[f] (null:
    // none), the buffer the neighbour context reads as its halo_ext of the opposite face in the NEXT stage -- possibly in
    // a peer GPU's memory (NVLink stores from inside the kernel instead of an export kernel and a message)
    double *halo_push[6];
    int bc[6];            // domain faces x-, x+, y-, y+, z-, z+: 0 periodic, 1 slip wall, 2 far field (R19)
    double qinf[DG_NV];   // far-field state (conserved variables)
};

struct DgTraceArgs {
    const double *Q;
    double *Txy, *Tz;
    int nx, ny, nz, nbx, nby, lz, nchunks;
};

// Arguments of the paper-shaped per-kernel mode (Table II): volume and surface kernels.
struct DgSplitArgs {
    const double *Q;
    double *R;            // residual accumulator, internal layout (volume kernel overwrites it, surface kernel adds)
    int nx, ny, nz, nbx, nby;
    double gamma, gm1;
    double scale[3];      // 2/h_a per axis
};

// Arguments of the viscous-term kernels (reading R20).
struct DgViscArgs {
    const double *Q;      // state, internal layout
    double *S[3];         // dg_visc_gradflux_kernel: out, the nodal viscous fluxes Fv_a; dg_visc_div_kernel: in
    double *out;          // dg_visc_div_kernel: the residual vector it adds div Fv to, internal layout
    int nx, ny, nz, nbx, nby;
    double scale3[3];     // 2/h_a per axis
    double gm1, mu, kappa;   // gamma - 1, dynamic viscosity, mu gamma / (Pr (gamma - 1))
};

struct DgLayoutArgs {
    double *internal;
    double *canonical;      // [e][k][j][i][n]
    int nx, ny, nz, nbx, nby;
    int to_internal;        // 1: canonical -> internal, 0: internal -> canonical
};

struct DgWaveArgs {
    const double *Q;
    unsigned long long *lam_bits;  // max reduced on the bit pattern (non-negative doubles order as integers)
    int nx, ny, nz, nbx, nby;
    double gamma, gm1;
};

// One compiled (N, column shape) variant.
struct DgKernelTable {
    int N, bx, by;
    int threads;             // threads per block of the stage kernel (compute warps + 1 copy warp)
    int smem_bytes;          // dynamic shared memory of the stage kernel
    long long slot;          // doubles per layer slot in Q/K
    long long txy;           // x/y face-trace doubles per layer slot
    long long tz;            // z face-trace doubles per chunk slot
    int cx, cy, cz;          // face nodes of a layer slot's x side, y side, and of a column's z side
    int reload;
    int minb;                // blocks per SM the kernel is compiled for (__launch_bounds__)
    // upload the reference operators, opt in to the shared memory size; *blocks_per_sm = resident blocks per SM
    cudaError_t (*prepare)(const DgRefOps &ref, int *blocks_per_sm);
    cudaError_t (*launch_stage)(const DgStageArgs &a, cudaStream_t s);
    cudaError_t (*launch_traces)(const DgTraceArgs &a, cudaStream_t s);
    cudaError_t (*launch_split_volume)(const DgSplitArgs &a, cudaStream_t s);
    cudaError_t (*launch_split_surface)(const DgSplitArgs &a, cudaStream_t s);
    cudaError_t (*launch_layout)(const DgLayoutArgs &a, int sms, cudaStream_t s);
    cudaError_t (*launch_wavespeed)(const DgWaveArgs &a, int sms, cudaStream_t s);
    cudaError_t (*launch_visc_gradflux)(const DgViscArgs &a, cudaStream_t s);
    cudaError_t (*launch_visc_div)(const DgViscArgs &a, cudaStream_t s);
};

// Each kernel TU exports its variants: dg_variants_N<N>(&count) -> array of tables, default first.
#define DG_DECLARE_VARIANTS(NN) const DgKernelTable *dg_variants_N##NN(int *count);
DG_DECLARE_VARIANTS(2)
DG_DECLARE_VARIANTS(3)
DG_DECLARE_VARIANTS(4)
DG_DECLARE_VARIANTS(5)
DG_DECLARE_VARIANTS(6)
DG_DECLARE_VARIANTS(7)
DG_DECLARE_VARIANTS(8)
