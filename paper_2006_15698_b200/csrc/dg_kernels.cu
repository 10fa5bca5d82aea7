// dg_kernels.cu -- CUDA kernels of the DG Euler time step for one N = p+1 (compile with -DDG_N=<N>,
// -gencode arch=compute_100a,code=sm_100a).  Hand-written for B200; fp64 throughout.
//
// The fused stage kernel does, for one "brick" of BX x BY x BZ elements per thread block and in one
// sweep over HBM:
//   P0  stage the brick's Q (5 x nodes) in shared memory, stage the 6 neighbour bricks' face traces,
//       prefetch the brick's K lines into L2
//   PA  one thread per node LINE and axis: pointwise Euler flux (eq (2)-(3)) at the
//       line's N nodes, V_i = sum_q Dhat_iq F_q in registers (eq (5) 2nd term, the
//       contraction of listing lines 220-237), and the two face traces T+- = sum_q l_q(+-1) Q_q
//   PB  local Lax-Friedrichs interface flux at the + end of every line, and at the - end
//       of the lines that start on the brick boundary (neighbour traces come from the trace buffer)
//   PC  lift and 2/h scaling: r_i = (2/h_a) (V_i - (l_i(+1) F*_+ - l_i(-1) F*_-)/w_i)  (eq (5) 3rd term)
//   PD  sum of the three axes; LSERK45 stage  K = A K + dt R, Q = Q + B K written
//       straight back to HBM; or R itself in residual mode
//   PE  face traces of the UPDATED Q on the brick boundary, written to the other trace buffer
// so that Q and K are read once and written once per stage and no element ever needs another
// element's nodal values: neighbours meet only through the double-buffered brick-boundary traces.
//
// Nothing here is shared with oracle/ (separate source, separate operator construction).
#include "dg_internal.h"

#ifndef DG_N
#error "compile with -DDG_N=<p+1>"
#endif

namespace {

__constant__ DgOps c_ops;

// ------------------------------------------------------------------------------------------------
// compile-time geometry of one variant
// ------------------------------------------------------------------------------------------------
template <int N_, int BX_, int BY_, int BZ_, int MINB_>
struct Cfg {
    static constexpr int N = N_, BX = BX_, BY = BY_, BZ = BZ_, MINB = MINB_;
    static constexpr int GX = BX * N, GY = BY * N, GZ = BZ * N;   // nodes of the brick per axis
    static constexpr int NODES = GX * GY * GZ;
    static constexpr int SLOT = DG_NV * NODES;                     // doubles per brick in Q, K, R
    static constexpr int GXP = GX | 1;                             // odd shared-memory pitch: x-lines conflict-free
    static constexpr int PLANE = GZ * GY * GXP;                    // shared doubles per variable
    static constexpr int L = NODES / N;                            // node lines per axis
    static constexpr int THREADS = (3 * L + 31) / 32 * 32;
    static constexpr int CX = GY * GZ, CY = GX * GZ, CZ = GX * GY; // face nodes of a brick side per axis
    static constexpr int CMAX = CX > CY ? (CX > CZ ? CX : CZ) : (CY > CZ ? CY : CZ);
    static constexpr int TSLOT = 2 * DG_NV * (CX + CY + CZ);       // trace doubles per brick
    static constexpr int SMEM_DOUBLES = 3 * DG_NV * PLANE + 2 * 3 * DG_NV * L + 3 * 2 * DG_NV * CMAX;
    static constexpr int SMEM_BYTES = SMEM_DOUBLES * 8;
};

__device__ __forceinline__ void prefetch_l2(const void *p) {
    asm volatile("prefetch.global.L2 [%0];" ::"l"(p));
}

// Column `axis` of the Euler flux matrix, eq (2)-(3) (listing lines 186-217).
// Same expression tree as DESIGN.md "arithmetic form".
__device__ __forceinline__ void euler_flux(const double (&Q)[DG_NV], int axis, double gm1, double (&F)[DG_NV],
                                           double &vel, double &pres, double &oneOrho) {
    oneOrho = 1.0 / Q[0];
    const double u = Q[1] * oneOrho, v = Q[2] * oneOrho, w = Q[3] * oneOrho;
    pres = gm1 * (Q[4] - 0.5 * Q[0] * (u * u + v * v + w * w));
    const double Ep = Q[4] + pres;
    vel = (axis == 0) ? u : (axis == 1) ? v : w;
    F[0] = Q[0] * vel;
    F[1] = Q[1] * vel + ((axis == 0) ? pres : 0.0);
    F[2] = Q[2] * vel + ((axis == 1) ? pres : 0.0);
    F[3] = Q[3] * vel + ((axis == 2) ? pres : 0.0);
    F[4] = Ep * vel;
}

// Local Lax-Friedrichs flux (reading R3):
//   F* = 1/2 (F(QL) + F(QR)) - 1/2 lam (QR - QL),  lam = max(|u_a^L| + c_L, |u_a^R| + c_R)
__device__ __forceinline__ void lax_friedrichs(const double (&QL)[DG_NV], const double (&QR)[DG_NV], int axis,
                                               double gamma, double gm1, double (&Fs)[DG_NV]) {
    double FL[DG_NV], FR[DG_NV], uL, uR, pL, pR, rL, rR;
    euler_flux(QL, axis, gm1, FL, uL, pL, rL);
    euler_flux(QR, axis, gm1, FR, uR, pR, rR);
    const double lamL = fabs(uL) + sqrt(gamma * pL * rL);
    const double lamR = fabs(uR) + sqrt(gamma * pR * rR);
    const double lam = (lamL > lamR) ? lamL : lamR;
#pragma unroll
    for (int n = 0; n < DG_NV; ++n) Fs[n] = 0.5 * (FL[n] + FR[n]) - 0.5 * lam * (QR[n] - QL[n]);
}

// ------------------------------------------------------------------------------------------------
// the fused stage kernel
// ------------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(C::THREADS, C::MINB) dg_stage_kernel(const __grid_constant__ DgStageArgs a) {
    constexpr int N = C::N, GX = C::GX, GY = C::GY, GXP = C::GXP;
    constexpr int NODES = C::NODES, PLANE = C::PLANE, L = C::L, THREADS = C::THREADS, CMAX = C::CMAX;
    constexpr int NV = DG_NV;

    extern __shared__ __align__(16) double smem[];
    double *Qs = smem;                  // [5][PLANE]   nodal values of the brick (old, then updated)
    double *S1 = Qs + NV * PLANE;       // [5][PLANE]   x-axis contribution to R
    double *S2 = S1 + NV * PLANE;       // [5][PLANE]   y-axis contribution to R
    double *Tms = S2 + NV * PLANE;      // [3][5][L]    T- of every line (right state of the line below)
    double *Fss = Tms + 3 * NV * L;     // [3][5][L]    F* at the + end of every line
    double *Hs = Fss + 3 * NV * L;      // [3][2][5][CMAX] neighbour bricks' traces (halo)

    const int tid = threadIdx.x;
    const long long brick = blockIdx.x;
    const int bxi = (int)(brick % a.nbx);
    const int byi = (int)((brick / a.nbx) % a.nby);
    const int bzi = (int)(brick / ((long long)a.nbx * a.nby));
    const int ext0 = min(C::BX, a.nx - bxi * C::BX);   // elements of this brick per axis (ragged last brick)
    const int ext1 = min(C::BY, a.ny - byi * C::BY);
    const int ext2 = min(C::BZ, a.nz - bzi * C::BZ);
    const int nodx = ext0 * N, nody = ext1 * N, nodz = ext2 * N;
    const size_t qbase = (size_t)brick * C::SLOT;
    const int mode = a.mode;

    // ---------------- P0: stage Q, stage neighbour traces, prefetch K -------------------------------
    {
        constexpr int ITERS = (NV * NODES + THREADS - 1) / THREADS;
        double tmp[ITERS];
#pragma unroll
        for (int it = 0; it < ITERS; ++it) {
            const int idx = tid + it * THREADS;
            const int n = idx / NODES, r = idx - n * NODES;
            const int gz = r / (GY * GX), r2 = r - gz * (GY * GX);
            const int gy = r2 / GX, gx = r2 - gy * GX;
            const bool ok = (idx < NV * NODES) && gx < nodx && gy < nody && gz < nodz;
            tmp[it] = ok ? a.Q[qbase + idx] : 0.0;
        }
#pragma unroll
        for (int it = 0; it < ITERS; ++it) {
            const int idx = tid + it * THREADS;
            const int n = idx / NODES, r = idx - n * NODES;
            const int gz = r / (GY * GX), r2 = r - gz * (GY * GX);
            const int gy = r2 / GX, gx = r2 - gy * GX;
            if (idx < NV * NODES) Qs[n * PLANE + (gz * GY + gy) * GXP + gx] = tmp[it];
        }
    }
    if (mode != DG_MODE_TRACES) {
        // halo: side 0 = T+ of the brick below along the axis (left state of my - faces),
        //       side 1 = T- of the brick above (right state of my + faces)
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            const int Ca = (ax == 0) ? C::CX : (ax == 1) ? C::CY : C::CZ;
            const int T1 = (ax == 0) ? GY : GX;                       // fastest transverse dimension
            const int lim1 = (ax == 0) ? nody : nodx;
            const int lim2 = (ax == 2) ? nody : nodz;
            const int tbase = (ax == 0) ? 0 : (ax == 1) ? 2 * NV * C::CX : 2 * NV * (C::CX + C::CY);
            int bm[3] = {bxi, byi, bzi}, bp[3] = {bxi, byi, bzi};
            const int nb = (ax == 0) ? a.nbx : (ax == 1) ? a.nby : a.nbz;
            bm[ax] = (bm[ax] + nb - 1) % nb;
            bp[ax] = (bp[ax] + 1) % nb;
            const size_t brm = (size_t)bm[0] + (size_t)a.nbx * ((size_t)bm[1] + (size_t)a.nby * bm[2]);
            const size_t brp = (size_t)bp[0] + (size_t)a.nbx * ((size_t)bp[1] + (size_t)a.nby * bp[2]);
            for (int idx = tid; idx < 2 * NV * Ca; idx += THREADS) {
                const int side = idx / (NV * Ca), r = idx - side * (NV * Ca);
                const int n = r / Ca, c = r - n * Ca;
                const int t2 = c / T1, t1 = c - t2 * T1;
                if (t1 < lim1 && t2 < lim2) {
                    const size_t src = (side == 0 ? brm : brp) * C::TSLOT + tbase + ((1 - side) * NV + n) * Ca + c;
                    Hs[((ax * 2 + side) * NV + n) * CMAX + c] = a.Told[src];
                }
            }
        }
        if (mode == DG_MODE_STAGE && a.rkA != 0.0) {
            constexpr int LINES = (C::SLOT + 15) / 16;
            for (int i = tid; i < LINES; i += THREADS) prefetch_l2(a.K + qbase + min(i * 16, C::SLOT - 1));
        }
    }
    __syncthreads();

    // ---------------- thread -> (axis, line) -------------------------------------------------------
    const int grp = tid / L;                  // 0,1,2 = lines along x,y,z
    const int l = tid - grp * L;
    const int axis = grp < 3 ? grp : 0;
    const int Ca = (axis == 0) ? C::CX : (axis == 1) ? C::CY : C::CZ;
    const int e = l / Ca, c = l - e * Ca;      // element along the axis, face node
    const int T1 = (axis == 0) ? GY : GX;
    const int t2 = c / T1, t1 = c - t2 * T1;
    int base, stride, exta;
    bool active;
    if (axis == 0) {        // (t1,t2) = (gy,gz)
        base = (t2 * GY + t1) * GXP + e * N; stride = 1; exta = ext0;
        active = t1 < nody && t2 < nodz;
    } else if (axis == 1) { // (t1,t2) = (gx,gz)
        base = (t2 * GY + e * N) * GXP + t1; stride = GXP; exta = ext1;
        active = t1 < nodx && t2 < nodz;
    } else {                // (t1,t2) = (gx,gy)
        base = (e * N * GY + t2) * GXP + t1; stride = GY * GXP; exta = ext2;
        active = t1 < nodx && t2 < nody;
    }
    active = active && grp < 3 && e < exta;
    const int tbase = (axis == 0) ? 0 : (axis == 1) ? 2 * NV * C::CX : 2 * NV * (C::CX + C::CY);

    double V[NV][N];

    if (mode != DG_MODE_TRACES) {
        double Tp[NV], Tm[NV];
        // ------------- PA: flux, sum-factorised derivative, traces ---------------------------------
        if (active) {
#pragma unroll
            for (int n = 0; n < NV; ++n) {
                Tp[n] = 0.0;
                Tm[n] = 0.0;
#pragma unroll
                for (int i = 0; i < N; ++i) V[n][i] = 0.0;
            }
#pragma unroll
            for (int q = 0; q < N; ++q) {
                double Qn[NV], F[NV], vel, pres, rinv;
#pragma unroll
                for (int n = 0; n < NV; ++n) Qn[n] = Qs[n * PLANE + base + q * stride];
                euler_flux(Qn, axis, a.gm1, F, vel, pres, rinv);
#pragma unroll
                for (int n = 0; n < NV; ++n) {
#pragma unroll
                    for (int i = 0; i < N; ++i) V[n][i] = fma(c_ops.Dhat[i * N + q], F[n], V[n][i]);
                    Tp[n] = fma(c_ops.lp[q], Qn[n], Tp[n]);
                    Tm[n] = fma(c_ops.lm[q], Qn[n], Tm[n]);
                }
            }
#pragma unroll
            for (int n = 0; n < NV; ++n) Tms[(grp * NV + n) * L + l] = Tm[n];
        }
        __syncthreads();

        // ------------- PB: interface fluxes ---------------------------------------------------------
        double Fp[NV], Fm[NV];
        if (active) {
            double Qo[NV];
            if (e + 1 < exta) {
#pragma unroll
                for (int n = 0; n < NV; ++n) Qo[n] = Tms[(grp * NV + n) * L + l + Ca];
            } else {
#pragma unroll
                for (int n = 0; n < NV; ++n) Qo[n] = Hs[((grp * 2 + 1) * NV + n) * CMAX + c];
            }
            lax_friedrichs(Tp, Qo, axis, a.gamma, a.gm1, Fp);
#pragma unroll
            for (int n = 0; n < NV; ++n) Fss[(grp * NV + n) * L + l] = Fp[n];
            if (e == 0) {
#pragma unroll
                for (int n = 0; n < NV; ++n) Qo[n] = Hs[((grp * 2 + 0) * NV + n) * CMAX + c];
                lax_friedrichs(Qo, Tm, axis, a.gamma, a.gm1, Fm);
            }
        }
        __syncthreads();

        // ------------- PC: lift, scale, hand the x and y contributions over -------------------------
        if (active) {
            if (e > 0) {
#pragma unroll
                for (int n = 0; n < NV; ++n) Fm[n] = Fss[(grp * NV + n) * L + l - Ca];
            }
            const double g = a.g[axis];
#pragma unroll
            for (int n = 0; n < NV; ++n) {
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    const double lift = c_ops.lpw[i] * Fp[n] - c_ops.lmw[i] * Fm[n];
                    const double r = g * (V[n][i] - lift);
                    if (grp == 0) S1[n * PLANE + base + i * stride] = r;
                    else if (grp == 1) S2[n * PLANE + base + i * stride] = r;
                    else V[n][i] = r;
                }
            }
        }
        __syncthreads();

        // ------------- PD: R = (Rx + Ry) + Rz; Runge-Kutta stage; write back ------------------------
        if (active && grp == 2) {
            const double A = a.rkA, B = a.rkB, dt = a.dt;
            const bool readK = (A != 0.0);
            const size_t g0 = qbase + (size_t)((e * N) * GY + t2) * GX + t1;   // node q=0 of this z-line, n=0
            if (mode == DG_MODE_RESIDUAL) {
#pragma unroll
                for (int n = 0; n < NV; ++n)
#pragma unroll
                    for (int q = 0; q < N; ++q) {
                        const int sa = n * PLANE + base + q * stride;
                        a.Rout[g0 + (size_t)n * NODES + (size_t)q * (GY * GX)] = (S1[sa] + S2[sa]) + V[n][q];
                    }
            } else {
                double Kold[NV][N];
                if (readK) {
#pragma unroll
                    for (int n = 0; n < NV; ++n)
#pragma unroll
                        for (int q = 0; q < N; ++q) Kold[n][q] = a.K[g0 + (size_t)n * NODES + (size_t)q * (GY * GX)];
                }
#pragma unroll
                for (int n = 0; n < NV; ++n)
#pragma unroll
                    for (int q = 0; q < N; ++q) {
                        const int sa = n * PLANE + base + q * stride;
                        const size_t go = g0 + (size_t)n * NODES + (size_t)q * (GY * GX);
                        const double R = (S1[sa] + S2[sa]) + V[n][q];
                        const double Kn = readK ? fma(A, Kold[n][q], dt * R) : dt * R;
                        const double Qn = fma(B, Kn, Qs[sa]);
                        a.K[go] = Kn;
                        a.Q[go] = Qn;
                        Qs[sa] = Qn;
                    }
            }
        }
        if (mode == DG_MODE_RESIDUAL) return;
        __syncthreads();
    }

    // ---------------- PE: traces of the (updated) Q on the brick boundary ---------------------------
    if (active && (e == 0 || e == exta - 1)) {
        double Tp[NV], Tm[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            Tp[n] = 0.0;
            Tm[n] = 0.0;
        }
#pragma unroll
        for (int q = 0; q < N; ++q) {
#pragma unroll
            for (int n = 0; n < NV; ++n) {
                const double Qv = Qs[n * PLANE + base + q * stride];
                Tp[n] = fma(c_ops.lp[q], Qv, Tp[n]);
                Tm[n] = fma(c_ops.lm[q], Qv, Tm[n]);
            }
        }
        double *dst = a.Tnew + (size_t)brick * C::TSLOT + tbase + c;
        if (e == 0) {
#pragma unroll
            for (int n = 0; n < NV; ++n) dst[(0 * NV + n) * Ca] = Tm[n];
        }
        if (e == exta - 1) {
#pragma unroll
            for (int n = 0; n < NV; ++n) dst[(1 * NV + n) * Ca] = Tp[n];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// layout conversion canonical [e][k][j][i][n] <-> internal [brick][n][gz][gy][gx]
// one thread per node; canonical side reads/writes 40 contiguous bytes per thread
// ------------------------------------------------------------------------------------------------
template <class C>
__device__ __forceinline__ size_t internal_offset(size_t node, int nx, int ny, int nbx, int nby) {
    constexpr int N = C::N;
    const int i = (int)(node % N);
    size_t r = node / N;
    const int j = (int)(r % N);
    r /= N;
    const int k = (int)(r % N);
    r /= N;                                    // element index e = ex + nx (ey + ny ez)
    const int ex = (int)(r % nx);
    r /= nx;
    const int ey = (int)(r % ny);
    const int ez = (int)(r / ny);
    const int bxi = ex / C::BX, byi = ey / C::BY, bzi = ez / C::BZ;
    const int gx = (ex - bxi * C::BX) * N + i, gy = (ey - byi * C::BY) * N + j, gz = (ez - bzi * C::BZ) * N + k;
    const size_t brick = (size_t)bxi + (size_t)nbx * ((size_t)byi + (size_t)nby * bzi);
    return brick * C::SLOT + (size_t)(gz * C::GY + gy) * C::GX + gx;
}

template <class C>
__global__ void __launch_bounds__(256) dg_layout_kernel(const DgLayoutArgs a) {
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    for (size_t node = (size_t)blockIdx.x * blockDim.x + threadIdx.x; node < total;
         node += (size_t)gridDim.x * blockDim.x) {
        const size_t io = internal_offset<C>(node, a.nx, a.ny, a.nbx, a.nby);
        if (a.to_internal) {
#pragma unroll
            for (int n = 0; n < DG_NV; ++n) a.internal[io + (size_t)n * C::NODES] = a.canonical[node * DG_NV + n];
        } else {
#pragma unroll
            for (int n = 0; n < DG_NV; ++n) a.canonical[node * DG_NV + n] = a.internal[io + (size_t)n * C::NODES];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// max wavespeed  lam = max_nodes sqrt(u^2+v^2+w^2) + sqrt(gamma p / rho)   (reading R10)
// ------------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(256) dg_wavespeed_kernel(const DgWaveArgs a) {
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    double best = 0.0;
    for (size_t node = (size_t)blockIdx.x * blockDim.x + threadIdx.x; node < total;
         node += (size_t)gridDim.x * blockDim.x) {
        const size_t io = internal_offset<C>(node, a.nx, a.ny, a.nbx, a.nby);
        const double Q0 = a.Q[io], Q1 = a.Q[io + (size_t)C::NODES], Q2 = a.Q[io + 2 * (size_t)C::NODES],
                     Q3 = a.Q[io + 3 * (size_t)C::NODES], Q4 = a.Q[io + 4 * (size_t)C::NODES];
        const double rinv = 1.0 / Q0;
        const double u = Q1 * rinv, v = Q2 * rinv, w = Q3 * rinv;
        const double pres = a.gm1 * (Q4 - 0.5 * Q0 * (u * u + v * v + w * w));
        const double s = sqrt(u * u + v * v + w * w) + sqrt(a.gamma * pres * rinv);
        best = (s > best) ? s : best;
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double o = __shfl_xor_sync(0xffffffffu, best, off);
        best = (o > best) ? o : best;
    }
    if ((threadIdx.x & 31) == 0) atomicMax(a.lam_bits, (unsigned long long)__double_as_longlong(best));
}

// ------------------------------------------------------------------------------------------------
// host-side launchers, one table per variant
// ------------------------------------------------------------------------------------------------
template <class C>
cudaError_t upload_ops(const DgOps *ops, cudaStream_t s) {
    cudaError_t err = cudaMemcpyToSymbolAsync(c_ops, ops, sizeof(DgOps), 0, cudaMemcpyHostToDevice, s);
    if (err != cudaSuccess) return err;
    err = cudaStreamSynchronize(s);   // ops lives on the caller's stack
    if (err != cudaSuccess) return err;
    return cudaFuncSetAttribute(dg_stage_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
}

template <class C>
cudaError_t launch_stage(const DgStageArgs &a, cudaStream_t s) {
    const long long bricks = (long long)a.nbx * a.nby * a.nbz;
    if (bricks <= 0 || bricks > 2147483647LL) return cudaErrorInvalidConfiguration;
    dg_stage_kernel<C><<<(unsigned)bricks, C::THREADS, C::SMEM_BYTES, s>>>(a);
    return cudaGetLastError();
}

inline unsigned flat_grid(size_t total) {
    const size_t want = (total + 255) / 256;
    const size_t cap = 148u * 16u;   // grid-stride: a few blocks per SM
    return (unsigned)(want < cap ? (want ? want : 1) : cap);
}

template <class C>
cudaError_t launch_layout(const DgLayoutArgs &a, cudaStream_t s) {
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    dg_layout_kernel<C><<<flat_grid(total), 256, 0, s>>>(a);
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_wavespeed(const DgWaveArgs &a, cudaStream_t s) {
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    dg_wavespeed_kernel<C><<<flat_grid(total), 256, 0, s>>>(a);
    return cudaGetLastError();
}

template <class C>
constexpr DgKernelTable make_table() {
    return DgKernelTable{C::N,       C::BX,          C::BY,           C::BZ,
                         C::THREADS, C::SMEM_BYTES,  C::SLOT,         C::TSLOT,
                         &upload_ops<C>, &launch_stage<C>, &launch_layout<C>, &launch_wavespeed<C>};
}

// Brick shapes per N (default first).  DESIGN.md "brick shapes" explains the choice: threads = 3 x
// lines per brick must leave >= 2 blocks per SM within the register file, and the brick-boundary
// trace traffic 160/(B_a N) bytes per node and axis should stay <= ~80 B per node.
#if DG_N == 2
using V0 = Cfg<2, 4, 4, 2, 2>;
using V1 = Cfg<2, 2, 2, 2, 4>;
using V2 = Cfg<2, 4, 4, 4, 1>;
#elif DG_N == 3
using V0 = Cfg<3, 2, 2, 2, 3>;
using V1 = Cfg<3, 1, 1, 1, 8>;
using V2 = Cfg<3, 4, 2, 2, 2>;
#elif DG_N == 4
using V0 = Cfg<4, 2, 2, 1, 3>;
using V1 = Cfg<4, 1, 1, 1, 6>;
using V2 = Cfg<4, 2, 2, 2, 1>;
#elif DG_N == 5
using V0 = Cfg<5, 2, 1, 1, 3>;
using V1 = Cfg<5, 1, 1, 1, 6>;
using V2 = Cfg<5, 2, 2, 1, 1>;
#elif DG_N == 6
using V0 = Cfg<6, 1, 1, 1, 4>;
using V1 = Cfg<6, 2, 1, 1, 2>;
using V2 = Cfg<6, 2, 2, 1, 1>;
#elif DG_N == 7
using V0 = Cfg<7, 1, 1, 1, 3>;
using V1 = Cfg<7, 2, 1, 1, 1>;
using V2 = Cfg<7, 1, 1, 1, 2>;
#elif DG_N == 8
using V0 = Cfg<8, 1, 1, 1, 2>;
using V1 = Cfg<8, 1, 1, 1, 1>;
using V2 = Cfg<8, 2, 1, 1, 1>;
#else
#error "DG_N must be 2..8"
#endif

const DgKernelTable k_tables[] = {make_table<V0>(), make_table<V1>(), make_table<V2>()};

}  // namespace

#define DG_CAT2(a, b) a##b
#define DG_CAT(a, b) DG_CAT2(a, b)
const DgKernelTable *DG_CAT(dg_variants_N, DG_N)(int *count) {
    *count = (int)(sizeof(k_tables) / sizeof(k_tables[0]));
    return k_tables;
}
