// dg_kernels.cu -- CUDA kernels of the DG Euler time step for one N = p+1 (compile with -DDG_N=<N>,
// -gencode arch=compute_100a,code=sm_100a).  Hand-written for B200; fp64 throughout.
//
// The fused stage kernel does, for one "brick" of BX x BY x BZ elements per thread block and in one
// sweep over HBM:
//   P0  asynchronous copies (cp.async, no registers): the brick's Q (5 x nodes) and the 6 neighbour
//       bricks' face traces into shared memory
//   then, one thread per node LINE, for the axes x, y, z in turn:
//   PA  pointwise Euler flux (eq (2)-(3)) at the line's N nodes,
//       V_i = sum_q Dhat_iq F_q in registers (eq (5) 2nd term, the contraction of
//       listing lines 220-237), and the two face traces T+- = sum_q l_q(+-1) Q_q
//   PB  local Lax-Friedrichs interface flux at the + end of the line, and at the - end of
//       the lines that start on the brick boundary (neighbour traces come from the trace buffer)
//   PC  lift and 2/h scaling: r_i = (2/h_a) (V_i - (l_i(+1) F*_+ - l_i(-1) F*_-)/w_i)  (eq (5) 3rd term),
//       accumulated over the axes in shared memory
//   PD  (with the z lines, whose global accesses coalesce) LSERK45 stage  K = A K + dt R, Q = Q + B K
//       (PAPER.md:80, 254): K read and K, Q written straight from/to HBM; or R itself in residual mode
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
    static constexpr int P = GX | 1;                               // odd shared-memory row pitch: x-lines conflict-free
    static constexpr int ROWS = GZ * GY;                           // rows per variable
    static constexpr int PLANE = ROWS * P;                         // shared doubles per variable
    static constexpr int L = NODES / N;                            // node lines per axis = threads that work
    static constexpr int THREADS = (L + 31) / 32 * 32;
    static constexpr int CX = GY * GZ, CY = GX * GZ, CZ = GX * GY; // face nodes of a brick side per axis
    static constexpr int TSLOT = 2 * DG_NV * (CX + CY + CZ);       // trace doubles per brick
    static constexpr bool MULTI = (BX > 1) || (BY > 1) || (BZ > 1);
    static constexpr int LINEBUF = MULTI ? DG_NV * L : 0;          // T- / F* hand-over between elements of a brick
    static constexpr int SMEM_DOUBLES = 2 * DG_NV * PLANE + TSLOT + 2 * LINEBUF;
    static constexpr int SMEM_BYTES = SMEM_DOUBLES * 8;
};

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit_wait_all() {
    asm volatile("cp.async.commit_group;\ncp.async.wait_group 0;" ::: "memory");
}

// Column AX of the Euler flux matrix, eq (2)-(3) (listing lines 186-217).
// Same expression tree as DESIGN.md "arithmetic form".
template <int AX>
__device__ __forceinline__ void euler_flux(const double (&Q)[DG_NV], double gm1, double (&F)[DG_NV], double &vel,
                                           double &pres, double &oneOrho) {
    oneOrho = 1.0 / Q[0];
    const double u = Q[1] * oneOrho, v = Q[2] * oneOrho, w = Q[3] * oneOrho;
    pres = gm1 * (Q[4] - 0.5 * Q[0] * (u * u + v * v + w * w));
    const double Ep = Q[4] + pres;
    vel = (AX == 0) ? u : (AX == 1) ? v : w;
    F[0] = Q[0] * vel;
    F[1] = Q[1] * vel + ((AX == 0) ? pres : 0.0);
    F[2] = Q[2] * vel + ((AX == 1) ? pres : 0.0);
    F[3] = Q[3] * vel + ((AX == 2) ? pres : 0.0);
    F[4] = Ep * vel;
}

// Local Lax-Friedrichs flux (reading R3):
//   F* = 1/2 (F(QL) + F(QR)) - 1/2 lam (QR - QL),  lam = max(|u_a^L| + c_L, |u_a^R| + c_R)
template <int AX>
__device__ __forceinline__ void lax_friedrichs(const double (&QL)[DG_NV], const double (&QR)[DG_NV], double gamma,
                                               double gm1, double (&Fs)[DG_NV]) {
    double FL[DG_NV], FR[DG_NV], uL, uR, pL, pR, rL, rR;
    euler_flux<AX>(QL, gm1, FL, uL, pL, rL);
    euler_flux<AX>(QR, gm1, FR, uR, pR, rR);
    const double lamL = fabs(uL) + sqrt(gamma * pL * rL);
    const double lamR = fabs(uR) + sqrt(gamma * pR * rR);
    const double lam = (lamL > lamR) ? lamL : lamR;
#pragma unroll
    for (int n = 0; n < DG_NV; ++n) Fs[n] = 0.5 * (FL[n] + FR[n]) - 0.5 * lam * (QR[n] - QL[n]);
}

// ------------------------------------------------------------------------------------------------
// geometry of one node line along axis AX inside the brick, for thread `l`
//   l = e * Ca + c,  e = element along the axis, c = face node = t2 * T1 + t1
//   axis x: (t1,t2) = (gy,gz);  y: (gx,gz);  z: (gx,gy)
// ------------------------------------------------------------------------------------------------
template <class C, int AX>
struct Line {
    static constexpr int Ca = (AX == 0) ? C::CX : (AX == 1) ? C::CY : C::CZ;
    static constexpr int T1 = (AX == 0) ? C::GY : C::GX;
    static constexpr int Ba = (AX == 0) ? C::BX : (AX == 1) ? C::BY : C::BZ;
    static constexpr int STRIDE = (AX == 0) ? 1 : (AX == 1) ? C::P : C::GY * C::P;   // shared-memory node stride
    static constexpr int TBASE = (AX == 0) ? 0 : (AX == 1) ? 2 * DG_NV * C::CX : 2 * DG_NV * (C::CX + C::CY);
    int e, c, t1, t2, base, exta;
    bool active;
    __device__ __forceinline__ Line(int l, int nodx, int nody, int nodz, int ext0, int ext1, int ext2) {
        e = (Ba == 1) ? 0 : l / Ca;
        c = l - e * Ca;
        t2 = c / T1;
        t1 = c - t2 * T1;
        if (AX == 0) {
            base = (t2 * C::GY + t1) * C::P + e * C::N;
            exta = ext0;
            active = t1 < nody && t2 < nodz;
        } else if (AX == 1) {
            base = (t2 * C::GY + e * C::N) * C::P + t1;
            exta = ext1;
            active = t1 < nodx && t2 < nodz;
        } else {
            base = (e * C::N * C::GY + t2) * C::P + t1;
            exta = ext2;
            active = t1 < nodx && t2 < nody;
        }
        active = active && l < C::L && e < exta;
    }
};

// PA..PC for one axis: returns r[n][i] = (2/h_a) (V - lift) of this thread's line.
template <class C, int AX>
__device__ __forceinline__ void axis_residual(const Line<C, AX> &ln, int l, const double *Qs, const double *Hs,
                                              double *Tms, double *Fss, const DgStageArgs &a,
                                              double (&V)[DG_NV][C::N]) {
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE, L = C::L;
    using LN = Line<C, AX>;
    constexpr int Ca = LN::Ca, STRIDE = LN::STRIDE, Ba = LN::Ba;
    double Tp[NV], Tm[NV];
    // ------------- PA: flux, sum-factorised derivative, traces -------------------------------------
    if (ln.active) {
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
            for (int n = 0; n < NV; ++n) Qn[n] = Qs[n * PLANE + ln.base + q * STRIDE];
            euler_flux<AX>(Qn, a.gm1, F, vel, pres, rinv);
#pragma unroll
            for (int n = 0; n < NV; ++n) {
#pragma unroll
                for (int i = 0; i < N; ++i) V[n][i] = fma(c_ops.Dhat[i * N + q], F[n], V[n][i]);
                Tp[n] = fma(c_ops.lp[q], Qn[n], Tp[n]);
                Tm[n] = fma(c_ops.lm[q], Qn[n], Tm[n]);
            }
        }
        if (Ba > 1) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Tms[n * L + l] = Tm[n];
        }
    }
    if (Ba > 1) __syncthreads();

    // ------------- PB: interface fluxes ------------------------------------------------------------
    double Fp[NV], Fm[NV];
    if (ln.active) {
        double Qo[NV];
        if (Ba > 1 && ln.e + 1 < ln.exta) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Qo[n] = Tms[n * L + l + Ca];
        } else {
#pragma unroll
            for (int n = 0; n < NV; ++n) Qo[n] = Hs[LN::TBASE + (NV + n) * Ca + ln.c];
        }
        lax_friedrichs<AX>(Tp, Qo, a.gamma, a.gm1, Fp);
        if (Ba > 1) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Fss[n * L + l] = Fp[n];
        }
        if (ln.e == 0) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Qo[n] = Hs[LN::TBASE + n * Ca + ln.c];
            lax_friedrichs<AX>(Qo, Tm, a.gamma, a.gm1, Fm);
        }
    }
    if (Ba > 1) __syncthreads();

    // ------------- PC: lift, scale -----------------------------------------------------------------
    if (ln.active) {
        if (Ba > 1 && ln.e > 0) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Fm[n] = Fss[n * L + l - Ca];
        }
        const double g = a.g[AX];
#pragma unroll
        for (int n = 0; n < NV; ++n) {
#pragma unroll
            for (int i = 0; i < N; ++i) {
                const double lift = c_ops.lpw[i] * Fp[n] - c_ops.lmw[i] * Fm[n];
                V[n][i] = g * (V[n][i] - lift);
            }
        }
    }
}

// PE for one axis: traces of the (updated) Q in shared memory on the brick boundary -> Tnew.
template <class C, int AX>
__device__ __forceinline__ void boundary_traces(const Line<C, AX> &ln, const double *Qs, double *Tbrick) {
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE;
    using LN = Line<C, AX>;
    if (ln.active && (ln.e == 0 || ln.e == ln.exta - 1)) {
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
                const double Qv = Qs[n * PLANE + ln.base + q * LN::STRIDE];
                Tp[n] = fma(c_ops.lp[q], Qv, Tp[n]);
                Tm[n] = fma(c_ops.lm[q], Qv, Tm[n]);
            }
        }
        double *dst = Tbrick + LN::TBASE + ln.c;
        if (ln.e == 0) {
#pragma unroll
            for (int n = 0; n < NV; ++n) dst[n * LN::Ca] = Tm[n];
        }
        if (ln.e == ln.exta - 1) {
#pragma unroll
            for (int n = 0; n < NV; ++n) dst[(NV + n) * LN::Ca] = Tp[n];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// the fused stage kernel
// ------------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(C::THREADS, C::MINB) dg_stage_kernel(const __grid_constant__ DgStageArgs a) {
    constexpr int N = C::N, GX = C::GX, GY = C::GY, P = C::P;
    constexpr int NODES = C::NODES, PLANE = C::PLANE, L = C::L, THREADS = C::THREADS;
    constexpr int NV = DG_NV;

    extern __shared__ __align__(16) double smem[];
    double *Qs = smem;                  // [5][PLANE]  nodal values of the brick (old, then updated)
    double *Rs = Qs + NV * PLANE;       // [5][PLANE]  x (+ y) contribution to R
    double *Hs = Rs + NV * PLANE;       // [TSLOT]     neighbour bricks' traces, laid out like a brick's own slot:
                                        //             [axis][side][5][Ca]; side 0 = T+ of the brick below,
                                        //             side 1 = T- of the brick above
    double *Tms = Hs + C::TSLOT;        // [5][L]      T- of every line (right state of the line below)
    double *Fss = Tms + C::LINEBUF;     // [5][L]      F* at the + end of every line

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

    // ---------------- P0: asynchronous staging of Q and of the neighbour traces ----------------------
    {
        const double *src = a.Q + qbase;
        constexpr int TOTAL = NV * NODES;
#pragma unroll 4
        for (int idx = tid; idx < TOTAL; idx += THREADS) {
            const int row = idx / GX;                         // row over all 5 variables: PLANE = ROWS * P
            cp_async8(Qs + idx + row * (P - GX), src + idx);
        }
    }
    if (mode != DG_MODE_TRACES) {
#pragma unroll
        for (int ax = 0; ax < 3; ++ax) {
            const int Ca = (ax == 0) ? C::CX : (ax == 1) ? C::CY : C::CZ;
            const int tbase = (ax == 0) ? 0 : (ax == 1) ? 2 * NV * C::CX : 2 * NV * (C::CX + C::CY);
            int bm[3] = {bxi, byi, bzi}, bp[3] = {bxi, byi, bzi};
            const int nb = (ax == 0) ? a.nbx : (ax == 1) ? a.nby : a.nbz;
            bm[ax] = (bm[ax] == 0) ? nb - 1 : bm[ax] - 1;
            bp[ax] = (bp[ax] + 1 == nb) ? 0 : bp[ax] + 1;
            const size_t brm = (size_t)bm[0] + (size_t)a.nbx * ((size_t)bm[1] + (size_t)a.nby * bm[2]);
            const size_t brp = (size_t)bp[0] + (size_t)a.nbx * ((size_t)bp[1] + (size_t)a.nby * bp[2]);
            const double *srcm = a.Told + brm * C::TSLOT + tbase + NV * Ca;   // T+ (side 1) of the brick below
            const double *srcp = a.Told + brp * C::TSLOT + tbase;             // T- (side 0) of the brick above
            for (int r = tid; r < NV * Ca; r += THREADS) {
                cp_async8(Hs + tbase + r, srcm + r);
                cp_async8(Hs + tbase + NV * Ca + r, srcp + r);
            }
        }
    }
    cp_async_commit_wait_all();
    __syncthreads();

    const int l = tid;
    const Line<C, 2> lz(l, nodx, nody, nodz, ext0, ext1, ext2);
    double *Tbrick = a.Tnew + (size_t)brick * C::TSLOT;

    if (mode != DG_MODE_TRACES) {
        double V[NV][N];
        // ---------------- x lines --------------------------------------------------------------------
        {
            const Line<C, 0> lx(l, nodx, nody, nodz, ext0, ext1, ext2);
            axis_residual<C, 0>(lx, l, Qs, Hs, Tms, Fss, a, V);
            if (lx.active) {
#pragma unroll
                for (int n = 0; n < NV; ++n)
#pragma unroll
                    for (int i = 0; i < N; ++i) Rs[n * PLANE + lx.base + i] = V[n][i];
            }
        }
        __syncthreads();
        // ---------------- y lines --------------------------------------------------------------------
        {
            const Line<C, 1> ly(l, nodx, nody, nodz, ext0, ext1, ext2);
            axis_residual<C, 1>(ly, l, Qs, Hs, Tms, Fss, a, V);
            if (ly.active) {
#pragma unroll
                for (int n = 0; n < NV; ++n)
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        const int sa = n * PLANE + ly.base + i * P;
                        Rs[sa] = Rs[sa] + V[n][i];
                    }
            }
        }
        __syncthreads();
        // ---------------- z lines: residual, Runge-Kutta stage, write back ---------------------------
        constexpr int ZS = Line<C, 2>::STRIDE;
        const size_t g0 = qbase + (size_t)(lz.e * N) * (GY * GX) + lz.c;   // node q=0 of this z-line, n=0
        const bool readK = (mode == DG_MODE_STAGE) && (a.rkA != 0.0);
        double Kold[NV][N];
        if (lz.active && readK) {   // issued before the z contraction: the loads land while it runs
#pragma unroll
            for (int n = 0; n < NV; ++n)
#pragma unroll
                for (int q = 0; q < N; ++q) Kold[n][q] = __ldcs(a.K + g0 + (size_t)n * NODES + (size_t)q * (GY * GX));
        }
        axis_residual<C, 2>(lz, l, Qs, Hs, Tms, Fss, a, V);
        if (lz.active) {
            if (mode == DG_MODE_RESIDUAL) {
#pragma unroll
                for (int n = 0; n < NV; ++n)
#pragma unroll
                    for (int q = 0; q < N; ++q)
                        a.Rout[g0 + (size_t)n * NODES + (size_t)q * (GY * GX)] = Rs[n * PLANE + lz.base + q * ZS] + V[n][q];
            } else {
                const double A = a.rkA, B = a.rkB, dt = a.dt;
                double Tp[NV], Tm[NV];
#pragma unroll
                for (int n = 0; n < NV; ++n) {
                    Tp[n] = 0.0;
                    Tm[n] = 0.0;
#pragma unroll
                    for (int q = 0; q < N; ++q) {
                        const int sa = n * PLANE + lz.base + q * ZS;
                        const size_t go = g0 + (size_t)n * NODES + (size_t)q * (GY * GX);
                        const double R = Rs[sa] + V[n][q];
                        const double Kn = readK ? fma(A, Kold[n][q], dt * R) : dt * R;
                        const double Qn = fma(B, Kn, Qs[sa]);
                        a.K[go] = Kn;
                        a.Q[go] = Qn;
                        Qs[sa] = Qn;
                        Tp[n] = fma(c_ops.lp[q], Qn, Tp[n]);
                        Tm[n] = fma(c_ops.lm[q], Qn, Tm[n]);
                    }
                }
                // z traces of the updated Q straight from registers
                double *dst = Tbrick + Line<C, 2>::TBASE + lz.c;
                if (lz.e == 0) {
#pragma unroll
                    for (int n = 0; n < NV; ++n) dst[n * C::CZ] = Tm[n];
                }
                if (lz.e == lz.exta - 1) {
#pragma unroll
                    for (int n = 0; n < NV; ++n) dst[(NV + n) * C::CZ] = Tp[n];
                }
            }
        }
        if (mode == DG_MODE_RESIDUAL) return;
        __syncthreads();
    } else {
        boundary_traces<C, 2>(lz, Qs, Tbrick);
    }

    // ---------------- PE: x and y traces of the updated Q on the brick boundary -----------------------
    {
        const Line<C, 0> lx(l, nodx, nody, nodz, ext0, ext1, ext2);
        boundary_traces<C, 0>(lx, Qs, Tbrick);
        const Line<C, 1> ly(l, nodx, nody, nodz, ext0, ext1, ext2);
        boundary_traces<C, 1>(ly, Qs, Tbrick);
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

// Brick shapes per N (default first).  DESIGN.md "brick shapes" explains the choice: about 350-650 nodes
// per brick keeps Q + R + halo under ~70 KB of shared memory (3+ blocks per SM overlap each other's load,
// compute and store phases) while the brick-boundary trace traffic 160/(B_a N) bytes per node and axis
// stays at 53-69 B per node.
#if DG_N == 2
using V0 = Cfg<2, 4, 4, 4, 3>;
using V1 = Cfg<2, 2, 2, 2, 4>;
using V2 = Cfg<2, 4, 4, 2, 4>;
#elif DG_N == 3
using V0 = Cfg<3, 3, 3, 2, 3>;
using V1 = Cfg<3, 1, 1, 1, 8>;
using V2 = Cfg<3, 2, 2, 2, 4>;
#elif DG_N == 4
using V0 = Cfg<4, 2, 2, 2, 3>;
using V1 = Cfg<4, 1, 1, 1, 8>;
using V2 = Cfg<4, 2, 2, 1, 4>;
#elif DG_N == 5
using V0 = Cfg<5, 1, 2, 2, 3>;
using V1 = Cfg<5, 1, 1, 1, 8>;
using V2 = Cfg<5, 2, 2, 1, 3>;
#elif DG_N == 6
using V0 = Cfg<6, 1, 1, 2, 4>;
using V1 = Cfg<6, 1, 1, 1, 6>;
using V2 = Cfg<6, 2, 2, 1, 2>;
#elif DG_N == 7
using V0 = Cfg<7, 1, 1, 1, 5>;
using V1 = Cfg<7, 2, 1, 1, 3>;
using V2 = Cfg<7, 1, 1, 2, 3>;
#elif DG_N == 8
using V0 = Cfg<8, 1, 1, 1, 4>;
using V1 = Cfg<8, 2, 1, 1, 2>;
using V2 = Cfg<8, 1, 1, 2, 2>;
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
