// dg_kernels.cu -- CUDA kernels of the DG Euler time step for one N = p+1 (compile with -DDG_N=<N>,
// -gencode arch=compute_100a,code=sm_100a).  Hand-written for B200; fp64 throughout.
//
// The fused stage kernel is PERSISTENT: each thread block strides over "bricks" of BX x BY x BZ elements
// and, for every brick, in one sweep over HBM:
//   P0  asynchronous copies (cp.async, no registers) of the NEXT brick's Q (5 x nodes) and of its 6
//       neighbour bricks' face traces into the other half of a double buffer in shared memory, plus an
//       L2 prefetch of its K, all of which land while the current brick is being computed
//   then, one thread per node LINE, for the axes x, y, z in turn (one rolled loop, small code):
//   PA  pointwise Euler flux (eq (2)-(3)) at the line's N nodes,
//       V_i = sum_q Dhat_iq F_q in registers (eq (5) 2nd term, the contraction of
//       listing lines 220-237), and the two face traces T+- = sum_q l_q(+-1) Q_q
//   PB  local Lax-Friedrichs interface flux at the + end of the line, and at the - end of
//       the lines that start on the brick boundary (neighbour traces come from the trace buffer)
//   PC  lift with 2/h folded in: r_i = V_i - (l_i(+1) F*_+ - l_i(-1) F*_-) (2/h_a)/w_i  (eq (5) 3rd term),
//       accumulated over the axes in shared memory
//   PD  (with the z lines, whose global accesses coalesce) LSERK45 stage  K = A K + dt R, Q = Q + B K
//       (PAPER.md:80, 254): K read and K, Q written straight from/to HBM; or R itself in residual mode
//   PE  face traces of the UPDATED Q on the brick boundary, written to the other trace buffer
// so that Q and K are read once and written once per stage and no element ever needs another
// element's nodal values: neighbours meet only through the double-buffered brick-boundary traces.
//
// Nothing here is shared with oracle/ (separate source, separate operator construction).
#include "dg_internal.h"

#include <stdint.h>

#ifndef DG_N
#error "compile with -DDG_N=<p+1>"
#endif

namespace {

// ------------------------------------------------------------------------------------------------
// compile-time geometry of one variant
// ------------------------------------------------------------------------------------------------
template <int N_, int BX_, int BY_, int BZ_, int MINB_, int NBUF_>
struct Cfg {
    static constexpr int N = N_, BX = BX_, BY = BY_, BZ = BZ_, MINB = MINB_, NBUF = NBUF_;
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
    static constexpr int SMEM_DOUBLES = (NBUF + 1) * DG_NV * PLANE + TSLOT + 2 * LINEBUF;
    static constexpr int SMEM_BYTES = SMEM_DOUBLES * 8;
};

__device__ __forceinline__ void cp_async8(double *smem_dst, const double *gsrc) {
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int PENDING>
__device__ __forceinline__ void cp_async_wait() {
    asm volatile("cp.async.wait_group %0;" ::"n"(PENDING) : "memory");
}
// Ask L2 to fetch [ptr, ptr + bytes) (rounded out to 16-byte granules): one instruction per brick of K.
__device__ __forceinline__ void l2_prefetch(const void *ptr, unsigned bytes) {
    const uintptr_t lo = (uintptr_t)ptr & ~(uintptr_t)15;
    const uintptr_t hi = ((uintptr_t)ptr + bytes + 15) & ~(uintptr_t)15;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(lo), "r"((unsigned)(hi - lo)) : "memory");
}

// Euler flux along the face/line normal, eq (2)-(3) (listing lines 186-217), for a state
// whose momentum components have been ROTATED so that slot 1 is the normal one:
//   slots = (rho, rho u_a, rho u_b, rho u_c, rho E),  (a,b,c) = (x,y,z), (y,z,x) or (z,x,y).
// One copy of the code then serves the three axes with no run-time selection.
__device__ __forceinline__ void euler_flux_normal(const double (&Q)[DG_NV], double gm1, double (&F)[DG_NV],
                                                  double &vel, double &pres, double &oneOrho) {
    oneOrho = 1.0 / Q[0];
    vel = Q[1] * oneOrho;
    const double ub = Q[2] * oneOrho, uc = Q[3] * oneOrho;
    pres = gm1 * (Q[4] - 0.5 * Q[0] * (vel * vel + ub * ub + uc * uc));
    F[0] = Q[0] * vel;
    F[1] = Q[1] * vel + pres;
    F[2] = Q[2] * vel;
    F[3] = Q[3] * vel;
    F[4] = (Q[4] + pres) * vel;
}

// Local Lax-Friedrichs flux (reading R3), rotated slots as above:
//   F* = 1/2 (F(QL) + F(QR)) - 1/2 lam (QR - QL),  lam = max(|u_a^L| + c_L, |u_a^R| + c_R)
// written for (own, other) with sgn = +1 when own is the left state, -1 when it is the right one.
__device__ __forceinline__ void lax_friedrichs(const double (&Qown)[DG_NV], const double (&Qoth)[DG_NV], double sgn,
                                               double gamma, double gm1, double (&Fs)[DG_NV]) {
    double Fa[DG_NV], Fb[DG_NV], ua, ub, pa, pb, ra, rb;
    euler_flux_normal(Qown, gm1, Fa, ua, pa, ra);
    euler_flux_normal(Qoth, gm1, Fb, ub, pb, rb);
    const double lama = fabs(ua) + sqrt(gamma * pa * ra);
    const double lamb = fabs(ub) + sqrt(gamma * pb * rb);
    const double hl = 0.5 * sgn * ((lama > lamb) ? lama : lamb);
#pragma unroll
    for (int n = 0; n < DG_NV; ++n) Fs[n] = 0.5 * (Fa[n] + Fb[n]) - hl * (Qoth[n] - Qown[n]);
}

// ------------------------------------------------------------------------------------------------
// geometry of the node line of thread `l` along axis `ax` inside the brick
//   l = e * Ca + c,  e = element along the axis, c = face node = t2 * T1 + t1
//   axis x: (t1,t2) = (gy,gz);  y: (gx,gz);  z: (gx,gy)
// ------------------------------------------------------------------------------------------------
struct Line {
    int e, c, base, stride, Ca, tbase, exta;
    bool active, multi;
};

template <class C>
__device__ __forceinline__ Line make_line(int ax, int l, int ext0, int ext1, int ext2) {
    constexpr int N = C::N;
    Line ln;
    int t1, t2;
    if (ax == 0) {
        ln.Ca = C::CX;
        ln.e = (C::BX == 1) ? 0 : l / C::CX;
        ln.c = l - ln.e * C::CX;
        t2 = ln.c / C::GY;
        t1 = ln.c - t2 * C::GY;
        ln.base = (t2 * C::GY + t1) * C::P + ln.e * N;
        ln.stride = 1;
        ln.tbase = 0;
        ln.exta = ext0;
        ln.multi = C::BX > 1;
        ln.active = t1 < ext1 * N && t2 < ext2 * N;
    } else if (ax == 1) {
        ln.Ca = C::CY;
        ln.e = (C::BY == 1) ? 0 : l / C::CY;
        ln.c = l - ln.e * C::CY;
        t2 = ln.c / C::GX;
        t1 = ln.c - t2 * C::GX;
        ln.base = (t2 * C::GY + ln.e * N) * C::P + t1;
        ln.stride = C::P;
        ln.tbase = 2 * DG_NV * C::CX;
        ln.exta = ext1;
        ln.multi = C::BY > 1;
        ln.active = t1 < ext0 * N && t2 < ext2 * N;
    } else {
        ln.Ca = C::CZ;
        ln.e = (C::BZ == 1) ? 0 : l / C::CZ;
        ln.c = l - ln.e * C::CZ;
        t2 = ln.c / C::GX;
        t1 = ln.c - t2 * C::GX;
        ln.base = (ln.e * N * C::GY + t2) * C::P + t1;
        ln.stride = C::GY * C::P;
        ln.tbase = 2 * DG_NV * (C::CX + C::CY);
        ln.exta = ext2;
        ln.multi = C::BZ > 1;
        ln.active = t1 < ext0 * N && t2 < ext1 * N;
    }
    ln.active = ln.active && l < C::L && ln.e < ln.exta;
    return ln;
}

// P0a: enqueue the asynchronous copy of one brick's Q, and ask L2 for its K and its neighbours' traces.
template <class C>
__device__ __forceinline__ void issue_q_loads(const DgStageArgs &a, int brick, double *Qd, int tid, bool want_k) {
    constexpr int NV = DG_NV, GX = C::GX, P = C::P, THREADS = C::THREADS;
    const double *src = a.Q + (size_t)brick * C::SLOT;
    constexpr int TOTAL = NV * C::NODES;
#pragma unroll 4
    for (int idx = tid; idx < TOTAL; idx += THREADS) {
        const int row = idx / GX;                         // row over all 5 variables: PLANE = ROWS * P
        cp_async8(Qd + idx + row * (P - GX), src + idx);
    }
    if (want_k && tid == 0) l2_prefetch(a.K + (size_t)brick * C::SLOT, C::SLOT * 8);
}

// Neighbour brick and offset of the trace block a brick needs for (axis, side): side 0 = T+ of the brick
// below (stored as that brick's side 1), side 1 = T- of the brick above (its side 0).
template <class C>
__device__ __forceinline__ const double *halo_source(const DgStageArgs &a, int bxi, int byi, int bzi, int ax, int side) {
    const int Ca = (ax == 0) ? C::CX : (ax == 1) ? C::CY : C::CZ;
    const int tbase = (ax == 0) ? 0 : (ax == 1) ? 2 * DG_NV * C::CX : 2 * DG_NV * (C::CX + C::CY);
    int bx = bxi, by = byi, bz = bzi;   // (no run-time indexed local array: it would live in local memory)
    if (ax == 0) bx = (side == 0) ? ((bx == 0) ? a.nbx - 1 : bx - 1) : ((bx + 1 == a.nbx) ? 0 : bx + 1);
    else if (ax == 1) by = (side == 0) ? ((by == 0) ? a.nby - 1 : by - 1) : ((by + 1 == a.nby) ? 0 : by + 1);
    else bz = (side == 0) ? ((bz == 0) ? a.nbz - 1 : bz - 1) : ((bz + 1 == a.nbz) ? 0 : bz + 1);
    const size_t nbr = (size_t)bx + (size_t)a.nbx * ((size_t)by + (size_t)a.nby * bz);
    return a.Told + nbr * C::TSLOT + tbase + (side == 0 ? DG_NV * Ca : 0);
}

// P0b: enqueue the asynchronous copies of the 6 neighbour trace blocks of this brick.
template <class C>
__device__ __forceinline__ void issue_halo_loads(const DgStageArgs &a, int bxi, int byi, int bzi, double *Hd, int tid) {
    constexpr int NV = DG_NV, THREADS = C::THREADS;
#pragma unroll
    for (int ax = 0; ax < 3; ++ax) {
        const int Ca = (ax == 0) ? C::CX : (ax == 1) ? C::CY : C::CZ;
        const int tbase = (ax == 0) ? 0 : (ax == 1) ? 2 * NV * C::CX : 2 * NV * (C::CX + C::CY);
        const double *srcm = halo_source<C>(a, bxi, byi, bzi, ax, 0);
        const double *srcp = halo_source<C>(a, bxi, byi, bzi, ax, 1);
        for (int r = tid; r < NV * Ca; r += THREADS) {
            cp_async8(Hd + tbase + r, srcm + r);
            cp_async8(Hd + tbase + NV * Ca + r, srcp + r);
        }
    }
}

// ... and the L2 prefetch of the same 6 blocks for the NEXT brick (6 threads, one instruction each).
template <class C>
__device__ __forceinline__ void prefetch_halo(const DgStageArgs &a, int brick, int tid) {
    if (tid < 6) {
        const int bxi = brick % a.nbx, byi = (brick / a.nbx) % a.nby, bzi = brick / (a.nbx * a.nby);
        const int ax = tid >> 1, side = tid & 1;
        const int Ca = (ax == 0) ? C::CX : (ax == 1) ? C::CY : C::CZ;
        l2_prefetch(halo_source<C>(a, bxi, byi, bzi, ax, side), DG_NV * Ca * 8);
    }
}

// PE for one axis: traces of the (updated) Q in shared memory on the brick boundary -> Tnew.
template <class C>
__device__ __forceinline__ void boundary_traces(const Line &ln, const double *Qs, double *Tbrick,
                                                const DgStageArgs &a) {
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE;
    if (ln.active && (ln.e == 0 || ln.e == ln.exta - 1)) {
        double Tp[NV], Tm[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            Tp[n] = 0.0;
            Tm[n] = 0.0;
        }
#pragma unroll
        for (int q = 0; q < N; ++q) {
            const double lpq = a.ops.lp[q], lmq = a.ops.lm[q];
#pragma unroll
            for (int n = 0; n < NV; ++n) {
                const double Qv = Qs[n * PLANE + ln.base + q * ln.stride];
                Tp[n] = fma(lpq, Qv, Tp[n]);
                Tm[n] = fma(lmq, Qv, Tm[n]);
            }
        }
        double *dst = Tbrick + ln.tbase + ln.c;
        if (ln.e == 0) {
#pragma unroll
            for (int n = 0; n < NV; ++n) dst[n * ln.Ca] = Tm[n];
        }
        if (ln.e == ln.exta - 1) {
#pragma unroll
            for (int n = 0; n < NV; ++n) dst[(NV + n) * ln.Ca] = Tp[n];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// the fused, persistent stage kernel
// ------------------------------------------------------------------------------------------------
template <class C, int MODE>
__global__ void __launch_bounds__(C::THREADS, C::MINB) dg_stage_kernel(const __grid_constant__ DgStageArgs a) {
    constexpr int N = C::N, GX = C::GX, GY = C::GY;
    constexpr int NODES = C::NODES, PLANE = C::PLANE, L = C::L;
    constexpr int NV = DG_NV, NBUF = C::NBUF;
    constexpr int mode = MODE;   // one kernel per mode: the hot stage kernel carries no residual/trace-only code

    extern __shared__ __align__(16) double smem[];
    double *Qbuf = smem;                       // [NBUF][5][PLANE] nodal values of a brick (old, then updated)
    double *Rs = Qbuf + NBUF * NV * PLANE;     // [5][PLANE]       x (+ y) contribution to R
    double *Hs = Rs + NV * PLANE;              // [TSLOT]          neighbour bricks' traces, laid out like a brick's
                                               //                  own slot: [axis][side][5][Ca]; side 0 = T+ of the
                                               //                  brick below, side 1 = T- of the brick above
    double *Tms = Hs + C::TSLOT;               // [5][L]           T- of every line (right state of the line below)
    double *Fss = Tms + C::LINEBUF;            // [5][L]           F* at the + end of every line

    const int tid = threadIdx.x, l = tid;
    const int nbricks = a.nbx * a.nby * a.nbz;
    const bool readK = (mode == DG_MODE_STAGE) && (a.rkA != 0.0);
    constexpr bool want_halo = (mode != DG_MODE_TRACES);

    int brick = blockIdx.x;
    int buf = 0;
    if (NBUF == 2) {
        if (brick < nbricks) issue_q_loads<C>(a, brick, Qbuf, tid, readK);
        cp_async_commit();
    }
    for (; brick < nbricks; brick += gridDim.x) {
        const int bxi = brick % a.nbx, byi = (brick / a.nbx) % a.nby, bzi = brick / (a.nbx * a.nby);
        // ---------------- P0: this brick's neighbour traces and the next brick's Q go out ---------------
        double *Qs;
        if (NBUF == 2) {
            if (want_halo) issue_halo_loads<C>(a, bxi, byi, bzi, Hs, tid);
            cp_async_commit();
            const int next = brick + gridDim.x;
            if (next < nbricks) {
                issue_q_loads<C>(a, next, Qbuf + (buf ^ 1) * NV * PLANE, tid, readK);
                if (want_halo) prefetch_halo<C>(a, next, tid);
            }
            cp_async_commit();
            cp_async_wait<2>();                    // this brick's Q (asked for one brick ago) has landed
            Qs = Qbuf + buf * NV * PLANE;
            buf ^= 1;
        } else {
            issue_q_loads<C>(a, brick, Qbuf, tid, readK);
            cp_async_commit();
            if (want_halo) issue_halo_loads<C>(a, bxi, byi, bzi, Hs, tid);
            cp_async_commit();
            cp_async_wait<1>();
            Qs = Qbuf;
        }
        __syncthreads();

        const int ext0 = min(C::BX, a.nx - bxi * C::BX);   // elements of this brick per axis (ragged last brick)
        const int ext1 = min(C::BY, a.ny - byi * C::BY);
        const int ext2 = min(C::BZ, a.nz - bzi * C::BZ);
        const size_t qbase = (size_t)brick * C::SLOT;
        double *Tbrick = a.Tnew + (size_t)brick * C::TSLOT;

        if (mode != DG_MODE_TRACES) {
            double V[NV][N];
#pragma unroll 1
            for (int ax = 0; ax < 3; ++ax) {
                const Line ln = make_line<C>(ax, l, ext0, ext1, ext2);
                // momentum slots rotated so that slot 1 is the component along this axis
                const int m1 = 1 + ax, m2 = (ax == 2) ? 1 : 2 + ax, m3 = (ax == 0) ? 3 : ax;
                const int po1 = m1 * PLANE, po2 = m2 * PLANE, po3 = m3 * PLANE;
                double Tp[NV], Tm[NV];
                // ------------- PA: flux, sum-factorised derivative, traces ---------------------------
                if (ln.active) {
#pragma unroll
                    for (int n = 0; n < NV; ++n) {
                        Tp[n] = 0.0;
                        Tm[n] = 0.0;
#pragma unroll
                        for (int i = 0; i < N; ++i) V[n][i] = 0.0;
                    }
                    const double *Q0p = Qs + ln.base;
#pragma unroll
                    for (int q = 0; q < N; ++q) {
                        double Qn[NV], F[NV], vel, pres, rinv;
                        const double *Qq = Q0p + q * ln.stride;
                        Qn[0] = Qq[0];
                        Qn[1] = Qq[po1];
                        Qn[2] = Qq[po2];
                        Qn[3] = Qq[po3];
                        Qn[4] = Qq[4 * PLANE];
                        euler_flux_normal(Qn, a.gm1, F, vel, pres, rinv);
                        const double *Dq = a.ops.Dg[ax][q];
                        const double lpq = a.ops.lp[q], lmq = a.ops.lm[q];
#pragma unroll
                        for (int n = 0; n < NV; ++n) {
#pragma unroll
                            for (int i = 0; i < N; ++i) V[n][i] = fma(Dq[i], F[n], V[n][i]);
                            Tp[n] = fma(lpq, Qn[n], Tp[n]);
                            Tm[n] = fma(lmq, Qn[n], Tm[n]);
                        }
                    }
                    if (ln.multi) {
#pragma unroll
                        for (int n = 0; n < NV; ++n) Tms[n * L + l] = Tm[n];
                    }
                }
                if (ax == 0) {
                    cp_async_wait<(NBUF == 2) ? 1 : 0>();   // the neighbour traces have landed
                    __syncthreads();
                } else if (ln.multi) {
                    __syncthreads();
                }

                // ------------- PB: interface fluxes ----------------------------------------------------
                double Fp[NV], Fm[NV];
                if (ln.active) {
                    double Qown[NV];
#pragma unroll
                    for (int n = 0; n < NV; ++n) Qown[n] = Tp[n];
#pragma unroll 1
                    for (int s = 0; s < 2; ++s) {
                        // s = 0: + face (own state is the left one); s = 1: - face, only for the lines that
                        // start on the brick boundary (own state is the right one)
                        double Qo[NV], Fs[NV];
                        const double *src;
                        int sstride;
                        if (s == 0 && ln.multi && ln.e + 1 < ln.exta) {
                            src = Tms + l + ln.Ca;        // T- of the next element of this brick (rotated slots)
                            sstride = L;
                            Qo[1] = src[1 * sstride];
                            Qo[2] = src[2 * sstride];
                            Qo[3] = src[3 * sstride];
                        } else {
                            src = Hs + ln.tbase + ((s == 0) ? NV * ln.Ca : 0) + ln.c;
                            sstride = ln.Ca;
                            Qo[1] = src[m1 * sstride];
                            Qo[2] = src[m2 * sstride];
                            Qo[3] = src[m3 * sstride];
                        }
                        Qo[0] = src[0];
                        Qo[4] = src[4 * sstride];
                        lax_friedrichs(Qown, Qo, (s == 0) ? 1.0 : -1.0, a.gamma, a.gm1, Fs);
                        if (s == 0) {
#pragma unroll
                            for (int n = 0; n < NV; ++n) {
                                Fp[n] = Fs[n];
                                Qown[n] = Tm[n];
                            }
                            if (ln.e != 0) break;
                        } else {
#pragma unroll
                            for (int n = 0; n < NV; ++n) Fm[n] = Fs[n];
                        }
                    }
                    if (ln.multi) {
#pragma unroll
                        for (int n = 0; n < NV; ++n) Fss[n * L + l] = Fp[n];
                    }
                }
                if (ln.multi) __syncthreads();

                // ------------- PC: lift (2/h and 1/w folded into the tables) ---------------------------
                if (ln.active) {
                    if (ln.multi && ln.e > 0) {
#pragma unroll
                        for (int n = 0; n < NV; ++n) Fm[n] = Fss[n * L + l - ln.Ca];
                    }
                    // K of this z line: asked for now (an L2 hit: prefetched a brick ago), used after the lift
                    const size_t g0 = qbase + (size_t)(ln.e * N) * (GY * GX) + ln.c;   // node q=0 of a z-line, n=0
                    double Kold[NV][N];
                    if (ax == 2 && readK) {
#pragma unroll
                        for (int n = 0; n < NV; ++n)
#pragma unroll
                            for (int q = 0; q < N; ++q)
                                Kold[n][q] = __ldcs(a.K + g0 + (size_t)n * NODES + (size_t)q * (GY * GX));
                    }
                    const double *lpg = a.ops.lpg[ax], *lmg = a.ops.lmg[ax];
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        const double cp = lpg[i], cm = lmg[i];
#pragma unroll
                        for (int n = 0; n < NV; ++n) V[n][i] = fma(cm, Fm[n], fma(-cp, Fp[n], V[n][i]));
                    }
                    if (ax < 2) {
                        // x: R = r_x;  y: R += r_y   (slot s holds variable 0, m1, m2, m3, 4)
                        double *R0p = Rs + ln.base;
#pragma unroll
                        for (int i = 0; i < N; ++i) {
                            double *Rq = R0p + i * ln.stride;
                            if (ax == 0) {
                                Rq[0] = V[0][i];
                                Rq[po1] = V[1][i];
                                Rq[po2] = V[2][i];
                                Rq[po3] = V[3][i];
                                Rq[4 * PLANE] = V[4][i];
                            } else {
                                Rq[0] += V[0][i];
                                Rq[po1] += V[1][i];
                                Rq[po2] += V[2][i];
                                Rq[po3] += V[3][i];
                                Rq[4 * PLANE] += V[4][i];
                            }
                        }
                    } else {
                        // z: slots (0,1,2,3,4) hold variables (0,3,1,2,4)
                        constexpr int var_of_slot[NV] = {0, 3, 1, 2, 4};
                        if (mode == DG_MODE_RESIDUAL) {
#pragma unroll
                            for (int s = 0; s < NV; ++s)
#pragma unroll
                                for (int q = 0; q < N; ++q) {
                                    const int n = var_of_slot[s];
                                    a.Rout[g0 + (size_t)n * NODES + (size_t)q * (GY * GX)] =
                                        Rs[n * PLANE + ln.base + q * ln.stride] + V[s][q];
                                }
                        } else {
                            // ------------- PD: LSERK45 stage, write back, z traces of the updated Q -----
                            const double A = a.rkA, B = a.rkB, dt = a.dt;
                            double *dst = Tbrick + ln.tbase + ln.c;
#pragma unroll
                            for (int s = 0; s < NV; ++s) {
                                const int n = var_of_slot[s];
                                double tp = 0.0, tm = 0.0;
#pragma unroll
                                for (int q = 0; q < N; ++q) {
                                    const int sa = n * PLANE + ln.base + q * ln.stride;
                                    const size_t go = g0 + (size_t)n * NODES + (size_t)q * (GY * GX);
                                    const double R = Rs[sa] + V[s][q];
                                    const double Kn = readK ? fma(A, Kold[n][q], dt * R) : dt * R;
                                    const double Qn = fma(B, Kn, Qs[sa]);
                                    a.K[go] = Kn;
                                    a.Q[go] = Qn;
                                    Qs[sa] = Qn;
                                    tp = fma(a.ops.lp[q], Qn, tp);
                                    tm = fma(a.ops.lm[q], Qn, tm);
                                }
                                if (ln.e == 0) dst[n * C::CZ] = tm;
                                if (ln.e == ln.exta - 1) dst[(NV + n) * C::CZ] = tp;
                            }
                        }
                    }
                }
                if (ax < 2) __syncthreads();
            }
        }

        // ---------------- PE: traces of the updated Q on the brick boundary (z came from registers) ----
        if (mode != DG_MODE_RESIDUAL) {
            if (mode == DG_MODE_STAGE) __syncthreads();
            const int nax = (mode == DG_MODE_TRACES) ? 3 : 2;
#pragma unroll 1
            for (int ax = 0; ax < nax; ++ax) boundary_traces<C>(make_line<C>(ax, l, ext0, ext1, ext2), Qs, Tbrick, a);
        }
        __syncthreads();   // everyone is done with this brick's buffers before they are refilled
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
cudaError_t prepare(int *blocks_per_sm) {
    cudaError_t err = cudaFuncSetAttribute(dg_stage_kernel<C, DG_MODE_STAGE>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_stage_kernel<C, DG_MODE_RESIDUAL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   C::SMEM_BYTES);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_stage_kernel<C, DG_MODE_TRACES>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, dg_stage_kernel<C, DG_MODE_STAGE>,
                                                         C::THREADS, C::SMEM_BYTES);
}

template <class C>
cudaError_t launch_stage(const DgStageArgs &a, cudaStream_t s) {
    if (a.grid <= 0) return cudaErrorInvalidConfiguration;
    if (a.mode == DG_MODE_STAGE)
        dg_stage_kernel<C, DG_MODE_STAGE><<<(unsigned)a.grid, C::THREADS, C::SMEM_BYTES, s>>>(a);
    else if (a.mode == DG_MODE_RESIDUAL)
        dg_stage_kernel<C, DG_MODE_RESIDUAL><<<(unsigned)a.grid, C::THREADS, C::SMEM_BYTES, s>>>(a);
    else
        dg_stage_kernel<C, DG_MODE_TRACES><<<(unsigned)a.grid, C::THREADS, C::SMEM_BYTES, s>>>(a);
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
                         &prepare<C>, &launch_stage<C>, &launch_layout<C>, &launch_wavespeed<C>};
}

// Brick shapes per N (default first): Cfg<N, BX, BY, BZ, min blocks per SM, Q buffers>.
// DESIGN.md "brick shapes" explains the choice.
#if DG_N == 2
using V0 = Cfg<2, 4, 4, 4, 2, 2>;
using V1 = Cfg<2, 4, 4, 4, 3, 1>;
using V2 = Cfg<2, 4, 4, 2, 4, 2>;
using V3 = Cfg<2, 2, 2, 2, 4, 1>;
#elif DG_N == 3
using V0 = Cfg<3, 4, 4, 2, 2, 2>;
using V1 = Cfg<3, 4, 4, 2, 2, 1>;
using V2 = Cfg<3, 2, 2, 2, 4, 2>;
using V3 = Cfg<3, 1, 1, 1, 8, 1>;
#elif DG_N == 4
using V0 = Cfg<4, 2, 2, 2, 2, 2>;
using V1 = Cfg<4, 2, 2, 2, 3, 1>;
using V2 = Cfg<4, 2, 2, 1, 4, 2>;
using V3 = Cfg<4, 1, 1, 1, 8, 1>;
#elif DG_N == 5
using V0 = Cfg<5, 1, 2, 2, 2, 2>;
using V1 = Cfg<5, 1, 2, 2, 3, 1>;
using V2 = Cfg<5, 2, 2, 2, 1, 2>;
using V3 = Cfg<5, 1, 1, 1, 6, 2>;
#elif DG_N == 6
using V0 = Cfg<6, 1, 2, 2, 1, 2>;
using V1 = Cfg<6, 1, 2, 2, 1, 1>;
using V2 = Cfg<6, 1, 1, 2, 2, 2>;
using V3 = Cfg<6, 1, 1, 1, 5, 2>;
#elif DG_N == 7
using V0 = Cfg<7, 1, 1, 2, 2, 2>;
using V1 = Cfg<7, 1, 1, 2, 2, 1>;
using V2 = Cfg<7, 1, 2, 2, 1, 2>;
using V3 = Cfg<7, 1, 1, 1, 4, 2>;
#elif DG_N == 8
using V0 = Cfg<8, 1, 1, 2, 1, 2>;
using V1 = Cfg<8, 1, 1, 2, 2, 1>;
using V2 = Cfg<8, 1, 1, 1, 3, 2>;
using V3 = Cfg<8, 1, 1, 1, 4, 1>;
#else
#error "DG_N must be 2..8"
#endif

const DgKernelTable k_tables[] = {make_table<V0>(), make_table<V1>(), make_table<V2>(), make_table<V3>()};

}  // namespace

#define DG_CAT2(a, b) a##b
#define DG_CAT(a, b) DG_CAT2(a, b)
const DgKernelTable *DG_CAT(dg_variants_N, DG_N)(int *count) {
    *count = (int)(sizeof(k_tables) / sizeof(k_tables[0]));
    return k_tables;
}
