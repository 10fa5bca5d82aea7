// dg_kernels.cu -- CUDA kernels of the DG Euler time step for one N = p+1 (compile with -DDG_N=<N>,
// -gencode arch=compute_100a,code=sm_100a).  Hand-written for B200; fp64 throughout.
//
// The fused stage kernel (v4): ONE thread block per "brick" of BX x BY x BZ elements, one thread per node
// LINE, every shared-memory stride a compile-time constant.  Per brick, in ONE sweep over HBM:
//   P0  cp.async (no registers) of the brick's Q and K (5 x nodes each, separate groups) into shared memory
//   then, for the axes x, y, z in turn (three instances of one template):
//   PH  the neighbour bricks' face traces this line touches go straight from HBM/L2 into registers
//   PT  the line's N nodal values into registers (RELOAD variants: read again later instead) and the two
//       face traces T+- = sum_q l_q(+-1) Q_q
//   PB  local Lax-Friedrichs interface flux, doubled, at the + end of the line, and at the
//       - end of the lines that start on the brick boundary (faces inside a brick: once, handed over
//       through shared memory; cluster variants: also across the blocks of a cluster)
//   PC  lift with 2/h, 1/2 and dt folded into the tables starts the accumulators:
//       r_i = sum_q Dhat_iq F_q - (l_i(+1) F*_+ - l_i(-1) F*_-) (2/h_a)/w_i       (eq (5) 3rd and 2nd term)
//   PA  pointwise Euler flux (eq (2)-(3)) at the line's N nodes and the sum-factorised
//       derivative (the contraction of listing lines 220-237), all in registers
//   PD  LSERK45 accumulated in place on the staged K:  x: K = A K + r_x,  y: K += r_y,
//       z: K += r_z, Q += B K, both written straight to HBM from the z lines (coalesced, streaming);
//       or R itself in residual mode.  Before the z pass: L2 prefetch of the follow-on brick's data.
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
// Shared-memory layout of a brick: [5][GZ] planes of pitch PP doubles, rows of pitch P doubles inside a
// plane, and, per axis, the order in which a warp's lanes walk the node lines (ORD):
//   0: t1 fastest, then t2, then the element e along the axis      1: t2, t1, e
//   2: t1, e, t2                                                   3: t2, e, t1
//   4: e, t1, t2                                                   5: e, t2, t1
// (t1,t2) = (gy,gz) for x lines, (gx,gz) for y lines, (gx,gy) for z lines.  P, PP and the orders are picked
// per brick shape so that the 16 lanes of a half-warp hit 16 different 8-byte bank pairs in all three
// passes (0 = dense).  z lines keep t1 = gx fastest: their lanes also
// address HBM.
// CLX x CLY x CLZ > 1: the blocks of that many neighbouring bricks form a thread-block CLUSTER and hand the traces
// of the faces they share to each other through distributed shared memory instead of the HBM trace buffer.
template <int N_, int BX_, int BY_, int BZ_, int MINB_, int RELOAD_ = 0, int P_ = 0, int PP_ = 0, int OX_ = 0,
          int OY_ = 0, int OZ_ = 0, int CLX_ = 1, int CLY_ = 1, int CLZ_ = 1>
struct Cfg {
    static constexpr int CLX = CLX_, CLY = CLY_, CLZ = CLZ_, CLUSTER = CLX_ * CLY_ * CLZ_;
    static constexpr int N = N_, BX = BX_, BY = BY_, BZ = BZ_, MINB = MINB_;
    // RELOAD = 1: the volume term reads the line's Q from shared memory a second time instead of keeping
    // it in 10 N registers across the interface fluxes (fewer registers, more blocks per SM, 15 more
    // shared loads per node)
    static constexpr bool RELOAD = RELOAD_ != 0;
    static constexpr int GX = BX * N, GY = BY * N, GZ = BZ * N;   // nodes of the brick per axis
    static constexpr int NODES = GX * GY * GZ;
    static constexpr int SLOT = DG_NV * NODES;                     // doubles per brick in Q, K, R (HBM, dense)
    static constexpr int P = P_ ? P_ : GX;                         // shared-memory row pitch
    static constexpr int PP = PP_ ? PP_ : GY * P;                  // shared-memory plane pitch
    static constexpr int PLANE = GZ * PP;                          // shared doubles per variable
    static constexpr int OX = OX_, OY = OY_, OZ = OZ_;
    static constexpr int L = NODES / N;                            // node lines per axis = threads that work
    static constexpr int THREADS = (L + 31) / 32 * 32;
    static constexpr int CX = GY * GZ, CY = GX * GZ, CZ = GX * GY; // face nodes of a brick side per axis
    static constexpr int TSLOT = 2 * DG_NV * (CX + CY + CZ);       // trace doubles per brick
    static constexpr bool MULTI = (BX > 1) || (BY > 1) || (BZ > 1);
    static constexpr int LINEBUF = MULTI ? DG_NV * L : 0;          // T- / F* hand-over between elements of a brick
    static constexpr int EXFACE = (CLX > 1 ? CX : 0) > (CLY > 1 ? CY : 0)
                                      ? ((CLX > 1 ? CX : 0) > (CLZ > 1 ? CZ : 0) ? (CLX > 1 ? CX : 0) : (CLZ > 1 ? CZ : 0))
                                      : ((CLY > 1 ? CY : 0) > (CLZ > 1 ? CZ : 0) ? (CLY > 1 ? CY : 0) : (CLZ > 1 ? CZ : 0));
    static constexpr int EXBUF = 2 * DG_NV * EXFACE;               // traces exported to the cluster neighbours
    static constexpr int SMEM_DOUBLES = 2 * DG_NV * PLANE + 2 * LINEBUF + EXBUF;
    static constexpr int SMEM_BYTES = SMEM_DOUBLES * 8;
    static_assert(P >= GX && PP >= GY * P, "pitches too small");
    static_assert(OZ == 0 || OZ == 2, "z lines must keep gx fastest across lanes");
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
// Ask L2 to fetch [ptr, ptr + bytes) (rounded out to 16-byte granules): one instruction per block of data.
__device__ __forceinline__ void l2_prefetch(const void *ptr, unsigned bytes) {
    const uintptr_t lo = (uintptr_t)ptr & ~(uintptr_t)15;
    const uintptr_t hi = ((uintptr_t)ptr + bytes + 15) & ~(uintptr_t)15;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(lo), "r"((unsigned)(hi - lo)) : "memory");
}

// Compiler-level fence on memory operations: bounds how far loads are hoisted (register pressure).
__device__ __forceinline__ void sched_fence() { asm volatile("" ::: "memory"); }

// Thread-block cluster primitives (split barrier; distributed shared memory loads).
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ unsigned map_to_rank(const void *smem_ptr, unsigned rank) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(smem_ptr);
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
__device__ __forceinline__ double ld_cluster(unsigned addr) {
    double v;
    asm volatile("ld.shared::cluster.f64 %0, [%1];" : "=d"(v) : "r"(addr) : "memory");
    return v;
}

// Euler flux along the face/line normal, eq (2)-(3) (listing lines 186-217), for a state
// whose momentum components have been ROTATED so that slot 1 is the normal one:
//   slots = (rho, rho u_a, rho u_b, rho u_c, rho E),  (a,b,c) = (x,y,z), (y,z,x) or (z,x,y).
// One copy of the code then serves the three axes with no run-time selection.
__device__ __forceinline__ void euler_flux_normal(const double (&Q)[DG_NV], double gm1, double (&F)[DG_NV],
                                                  double &vel, double &pres, double &oneOrho) {
    oneOrho = rcp_pos(Q[0]);
    vel = Q[1] * oneOrho;
    // 1/2 rho |u|^2 = 1/2 |rho u|^2 / rho
    const double m2 = fma(Q[3], Q[3], fma(Q[2], Q[2], Q[1] * Q[1]));
    pres = gm1 * fma(-0.5, m2 * oneOrho, Q[4]);
    F[0] = Q[1];                                    // rho u_a
    F[1] = fma(Q[1], vel, pres);
    F[2] = Q[2] * vel;
    F[3] = Q[3] * vel;
    F[4] = (Q[4] + pres) * vel;
}

// Local Lax-Friedrichs flux (reading R3), rotated slots as above, returned DOUBLED
// (the factor 1/2 is folded into the lift tables):
//   2 F* = F(QL) + F(QR) - lam (QR - QL),  lam = max(|u_a^L| + c_L, |u_a^R| + c_R)
// written for (own, other) with sgn = +1 when own is the left state, -1 when it is the right one.
__device__ __forceinline__ void lax_friedrichs2(const double (&Qown)[DG_NV], const double (&Qoth)[DG_NV], double sgn,
                                                double gamma, double gm1, double (&Fs)[DG_NV]) {
    double Fa[DG_NV], Fb[DG_NV], ua, ub, pa, pb, ra, rb;
    euler_flux_normal(Qown, gm1, Fa, ua, pa, ra);
    euler_flux_normal(Qoth, gm1, Fb, ub, pb, rb);
    const double lama = fabs(ua) + sqrt_pos(gamma * pa * ra);
    const double lamb = fabs(ub) + sqrt_pos(gamma * pb * rb);
    const double sl = sgn * ((lama > lamb) ? lama : lamb);
#pragma unroll
    for (int n = 0; n < DG_NV; ++n) Fs[n] = fma(-sl, Qoth[n] - Qown[n], Fa[n] + Fb[n]);
}

// ------------------------------------------------------------------------------------------------
// per-axis compile-time traits and the (brick-independent) geometry of a thread's node line
//   line l = e * Ca + c,  e = element along the axis, c = face node = t2 * T1 + t1
//   axis x: (t1,t2) = (gy,gz);  y: (gx,gz);  z: (gx,gy)
// ------------------------------------------------------------------------------------------------
template <class C, int AX>
struct Axis {
    static constexpr int S = (AX == 0) ? 1 : (AX == 1) ? C::P : C::PP;                 // shared stride along the line
    static constexpr int Ca = (AX == 0) ? C::CX : (AX == 1) ? C::CY : C::CZ;           // face nodes of a brick side
    static constexpr int T1 = (AX == 0) ? C::GY : C::GX;
    static constexpr int T2 = (AX == 2) ? C::GY : C::GZ;
    static constexpr int ORD = (AX == 0) ? C::OX : (AX == 1) ? C::OY : C::OZ;
    static constexpr int B = (AX == 0) ? C::BX : (AX == 1) ? C::BY : C::BZ;            // elements along the axis
    static constexpr int TBASE = (AX == 0) ? 0 : (AX == 1) ? 2 * DG_NV * C::CX : 2 * DG_NV * (C::CX + C::CY);
    static constexpr bool MULTI = B > 1;
    static constexpr int CL = (AX == 0) ? C::CLX : (AX == 1) ? C::CLY : C::CLZ;     // cluster blocks along the axis
    // momentum slots rotated so that slot 1 is the component along this axis: slot s holds variable VAR[s]
    static constexpr int M1 = 1 + AX, M2 = (AX == 2) ? 1 : 2 + AX, M3 = (AX == 0) ? 3 : AX;
};
template <class C, int AX>
__device__ __forceinline__ constexpr int var_of_slot(int s) {
    return s == 0 ? 0 : s == 1 ? Axis<C, AX>::M1 : s == 2 ? Axis<C, AX>::M2 : s == 3 ? Axis<C, AX>::M3 : 4;
}

struct Geo {
    int base;   // shared-memory offset (doubles, inside one variable plane) of node 0 of the line
    int c;      // face-node index of the line on the brick side (lane order: this is how the traces are stored)
    int e;      // element along the axis
    int t1, t2; // transverse node indices
};

template <class C, int AX>
__device__ __forceinline__ Geo make_geo(int l) {
    using A = Axis<C, AX>;
    constexpr int N = C::N, T1 = A::T1, T2 = A::T2, B = A::B;
    Geo g;
    if (A::ORD == 0) {
        g.t1 = l % T1;
        g.t2 = (l / T1) % T2;
        g.e = l / (T1 * T2);
        g.c = g.t2 * T1 + g.t1;
    } else if (A::ORD == 1) {
        g.t2 = l % T2;
        g.t1 = (l / T2) % T1;
        g.e = l / (T1 * T2);
        g.c = g.t1 * T2 + g.t2;
    } else if (A::ORD == 2) {
        g.t1 = l % T1;
        g.e = (l / T1) % B;
        g.t2 = l / (T1 * B);
        g.c = g.t2 * T1 + g.t1;
    } else if (A::ORD == 3) {
        g.t2 = l % T2;
        g.e = (l / T2) % B;
        g.t1 = l / (T2 * B);
        g.c = g.t1 * T2 + g.t2;
    } else if (A::ORD == 4) {
        g.e = l % B;
        g.t1 = (l / B) % T1;
        g.t2 = l / (B * T1);
        g.c = g.t2 * T1 + g.t1;
    } else {
        g.e = l % B;
        g.t2 = (l / B) % T2;
        g.t1 = l / (B * T2);
        g.c = g.t1 * T2 + g.t2;
    }
    if (AX == 0) g.base = g.t2 * C::PP + g.t1 * C::P + g.e * N;
    else if (AX == 1) g.base = g.t2 * C::PP + g.e * N * C::P + g.t1;
    else g.base = g.e * N * C::PP + g.t2 * C::P + g.t1;
    return g;
}

// Is the line inside a ragged (last) brick of ext0 x ext1 x ext2 elements?
template <class C, int AX>
__device__ __forceinline__ bool line_inside(const Geo &g, int ext0, int ext1, int ext2) {
    const int lim1 = ((AX == 0) ? ext1 : ext0) * C::N, lim2 = ((AX == 2) ? ext1 : ext2) * C::N;
    const int exta = (AX == 0) ? ext0 : (AX == 1) ? ext1 : ext2;
    return g.t1 < lim1 && g.t2 < lim2 && g.e < exta;
}

// P0: enqueue the asynchronous copy of one dense HBM slot [5][GZ][GY][GX] into the pitched shared planes.
// Thread tid < L = BZ * GX * GY owns one node of a group of BZ consecutive z planes; the 5 N groups of the
// slot are then a fixed stride apart on both sides, so the whole copy is 5 N instructions per thread with
// immediate offsets (consecutive lanes read consecutive doubles of HBM).
template <class C>
__device__ __forceinline__ void stage_in(double *dst, const double *src, int tid) {
    if (tid < C::L) {
        const int pz = tid / (C::GX * C::GY), k = tid - pz * (C::GX * C::GY);
        const int gy = k / C::GX, gx = k - gy * C::GX;
        double *d = dst + pz * C::PP + gy * C::P + gx;
        const double *g = src + tid;
#pragma unroll
        for (int j = 0; j < DG_NV * C::N; ++j) cp_async8(d + j * (C::BZ * C::PP), g + j * C::L);
    }
}

// Trace block [5][Ca] a brick needs for (axis, side): side 0 = T+ of the brick below (stored as that brick's
// side 1), side 1 = T- of the brick above (its side 0).  Periodic in every direction.
template <class C, int AX>
__device__ __forceinline__ const double *halo_source(const DgStageArgs &a, int bx, int by, int bz, int side) {
    using A = Axis<C, AX>;
    if (AX == 0) bx = (side == 0) ? ((bx == 0) ? a.nbx - 1 : bx - 1) : ((bx + 1 == a.nbx) ? 0 : bx + 1);
    else if (AX == 1) by = (side == 0) ? ((by == 0) ? a.nby - 1 : by - 1) : ((by + 1 == a.nby) ? 0 : by + 1);
    else bz = (side == 0) ? ((bz == 0) ? a.nbz - 1 : bz - 1) : ((bz + 1 == a.nbz) ? 0 : bz + 1);
    const size_t nbr = (size_t)bx + (size_t)a.nbx * ((size_t)by + (size_t)a.nby * bz);
    return a.Told + nbr * C::TSLOT + A::TBASE + (side == 0 ? DG_NV * A::Ca : 0);
}

// L2 prefetch of everything the block's NEXT brick will read: 8 threads, one instruction each.
template <class C>
__device__ __forceinline__ void prefetch_brick(const DgStageArgs &a, int brick, int tid, bool want_k, bool want_halo) {
    if (tid == 0) l2_prefetch(a.Q + (size_t)brick * C::SLOT, C::SLOT * 8);
    if (tid == 1 && want_k) l2_prefetch(a.K + (size_t)brick * C::SLOT, C::SLOT * 8);
    if (tid >= 2 && tid < 8 && want_halo) {
        const int bx = brick % a.nbx, by = (brick / a.nbx) % a.nby, bz = brick / (a.nbx * a.nby);
        const int side = tid & 1;
        if (tid < 4) l2_prefetch(halo_source<C, 0>(a, bx, by, bz, side), DG_NV * C::CX * 8);
        else if (tid < 6) l2_prefetch(halo_source<C, 1>(a, bx, by, bz, side), DG_NV * C::CY * 8);
        else l2_prefetch(halo_source<C, 2>(a, bx, by, bz, side), DG_NV * C::CZ * 8);
    }
}

// PE for one axis: traces of the (updated) Q in shared memory on the brick boundary -> Tnew.
template <class C, int AX>
__device__ __forceinline__ void boundary_traces(const Geo &g, bool act, int exta, const double *Qs, double *Tbrick,
                                                const DgStageArgs &a, bool wlo = true, bool whi = true) {
    using A = Axis<C, AX>;
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE;
    // wlo / whi: does the low / high face of the brick go through HBM (false: a cluster neighbour takes it)
    const bool first = g.e == 0 && wlo, last = g.e == exta - 1 && whi;
    if (!act || !(first || last)) return;
    double *dst = Tbrick + A::TBASE + g.c;
    const double *Q0 = Qs + g.base;
    if (first && last) {
        double Tp[NV], Tm[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) Tp[n] = Tm[n] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q)
#pragma unroll
            for (int n = 0; n < NV; ++n) {
                const double Qv = Q0[n * PLANE + q * A::S];
                Tp[n] = fma(a.ops.lp[q], Qv, Tp[n]);
                Tm[n] = fma(a.ops.lm[q], Qv, Tm[n]);
            }
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            dst[n * A::Ca] = Tm[n];
            dst[(NV + n) * A::Ca] = Tp[n];
        }
    } else {
        // one end only: the interpolation weights of the - end are those of the + end reversed
        double T[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) T[n] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q) {
            const double w = first ? a.ops.lm[q] : a.ops.lp[q];
#pragma unroll
            for (int n = 0; n < NV; ++n) T[n] = fma(w, Q0[n * PLANE + q * A::S], T[n]);
        }
        if (!first) dst += NV * A::Ca;
#pragma unroll
        for (int n = 0; n < NV; ++n) dst[n * A::Ca] = T[n];
    }
}

// ------------------------------------------------------------------------------------------------
// one axis of the residual for one brick
// ------------------------------------------------------------------------------------------------
// PH: the neighbour bricks' traces this line touches, momentum slots rotated, HBM/L2 -> registers.
template <class C, int AX>
__device__ __forceinline__ void load_halo(const Geo &g, bool act, int exta, const double *halo_lo,
                                          const double *halo_hi, bool ilo, bool ihi, double (&Hlo)[DG_NV],
                                          double (&Hhi)[DG_NV]) {
    constexpr int Ca = Axis<C, AX>::Ca;
    if (act && g.e == 0 && !ilo) {
#pragma unroll
        for (int s = 0; s < DG_NV; ++s) Hlo[s] = __ldg(halo_lo + var_of_slot<C, AX>(s) * Ca + g.c);
    }
    if (act && g.e == exta - 1 && !ihi) {
#pragma unroll
        for (int s = 0; s < DG_NV; ++s) Hhi[s] = __ldg(halo_hi + var_of_slot<C, AX>(s) * Ca + g.c);
    }
}

// PA..PD for one axis.  Order chosen for register pressure: the line's Q goes into registers once; the
// face traces and the two interface fluxes come first (no accumulators alive yet); the accumulators then
// START from the lift term and the volume term is added node by node.
//   r_i = sum_q Dhat_iq F_q - (l_i(+1) F*_+ - l_i(-1) F*_-) (2/h_a)/w_i
// Cluster variants (A::CL > 1): `ilo` / `ihi` say that the low / high face of the brick is shared with the
// cluster block of rank `rlo` / `rhi`; the traces on those faces are exported to Ex in this block's shared
// memory and the neighbour's are read from ITS Ex.  One cluster barrier between export and import; the
// barrier that protects Ex against the next export is split (arrive after the import, wait before the next
// export or the end of the kernel: PENDING says that such a wait is still owed on entry).
template <class C, int AX, int MODE, bool PENDING>
__device__ __forceinline__ void axis_pass(const DgStageArgs &a, const Geo &g, int l, bool act, int exta,
                                          const double *halo_lo, const double *halo_hi, double *Qs, double *Ks,
                                          double *Tms, double *Fss, double *Ex, bool readK, size_t qbase,
                                          double *Tbrick, bool ilo, bool ihi, unsigned rlo, unsigned rhi) {
    using A = Axis<C, AX>;
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE, L = C::L, S = A::S, Ca = A::Ca;
    const bool first = g.e == 0, last = g.e == exta - 1;
    const int lb = g.e * Ca + g.c;   // slot of this line in the hand-over buffers
    double Hlo[NV], Hhi[NV];
    load_halo<C, AX>(g, act, exta, halo_lo, halo_hi, ilo, ihi, Hlo, Hhi);

    double QL[C::RELOAD ? 1 : NV][C::RELOAD ? 1 : N], Tp[NV], Tm[NV];
    if (act) {
        // ------------- the line's nodal values (slot s holds variable var_of_slot(s)) and its traces ----
        const double *Q0 = Qs + g.base;
#pragma unroll
        for (int s = 0; s < NV; ++s) {
            Tp[s] = 0.0;
            Tm[s] = 0.0;
#pragma unroll
            for (int q = 0; q < N; ++q) {
                const double Qv = Q0[var_of_slot<C, AX>(s) * PLANE + q * S];
                if (!C::RELOAD) QL[s][q] = Qv;
                Tp[s] = fma(a.ops.lp[q], Qv, Tp[s]);
                Tm[s] = fma(a.ops.lm[q], Qv, Tm[s]);
            }
        }
        if (A::MULTI) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Tms[n * L + lb] = Tm[n];
        }
    }
    if (A::CL > 1) {
        if (PENDING) cluster_wait();   // the neighbours are done with the previous axis' exports
        if (act && first && ilo) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Ex[n * Ca + g.c] = Tm[n];
        }
        if (act && last && ihi) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Ex[(NV + n) * Ca + g.c] = Tp[n];
        }
        cluster_arrive();              // (a cluster barrier is also a block barrier: covers Tms)
        cluster_wait();
    } else if (A::MULTI) {
        __syncthreads();
    }

    // ------------- PB: interface fluxes ----------------------------------------------------------------
    double Fp[NV], Fm[NV];
    if (act) {
        if (A::MULTI && !last) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Hhi[n] = Tms[n * L + lb + Ca];   // T- of the next element of this brick
        } else if (A::CL > 1 && ihi) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Hhi[n] = ld_cluster(map_to_rank(Ex + n * Ca + g.c, rhi));        // its T-
        }
        if (A::CL > 1 && first && ilo) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Hlo[n] = ld_cluster(map_to_rank(Ex + (NV + n) * Ca + g.c, rlo));  // its T+
        }
        lax_friedrichs2(Tp, Hhi, 1.0, a.gamma, a.gm1, Fp);
        if (A::MULTI) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Fss[n * L + lb] = Fp[n];
        }
        if (first) lax_friedrichs2(Tm, Hlo, -1.0, a.gamma, a.gm1, Fm);
    }
    if (A::CL > 1) cluster_arrive();   // done reading the neighbours' exports (waited for before Ex is reused)
    if (A::MULTI) __syncthreads();

    double V[NV][N];
    if (act) {
        if (A::MULTI && !first) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Fm[n] = Fss[n * L + lb - Ca];
        }
        // ------------- PC: lift (2/h and 1/w folded into the tables) starts the accumulators -----------
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const double cp = a.ops.lpg[AX][i], cm = a.ops.lmg[AX][i];
#pragma unroll
            for (int n = 0; n < NV; ++n) V[n][i] = fma(cm, Fm[n], -cp * Fp[n]);
        }
        // ------------- PA: pointwise flux and sum-factorised derivative --------------------------------
#pragma unroll
        for (int q = 0; q < N; ++q) {
            double Qn[NV], F[NV], vel, pres, rinv;
#pragma unroll
            for (int s = 0; s < NV; ++s)
                Qn[s] = C::RELOAD ? Qs[g.base + var_of_slot<C, AX>(s) * PLANE + q * S] : QL[C::RELOAD ? 0 : s][C::RELOAD ? 0 : q];
            euler_flux_normal(Qn, a.gm1, F, vel, pres, rinv);
#pragma unroll
            for (int n = 0; n < NV; ++n)
#pragma unroll
                for (int i = 0; i < N; ++i) V[n][i] = fma(a.ops.Dg[AX][q][i], F[n], V[n][i]);
        }
    }
    if (AX == 0) {
        cp_async_wait<0>();            // the staged K (its own cp.async group) has landed
        if (readK) __syncthreads();
    }
    if (act) {
        // ------------- PD: Runge-Kutta accumulation on the staged K ------------------------------------
        double *K0 = Ks + g.base;
        if (AX == 0) {
            if (readK) {
                const double rkA = a.rkA;
#pragma unroll
                for (int s = 0; s < NV; ++s)
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        double *p = K0 + var_of_slot<C, AX>(s) * PLANE + i * S;
                        *p = fma(rkA, *p, V[s][i]);
                    }
            } else {
#pragma unroll
                for (int s = 0; s < NV; ++s)
#pragma unroll
                    for (int i = 0; i < N; ++i) K0[var_of_slot<C, AX>(s) * PLANE + i * S] = V[s][i];
            }
        } else if (AX == 1) {
#pragma unroll
            for (int s = 0; s < NV; ++s)
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    double *p = K0 + var_of_slot<C, AX>(s) * PLANE + i * S;
                    *p += V[s][i];
                }
        } else {
            // z lines: consecutive threads hold consecutive (gx, gy), so HBM accesses coalesce
            const size_t g0 = qbase + (size_t)(g.e * N) * (C::GY * C::GX) + g.t2 * C::GX + g.t1;   // node 0, variable 0
            if (MODE == DG_MODE_RESIDUAL) {
#pragma unroll
                for (int s = 0; s < NV; ++s)
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        const int n = var_of_slot<C, AX>(s);
                        a.Rout[g0 + (size_t)n * C::NODES + (size_t)i * (C::GY * C::GX)] =
                            K0[n * PLANE + i * S] + V[s][i];
                    }
            } else {
                const double rkB = a.rkB;
                double *Q0w = Qs + g.base;
                double *dst = Tbrick + A::TBASE + g.c;
#pragma unroll
                for (int s = 0; s < NV; ++s) {
                    const int n = var_of_slot<C, AX>(s);
                    double Qn[N];
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        const size_t go = g0 + (size_t)n * C::NODES + (size_t)i * (C::GY * C::GX);
                        const double Kn = K0[n * PLANE + i * S] + V[s][i];
                        const double Qold = C::RELOAD ? Q0w[n * PLANE + i * S] : QL[C::RELOAD ? 0 : s][C::RELOAD ? 0 : i];
                        Qn[i] = fma(rkB, Kn, Qold);
                        __stcs(a.K + go, Kn);   // streaming: written once, not read again in this stage
                        __stcs(a.Q + go, Qn[i]);
                        Q0w[n * PLANE + i * S] = Qn[i];
                    }
                    // PE for the z faces: traces of the updated Q, only at the ends that lie on the brick boundary
                    if (first && !ilo) {
                        double tm = 0.0;
#pragma unroll
                        for (int i = 0; i < N; ++i) tm = fma(a.ops.lm[i], Qn[i], tm);
                        dst[n * Ca] = tm;
                    }
                    if (last && !ihi) {
                        double tp = 0.0;
#pragma unroll
                        for (int i = 0; i < N; ++i) tp = fma(a.ops.lp[i], Qn[i], tp);
                        dst[(NV + n) * Ca] = tp;
                    }
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// ------------------------------------------------------------------------------------------------
// the fused, persistent stage kernel
// ------------------------------------------------------------------------------------------------
template <class C, int MODE>
__global__ void __launch_bounds__(C::THREADS, C::MINB) dg_stage_kernel(const __grid_constant__ DgStageArgs a) {
    constexpr int NV = DG_NV, PLANE = C::PLANE, L = C::L;
    constexpr bool EXCH = (C::CLUSTER > 1) && (MODE != DG_MODE_TRACES);   // do cluster neighbours trade traces?
    extern __shared__ __align__(16) double smem[];
    double *Qs = smem;                     // [5][PLANE] nodal values of the brick (old, then updated)
    double *Ks = Qs + NV * PLANE;          // [5][PLANE] Runge-Kutta register of the brick, accumulated in place
    double *Tms = Ks + NV * PLANE;         // [5][L]     T- of every line (right state of the line below)
    double *Fss = Tms + C::LINEBUF;        // [5][L]     F* at the + end of every line
    double *Ex = Fss + C::LINEBUF;         // [2][5][EXFACE] traces exported to the cluster neighbours

    // One brick per block, blockIdx = brick coordinates (no persistent loop: a loop over bricks makes the
    // compiler hoist the operator tables out of it into registers).  The grid is rounded up to whole
    // clusters; a block past the last brick only takes part in the cluster barriers.
    const int tid = threadIdx.x, l = tid;
    const int bxi = blockIdx.x, byi = blockIdx.y, bzi = blockIdx.z;
    const bool real = bxi < a.nbx && byi < a.nby && bzi < a.nbz;
    const int brick = bxi + a.nbx * (byi + a.nby * bzi);
    const bool readK = (MODE == DG_MODE_STAGE) && (a.rkA != 0.0);
    const Geo gx = make_geo<C, 0>(l), gy = make_geo<C, 1>(l), gz = make_geo<C, 2>(l);
    const bool inL = (l < L) && real;
    const size_t qbase = (size_t)brick * C::SLOT;

    // ---------------- P0: this brick's Q and K come in ----------------------------------------------------
    if (real) stage_in<C>(Qs, a.Q + qbase, tid);
    cp_async_commit();
    if (real && readK) stage_in<C>(Ks, a.K + qbase, tid);
    cp_async_commit();   // K is not needed before the end of the x pass: its own group

    // The brick that takes this block's place when it ends: blocks are dispatched cluster by cluster in
    // index order, so it is the one `a.grid` (= resident blocks of the whole GPU) further on in that order.
    int next = -1;
    {
        const int ncx = gridDim.x / C::CLX, ncy = gridDim.y / C::CLY;
        const int px = bxi % C::CLX, py = byi % C::CLY, pz = bzi % C::CLZ;
        const long long cid = (bxi / C::CLX) + (long long)ncx * ((byi / C::CLY) + (long long)ncy * (bzi / C::CLZ));
        const long long d = cid * C::CLUSTER + (px + C::CLX * (py + C::CLY * pz)) + a.grid;
        const long long ncid = d / C::CLUSTER;
        const int r = (int)(d - ncid * C::CLUSTER);
        const int cx = (int)(ncid % ncx), cy = (int)((ncid / ncx) % ncy), cz = (int)(ncid / ((long long)ncx * ncy));
        const int nx_ = cx * C::CLX + r % C::CLX, ny_ = cy * C::CLY + (r / C::CLX) % C::CLY, nz_ = cz * C::CLZ + r / (C::CLX * C::CLY);
        if (nx_ < a.nbx && ny_ < a.nby && nz_ < a.nbz) next = nx_ + a.nbx * (ny_ + a.nby * nz_);
    }

    const int ext0 = min(C::BX, a.nx - bxi * C::BX);   // elements of this brick per axis (ragged last brick)
    const int ext1 = min(C::BY, a.ny - byi * C::BY);
    const int ext2 = min(C::BZ, a.nz - bzi * C::BZ);
    const bool full = (ext0 == C::BX) && (ext1 == C::BY) && (ext2 == C::BZ);
    bool actx = inL, acty = inL, actz = inL;
    if (!full && real) {
        actx = inL && line_inside<C, 0>(gx, ext0, ext1, ext2);
        acty = inL && line_inside<C, 1>(gy, ext0, ext1, ext2);
        actz = inL && line_inside<C, 2>(gz, ext0, ext1, ext2);
    }
    double *Tbrick = a.Tnew + (size_t)brick * C::TSLOT;

    // faces shared with a block of the same cluster (never across the periodic wrap, never with a padding block)
    const int px = bxi % C::CLX, py = byi % C::CLY, pz = bzi % C::CLZ;
    const unsigned rank = px + C::CLX * (py + C::CLY * pz);
    const bool ixl = EXCH && px > 0, ixh = EXCH && px < C::CLX - 1 && bxi + 1 < a.nbx;
    const bool iyl = EXCH && py > 0, iyh = EXCH && py < C::CLY - 1 && byi + 1 < a.nby;
    const bool izl = EXCH && pz > 0, izh = EXCH && pz < C::CLZ - 1 && bzi + 1 < a.nbz;

    cp_async_wait<1>();   // Q has landed
    __syncthreads();
    if (MODE != DG_MODE_TRACES) {
        constexpr bool PY = C::CLX > 1, PZ = (C::CLX > 1) || (C::CLY > 1);
        axis_pass<C, 0, MODE, false>(a, gx, l, actx, ext0, halo_source<C, 0>(a, bxi, byi, bzi, 0),
                                     halo_source<C, 0>(a, bxi, byi, bzi, 1), Qs, Ks, Tms, Fss, Ex, readK, qbase, Tbrick,
                                     ixl, ixh, rank - 1, rank + 1);
        __syncthreads();
        axis_pass<C, 1, MODE, PY>(a, gy, l, acty, ext1, halo_source<C, 1>(a, bxi, byi, bzi, 0),
                                  halo_source<C, 1>(a, bxi, byi, bzi, 1), Qs, Ks, Tms, Fss, Ex, readK, qbase, Tbrick,
                                  iyl, iyh, rank - C::CLX, rank + C::CLX);
        __syncthreads();
        // ask L2 for the follow-on brick's data now, about a third of a brick ahead of its use
        if (next >= 0 && !(a.flags & 1)) prefetch_brick<C>(a, next, tid, readK, true);
        axis_pass<C, 2, MODE, PZ>(a, gz, l, actz, ext2, halo_source<C, 2>(a, bxi, byi, bzi, 0),
                                  halo_source<C, 2>(a, bxi, byi, bzi, 1), Qs, Ks, Tms, Fss, Ex, readK, qbase, Tbrick,
                                  izl, izh, rank - C::CLX * C::CLY, rank + C::CLX * C::CLY);
    }
    // ---------------- PE: traces of the updated Q on the brick boundary (z came from registers) --------
    if (MODE != DG_MODE_RESIDUAL) {
        if (MODE == DG_MODE_STAGE) __syncthreads();
        boundary_traces<C, 0>(gx, actx, ext0, Qs, Tbrick, a, !ixl, !ixh);
        boundary_traces<C, 1>(gy, acty, ext1, Qs, Tbrick, a, !iyl, !iyh);
        if (MODE == DG_MODE_TRACES) boundary_traces<C, 2>(gz, actz, ext2, Qs, Tbrick, a);
    }
    // nobody may leave while a cluster neighbour can still read its exports
    if (EXCH) cluster_wait();
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
void stage_config(cudaLaunchConfig_t &cfg, cudaLaunchAttribute &attr, int nbx, int nby, int nbz, cudaStream_t s) {
    // one block per brick, blockIdx = brick coordinates, rounded up to whole clusters
    cfg.gridDim = dim3((unsigned)((nbx + C::CLX - 1) / C::CLX * C::CLX), (unsigned)((nby + C::CLY - 1) / C::CLY * C::CLY),
                       (unsigned)((nbz + C::CLZ - 1) / C::CLZ * C::CLZ));
    cfg.blockDim = dim3(C::THREADS, 1, 1);
    cfg.dynamicSmemBytes = C::SMEM_BYTES;
    cfg.stream = s;
    attr.id = cudaLaunchAttributeClusterDimension;
    attr.val.clusterDim.x = C::CLX;
    attr.val.clusterDim.y = C::CLY;
    attr.val.clusterDim.z = C::CLZ;
    cfg.attrs = &attr;
    cfg.numAttrs = 1;
}

// Opt in to the shared-memory size; *resident = blocks of the stage kernel the whole GPU holds at once.
template <class C>
cudaError_t prepare(int *resident) {
    cudaError_t err = cudaFuncSetAttribute(dg_stage_kernel<C, DG_MODE_STAGE>,
                                           cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_stage_kernel<C, DG_MODE_RESIDUAL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   C::SMEM_BYTES);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_stage_kernel<C, DG_MODE_TRACES>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   C::SMEM_BYTES);
    if (err != cudaSuccess) return err;
    if (C::CLUSTER > 1) {
        cudaLaunchConfig_t cfg = {};
        cudaLaunchAttribute attr;
        stage_config<C>(cfg, attr, C::CLX * 64, C::CLY * 64, C::CLZ * 64, 0);
        int clusters = 0;
        err = cudaOccupancyMaxActiveClusters(&clusters, dg_stage_kernel<C, DG_MODE_STAGE>, &cfg);
        *resident = clusters * C::CLUSTER;
        return err;
    }
    int dev = 0, sms = 0, per_sm = 0;
    err = cudaGetDevice(&dev);
    if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (err == cudaSuccess)
        err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, dg_stage_kernel<C, DG_MODE_STAGE>, C::THREADS,
                                                            C::SMEM_BYTES);
    *resident = per_sm * sms;
    return err;
}

template <class C>
cudaError_t launch_stage(const DgStageArgs &a, cudaStream_t s) {
    if (a.grid <= 0) return cudaErrorInvalidConfiguration;
    cudaLaunchConfig_t cfg = {};
    cudaLaunchAttribute attr;
    stage_config<C>(cfg, attr, a.nbx, a.nby, a.nbz, s);
    if (a.mode == DG_MODE_STAGE) return cudaLaunchKernelEx(&cfg, dg_stage_kernel<C, DG_MODE_STAGE>, a);
    if (a.mode == DG_MODE_RESIDUAL) return cudaLaunchKernelEx(&cfg, dg_stage_kernel<C, DG_MODE_RESIDUAL>, a);
    return cudaLaunchKernelEx(&cfg, dg_stage_kernel<C, DG_MODE_TRACES>, a);
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

// Variants per N (default first): Cfg<N, BX, BY, BZ, min blocks per SM, RELOAD, P, PP, OX, OY, OZ>.
// DESIGN.md "brick shapes" and "shared-memory layout" explain the choices.
#if DG_N == 2
using V0 = Cfg<2, 4, 4, 2, 6, 1, 9, 76, 1, 1, 2>;
using V1 = Cfg<2, 4, 4, 2, 6, 0, 9, 76, 1, 1, 2>;
using V2 = Cfg<2, 4, 4, 4, 3, 1, 8, 65, 1, 0, 0>;
using V3 = Cfg<2, 4, 4, 4, 3, 0, 8, 65, 1, 0, 0>;
#elif DG_N == 3
using V0 = Cfg<3, 4, 4, 2, 2, 1, 12, 156, 3, 0, 0>;
using V1 = Cfg<3, 2, 2, 2, 7, 0, 6, 38, 2, 0, 0>;
using V2 = Cfg<3, 2, 2, 2, 7, 1, 6, 38, 2, 0, 0>;
using V3 = Cfg<3, 4, 4, 2, 2, 0, 12, 156, 3, 0, 0>;
#elif DG_N == 4
using V0 = Cfg<4, 2, 2, 2, 3, 0, 9, 74, 1, 1, 2>;
using V1 = Cfg<4, 2, 2, 2, 3, 1, 9, 74, 1, 1, 2>;
using V2 = Cfg<4, 2, 2, 1, 6, 1, 8, 65, 3, 0, 0>;
using V3 = Cfg<4, 2, 2, 1, 6, 0, 8, 65, 3, 0, 0>;
#elif DG_N == 5
using V0 = Cfg<5, 1, 2, 2, 4, 0, 0, 0, 0, 1, 0>;
using V1 = Cfg<5, 1, 2, 2, 4, 1, 0, 0, 0, 1, 0>;
using V2 = Cfg<5, 1, 2, 2, 4, 0, 0, 0, 0, 1, 0, 2, 2, 2>;
using V3 = Cfg<5, 1, 2, 2, 4, 0, 0, 0, 0, 1, 0, 2, 1, 1>;
using V4 = Cfg<5, 5, 1, 1, 3, 0, 0, 0, 4, 1, 0>;   // 125 lines on 128 threads
using V5 = Cfg<5, 1, 2, 3, 3, 1, 0, 0, 0, 1, 0>;
#define DG_MORE_VARIANTS make_table<V4>(), make_table<V5>(),
#elif DG_N == 6
using V0 = Cfg<6, 1, 1, 2, 4, 1, 6, 38, 1, 0, 0>;
using V1 = Cfg<6, 1, 1, 2, 4, 0, 6, 38, 1, 0, 0>;
using V2 = Cfg<6, 1, 2, 2, 2, 1, 6, 75, 0, 3, 0>;
using V3 = Cfg<6, 1, 2, 2, 2, 0, 6, 75, 0, 3, 0>;
#elif DG_N == 7
using V0 = Cfg<7, 1, 1, 2, 3, 1, 7, 55, 1, 0, 0>;
using V1 = Cfg<7, 1, 1, 2, 3, 0, 7, 55, 1, 0, 0>;
using V2 = Cfg<7, 1, 1, 1, 6, 1, 7, 55, 1, 0, 0>;
using V3 = Cfg<7, 1, 1, 1, 6, 0, 7, 55, 1, 0, 0>;
#elif DG_N == 8
using V0 = Cfg<8, 1, 1, 2, 2, 0, 8, 65, 1, 1, 0>;
using V1 = Cfg<8, 1, 1, 2, 2, 1, 8, 65, 1, 1, 0>;
using V2 = Cfg<8, 1, 1, 1, 4, 1, 8, 65, 1, 0, 0>;
using V3 = Cfg<8, 1, 1, 1, 4, 0, 8, 65, 1, 0, 0>;
#else
#error "DG_N must be 2..8"
#endif

using VE = Cfg<DG_N, 1, 1, 1, 4, 1>;   // one element per block: always there (tiny and ragged meshes, tests)

#ifndef DG_MORE_VARIANTS
#define DG_MORE_VARIANTS
#endif
const DgKernelTable k_tables[] = {make_table<V0>(), make_table<V1>(), make_table<V2>(), make_table<V3>(),
                                  DG_MORE_VARIANTS make_table<VE>()};

}  // namespace

#define DG_CAT2(a, b) a##b
#define DG_CAT(a, b) DG_CAT2(a, b)
const DgKernelTable *DG_CAT(dg_variants_N, DG_N)(int *count) {
    *count = (int)(sizeof(k_tables) / sizeof(k_tables[0]));
    return k_tables;
}
