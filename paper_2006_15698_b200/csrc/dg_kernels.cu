// dg_kernels.cu -- CUDA kernels of the DG Euler time step for one N = p+1 (compile with -DDG_N=<N>,
// -gencode arch=compute_100a,code=sm_100a).  Hand-written for B200; fp64 throughout.
//
// The fused stage kernel (v5, "column sweep"): the mesh is cut into columns of BX x BY elements; ONE thread
// block marches through `lz` consecutive z layers (BX x BY x 1 elements each) of one column.  Per layer, in
// ONE sweep over HBM:
//   copy warp   cp.async.bulk (TMA engine, mbarrier completion) brings the layer's Q and K slots into a ring
//               of shared-memory buffers one to two layers ahead of their use and writes the updated Q and K
//               back with cp.async.bulk stores: no thread ever touches Q or K in global memory
//   compute warps, one thread per node LINE, for the axes x, y, z in turn (instances of one template):
//   PH  the neighbour columns' face traces this line touches go straight from HBM/L2 into registers (x, y);
//       along z the upper neighbour is the NEXT layer of the ring (its trace is taken from shared memory) and
//       the lower face's flux is the one this thread computed for the previous layer (kept in registers):
//       z traces go through HBM only at the two ends of a chunk
//   PT  the line's N nodal values into registers and the two face traces T+- = sum_q l_q(+-1) Q_q
//   PB  local Lax-Friedrichs interface flux, doubled: faces inside a column once (x, y: handed
//       over through shared memory; z: carried in registers), faces on the column boundary by both sides
//   PC  lift with 2/h, 1/2 and dt folded into the tables starts the accumulators:
//       r_i = sum_q Dhat_iq F_q - (l_i(+1) F*_+ - l_i(-1) F*_-) (2/h_a)/w_i       (eq (5) 3rd and 2nd term)
//   PA  pointwise Euler flux (eq (2)-(3)) at the line's N nodes and the sum-factorised
//       derivative (the contraction of listing lines 220-237), all in registers
//   PD  LSERK45 accumulated in place on the staged K:  x: K = A K + s_x r_x,  y: K += s_y r_y,
//       z: K += s_z r_z (s_a = dt 2/h_a), written straight to HBM from the z lines; Q += B K left in shared memory
//       for the copy warp; or R itself in residual mode
//   PE  x / y face traces of the UPDATED Q on the column boundary, written to the other trace buffer
// so that Q and K are read once and written once per stage and no block ever needs another block's nodal
// values: neighbours meet only through the double-buffered column-boundary traces.
//
// Nothing here is shared with oracle/ (separate source, separate operator construction).
#include "dg_internal.h"

#include <stdint.h>

#include <type_traits>

#ifndef DG_N
#error "compile with -DDG_N=<p+1>"
#endif

namespace {

// ------------------------------------------------------------------------------------------------
// compile-time geometry of one variant
// ------------------------------------------------------------------------------------------------
// Shared-memory layout of a layer: [5][N] planes (variable, z node k) of pitch PP doubles, dense rows of GX
// doubles inside a plane, and, per axis, the order in which a warp's lanes walk the node lines (ORD):
//   0: t1 fastest, then t2, then the element e along the axis      1: t2, t1, e
//   2: t1, e, t2                                                   3: t2, e, t1
//   4: e, t1, t2                                                   5: e, t2, t1
//   6: e, t1 inside a group of 32 (or, if t1 x e fits, 16) lanes per t2: every t2 plane of lines has a warp or half-warp
//      of its own (idle lanes at its end), so that no half-warp straddles two planes
// (t1,t2) = (gy,k) for x lines, (gx,k) for y lines, (gx,gy) for z lines.  PP (even: planes stay 16-byte
// aligned for the bulk copies) and the orders are picked per column shape so that the 16 lanes of a
// half-warp hit different 8-byte bank pairs where such a choice exists.
template <int N_, int BX_, int BY_, int MINB_, int RELOAD_ = 0, int PP_ = 0, int OX_ = 0, int OY_ = 0, int SHFL_ = 0>
struct Cfg {
    static constexpr int N = N_, BX = BX_, BY = BY_, MINB = MINB_;
    // RELOAD = 1: the volume term reads the line's Q from shared memory a second time instead of keeping
    // it in 10 N registers across the interface fluxes
    static constexpr bool RELOAD = RELOAD_ != 0;
    static constexpr int GX = BX * N, GY = BY * N;                 // nodes of a layer per axis (z: N)
    // pitch of one (gy,gx) plane, doubles, in HBM AND in shared memory (a layer is ONE bulk copy): even, and
    // padded by PP_ - GX GY where that removes shared-memory bank conflicts at a few per cent more traffic
    static constexpr int HP = PP_ ? PP_ : ((GX * GY + 1) & ~1);
    static constexpr int NPL = DG_NV * N;                          // planes per slot
    static constexpr int SLOT = (NPL * HP + 15) & ~15;             // doubles per layer slot in Q, K (128-byte multiple)
    static constexpr int P = GX;                                   // shared-memory row pitch (dense)
    static constexpr int PP = HP;                                  // shared-memory plane pitch
    static constexpr int PLANE = N * PP;                           // shared doubles per variable
    static constexpr int BUF = DG_NV * PLANE;                      // shared doubles per layer buffer
    static constexpr int OX = OX_, OY = OY_;
    // SHFL = 1: an axis with two elements whose element index runs fastest in the lane order (ORD 4) hands its interior
    // face over with warp shuffles instead of shared memory and two block barriers (measured: +1.5 % at N = 7, -4 % at N = 5)
    static constexpr bool SHFL = SHFL_ != 0;
    // the barrier between the y pass and the z-pass update as a SPLIT barrier (mbarrier: a warp arrives when its y pass ends
    // and waits only before the update): + 1.5 % at N = 8, + 0.6 % at N = 7, - 1 % at N = 5 and N = 2 (A/B measured)
    static constexpr bool YSPLIT = N_ >= 7;
    // the x and y boundary traces of the updated Q (phase PE) computed by the copy warp instead of the compute warps
    // (A/B measured: p = 1 +2.6 %, p = 2 +0.8 %, p = 3 +1.8 %, p = 7 +3.8 %, cfg5 +3 %; none at N = 5, 6, -1 % at N = 7)
    static constexpr bool XPE = N_ <= 4 || N_ == 8;
    static constexpr int L = GX * GY;                              // node lines per axis = threads that work
    static constexpr int NCOMP = (L + 31) / 32 * 32;               // compute threads
    static constexpr int THREADS = NCOMP + 32;                     // + the copy warp
    static constexpr int CX = GY * N, CY = GX * N, CZ = GX * GY;   // face nodes of a layer side per axis
    static constexpr int TXY = 2 * DG_NV * (CX + CY);              // x/y trace doubles per layer slot
    static constexpr int TZ = 2 * DG_NV * CZ;                      // z trace doubles per chunk slot
    static constexpr bool MULTI = (BX > 1) || (BY > 1);
    static constexpr int LINEBUF = MULTI ? ((DG_NV * L + 1) & ~1) : 0;   // T- / F* hand-over between elements of a layer
    static_assert(PP >= HP && (PP % 2) == 0, "plane pitch must be even and hold a plane");
    static_assert((BUF % 2) == 0 && (LINEBUF % 2) == 0, "buffers must stay 16-byte aligned");
};

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// ---- mbarrier + bulk-copy (TMA engine) primitives ---------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t *b, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *b, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *b, unsigned parity) {
    const unsigned addr = smem_u32(b);
    unsigned done;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(addr), "r"(parity)
            : "memory");
    } while (!done);
}
// global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_load(double *sdst, const double *gsrc, unsigned bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(sdst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// shared -> global, completion tracked by the issuing thread's bulk groups
__device__ __forceinline__ void bulk_store(double *gdst, const double *ssrc, unsigned bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)),
                 "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// generic-proxy writes to shared memory become visible to the async proxy (the bulk stores)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// Ask L2 to fetch [ptr, ptr + bytes) (rounded out to 16-byte granules): one instruction per block of data.
__device__ __forceinline__ void l2_prefetch(const void *ptr, unsigned bytes) {
    const uintptr_t lo = (uintptr_t)ptr & ~(uintptr_t)15;
    const uintptr_t hi = ((uintptr_t)ptr + bytes + 15) & ~(uintptr_t)15;
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(lo), "r"((unsigned)(hi - lo)) : "memory");
}
// named barriers: 1 = the compute warps among themselves, 2 = compute warps -> copy warp ("layer finished")
template <int NTHREADS>
__device__ __forceinline__ void bar_sync(int id) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(NTHREADS) : "memory");
}
template <int NTHREADS>
__device__ __forceinline__ void bar_arrive(int id) {
    asm volatile("bar.arrive %0, %1;" ::"r"(id), "n"(NTHREADS) : "memory");
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
    // Products rounded on their own (never contracted into a later add): the interface flux below adds the
    // fluxes of the two sides, and a product fused into that sum on one side only would make the two blocks
    // that share a face compute fluxes that differ in the last bit.
    F[0] = Q[1];                                    // rho u_a
    F[1] = fma(Q[1], vel, pres);
    F[2] = __dmul_rn(Q[2], vel);
    F[3] = __dmul_rn(Q[3], vel);
    F[4] = __dmul_rn(Q[4] + pres, vel);
}

// Local Lax-Friedrichs flux (reading R3), rotated slots as above, returned DOUBLED
// (the factor 1/2 is folded into the lift tables):
//   2 F* = F(QL) + F(QR) - lam (QR - QL),  lam = max(|u_a^L| + c_L, |u_a^R| + c_R)
// written for (own, other) with sgn = +1 when own is the left state, -1 when it is the right one; the two
// evaluations of one face (by the blocks on either side) are bit-identical.
__device__ __forceinline__ void lax_friedrichs2(const double (&Qown)[DG_NV], const double (&Qoth)[DG_NV], double sgn,
                                                double gamma, double gm1, double (&Fs)[DG_NV]) {
    double Fa[DG_NV], Fb[DG_NV], ua, ub, pa, pb, ra, rb;
    euler_flux_normal(Qown, gm1, Fa, ua, pa, ra);
    euler_flux_normal(Qoth, gm1, Fb, ub, pb, rb);
    const double lama = fabs(ua) + sqrt_pos(gamma * pa * ra);
    const double lamb = fabs(ub) + sqrt_pos(gamma * pb * rb);
    const double sl = sgn * ((lama > lamb) ? lama : lamb);
#pragma unroll
    for (int n = 0; n < DG_NV; ++n) Fs[n] = fma(-sl, Qoth[n] - Qown[n], __dadd_rn(Fa[n], Fb[n]));
}

// ------------------------------------------------------------------------------------------------
// per-axis compile-time traits and the (layer-independent) geometry of a thread's node line
//   line l = e * Ca + c,  e = element along the axis, c = face node = position in the lane order
//   axis x: (t1,t2) = (gy,k);  y: (gx,k);  z: (gx,gy)
// ------------------------------------------------------------------------------------------------
template <class C, int AX>
struct Axis {
    static constexpr int S = (AX == 0) ? 1 : (AX == 1) ? C::P : C::PP;                 // shared stride along the line
    static constexpr int Ca = (AX == 0) ? C::CX : (AX == 1) ? C::CY : C::CZ;           // face nodes of a layer side
    static constexpr int T1 = (AX == 0) ? C::GY : C::GX;
    static constexpr int T2 = (AX == 2) ? C::GY : C::N;
    static constexpr int ORD = (AX == 0) ? C::OX : (AX == 1) ? C::OY : 0;
    static constexpr int B = (AX == 0) ? C::BX : (AX == 1) ? C::BY : 1;                // elements along the axis
    static constexpr int TBASE = (AX == 0) ? 0 : 2 * DG_NV * C::CX;                    // inside a Txy slot
    static constexpr bool MULTI = B > 1;
    // momentum slots rotated so that slot 1 is the component along this axis: slot s holds variable VAR[s]
    static constexpr int M1 = 1 + AX, M2 = (AX == 2) ? 1 : 2 + AX, M3 = (AX == 0) ? 3 : AX;
};
template <class C, int AX>
__device__ __forceinline__ constexpr int var_of_slot(int s) {
    return s == 0 ? 0 : s == 1 ? Axis<C, AX>::M1 : s == 2 ? Axis<C, AX>::M2 : s == 3 ? Axis<C, AX>::M3 : 4;
}

struct Geo {
    int base;   // shared-memory offset (doubles, inside one variable's planes) of node 0 of the line
    int c;      // face-node index of the line on the layer side (lane order: this is how the traces are stored)
    int e;      // element along the axis
    int t1, t2; // transverse node indices
    bool ok;    // the thread has a line of its own (false: it computes on a valid line and stores nothing)
};

template <class C, int AX>
__device__ __forceinline__ Geo make_geo(int l) {
    using A = Axis<C, AX>;
    constexpr int N = C::N, T1 = A::T1, T2 = A::T2, B = A::B;
    Geo g;
    if (A::ORD == 6) {
        // one (t2) plane of lines per warp -- or per half-warp when it fits --, element index fastest: no half-warp
        // straddles two planes, so that its lanes' addresses stay an arithmetic sequence whatever the plane pitch
        constexpr int G = (T1 * B <= 16) ? 16 : 32;
        static_assert(A::ORD != 6 || (T1 * B <= 32 && T2 * G <= C::NCOMP), "ORD 6 does not fit this shape");
        const int r = min(l % G, T1 * B - 1);
        g.ok = (l % G) < T1 * B && (l / G) < T2;
        g.e = r % B;
        g.t1 = r / B;
        g.t2 = min(l / G, T2 - 1);
        g.c = g.t2 * T1 + g.t1;
    } else {
    g.ok = l < C::L;
    l = min(l, C::L - 1);
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
    }
    if (AX == 0) g.base = g.t2 * C::PP + g.t1 * C::P + g.e * N;
    else if (AX == 1) g.base = g.t2 * C::PP + g.e * N * C::P + g.t1;
    else g.base = g.t2 * C::P + g.t1;
    return g;
}

// Is the line inside a ragged (last) column of ext0 x ext1 elements?
template <class C, int AX>
__device__ __forceinline__ bool line_inside(const Geo &g, int ext0, int ext1) {
    if (AX == 0) return g.t1 < ext1 * C::N && g.e < ext0;
    if (AX == 1) return g.t1 < ext0 * C::N && g.e < ext1;
    return g.t1 < ext0 * C::N && g.t2 < ext1 * C::N;
}

// Reference-element operators of this N (DgRefOps; uploaded by prepare()).  "-" side tables are the "+" side
// tables read backwards (symmetric nodes).
__constant__ DgRefOps c_ref;
#define DG_LP(q) c_ref.lp[q]
#define DG_LM(q) c_ref.lp[DG_N - 1 - (q)]
#define DG_LQP(i) c_ref.lq[i]
#define DG_LQM(i) c_ref.lq[DG_N - 1 - (i)]

// What the compute warps need of the kernel arguments and the block's position, written to shared memory once
// per block: layer_body() is a separate (not inlined) function and takes everything from here.
struct BlockInfo {
    const double *halo[4];     // Txy_old blocks of layer z0 this column reads: x low, x high, y low, y high
    double *txy_out;           // this column's Txy_new slot of layer z0
    const double *tz_lo, *tz_hi;
    double *tz_out;
    double *kslot;             // this column's K slot of layer z0
    long long tstride;         // doubles between consecutive layers in Txy
    long long hstride[4];      // ... in the four blocks of halo[] (Txy, or an external halo buffer)
    long long kstride;         // ... in Q and K
    double gamma, gm1, rkA, rkB, scale[3];
    int ext0, ext1, readK, storeK, nl;
    int bc[6];                 // boundary condition of this block's x-, x+, y-, y+, z-, z+ side if it lies on a non-periodic
                               // domain face (1 slip wall, 2 far field), else 0
    double qinf[DG_NV];
    // "push" mode of a block decomposition: where this block ALSO stores the traces of the updated state on the domain
    // faces it touches (the neighbour context's halo buffer, possibly in a peer GPU's memory), or null
    double *push[4];           // x low, x high, y low, y high: the [5][Ca] block of layer z0
    long long pstride[4];      // doubles between consecutive layers
    double *push_z[2];         // z low (first chunk), z high (last chunk): the [5][CZ] block of this column
};

// PE for one of the axes x, y: traces of the Q in shared memory on the column boundary -> Tslot.
template <class C, int AX>
__device__ __forceinline__ void boundary_traces(const Geo &g, bool act, int exta, const double *Qs, double *Tslot,
                                                double *push_lo = nullptr, double *push_hi = nullptr) {
    using A = Axis<C, AX>;
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE;
    const bool first = g.e == 0, last = g.e == exta - 1;
    if (!act || !(first || last)) return;
    double *dst = Tslot + A::TBASE + g.c;
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
                Tp[n] = fma(DG_LP(q), Qv, Tp[n]);
                Tm[n] = fma(DG_LM(q), Qv, Tm[n]);
            }
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            dst[n * A::Ca] = Tm[n];
            dst[(NV + n) * A::Ca] = Tp[n];
            if (push_lo) push_lo[n * A::Ca + g.c] = Tm[n];
            if (push_hi) push_hi[n * A::Ca + g.c] = Tp[n];
        }
    } else if (A::ORD < 4 && first) {   // (the lines of the first and of the last element sit in different warps)
        double T[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) T[n] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q)
#pragma unroll
            for (int n = 0; n < NV; ++n) T[n] = fma(DG_LM(q), Q0[n * PLANE + q * A::S], T[n]);
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            dst[n * A::Ca] = T[n];
            if (push_lo) push_lo[n * A::Ca + g.c] = T[n];
        }
    } else if (A::ORD < 4) {
        double T[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) T[n] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q)
#pragma unroll
            for (int n = 0; n < NV; ++n) T[n] = fma(DG_LP(q), Q0[n * PLANE + q * A::S], T[n]);
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            dst[(NV + n) * A::Ca] = T[n];
            if (push_hi) push_hi[n * A::Ca + g.c] = T[n];
        }
    } else {
        // element index fastest in the lane order: lines of the first and of the last element share every warp.  One
        // trace per line, T- for the former and T+ for the latter, in ONE instruction stream (two divergent branches
        // would run every load twice with half the lanes, and those lanes' addresses collide in the banks)
        double T[NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) T[n] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q) {
            const double w = first ? DG_LM(q) : DG_LP(q);
#pragma unroll
            for (int n = 0; n < NV; ++n) T[n] = fma(w, Q0[n * PLANE + q * A::S], T[n]);
        }
        double *d1 = dst + (first ? 0 : NV * A::Ca);
        double *push = first ? push_lo : push_hi;
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            d1[n * A::Ca] = T[n];
            if (push) push[n * A::Ca + g.c] = T[n];
        }
    }
}

// Trace block [5][Ca] a column needs for (axis x or y, side) in layer ez: side 0 = T+ of the column below
// (stored as that column's side 1), side 1 = T- of the column above (its side 0).  Periodic.
template <class C, int AX>
__device__ __forceinline__ const double *halo_source(const double *T, int nbx, int nby, int bx, int by, int ez, int side) {
    using A = Axis<C, AX>;
    if (AX == 0) bx = (side == 0) ? ((bx == 0) ? nbx - 1 : bx - 1) : ((bx + 1 == nbx) ? 0 : bx + 1);
    else by = (side == 0) ? ((by == 0) ? nby - 1 : by - 1) : ((by + 1 == nby) ? 0 : by + 1);
    const size_t nbr = (size_t)bx + (size_t)nbx * ((size_t)by + (size_t)nby * ez);
    return T + nbr * C::TXY + A::TBASE + (side == 0 ? DG_NV * A::Ca : 0);
}

// Exterior (ghost) state of a non-periodic domain face from the interior trace T, momentum slots rotated for AX
// (reading R19): slip wall = T with the normal momentum (slot 1) negated; far field = the prescribed state.
template <class C, int AX>
__device__ __forceinline__ void ghost_state(int kind, const double (&T)[DG_NV], const double *qinf, double (&G)[DG_NV]) {
#pragma unroll
    for (int s = 0; s < DG_NV; ++s) G[s] = (kind == 2) ? qinf[var_of_slot<C, AX>(s)] : T[s];
    if (kind == 1) G[1] = -T[1];
}

// PC + PA for one line: V_i = sum_q Dhat_iq F_q - (l_i(+1) 2F*_+ - l_i(-1) 2F*_-)/(2 w_i), F_q the pointwise Euler flux
// of the line's node q (loadQ(q, Qn) delivers its state, slots rotated).  N >= 5: even-odd form (DgRefOps): the
// nodes are taken in mirror pairs, half-size operators act on the sum and the difference of the pair's fluxes.
template <class C, class LoadQ>
__device__ __forceinline__ void lift_and_volume(LoadQ loadQ, double gm1, const double (&Fm)[DG_NV], const double (&Fp)[DG_NV],
                                                double (&V)[DG_NV][C::N]) {
    constexpr int N = C::N, NV = DG_NV;
    if constexpr (N < 5) {
#pragma unroll
        for (int i = 0; i < N; ++i) {
            const double cp = DG_LQP(i), cm = DG_LQM(i);
#pragma unroll
            for (int n = 0; n < NV; ++n) V[n][i] = fma(cm, Fm[n], -cp * Fp[n]);
        }
#pragma unroll
        for (int q = 0; q < N; ++q) {
            double Qn[NV], F[NV], vel, pres, rinv;
            loadQ(q, Qn);
            euler_flux_normal(Qn, gm1, F, vel, pres, rinv);
#pragma unroll
            for (int n = 0; n < NV; ++n)
#pragma unroll
                for (int i = 0; i < N; ++i) V[n][i] = fma(c_ref.D[q][i], F[n], V[n][i]);
        }
    } else {
        constexpr int H = N / 2, ODD = N & 1, MID = N / 2;
        double A[NV][H], S[NV][H + ODD];
        // lift: L_i + L_i' = (lq_i + lq_i')(F*_- - F*_+),  L_i - L_i' = (lq_i' - lq_i)(F*_- + F*_+)   (halved in the tables)
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            const double fd = Fm[n] - Fp[n], fs = Fm[n] + Fp[n];
#pragma unroll
            for (int i = 0; i < H; ++i) {
                S[n][i] = c_ref.ls[i] * fd;
                A[n][i] = c_ref.la[i] * fs;
            }
            if (ODD) S[n][ODD ? MID : 0] = c_ref.ls[MID] * fd;
        }
#pragma unroll
        for (int q = 0; q < H; ++q) {
            double Qa[NV], Qb[NV], Fa[NV], Fb[NV], vel, pres, rinv;
            loadQ(q, Qa);
            loadQ(N - 1 - q, Qb);
            euler_flux_normal(Qa, gm1, Fa, vel, pres, rinv);
            euler_flux_normal(Qb, gm1, Fb, vel, pres, rinv);
#pragma unroll
            for (int n = 0; n < NV; ++n) {
                const double fe = Fa[n] + Fb[n], fo = Fa[n] - Fb[n];
#pragma unroll
                for (int i = 0; i < H; ++i) A[n][i] = fma(c_ref.Pe[q][i], fe, A[n][i]);
#pragma unroll
                for (int i = 0; i < H + ODD; ++i) S[n][i] = fma(c_ref.Po[q][i], fo, S[n][i]);
            }
        }
        if (ODD) {
            double Qc[NV], Fc[NV], vel, pres, rinv;
            loadQ(MID, Qc);
            euler_flux_normal(Qc, gm1, Fc, vel, pres, rinv);
#pragma unroll
            for (int n = 0; n < NV; ++n)
#pragma unroll
                for (int i = 0; i < H; ++i) A[n][i] = fma(c_ref.Dm[i], Fc[n], A[n][i]);
        }
#pragma unroll
        for (int n = 0; n < NV; ++n) {
#pragma unroll
            for (int i = 0; i < H; ++i) {
                V[n][i] = S[n][i] + A[n][i];
                V[n][N - 1 - i] = S[n][i] - A[n][i];
            }
            if (ODD) V[n][MID] = S[n][ODD ? MID : 0];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// the x and y passes of one layer
// ------------------------------------------------------------------------------------------------
// Order chosen for register pressure: the line's Q goes into registers once; the face traces and the two
// interface fluxes come first (no accumulators alive yet); the accumulators then START from the lift term
// and the volume term is added node by node.
//   r_i = (2/h_a) [ sum_q Dhat_iq F_q - (l_i(+1) F*_+ - l_i(-1) F*_-)/w_i ]
// Threads without a line of their own (`act` false: the tail of the last warp, lines in the padding of a ragged
// column) run the arithmetic on a valid line all the same and only their stores are switched off.
template <class C, int AX, int MODE, bool BC>
__device__ __forceinline__ void xy_pass(const BlockInfo *bi, const Geo &g, bool act, int exta, const double *halo_lo,
                                        const double *halo_hi, const double *Qs, double *KR, double *Tms, double *Fss,
                                        uint64_t *fullk, unsigned kparity) {
    using A = Axis<C, AX>;
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE, L = C::L, S = A::S, Ca = A::Ca;
    const bool first = g.e == 0, last = g.e == exta - 1;
    // slot of this line in the hand-over buffers: neighbouring lanes write neighbouring slots (element index fastest
    // where it is fastest in the lane order); HS = distance to the next element's line
    constexpr int HS = (A::ORD >= 4) ? 1 : Ca;
    const int lb = (A::ORD >= 4) ? g.c * A::B + g.e : g.e * Ca + g.c;
    const double gamma = bi->gamma, gm1 = bi->gm1;
    // PH: the neighbour columns' traces this line touches, momentum slots rotated, HBM/L2 -> registers
    double Hlo[NV], Hhi[NV];
#pragma unroll
    for (int s = 0; s < NV; ++s) {
        Hlo[s] = 1.0;
        Hhi[s] = 1.0;
    }
    if (act && first) {
#pragma unroll
        for (int s = 0; s < NV; ++s) Hlo[s] = __ldg(halo_lo + var_of_slot<C, AX>(s) * Ca + g.c);
    }
    if (act && last) {
#pragma unroll
        for (int s = 0; s < NV; ++s) Hhi[s] = __ldg(halo_hi + var_of_slot<C, AX>(s) * Ca + g.c);
    }

    // ------------- PT: the line's nodal values (slot s holds variable var_of_slot(s)) and its traces ----
    double QL[C::RELOAD ? 1 : NV][C::RELOAD ? 1 : N], Tp[NV], Tm[NV];
    const double *Q0 = Qs + g.base;
#pragma unroll
    for (int s = 0; s < NV; ++s) {
        Tp[s] = 0.0;
        Tm[s] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q) {
            const double Qv = Q0[var_of_slot<C, AX>(s) * PLANE + q * S];
            if (!C::RELOAD) QL[s][q] = Qv;
            Tp[s] = fma(DG_LP(q), Qv, Tp[s]);
            Tm[s] = fma(DG_LM(q), Qv, Tm[s]);
        }
    }
    // non-periodic domain faces (BC instances only): the neighbour's trace is the ghost state of the own one
    if (BC) {
        const int blo = bi->bc[2 * AX], bhi = bi->bc[2 * AX + 1];
        if (blo && first) ghost_state<C, AX>(blo, Tm, bi->qinf, Hlo);
        if (bhi && last) ghost_state<C, AX>(bhi, Tp, bi->qinf, Hhi);
    }
    // Two elements along the axis with the element index fastest in the lane order: the two lines that share an
    // interior face sit in neighbouring lanes of one warp, and the hand-over is two warp shuffles (no shared
    // memory, no block barrier).
    constexpr bool SHF = C::SHFL && A::MULTI && A::B == 2 && A::ORD == 4;
    if (A::MULTI && !SHF) {
        if (act) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Tms[n * L + lb] = Tm[n];
        }
        bar_sync<C::NCOMP>(1);
    }

    // ------------- PB: interface fluxes ----------------------------------------------------------------
    double Fp[NV], Fm[NV];
    if (SHF) {
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            const double t = __shfl_down_sync(0xffffffffu, Tm[n], 1);   // T- of the next element of this layer
            if (!last) Hhi[n] = t;
        }
    } else if (A::MULTI && act && !last) {
#pragma unroll
        for (int n = 0; n < NV; ++n) Hhi[n] = Tms[n * L + lb + HS];   // T- of the next element of this layer
    }
    lax_friedrichs2(Tp, Hhi, 1.0, gamma, gm1, Fp);
    if (SHF) {
        // every warp holds lines of both elements: evaluated by all lanes (no divergence, the two evaluations
        // interleave); the lanes of the upper element take the shuffled flux instead
        lax_friedrichs2(Tm, Hlo, -1.0, gamma, gm1, Fm);
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            const double t = __shfl_up_sync(0xffffffffu, Fp[n], 1);     // the face this line shares with the element below
            if (!first) Fm[n] = t;
        }
    } else if (A::MULTI) {
        if (act) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Fss[n * L + lb] = Fp[n];
        }
        if (first) lax_friedrichs2(Tm, Hlo, -1.0, gamma, gm1, Fm);
        bar_sync<C::NCOMP>(1);
        if (!first) {
#pragma unroll
            for (int n = 0; n < NV; ++n) Fm[n] = Fss[n * L + lb - HS];
        }
    } else {
        lax_friedrichs2(Tm, Hlo, -1.0, gamma, gm1, Fm);
    }

    // ------------- PC + PA: lift, pointwise flux and sum-factorised derivative -------------------------------
    double V[NV][N];
    lift_and_volume<C>(
        [&](int q, double(&Qn)[NV]) {
#pragma unroll
            for (int s = 0; s < NV; ++s)
                Qn[s] = C::RELOAD ? Q0[var_of_slot<C, AX>(s) * PLANE + q * S] : QL[C::RELOAD ? 0 : s][C::RELOAD ? 0 : q];
        },
        gm1, Fm, Fp, V);
    // ------------- PD: Runge-Kutta accumulation on the staged K -----------------------------------------
    if (AX == 0) {
        if (bi->readK) mbar_wait(fullk, kparity);   // this layer's K has landed in KR
    } else if (!A::MULTI || SHF) {
        bar_sync<C::NCOMP>(1);         // the x pass of every line is done (the hand-over barriers above said so otherwise)
    }
    if (act) {
        double *K0 = KR + g.base;
        const double sc = bi->scale[AX];
        if (AX == 0) {
            if (bi->readK) {
                const double rkA = bi->rkA;
#pragma unroll
                for (int s = 0; s < NV; ++s)
#pragma unroll
                    for (int i = 0; i < N; ++i) {
                        double *p = K0 + var_of_slot<C, AX>(s) * PLANE + i * S;
                        *p = fma(rkA, *p, sc * V[s][i]);
                    }
            } else {
#pragma unroll
                for (int s = 0; s < NV; ++s)
#pragma unroll
                    for (int i = 0; i < N; ++i) K0[var_of_slot<C, AX>(s) * PLANE + i * S] = sc * V[s][i];
            }
        } else {
#pragma unroll
            for (int s = 0; s < NV; ++s)
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    double *p = K0 + var_of_slot<C, AX>(s) * PLANE + i * S;
                    *p = fma(sc, V[s][i], *p);
                }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// the z pass of one layer: thread (gx, gy) owns the z line; the flux on the lower face of the layer is the one
// this thread computed for the upper face of the previous layer, kept in FmS (shared memory, [5][L])
// ------------------------------------------------------------------------------------------------
template <class C, int MODE, bool LAM, bool BC>
__device__ __forceinline__ void z_pass(const BlockInfo *bi, const Geo &g, int l, bool act, double *Qs, const double *Qnext,
                                       const double *KR, double *FmS, double *Kg, bool first_layer, bool last_layer,
                                       uint64_t *ydone, unsigned yparity, double &lam_best) {
    constexpr int AX = 2;
    using A = Axis<C, AX>;
    constexpr int N = C::N, NV = DG_NV, PLANE = C::PLANE, S = A::S, Ca = A::Ca, L = C::L;
    const double gamma = bi->gamma, gm1 = bi->gm1;
    double QL[C::RELOAD ? 1 : NV][C::RELOAD ? 1 : N], V[NV][N], Fp[NV], Fm[NV];
    // PH: T- of the line above: from the next layer of the ring, or (top of the chunk) from HBM
    double Hhi[NV];
    if (!last_layer) {
        const double *Q1 = Qnext + g.base;
#pragma unroll
        for (int s = 0; s < NV; ++s) {
            double t = 0.0;
#pragma unroll
            for (int q = 0; q < N; ++q) t = fma(DG_LM(q), Q1[var_of_slot<C, AX>(s) * PLANE + q * S], t);
            Hhi[s] = t;
        }
    } else {
        const double *tz_hi = bi->tz_hi;
#pragma unroll
        for (int s = 0; s < NV; ++s) Hhi[s] = __ldg(tz_hi + var_of_slot<C, AX>(s) * Ca + g.c);
    }
    // PT
    double Tp[NV];
    const double *Q0 = Qs + g.base;
#pragma unroll
    for (int s = 0; s < NV; ++s) {
        Tp[s] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q) {
            const double Qv = Q0[var_of_slot<C, AX>(s) * PLANE + q * S];
            if (!C::RELOAD) QL[s][q] = Qv;
            Tp[s] = fma(DG_LP(q), Qv, Tp[s]);
        }
    }
    if (BC && last_layer && bi->bc[5]) ghost_state<C, AX>(bi->bc[5], Tp, bi->qinf, Hhi);   // non-periodic top of the domain
    // PB
    if (first_layer) {   // bottom of the chunk: own T- against T+ of the layer below (from HBM)
        double Tm[NV], Hlo[NV];
        const double *tz_lo = bi->tz_lo;
#pragma unroll
        for (int s = 0; s < NV; ++s) {
            double t = 0.0;
#pragma unroll
            for (int q = 0; q < N; ++q) t = fma(DG_LM(q), Q0[var_of_slot<C, AX>(s) * PLANE + q * S], t);
            Tm[s] = t;
            Hlo[s] = __ldg(tz_lo + var_of_slot<C, AX>(s) * Ca + g.c);
        }
        if (BC && bi->bc[4]) ghost_state<C, AX>(bi->bc[4], Tm, bi->qinf, Hlo);   // non-periodic bottom of the domain
        lax_friedrichs2(Tm, Hlo, -1.0, gamma, gm1, Fm);
    } else {
#pragma unroll
        for (int n = 0; n < NV; ++n) Fm[n] = FmS[n * L + l];
    }
    lax_friedrichs2(Tp, Hhi, 1.0, gamma, gm1, Fp);
    if (!last_layer) {
#pragma unroll
        for (int n = 0; n < NV; ++n) FmS[n * L + l] = Fp[n];   // the next layer's lower face (same thread reads it)
    }
    // PC + PA
    lift_and_volume<C>(
        [&](int q, double(&Qn)[NV]) {
#pragma unroll
            for (int s = 0; s < NV; ++s)
                Qn[s] = C::RELOAD ? Q0[var_of_slot<C, AX>(s) * PLANE + q * S] : QL[C::RELOAD ? 0 : s][C::RELOAD ? 0 : q];
        },
        gm1, Fm, Fp, V);
    // every warp's y pass is done with K and with Q (YSPLIT: each warp arrived when its y pass ended, so a warp that is
    // ahead waits for the others' y passes only, not for their z-pass arithmetic above)
    if (C::YSPLIT) mbar_wait(ydone, yparity);
    else bar_sync<C::NCOMP>(1);
    if (act) {
        // PD: the updated K (or R) goes straight to HBM from the z lines (coalesced across the lanes, streaming),
        // so that KR is free for the next layer's K as soon as every line has read it
        const double *K0 = KR + g.base;
        double *Kline = Kg + g.base;
        double *Q0w = Qs + g.base;
        const double sc = bi->scale[AX];
        if (MODE == DG_MODE_RESIDUAL) {
#pragma unroll
            for (int s = 0; s < NV; ++s)
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    const int n = var_of_slot<C, AX>(s);
                    __stcs(Kline + (n * N + i) * C::HP, fma(sc, V[s][i], K0[n * PLANE + i * S]));
                }
        } else {
            const double rkB = bi->rkB;
            const bool storeK = bi->storeK != 0;
            double *tz_out = bi->tz_out;
            double Qn[LAM ? NV : 1][N];
#pragma unroll
            for (int s = 0; s < NV; ++s) {
                const int n = var_of_slot<C, AX>(s);
                const int sq = LAM ? s : 0;
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    const double Kn = fma(sc, V[s][i], K0[n * PLANE + i * S]);
                    const double Qold = C::RELOAD ? Q0w[n * PLANE + i * S] : QL[C::RELOAD ? 0 : s][C::RELOAD ? 0 : i];
                    Qn[sq][i] = fma(rkB, Kn, Qold);
                    if (storeK) __stcs(Kline + (n * N + i) * C::HP, Kn);
                    Q0w[n * PLANE + i * S] = Qn[sq][i];
                }
                // PE for the z faces: traces of the updated Q, only at the two ends of the chunk
                if (first_layer) {
                    double tm = 0.0;
#pragma unroll
                    for (int i = 0; i < N; ++i) tm = fma(DG_LM(i), Qn[sq][i], tm);
                    tz_out[n * Ca + g.c] = tm;
                    if (BC && bi->push_z[0]) bi->push_z[0][n * Ca + g.c] = tm;
                }
                if (last_layer) {
                    double tp = 0.0;
#pragma unroll
                    for (int i = 0; i < N; ++i) tp = fma(DG_LP(i), Qn[sq][i], tp);
                    tz_out[(NV + n) * Ca + g.c] = tp;
                    if (BC && bi->push_z[1]) bi->push_z[1][n * Ca + g.c] = tp;
                }
            }
            if (LAM) {
                // max wavespeed of the updated state (reading R10) with the kernels' own reciprocal and
                // square root (a few ulp; the IEEE routines' slow paths cost 4 % of a step here); slots are
                // (rho, rho w, rho u, rho v, rho E): the speed does not care about the rotation.  A negative
                // density or pressure still gives NaN (the seeds of rcp / rsqrt propagate it).
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    const double rinv = rcp_pos(Qn[0][i]);
                    const double m2 = fma(Qn[LAM ? 3 : 0][i], Qn[LAM ? 3 : 0][i],
                                          fma(Qn[LAM ? 2 : 0][i], Qn[LAM ? 2 : 0][i], Qn[LAM ? 1 : 0][i] * Qn[LAM ? 1 : 0][i]));
                    const double pres = gm1 * fma(-0.5, m2 * rinv, Qn[LAM ? 4 : 0][i]);
                    const double um = (m2 > 1e-280) ? sqrt_pos(m2) * rinv : 0.0;   // fluid at rest: the seed of 0 is inf
                    const double sp = um + sqrt_pos(gamma * pres * rinv);
                    if (sp > lam_best || sp != sp) lam_best = sp;   // NaN sticks
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// the copy warp: every byte of Q and K between HBM and shared memory moves here, by the TMA engine
// ------------------------------------------------------------------------------------------------
// A layer slot is one contiguous block on both sides: one bulk copy each way, issued by one lane.
template <class C>
__device__ __forceinline__ void copy_in(double *sdst, const double *gsrc, uint64_t *bar, int lane) {
    constexpr unsigned BYTES = C::NPL * C::HP * 8;
    if (lane != 0) return;
    mbar_expect_tx(bar, BYTES);
    bulk_load(sdst, gsrc, BYTES, bar);
}
template <class C>
__device__ __forceinline__ void copy_out(double *gdst, const double *ssrc, int lane) {
    if (lane == 0) bulk_store(gdst, ssrc, C::NPL * C::HP * 8);
}

template <class C, int MODE, bool BC>
__device__ __forceinline__ void copy_warp(const DgStageArgs &a, const BlockInfo *bi, int lane, int bxi, int byi, int z0, int nl,
                                          bool readK, double *Qb0, double *Qb1, double *KR, uint64_t *fullq, uint64_t *fullk) {
    const size_t lstride = (size_t)a.nbx * a.nby;                    // slots per layer
    const size_t slot0 = (size_t)z0 * lstride + (size_t)byi * a.nbx + bxi;
    // (the loads of the first two Q layers and of the first K layer were issued in the kernel's prologue; the K
    // loads of later layers are issued by the compute warps)
    // L2 prefetch of the neighbour columns' traces of the first layer (4 blocks of 5 Ca doubles)
    if (lane < 4) l2_prefetch(bi->halo[lane], DG_NV * (lane < 2 ? C::CX : C::CY) * 8);
    for (int it = 0; it < nl; ++it) {
        double *Qcur = (it & 1) ? Qb1 : Qb0;
        const size_t slot = slot0 + (size_t)it * lstride;
        bar_sync<C::THREADS>(2);                                     // the compute warps are done with layer `it`
        if (MODE == DG_MODE_STAGE) {
            copy_out<C>(a.Q + slot * C::SLOT, Qcur, lane);
            bulk_commit();
            if (C::XPE) {
                // PE of the x axis, done by this otherwise idle warp while the bulk store reads the same buffer: the x
                // traces of the updated Q on the column boundary (the compute warps have gone on to the next layer)
                const int ext0 = bi->ext0, ext1 = bi->ext1;
                double *Tslot = bi->txy_out + (long long)it * bi->tstride;
                for (int r = lane; r < C::NCOMP; r += 32) {
                    const Geo gx = make_geo<C, 0>(r);
                    boundary_traces<C, 0>(gx, gx.ok && line_inside<C, 0>(gx, ext0, ext1), ext0, Qcur, Tslot,
                                          (BC && bi->push[0]) ? bi->push[0] + it * bi->pstride[0] : nullptr,
                                          (BC && bi->push[1]) ? bi->push[1] + it * bi->pstride[1] : nullptr);
                    const Geo gy = make_geo<C, 1>(r);
                    boundary_traces<C, 1>(gy, gy.ok && line_inside<C, 1>(gy, ext0, ext1), ext1, Qcur, Tslot,
                                          (BC && bi->push[2]) ? bi->push[2] + it * bi->pstride[2] : nullptr,
                                          (BC && bi->push[3]) ? bi->push[3] + it * bi->pstride[3] : nullptr);
                }
            }
            bulk_wait_read();                                        // shared memory has been read out
            __syncwarp();
        }
        if (it + 2 < nl) copy_in<C>(Qcur, a.Q + (slot + 2 * lstride) * C::SLOT, &fullq[it & 1], lane);
    }
}

// ------------------------------------------------------------------------------------------------
// one layer of the sweep, as a function of its own
// ------------------------------------------------------------------------------------------------
// NOT inlined on purpose: inside the layer loop of the kernel ptxas treats the ~(N^2 + 2N) operator-table loads
// as loop invariants, hoists them out, overflows the uniform register file and brings them back through local
// memory (measured: 50 spill slots per DOF, 29 % of the stall samples).  As a function with no loop of its own
// the body compiles as it did when a block owned one brick.  Everything it needs comes from shared memory.
template <class C>
struct Smem {
    static constexpr int QB0 = 0, QB1 = C::BUF, KR = 2 * C::BUF, TMS = 3 * C::BUF, FSS = TMS + C::LINEBUF,
                         FMS = FSS + C::LINEBUF, INFO = FMS + ((DG_NV * C::L + 1) & ~1), BARS = INFO + (int)((sizeof(BlockInfo) + 15) / 16 * 2),
                         DOUBLES = BARS + 4;
    static constexpr int BYTES = DOUBLES * 8;
};

template <class C, int MODE, bool LAM, bool BC>
__device__ __noinline__ double layer_body(int it, double lam_best) {
    extern __shared__ __align__(128) double smem[];
    using SM = Smem<C>;
    constexpr int L = C::L;
    const BlockInfo *bi = reinterpret_cast<const BlockInfo *>(smem + SM::INFO);
    uint64_t *fullq = reinterpret_cast<uint64_t *>(smem + SM::BARS), *fullk = fullq + 2;
    double *Qs = smem + ((it & 1) ? SM::QB1 : SM::QB0);
    const double *Qnext = smem + ((it & 1) ? SM::QB0 : SM::QB1);
    double *KR = smem + SM::KR, *Tms = smem + SM::TMS, *Fss = smem + SM::FSS, *FmS = smem + SM::FMS;
    const int l = threadIdx.x, lx = min(l, L - 1);
    const int ext0 = bi->ext0, ext1 = bi->ext1;
    const long long toff = (long long)it * bi->tstride;
    mbar_wait(&fullq[it & 1], (it >> 1) & 1);
    {
        const Geo gx = make_geo<C, 0>(l);
        xy_pass<C, 0, MODE, BC>(bi, gx, gx.ok && line_inside<C, 0>(gx, ext0, ext1), ext0, bi->halo[0] + it * bi->hstride[0],
                                bi->halo[1] + it * bi->hstride[1], Qs,
                            KR, Tms, Fss, fullk, it & 1);
    }
    {
        const Geo gy = make_geo<C, 1>(l);
        xy_pass<C, 1, MODE, BC>(bi, gy, gy.ok && line_inside<C, 1>(gy, ext0, ext1), ext1, bi->halo[2] + it * bi->hstride[2],
                                bi->halo[3] + it * bi->hstride[3], Qs,
                            KR, Tms, Fss, fullk, it & 1);
    }
    if (C::YSPLIT) {
        __syncwarp();
        if ((l & 31) == 0) mbar_arrive(fullk + 1);   // this warp's y pass is done (`ydone`, counted in warps)
    }
    const bool last_layer = it + 1 == bi->nl;
    // Ask L2 for what the NEXT layer reads with a short lead (about a third of a layer): its K slot, which the
    // copy warp can only fetch once this layer's K has left shared memory, and the neighbour columns' traces.
    // Asked for earlier, L2 has evicted them again by the time they are used (measured: +25 % DRAM reads).
    if (!last_layer && l < 5) {
        if (l < 4) l2_prefetch(bi->halo[l] + (it + 1) * bi->hstride[l], DG_NV * (l < 2 ? C::CX : C::CY) * 8);
        else if (bi->readK) l2_prefetch(bi->kslot + (long long)(it + 1) * bi->kstride, C::NPL * C::HP * 8);
    }
    if (!last_layer) mbar_wait(&fullq[(it + 1) & 1], ((it + 1) >> 1) & 1);
    {
        const Geo gz = make_geo<C, 2>(l);
        z_pass<C, MODE, LAM, BC>(bi, gz, lx, gz.ok && line_inside<C, 2>(gz, ext0, ext1), Qs, Qnext, KR, FmS,
                             bi->kslot + (long long)it * bi->kstride, it == 0, last_layer, fullk + 1, it & 1, lam_best);
    }
    bar_sync<C::NCOMP>(1);   // the updated Q of the whole layer is in shared memory; every line has read KR
    if (MODE == DG_MODE_STAGE) {
        // the next layer's K can come in now (needed at the end of its x pass)
        if (l < 32 && bi->readK && !last_layer) copy_in<C>(KR, bi->kslot + (long long)(it + 1) * bi->kstride, fullk, l);
        double *Tslot = bi->txy_out + toff;
        const Geo gx = make_geo<C, 0>(l), gy = make_geo<C, 1>(l);
        // (push mode runs the BC instances: the periodic, single-context instances carry none of this)
        if (!C::XPE)
            boundary_traces<C, 0>(gx, gx.ok && line_inside<C, 0>(gx, ext0, ext1), ext0, Qs, Tslot,
                                  (BC && bi->push[0]) ? bi->push[0] + it * bi->pstride[0] : nullptr,
                                  (BC && bi->push[1]) ? bi->push[1] + it * bi->pstride[1] : nullptr);
        if (!C::XPE)
            boundary_traces<C, 1>(gy, gy.ok && line_inside<C, 1>(gy, ext0, ext1), ext1, Qs, Tslot,
                                  (BC && bi->push[2]) ? bi->push[2] + it * bi->pstride[2] : nullptr,
                                  (BC && bi->push[3]) ? bi->push[3] + it * bi->pstride[3] : nullptr);
    }
    fence_proxy_async();
    bar_arrive<C::THREADS>(2);   // hand the layer to the copy warp
    return lam_best;
}

// ------------------------------------------------------------------------------------------------
// the fused stage kernel: block (bx, by, chunk) marches through layers z0 .. z0 + nl - 1 of column (bx, by)
// ------------------------------------------------------------------------------------------------
// BC = false: every domain face periodic (the paper's benchmark; no boundary code in the instance).
template <class C, int MODE, bool LAM, bool BC>
__global__ void __launch_bounds__(C::THREADS, C::MINB) dg_stage_kernel(const __grid_constant__ DgStageArgs a) {
    extern __shared__ __align__(128) double smem[];
    using SM = Smem<C>;
    uint64_t *fullq = reinterpret_cast<uint64_t *>(smem + SM::BARS), *fullk = fullq + 2;
    const int tid = threadIdx.x;
    const int bxi = blockIdx.x, byi = blockIdx.y, chunk = blockIdx.z;
    const int z0 = chunk * a.lz;
    const int nl = min(a.lz, a.nz - z0);
    const bool readK = (MODE == DG_MODE_STAGE) && (a.rkA != 0.0);
    if (tid == C::NCOMP) {
        // the copy warp's first lane sets the mbarriers up and sends the first bulk loads off at once, while thread 0
        // fills BlockInfo: the loads' latency overlaps the block's prologue
        mbar_init(&fullq[0], 1);
        mbar_init(&fullq[1], 1);
        mbar_init(fullk, 1);
        mbar_init(fullk + 1, C::NCOMP / 32);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const size_t lstride = (size_t)a.nbx * a.nby;
        const size_t slot0 = (size_t)z0 * lstride + (size_t)byi * a.nbx + bxi;
        copy_in<C>(smem + SM::QB0, a.Q + slot0 * C::SLOT, &fullq[0], 0);
        if (readK) copy_in<C>(smem + SM::KR, a.K + slot0 * C::SLOT, fullk, 0);
        if (nl > 1) copy_in<C>(smem + SM::QB1, a.Q + (slot0 + lstride) * C::SLOT, &fullq[1], 0);
    }
    if (tid == 0) {
        BlockInfo *bi = reinterpret_cast<BlockInfo *>(smem + SM::INFO);
        const size_t cstride = (size_t)a.nbx * a.nby, col = (size_t)byi * a.nbx + bxi;
        // neighbour columns' traces: the periodic neighbour's Txy block, or (block decomposition over GPUs) the
        // caller's halo buffer of that domain face
        bi->halo[0] = halo_source<C, 0>(a.Txy_old, a.nbx, a.nby, bxi, byi, z0, 0);
        bi->halo[1] = halo_source<C, 0>(a.Txy_old, a.nbx, a.nby, bxi, byi, z0, 1);
        bi->halo[2] = halo_source<C, 1>(a.Txy_old, a.nbx, a.nby, bxi, byi, z0, 0);
        bi->halo[3] = halo_source<C, 1>(a.Txy_old, a.nbx, a.nby, bxi, byi, z0, 1);
        for (int f = 0; f < 4; ++f) bi->hstride[f] = (long long)cstride * C::TXY;
        if (a.halo_ext[0] && bxi == 0) { bi->halo[0] = a.halo_ext[0] + ((size_t)z0 * a.nby + byi) * (DG_NV * C::CX); bi->hstride[0] = (long long)a.nby * (DG_NV * C::CX); }
        if (a.halo_ext[1] && bxi + 1 == a.nbx) { bi->halo[1] = a.halo_ext[1] + ((size_t)z0 * a.nby + byi) * (DG_NV * C::CX); bi->hstride[1] = (long long)a.nby * (DG_NV * C::CX); }
        if (a.halo_ext[2] && byi == 0) { bi->halo[2] = a.halo_ext[2] + ((size_t)z0 * a.nbx + bxi) * (DG_NV * C::CY); bi->hstride[2] = (long long)a.nbx * (DG_NV * C::CY); }
        if (a.halo_ext[3] && byi + 1 == a.nby) { bi->halo[3] = a.halo_ext[3] + ((size_t)z0 * a.nbx + bxi) * (DG_NV * C::CY); bi->hstride[3] = (long long)a.nbx * (DG_NV * C::CY); }
        bi->txy_out = a.Txy_new + ((size_t)z0 * cstride + col) * C::TXY;
        // z traces at the ends of the chunk: T+ of the chunk below (its side 1), T- of the chunk above (its side 0)
        const int clo = (chunk == 0) ? a.nchunks - 1 : chunk - 1, chi = (chunk + 1 == a.nchunks) ? 0 : chunk + 1;
        bi->tz_lo = a.Tz_old + ((size_t)clo * cstride + col) * C::TZ + DG_NV * C::CZ;
        bi->tz_hi = a.Tz_old + ((size_t)chi * cstride + col) * C::TZ;
        if (a.halo_ext[4] && chunk == 0) bi->tz_lo = a.halo_ext[4] + col * (DG_NV * C::CZ);
        if (a.halo_ext[5] && chunk + 1 == a.nchunks) bi->tz_hi = a.halo_ext[5] + col * (DG_NV * C::CZ);
        bi->tz_out = a.Tz_new + ((size_t)chunk * cstride + col) * C::TZ;
        // push mode: the same blocks of the neighbour contexts' halo buffers that those contexts read (layout of halo_ext)
        for (int f = 0; f < 4; ++f) bi->push[f] = nullptr;
        if (a.halo_push[0] && bxi == 0) { bi->push[0] = a.halo_push[0] + ((size_t)z0 * a.nby + byi) * (DG_NV * C::CX); bi->pstride[0] = (long long)a.nby * (DG_NV * C::CX); }
        if (a.halo_push[1] && bxi + 1 == a.nbx) { bi->push[1] = a.halo_push[1] + ((size_t)z0 * a.nby + byi) * (DG_NV * C::CX); bi->pstride[1] = (long long)a.nby * (DG_NV * C::CX); }
        if (a.halo_push[2] && byi == 0) { bi->push[2] = a.halo_push[2] + ((size_t)z0 * a.nbx + bxi) * (DG_NV * C::CY); bi->pstride[2] = (long long)a.nbx * (DG_NV * C::CY); }
        if (a.halo_push[3] && byi + 1 == a.nby) { bi->push[3] = a.halo_push[3] + ((size_t)z0 * a.nbx + bxi) * (DG_NV * C::CY); bi->pstride[3] = (long long)a.nbx * (DG_NV * C::CY); }
        bi->push_z[0] = (a.halo_push[4] && chunk == 0) ? a.halo_push[4] + col * (DG_NV * C::CZ) : nullptr;
        bi->push_z[1] = (a.halo_push[5] && chunk + 1 == a.nchunks) ? a.halo_push[5] + col * (DG_NV * C::CZ) : nullptr;
        bi->tstride = (long long)cstride * C::TXY;
        bi->kslot = a.K + ((size_t)z0 * cstride + col) * C::SLOT;
        bi->kstride = (long long)cstride * C::SLOT;
        bi->gamma = a.gamma;
        bi->gm1 = a.gm1;
        bi->rkA = a.rkA;
        bi->rkB = a.rkB;
        double dtf = 1.0;
        if (a.lam_in) {   // CFL time step from the wavespeed reduced on the device (reading R10)
            dtf = a.cfl_factor / __longlong_as_double((long long)*a.lam_in);
            if (a.t_acc && bxi == 0 && byi == 0 && chunk == 0) {
                a.t_acc[0] += dtf;
                a.t_acc[1] = dtf;
            }
        }
        bi->scale[0] = a.scale[0] * dtf;
        bi->scale[1] = a.scale[1] * dtf;
        bi->scale[2] = a.scale[2] * dtf;
        bi->ext0 = min(C::BX, a.nx - bxi * C::BX);   // elements of this column per axis (ragged last column)
        bi->ext1 = min(C::BY, a.ny - byi * C::BY);
        bi->readK = readK ? 1 : 0;
        bi->storeK = a.store_k;
        bi->bc[0] = (bxi == 0) ? a.bc[0] : 0;
        bi->bc[1] = (bxi + 1 == a.nbx) ? a.bc[1] : 0;
        bi->bc[2] = (byi == 0) ? a.bc[2] : 0;
        bi->bc[3] = (byi + 1 == a.nby) ? a.bc[3] : 0;
        bi->bc[4] = (chunk == 0) ? a.bc[4] : 0;
        bi->bc[5] = (chunk + 1 == a.nchunks) ? a.bc[5] : 0;
        for (int n = 0; n < DG_NV; ++n) bi->qinf[n] = a.qinf[n];
        bi->nl = nl;
    }
    __syncthreads();
    if (tid >= C::NCOMP) {
        copy_warp<C, MODE, BC>(a, reinterpret_cast<const BlockInfo *>(smem + SM::INFO), tid - C::NCOMP, bxi, byi, z0, nl, readK, smem + SM::QB0, smem + SM::QB1, smem + SM::KR, fullq,
                           fullk);
        return;
    }
    double lam_best = 0.0;
#pragma unroll 1
    for (int it = 0; it < nl; ++it) lam_best = layer_body<C, MODE, LAM, BC>(it, lam_best);
    if (LAM) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            const double o = __shfl_xor_sync(0xffffffffu, lam_best, off);
            if (o > lam_best || o != o) lam_best = o;
        }
        if ((tid & 31) == 0) atomicMax(a.lam_bits, (unsigned long long)__double_as_longlong(lam_best));
    }
}

// ------------------------------------------------------------------------------------------------
// face traces of a freshly set state (after dg_set_state): one block per layer slot
// ------------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(C::NCOMP) dg_traces_kernel(const __grid_constant__ DgTraceArgs a) {
    constexpr int NV = DG_NV, N = C::N;
    extern __shared__ __align__(128) double smem[];
    const int tid = threadIdx.x, bxi = blockIdx.x, byi = blockIdx.y, ez = blockIdx.z;
    const size_t cstride = (size_t)a.nbx * a.nby, col = (size_t)byi * a.nbx + bxi;
    const size_t slot = (size_t)ez * cstride + col;
    const double *src = a.Q + slot * C::SLOT;
    for (int idx = tid; idx < C::NPL * C::HP; idx += C::NCOMP) {
        const int pl = idx / C::HP;
        smem[pl * C::PP + (idx - pl * C::HP)] = src[idx];
    }
    __syncthreads();
    const Geo gx = make_geo<C, 0>(tid), gy = make_geo<C, 1>(tid), gz = make_geo<C, 2>(tid);
    const int ext0 = min(C::BX, a.nx - bxi * C::BX), ext1 = min(C::BY, a.ny - byi * C::BY);
    double *Tslot = a.Txy + slot * C::TXY;
    boundary_traces<C, 0>(gx, gx.ok && line_inside<C, 0>(gx, ext0, ext1), ext0, smem, Tslot);
    boundary_traces<C, 1>(gy, gy.ok && line_inside<C, 1>(gy, ext0, ext1), ext1, smem, Tslot);
    const int chunk = ez / a.lz;
    const bool zfirst = ez == chunk * a.lz, zlast = (ez + 1 == a.nz) || (ez + 1 == (chunk + 1) * a.lz);
    if ((zfirst || zlast) && gz.ok && line_inside<C, 2>(gz, ext0, ext1)) {
        double *dst = a.Tz + ((size_t)chunk * cstride + col) * C::TZ + gz.c;
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            double tp = 0.0, tm = 0.0;
#pragma unroll
            for (int q = 0; q < N; ++q) {
                const double Qv = smem[n * C::PLANE + gz.base + q * C::PP];
                tp = fma(DG_LP(q), Qv, tp);
                tm = fma(DG_LM(q), Qv, tm);
            }
            if (zfirst) dst[n * C::CZ] = tm;
            if (zlast) dst[(NV + n) * C::CZ] = tp;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// paper-shaped per-kernel mode (Table II): the volume kernel (K1) and the
// surface kernel (K2) as launches of their own over the same layout; one block per layer slot, one thread per
// node line and axis.  Not the hot path: it exists to print the paper's per-kernel breakdown next to the fused
// step and is parity-tested against the oracle's volume and surface terms.
// ------------------------------------------------------------------------------------------------
template <class C>
__device__ __forceinline__ void stage_layer_in(double *smem_dst, const double *gsrc, int tid) {
    for (int idx = tid; idx < C::NPL * C::HP; idx += C::NCOMP) smem_dst[idx] = gsrc[idx];
}

// R <- sum over the axes of (2/h_a) sum_q Dhat_iq F^a_q   (eq (5) 2nd term / mass; overwrites R like the listing)
template <class C>
__global__ void __launch_bounds__(C::NCOMP) dg_split_volume_kernel(const __grid_constant__ DgSplitArgs a) {
    constexpr int NV = DG_NV, N = C::N, PLANE = C::PLANE;
    extern __shared__ __align__(128) double smem[];
    double *Qs = smem, *Rs = smem + C::BUF;
    const int tid = threadIdx.x, bxi = blockIdx.x, byi = blockIdx.y, ez = blockIdx.z;
    const size_t slot = ((size_t)ez * a.nby + byi) * a.nbx + bxi;
    stage_layer_in<C>(Qs, a.Q + slot * C::SLOT, tid);
    __syncthreads();
    const int ext0 = min(C::BX, a.nx - bxi * C::BX), ext1 = min(C::BY, a.ny - byi * C::BY);
    auto axis = [&](auto AXT) {
        constexpr int AX = decltype(AXT)::value;
        using A = Axis<C, AX>;
        const Geo g = make_geo<C, AX>(tid);
        const bool act = g.ok && line_inside<C, AX>(g, ext0, ext1);
        double V[NV][N];
#pragma unroll
        for (int q = 0; q < N; ++q) {
            double Qn[NV], F[NV], vel, pres, rinv;
#pragma unroll
            for (int s = 0; s < NV; ++s) Qn[s] = Qs[g.base + var_of_slot<C, AX>(s) * PLANE + q * A::S];
            euler_flux_normal(Qn, a.gm1, F, vel, pres, rinv);
#pragma unroll
            for (int n = 0; n < NV; ++n)
#pragma unroll
                for (int i = 0; i < N; ++i) V[n][i] = (q == 0) ? c_ref.D[q][i] * F[n] : fma(c_ref.D[q][i], F[n], V[n][i]);
        }
        if (act) {
#pragma unroll
            for (int s = 0; s < NV; ++s)
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    double *p = Rs + g.base + var_of_slot<C, AX>(s) * PLANE + i * A::S;
                    *p = (AX == 0) ? a.scale[AX] * V[s][i] : fma(a.scale[AX], V[s][i], *p);
                }
        }
        __syncthreads();
    };
    axis(std::integral_constant<int, 0>{});
    axis(std::integral_constant<int, 1>{});
    axis(std::integral_constant<int, 2>{});
    double *dst = a.R + slot * C::SLOT;
    for (int idx = tid; idx < C::NPL * C::HP; idx += C::NCOMP) dst[idx] = Rs[idx];
}

// Trace of the line through node (j, k transverse) of element (ex, ey, ez) along axis AX, at its + or - end,
// read from the state in HBM (any element of the mesh; periodic wrap by the caller), slots rotated for AX.
template <class C, int AX>
__device__ __forceinline__ void global_line_trace_of(const double *field, int nbx, int nby, int ex, int ey, int ez, int t1, int t2,
                                                     bool plus, double (&T)[DG_NV]) {
    constexpr int N = C::N;
    const int bxi = ex / C::BX, byi = ey / C::BY;
    const int lx = ex - bxi * C::BX, ly = ey - byi * C::BY;
    const double *src = field + (((size_t)ez * nby + byi) * nbx + bxi) * C::SLOT;
    // (t1, t2) are node indices INSIDE the element here: x lines (j, k), y lines (i, k), z lines (i, j)
    int base, stride;
    if (AX == 0) { base = t2 * C::HP + (ly * N + t1) * C::GX + lx * N; stride = 1; }
    else if (AX == 1) { base = t2 * C::HP + (ly * N) * C::GX + lx * N + t1; stride = C::GX; }
    else { base = (ly * N + t2) * C::GX + lx * N + t1; stride = C::HP; }
#pragma unroll
    for (int s = 0; s < DG_NV; ++s) {
        double t = 0.0;
        const double *p = src + var_of_slot<C, AX>(s) * (N * C::HP) + base;
#pragma unroll
        for (int q = 0; q < N; ++q) t = fma(plus ? DG_LP(q) : DG_LM(q), __ldg(p + q * stride), t);
        T[s] = t;
    }
}

template <class C, int AX>
__device__ __forceinline__ void global_line_trace(const DgSplitArgs &a, int ex, int ey, int ez, int t1, int t2, bool plus,
                                                  double (&T)[DG_NV]) {
    global_line_trace_of<C, AX>(a.Q, a.nbx, a.nby, ex, ey, ez, t1, t2, plus, T);
}

// R += -(2/h_a) (l_i(+1) F*_+ - l_i(-1) F*_-)/w_i for the three axes: every line evaluates the local Lax-Friedrichs
// flux at both of its ends from its own traces and the two neighbour elements' (eq (5) 3rd term / mass)
template <class C>
__global__ void __launch_bounds__(C::NCOMP) dg_split_surface_kernel(const __grid_constant__ DgSplitArgs a) {
    constexpr int NV = DG_NV, N = C::N, PLANE = C::PLANE;
    extern __shared__ __align__(128) double smem[];
    double *Qs = smem, *Rs = smem + C::BUF;
    const int tid = threadIdx.x, bxi = blockIdx.x, byi = blockIdx.y, ez = blockIdx.z;
    const size_t slot = ((size_t)ez * a.nby + byi) * a.nbx + bxi;
    stage_layer_in<C>(Qs, a.Q + slot * C::SLOT, tid);
    stage_layer_in<C>(Rs, a.R + slot * C::SLOT, tid);
    __syncthreads();
    const int ext0 = min(C::BX, a.nx - bxi * C::BX), ext1 = min(C::BY, a.ny - byi * C::BY);
    auto axis = [&](auto AXT) {
        constexpr int AX = decltype(AXT)::value;
        using A = Axis<C, AX>;
        const Geo g = make_geo<C, AX>(tid);
        const bool act = g.ok && line_inside<C, AX>(g, ext0, ext1);
        if (act) {
            double Tp[NV], Tm[NV], Hlo[NV], Hhi[NV], Fp[NV], Fm[NV];
#pragma unroll
            for (int s = 0; s < NV; ++s) {
                Tp[s] = Tm[s] = 0.0;
#pragma unroll
                for (int q = 0; q < N; ++q) {
                    const double Qv = Qs[g.base + var_of_slot<C, AX>(s) * PLANE + q * A::S];
                    Tp[s] = fma(DG_LP(q), Qv, Tp[s]);
                    Tm[s] = fma(DG_LM(q), Qv, Tm[s]);
                }
            }
            // this line's element and its two neighbours along AX (periodic), node indices in the element
            int ex = bxi * C::BX, ey = byi * C::BY, e2 = ez, n1, n2;
            if (AX == 0) { ex += g.e; ey += g.t1 / N; n1 = g.t1 % N; n2 = g.t2; }
            else if (AX == 1) { ey += g.e; ex += g.t1 / N; n1 = g.t1 % N; n2 = g.t2; }
            else { ex += g.t1 / N; ey += g.t2 / N; n1 = g.t1 % N; n2 = g.t2 % N; }
            const int na = (AX == 0) ? a.nx : (AX == 1) ? a.ny : a.nz;
            const int ea = (AX == 0) ? ex : (AX == 1) ? ey : e2;
            const int up = (ea + 1 == na) ? 0 : ea + 1, dn = (ea == 0) ? na - 1 : ea - 1;
            global_line_trace<C, AX>(a, AX == 0 ? up : ex, AX == 1 ? up : ey, AX == 2 ? up : e2, n1, n2, false, Hhi);
            global_line_trace<C, AX>(a, AX == 0 ? dn : ex, AX == 1 ? dn : ey, AX == 2 ? dn : e2, n1, n2, true, Hlo);
            lax_friedrichs2(Tp, Hhi, 1.0, a.gamma, a.gm1, Fp);
            lax_friedrichs2(Tm, Hlo, -1.0, a.gamma, a.gm1, Fm);
#pragma unroll
            for (int s = 0; s < NV; ++s)
#pragma unroll
                for (int i = 0; i < N; ++i) {
                    double *p = Rs + g.base + var_of_slot<C, AX>(s) * PLANE + i * A::S;
                    *p = fma(a.scale[AX], fma(DG_LQM(i), Fm[s], -DG_LQP(i) * Fp[s]), *p);
                }
        }
        __syncthreads();
    };
    axis(std::integral_constant<int, 0>{});
    axis(std::integral_constant<int, 1>{});
    axis(std::integral_constant<int, 2>{});
    double *dst = a.R + slot * C::SLOT;
    for (int idx = tid; idx < C::NPL * C::HP; idx += C::NCOMP) dst[idx] = Rs[idx];
}

// ------------------------------------------------------------------------------------------------
// viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4.  The paper names them only and prints no equations:
// DESIGN.md reading R20 -- constant viscosity, Stokes hypothesis, Fourier conduction with constant Prandtl number,
// first Bassi-Rebay scheme in the basis of eq (4)-(7), periodic meshes.  Run as kernels of their own on top of the
// per-kernel mode (not the fused hot path):
//   cwd_axis ("central weak derivative")  (2/h_a) [ (l_i(+1) G*_+ - l_i(-1) G*_-)/w_i - sum_q Dhat_iq G_q ] along one axis
//                       with the CENTRAL interface value G* = (G_L + G_R)/2: the weak form of eq (5) for d_a G.  Applied to
//                       Q it gives the gradient S_a, applied to the nodal viscous flux Fv_a it gives div Fv.
//   dg_visc_gradflux_kernel  S_x, S_y, S_z of a layer slot into shared memory, then pointwise (velocity and p/rho gradients
//                       from S by the quotient rule) the viscous fluxes Fv_a -> three vectors in HBM
//   dg_visc_div_kernel  R += d_x Fv_x + d_y Fv_y + d_z Fv_z, the slot of R accumulated in shared memory
// ------------------------------------------------------------------------------------------------
// One line of the central weak derivative along AX: Gs = the block's own layer slot of the field in shared memory, Gg = the
// whole field in HBM (the two neighbour elements' traces), o = this slot's output (shared or global memory, slot layout).
template <class C, int AX>
__device__ __forceinline__ void cwd_axis(const DgViscArgs &a, const double *Gs, const double *Gg, double *o, bool accumulate,
                                         double scale, int tid, int bxi, int byi, int ez) {
    using A = Axis<C, AX>;
    constexpr int NV = DG_NV, N = C::N, PLANE = C::PLANE;
    const int ext0 = min(C::BX, a.nx - bxi * C::BX), ext1 = min(C::BY, a.ny - byi * C::BY);
    const Geo g = make_geo<C, AX>(tid);
    if (!g.ok || !line_inside<C, AX>(g, ext0, ext1)) return;
    double Gl[NV][N], Tp[NV], Tm[NV], Hlo[NV], Hhi[NV];
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        Tp[n] = Tm[n] = 0.0;
#pragma unroll
        for (int q = 0; q < N; ++q) {
            const double v = Gs[g.base + n * PLANE + q * A::S];
            Gl[n][q] = v;
            Tp[n] = fma(DG_LP(q), v, Tp[n]);
            Tm[n] = fma(DG_LM(q), v, Tm[n]);
        }
    }
    // this line's element and its two neighbours along AX (periodic), node indices in the element
    int ex = bxi * C::BX, ey = byi * C::BY, n1, n2;
    if (AX == 0) { ex += g.e; ey += g.t1 / N; n1 = g.t1 % N; n2 = g.t2; }
    else if (AX == 1) { ey += g.e; ex += g.t1 / N; n1 = g.t1 % N; n2 = g.t2; }
    else { ex += g.t1 / N; ey += g.t2 / N; n1 = g.t1 % N; n2 = g.t2 % N; }
    const int na = (AX == 0) ? a.nx : (AX == 1) ? a.ny : a.nz;
    const int ea = (AX == 0) ? ex : (AX == 1) ? ey : ez;
    const int up = (ea + 1 == na) ? 0 : ea + 1, dn = (ea == 0) ? na - 1 : ea - 1;
    // identity slots here (no momentum rotation): global_line_trace_of returns slot s = variable var_of_slot(s)
    double Ru[NV], Rd[NV];
    global_line_trace_of<C, AX>(Gg, a.nbx, a.nby, AX == 0 ? up : ex, AX == 1 ? up : ey, AX == 2 ? up : ez, n1, n2, false, Ru);
    global_line_trace_of<C, AX>(Gg, a.nbx, a.nby, AX == 0 ? dn : ex, AX == 1 ? dn : ey, AX == 2 ? dn : ez, n1, n2, true, Rd);
#pragma unroll
    for (int s = 0; s < NV; ++s) {
        Hhi[var_of_slot<C, AX>(s)] = Ru[s];
        Hlo[var_of_slot<C, AX>(s)] = Rd[s];
    }
    o += g.base;
#pragma unroll
    for (int n = 0; n < NV; ++n) {
        const double sp = Tp[n] + Hhi[n], sm = Hlo[n] + Tm[n];   // 2 G*_+, 2 G*_-; c_ref.lq carries the 1/2 and 1/w
#pragma unroll
        for (int i = 0; i < N; ++i) {
            double v = fma(DG_LQP(i), sp, -DG_LQM(i) * sm);
#pragma unroll
            for (int q = 0; q < N; ++q) v = fma(-c_ref.D[q][i], Gl[n][q], v);
            double *dst = o + n * PLANE + i * A::S;
            *dst = accumulate ? fma(scale, v, *dst) : scale * v;
        }
    }
}

// steps v1 + v2 of reading R20 in one sweep: the three gradients S_a = d_a Q of the block's layer into shared memory, then
// the viscous fluxes Fv_a at the layer's nodes, written to the three vectors a.S[]
template <class C>
__global__ void __launch_bounds__(C::NCOMP) dg_visc_gradflux_kernel(const __grid_constant__ DgViscArgs a) {
    constexpr int NV = DG_NV, N = C::N, PLANE = C::PLANE;
    extern __shared__ __align__(128) double smem[];
    double *Qs = smem, *Ss = smem + C::BUF;   // Ss[d * BUF ...]
    const int tid = threadIdx.x, bxi = blockIdx.x, byi = blockIdx.y, ez = blockIdx.z;
    const size_t slot = ((size_t)ez * a.nby + byi) * a.nbx + bxi;
    stage_layer_in<C>(Qs, a.Q + slot * C::SLOT, tid);
    __syncthreads();
    cwd_axis<C, 0>(a, Qs, a.Q, Ss, false, a.scale3[0], tid, bxi, byi, ez);
    cwd_axis<C, 1>(a, Qs, a.Q, Ss + C::BUF, false, a.scale3[1], tid, bxi, byi, ez);
    cwd_axis<C, 2>(a, Qs, a.Q, Ss + 2 * C::BUF, false, a.scale3[2], tid, bxi, byi, ez);
    __syncthreads();
    // pointwise, one thread per z line of the layer
    const int ext0 = min(C::BX, a.nx - bxi * C::BX), ext1 = min(C::BY, a.ny - byi * C::BY);
    const Geo g = make_geo<C, 2>(tid);
    if (!g.ok || !line_inside<C, 2>(g, ext0, ext1)) return;
#pragma unroll 1
    for (int i = 0; i < N; ++i) {
        const int io = g.base + i * C::PP;
        double Q[NV], S[3][NV];
#pragma unroll
        for (int n = 0; n < NV; ++n) {
            Q[n] = Qs[io + n * PLANE];
#pragma unroll
            for (int d = 0; d < 3; ++d) S[d][n] = Ss[d * C::BUF + io + n * PLANE];
        }
        const double rinv = 1.0 / Q[0];
        const double u[3] = {Q[1] * rinv, Q[2] * rinv, Q[3] * rinv};
        const double E = Q[4] * rinv;
        double du[3][3], dT[3];   // du[d][b] = d_d u_b, dT[d] = d_d (p/rho)
#pragma unroll
        for (int d = 0; d < 3; ++d) {
#pragma unroll
            for (int b = 0; b < 3; ++b) du[d][b] = (S[d][1 + b] - u[b] * S[d][0]) * rinv;
            const double dE = (S[d][4] - E * S[d][0]) * rinv;
            dT[d] = a.gm1 * (dE - (u[0] * du[d][0] + u[1] * du[d][1] + u[2] * du[d][2]));
        }
        const double divu = du[0][0] + du[1][1] + du[2][2];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            double tau[3];
#pragma unroll
            for (int b = 0; b < 3; ++b) tau[b] = a.mu * (du[d][b] + du[b][d]);
            tau[d] -= a.mu * (2.0 / 3.0) * divu;
            double *o = a.S[d] + slot * C::SLOT + io;
            o[0] = 0.0;
            o[PLANE] = tau[0];
            o[2 * PLANE] = tau[1];
            o[3 * PLANE] = tau[2];
            o[4 * PLANE] = (u[0] * tau[0] + u[1] * tau[1] + u[2] * tau[2]) + a.kappa * dT[d];
        }
    }
}

// step v3: R += sum_a d_a Fv_a, the residual's layer slot accumulated in shared memory and written once
template <class C>
__global__ void __launch_bounds__(C::NCOMP) dg_visc_div_kernel(const __grid_constant__ DgViscArgs a) {
    extern __shared__ __align__(128) double smem[];
    double *Gs = smem, *Rs = smem + C::BUF;
    const int tid = threadIdx.x, bxi = blockIdx.x, byi = blockIdx.y, ez = blockIdx.z;
    const size_t slot = ((size_t)ez * a.nby + byi) * a.nbx + bxi;
    stage_layer_in<C>(Rs, a.out + slot * C::SLOT, tid);
    stage_layer_in<C>(Gs, a.S[0] + slot * C::SLOT, tid);
    __syncthreads();
    cwd_axis<C, 0>(a, Gs, a.S[0], Rs, true, a.scale3[0], tid, bxi, byi, ez);
    __syncthreads();
    stage_layer_in<C>(Gs, a.S[1] + slot * C::SLOT, tid);
    __syncthreads();
    cwd_axis<C, 1>(a, Gs, a.S[1], Rs, true, a.scale3[1], tid, bxi, byi, ez);
    __syncthreads();
    stage_layer_in<C>(Gs, a.S[2] + slot * C::SLOT, tid);
    __syncthreads();
    cwd_axis<C, 2>(a, Gs, a.S[2], Rs, true, a.scale3[2], tid, bxi, byi, ez);
    __syncthreads();
    double *dst = a.out + slot * C::SLOT;
    for (int idx = tid; idx < C::NPL * C::HP; idx += C::NCOMP) dst[idx] = Rs[idx];
}

// ------------------------------------------------------------------------------------------------
// layout conversion canonical [e][k][j][i][n] <-> internal [slot][n][k][HP: gy, gx]
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
    const int bxi = ex / C::BX, byi = ey / C::BY;
    const int gx = (ex - bxi * C::BX) * N + i, gy = (ey - byi * C::BY) * N + j;
    const size_t slot = (size_t)bxi + (size_t)nbx * ((size_t)byi + (size_t)nby * ez);
    return slot * C::SLOT + (size_t)k * C::HP + (size_t)(gy * C::GX + gx);
}

template <class C>
__global__ void __launch_bounds__(256) dg_layout_kernel(const DgLayoutArgs a) {
    constexpr size_t VS = (size_t)C::N * C::HP;   // doubles per variable inside a slot
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    for (size_t node = (size_t)blockIdx.x * blockDim.x + threadIdx.x; node < total;
         node += (size_t)gridDim.x * blockDim.x) {
        const size_t io = internal_offset<C>(node, a.nx, a.ny, a.nbx, a.nby);
        if (a.to_internal) {
#pragma unroll
            for (int n = 0; n < DG_NV; ++n) a.internal[io + n * VS] = a.canonical[node * DG_NV + n];
        } else {
#pragma unroll
            for (int n = 0; n < DG_NV; ++n) a.canonical[node * DG_NV + n] = a.internal[io + n * VS];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// max wavespeed  lam = max_nodes sqrt(u^2+v^2+w^2) + sqrt(gamma p / rho)   (reading R10)
// of a freshly set state (after a Runge-Kutta step the last stage has already reduced it)
// ------------------------------------------------------------------------------------------------
template <class C>
__global__ void __launch_bounds__(256) dg_wavespeed_kernel(const DgWaveArgs a) {
    constexpr size_t VS = (size_t)C::N * C::HP;
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    double best = 0.0;
    for (size_t node = (size_t)blockIdx.x * blockDim.x + threadIdx.x; node < total;
         node += (size_t)gridDim.x * blockDim.x) {
        const size_t io = internal_offset<C>(node, a.nx, a.ny, a.nbx, a.nby);
        const double Q0 = a.Q[io], Q1 = a.Q[io + VS], Q2 = a.Q[io + 2 * VS], Q3 = a.Q[io + 3 * VS], Q4 = a.Q[io + 4 * VS];
        const double rinv = 1.0 / Q0;
        const double u = Q1 * rinv, v = Q2 * rinv, w = Q3 * rinv;
        const double pres = a.gm1 * (Q4 - 0.5 * Q0 * (u * u + v * v + w * w));
        const double s = sqrt(u * u + v * v + w * w) + sqrt(a.gamma * pres * rinv);
        if (s > best || s != s) best = s;   // NaN sticks
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        const double o = __shfl_xor_sync(0xffffffffu, best, off);
        if (o > best || o != o) best = o;
    }
    if ((threadIdx.x & 31) == 0) atomicMax(a.lam_bits, (unsigned long long)__double_as_longlong(best));
}

// ------------------------------------------------------------------------------------------------
// host-side launchers, one table per variant
// ------------------------------------------------------------------------------------------------
template <class C>
cudaError_t prepare(const DgRefOps &ref, int *blocks_per_sm) {
    cudaError_t err = cudaMemcpyToSymbol(c_ref, &ref, sizeof(DgRefOps));
    auto opt_in = [&](auto kernel) {
        if (err == cudaSuccess) err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, Smem<C>::BYTES);
    };
    opt_in(dg_stage_kernel<C, DG_MODE_STAGE, false, false>);
    opt_in(dg_stage_kernel<C, DG_MODE_STAGE, true, false>);
    opt_in(dg_stage_kernel<C, DG_MODE_RESIDUAL, false, false>);
    opt_in(dg_stage_kernel<C, DG_MODE_STAGE, false, true>);
    opt_in(dg_stage_kernel<C, DG_MODE_STAGE, true, true>);
    opt_in(dg_stage_kernel<C, DG_MODE_RESIDUAL, false, true>);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_traces_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, C::BUF * 8);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_split_volume_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * C::BUF * 8);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_split_surface_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * C::BUF * 8);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_visc_gradflux_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, 4 * C::BUF * 8);
    if (err == cudaSuccess)
        err = cudaFuncSetAttribute(dg_visc_div_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, 2 * C::BUF * 8);
    if (err != cudaSuccess) return err;
    return cudaOccupancyMaxActiveBlocksPerMultiprocessor(blocks_per_sm, dg_stage_kernel<C, DG_MODE_STAGE, false, false>,
                                                         C::THREADS, Smem<C>::BYTES);
}

template <class C>
cudaError_t launch_stage(const DgStageArgs &a, cudaStream_t s) {
    const dim3 grid((unsigned)a.nbx, (unsigned)a.nby, (unsigned)a.nchunks);
    // the instances with boundary code also hold the push-mode stores
    const bool bc = a.bc[0] || a.bc[1] || a.bc[2] || a.bc[3] || a.bc[4] || a.bc[5] || a.halo_push[0] || a.halo_push[1] ||
                    a.halo_push[2] || a.halo_push[3] || a.halo_push[4] || a.halo_push[5];
    const size_t sm = Smem<C>::BYTES;
    if (a.mode == DG_MODE_RESIDUAL) {
        if (bc) dg_stage_kernel<C, DG_MODE_RESIDUAL, false, true><<<grid, C::THREADS, sm, s>>>(a);
        else dg_stage_kernel<C, DG_MODE_RESIDUAL, false, false><<<grid, C::THREADS, sm, s>>>(a);
    } else if (a.want_lam) {
        if (bc) dg_stage_kernel<C, DG_MODE_STAGE, true, true><<<grid, C::THREADS, sm, s>>>(a);
        else dg_stage_kernel<C, DG_MODE_STAGE, true, false><<<grid, C::THREADS, sm, s>>>(a);
    } else {
        if (bc) dg_stage_kernel<C, DG_MODE_STAGE, false, true><<<grid, C::THREADS, sm, s>>>(a);
        else dg_stage_kernel<C, DG_MODE_STAGE, false, false><<<grid, C::THREADS, sm, s>>>(a);
    }
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_traces(const DgTraceArgs &a, cudaStream_t s) {
    const dim3 grid((unsigned)a.nbx, (unsigned)a.nby, (unsigned)a.nz);
    dg_traces_kernel<C><<<grid, C::NCOMP, C::BUF * 8, s>>>(a);
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_split_volume(const DgSplitArgs &a, cudaStream_t s) {
    const dim3 grid((unsigned)a.nbx, (unsigned)a.nby, (unsigned)a.nz);
    dg_split_volume_kernel<C><<<grid, C::NCOMP, 2 * C::BUF * 8, s>>>(a);
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_split_surface(const DgSplitArgs &a, cudaStream_t s) {
    const dim3 grid((unsigned)a.nbx, (unsigned)a.nby, (unsigned)a.nz);
    dg_split_surface_kernel<C><<<grid, C::NCOMP, 2 * C::BUF * 8, s>>>(a);
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_visc_gradflux(const DgViscArgs &a, cudaStream_t s) {
    const dim3 grid((unsigned)a.nbx, (unsigned)a.nby, (unsigned)a.nz);
    dg_visc_gradflux_kernel<C><<<grid, C::NCOMP, 4 * C::BUF * 8, s>>>(a);
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_visc_div(const DgViscArgs &a, cudaStream_t s) {
    const dim3 grid((unsigned)a.nbx, (unsigned)a.nby, (unsigned)a.nz);
    dg_visc_div_kernel<C><<<grid, C::NCOMP, 2 * C::BUF * 8, s>>>(a);
    return cudaGetLastError();
}

inline unsigned flat_grid(size_t total, int sms) {
    const size_t want = (total + 255) / 256;
    const size_t cap = (size_t)(sms > 0 ? sms : 1) * 16u;   // grid-stride: a few blocks per SM
    return (unsigned)(want < cap ? (want ? want : 1) : cap);
}

template <class C>
cudaError_t launch_layout(const DgLayoutArgs &a, int sms, cudaStream_t s) {
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    dg_layout_kernel<C><<<flat_grid(total, sms), 256, 0, s>>>(a);
    return cudaGetLastError();
}

template <class C>
cudaError_t launch_wavespeed(const DgWaveArgs &a, int sms, cudaStream_t s) {
    const size_t total = (size_t)a.nx * a.ny * a.nz * (C::N * C::N * C::N);
    dg_wavespeed_kernel<C><<<flat_grid(total, sms), 256, 0, s>>>(a);
    return cudaGetLastError();
}

template <class C>
constexpr DgKernelTable make_table() {
    return DgKernelTable{C::N,       C::BX,          C::BY,         C::THREADS,      Smem<C>::BYTES,     C::SLOT,
                         C::TXY,     C::TZ,          C::CX, C::CY, C::CZ, C::RELOAD ? 1 : 0, C::MINB, &prepare<C>, &launch_stage<C>,  &launch_traces<C>, &launch_split_volume<C>, &launch_split_surface<C>,
                         &launch_layout<C>, &launch_wavespeed<C>, &launch_visc_gradflux<C>, &launch_visc_div<C>};
}

// Variants per N (default first): Cfg<N, BX, BY, min blocks per SM, RELOAD, PP, OX, OY>.
// DESIGN.md "column shapes" and "shared-memory layout" explain the choices.
// dg_create and dg_set_brick select by column SHAPE and take the first variant of a shape, so a later variant with the
// same (BX, BY) can only be reached through dg_set_variant: those (other residency / reload / offset settings of a shape,
// all measured slower than the first) are compiled only with -DDG_ALL_VARIANTS (python -m
// paper_2006_15698_b200.build --all-variants, for bench.py --sweep-variants); DG_X(...) marks them.
#define DG_T(...) make_table<Cfg<__VA_ARGS__>>(),
#ifdef DG_ALL_VARIANTS
#define DG_X(...) DG_T(__VA_ARGS__)
#else
#define DG_X(...)
#endif
#if DG_N == 2
#define DG_VARIANTS DG_T(2, 9, 8, 2, 1, 290, 0, 0) DG_T(2, 8, 4, 3, 0, 0, 3, 0) DG_T(2, 4, 4, 6, 0, 0, 3, 0) DG_T(2, 8, 8, 2, 0, 0, 3, 0) \
                    DG_T(2, 9, 7, 2, 1, 258, 3, 0) DG_X(2, 9, 7, 3, 1, 258, 3, 0)
#elif DG_N == 3
#define DG_VARIANTS DG_T(3, 6, 4, 2, 0, 0, 4, 0) DG_T(3, 4, 4, 2, 0, 0, 4, 4) DG_T(3, 2, 7, 3, 0, 134, 4, 0) DG_T(3, 6, 3, 2, 0, 0, 4, 0) \
                    DG_X(3, 4, 4, 3, 1, 0, 4, 4) DG_T(3, 4, 2, 4, 1, 0, 4, 0)
#elif DG_N == 4
#define DG_VARIANTS DG_T(4, 2, 2, 4, 0, 66, 1, 0) DG_X(4, 2, 2, 5, 1, 66, 1, 0) DG_T(4, 4, 2, 2, 0, 130, 3, 0) DG_X(4, 4, 2, 3, 1, 130, 3, 0) \
                    DG_X(4, 2, 2, 3, 0, 66, 1, 0)
#elif DG_N == 5
#define DG_VARIANTS DG_T(5, 2, 3, 2, 0, 154, 6, 0) DG_X(5, 2, 3, 2, 0, 154, 4, 0) DG_T(5, 3, 2, 2, 0, 0, 4, 0) DG_T(5, 2, 2, 3, 1, 106, 4, 0) DG_T(5, 5, 1, 2, 0, 0, 4, 0) \
                    DG_X(5, 5, 1, 2, 1, 0, 4, 0) DG_T(5, 1, 5, 2, 0, 138, 0, 1)
#elif DG_N == 6
#define DG_VARIANTS DG_T(6, 1, 3, 2, 1, 118, 0, 0) DG_X(6, 1, 3, 2, 0, 118, 0, 0) DG_T(6, 3, 1, 2, 0, 114, 2, 0) DG_T(6, 2, 1, 3, 0, 0, 4, 0) DG_X(6, 2, 1, 3, 1, 0, 4, 0) \
                    DG_T(6, 1, 1, 5, 1, 0, 0, 0) DG_X(6, 1, 1, 4, 0, 0, 0, 0)
#elif DG_N == 7
#define DG_VARIANTS DG_T(7, 2, 1, 2, 1, 0, 4, 6, 1) DG_X(7, 2, 1, 2, 1, 0, 4, 0, 1) DG_X(7, 2, 1, 2, 1, 0, 4, 0) DG_T(7, 1, 1, 4, 1, 0, 0, 1) DG_X(7, 1, 1, 4, 0, 0, 0, 1) DG_X(7, 1, 1, 3, 0, 0, 0, 1)
#elif DG_N == 8
#define DG_VARIANTS DG_T(8, 1, 1, 3, 1, 66, 1, 1) DG_X(8, 1, 1, 3, 0, 66, 1, 1) DG_T(8, 2, 1, 1, 0, 130, 1, 0) DG_T(8, 1, 2, 1, 0, 130, 1, 1)
#else
#error "DG_N must be 2..8"
#endif

// last: one element per layer, always there (tiny and ragged meshes, tests); for N >= 6 the list above already has a
// 1 x 1 shape in front of it, so this one is unreachable there and is kept for DG_ALL_VARIANTS only
#if DG_N <= 5 || defined(DG_ALL_VARIANTS)
const DgKernelTable k_tables[] = {DG_VARIANTS DG_T(DG_N, 1, 1, 2, 1)};
#else
const DgKernelTable k_tables[] = {DG_VARIANTS};
#endif

}  // namespace

#define DG_CAT2(a, b) a##b
#define DG_CAT(a, b) DG_CAT2(a, b)
const DgKernelTable *DG_CAT(dg_variants_N, DG_N)(int *count) {
    *count = (int)(sizeof(k_tables) / sizeof(k_tables[0]));
    return k_tables;
}
