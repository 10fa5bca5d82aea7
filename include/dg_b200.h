/*
 * dg_b200.h -- C ABI of the B200-native (sm_100a, fp64) explicit time step of the nodal
 * discontinuous Galerkin discretisation of the 3-D compressible Euler equations on a uniform
 * periodic Cartesian hex mesh with collocated Gauss-Legendre points
 * (Kirby & Mavriplis, arXiv 2006.15698; citations are PAPER.md:<line>).
 *
 * One context = one mesh + one state vector resident in GPU memory.  The hot path is
 *     dg_rk_step : 5 x [ pointwise flux -> sum-factorised differentiation -> face traces ->
 *                        Lax-Friedrichs interface flux -> lift -> 2/h scaling -> LSERK45 stage ]
 * every step of which runs in this library's CUDA kernels (no CPU fallback, no other library).
 *
 * Memory ownership: the CALLER allocates all device memory (one workspace of
 * dg_workspace_bytes(), e.g. a torch uint8 tensor) and owns the CUDA stream; the library borrows
 * both from dg_bind() until dg_destroy().  The context itself (a host struct holding the small
 * operator tables, which travel to the GPU inside the kernel arguments) is owned by the library.
 *
 * Stream and device contract: every call after dg_bind() enqueues its work on the stream given to
 * dg_bind() and assumes that the workspace's device is the calling thread's CURRENT device (the
 * library never calls cudaSetDevice).  Device pointers passed to dg_set_state / dg_get_state /
 * dg_residual are read or written in that stream's order: data produced or consumed on another
 * stream must be ordered against it by the caller (event or synchronise).
 *
 * Canonical array layout of every state-sized argument (`q`, `r`), N = p+1:
 *     a[ ((((e*N + k)*N + j)*N + i)*5 + n ],   n = rho, rho u, rho v, rho w, rho E   (eq (2))
 *     e = ex + nx*(ey + ny*ez)                 (element order: DESIGN.md reading R13)
 * Node (i,j,k) of element (ex,ey,ez) is at x = (ex + (xi_i+1)/2) Lx/nx, ... with xi the
 * N Gauss-Legendre points on [-1,1], ascending.  The library keeps the state in its
 * own column-layer-major, variable-planar layout; dg_set_state /
 * dg_get_state convert on the device.
 *
 * Pointers flagged `on_device` are device pointers (same device as the workspace) when
 * on_device != 0, host pointers otherwise (pinned memory makes the copies asynchronous).
 *
 * Errors: every int-returning call returns DG_OK or one of the codes below and never throws or
 * aborts; dg_last_error() gives the text.  Invalid arguments leave the context unchanged.  CUDA
 * errors of asynchronous work surface at the next synchronising call.  Non-physical states
 * (rho <= 0, p <= 0) are not trapped: the paper has no limiter; NaNs propagate (reading R15).
 *
 * Thread safety: calls on one context must be serialised by the caller.
 */
#ifndef DG_B200_H
#define DG_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dg_ctx dg_ctx; /* opaque */

enum {
    DG_OK = 0,
    DG_EINVAL = 1,       /* bad argument */
    DG_EUNSUPPORTED = 2, /* p outside 1..7 */
    DG_ENOMEM = 3,       /* workspace too small / host allocation failed */
    DG_ECUDA = 4,        /* CUDA runtime error (text in dg_last_error) */
    DG_ESTATE = 5,       /* call out of order: not bound, or no state set */
    DG_ENONPHYSICAL = 6  /* dg_rk_step_cfl only: the state has a node with rho <= 0, p <= 0 or a non-finite value, so its
                            wavespeed gives no time step (the call itself was in order; the paper has no limiter) */
};

/* Create a context for nx*ny*nz periodic elements on [0,Lx]x[0,Ly]x[0,Lz], extent = {Lx,Ly,Lz},
 * polynomial degree p (N = p+1 Gauss-Legendre points per direction) and ratio of
 * specific heats gamma.  nx,ny,nz >= 1; 1 <= p <= 7 else DG_EUNSUPPORTED;
 * gamma > 1; extents > 0.  Touches no GPU.  *out is set only on DG_OK. */
int dg_create(dg_ctx **out, int nx, int ny, int nz, int p, double gamma, const double extent[3]);

/* Optional tuning knob, before dg_bind: the stage kernel cuts the mesh into COLUMNS of bx x by elements
 * and a thread block marches through lz consecutive z layers of one column.  Only the
 * column shapes compiled into the library for this p are accepted (DG_EUNSUPPORTED otherwise);
 * bx = by = 0 keeps the current shape; lz = 0 lets the library choose the chunk length.  Changes layout
 * sizes, so it is refused after dg_bind (DG_ESTATE). */
int dg_set_brick(dg_ctx *ctx, int bx, int by, int lz);

/* Boundary conditions of the six domain faces, bc = {x-, x+, y-, y+, z-, z+}.  The paper's
 * benchmark is periodic and gives no other condition; these are DESIGN.md reading R19:
 *   DG_BC_PERIODIC : the neighbour across the face is the element at the other end of the axis (default; an axis is
 *                    periodic on both of its faces or on neither, DG_EINVAL otherwise)
 *   DG_BC_WALL     : slip wall; the exterior state of the Lax-Friedrichs flux is the interior trace with
 *                    its face-normal momentum negated
 *   DG_BC_FARFIELD : the exterior state is q_inf[5] = (rho, rho u, rho v, rho w, rho E), a host array copied by the call
 *                    (may be NULL when no face is a far field)
 *   DG_BC_HALO     : the elements beyond the face belong to ANOTHER context (block decomposition of a larger mesh over
 *                    several GPUs; nearest-neighbour coupling only); their face
 *                    traces are read from the buffer given to dg_set_halo, which the caller fills from the
 *                    neighbour's dg_halo_export before every stage (see below)
 * May be called at any time between dg_create and dg_destroy; takes effect with the next dg_residual / dg_rk_step.
 * dg_split_surface supports periodic faces only (DG_EUNSUPPORTED otherwise). */
enum { DG_BC_PERIODIC = 0, DG_BC_WALL = 1, DG_BC_FARFIELD = 2, DG_BC_HALO = 3 };
int dg_set_boundary(dg_ctx *ctx, const int bc[6], const double q_inf[5]);

/* Number of stage-kernel variants (column shape x shared-memory layout x residency) compiled into the
 * library for degree p; 0 when p is outside 1..7.  dg_create picks the first variant whose columns
 * pad the mesh by less than 4 % (variants are listed fastest first). */
int dg_variant_count(int p);

/* Tuning knob, before dg_bind: select variant 0 <= index < dg_variant_count(p) (DG_EINVAL otherwise). */
int dg_set_variant(dg_ctx *ctx, int index);

/* 5*(p+1)^3*nx*ny*nz: number of doubles in a canonical state vector (size_t: config 5 > 2^31). */
size_t dg_state_len(const dg_ctx *ctx);

/* Device bytes the caller must provide to dg_bind: state Q, Runge-Kutta register K, one
 * canonical staging vector, two pairs of face-trace buffers (column boundaries, chunk ends), scalars. */
size_t dg_workspace_bytes(const dg_ctx *ctx);

/* Borrow `bytes` (>= dg_workspace_bytes) of device memory, 256-byte aligned, and a CUDA stream
 * (cudaStream_t passed as void*; NULL = legacy default stream).  All later work of this context
 * is enqueued on that stream.  First CUDA call of the context: queries the device, opts the kernels in
 * to their shared-memory size, and zero-fills Q and K when the layout has padding nodes. */
int dg_bind(dg_ctx *ctx, void *dev_workspace, size_t bytes, void *cuda_stream);

/* Copy a canonical state vector in (host or device), convert it to the internal layout and
 * compute its face traces.  Asynchronous for device / pinned-host sources. */
int dg_set_state(dg_ctx *ctx, const double *q, int on_device);

/* r_out = dQ/dt = L(Q) of the current state, canonical layout: eq (5) solved
 * for the time derivative, with the local Lax-Friedrichs flux (reading R3).  Does
 * not change the state.  Synchronises the stream when r_out is a host pointer. */
int dg_residual(dg_ctx *ctx, double *r_out, int on_device);

/* *lam_host = max over nodes of sqrt(u^2+v^2+w^2) + sqrt(gamma p/rho) of the current state
 * (for the caller's CFL time step; not in the paper: DESIGN.md reading R10).  After dg_set_state or
 * dg_rk_step this runs a reduction kernel over the state; after dg_rk_step_cfl the last stage has
 * already reduced it and the call is an 8-byte read-back.  NaN if any node is non-finite or has
 * negative pressure or density.  Synchronises the stream. */
int dg_max_wavespeed(dg_ctx *ctx, double *lam_host);

/* The same maximum (reading R10) for callers that CANNOT give the library device memory -- the one call of
 * this header that needs no context, no workspace and no dg_bind, and that never allocates (no cudaMalloc, cudaFree
 * or allocating library routine, on any call).  It is meant for code that holds nothing but a pointer to the
 * solution and a slot for the answer: a time-step or blow-up monitor hooked into another application's time loop;
 * a plug-in under an application that hands out all device memory at start-up and forbids allocation afterwards
 * (cudaMalloc synchronises the whole device and can fail in the middle of a run on a full card); code that has no
 * way of reporting an out-of-memory failure upwards.
 *   q_dev        DEVICE pointer, canonical layout [node][5] (see above), n_nodes = (p+1)^3 nx ny nz nodes; read only
 *   gamma        ratio of specific heats, > 1
 *   lam_out_dev  DEVICE pointer to one double on the same device: receives the maximum, NaN under the rule above,
 *                in stream order (nothing is copied to the host, nothing synchronises)
 *   cuda_stream  cudaStream_t as void* (NULL = legacy default stream); the caller's current device must be the one
 *                that holds q_dev and lam_out_dev
 *   err, err_len optional host buffer for the error text (there is no context for dg_last_error); may be NULL / 0
 * The scratch memory of the reduction (one partial maximum per thread block and a block counter) is a fixed array
 * inside the library, 256.25 KiB, which every GPU that loads the library holds until the process exits.  Its size sets
 * the limit: n_nodes <= DG_NOALLOC_MAX_NODES (2^29; config 5 has 452,984,832), beyond that the call returns DG_ENOMEM
 * with a text that says so and touches no GPU.  Other returns: DG_OK, DG_EINVAL (null pointer, gamma <= 1,
 * n_nodes = 0), DG_ECUDA.
 * The FIRST call on each device looks up where that device keeps the array (cudaGetSymbolAddress; the address is
 * cached per device): make that first call during set-up, with the device current, and before any stream capture.
 * ALL calls on one device share the one array, which keeps what the last call left (the call clears the counter it
 * needs at zero itself): calls that may overlap on the GPU -- different streams, different host threads, different
 * contexts of this library -- race on it and must be ordered by the caller; calls on one stream are safe.
 * Gives the same double as dg_set_state + dg_max_wavespeed (tests/test_zz_no_alloc.py). */
#define DG_NOALLOC_MAX_NODES 536870912ull
int dg_max_wavespeed_noalloc(const double *q_dev, size_t n_nodes, double gamma, double *lam_out_dev, void *cuda_stream,
                             char *err, size_t err_len);

/* Advance nsteps >= 0 LSERK45 steps of fixed dt:
 * K = 0; for s = 1..5: K = A_s K + dt L(Q); Q = Q + B_s K.  One fused kernel per stage,
 * enqueued on the stream, no host synchronisation. */
int dg_rk_step(dg_ctx *ctx, double dt, int nsteps);

/* nsteps >= 0 LSERK45 steps, each with its own time step from the CFL rule of reading R10,
 *     dt = cfl * min(hx,hy,hz) / ((2p+1) * lam_max(Q at the start of the step)),
 * formed ON THE DEVICE: lam_max is reduced by the last stage of the previous step (no extra sweep over the state)
 * and the next step's kernels read it from device memory, so the steps are enqueued without a host round trip.
 * One read-back at the start checks the wavespeed of the current state (DG_ENONPHYSICAL if not positive and
 * finite, nothing stepped) and one at the end returns *t_advanced = sum of the time steps taken and *dt_last = the last
 * one (host pointers, either may be NULL; DG_ENONPHYSICAL if the state went non-physical on the way).  cfl > 0. */
int dg_rk_step_cfl(dg_ctx *ctx, double cfl, int nsteps, double *t_advanced, double *dt_last);

/* The time step of the same rule (reading R10) as a plain host computation, for callers that reduce the wavespeed
 * themselves -- a block decomposition takes the maximum of dg_max_wavespeed over all contexts (below):
 *     *dt = (cfl * min(hx,hy,hz) / (2p+1)) / lam_max,
 * the operations dg_rk_step_cfl performs on the device, in the same order.  Touches no GPU and does not change the
 * context.  cfl, lam_max positive and finite and dt non-null, else DG_EINVAL (no text: the context is const). */
int dg_cfl_dt(const dg_ctx *ctx, double cfl, double lam_max, double *dt);

/* Block decomposition over several contexts / GPUs (one exchange of face
 * data per Runge-Kutta stage).  The library does no communication itself: it exports and imports face traces, the
 * caller moves them (NCCL / peer copies between GPUs, plain copies between contexts of one GPU).  All contexts of a
 * decomposition must use the same p, the same column shape (variant) and, across a shared face, the same number of
 * elements in the two transverse directions.
 *   dg_halo_len(ctx, f)      doubles in the trace buffer of domain face f = 0..5 (x-, x+, y-, y+, z-, z+)
 *   dg_halo_export(ctx, f, dst_dev)  gathers the face traces of the CURRENT state on face f (the T- of the first /
 *                            T+ of the last elements along the axis) into the DEVICE buffer dst_dev,
 *                            enqueued on the stream; this is what the neighbour across f needs
 *   dg_set_halo(ctx, f, halo_dev)    the DEVICE buffer (dg_halo_len doubles, caller-owned, must stay valid) from which
 *                            the kernels read the traces of the elements beyond face f when its condition is
 *                            DG_BC_HALO: the export of the opposite face of the neighbour context; it must hold
 *                            the neighbour's traces of the current state whenever dg_residual / dg_rk_stage runs
 *   dg_rk_stage(ctx, dt, s)  ONE stage s = 0..4 of the LSERK45 step (dg_rk_step = stages 0..4 in a row), so that the
 *                            caller can exchange the faces between stages: export -> move -> next stage.
 * The interface flux of a shared face is evaluated by both contexts, bit-identically, so a decomposed run reproduces
 * the single-context run bit for bit (tests/test_gpu_halo.py).  With halo faces dg_rk_step is refused (DG_EUNSUPPORTED:
 * five stages back to back would read stale neighbour traces) and so is dg_rk_step_cfl (the CFL wavespeed is a maximum
 * over all contexts: reduce dg_max_wavespeed across them, form dt with dg_cfl_dt and use dg_rk_stage). */
/* Before dg_bind: element sizes h = {hx, hy, hz} given directly instead of extent / n (a block of a decomposed mesh
 * must use the SAME doubles as its neighbours; extent * n_local / n_global divided by n_local again can differ in
 * the last bit).  DG_ESTATE after dg_bind. */
int dg_set_spacing(dg_ctx *ctx, const double h[3]);
size_t dg_halo_len(const dg_ctx *ctx, int face);
int dg_halo_export(dg_ctx *ctx, int face, double *dst_dev);
int dg_set_halo(dg_ctx *ctx, int face, const double *halo_dev);
int dg_rk_stage(dg_ctx *ctx, double dt, int stage);

/* "Push" mode of the same decomposition: the face exchange done BY THE STAGE KERNEL, with no export kernel and no message.
 * Every halo face gets a PAIR of trace buffers, read alternately:
 *   dg_set_halo_pair(ctx, f, buf0, buf1)  the kernels of a stage read the traces beyond face f from buf[parity], parity =
 *                            number of stages run since dg_set_state, mod 2 (device buffers of dg_halo_len doubles each)
 *   dg_set_halo_push(ctx, f, peer0, peer1)  the NEIGHBOUR's pair for ITS opposite face (f ^ 1): while a stage computes,
 *                            the blocks on face f store the traces of the updated state straight into
 *                            peer[1 - parity], which is what the neighbour reads in the next stage.  The pointers may be
 *                            peer-mapped memory of another GPU (CUDA peer access / IPC): the stores then travel over
 *                            NVLink while the rest of the stage computes -- the paper's computation-communication
 *                            overlap, tile by tile.  The call looks up the device that holds the buffers
 *                            and, if it is not the current one, enables peer access to it (DG_EUNSUPPORTED if the two
 *                            GPUs have none).  UNVERIFIED across GPUs: this code has only ever run with both
 *                            contexts on ONE GPU (the tests' CUDA-IPC case included).
 * The caller provides the ordering only: every context's stage s must have completed before any neighbour's stage s + 1
 * starts (same stream, events, or a barrier between processes), and both sides must have run the same number of stages
 * since dg_set_state.  After dg_set_state the initial traces go to the neighbour's buffer 0 with dg_halo_export.
 * dg_residual reads buf[parity] and pushes nothing.  Not combined with the per-kernel mode (dg_split_update resets the parity).
 * Results are bit-identical to the export / import mode and to the single-context run. */
int dg_set_halo_pair(dg_ctx *ctx, int face, const double *halo0_dev, const double *halo1_dev);
int dg_set_halo_push(dg_ctx *ctx, int face, double *peer0_dev, double *peer1_dev);

/* Paper-shaped per-kernel mode (Table II): the same spatial residual and stage
 * update as dg_rk_step, run as the paper's three kernels so that their times can be measured one by one (the fused
 * path is the product; this mode exists for the breakdown and is parity-tested against the oracle's terms).
 *   dg_split_volume : R  = volume term of the current state (eq (5) 2nd term / mass; "overwrites R")
 *   dg_split_surface: R -= lift of the local Lax-Friedrichs interface fluxes (eq (5) 3rd term / mass)
 *   dg_split_update : K = A_s K + dt R; Q = Q + B_s K for stage s = 0..4 of LSERK45, then the face traces of the new
 *                     state ("update-project")
 * After volume + surface R = dQ/dt = L(Q) as dg_residual returns it.  R lives in the library's staging vector: do
 * not interleave host-pointer dg_set_state / dg_get_state / dg_residual calls between volume and update.  All three
 * are enqueued on the stream without synchronisation.  dg_split_get_r copies R out in canonical layout (host or
 * device pointer).  The HOST variant stages the copy through the Runge-Kutta register K and destroys its contents: K is
 * dead only BETWEEN steps (after stage 4 and before the next stage 0), so call it there -- between dg_split_update
 * stages 0..3 of one step it would corrupt the step.  The device variant touches nothing but R and r_out. */
int dg_split_volume(dg_ctx *ctx);
int dg_split_surface(dg_ctx *ctx);
int dg_split_update(dg_ctx *ctx, double dt, int stage);
int dg_split_get_r(dg_ctx *ctx, double *r_out, int on_device);

/* Viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4.  The paper names "the viscous formulation" of its CPU code
 * and prints no viscous equations; the formulation is DESIGN.md reading R20:
 *     dQ/dt = L(Q) + div Fv(Q, grad Q),  Fv_a = (0, tau_a1, tau_a2, tau_a3, u_b tau_ab + mu gamma/(Pr (gamma-1)) d_a(p/rho)),
 *     tau_ab = mu (d_a u_b + d_b u_a - 2/3 delta_ab d_c u_c)
 * (constant dynamic viscosity mu, Stokes hypothesis, Fourier conduction with constant Prandtl number Pr, ideal gas),
 * discretised in the basis of eq (4)-(7) by the first Bassi-Rebay scheme: the gradient of the conserved variables and
 * the divergence of the nodal viscous flux both use the weak form of eq (5) with the central interface value.
 * Periodic meshes only (DG_EUNSUPPORTED otherwise).  Runs as kernels of its own on top of the per-kernel mode, not
 * in the fused stage kernel.
 *   dg_set_viscosity : before dg_bind (three more state-sized vectors in the workspace when mu > 0; DG_ESTATE after);
 *                      mu >= 0, prandtl > 0 (DG_EINVAL otherwise); mu = 0 switches the terms off
 *   dg_split_viscous : R += div Fv of the current state (after dg_split_volume + dg_split_surface R = L(Q) + div Fv);
 *                      two sweeps: gradients + pointwise viscous flux (one kernel), divergence (one kernel)
 *   dg_rk_step_ns    : nsteps LSERK45 steps of fixed dt of dQ/dt = L(Q) + div Fv
 *                      (per stage: dg_split_volume, dg_split_surface, dg_split_viscous, dg_split_update)
 * All enqueued on the stream without synchronisation. */
int dg_set_viscosity(dg_ctx *ctx, double mu, double prandtl);
int dg_split_viscous(dg_ctx *ctx);
int dg_rk_step_ns(dg_ctx *ctx, double dt, int nsteps);

/* Copy the current state out in canonical layout.  Synchronises when q_out is a host pointer. */
int dg_get_state(dg_ctx *ctx, double *q_out, int on_device);

/* The library's own N Gauss-Legendre nodes and weights (host arrays of p+1 doubles). */
int dg_nodes(const dg_ctx *ctx, double *xi, double *w);

/* Number of CUDA kernels this context has launched so far (bench.py's `gpu_launches`). */
unsigned long long dg_launch_count(const dg_ctx *ctx);

/* Launch geometry of the fused stage kernel, for reports: out[0..7] = column elements bx, by, layers per
 * chunk lz, threads per block, dynamic shared bytes per block, resident blocks of the whole GPU (once
 * bound; thread blocks per launch before), internal (padded) state length in doubles / 2^20 rounded
 * up, index of the variant in use. */
int dg_kernel_info(const dg_ctx *ctx, long long out[8]);

/* Release the context (never the borrowed workspace).  NULL is accepted. */
int dg_destroy(dg_ctx *ctx);

/* Text of the last error on this context ("" if none).  Valid until the next call on ctx. */
const char *dg_last_error(const dg_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* DG_B200_H */
