/*
 * dg_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded CPU oracle for the explicit time step of the nodal
 * discontinuous Galerkin discretisation of the 3-D compressible Euler equations on a
 * uniform periodic Cartesian hex mesh (arXiv 2006.15698, section II).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call anything under oracle/.  It shares no code with the CUDA path in
 * paper_2006_15698_b200/csrc/ and includes none of its headers.
 *
 * Arithmetic type: `real` = double by default; compile with -DORACLE_REAL="long double" for
 * the higher-precision arbiter build (same source, same interface; all arrays crossing this
 * interface stay double).
 *
 * Canonical array layout (listing index `idx1`): for N = p+1,
 *     q[ ((((e*N + k)*N + j)*N + i)*5 + n ],   n = rho, rho*u, rho*v, rho*w, rho*E
 * with element index e = ex + nx*(ey + ny*ez) (element ordering is not in the paper;
 * DESIGN.md reading R13).  Node (i,j,k) of element (ex,ey,ez) sits at
 *     x = (ex + (xi_i+1)/2) * Lx/nx, etc., xi = Gauss-Legendre nodes on [-1,1], ascending.
 *
 * Every function returns 0 on success, nonzero on invalid arguments.
 */
#ifndef DG_ORACLE_H
#define DG_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

/* N-point Gauss-Legendre nodes (ascending) and weights on [-1,1]. */
int oracle_gauss_legendre(int N, double *xi, double *w);

/* 1-D operators of the collocated Lagrange basis, eq (7):
 *   D[q*N+i]    = l_i'(xi_q)               (differentiation matrix)
 *   lp[i], lm[i] = l_i(+1), l_i(-1)        (face interpolation)
 *   Dhat[i*N+q] = w_q * D[q*N+i] / w_i     (weak-form volume operator, eq (5) 2nd term
 *                                           divided by the diagonal mass matrix)        */
int oracle_operators(int N, double *xi, double *w, double *D, double *lp, double *lm,
                     double *Dhat);

/* Carpenter-Kennedy (5,4) 2N-storage coefficients (reading R9). */
void oracle_lserk45(double A[5], double B[5]);

/* r = volume term V only (eq (5) 2nd term / mass).  Canonical layout, overwritten. */
int oracle_volume_term(int nx, int ny, int nz, int p, double gamma, const double extent[3],
                       const double *q, double *r);

/* r = surface term S only (eq (5) 3rd term / mass), local Lax-Friedrichs flux. */
int oracle_surface_term(int nx, int ny, int nz, int p, double gamma, const double extent[3],
                        const double *q, double *r);

/* r = dQ/dt = L(Q) = V - S  (eq (5) solved for the time derivative). */
int oracle_residual(int nx, int ny, int nz, int p, double gamma, const double extent[3],
                    const double *q, double *r);

/* nsteps LSERK45 steps of fixed dt, in place on q. */
int oracle_rk_step(int nx, int ny, int nz, int p, double gamma, const double extent[3],
                   double *q, double dt, int nsteps);

/* The same two with non-periodic domain faces (the paper gives no boundary condition, PAPER.md:126
 * "periodic domain": DESIGN.md reading R19).  bc[6] = condition of the faces x-, x+, y-, y+, z-, z+: 0 periodic (both
 * faces of an axis or neither), 1 slip wall (exterior state = interior trace with the normal momentum negated),
 * 2 far field (exterior state = qinf[5], conserved variables).  bc == NULL means periodic everywhere. */
int oracle_residual_bc(int nx, int ny, int nz, int p, double gamma, const double extent[3], const int bc[6],
                       const double qinf[5], const double *q, double *r);
int oracle_rk_step_bc(int nx, int ny, int nz, int p, double gamma, const double extent[3], const int bc[6],
                      const double qinf[5], double *q, double dt, int nsteps);

/* Viscous (Navier-Stokes) terms, SURVEY.md 8(f)-4.  The paper names them only and prints no equations:
 * DESIGN.md reading R20, PARITY UNPINNED BY THE PAPER.  Constant dynamic viscosity mu >= 0, Stokes hypothesis, Fourier
 * conduction with constant Prandtl number, first Bassi-Rebay scheme (central interface values for Q and for the viscous
 * flux) in the basis of eq (4)-(7); periodic meshes only.
 *   oracle_gradient:     s = d_axis Q, the BR1 gradient of the five conserved variables (canonical layout)
 *   oracle_viscous_term: r = div Fv(Q, grad Q),  Fv_a = (0, tau_a1, tau_a2, tau_a3, u_b tau_ab + mu gamma/(Pr (gamma-1)) d_a(p/rho))
 *   oracle_residual_ns:  r = L(Q) + div Fv;  oracle_rk_step_ns: LSERK45 steps of dQ/dt = L(Q) + div Fv */
int oracle_gradient(int nx, int ny, int nz, int p, const double extent[3], int axis, const double *q, double *s);
int oracle_viscous_term(int nx, int ny, int nz, int p, double gamma, const double extent[3], double mu, double prandtl,
                        const double *q, double *r);
int oracle_residual_ns(int nx, int ny, int nz, int p, double gamma, const double extent[3], double mu, double prandtl,
                       const double *q, double *r);
int oracle_rk_step_ns(int nx, int ny, int nz, int p, double gamma, const double extent[3], double mu, double prandtl,
                      double *q, double dt, int nsteps);

/* lam = max over nodes of sqrt(u^2+v^2+w^2) + c   (reading R10). */
int oracle_max_wavespeed(int nx, int ny, int nz, int p, double gamma, const double *q,
                         double *lam);

/* Bytes per `real` in this build (8 = double; 16 = x87 long double arbiter). */
int oracle_real_bytes(void);

/* Threads the element loops use (1 unless built with -fopenmp). */
int oracle_threads(void);

#ifdef __cplusplus
}
#endif
#endif
