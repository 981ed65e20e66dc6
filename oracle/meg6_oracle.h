/*
 * meg6_oracle.h -- C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, FP64 restatement of the MEG6 + alpha-damping + SSP-RK3 discretisation of
 * arXiv 2303.10785 ("P:n" = line n of /root/reference/PAPER.md).  Only tests/, bench.py's
 * cpu_baseline / --impl reference legs and __graft_entry__.smoke() may load this library.
 * It shares no source, header, table or helper with the CUDA path (paper_2303_10785_b200/).
 *
 * All pointers are HOST pointers.  State arrays are interior-only structure-of-arrays
 * U[5][nk][nj][ni] (rho, rho u, rho v, rho w, E), i (xi) fastest.  Node arrays are
 * (ni+1)(nj+1)(nk+1), i fastest.
 */
#ifndef MEG6_ORACLE_H
#define MEG6_ORACLE_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct meg6o_grid meg6o_grid;

typedef struct {
  int ni, nj, nk;           /* interior cells                                                   */
  int periodic[3];          /* per direction                                                    */
  double period[3][3];      /* period[d] = (dx,dy,dz) added to ghost coordinates across dir d   */
  int scheme;               /* 0 = MEG6 (E6 gradients, Eq. 17), 1 = MIG4 (IG4, Eq. 18)          */
  int viscous;              /* 0/1                                                              */
  double gamma, r_gas, prandtl;
  double mu_ref, t_ref, s_suth; /* Sutherland; s_suth < 0 => constant mu = mu_ref               */
  double mp_alpha;          /* MP limiter alpha (App. E), default 4                             */
  int moving;               /* 1: x(t) = x0 + sin(2 pi omega t) dx_mode                         */
  double omega;
  int bc[6];                /* faces imin,imax,jmin,jmax,kmin,kmax: 0 periodic, 1 inflow, 2 outflow, 3 inviscid wall, 4 adiabatic wall, 5 block interface */
  double p_out;             /* outflow reference pressure                                       */
  int metric_form;          /* ORACLE ONLY: 0 = conservative Eq. 10 + consistent delta/H (Sec. 7),
                               1 = non-conservative App. D (negative control for freestream)    */
} meg6o_params;

meg6o_grid* meg6o_create(const meg6o_params* p, const double* x, const double* y, const double* z,
                         const double* dxm, const double* dym, const double* dzm);
void meg6o_destroy(meg6o_grid* g);
void meg6o_set_threads(int n);
int  meg6o_get_threads(void);

void meg6o_metrics_compute(meg6o_grid* g, double t);
/* tests only: padded cell centres [(nk+20)(nj+20)(ni+20)], ghost depth 10, used instead of the nodes */
void meg6o_set_centres(meg6o_grid* g, const double* xc, const double* yc, const double* zc);
void meg6o_set_inflow(meg6o_grid* g, int face, const double* P_in);   /* [5][n2][n1] of that face */
void meg6o_set_sponge(meg6o_grid* g, const double* sigma, const double* U_ref);
void meg6o_rhs(meg6o_grid* g, const double* U, double* dUdt);
void meg6o_rk3_step(meg6o_grid* g, double* U, double t, double dt);
/* Multi-block (Sec. 6; Table 1 last column; R28): face `face` (bc 5) of `home` takes its ghost primitives
 * from the interior cells of `nb` next to nb's opposite face; aligned blocks, equal transverse sizes.  Returns 0 if ok.
 * The *_blocks calls advance all blocks together (ghost exchange before every right-hand side). */
int meg6o_link_blocks(meg6o_grid* home, int face, meg6o_grid* nb);
/* The same for blocks with their own coordinate systems: home's `face` is the neighbour's `nb_face`; home's
 * transverse axes (storage order) run along the neighbour's transverse axes in that order (swap 0) or exchanged (swap 1),
 * forwards or backwards (flip_a, flip_b); off[3] (may be NULL) is added to the neighbour's cell-centre coordinates seen
 * from home (the period vector across a wrap-around link).  Ghost CELLS come from the neighbour: primitives and the
 * cell-centre coordinates the metrics are formed from (R28, R29). */
int meg6o_link_blocks_oriented(meg6o_grid* home, int face, meg6o_grid* nb, int nb_face, int swap, int flip_a, int flip_b,
                               const double* off);
/* geometry of linked blocks together: cell centres of all, ghost coordinates direction by direction over all, metrics */
void meg6o_metrics_compute_blocks(int nb, meg6o_grid* const* g, double t);
/* staged geometry for blocks in different processes: centres -> for d: [pack / deliver] extend(d) -> finish */
size_t meg6o_geom_interface_doubles(const meg6o_grid* g, int face);
void meg6o_set_geom_interface_buffer(meg6o_grid* g, int face, const double* layers, const double* off);
void meg6o_stage_geom_centres(meg6o_grid* g, double t);
void meg6o_stage_geom_pack(meg6o_grid* g, int face, double* layers);
void meg6o_stage_geom_extend(meg6o_grid* g, int d);
void meg6o_stage_geom_finish(meg6o_grid* g);
/* Staged evaluation for blocks in different processes: prim -> for d: [pack / deliver / set_interface_buffer] ghosts(d)
 * -> stage_rhs.  The packed layers of a face: meg6o_interface_doubles doubles. */
size_t meg6o_interface_doubles(const meg6o_grid* g, int face);
void meg6o_set_interface_buffer(meg6o_grid* g, int face, const double* layers);
void meg6o_stage_prim(meg6o_grid* g, const double* U);
void meg6o_stage_ghosts(meg6o_grid* g, int d);
void meg6o_stage_pack(meg6o_grid* g, int face, double* layers);
void meg6o_stage_rhs(meg6o_grid* g, const double* U, double* dUdt);
void meg6o_rhs_blocks(int nb, meg6o_grid* const* g, const double* const* U, double* const* dUdt);
void meg6o_rk3_step_blocks(int nb, meg6o_grid* const* g, double* const* U, double t, double dt);
double meg6o_cfl_dt(meg6o_grid* g, const double* U, double cfl);
/* volume-averaged kinetic energy, enstrophy (Eq. 54, in 3-D with dV = 1/J) and the volume: out[3] */
void meg6o_diagnostics(meg6o_grid* g, const double* U, double* out);
void meg6o_limiter_stats(meg6o_grid* g, unsigned long long* n_limited, unsigned long long* n_tested);
/* Branch record of the LAST right-hand side (last stage of the last rk3_step), kept while enabled: one 16-bit word per
 * interface of family d (n_d + 1 interfaces along d, interior extents along the others, i fastest, as meg6o_get_face):
 * bit r (0..4): the left state of characteristic component r failed test E.1 and was limited; bit 5+r: the
 * right state; bits 10-11: the branch 0..3 of Eq. 26 (cascade R10) the HLLC flux took; bit 12 (oracle only):
 * that branch was a tie -- a wave speed the cascade tested lies within 1e-10 of zero relative to the fastest wave, so
 * either neighbouring branch gives the same flux up to round-off (R10).
 * get returns the number of words (out may be NULL). */
void meg6o_branch_masks_enable(meg6o_grid* g, int on);
size_t meg6o_get_branch_mask(meg6o_grid* g, int d, unsigned short* out);

/* inspection (tests): which = 0..8 hatted metrics (xi_x..zeta_z), 9 = 1/J, 10..12 = xi_t,eta_t,zeta_t
 * (hatted), 13 = (1/J)_t, 14..16 = cell-centre x,y,z.   out[nk][nj][ni]                          */
void meg6o_get_cell(meg6o_grid* g, int which, double* out);
/* interface arrays of family d (0,1,2): q = 0..8 hatted metrics, 9 = 1/J, 10 = own time metric.
 * out has (n_d + 1) entries along d, interior extents along the others, i fastest.              */
void meg6o_get_face(meg6o_grid* g, int d, int q, double* out);
/* primitives (rho,u,v,w,p,T) and their D1 gradients after the last rhs(): interior only          */
void meg6o_get_prim(meg6o_grid* g, int field, double* out);
void meg6o_get_grad(meg6o_grid* g, int d, int field, double* out);

/* ---- fine-grained pieces exported so that tests can pin each formula by itself ---- */
/* 1-D line operators on f[0..n-1]; out[i] is written where the stencil fits, else NaN.
 * op: 0 D1 (Eq. 17), 1 D2 (Eq. 19), 2 Lft, 3 Rgt (Eq. 16), 4 H at i+1/2 (Eq. 36/38),
 *     5 delta (Eq. 37), 6 alpha-damping interface gradient at i+1/2 (Eq. 29-31)
 *     7 fourth-order central difference (Eq. D.2)                                               */
void meg6o_line_op(int op, int n, const double* f, double* out);
/* eigenvector matrices of App. A for unit normal n, mean density rho, sound speed a (row major 5x5) */
void meg6o_eigen(const double n[3], double rho, double a, double Linv[25], double Rmat[25]);
/* MP limiter (App. E) for one component: returns limited value; *limited = 1 if E.1 failed.     */
double meg6o_mp_limit(double w_unl, double c0, double cm, double cp, double dm_near, double dm_far,
                      double alpha, int* limited);
/* contravariant HLLC (Eq. 26-27): PL,PR = (rho,u,v,w,p); m = (mx,my,mz,mt); F[5]; returns branch 0..3 */
int meg6o_hllc(const double PL[5], const double PR[5], const double m[4], double gamma, double F[5]);
/* full inviscid interface flux (O3): Pc = 4 cells i-1..i+2, P1 = P' at i,i+1, P2 = P'' at i-1..i+2 */
void meg6o_inviscid_face(const double Pc[4][5], const double P1[2][5], const double P2[4][5],
                         const double m[4], double gamma, double alpha, double F[5]);
/* viscous interface flux (O4) on an interface of family d (0 xi, 1 eta, 2 zeta).
 * phi[2][4] = (u,v,w,T) at cells i,i+1 (along d); g[2][3][4] = D1 gradients [cell][xi|eta|zeta][field];
 * mh[9] = hatted interface metrics (xi_x,xi_y,xi_z,eta_x,...,zeta_z); rj = interface 1/J        */
void meg6o_viscous_face(int d, const double phi[2][4], const double g[2][3][4], const double mh[9],
                        double rj, const meg6o_params* p, double Fv[5]);
double meg6o_sutherland(const meg6o_params* p, double T);

#ifdef __cplusplus
}
#endif
#endif
