/*
 * meg6.h -- C ABI of the B200 (sm_100a) implementation of the MEG6 right-hand side + SSP-RK3 step of
 * arXiv 2303.10785 (Chandravamsi et al., gradient-based reconstruction on curvilinear / dynamic meshes).
 *
 * Citations: "P:n" = line n of the paper text; "Rn" = reading n of a garbled or silent
 * passage, listed in DESIGN.md.
 *
 * Conventions (all entry points):
 *  - Every array pointer is a DEVICE pointer owned by the caller unless stated otherwise; FP64 only.
 *  - State arrays U, dUdt are interior-only structure-of-arrays [5][nk][nj][ni] of the conservative
 *    variables Q = (rho, rho u, rho v, rho w, E), index ((c*nk + k)*nj + j)*ni + i, xi fastest.
 *  - Node coordinate arrays are [(nk+1)][(nj+1)][(ni+1)], xi fastest (hexahedral cell vertices).
 *  - The library never allocates device memory: the caller passes one workspace block of
 *    meg6_workspace_bytes() bytes (256-byte aligned) that must outlive the grid handle.
 *  - All work is enqueued on the CUDA stream given at grid_create; nothing synchronises the stream
 *    except meg6_limiter_stats, meg6_cfl_dt and meg6_get_array (which copy to the host).
 *  - Every function returns a status code; meg6_last_error() gives a message for the last failure on
 *    the calling thread.  Nothing throws.  There is no CPU fallback: without a CUDA device every
 *    compute entry point returns MEG6_ECUDA.
 */
#ifndef MEG6_H
#define MEG6_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct meg6_grid meg6_grid; /* opaque; host memory owned by the library */

typedef enum {
  MEG6_OK = 0,
  MEG6_EINVAL = 1, /* bad argument (null pointer, size < stencil, unsupported option) */
  MEG6_ENOMEM = 2, /* workspace too small                                            */
  MEG6_ECUDA = 3,  /* CUDA runtime error (message in meg6_last_error)                */
  MEG6_ESTATE = 4  /* call order violated (e.g. rhs before metrics_compute)          */
} meg6_status;

typedef struct {
  int ni, nj, nk;     /* interior cells per direction; each >= 10 (periodic wrap of the 10-deep metric halo) */
  int periodic[3];    /* per direction; a periodic direction ignores bc[] of its two faces           */
  double period[3][3];/* period[d] = (dx,dy,dz) added to ghost-cell coordinates across direction d (R14) */
  int scheme;         /* 0 = MEG6 (E6 gradients, Eq. 17); 1 = MIG4 (implicit IG4 gradients, Eq. 18 P:217,
                         in reconstruction, viscous flux and metrics; line systems closed per R26)      */
  int viscous;        /* 0: Euler; 1: + alpha-damping viscous flux (Eq. 29-35)            */
  double gamma, r_gas, prandtl; /* T = p/(rho r_gas); kappa = mu gamma r_gas/((gamma-1) Pr)   */
  double mu_ref, t_ref, s_suth; /* mu = mu_ref (T/t_ref)^1.5 (t_ref+s_suth)/(T+s_suth); s_suth<0: mu = mu_ref (R15) */
  double mp_alpha;    /* alpha of the MP limiter (App. E; R7), 4 by default              */
  int moving;         /* 0 static mesh; 1: nodes x(t) = x0 + sin(2 pi omega t) * dx_mode (form of Eq. 49) */
  double omega;
  int bc[6];          /* faces imin,imax,jmin,jmax,kmin,kmax of non-periodic directions:
                         1 fixed inflow (ghost = 2 P_in - P_mirror), 2 outflow (ghost = last interior cell,
                         p = p_out where the outward normal Mach number < 1)   (Table 1, R20),
                         3 inviscid wall (ghost layer q = rho, p of the q-th interior cell, its velocity reflected
                         about the unit vector of that cell's own hatted metrics of the direction: u - 2 V k~),
                         4 adiabatic no-slip wall (rho, p mirrored, velocity negated)   (Table 1, R27),
                         5 block interface (ghost = neighbour block's interior, meg6_link_blocks; R28);
                         walls need moving == 0 (MEG6_EINVAL otherwise)                                  */
  double p_out;
} meg6_params;

/* Bytes of device workspace the grid needs (0 on invalid params). */
size_t meg6_workspace_bytes(const meg6_params* p);

/* Creates a grid.  x,y,z: node coordinates (device); dx_mode,dy_mode,dz_mode: node displacement modes
 * (device; NULL when moving == 0).  The node arrays are copied into the workspace (the caller may free
 * them after the call has been enqueued and the stream synchronised).  cuda_stream is a cudaStream_t
 * (NULL = default stream).  *out is written on success only. */
meg6_status meg6_grid_create(const meg6_params* p, const double* x, const double* y, const double* z,
                             const double* dx_mode, const double* dy_mode, const double* dz_mode,
                             void* workspace, size_t workspace_bytes, void* cuda_stream, meg6_grid** out);
void meg6_grid_destroy(meg6_grid* g);

/* Metric/Jacobian kernels (Sec. 4 and 7): cell centres = 8-vertex mean; ghost coordinates
 * (R13, R14); Thomas-Lombard conservative metrics Eq. 10 with every derivative the consistent
 * central derivative of Eq. 36-37 / 41; 1/J Eq. 13; time metrics Eq. 11; interface values by
 * the central interpolation Eq. 38; (1/J)_t Eq. 14 from the same interface values.
 * Static meshes: t ignored, idempotent.  Moving meshes: geometry at time t.
 * Environment: MEG6_GEOM_BLOCKED=0|1 forces the one-cell-per-thread or the line-blocked form of the coordinate
 * derivative and interface-metric kernels (default: blocked from 2^21 cells); both give the same bits. */
meg6_status meg6_metrics_compute(meg6_grid* g, double t);

/* Inflow data of one bc==1 face: P_in[5][n2][n1] = (rho,u,v,w,p) per face cell, (n1,n2) = the two
 * transverse extents in storage order (i before j before k).  Copied into the workspace. */
meg6_status meg6_set_inflow(meg6_grid* g, int face, const double* P_in);
/* Sponge source -sigma (Q - Q_ref) (R16): sigma[nk][nj][ni], U_ref[5][nk][nj][ni]; the POINTERS are
 * kept (caller keeps the arrays alive); NULL, NULL switches the sponge off. */
meg6_status meg6_set_sponge(meg6_grid* g, const double* sigma, const double* U_ref);

/* dUdt = dQ/dt = J (Res - (1/J)_t Q) - sigma (Q - Q_ref) with Res of Eq. 8-9: E6 gradients
 * (Eq. 17), characteristic gradient-based reconstruction (Eq. 19-23), improved MP limiter (App. E),
 * contravariant HLLC (Eq. 26-27), alpha-damping viscous flux (Eq. 29-35), at the geometry of the last
 * metrics_compute.  U and dUdt must not overlap. */
meg6_status meg6_rhs(meg6_grid* g, const double* U, double* dUdt);

/* One SSP-RK3 step (Eq. B.1) in place on U, from time t to t+dt.  Moving meshes recompute the
 * geometry at the stage times t, t+dt, t+dt/2 (R17) and leave it at t+dt/2.  U is read and written by the last
 * sweep of every stage; it must not be touched by other streams while the step is in flight. */
meg6_status meg6_rk3_step(meg6_grid* g, double* U, double t, double dt);
/* nsteps SSP-RK3 steps of constant dt (t, t+dt, ...): the same arithmetic as nsteps calls of meg6_rk3_step, bit for bit;
 * since U stays with the library between the steps (the paper's time loop is device-resident), the
 * primitive conversion of U^{n+1} is done by the last sweep of step n instead of a separate kernel per step. */
meg6_status meg6_rk3_steps(meg6_grid* g, double* U, double t, double dt, int nsteps);

/* Multi-block (Sec. 6; Table 1 last column P:354-362; readings R28, R29).  A face with bc == 5 is a block
 * interface: its ghost CELLS are the neighbour block's cells next to the face the two blocks share -- the six ghost
 * layers of primitives at every stage, and the ten ghost layers of cell-centre coordinates (and grid velocities) the
 * metrics are formed from, so that both blocks difference the same coordinates across the interface (the interface
 * metrics of a cut mesh are those of the uncut one, bit for bit; fluxes across the cut are equal and opposite).
 * meg6_link_blocks: aligned blocks -- the three computational axes of the two blocks point the same way, the
 * neighbour's face is face ^ 1, the transverse cell counts and periodicity agree.
 * meg6_link_blocks_oriented: "each block possesses its own coordinate system" -- home's `face` is the
 * neighbour's `nb_face`; home's two transverse axes, in storage order (a < b), run along the neighbour's transverse axes
 * (a' < b') as a -> a', b -> b' (swap 0) or a -> b', b -> a' (swap 1), each forwards (flip 0) or backwards (flip 1); the
 * cell counts of the interface plane must agree.  off[3] (HOST pointer, may be NULL = 0) is added to the
 * neighbour's coordinates seen from home: the period vector across a wrap-around link.  Velocities and coordinates are
 * Cartesian components: only indices are mapped.  Where some link is not the aligned one the direction-by-direction
 * ghost fills are repeated three times, so that edge and corner ghosts that reach a rotated neighbour's own ghost cells
 * are the fixed point of the exchange (R29).  MEG6_EINVAL on mismatching sizes / scheme / stream.
 * A block may be linked to itself (wrap-around).  The link is a pointer: the neighbour must outlive the home grid's
 * last call.  A link invalidates the home block's metrics (call meg6_metrics_compute[_blocks] again).
 * meg6_metrics_compute_blocks / meg6_rhs_blocks / meg6_rk3_step_blocks work on n blocks together: geometry -- cell
 * centres of all blocks, then the ghost coordinates direction by direction over all blocks, then each block's metrics;
 * flow -- primitives of all blocks, then the ghost exchange direction by direction over all blocks (edge and corner
 * ghosts come from diagonal neighbours in two steps), then the sweeps of each block; per block the semantics of the
 * single-grid calls.  g, U, dUdt: HOST arrays of n pointers (grids; DEVICE state arrays).  Every neighbour of a listed
 * block must be listed.  The single-grid calls return MEG6_ESTATE on a grid that has an interface to another block or
 * an unlinked one. */
meg6_status meg6_link_blocks(meg6_grid* home, int face, meg6_grid* neighbour);
meg6_status meg6_link_blocks_oriented(meg6_grid* home, int face, meg6_grid* neighbour, int nb_face, int swap, int flip_a,
                                      int flip_b, const double* off);
meg6_status meg6_metrics_compute_blocks(int n, meg6_grid* const* g, double t);
meg6_status meg6_rhs_blocks(int n, meg6_grid* const* g, const double* const* U, double* const* dUdt);
meg6_status meg6_rk3_step_blocks(int n, meg6_grid* const* g, double* const* U, double t, double dt);

/* Staged stepping: one RK stage as separate calls, for blocks that live on different devices (a slab decomposition:
 * SURVEY 8(e)) -- the caller moves the interface layers itself between the ghost fill of one direction and the next.
 * Per SSP-RK3 step (stage s = 0, 1, 2 at times t, t+dt, t+dt/2; moving meshes: meg6_metrics_compute before each):
 *   s == 0:  meg6_stage_prim(g, U)                       primitives of U (later stages: written by the previous sweeps)
 *   for d = 0, 1, 2:
 *       meg6_stage_pack(g, s, face, layers)              for each interface face of direction d: the six cell layers
 *                                                        next to `face`, all fields, every transverse position of the
 *                                                        padded array (ghosts of lower directions included, so edge
 *                                                        and corner ghosts travel with them); meg6_interface_doubles
 *                                                        doubles.  The caller delivers them to the neighbour, whose
 *                                                        buffer was registered with meg6_set_interface_buffer(g, face^1
 *                                                        seen from there, layers) -- pointer kept; replaces a link.
 *       meg6_stage_ghosts(g, s, d)                       ghost fill of direction d (all boundary kinds)
 *   meg6_stage_sweeps(g, U, NULL, s, dt)                 gradients + sweeps + fused RK stage update of U
 * meg6_stage_sweeps(g, U, dUdt, 0, 0) writes dQ/dt instead (after stage_prim and the ghost fills with s = 0).
 * Identical, kernel for kernel, to what meg6_rk3_step_blocks launches -- except for its edge round: after the three
 * directions the block calls copy, once more and over the ghost ranges of BOTH transverse directions, the ghost layers
 * of every face linked by pointer, so that an edge ghost cell beyond an interface is the neighbour's own ghost cell
 * there (R28).  That matters only where a fixed-inflow face with non-uniform data lies in a direction filled AFTER a
 * cut direction (the block's own P_in at a clamped index otherwise); a slab decomposition cuts the last direction and
 * needs no such round, and the staged calls have none. */
/* The geometry in pieces, for the same callers: meg6_stage_geom_centres(g, t); for d = 0, 1, 2: [meg6_stage_geom_pack
 * (g, face, layers) for the interface faces of direction d -- the ten layers of cell-centre coordinates (moving meshes:
 * and grid velocities) next to `face` over the padded transverse extent, meg6_geom_interface_doubles doubles -- delivered
 * to the neighbour, which registered its receive buffer with meg6_set_geom_interface_buffer(g, face, layers, off)],
 * meg6_stage_geom_extend(g, d); then meg6_stage_geom_finish(g).  Remote neighbours are aligned blocks at least ten
 * cells thick along the link.  Static meshes: once; moving meshes: at every stage time. */
size_t      meg6_geom_interface_doubles(const meg6_grid* g, int face);
meg6_status meg6_set_geom_interface_buffer(meg6_grid* g, int face, const double* layers, const double* off);
meg6_status meg6_stage_geom_centres(meg6_grid* g, double t);
meg6_status meg6_stage_geom_pack(meg6_grid* g, int face, double* layers);
meg6_status meg6_stage_geom_extend(meg6_grid* g, int d);
meg6_status meg6_stage_geom_finish(meg6_grid* g);

size_t      meg6_interface_doubles(const meg6_grid* g, int face);
meg6_status meg6_set_interface_buffer(meg6_grid* g, int face, const double* layers);
meg6_status meg6_stage_prim(meg6_grid* g, const double* U);
meg6_status meg6_stage_pack(meg6_grid* g, int s, int face, double* layers);
meg6_status meg6_stage_ghosts(meg6_grid* g, int s, int d);
meg6_status meg6_stage_sweeps(meg6_grid* g, double* U, double* dUdt, int s, double dt);

/* Eq. B.2 / B.3 time step for the state U at the geometry of the last metrics_compute.
 * Synchronises the stream.  *dt is a HOST pointer. */
meg6_status meg6_cfl_dt(meg6_grid* g, const double* U, double cfl, double* dt);

/* The same time step for callers that may not allocate and may not wait (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the partial minima of the reduction live in a file-scope
 * `static __device__` array of the library (256 KiB on every GPU that loads libmeg6.so, held until exit) instead of the
 * workspace, the reduction is finished on the device, and the result goes to *dt_device, a DEVICE pointer (one double)
 * owned by the caller.  Two kernel launches on the grid's stream; no cudaMalloc / cudaFree / allocating library call, no
 * copy to the host, no synchronisation.  Limit: grids of at most 16 777 216 = 2^24 cells (one pair of partial minima
 * per 1024 cells, 16 384 pairs); larger grids get MEG6_EINVAL with a message that says so (use meg6_cfl_dt).  Other
 * errors as meg6_cfl_dt.  The array is shared by every call on that GPU and keeps the last call's contents: a call
 * overwrites every slot it reads (nothing has to start at zero), but calls that overlap on the GPU -- two grids on
 * different streams, or the same grid from two threads -- race on it; callers serialise them. */
meg6_status meg6_cfl_dt_noalloc(meg6_grid* g, const double* U, double cfl, double* dt_device);

/* Volume-averaged kinetic energy and enstrophy of the state U (Eq. 54, written for three dimensions with
 * dV = 1/J; vorticity from the shared first gradients of the velocity) and the volume, at the geometry of the
 * last metrics_compute: out[0] = E_k, out[1] = enstrophy, out[2] = sum of 1/J.  out is a HOST pointer (3 doubles);
 * synchronises the stream.  Overwrites the library's primitive buffer (like meg6_rhs). */
meg6_status meg6_diagnostics(meg6_grid* g, const double* U, double* out);

/* Counters of interface-components tested / limited by the MP limiter (test E.1 failed) since grid
 * creation, accumulated only while enabled (default off; costs atomics).  HOST pointers; synchronises. */
meg6_status meg6_limiter_stats_enable(meg6_grid* g, int on);
meg6_status meg6_limiter_stats(meg6_grid* g, unsigned long long* n_limited, unsigned long long* n_tested);

/* Per-interface branch record (north_star: "any cell where an MP-limiter branch flips is reported separately").  While a
 * pointer is set, every right-hand side (each stage of rk3_step) overwrites it with one 16-bit word per interface of that
 * family -- (ni+1) nj nk words for xi, ni (nj+1) nk for eta, ni nj (nk+1) for zeta, index along the family's direction
 * running over n_d + 1, i fastest:
 *   bit r (0..4)  the LEFT state of characteristic component r failed test E.1 and went through E.2-E.4,
 *   bit 5 + r     the same for the RIGHT state (R8),
 *   bits 10-11    the branch of Eq. 26 (cascade R10) the HLLC flux took: 0 F_L, 1 F*_L, 2 F*_R, 3 F_R.
 * DEVICE pointers owned by the caller, each may be NULL (that family is not recorded); the decisions are taken in FP64
 * as in the flux itself.  Costs one 2-byte store per interface while set. */
meg6_status meg6_set_branch_masks(meg6_grid* g, unsigned short* xi, unsigned short* eta, unsigned short* zeta);

/* Inspection for tests: copies an internal array to HOST memory `out` (interior cells, [nk][nj][ni], or
 * for interface arrays n_d+1 entries along d).  kind 0: cell array `which` = 0..8 hatted metrics
 * (xi_x..zeta_z), 9 = 1/J, 10..12 = hatted time metrics, 13 = (1/J)_t, 14..16 = cell-centre x,y,z;
 * kind 1: interface array, which = 16*d + q, q = 0..8 hatted metrics, 9 = 1/J, 10 = own time metric;
 * kind 2: primitive field which = 0..5 (rho,u,v,w,p,T) after the last rhs. */
meg6_status meg6_get_array(meg6_grid* g, int kind, int which, double* out);

/* Per-kernel timing for bench.py: while enabled, every kernel launch of the library is bracketed by CUDA
 * events on the grid's stream.  meg6_profile_read synchronises the stream, adds up the elapsed time and the
 * number of kernel launches per kind since the last read, and clears the record.  HOST pointers, 16 entries
 * each.  Kinds: 0 metric/Jacobian kernels (all of one metrics_compute), 1 primitive conversion (once per step),
 * 2 ghost fill, 3 stored E6 gradients, 4 xi sweep (the last one: fused with residual assembly, the RK3 stage update
 * and the primitive conversion of the new state), 5 eta sweep (first), 6 zeta sweep, 7-8 unused, 9 CFL reduction. */
meg6_status meg6_profile_enable(meg6_grid* g, int on);
meg6_status meg6_profile_read(meg6_grid* g, double* ms_per_kind, unsigned long long* launches_per_kind);

/* FP64-pipe roof of the device by measurement (bench.py prints it beside the HBM roof): runs a
 * register-resident loop of independent DFMA chains that fills every SM (4 launches, ~10 ms) and returns the best rate
 * in DFMA thread-instructions per second (x 2 = flop/s).  scratch: DEVICE pointer to one double (never written in
 * practice); dfma_per_second: HOST pointer.  Synchronises the stream.  Needs no grid. */
meg6_status meg6_fp64_peak(void* cuda_stream, double* scratch, double* dfma_per_second);

const char* meg6_last_error(void);
/* Library/ABI version: 1000*major + minor. */
int meg6_version(void);

#ifdef __cplusplus
}
#endif
#endif
