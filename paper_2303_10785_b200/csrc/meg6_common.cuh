// meg6_common.cuh -- layouts, constants and the grid object of the B200 MEG6 library.
// Part of the single translation unit meg6.cu.  Shares nothing with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <vector>
#include "../../include/meg6.h"

namespace meg6 {

// Ghost depths.  GX: cell-centre coordinates and metrics (two nested consistent derivatives of reach 5,
// Eq. 10 + Eq. 41).  Primitives need 6 cells beyond an interface stencil (P' on i-2..i+3 from P on i-5..i+6);
// the i-axis ghost is widened to 8 so that interior rows start on a 64-byte boundary.
constexpr int GX = 10;
constexpr int GPI = 8, GPJ = 6, GPK = 6;
constexpr int GGI = 4, GGJ = 1, GGK = 1;   // stored gradients: one ghost layer (cells i and i+1 of boundary faces)

// Consistent central derivative, Eq. 41: delta f_i = sum_m CD[m-1] (f_{i+m} - f_{i-m})
__device__ constexpr double CD1 = 2282.0 / 2880.0, CD2 = -546.0 / 2880.0, CD3 = 89.0 / 2880.0,
                            CD4 = -3.0 / 2880.0, CD5 = -1.0 / 2880.0;
// Central interface value, Eq. 36/38 with Eq. 17 and 19 substituted:
// H_{i+1/2} = sum_{q=1..5} CH[q-1] (f_{i+1-q} + f_{i+q})
__device__ constexpr double CH1 = 1821.0 / 2880.0, CH2 = -461.0 / 2880.0, CH3 = 85.0 / 2880.0,
                            CH4 = -4.0 / 2880.0, CH5 = -1.0 / 2880.0;
// E6 gradient, Eq. 17
__device__ constexpr double CE1 = 3.0 / 4.0, CE2 = -3.0 / 20.0, CE3 = 1.0 / 60.0;
// Eq. 19 with Eq. 17 substituted: D2 f_i = CS0 f_i + sum_{m=1..4} CS[m] (f_{i+m} + f_{i-m})
__device__ constexpr double CS0 = -13.0 / 4.0, CS1 = 77.0 / 40.0, CS2 = -11.0 / 30.0, CS3 = 3.0 / 40.0,
                            CS4 = -1.0 / 120.0;

struct Lay {   // padded 3-D layout, i fastest
  int gi, gj, gk;
  int pi, pj, pk;
  long long sj, sk, n;
  __host__ __device__ __forceinline__ long long at(int i, int j, int k) const {
    return (long long)(k + gk) * sk + (long long)(j + gj) * sj + (long long)(i + gi);
  }
  __host__ __device__ __forceinline__ long long stride(int d) const { return d == 0 ? 1 : d == 1 ? sj : sk; }
};

inline Lay make_lay(int ni, int nj, int nk, int gi, int gj, int gk, int align_i = 1) {
  Lay L;
  L.gi = gi; L.gj = gj; L.gk = gk;
  L.pi = ni + 2 * gi;
  if (align_i > 1) L.pi = (L.pi + align_i - 1) / align_i * align_i;
  L.pj = nj + 2 * gj; L.pk = nk + 2 * gk;
  L.sj = L.pi; L.sk = (long long)L.pi * L.pj;
  L.n = L.sk * L.pk;
  return L;
}

struct Box { int lo[3], hi[3]; };   // valid cell range [lo, hi) of an array, per direction (MIG4 passes)

struct Consts {   // per-grid constants passed by value to kernels
  int n[3];
  int periodic[3];
  double period[3][3];
  int viscous, moving;
  int bc[6];
  double gamma, r_gas, prandtl, mu_ref, t_ref, s_suth, mp_alpha, p_out;
  double kappa_fac;   // gamma r_gas / ((gamma-1) Pr)
  double igm1;        // 1/(gamma-1)
  double suth_c;      // mu_ref (t_ref + s_suth) / t_ref^1.5: mu = suth_c T sqrt(T)/(T + s_suth)  (R15)
  Lay LX, LP, LG, LC; // coordinates/metrics, primitives, gradients, interior cells (caller's U layout)
  Lay LR;             // residual accumulator: interior cells, even row pitch (TMA strides are multiples of 16 B)
  Lay LF[3];          // interface families
  long long fsP, fsG, fsR, fsM[3];   // distance in doubles between consecutive fields of P, G, res, fmet[d]
};

}  // namespace meg6

// P primitives, M interface metrics, Mt time metric, G stored tangential gradients (MEG6); MIG4: Q = implicit
// gradients along the sweep, G3[s] = gradients (u,v,w,p,T) of tangential direction s
// R: running residual; U, U0, J, Sg: the caller's state, U^n, 1/J and the sponge coefficient (final phase of the fused xi sweep)
namespace meg6 { struct TmaMaps { CUtensorMap P, M, Mt, G, Q, G3[2], R, U, U0, J, Sg; }; }

struct meg6_grid {
  meg6_params p;
  meg6::TmaMaps tmaps3[2][3];   // per primitive buffer and sweep direction
  // tensor maps of the fused final phase: U^n and 1/J (fixed), sigma (set_sponge), the caller's U (re-encoded when the
  // pointer changes); tail_ok: the layouts allow them (even ni: every global stride a multiple of 16 bytes)
  void* encode_fn; bool tail_ok;
  CUtensorMap mapU0, mapJ, mapSg, mapU; const double* mapU_ptr; const double* mapSg_ptr;
  meg6::Consts c;
  cudaStream_t stream;
  char* ws; size_t ws_bytes;
  // geometry inputs (copied nodes)
  double* nodes[3]; double* modes[3];
  // geometry
  double* xc[3]; double* xt[3];
  double* cd[9];      // delta_d(x_c): cd[3*c + d]
  double* met[9]; double* rj; double* mt[3];
  double* fmet[3][10]; double* fmt[3];
  double* rjt;
  // MIG4 (scheme 1): scratch arrays of the pass-based geometry (layout LX), Thomas coefficients, stored gradients
  double* scr[6];
  double* Gi[3][6];   // IG4 gradients of the six primitive fields along xi, eta, zeta (layout LP, field stride fsP)
  double* ig4_cc; double* ig4_den;
  // flow
  double* P[6];       // primitives + T with ghosts, buffer 0
  double* Pb[6];      // buffer 1 (the fused last sweep writes the next stage's primitives into the other buffer)
  double* G[3][4];    // D1 gradients of (u,v,w,T) along xi,eta,zeta (viscous)
  double* res;        // [5][N]
  double* U0;         // [5][N]
  double* inflow[6];
  meg6_grid* link[6];          // bc 5: the neighbour block of each face (meg6_link_blocks[_oriented])
  // orientation of the neighbour seen from this block ("each block possesses its own coordinate system"; R28, R29):
  // the cell with index vector h of THIS block (ghost ranges included) is the neighbour's cell m with
  //   m[lax[e]] = lsg[e] > 0 ? h[e] + lsh[e] : lsh[e] - h[e];   loff: added to the neighbour's coordinates seen from here
  int lax[6][3], lsg[6][3], lsh[6][3];
  double loff[6][3];
  bool rotated;                // some link of this block (or to it) is not the aligned one: ghost fills are repeated (R29)
  const double* ibuf[6];       // bc 5: or a packed copy of the neighbour's layers (meg6_set_interface_buffer)
  const double* gbuf[6];       // ... and of its cell-centre coordinates (meg6_set_geom_interface_buffer)
  double goff[6][3];
  const double* sigma; const double* uref;
  unsigned long long* stats;   // [2] device counters: limited, tested
  unsigned short* bmask[3];    // caller's branch-record arrays per interface family (meg6_set_branch_masks) or null
  double* red;                 // reduction scratch
  double* noalloc_scratch;     // device address of the library's static scratch array on this grid's device (meg6_cfl_dt_noalloc)
  int stats_on;
  bool have_metrics;
  int geom_blocked;            // -1 by size, 0 / 1 forced (MEG6_GEOM_BLOCKED in the environment at grid_create; tests)
  int geom_launches;           // kernels launched by the last metrics_compute
  // meg6_rk3_steps on static meshes: the launches of two consecutive steps (the period of the primitive-buffer parity)
  // captured once as a CUDA graph and replayed; the key is what the captured kernel arguments depend on
  double* tp;                  // 12 doubles: (sin, 2 pi omega cos) of the six stage times of a replayed two-step graph
  const double* tp_cur;        // non-null while such a graph is captured: where k_centres reads its two numbers
  cudaGraphExec_t steps_graph;
  struct GraphKey { const double* U; double dt; const double* sigma; const double* uref; int stats_on; unsigned short* bm[3]; } steps_key;
  // per-kernel timing (meg6_profile_*): event pairs of the launches since the last read
  int prof_on;
  std::vector<cudaEvent_t> prof_pool;
  struct ProfRec { int kind; int launches; size_t e0, e1; };
  std::vector<ProfRec> prof_recs;
  size_t prof_used;
};
