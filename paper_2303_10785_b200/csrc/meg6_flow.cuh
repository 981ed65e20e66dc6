// meg6_flow.cuh -- primitive conversion, ghost fill, stored gradients, CFL reduction.
// Residual assembly and the SSP-RK3 update (rows S, T) are fused into the last sweep, meg6_flux3.cuh.
#pragma once
#include "meg6_common.cuh"

namespace meg6 {

struct P5c { const double* p[5]; };
struct P6 { double* p[6]; };
struct P12 { double* p[12]; };

// G(a): Q -> P = (rho,u,v,w,p) (Eq. 5, P:83 inverted) and T = p/(rho R), interior cells.
__global__ void __launch_bounds__(256) k_prim(Consts c, const double* __restrict__ U, P6 P) {
  const long long N = c.LC.n;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= N) return;
  const int i = (int)(tid % c.n[0]), j = (int)((tid / c.n[0]) % c.n[1]), k = (int)(tid / ((long long)c.n[0] * c.n[1]));
  const double r = U[tid], ir = 1.0 / r;
  const double u = U[N + tid] * ir, v = U[2 * N + tid] * ir, w = U[3 * N + tid] * ir;
  const double p = (c.gamma - 1.0) * (U[4 * N + tid] - 0.5 * r * (u * u + v * v + w * w));
  const long long at = c.LP.at(i, j, k);
  P.p[0][at] = r; P.p[1][at] = u; P.p[2][at] = v; P.p[3][at] = w; P.p[4][at] = p;
  P.p[5][at] = p / (r * c.r_gas);
}

struct GhostIn {
  const double* inflow[2]; const double* mx; const double* my; const double* mz;
  // block interfaces (bc 5): field 0 of the neighbour's primitive buffer, its layout, field stride and cell count
  // along this direction, per side
  const double* nbP[2]; Lay nbL[2]; long long nbfs[2];
  int nax[2][3], nsg[2][3], nsh[2][3];   // index map home -> neighbour: m[nax[e]] = nsg[e] > 0 ? h[e] + nsh[e] : nsh[e] - h[e]
  // edge round of a multi-block fill (R28): only the sides with edge[side] set (faces linked to a block of this call),
  // over the ghost ranges of BOTH transverse directions -- an edge ghost cell beyond an interface is the neighbour's
  // own ghost cell there (its boundary rule with its face data), also where the other direction is filled later
  int edges, edge[2];
};

// B: ghost layers of direction d (6 deep), after the lower directions have been filled: periodic wrap, fixed
// inflow ghost = 2 P_in - P_mirror, outflow ghost = last interior cell with p = p_out where the outward normal
// Mach number is below one (Table 1, R20), walls (R27), block interfaces (R28).  One thread per GHOST CELL (all six fields): the twelve ghost
// cells of a xi line, or the xi-contiguous cells of an eta/zeta ghost layer, go to consecutive threads.
__global__ void __launch_bounds__(256) k_ghost(Consts c, int d, P6 P, GhostIn in) {
  int a = (d + 1) % 3, b = (d + 2) % 3;
  if (a > b) { int t = a; a = b; b = t; }
  constexpr int NG = 6;
  // transverse ranges: directions below d are already extended
  const int loa = (a < d || in.edges) ? -NG : 0, ea = c.n[a] + ((a < d || in.edges) ? 2 * NG : 0);
  const int lob = (b < d || in.edges) ? -NG : 0, eb = c.n[b] + ((b < d || in.edges) ? 2 * NG : 0);
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)ea * eb * 2 * NG) return;
  int qs, ta, tb;   // qs = layer + 6 * side
  if (d == 0) { qs = (int)(tid % (2 * NG)); const long long r = tid / (2 * NG); ta = loa + (int)(r % ea); tb = lob + (int)(r / ea); }
  else if (d == 1) { ta = loa + (int)(tid % ea); const long long r = tid / ea; qs = (int)(r % (2 * NG)); tb = lob + (int)(r / (2 * NG)); }
  else { ta = loa + (int)(tid % ea); const long long r = tid / ea; tb = lob + (int)(r % eb); qs = (int)(r / eb); }
  const int side = qs / NG, q = qs % NG + 1;   // q-th ghost layer, 1 = next to the boundary
  int ix[3];
  ix[a] = ta; ix[b] = tb; ix[d] = 0;
  const int n = c.n[d];
  const long long s = c.LP.stride(d);
  const long long base = c.LP.at(ix[0], ix[1], ix[2]);   // cell 0 of this line
  const int last = side ? n - 1 : 0, sg = side ? 1 : -1;
  const long long dst = base + (long long)(last + sg * q) * s;
  if (in.edges && !in.edge[side]) return;
  if (c.periodic[d]) {
    const long long src = side ? base + (long long)(q - 1) * s : base + (long long)(n - q) * s;
    double v[6];
#pragma unroll
    for (int f = 0; f < 6; ++f) v[f] = P.p[f][src];
#pragma unroll
    for (int f = 0; f < 6; ++f) P.p[f][dst] = v[f];
    return;
  }
  const int bc = c.bc[2 * d + side];
  // face data: interior positions; in the ghost columns of a periodic transverse direction the periodic image's
  const int ca = c.periodic[a] ? (ta % c.n[a] + c.n[a]) % c.n[a] : min(max(ta, 0), c.n[a] - 1);
  const int cb = c.periodic[b] ? (tb % c.n[b] + c.n[b]) % c.n[b] : min(max(tb, 0), c.n[b] - 1);
  // metric lookups of the wall / outflow rules: wherever the cell-centre metrics exist (five ghost layers; beyond a block
  // interface those are the neighbour's true metrics, R27 / R28)
  const int ma = min(max(ta, -5), c.n[a] + 4), mb = min(max(tb, -5), c.n[b] + 4);
  if (bc == 5) {
    // block interface (Table 1 last column; R28, R29): ghost layer q = the q-th interior cell of the neighbour
    // block counted from the face it shares with this one, at the transverse position the link's orientation gives
    int h[3], is[3];
    h[a] = ta; h[b] = tb; h[d] = last + sg * q;
#pragma unroll
    for (int e = 0; e < 3; ++e) {
      const int m = in.nsg[side][e] > 0 ? h[e] + in.nsh[side][e] : in.nsh[side][e] - h[e];
      const int ax = in.nax[side][e];
      if (ax == 0) is[0] = m; else if (ax == 1) is[1] = m; else is[2] = m;
    }
    const double* src = in.nbP[side] + in.nbL[side].at(is[0], is[1], is[2]);
    double v[6];
#pragma unroll
    for (int f = 0; f < 6; ++f) v[f] = src[f * in.nbfs[side]];
#pragma unroll
    for (int f = 0; f < 6; ++f) P.p[f][dst] = v[f];
  } else if (bc == 1) {
    const long long nf = (long long)c.n[a] * c.n[b];
    const double* pin = in.inflow[side] + (long long)cb * c.n[a] + ca;
    const long long mir = base + (long long)(last - sg * (q - 1)) * s;
    double v[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) v[f] = 2.0 * pin[f * nf] - P.p[f][mir];
#pragma unroll
    for (int f = 0; f < 5; ++f) P.p[f][dst] = v[f];
    P.p[5][dst] = v[4] / (v[0] * c.r_gas);
  } else if (bc == 3 || bc == 4) {
    // walls (Table 1, R27): rho and p of the mirror cell m; inviscid wall: velocity minus twice its
    // component along the unit vector of m's own hatted metrics of this direction; adiabatic wall: velocity negated
    const int m = last - sg * (q - 1);
    const long long mir = base + (long long)m * s;
    double pv[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) pv[f] = P.p[f][mir];
    if (bc == 3) {
      int im[3];
      im[a] = ma; im[b] = mb; im[d] = m;
      const long long am = c.LX.at(im[0], im[1], im[2]);
      const double mx = in.mx[am], my = in.my[am], mz = in.mz[am];
      const double gm = sqrt(mx * mx + my * my + mz * mz);
      const double kx = mx / gm, ky = my / gm, kz = mz / gm;
      const double V = pv[1] * kx + pv[2] * ky + pv[3] * kz;
      pv[1] = pv[1] - 2.0 * V * kx; pv[2] = pv[2] - 2.0 * V * ky; pv[3] = pv[3] - 2.0 * V * kz;
    } else {
      pv[1] = -pv[1]; pv[2] = -pv[2]; pv[3] = -pv[3];
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) P.p[f][dst] = pv[f];
    P.p[5][dst] = pv[4] / (pv[0] * c.r_gas);
  } else {
    double pv[5];
#pragma unroll
    for (int f = 0; f < 5; ++f) pv[f] = P.p[f][base + (long long)last * s];
    int im[3];
    im[a] = ma; im[b] = mb; im[d] = last;
    const long long am = c.LX.at(im[0], im[1], im[2]);
    const double mx = in.mx[am], my = in.my[am], mz = in.mz[am];
    const double gm = sqrt(mx * mx + my * my + mz * mz);
    const double cs = sqrt(c.gamma * pv[4] / pv[0]);
    const double mn = sg * (mx * pv[1] + my * pv[2] + mz * pv[3]) / (gm * cs);
    if (mn < 1.0) pv[4] = c.p_out;
#pragma unroll
    for (int f = 0; f < 5; ++f) P.p[f][dst] = pv[f];
    P.p[5][dst] = pv[4] / (pv[0] * c.r_gas);
  }
}

// B for a block that is periodic in all three directions (configs 1, 2, 3, 5): every ghost cell is the copy of the interior
// cell at the wrapped index -- what the three direction-ordered passes of k_ghost produce, value for value -- in ONE
// launch (the small configs are bound by launches: three ghost kernels were 45 % of a 32^3 stage).  One thread per
// ghost cell: the zeta slabs over the whole padded (i, j) extent, the eta slabs over the padded i extent, the xi slabs.
__global__ void __launch_bounds__(256) k_ghost_periodic(Consts c, P6 P) {
  constexpr int NG = 6;
  const int n0 = c.n[0], n1 = c.n[1], n2 = c.n[2];
  const long long e0 = n0 + 2 * NG, e1 = n1 + 2 * NG;
  const long long nz = e0 * e1 * (2 * NG), ny = e0 * (2 * NG) * n2, nx = (long long)(2 * NG) * n1 * n2;
  long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int i, j, k;
  if (tid < nz) {
    i = (int)(tid % e0) - NG; j = (int)((tid / e0) % e1) - NG;
    const int q = (int)(tid / (e0 * e1));
    k = q < NG ? q - NG : n2 + q - NG;
  } else if ((tid -= nz) < ny) {
    i = (int)(tid % e0) - NG;
    const int q = (int)((tid / e0) % (2 * NG));
    j = q < NG ? q - NG : n1 + q - NG;
    k = (int)(tid / (e0 * 2 * NG));
  } else if ((tid -= ny) < nx) {
    const int q = (int)(tid % (2 * NG));
    i = q < NG ? q - NG : n0 + q - NG;
    j = (int)((tid / (2 * NG)) % n1); k = (int)(tid / ((long long)(2 * NG) * n1));
  } else return;
  const int si = i < 0 ? i + n0 : i >= n0 ? i - n0 : i, sj = j < 0 ? j + n1 : j >= n1 ? j - n1 : j,
            sk = k < 0 ? k + n2 : k >= n2 ? k - n2 : k;
  const long long src = c.LP.at(si, sj, sk), dst = c.LP.at(i, j, k);
  double v[6];
#pragma unroll
  for (int f = 0; f < 6; ++f) v[f] = P.p[f][src];
#pragma unroll
  for (int f = 0; f < 6; ++f) P.p[f][dst] = v[f];
}

// Packed interface layers (meg6_stage_pack): the six cell layers of direction d next to one face, all six fields,
// every transverse position of the padded primitive array.  The packed array is a padded layout itself: as LP, but
// with 6 cells and no ghosts along d -- k_ghost reads it like a neighbour block that is six cells thick.
inline Lay pack_lay(const Lay& LP, int d) {
  Lay L = LP;
  if (d == 0) { L.gi = 0; L.pi = 6; } else if (d == 1) { L.gj = 0; L.pj = 6; } else { L.gk = 0; L.pk = 6; }
  L.sj = L.pi; L.sk = (long long)L.pi * L.pj; L.n = L.sk * L.pk;
  return L;
}

__global__ void __launch_bounds__(256) k_pack(Lay LP, Lay LQ, int d, int first, long long fsP, const double* __restrict__ P,
                                              double* __restrict__ out) {
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= LQ.n) return;
  const int pi = (int)(tid % LQ.pi), pj = (int)((tid / LQ.pi) % LQ.pj), pk = (int)(tid / LQ.sk);
  int ix[3] = {pi - LQ.gi, pj - LQ.gj, pk - LQ.gk};   // cell indices of the packed array
  ix[d] += first;                                     // ... of the source array
  const long long src = LP.at(ix[0], ix[1], ix[2]);
#pragma unroll
  for (int f = 0; f < 6; ++f) out[f * LQ.n + tid] = P[f * fsP + src];
}

// E6 gradient, Eq. 17 (R1)
__device__ __forceinline__ double d1_op(const double* __restrict__ f, long long s) {
  double r = CE1 * (f[s] - f[-s]);
  r = fma(CE2, f[2 * s] - f[-2 * s], r);
  r = fma(CE3, f[3 * s] - f[-3 * s], r);
  return r;
}

// G(b): stored gradients of (u,v,w,T) along xi and zeta on cells [-1, n+1)^3 (viscous flux, Fig. 5 P:295;
// R18: T is differentiated with the same E6 scheme).  G.p[4*e + f].
// A thread takes TWO xi-neighbouring cells (an aligned pair: every load and store is 16 bytes wide) and walks GRAD_KB cells
// along zeta: the zeta stencil re-uses its loads in registers, the xi stencils of the pair share one ten-value window
// (4 + 1 wide loads instead of 12 narrow ones; ncu r2: the one-cell form was bound by L1 wavefronts, 66-72 %, half of its
// instructions address arithmetic around 8.5 loads per value).  A block of 32 x 8 threads covers 64 x 8 x GRAD_KB cells.
// The eta gradients of the interior columns (0 <= i < ni, 0 <= k < nk) are stored by the eta sweep, which has them in its
// tiles; with eta_ghost_only they are formed here only in the ghost columns i = -1, ni and k = -1, nk, which no eta tile covers.
constexpr int GRAD_KB = 4;   // cells per thread along zeta (2 and 8: +10 %, r2c)
__device__ __forceinline__ double e6_vals(double m3, double m2, double m1, double p1, double p2, double p3) {   // as d1_op
  double r = CE1 * (p1 - m1);
  r = fma(CE2, p2 - m2, r);
  r = fma(CE3, p3 - m3, r);
  return r;
}
__global__ void __launch_bounds__(256, 4) k_grad(Consts c, P6 P, P12 G, int eta_ghost_only) {
  // i runs over the whole padded row of G (-GGI .. pitch-GGI): the cells beyond -1 and n are padding nobody reads, but
  // writing them makes every warp store start and end on a 32-byte sector (no partial-sector fills in L2/DRAM)
  const int i0 = 2 * (blockIdx.x * 32 + threadIdx.x) - GGI;     // even: the pair (i0, i0 + 1) is 16-byte aligned in P and G
  const int j = blockIdx.y * 8 + threadIdx.y - 1;
  const int k0 = blockIdx.z * GRAD_KB - 1;
  if (i0 >= c.LG.pi - GGI || j > c.n[1]) return;
  const long long sj = c.LP.sj, sk = c.LP.sk;
  const long long ap0 = c.LP.at(i0, j, k0), ag0 = c.LG.at(i0, j, k0);
#pragma unroll
  for (int f = 0; f < 4; ++f) {
    const double* __restrict__ q = P.p[(f < 3) ? f + 1 : 5] + ap0;
    double2 z[GRAD_KB + 6];
#pragma unroll
    for (int m = 0; m < GRAD_KB + 6; ++m)
      z[m] = (k0 + m - 3 <= c.n[2] + 3) ? *reinterpret_cast<const double2*>(q + (m - 3) * sk) : make_double2(0.0, 0.0);
#pragma unroll
    for (int m = 0; m < GRAD_KB; ++m) {
      // no early exit: the planes beyond n+1 are inside the 6-deep ghost padding of P, only the stores are guarded, so
      // the loads of the next cells can be issued before the stores of this one
      const bool ok = k0 + m <= c.n[2];
      const double* __restrict__ qq = q + m * sk;
      const long long ag = ag0 + m * c.LG.sk;
      const double2 a = *reinterpret_cast<const double2*>(qq - 4), b = *reinterpret_cast<const double2*>(qq - 2),
                    d = *reinterpret_cast<const double2*>(qq + 2), e = *reinterpret_cast<const double2*>(qq + 4);
      const double2 cc = z[m + 3];
      double2 vx, vz;
      vx.x = e6_vals(a.y, b.x, b.y, cc.y, d.x, d.y);
      vx.y = e6_vals(b.x, b.y, cc.x, d.x, d.y, e.x);
      vz.x = e6_vals(z[m].x, z[m + 1].x, z[m + 2].x, z[m + 4].x, z[m + 5].x, z[m + 6].x);
      vz.y = e6_vals(z[m].y, z[m + 1].y, z[m + 2].y, z[m + 4].y, z[m + 5].y, z[m + 6].y);
      if (ok) {
        *reinterpret_cast<double2*>(G.p[f] + ag) = vx;
        *reinterpret_cast<double2*>(G.p[8 + f] + ag) = vz;
        const bool kg = k0 + m < 0 || k0 + m >= c.n[2];
#pragma unroll
        for (int h = 0; h < 2; ++h)
          if (!eta_ghost_only || kg || i0 + h < 0 || i0 + h >= c.n[0]) G.p[4 + f][ag + h] = d1_op(qq + h, sj);
      }
    }
  }
}

// Eq. B.2 / B.3: per-block minima of 1/(|U|+c|grad xi|) and 1/(mu |grad xi|^2) over cells and
// directions (un-hatted metrics = hatted * J).  red[2*b], red[2*b+1]; the host finishes the reduction.
struct CflIn { const double* met[9]; const double* mt[3]; const double* rj; };

__device__ __forceinline__ double sutherland(const Consts& c, double T) {
  if (c.s_suth < 0.0) return c.mu_ref;
  const double r = T / c.t_ref;
  return c.mu_ref * r * sqrt(r) * (c.t_ref + c.s_suth) / (T + c.s_suth);
}

constexpr int CFL_BLOCKS = 1024;

__global__ void __launch_bounds__(256) k_cfl(Consts c, const double* __restrict__ U, CflIn in, double* __restrict__ red) {
  const long long N = c.LC.n;
  double inv_min = INFINITY, vis_min = INFINITY;
  for (long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x; tid < N; tid += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(tid % c.n[0]), j = (int)((tid / c.n[0]) % c.n[1]), k = (int)(tid / ((long long)c.n[0] * c.n[1]));
    const long long at = c.LX.at(i, j, k);
    const double r = U[tid], u = U[N + tid] / r, v = U[2 * N + tid] / r, w = U[3 * N + tid] / r;
    const double p = (c.gamma - 1.0) * (U[4 * N + tid] - 0.5 * r * (u * u + v * v + w * w));
    const double cs = sqrt(c.gamma * p / r), J = 1.0 / in.rj[at];
    const double mu = c.viscous ? sutherland(c, p / (r * c.r_gas)) : 0.0;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double mx = J * in.met[3 * d][at], my = J * in.met[3 * d + 1][at], mz = J * in.met[3 * d + 2][at];
      const double mtt = c.moving ? J * in.mt[d][at] : 0.0;
      const double gn = sqrt(mx * mx + my * my + mz * mz);
      inv_min = fmin(inv_min, 1.0 / (fabs(mtt + mx * u + my * v + mz * w) + cs * gn));
      if (c.viscous) vis_min = fmin(vis_min, 1.0 / (mu * gn * gn));
    }
  }
  __shared__ double sa[256], sb[256];
  sa[threadIdx.x] = inv_min; sb[threadIdx.x] = vis_min;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      sa[threadIdx.x] = fmin(sa[threadIdx.x], sa[threadIdx.x + o]);
      sb[threadIdx.x] = fmin(sb[threadIdx.x], sb[threadIdx.x + o]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { red[2 * blockIdx.x] = sa[0]; red[2 * blockIdx.x + 1] = sb[0]; }
}

// Volume-averaged kinetic energy and enstrophy (Eq. 54, in three dimensions with dV = 1/J): per-block sums
// of rho |u|^2/2 dV, rho |omega|^2/2 dV and dV.  The vorticity comes from the shared first gradients of the velocity
// -- E6 stencils of the primitive arrays, or the stored IG4 gradients for MIG4 -- through the chain rule with
// the cell-centre metrics.  red[3*b + {0,1,2}]; the host finishes the sums.
struct DiagIn { const double* met[9]; const double* rj; const double* P[4]; const double* g[9]; int ig4; };

__global__ void __launch_bounds__(256) k_diag(Consts c, DiagIn in, double* __restrict__ red) {
  const long long N = c.LC.n;
  double ke = 0.0, en = 0.0, vol = 0.0;
  for (long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x; tid < N; tid += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(tid % c.n[0]), j = (int)((tid / c.n[0]) % c.n[1]), k = (int)(tid / ((long long)c.n[0] * c.n[1]));
    const long long ax = c.LX.at(i, j, k), ap = c.LP.at(i, j, k);
    const double rj = in.rj[ax], J = 1.0 / rj;
    double gq[3][3];   // gq[d][comp]
#pragma unroll
    for (int d = 0; d < 3; ++d)
#pragma unroll
      for (int cc = 0; cc < 3; ++cc)
        gq[d][cc] = in.ig4 ? in.g[3 * d + cc][ap] : d1_op(in.P[1 + cc] + ap, c.LP.stride(d));
    double dv[3][3];   // dv[comp][x]
#pragma unroll
    for (int cc = 0; cc < 3; ++cc)
#pragma unroll
      for (int x = 0; x < 3; ++x)
        dv[cc][x] = J * (in.met[x][ax] * gq[0][cc] + in.met[3 + x][ax] * gq[1][cc] + in.met[6 + x][ax] * gq[2][cc]);
    const double ox = dv[2][1] - dv[1][2], oy = dv[0][2] - dv[2][0], oz = dv[1][0] - dv[0][1];
    const double r = in.P[0][ap], u = in.P[1][ap], v = in.P[2][ap], w = in.P[3][ap];
    ke += r * 0.5 * (u * u + v * v + w * w) * rj;
    en += r * 0.5 * (ox * ox + oy * oy + oz * oz) * rj;
    vol += rj;
  }
  __shared__ double sa[256], sb[256], sc[256];
  sa[threadIdx.x] = ke; sb[threadIdx.x] = en; sc[threadIdx.x] = vol;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      sa[threadIdx.x] += sa[threadIdx.x + o]; sb[threadIdx.x] += sb[threadIdx.x + o]; sc[threadIdx.x] += sc[threadIdx.x + o];
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) { red[3 * blockIdx.x] = sa[0]; red[3 * blockIdx.x + 1] = sb[0]; red[3 * blockIdx.x + 2] = sc[0]; }
}

}  // namespace meg6
