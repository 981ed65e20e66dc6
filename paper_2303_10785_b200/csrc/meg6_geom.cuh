// meg6_geom.cuh -- metric / Jacobian kernels (paper Sec. 4 and 7).
#pragma once
#include "meg6_common.cuh"

namespace meg6 {

struct GeomIn {
  const double* node[3];
  const double* mode[3];
  double s, sd;   // sin(2 pi omega t), 2 pi omega cos(2 pi omega t)
  const double* tp;   // or, if not null: the same two numbers in device memory (tp[0], tp[1]; replayed CUDA graphs)
};

// 8-vertex mean of node positions x0 + s*mode (vel == false) or node velocities sd*mode.
__device__ __forceinline__ double cell_mean(const Consts& c, const GeomIn& g, int comp, bool vel, int i, int j, int k) {
  const long long sj = c.n[0] + 1, sk = (long long)(c.n[0] + 1) * (c.n[1] + 1);
  const long long b = (long long)k * sk + (long long)j * sj + i;
  const long long o[8] = {0, 1, sj, sj + 1, sk, sk + 1, sk + sj, sk + sj + 1};
  double acc = 0.0;
  const double gs = g.tp ? g.tp[0] : g.s, gsd = g.tp ? g.tp[1] : g.sd;
#pragma unroll
  for (int q = 0; q < 8; ++q) {
    double v;
    if (vel) v = gsd * g.mode[comp][b + o[q]];
    else {
      v = g.node[comp][b + o[q]];
      if (c.moving) v = v + gs * g.mode[comp][b + o[q]];
    }
    acc = (q == 0) ? v : acc + v;
  }
  return acc / 8.0;
}

struct P3 { double* p[3]; };
struct P9 { double* p[9]; };

// M1a: cell-centre coordinates (and grid velocities) of the interior cells: 8-vertex mean.
__global__ void __launch_bounds__(256) k_centres(Consts c, GeomIn g, P3 xc, P3 xt) {
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= c.LC.n) return;
  const int i = (int)(tid % c.n[0]), j = (int)((tid / c.n[0]) % c.n[1]), k = (int)(tid / ((long long)c.n[0] * c.n[1]));
  const long long at = c.LX.at(i, j, k);
#pragma unroll
  for (int comp = 0; comp < 3; ++comp) {
    xc.p[comp][at] = cell_mean(c, g, comp, false, i, j, k);
    if (c.moving) xt.p[comp][at] = cell_mean(c, g, comp, true, i, j, k);
  }
}

// M1b: ghost layers of direction d (R13, R14), after the lower directions: periodic -> image -/+ period (velocities:
// plain copy); otherwise linear extrapolation of the last spacing.  The same values, operation by operation, as the
// recursive definition ext_val (xi innermost, zeta outermost).  One thread per ghost cell.
// Block-interface faces (bc 5; R28, R29): the ghost cell centres are the neighbour block's own cell centres (plus the
// period across a wrap-around link) -- both blocks then difference the same coordinates across their common face, and
// the interface metrics of a cut mesh are those of the uncut one, bit for bit.  Per side: field 0 of the neighbour's
// coordinate (velocity) array, or of a packed copy of its ten layers next to the face; index map as in k_ghost.
struct ExtIn {
  const double* nbx[2][3]; const double* nbv[2][3]; Lay nbL[2];
  int nax[2][3], nsg[2][3], nsh[2][3];
  double off[2][3];
};

__global__ void __launch_bounds__(256) k_extend(Consts c, int d, P3 xc, P3 xt, ExtIn in) {
  int a = (d + 1) % 3, b = (d + 2) % 3;
  if (a > b) { int t = a; a = b; b = t; }
  const int loa = (a < d) ? -GX : 0, ea = c.n[a] + ((a < d) ? 2 * GX : 0);
  const int lob = (b < d) ? -GX : 0, eb = c.n[b] + ((b < d) ? 2 * GX : 0);
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)ea * eb * 2 * GX) return;
  int qs, ta, tb;
  if (d == 0) { qs = (int)(tid % (2 * GX)); const long long r = tid / (2 * GX); ta = loa + (int)(r % ea); tb = lob + (int)(r / ea); }
  else if (d == 1) { ta = loa + (int)(tid % ea); const long long r = tid / ea; qs = (int)(r % (2 * GX)); tb = lob + (int)(r / (2 * GX)); }
  else { ta = loa + (int)(tid % ea); const long long r = tid / ea; tb = lob + (int)(r % eb); qs = (int)(r / eb); }
  const int side = qs / GX, q = qs % GX + 1;
  const int n = c.n[d];
  const int ai = side ? n - 1 + q : -q;          // ghost index along d
  int ix[3];
  ix[a] = ta; ix[b] = tb; ix[d] = 0;
  const long long base = c.LX.at(ix[0], ix[1], ix[2]), s = c.LX.stride(d);
  const long long dst = base + (long long)ai * s;
#pragma unroll
  for (int comp = 0; comp < 3; ++comp) {
#pragma unroll
    for (int vel = 0; vel < 2; ++vel) {
      if (vel && !c.moving) continue;
      double* f = vel ? xt.p[comp] : xc.p[comp];
      const double* nbf = vel ? in.nbv[side][comp] : in.nbx[side][comp];
      if (!c.periodic[d] && c.bc[2 * d + side] == 5 && nbf) {
        int h[3], is[3];
        h[a] = ta; h[b] = tb; h[d] = ai;
#pragma unroll
        for (int e = 0; e < 3; ++e) {
          const int m = in.nsg[side][e] > 0 ? h[e] + in.nsh[side][e] : in.nsh[side][e] - h[e];
          const int ax = in.nax[side][e];
          if (ax == 0) is[0] = m; else if (ax == 1) is[1] = m; else is[2] = m;
        }
        const double v = nbf[in.nbL[side].at(is[0], is[1], is[2])];
        f[dst] = vel ? v : v + in.off[side][comp];
      } else if (c.periodic[d]) {
        const double off = vel ? 0.0 : c.period[d][comp];
        f[dst] = side ? f[base + (long long)(ai - n) * s] + off : f[base + (long long)(ai + n) * s] - off;
      } else if (!side) {
        const double v0 = f[base], v1 = f[base + s];
        f[dst] = v0 - (double)(-ai) * (v1 - v0);
      } else {
        const double v0 = f[base + (long long)(n - 1) * s], v1 = f[base + (long long)(n - 2) * s];
        f[dst] = v0 + (double)(ai - (n - 1)) * (v0 - v1);
      }
    }
  }
}

// M1b for a block that is periodic in all three directions: every ghost cell centre in ONE launch.  The three
// direction-ordered passes give  ((interior -+ period_xi) -+ period_eta) -+ period_zeta  with the offsets of the directions
// in which the index wrapped, added in that order; the same additions in the same order here (bit-identical), velocities
// plain copies.  One thread per ghost cell: zeta slabs over the padded (i, j) extent, eta slabs over padded i, xi slabs.
__global__ void __launch_bounds__(256) k_extend_periodic(Consts c, P3 xc, P3 xt) {
  const int n0 = c.n[0], n1 = c.n[1], n2 = c.n[2];
  const long long e0 = n0 + 2 * GX, e1 = n1 + 2 * GX;
  const long long nz = e0 * e1 * (2 * GX), ny = e0 * (2 * GX) * n2, nx = (long long)(2 * GX) * n1 * n2;
  long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  int i, j, k;
  if (tid < nz) {
    i = (int)(tid % e0) - GX; j = (int)((tid / e0) % e1) - GX;
    const int q = (int)(tid / (e0 * e1));
    k = q < GX ? q - GX : n2 + q - GX;
  } else if ((tid -= nz) < ny) {
    i = (int)(tid % e0) - GX;
    const int q = (int)((tid / e0) % (2 * GX));
    j = q < GX ? q - GX : n1 + q - GX;
    k = (int)(tid / (e0 * 2 * GX));
  } else if ((tid -= ny) < nx) {
    const int q = (int)(tid % (2 * GX));
    i = q < GX ? q - GX : n0 + q - GX;
    j = (int)((tid / (2 * GX)) % n1); k = (int)(tid / ((long long)(2 * GX) * n1));
  } else return;
  const int wi = i < 0 ? -1 : i >= n0 ? 1 : 0, wj = j < 0 ? -1 : j >= n1 ? 1 : 0, wk = k < 0 ? -1 : k >= n2 ? 1 : 0;
  const long long src = c.LX.at(i - wi * n0, j - wj * n1, k - wk * n2), dst = c.LX.at(i, j, k);
#pragma unroll
  for (int comp = 0; comp < 3; ++comp) {
    double v = xc.p[comp][src];
    if (wi) v = wi > 0 ? v + c.period[0][comp] : v - c.period[0][comp];
    if (wj) v = wj > 0 ? v + c.period[1][comp] : v - c.period[1][comp];
    if (wk) v = wk > 0 ? v + c.period[2][comp] : v - c.period[2][comp];
    xc.p[comp][dst] = v;
    if (c.moving) xt.p[comp][dst] = xt.p[comp][src];
  }
}

// Packed cell-centre layers of one face (meg6_stage_geom_pack): the ten layers of direction d next to the face over the
// whole padded transverse extent, coordinates (and grid velocities).  The packed array is a padded layout itself: LX
// with ten cells and no ghosts along d; k_extend of the receiving block reads it like a neighbour ten cells thick.
inline Lay geom_pack_lay(const Lay& LX, int d) {
  Lay L = LX;
  if (d == 0) { L.gi = 0; L.pi = GX; } else if (d == 1) { L.gj = 0; L.pj = GX; } else { L.gk = 0; L.pk = GX; }
  L.sj = L.pi; L.sk = (long long)L.pi * L.pj; L.n = L.sk * L.pk;
  return L;
}
struct P6c { const double* p[6]; };
__global__ void __launch_bounds__(256) k_pack_geom(Lay LX, Lay LQ, int d, int first, int nf, P6c src, double* __restrict__ out) {
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= LQ.n) return;
  const int pi = (int)(tid % LQ.pi), pj = (int)((tid / LQ.pi) % LQ.pj), pk = (int)(tid / LQ.sk);
  int ix[3] = {pi - LQ.gi, pj - LQ.gj, pk - LQ.gk};
  ix[d] += first;
  const long long at = LX.at(ix[0], ix[1], ix[2]);
  for (int f = 0; f < nf; ++f) out[f * LQ.n + tid] = src.p[f][at];
}

// ---- linear operators in the paper's own step-by-step form (Eq. 17, 19, 16, 36-38), evaluated in exactly
// the order the discretisation states them.  This translation unit is compiled with -fmad=false: at low Mach
// number a relative metric perturbation of 1e-15 is amplified by p/(rho u^2 k h) ~ 1e4 in the flux
// difference, so the metric arithmetic is kept free of contraction-dependent rounding.
// x / 12, correctly rounded, in three operations instead of the division sequence (the metric kernels are bound by the
// FP64 pipe, ncu r1m, and delta_vals divides three times).  y = RN(1/12); q = RN(x y) is within 1.5 ulp of x/12;
// r = x - 12 q is exact (a multiple of 4 ulp(q), at most 18 ulp(q)); q + r y differs from x/12 by less than 2e-16 ulp(q),
// while x/12 = (x/3)/4 sits on a third of an ulp -- at least 1/6 ulp from every rounding boundary -- so the last
// rounding gives RN(x/12), the value the oracle's division gives (no overflow or underflow at metric magnitudes;
// x = 0 gives 0).  The fma is explicit: -fmad=false only forbids contraction.
__device__ __forceinline__ double div12(double x) {
  constexpr double y = 1.0 / 12.0;
  const double q = x * y;
  const double r = fma(-12.0, q, x);
  return fma(r, y, q);
}

__device__ __forceinline__ double e6(const double* v) {   // Eq. 17 (R1) at v[0]
  return 3.0 / 4.0 * (v[1] - v[-1]) - 3.0 / 20.0 * (v[2] - v[-2]) + 1.0 / 60.0 * (v[3] - v[-3]);
}
// Products with 2, -2, 0.5 and -0.5 are exact (no underflow at metric magnitudes), so a * b + c with such an a is
// written as fma(a, b, c): the same single rounding as the multiply-then-add of the stated formula, one operation less.
// consistent derivative Eq. 37 at the centre v[5] of 11 consecutive values v[0..10]
__device__ __forceinline__ double delta_vals(const double* v) {
  const double* c = v + 5;
  double d1[5], d2[3];
#pragma unroll
  for (int j = -2; j <= 2; ++j) d1[j + 2] = e6(c + j);
#pragma unroll
  for (int j = -1; j <= 1; ++j)   // Eq. 19
    d2[j + 1] = fma(-0.5, d1[j + 3] - d1[j + 1], 2.0 * (fma(-2.0, c[j], c[j + 1]) + c[j - 1]));
  const double q0 = div12(d2[0]), q1 = div12(d2[1]), q2 = div12(d2[2]);
  const double Lm = fma(0.5, d1[1], c[-1]) + q0;    // Eq. 16: left state of face -1/2
  const double R0 = fma(-0.5, d1[2], c[0]) + q1;    // right state of face -1/2
  const double L0 = fma(0.5, d1[2], c[0]) + q1;     // left state of face +1/2
  const double Rp = fma(-0.5, d1[3], c[1]) + q2;    // right state of face +1/2
  // Eq. 36-37: H+ - H- with H = 0.5 (L + R); the halves are exact, so one scaling of the difference
  return 0.5 * ((L0 + Rp) - (Lm + R0));
}
// central interface value Eq. 38 between v[4] and v[5] of 10 consecutive values v[0..9]
__device__ __forceinline__ double H_vals(const double* v) {
  double d1[4], d2[2];
#pragma unroll
  for (int j = 0; j < 4; ++j) d1[j] = e6(v + 3 + j);
#pragma unroll
  for (int j = 0; j < 2; ++j)
    d2[j] = fma(-0.5, d1[j + 2] - d1[j], 2.0 * (fma(-2.0, v[4 + j], v[5 + j]) + v[3 + j]));
  const double L = fma(0.5, d1[1], v[4]) + div12(d2[0]);
  const double R = fma(-0.5, d1[2], v[5]) + div12(d2[1]);
  return 0.5 * (L + R);
}

__device__ __forceinline__ double delta_op(const double* __restrict__ f, long long s) {
  double v[11];
#pragma unroll
  for (int m = 0; m < 11; ++m) v[m] = f[(m - 5) * s];
  return delta_vals(v);
}

// M2: cd[3*comp + d] = delta_d(x_comp) wherever the 11-point stencil fits inside the padded box.
__global__ void k_coord_deriv(Consts c, P3 xc, P9 cd, double* __restrict__ rj) {
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= c.LX.n) return;
  const int pi = (int)(tid % c.LX.pi);
  const int pj = (int)((tid / c.LX.pi) % c.LX.pj);
  const int pk = (int)(tid / c.LX.sk);
  const int pos[3] = {pi, pj, pk};
  const int ext[3] = {c.n[0] + 2 * GX, c.n[1] + 2 * GX, c.n[2] + 2 * GX};
  if (pi >= ext[0]) return;
  double v[9];
  bool all = true;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (pos[d] < 5 || pos[d] >= ext[d] - 5) { all = false; continue; }
    const long long s = c.LX.stride(d);
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
      v[3 * comp + d] = delta_op(xc.p[comp] + tid, s);
      cd.p[3 * comp + d][tid] = v[3 * comp + d];
    }
  }
  if (all) {   // 1/J = det of the coordinate derivatives, Eq. 13, on cells [-5, n+5)^3
    const double xx = v[0], xe = v[1], xz = v[2], yx = v[3], ye = v[4], yz = v[5], zx = v[6], ze = v[7], zz = v[8];
    rj[tid] = xx * (ye * zz - ze * yz) - yx * (xe * zz - ze * xz) + zx * (xe * yz - ye * xz);
  }
}

// M2, blocked along zeta: a thread takes KB consecutive cells of a zeta column.  The three zeta derivatives of the
// block share their E6 gradients, second derivatives, one-sided states and interface values in registers (33 FP64
// operations per derivative instead of 76 at KB = 6; the kernel is FP64-pipe-bound, ncu r1m); the xi and eta derivatives
// are formed per cell as before.  Every value goes through the operations of delta_vals in its order (bit-identical).
constexpr int CD_KB = 6;      // cells of a zeta column per thread (measured: 4 and 8 no better, r1m)
template <int KB>
__global__ void __launch_bounds__(256) k_coord_deriv_blk(Consts c, P3 xc, P9 cd, double* __restrict__ rj) {
  const int ext[3] = {c.n[0] + 2 * GX, c.n[1] + 2 * GX, c.n[2] + 2 * GX};
  const int nb = (ext[2] + KB - 1) / KB;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)c.LX.pi * c.LX.pj * nb) return;
  const int pi = (int)(tid % c.LX.pi);
  const int pj = (int)((tid / c.LX.pi) % c.LX.pj);
  const int pk0 = (int)(tid / ((long long)c.LX.pi * c.LX.pj)) * KB;
  if (pi >= ext[0] || pj >= ext[1]) return;
  const long long a0 = (long long)pk0 * c.LX.sk + (long long)pj * c.LX.sj + pi, sk = c.LX.sk;
  double dz[3][KB];
#pragma unroll
  for (int comp = 0; comp < 3; ++comp) {
    const double* __restrict__ p = xc.p[comp] + a0;
    double v[KB + 10], d1[KB + 10], hl[KB + 10], hr[KB + 10], H[KB + 10];   // index m <-> plane pk0 + m - 5
#pragma unroll
    for (int m = 0; m < KB + 10; ++m) v[m] = p[(long long)(min(max(pk0 + m - 5, 0), ext[2] - 1) - pk0) * sk];
#pragma unroll
    for (int m = 3; m <= KB + 6; ++m) d1[m] = e6(v + m);
#pragma unroll
    for (int m = 4; m <= KB + 5; ++m) {
      const double d2 = fma(-0.5, d1[m + 1] - d1[m - 1], 2.0 * (fma(-2.0, v[m], v[m + 1]) + v[m - 1]));   // Eq. 19
      const double qd = div12(d2);
      hl[m] = fma(0.5, d1[m], v[m]) + qd;          // Eq. 16: state of plane m at its face +1/2
      hr[m] = fma(-0.5, d1[m], v[m]) + qd;         //         and at its face -1/2
    }
#pragma unroll
    for (int m = 4; m <= KB + 4; ++m) H[m] = hl[m] + hr[m + 1];       // twice the interface value of face m+1/2
#pragma unroll
    for (int b = 0; b < KB; ++b) dz[comp][b] = 0.5 * (H[b + 5] - H[b + 4]);   // Eq. 36-37 as in delta_vals
  }
#pragma unroll
  for (int b = 0; b < KB; ++b) {
    const int pk = pk0 + b;
    if (pk >= ext[2]) break;
    const long long at = a0 + b * sk;
    const int pos[3] = {pi, pj, pk};
    double v[9];
    bool all = true;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      if (pos[d] < 5 || pos[d] >= ext[d] - 5) { all = false; continue; }
      const long long s = c.LX.stride(d);
#pragma unroll
      for (int comp = 0; comp < 3; ++comp) {
        v[3 * comp + d] = (d == 2) ? dz[comp][b] : delta_op(xc.p[comp] + at, s);
        cd.p[3 * comp + d][at] = v[3 * comp + d];
      }
    }
    if (all) {   // 1/J = det of the coordinate derivatives, Eq. 13, on cells [-5, n+5)^3
      const double xx = v[0], xe = v[1], xz = v[2], yx = v[3], ye = v[4], yz = v[5], zx = v[6], ze = v[7], zz = v[8];
      rj[at] = xx * (ye * zz - ze * yz) - yx * (xe * zz - ze * xz) + zx * (xe * yz - ye * xz);
    }
  }
}

// M3 (tiled): the Thomas-Lombard metrics, Eq. 10, one sweep per direction D.  Every metric is
//     m[r][c] = delta_b( delta_a(q) s ) - delta_a( delta_b(q) s ),  (a,b) = (r+1,r+2), (q,s) = (c+1,c+2) mod 3,
// so direction D carries six consistent derivatives: the FIRST terms of row (D+1)%3 and the SECOND terms of row
// (D+2)%3.  A CTA forms the six products on a pencil tile (5-cell halo along D) in shared memory once, each thread
// then differentiates them for its cell (delta_vals: the operation order of Eq. 17/19/16/36-37, bit for bit the
// oracle's).  Sweeps run in the order D = 0, 1, 2; the second term to arrive completes the metric with the one
// subtraction of Eq. 10 (the first to arrive is parked in the metric array itself).  The last sweep also forms the
// hatted time metrics, Eq. 11.  (ncu r1: the one-thread-per-cell version read ~400 values per cell through
// L1 and took 60 % of a moving-mesh RK stage.  The same tiling applied to the coordinate derivatives and the
// interface metrics -- one array at a time through shared memory -- was measured SLOWER than their L1 versions.)
template <int D>
struct MetCfg {
  static constexpr int TS = (D == 0) ? 64 : 8;     // cells along D per tile
  static constexpr int TW = (D == 0) ? 4 : 32;     // transverse extent: rows j (D = 0) or xi lanes (D != 0)
  static constexpr int LS = TS + 10;
};

template <int D>
__global__ void __launch_bounds__(256) k_met_dir(Consts c, P3 xc, P3 xt, P9 cd, P9 met, P3 mt) {
  using C = MetCfg<D>;
  constexpr int TS = C::TS, TW = C::TW, LS = C::LS;
  __shared__ double sp[6 * LS * TW];
  auto sidx = [](int p, int pos, int t) { return (D == 0) ? (p * TW + t) * LS + pos : (p * LS + pos) * TW + t; };
  // tile origin (cells); outputs cover [-5, n+5) in every direction
  int o[3];
  if (D == 0) { o[0] = -5 + (int)blockIdx.x * TS; o[1] = -5 + (int)blockIdx.y * TW; o[2] = -5 + (int)blockIdx.z; }
  else if (D == 1) { o[0] = -5 + (int)blockIdx.x * TW; o[1] = -5 + (int)blockIdx.y * TS; o[2] = -5 + (int)blockIdx.z; }
  else { o[0] = -5 + (int)blockIdx.x * TW; o[1] = -5 + (int)blockIdx.z; o[2] = -5 + (int)blockIdx.y * TS; }   // zeta tiles of a line back to back: halo planes re-used in L2
  constexpr int TD = (D == 0) ? 1 : 0;             // the transverse direction inside the tile
  constexpr int A_RB = (D + 2) % 3, B_RA = (D + 1) % 3;
  const int tid = threadIdx.x;
  // ---- the six products on the tile, positions -5 .. TS+4 along D (clamped inside the padded arrays) ----
  for (int it = tid; it < LS * TW; it += 256) {
    int pos, t;
    if (D == 0) { pos = it % LS; t = it / LS; } else { t = it % TW; pos = it / TW; }
    int ix[3] = {o[0], o[1], o[2]};
    ix[D] = min(o[D] + pos - 5, c.n[D] + GX - 1);
    ix[TD] = min(o[TD] + t, c.n[TD] + GX - 1);
    const long long at = c.LX.at(ix[0], ix[1], ix[2]);
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
      const int q = (cc + 1) % 3, sc = (cc + 2) % 3;
      const double xs = xc.p[sc][at];
      sp[sidx(cc, pos, t)] = cd.p[3 * q + A_RB][at] * xs;        // first terms of row (D+1)%3
      sp[sidx(3 + cc, pos, t)] = cd.p[3 * q + B_RA][at] * xs;    // second terms of row (D+2)%3
    }
  }
  __syncthreads();
  int s, t;
  if (D == 0) { s = tid % TS; t = tid / TS; } else { t = tid % TW; s = tid / TW; }
  int ix[3] = {o[0], o[1], o[2]};
  ix[D] += s; ix[TD] += t;
  if (ix[0] >= c.n[0] + 5 || ix[1] >= c.n[1] + 5 || ix[2] >= c.n[2] + 5) return;
  const long long at = c.LX.at(ix[0], ix[1], ix[2]);
  constexpr int RB = (D + 1) % 3, RA = (D + 2) % 3;
  constexpr int SP = (D == 0) ? 1 : TW;            // shared-memory stride along D
  double mrb[3], mra[3];
#pragma unroll
  for (int cc = 0; cc < 3; ++cc) {
    double v[11];
#pragma unroll
    for (int m = 0; m < 11; ++m) v[m] = sp[sidx(cc, s, t) + m * SP];
    const double d1 = delta_vals(v);
#pragma unroll
    for (int m = 0; m < 11; ++m) v[m] = sp[sidx(3 + cc, s, t) + m * SP];
    const double d2 = delta_vals(v);
    // row RB: D is its b; its a = (D+2)%3 has already run iff a < D, i.e. D != 0
    mrb[cc] = (D == 0) ? d1 : d1 - met.p[3 * RB + cc][at];
    // row RA: D is its a; its b = (D+1)%3 has already run iff b < D, i.e. D == 2
    mra[cc] = (D == 2) ? met.p[3 * RA + cc][at] - d2 : d2;
    met.p[3 * RB + cc][at] = mrb[cc];
    met.p[3 * RA + cc][at] = mra[cc];
  }
  if (D == 2 && c.moving) {   // rows 0 (= RB) and 1 (= RA) are final here, row 2 was finished by the eta sweep
    const double vx = xt.p[0][at], vy = xt.p[1][at], vz = xt.p[2][at];
    mt.p[0][at] = -(vx * mrb[0] + vy * mrb[1] + vz * mrb[2]);
    mt.p[1][at] = -(vx * mra[0] + vy * mra[1] + vz * mra[2]);
    mt.p[2][at] = -(vx * met.p[6][at] + vy * met.p[7][at] + vz * met.p[8][at]);
  }
}

// Central interface value Eq. 38: face f lies between cells f-1 and f.
__device__ __forceinline__ double H_op(const double* __restrict__ f /* at cell f */, long long s) {
  double v[10];
#pragma unroll
  for (int m = 0; m < 10; ++m) v[m] = f[(m - 5) * s];
  return H_vals(v);
}

struct FaceJob { const double* src[11]; double* dst[11]; int n; };

// M4: interface arrays of family d: each hatted quantity (and 1/J) interpolated as a whole.
__global__ void k_face_metrics(Consts c, int d, FaceJob job) {
  const Lay& LF = c.LF[d];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= LF.n) return;
  const int i = (int)(tid % LF.pi), j = (int)((tid / LF.pi) % LF.pj), k = (int)(tid / LF.sk);
  const long long at = c.LX.at(i, j, k), s = c.LX.stride(d);
  for (int q = 0; q < job.n; ++q) job.dst[q][tid] = H_op(job.src[q] + at, s);
}

// M4, the three families in one launch (blockIdx.y = family): on small grids each family alone is less than one wave of
// CTAs (64^3: 1040 of 1184 slots, three launches of 10 us each)
struct FaceJob3 { FaceJob job[3]; };
__global__ void k_face_metrics3(Consts c, FaceJob3 jobs) {
  const int d = blockIdx.y;
  const Lay& LF = c.LF[d];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= LF.n) return;
  const int i = (int)(tid % LF.pi), j = (int)((tid / LF.pi) % LF.pj), k = (int)(tid / LF.sk);
  const long long at = c.LX.at(i, j, k), s = c.LX.stride(d);
  const FaceJob& job = jobs.job[d];
  for (int q = 0; q < job.n; ++q) job.dst[q][tid] = H_op(job.src[q] + at, s);
}

// M4 for the eta and zeta families: a thread forms KB consecutive interfaces of one grid line.  Neighbouring
// interfaces share the E6 gradients, second derivatives and one-sided states of their cells, which the thread keeps in
// registers: 30 FP64 operations per interface instead of 56 at KB = 4 (k_face_metrics is FP64-pipe-bound, ncu r1m);
// the operations on every value are those of H_vals, in its order (bit-identical results).  Lanes run along xi.
constexpr int FACE_KB = 6;    // interfaces of a grid line per thread
template <int KB>
__global__ void __launch_bounds__(256) k_face_metrics_blk(Consts c, int d, FaceJob job) {
  const Lay& LF = c.LF[d];
  const int nfd = (d == 1) ? LF.pj : LF.pk, nb = (nfd + KB - 1) / KB, no = (d == 1) ? LF.pk : LF.pj;
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)LF.pi * nb * no) return;
  const int i = (int)(tid % LF.pi);
  const long long r = tid / LF.pi;
  int j, k, f0;
  if (d == 1) { f0 = (int)(r % nb) * KB; j = f0; k = (int)(r / nb); }
  else { j = (int)(r % LF.pj); f0 = (int)(r / LF.pj) * KB; k = f0; }
  const long long at = c.LX.at(i, j, k), s = c.LX.stride(d);
  const long long ao = LF.at(i, j, k), so = LF.stride(d);
  const int lim = c.n[d] + GX - 1 - f0;            // last cell inside the padded array, relative to f0
  for (int q = 0; q < job.n; ++q) {
    const double* __restrict__ p = job.src[q] + at;
    double v[KB + 9], d1[KB + 9], hl[KB + 9], hr[KB + 9];   // index m <-> cell f0 + m - 5
#pragma unroll
    for (int m = 0; m < KB + 9; ++m) v[m] = p[(long long)min(m - 5, lim) * s];
#pragma unroll
    for (int m = 3; m <= KB + 5; ++m) d1[m] = e6(v + m);
#pragma unroll
    for (int m = 4; m <= KB + 4; ++m) {
      const double d2 = fma(-0.5, d1[m + 1] - d1[m - 1], 2.0 * (fma(-2.0, v[m], v[m + 1]) + v[m - 1]));   // Eq. 19
      const double qd = div12(d2);
      hl[m] = fma(0.5, d1[m], v[m]) + qd;          // Eq. 16: state of cell m at its face +1/2
      hr[m] = fma(-0.5, d1[m], v[m]) + qd;         //         and at its face -1/2
    }
#pragma unroll
    for (int b = 0; b < KB; ++b)
      if (f0 + b < nfd) job.dst[q][ao + b * so] = 0.5 * (hl[b + 4] + hr[b + 5]);   // Eq. 38
  }
}

// M5: GCL, Eq. 14: (1/J)_t = -sum_d [ (m_t)_{+1/2} - (m_t)_{-1/2} ] of the interface values above.
__global__ void k_rjt(Consts c, const double* __restrict__ f0, const double* __restrict__ f1,
                      const double* __restrict__ f2, double* __restrict__ rjt) {
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= c.LC.n) return;
  const int i = (int)(tid % c.n[0]), j = (int)((tid / c.n[0]) % c.n[1]), k = (int)(tid / ((long long)c.n[0] * c.n[1]));
  const long long a0 = c.LF[0].at(i, j, k), a1 = c.LF[1].at(i, j, k), a2 = c.LF[2].at(i, j, k);
  const double d0 = f0[a0 + 1] - f0[a0];
  const double d1 = f1[a1 + c.LF[1].sj] - f1[a1];
  const double d2 = f2[a2 + c.LF[2].sk] - f2[a2];
  rjt[tid] = -(d0 + d1 + d2);
}

}  // namespace meg6
