/*
 * meg6_oracle.cpp -- CPU ORACLE (test infrastructure, NOT the product path).
 *
 * Plain FP64 restatement, step by step and in the paper's order, of the per-RK-stage right-hand
 * side of arXiv 2303.10785 (MEG6 gradients + characteristic gradient-based reconstruction + improved
 * MP limiter + contravariant HLLC + alpha-damping viscous flux + freestream-preserving conservative
 * metrics + SSP-RK3).  "P:n" cites line n of /root/reference/PAPER.md; "Rn" cites a reading of a
 * garbled / silent passage listed in DESIGN.md (section "Readings").
 *
 * No tiling, no fusion: whole padded arrays, one loop nest per formula.  Build with
 * -O2 -ffp-contract=off.  OpenMP only splits the outermost loop of each nest.
 *
 * Parity status of individual readings ("parity unpinned" = nothing in the paper or the mathematics
 * fixes the choice; oracle and CUDA path simply share the reading):
 *   - eigenvector averaging state (R5), MP alpha value (R7), tangential viscous gradients (R11),
 *     un-hatted interface metrics (R12), Sutherland constants (R15), sponge form (R16),
 *     WHICH inflow/outflow ghost rules the garbled Table 1 meant (R20; the rules as read are pinned: the box is the
 *     inner part of a longer periodic box holding the ghost states, tests/test_oracle_inout.py),
 *     the VALUE of the alpha in Eq. B.3 (R25; the formula around it is pinned),
 *     the cell whose metrics give the wall normal of the inviscid-wall rule (R27),
 *     where the IG4 line systems of the MIG4 variant end and how they are closed (R26):
 *     parity unpinned.
 *     (block interfaces, R28, are pinned: cut domain == uncut domain)
 *   - everything else is pinned by tests/test_oracle_*.py (-m "not gpu"); in particular the grid-velocity path
 *     (node velocities P:166, time metrics Eq. 11, interface time metric, GCL Eq. 14, stage times of Eq. B.1 / R17) by
 *     tests/test_oracle_moving.py (rigidly translating mesh in closed form, stationary vortex on a deforming mesh
 *     P:573-579, third order in time) and meg6o_cfl_dt (Eq. B.2/B.3) by tests/test_oracle_cfl.py (closed forms).
 */
#include "meg6_oracle.h"

#include <algorithm>
#include <cassert>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

int g_threads = 1;

#ifdef _OPENMP
#define OMP_FOR _Pragma("omp parallel for schedule(static) num_threads(g_threads)")
#else
#define OMP_FOR
#endif

/* ------------------------------------------------------------------------------------------ */
/* Padded 3-D array with a uniform ghost depth g; index (i,j,k), i fastest; valid box [lo,hi). */
struct Arr {
  int n[3] = {0, 0, 0};
  int g = 0;
  int lo[3] = {0, 0, 0}, hi[3] = {0, 0, 0};
  std::vector<double> d;
  Arr() {}
  Arr(const int nn[3], int gg) { init(nn, gg); }
  void init(const int nn[3], int gg) {
    g = gg;
    for (int a = 0; a < 3; ++a) { n[a] = nn[a]; lo[a] = 0; hi[a] = nn[a]; }
    d.assign((size_t)(n[0] + 2 * g) * (n[1] + 2 * g) * (n[2] + 2 * g),
             std::numeric_limits<double>::quiet_NaN());
  }
  ptrdiff_t stride(int a) const {
    return a == 0 ? 1 : a == 1 ? (ptrdiff_t)(n[0] + 2 * g) : (ptrdiff_t)(n[0] + 2 * g) * (n[1] + 2 * g);
  }
  size_t idx(int i, int j, int k) const {
    return ((size_t)(k + g) * (n[1] + 2 * g) + (size_t)(j + g)) * (n[0] + 2 * g) + (size_t)(i + g);
  }
  double& operator()(int i, int j, int k) { return d[idx(i, j, k)]; }
  double operator()(int i, int j, int k) const { return d[idx(i, j, k)]; }
  void valid_all() { for (int a = 0; a < 3; ++a) { lo[a] = -g; hi[a] = n[a] + g; } }
  void free_mem() { std::vector<double>().swap(d); }
};

/* out(valid box) = fn(pointer to centre of `in`, stride along dir); the valid box of `in` shrinks by
 * rl cells on the low side and rh on the high side along dir. */
template <class F>
void line_apply(const Arr& in, int dir, int rl, int rh, Arr& out, F fn) {
  out.init(in.n, in.g);
  for (int a = 0; a < 3; ++a) { out.lo[a] = in.lo[a]; out.hi[a] = in.hi[a]; }
  out.lo[dir] += rl; out.hi[dir] -= rh;
  const ptrdiff_t s = in.stride(dir);
  OMP_FOR
  for (int k = out.lo[2]; k < out.hi[2]; ++k)
    for (int j = out.lo[1]; j < out.hi[1]; ++j)
      for (int i = out.lo[0]; i < out.hi[0]; ++i)
        out(i, j, k) = fn(&in.d[in.idx(i, j, k)], s);
}

/* out = fn(a, b) pointwise on the intersection of valid boxes */
template <class F>
void point_apply2(const Arr& a, const Arr& b, Arr& out, F fn) {
  out.init(a.n, a.g);
  for (int c = 0; c < 3; ++c) { out.lo[c] = std::max(a.lo[c], b.lo[c]); out.hi[c] = std::min(a.hi[c], b.hi[c]); }
  OMP_FOR
  for (int k = out.lo[2]; k < out.hi[2]; ++k)
    for (int j = out.lo[1]; j < out.hi[1]; ++j)
      for (int i = out.lo[0]; i < out.hi[0]; ++i)
        out(i, j, k) = fn(a(i, j, k), b(i, j, k));
}

/* ---------------------------------- 1-D operators ----------------------------------------- */
/* Eq. 17, explicit sixth-order gradient E6; the printed "+" inside the brackets are "-" (R1). */
inline double op_D1(const double* f, ptrdiff_t s) {
  return 3.0 / 4.0 * (f[s] - f[-s]) - 3.0 / 20.0 * (f[2 * s] - f[-2 * s]) + 1.0 / 60.0 * (f[3 * s] - f[-3 * s]);
}
/* Eq. D.2 fourth-order explicit central difference (negative control only). */
inline double op_C4(const double* f, ptrdiff_t s) {
  return 2.0 / 3.0 * (f[s] - f[-s]) - 1.0 / 12.0 * (f[2 * s] - f[-2 * s]);
}
/* Eq. 19: second derivative from values and first gradients (hats = cell values, R4). */
inline double op_D2(const double* f, const double* f1, ptrdiff_t s) {
  return 2.0 * (f[s] - 2.0 * f[0] + f[-s]) - 0.5 * (f1[s] - f1[-s]);
}
/* Eq. 16: value at i+1/2 seen from cell i (Lft) and at i-1/2 seen from cell i (Rgt). */
inline double op_Lft(double f, double f1, double f2) { return f + 0.5 * f1 + f2 / 12.0; }
inline double op_Rgt(double f, double f1, double f2) { return f - 0.5 * f1 + f2 / 12.0; }

/* Eq. 18, implicit fourth-order gradient IG4 (the printed "+" are "-", R2):
 *     alpha f'_{i-1} + f'_i + alpha f'_{i+1} = (2+alpha)/3 (f_{i+1}-f_{i-1}) + (4 alpha-1)/12 (f_{i+2}-f_{i-2}),
 * alpha = 5/14, one tridiagonal system along every grid line of the array.  The paper does not say where the
 * systems end (R26): here a system spans every cell of the padded line whose right-hand side exists, and its
 * first and last unknowns are given by the explicit fourth-order difference of Eq. D.2 (same reach, same order).
 * Thomas algorithm, written out: forward  den_i = 1 - alpha c_{i-1}, c_i = alpha/den_i,
 * d_i = (r_i - alpha d_{i-1})/den_i ;  backward  x_i = d_i - c_i x_{i+1}. */
const double IG4_ALPHA = 5.0 / 14.0;
void grad_ig4(const Arr& f, int dir, Arr& out) {
  out.init(f.n, f.g);
  for (int a = 0; a < 3; ++a) { out.lo[a] = f.lo[a]; out.hi[a] = f.hi[a]; }
  out.lo[dir] += 2; out.hi[dir] -= 2;
  const int m = out.hi[dir] - out.lo[dir];
  if (m < 3) { out.hi[dir] = out.lo[dir]; return; }
  const double al = IG4_ALPHA, ca = (2.0 + al) / 3.0, cb = (4.0 * al - 1.0) / 12.0;
  std::vector<double> cc(m, 0.0), den(m, 1.0);
  for (int q = 1; q < m - 1; ++q) { den[q] = 1.0 - al * cc[q - 1]; cc[q] = al / den[q]; }
  const ptrdiff_t s = f.stride(dir);
  const int a1 = (dir + 1) % 3, a2 = (dir + 2) % 3;
  OMP_FOR
  for (int v = out.lo[a2]; v < out.hi[a2]; ++v)
    for (int u = out.lo[a1]; u < out.hi[a1]; ++u) {
      int ix[3];
      ix[a1] = u; ix[a2] = v; ix[dir] = out.lo[dir];
      const double* pf = &f.d[f.idx(ix[0], ix[1], ix[2])];
      double* px = &out.d[out.idx(ix[0], ix[1], ix[2])];
      px[0] = op_C4(pf, s);                                        /* first unknown: explicit */
      for (int q = 1; q < m - 1; ++q) {
        const double* c = pf + q * s;
        const double r = ca * (c[s] - c[-s]) + cb * (c[2 * s] - c[-2 * s]);
        px[q * s] = (r - al * px[(q - 1) * s]) / den[q];
      }
      px[(m - 1) * s] = op_C4(pf + (m - 1) * s, s);                /* last unknown: explicit */
      for (int q = m - 2; q >= 1; --q) px[q * s] = px[q * s] - cc[q] * px[(q + 1) * s];
    }
}
/* first gradient of a whole array along dir (scheme 0: MEG6 = E6, Eq. 17; scheme 1: MIG4 = IG4, Eq. 18) */
void grad_dir(const Arr& f, int dir, int scheme, Arr& out) {
  if (scheme == 1) { grad_ig4(f, dir, out); return; }
  line_apply(f, dir, 3, 3, out, [](const double* p, ptrdiff_t s) { return op_D1(p, s); });
}
void grad_c4(const Arr& f, int dir, Arr& out) {
  line_apply(f, dir, 2, 2, out, [](const double* p, ptrdiff_t s) { return op_C4(p, s); });
}
/* second derivative Eq. 19 from f and its gradient f1 (same dir) */
void d2_dir(const Arr& f, const Arr& f1, int dir, Arr& out) {
  out.init(f.n, f.g);
  for (int a = 0; a < 3; ++a) { out.lo[a] = std::max(f.lo[a], f1.lo[a]); out.hi[a] = std::min(f.hi[a], f1.hi[a]); }
  out.lo[dir] += 1; out.hi[dir] -= 1;
  const ptrdiff_t s = f.stride(dir);
  OMP_FOR
  for (int k = out.lo[2]; k < out.hi[2]; ++k)
    for (int j = out.lo[1]; j < out.hi[1]; ++j)
      for (int i = out.lo[0]; i < out.hi[0]; ++i) {
        size_t c = f.idx(i, j, k);
        out(i, j, k) = op_D2(&f.d[c], &f1.d[c], s);
      }
}
/* Eq. 36/38: central interface value H at i+1/2 = average of the L and R states.
 * Index i of `out` means the interface between cell i and cell i+1 along dir.  `c4` selects the
 * App. D variant (gradients by Eq. D.2) used only by the negative control. */
void H_dir(const Arr& f, int dir, int scheme, bool c4, Arr& out) {
  Arr f1, f2;
  if (c4) grad_c4(f, dir, f1); else grad_dir(f, dir, scheme, f1);
  d2_dir(f, f1, dir, f2);
  out.init(f.n, f.g);
  for (int a = 0; a < 3; ++a) { out.lo[a] = f2.lo[a]; out.hi[a] = f2.hi[a]; }
  out.hi[dir] -= 1;
  const ptrdiff_t s = f.stride(dir);
  OMP_FOR
  for (int k = out.lo[2]; k < out.hi[2]; ++k)
    for (int j = out.lo[1]; j < out.hi[1]; ++j)
      for (int i = out.lo[0]; i < out.hi[0]; ++i) {
        size_t c = f.idx(i, j, k);
        double L = op_Lft(f.d[c], f1.d[c], f2.d[c]);
        double R = op_Rgt(f.d[c + s], f1.d[c + s], f2.d[c + s]);
        out(i, j, k) = 0.5 * (L + R);
      }
}
/* Eq. 37: consistent derivative = difference of the two central interface values. */
void delta_from_H(const Arr& H, int dir, Arr& out) {
  line_apply(H, dir, 1, 0, out, [](const double* p, ptrdiff_t s) { return p[0] - p[-s]; });
}
void delta_dir(const Arr& f, int dir, int scheme, Arr& out) {
  Arr H;
  H_dir(f, dir, scheme, false, H);
  delta_from_H(H, dir, out);
}

inline double sgn(double a) { return (a > 0.0) - (a < 0.0); }
/* E.2 */
inline double minmod(double a, double b) { return 0.5 * (sgn(a) + sgn(b)) * std::min(std::fabs(a), std::fabs(b)); }

}  // namespace

/* ------------------------------------------------------------------------------------------ */
struct meg6o_grid {
  meg6o_params p;
  int n[3];
  std::vector<double> xn, yn, zn, dxm, dym, dzm;   /* nodes */
  /* geometry at the time of the last metrics_compute */
  Arr xc[3];         /* cell-centre coordinates, ghost 10 */
  Arr xt[3];         /* cell-centre grid velocities (moving meshes), ghost 10 */
  Arr met[9];        /* hatted metrics at cell centres, valid on [-5,n+5) */
  Arr rj;            /* 1/J */
  Arr mt[3];         /* hatted time metrics */
  Arr fmet[3][10];   /* interface metrics per family: 9 hatted + 1/J (all ten only if viscous) */
  Arr fmt[3];        /* interface time metric of the family's own direction */
  Arr rjt;           /* (1/J)_t, interior */
  bool have_metrics = false;
  bool user_centres = false;   /* tests only: cell centres (ghosts included) supplied directly */
  /* flow scratch */
  Arr P[6];          /* rho,u,v,w,p,T, ghost 6 */
  Arr G1[3][6];      /* D1 gradients */
  std::vector<double> inflow[6];
  std::vector<double> sigma, uref;
  unsigned long long n_limited = 0, n_tested = 0;
  /* branch record of the last right-hand side (tests: which interfaces took which branch), per interface family:
   * bit r (0..4) = left state of characteristic component r failed E.1, bit 5+r = right state, bits 10-11 = branch
   * 0..3 of Eq. 26.  Interface index along d runs over n_d + 1, i fastest. */
  bool want_masks = false;
  std::vector<unsigned short> mask[3];
  meg6o_grid* link[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};   /* bc 5: neighbour block per face */
  /* orientation of the neighbour seen from this block (Sec. 6: "each block possesses its own coordinate
   * system"; R28/R29): a cell with index vector h of THIS block (ghost ranges included) is the neighbour's cell m with
   * m[lax[e]] = lsg[e] > 0 ? h[e] + lsh[e] : lsh[e] - h[e]; loff = what is added to the neighbour's coordinates when
   * they are seen from here (zero, or the period vector across a wrap-around link) */
  int lax[6][3], lsg[6][3], lsh[6][3];
  double loff[6][3];
  bool rotated = false;            /* some link is not the aligned one: the ghost fills are repeated (R29) */
  bool thin_nb = false;            /* a neighbour has fewer cells along the link than the coordinate ghost depth: its own
                                      ghost coordinates (from ITS neighbour) are read, so the extension runs twice */
  const double* ibuf[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr}; /* bc 5: or packed neighbour layers */
  const double* gbuf[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr}; /* ... and packed cell-centre layers */
  double goff[6][3];
};

namespace {

const int GX = 10; /* ghost depth of coordinates (two nested delta of reach 5, R13/R19) */
const int GP = 6;  /* ghost depth of primitives (R19) */

/* O1.3: extend a cell-centre array along dir: periodic image + offset, or linear extrapolation (R13, R14), or -- at a
 * block-interface face (bc 5) -- the neighbour block's own cell centres (R28: the two blocks then difference the same
 * coordinates across their common face, so the interface metrics of the cut are those of the uncut mesh).
 * comp = coordinate component (0..2) of `a`, vel: `a` is a grid-velocity array (no offsets).  which: 0 -> G->xc, 1 -> xt
 * of the neighbour (passed in nbarr per face, null where the face is no linked interface). */
void extend_dir(Arr& a, int dir, bool periodic, double offset, const meg6o_grid* G = nullptr, int comp = 0,
                const Arr* const nbarr[2] = nullptr, bool vel = false) {
  const int n = a.n[dir], g = a.g;
  int lo[3], hi[3];
  for (int c = 0; c < 3; ++c) { lo[c] = a.lo[c]; hi[c] = a.hi[c]; }
  for (int k = (dir == 2 ? 0 : lo[2]); k < (dir == 2 ? 1 : hi[2]); ++k)
    for (int j = (dir == 1 ? 0 : lo[1]); j < (dir == 1 ? 1 : hi[1]); ++j)
      for (int i = (dir == 0 ? 0 : lo[0]); i < (dir == 0 ? 1 : hi[0]); ++i) {
        double* base = &a.d[a.idx(i, j, k)];   /* index 0 along dir */
        const ptrdiff_t s = a.stride(dir);
        for (int q = 1; q <= g; ++q) {
          if (periodic) {
            base[-q * s] = base[(n - q) * s] - offset;
            base[(n - 1 + q) * s] = base[(q - 1) * s] + offset;
            continue;
          }
          for (int side = 0; side < 2; ++side) {
            const int face = 2 * dir + side;
            const int hd = side ? n - 1 + q : -q;
            double v;
            if (G && G->p.bc[face] == 5 && nbarr && nbarr[side]) {
              int h[3] = {i, j, k}, m[3];
              h[dir] = hd;
              for (int e = 0; e < 3; ++e)
                m[G->lax[face][e]] = G->lsg[face][e] > 0 ? h[e] + G->lsh[face][e] : G->lsh[face][e] - h[e];
              v = (*nbarr[side])(m[0], m[1], m[2]) + (vel ? 0.0 : G->loff[face][comp]);
            } else if (G && G->p.bc[face] == 5 && G->gbuf[face]) {
              /* packed layers of a remote neighbour (meg6o_stage_geom_pack on its side): [vel*3 + comp][tb][ta][l] */
              int ta = (dir == 0) ? j : i, tb = (dir == 2) ? j : k;
              int e1 = (dir == 0) ? 1 : 0, e2 = (dir == 2) ? 1 : 2;
              const size_t ea = a.n[e1] + 2 * GX, eb = a.n[e2] + 2 * GX;
              const int l = side ? q - 1 : GX - q;
              v = G->gbuf[face][((((size_t)(vel ? 3 : 0) + comp) * eb + (size_t)(tb + GX)) * ea + (size_t)(ta + GX)) * GX + l] +
                  (vel ? 0.0 : G->goff[face][comp]);
            } else if (!side) {
              v = base[0] - q * (base[s] - base[0]);
            } else {
              v = base[(n - 1) * s] + q * (base[(n - 1) * s] - base[(n - 2) * s]);
            }
            base[hd * s] = v;
          }
        }
      }
  a.lo[dir] = -g; a.hi[dir] = n + g;
}

/* O1.2: cell centre = mean of the 8 vertices */
void cell_mean(const meg6o_grid& G, const std::vector<double>& nodes, Arr& out) {
  const int ni = G.n[0], nj = G.n[1], nk = G.n[2];
  out.init(G.n, GX);
  const size_t sj = ni + 1, sk = (size_t)(ni + 1) * (nj + 1);
  for (int k = 0; k < nk; ++k)
    for (int j = 0; j < nj; ++j)
      for (int i = 0; i < ni; ++i) {
        size_t b = (size_t)k * sk + (size_t)j * sj + i;
        out(i, j, k) = (nodes[b] + nodes[b + 1] + nodes[b + sj] + nodes[b + sj + 1] + nodes[b + sk] +
                        nodes[b + sk + 1] + nodes[b + sk + sj] + nodes[b + sk + sj + 1]) / 8.0;
      }
}

void interior_copy(const Arr& a, double* out) {
  size_t m = 0;
  for (int k = 0; k < a.n[2]; ++k)
    for (int j = 0; j < a.n[1]; ++j)
      for (int i = 0; i < a.n[0]; ++i) out[m++] = a(i, j, k);
}

}  // namespace

extern "C" {

void meg6o_set_threads(int n) { g_threads = n < 1 ? 1 : n; }
int meg6o_get_threads(void) { return g_threads; }

meg6o_grid* meg6o_create(const meg6o_params* p, const double* x, const double* y, const double* z,
                         const double* dxm, const double* dym, const double* dzm) {
  for (int f = 0; f < 6; ++f)   /* Table 1 gives the wall rules without a wall velocity: static meshes only (R27) */
    if (p->moving && !p->periodic[f / 2] && (p->bc[f] == 3 || p->bc[f] == 4)) return nullptr;
  meg6o_grid* G = new meg6o_grid();
  G->p = *p;
  G->n[0] = p->ni; G->n[1] = p->nj; G->n[2] = p->nk;
  size_t nn = (size_t)(p->ni + 1) * (p->nj + 1) * (p->nk + 1);
  G->xn.assign(x, x + nn); G->yn.assign(y, y + nn); G->zn.assign(z, z + nn);
  if (p->moving) { G->dxm.assign(dxm, dxm + nn); G->dym.assign(dym, dym + nn); G->dzm.assign(dzm, dzm + nn); }
  return G;
}

void meg6o_destroy(meg6o_grid* G) { delete G; }

/* ---------------------------------- O1 geometry ------------------------------------------- */
namespace {
/* O1.1-O1.2: node positions and analytic node velocities (form of Eq. 49-50), cell centres */
void geom_centres(meg6o_grid* G, double t) {
  const meg6o_params& p = G->p;
  const double two_pi = 2.0 * M_PI;
  const std::vector<double>* base[3] = {&G->xn, &G->yn, &G->zn};
  const std::vector<double>* mode[3] = {&G->dxm, &G->dym, &G->dzm};
  for (int c = 0; c < 3; ++c) {
    if (G->user_centres) continue;
    if (p.moving) {
      const double s = std::sin(two_pi * p.omega * t), sd = two_pi * p.omega * std::cos(two_pi * p.omega * t);
      std::vector<double> pos(base[c]->size()), vel(base[c]->size());
      for (size_t q = 0; q < pos.size(); ++q) { pos[q] = (*base[c])[q] + s * (*mode[c])[q]; vel[q] = sd * (*mode[c])[q]; }
      cell_mean(*G, pos, G->xc[c]);
      cell_mean(*G, vel, G->xt[c]);
    } else {
      cell_mean(*G, *base[c], G->xc[c]);
    }
  }
}
/* O1.3 ghost layers of direction d (after the lower directions; with several blocks: direction d in every block
 * before direction d+1 in any, like the ghost fill of the primitives) */
void geom_extend(meg6o_grid* G, int d) {
  const meg6o_params& p = G->p;
  if (G->user_centres) return;
  for (int c = 0; c < 3; ++c) {
    const Arr* nbx[2] = {nullptr, nullptr};
    const Arr* nbv[2] = {nullptr, nullptr};
    for (int side = 0; side < 2; ++side) {
      const meg6o_grid* nb = (!p.periodic[d] && p.bc[2 * d + side] == 5) ? G->link[2 * d + side] : nullptr;
      if (nb) {
        if (nb->xc[c].d.empty()) { fprintf(stderr, "meg6o geometry: the neighbour block has no cell centres yet (use meg6o_metrics_compute_blocks)\n"); abort(); }
        nbx[side] = &nb->xc[c]; nbv[side] = &nb->xt[c];
      }
    }
    extend_dir(G->xc[c], d, p.periodic[d] != 0, p.period[d][c], G, c, nbx, false);
    if (p.moving) extend_dir(G->xt[c], d, p.periodic[d] != 0, 0.0, G, c, nbv, true);
  }
}
void geom_finish(meg6o_grid* G);
}  // namespace

/* geometry of several linked blocks: centres everywhere, then the ghost coordinates direction by direction over all
 * blocks (repeated where a link is rotated, R29), then each block's metrics */
void meg6o_metrics_compute_blocks(int nb, meg6o_grid* const* G, double t) {
  bool rot = false, thin = false;
  for (int b = 0; b < nb; ++b) { geom_centres(G[b], t); rot = rot || G[b]->rotated; thin = thin || G[b]->thin_nb; }
  for (int pass = 0; pass < (rot ? 3 : thin ? 2 : 1); ++pass)
    for (int d = 0; d < 3; ++d)
      for (int b = 0; b < nb; ++b) geom_extend(G[b], d);
  for (int b = 0; b < nb; ++b) geom_finish(G[b]);
}

void meg6o_metrics_compute(meg6o_grid* G, double t) { meg6o_metrics_compute_blocks(1, &G, t); }

/* staged geometry for blocks in different processes (the caller carries the packed cell-centre layers) */
void meg6o_stage_geom_centres(meg6o_grid* G, double t) { geom_centres(G, t); }
void meg6o_stage_geom_extend(meg6o_grid* G, int d) { geom_extend(G, d); }
void meg6o_stage_geom_finish(meg6o_grid* G) { geom_finish(G); }
size_t meg6o_geom_interface_doubles(const meg6o_grid* G, int face) {
  const int d = face / 2;
  const int e1 = (d == 0) ? 1 : 0, e2 = (d == 2) ? 1 : 2;
  return (size_t)(G->p.moving ? 6 : 3) * GX * (G->n[e1] + 2 * GX) * (G->n[e2] + 2 * GX);
}
void meg6o_set_geom_interface_buffer(meg6o_grid* G, int face, const double* layers, const double* off) {
  G->gbuf[face] = layers;
  for (int c = 0; c < 3; ++c) G->goff[face][c] = off ? off[c] : 0.0;
}
void meg6o_stage_geom_pack(meg6o_grid* G, int face, double* layers) {
  const int d = face / 2, side = face & 1;
  if (G->n[d] < GX) { fprintf(stderr, "meg6o_stage_geom_pack: a block must be at least %d cells thick along a remote link\n", GX); abort(); }
  const int e1 = (d == 0) ? 1 : 0, e2 = (d == 2) ? 1 : 2;
  const size_t ea = G->n[e1] + 2 * GX, eb = G->n[e2] + 2 * GX;
  const int first = side ? G->n[d] - GX : 0;
  for (int f = 0; f < (G->p.moving ? 6 : 3); ++f) {
    const Arr& a = (f < 3) ? G->xc[f] : G->xt[f - 3];
    for (int tb = -GX; tb < G->n[e2] + GX; ++tb)
      for (int ta = -GX; ta < G->n[e1] + GX; ++ta)
        for (int l = 0; l < GX; ++l) {
          int is[3]; is[e1] = ta; is[e2] = tb; is[d] = first + l;
          layers[((f * eb + (size_t)(tb + GX)) * ea + (size_t)(ta + GX)) * GX + l] = a.d[a.idx(is[0], is[1], is[2])];
        }
  }
}

namespace {
void geom_finish(meg6o_grid* G) {
  const meg6o_params& p = G->p;
  const int sch = p.scheme;
  Arr* xt = G->xt;
  auto mul = [](double a, double b) { return a * b; };
  auto sub = [](double a, double b) { return a - b; };

  /* derivatives of the coordinates: c_d[c][d] = d(coordinate c)/d(direction d) */
  Arr cd[3][3];
  for (int c = 0; c < 3; ++c)
    for (int d = 0; d < 3; ++d) {
      if (p.metric_form == 0) delta_dir(G->xc[c], d, sch, cd[c][d]);
      else grad_c4(G->xc[c], d, cd[c][d]);
    }

  if (p.metric_form == 0) {
    /* O1.4 Thomas-Lombard conservative metrics, Eq. 10; every derivative is the consistent
     * delta of Eq. 36-37.  met[3*r + c]: r = xi,eta,zeta ; c = x,y,z.
     * Row r uses directions (a,b) = (eta,zeta), (zeta,xi), (xi,eta); component c uses coordinates
     * (q,s) = (y,z), (z,x), (x,y):   m = delta_b( delta_a(q) * s ) - delta_a( delta_b(q) * s ).        */
    for (int r = 0; r < 3; ++r) {
      const int a = (r + 1) % 3, b = (r + 2) % 3;
      for (int c = 0; c < 3; ++c) {
        const int q = (c + 1) % 3, s = (c + 2) % 3;
        Arr t1, t2, d1, d2;
        point_apply2(cd[q][a], G->xc[s], t1, mul);   /* delta_a(q) * s */
        point_apply2(cd[q][b], G->xc[s], t2, mul);   /* delta_b(q) * s */
        delta_dir(t1, b, sch, d1);
        delta_dir(t2, a, sch, d2);
        point_apply2(d1, d2, G->met[3 * r + c], sub);
      }
    }
  } else {
    /* App. D: non-conservative products of fourth-order central differences */
    for (int r = 0; r < 3; ++r) {
      const int a = (r + 1) % 3, b = (r + 2) % 3;
      for (int c = 0; c < 3; ++c) {
        const int q = (c + 1) % 3, s = (c + 2) % 3;
        Arr t1, t2;
        point_apply2(cd[q][a], cd[s][b], t1, mul);
        point_apply2(cd[q][b], cd[s][a], t2, mul);
        point_apply2(t1, t2, G->met[3 * r + c], sub);
      }
    }
  }
  /* O1.5 Jacobian, Eq. 13: determinant of the coordinate derivatives */
  {
    Arr& rj = G->rj;
    rj.init(G->n, GX);
    for (int a = 0; a < 3; ++a) {
      rj.lo[a] = -GX; rj.hi[a] = G->n[a] + GX;
      for (int c = 0; c < 3; ++c)
        for (int d = 0; d < 3; ++d) { rj.lo[a] = std::max(rj.lo[a], cd[c][d].lo[a]); rj.hi[a] = std::min(rj.hi[a], cd[c][d].hi[a]); }
    }
    OMP_FOR
    for (int k = rj.lo[2]; k < rj.hi[2]; ++k)
      for (int j = rj.lo[1]; j < rj.hi[1]; ++j)
        for (int i = rj.lo[0]; i < rj.hi[0]; ++i) {
          const double xx = cd[0][0](i, j, k), yx = cd[1][0](i, j, k), zx = cd[2][0](i, j, k);
          const double xe = cd[0][1](i, j, k), ye = cd[1][1](i, j, k), ze = cd[2][1](i, j, k);
          const double xz = cd[0][2](i, j, k), yz = cd[1][2](i, j, k), zz = cd[2][2](i, j, k);
          rj(i, j, k) = xx * (ye * zz - ze * yz) - yx * (xe * zz - ze * xz) + zx * (xe * yz - ye * xz);
        }
  }
  /* O1.6 time metrics at cell centres, Eq. 11 in hatted form */
  if (p.moving) {
    for (int r = 0; r < 3; ++r) {
      Arr& m = G->mt[r];
      const Arr &mx = G->met[3 * r], &my = G->met[3 * r + 1], &mz = G->met[3 * r + 2];
      m.init(G->n, GX);
      for (int a = 0; a < 3; ++a) { m.lo[a] = mx.lo[a]; m.hi[a] = mx.hi[a]; }
      OMP_FOR
      for (int k = m.lo[2]; k < m.hi[2]; ++k)
        for (int j = m.lo[1]; j < m.hi[1]; ++j)
          for (int i = m.lo[0]; i < m.hi[0]; ++i)
            m(i, j, k) = -(xt[0](i, j, k) * mx(i, j, k) + xt[1](i, j, k) * my(i, j, k) + xt[2](i, j, k) * mz(i, j, k));
    }
  }
  /* O1.7 interface metrics: each hatted quantity interpolated as a whole, Eq. 38 */
  const bool c4 = (p.metric_form != 0);
  for (int d = 0; d < 3; ++d) {
    for (int q = 0; q < 10; ++q) {
      const bool own = (q >= 3 * d && q < 3 * d + 3);
      if (!own && !p.viscous) { G->fmet[d][q].free_mem(); continue; }
      H_dir(q < 9 ? G->met[q] : G->rj, d, sch, c4, G->fmet[d][q]);
    }
    if (p.moving) H_dir(G->mt[d], d, sch, c4, G->fmt[d]);
  }
  /* O1.8 GCL, Eq. 14: differences of exactly the interface values of step 7 */
  if (p.moving) {
    Arr d0, d1, d2;
    delta_from_H(G->fmt[0], 0, d0);
    delta_from_H(G->fmt[1], 1, d1);
    delta_from_H(G->fmt[2], 2, d2);
    G->rjt.init(G->n, 0);
    OMP_FOR
    for (int k = 0; k < G->n[2]; ++k)
      for (int j = 0; j < G->n[1]; ++j)
        for (int i = 0; i < G->n[0]; ++i) G->rjt(i, j, k) = -(d0(i, j, k) + d1(i, j, k) + d2(i, j, k));
  }
  G->have_metrics = true;
}
}  // namespace

/* tests only: supply padded cell-centre coordinates [(nk+20)(nj+20)(ni+20)] (ghost depth 10) directly,
 * bypassing O1.1-O1.3, so that single coefficients of the metric stencils can be probed (Eq. 43). */
void meg6o_set_centres(meg6o_grid* G, const double* xc, const double* yc, const double* zc) {
  const double* src[3] = {xc, yc, zc};
  for (int c = 0; c < 3; ++c) {
    G->xc[c].init(G->n, GX);
    G->xc[c].valid_all();
    std::copy(src[c], src[c] + G->xc[c].d.size(), G->xc[c].d.begin());
  }
  G->user_centres = true;
}

void meg6o_set_inflow(meg6o_grid* G, int face, const double* P_in) {
  const int d = face / 2, a = (d + 1) % 3, b = (d + 2) % 3;
  (void)a; (void)b;
  int n1, n2;
  if (d == 0) { n1 = G->n[1]; n2 = G->n[2]; } else if (d == 1) { n1 = G->n[0]; n2 = G->n[2]; } else { n1 = G->n[0]; n2 = G->n[1]; }
  G->inflow[face].assign(P_in, P_in + (size_t)5 * n1 * n2);
}

void meg6o_set_sponge(meg6o_grid* G, const double* sigma, const double* U_ref) {
  size_t N = (size_t)G->n[0] * G->n[1] * G->n[2];
  if (!sigma) { G->sigma.clear(); G->uref.clear(); return; }
  G->sigma.assign(sigma, sigma + N);
  G->uref.assign(U_ref, U_ref + 5 * N);
}

/* ------------------------------- pieces of the flux --------------------------------------- */

/* App. A, de-garbled (R6): left (A.6a) and right (A.4b) eigenvector matrices of B_xi acting
 * on (rho,u,v,w,p), with unit normal n, frozen density rho and sound speed a. */
void meg6o_eigen(const double n[3], double rho, double a, double L[25], double R[25]) {
  const double nx = n[0], ny = n[1], nz = n[2], ra = rho * a, a2 = a * a;
  const double Lm[5][5] = {{0.0, -nx * ra, -ny * ra, -nz * ra, 1.0},
                           {nx * a2, 0.0, -nz, ny, -nx},
                           {nz * a2, -ny, nx, 0.0, -nz},
                           {-ny * a2, -nz, 0.0, nx, ny},
                           {0.0, nx * ra, ny * ra, nz * ra, 1.0}};
  const double Rm[5][5] = {{1.0 / (2.0 * a2), nx / a2, nz / a2, -ny / a2, 1.0 / (2.0 * a2)},
                           {-nx / (2.0 * ra), 0.0, -ny, -nz, nx / (2.0 * ra)},
                           {-ny / (2.0 * ra), -nz, nx, 0.0, ny / (2.0 * ra)},
                           {-nz / (2.0 * ra), ny, 0.0, nx, nz / (2.0 * ra)},
                           {0.5, 0.0, 0.0, 0.0, 0.5}};
  for (int r = 0; r < 5; ++r)
    for (int c = 0; c < 5; ++c) { L[5 * r + c] = Lm[r][c]; R[5 * r + c] = Rm[r][c]; }
}

/* App. E, de-garbled (R7): hats = cell values, min -> minmod, beta == alpha. */
double meg6o_mp_limit(double w, double c0, double cm, double cp, double dm_near, double dm_far,
                      double alpha, int* limited) {
  const double wmp = c0 + minmod(cp - c0, alpha * (c0 - cm));                 /* E.2 */
  if ((w - c0) * (w - wmp) <= 1e-20) { if (limited) *limited = 0; return w; } /* E.1 */
  if (limited) *limited = 1;
  const double wmd = 0.5 * (c0 + cp) - 0.5 * dm_near;
  const double wul = c0 + alpha * (c0 - cm);
  const double wlc = 0.5 * (3.0 * c0 - cm) + 4.0 / 3.0 * dm_far;
  const double wmin = std::max(std::min(std::min(c0, cp), wmd), std::min(std::min(c0, wul), wlc));
  const double wmax = std::min(std::max(std::max(c0, cp), wmd), std::max(std::max(c0, wul), wlc));
  return w + minmod(wmin - w, wmax - w);                                      /* E.4 */
}

/* Eq. 26-27 with the flux vector of Eq. 2; energy row of Eq. 27 from the
 * Rankine-Hugoniot jump (R9); branch cascade (R10). */
int meg6o_hllc(const double PL[5], const double PR[5], const double m[4], double gamma, double F[5]) {
  const double mx = m[0], my = m[1], mz = m[2], mt = m[3];
  const double g2 = mx * mx + my * my + mz * mz, g = std::sqrt(g2);
  const double* PK[2] = {PL, PR};
  double Uh[2], c[2], E[2], Q[2][5], FK[2][5];
  for (int K = 0; K < 2; ++K) {
    const double r = PK[K][0], u = PK[K][1], v = PK[K][2], w = PK[K][3], pp = PK[K][4];
    Uh[K] = mt + mx * u + my * v + mz * w;                        /* Eq. 4 */
    c[K] = std::sqrt(gamma * pp / r);
    E[K] = pp / (gamma - 1.0) + 0.5 * r * (u * u + v * v + w * w); /* Eq. 5 */
    Q[K][0] = r; Q[K][1] = r * u; Q[K][2] = r * v; Q[K][3] = r * w; Q[K][4] = E[K];
    FK[K][0] = r * Uh[K];
    FK[K][1] = r * u * Uh[K] + mx * pp;
    FK[K][2] = r * v * Uh[K] + my * pp;
    FK[K][3] = r * w * Uh[K] + mz * pp;
    FK[K][4] = (E[K] + pp) * Uh[K] - mt * pp;
  }
  const double SL = std::min(Uh[0] - c[0] * g, Uh[1] - c[1] * g);
  const double SR = std::max(Uh[0] + c[0] * g, Uh[1] + c[1] * g);
  const double SS = (PR[0] * Uh[1] * (SR - Uh[1]) - PL[0] * Uh[0] * (SL - Uh[0]) + (PL[4] - PR[4]) * g2) /
                    (PR[0] * (SR - Uh[1]) - PL[0] * (SL - Uh[0]));
  int branch, K;
  if (SL >= 0.0) { branch = 0; K = 0; }
  else if (SS >= 0.0) { branch = 1; K = 0; }
  else if (SR >= 0.0) { branch = 2; K = 1; }
  else { branch = 3; K = 1; }
  if (branch == 0 || branch == 3) { for (int q = 0; q < 5; ++q) F[q] = FK[K][q]; return branch; }
  const double SK = (K == 0) ? SL : SR;
  const double r = PK[K][0], u = PK[K][1], v = PK[K][2], w = PK[K][3], pp = PK[K][4];
  const double fac = r * (SK - Uh[K]) / (SK - SS);
  double Qs[5];
  Qs[0] = fac;
  Qs[1] = fac * (u + mx * (SS - Uh[K]) / g2);
  Qs[2] = fac * (v + my * (SS - Uh[K]) / g2);
  Qs[3] = fac * (w + mz * (SS - Uh[K]) / g2);
  Qs[4] = fac * (E[K] / r + (SS - Uh[K]) * ((SS - mt) / g2 + pp / (r * (SK - Uh[K]))));
  for (int q = 0; q < 5; ++q) F[q] = FK[K][q] + SK * (Qs[q] - Q[K][q]);
  return branch;
}

namespace {
struct FaceStats { unsigned long long limited = 0, tested = 0; unsigned mask = 0; };

/* O3 steps 1-8 for one interface */
void inviscid_face_impl(const double Pc[4][5], const double P1[2][5], const double P2[4][5],
                        const double m[4], double gamma, double alpha, double F[5], FaceStats* st) {
  /* step 1: unit normal from the interface metrics (A.5) */
  const double g = std::sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
  const double n[3] = {m[0] / g, m[1] / g, m[2] / g};
  /* step 2: averaged state (R5); Pc[1] = cell i, Pc[2] = cell i+1 */
  const double rb = 0.5 * (Pc[1][0] + Pc[2][0]), pb = 0.5 * (Pc[1][4] + Pc[2][4]);
  const double a = std::sqrt(gamma * pb / rb);
  /* step 3 */
  double L[25], R[25];
  meg6o_eigen(n, rb, a, L, R);
  /* step 4: Eq. 20, matrix frozen per interface */
  double W[4][5], D[4][5], W1[2][5];
  for (int c = 0; c < 4; ++c)
    for (int r = 0; r < 5; ++r) {
      double s = 0.0, sd = 0.0;
      for (int q = 0; q < 5; ++q) { s += L[5 * r + q] * Pc[c][q]; sd += L[5 * r + q] * P2[c][q]; }
      W[c][r] = s; D[c][r] = sd;
    }
  for (int c = 0; c < 2; ++c)
    for (int r = 0; r < 5; ++r) {
      double s = 0.0;
      for (int q = 0; q < 5; ++q) s += L[5 * r + q] * P1[c][q];
      W1[c][r] = s;
    }
  double WL[5], WR[5];
  for (int r = 0; r < 5; ++r) {
    /* step 5: Eq. 21-22; cell i = index 1, cell i+1 = index 2 */
    const double wl = W[1][r] + 0.5 * W1[0][r] + D[1][r] / 12.0;
    const double wr = W[2][r] - 0.5 * W1[1][r] + D[2][r] / 12.0;
    /* step 6: MP limiter, left state and its mirror image for the right state (R8) */
    int fl = 0, fr = 0;
    const double dm_mid = minmod(D[1][r], D[2][r]);
    WL[r] = meg6o_mp_limit(wl, W[1][r], W[0][r], W[2][r], dm_mid, minmod(D[0][r], D[1][r]), alpha, &fl);
    WR[r] = meg6o_mp_limit(wr, W[2][r], W[3][r], W[1][r], dm_mid, minmod(D[2][r], D[3][r]), alpha, &fr);
    if (st) { st->tested += 2; st->limited += fl + fr; st->mask |= ((unsigned)fl << r) | ((unsigned)fr << (5 + r)); }
  }
  /* step 7: Eq. 23 */
  double PL[5], PR[5];
  for (int r = 0; r < 5; ++r) {
    double s = 0.0, t = 0.0;
    for (int q = 0; q < 5; ++q) { s += R[5 * r + q] * WL[q]; t += R[5 * r + q] * WR[q]; }
    PL[r] = s; PR[r] = t;
  }
  /* step 8 */
  const int branch = meg6o_hllc(PL, PR, m, gamma, F);
  if (st) {
    st->mask |= (unsigned)branch << 10;
    /* tie flag for the branch record (tests): a wave speed the cascade of Eq. 26 actually tested lies within 1e-10 of
     * zero relative to the fastest wave -- R10: both sides of such a tie give the same flux up to round-off, and which
     * side is taken depends on the rounding order (fluid at rest: S* = +-1e-17) */
    const double mx = m[0], my = m[1], mz = m[2], mt = m[3], gg = std::sqrt(mx * mx + my * my + mz * mz);
    const double UL = mt + mx * PL[1] + my * PL[2] + mz * PL[3], UR = mt + mx * PR[1] + my * PR[2] + mz * PR[3];
    const double cL = std::sqrt(gamma * PL[4] / PL[0]), cR = std::sqrt(gamma * PR[4] / PR[0]);
    const double SL = std::min(UL - cL * gg, UR - cR * gg), SR = std::max(UL + cL * gg, UR + cR * gg);
    const double SS = (PR[0] * UR * (SR - UR) - PL[0] * UL * (SL - UL) + (PL[4] - PR[4]) * gg * gg) /
                      (PR[0] * (SR - UR) - PL[0] * (SL - UL));
    const double tol = 1e-10 * std::max(std::fabs(SL), std::fabs(SR));
    bool tie = std::fabs(SL) <= tol;
    if (SL < 0.0) tie = tie || std::fabs(SS) <= tol;
    if (SL < 0.0 && SS < 0.0) tie = tie || std::fabs(SR) <= tol;
    if (tie) st->mask |= 1u << 12;
  }
}
}  // namespace

void meg6o_inviscid_face(const double Pc[4][5], const double P1[2][5], const double P2[4][5],
                         const double m[4], double gamma, double alpha, double F[5]) {
  inviscid_face_impl(Pc, P1, P2, m, gamma, alpha, F, nullptr);
}

/* Sutherland's law in dimensional-form parameters (R15) */
double meg6o_sutherland(const meg6o_params* p, double T) {
  if (p->s_suth < 0.0) return p->mu_ref;
  const double r = T / p->t_ref;
  return p->mu_ref * r * std::sqrt(r) * (p->t_ref + p->s_suth) / (T + p->s_suth);
}

/* O4: alpha-damping viscous flux at one interface of family d (Fig. 5) */
void meg6o_viscous_face(int d, const double phi[2][4], const double g[2][3][4], const double mh[9],
                        double rj, const meg6o_params* p, double Fv[5]) {
  const double alphaD = 4.0;   /* P:312, beta^D = 0 */
  double val[4], gr[3][4];
  for (int f = 0; f < 4; ++f) {
    const double phiL = phi[0][f] + 0.5 * g[0][d][f];                  /* Eq. 30 */
    const double phiR = phi[1][f] - 0.5 * g[1][d][f];                  /* Eq. 31 */
    for (int e = 0; e < 3; ++e) gr[e][f] = 0.5 * (g[0][e][f] + g[1][e][f]);   /* consistent term; tangential (R11) */
    gr[d][f] += alphaD / 2.0 * (phiR - phiL);                          /* Eq. 29 damping term */
    val[f] = 0.5 * (phiL + phiR);
  }
  const double mu = meg6o_sutherland(p, val[3]);
  const double lam = -2.0 / 3.0 * mu;                                  /* Stokes */
  const double kap = mu * p->gamma * p->r_gas / ((p->gamma - 1.0) * p->prandtl);
  /* un-hatted interface metrics (R12) and chain rule Eq. 32 */
  double k[9];
  for (int q = 0; q < 9; ++q) k[q] = mh[q] / rj;
  double dx[3][4];   /* dx[c][f] = d(field f)/d(x_c) */
  for (int c = 0; c < 3; ++c)
    for (int f = 0; f < 4; ++f) dx[c][f] = k[0 + c] * gr[0][f] + k[3 + c] * gr[1][f] + k[6 + c] * gr[2][f];
  const double ux = dx[0][0], uy = dx[1][0], uz = dx[2][0];
  const double vx = dx[0][1], vy = dx[1][1], vz = dx[2][1];
  const double wx = dx[0][2], wy = dx[1][2], wz = dx[2][2];
  const double Tx = dx[0][3], Ty = dx[1][3], Tz = dx[2][3];
  const double div = ux + vy + wz;
  const double txx = 2.0 * mu * ux + lam * div, tyy = 2.0 * mu * vy + lam * div, tzz = 2.0 * mu * wz + lam * div; /* Eq. 6, 33 */
  const double txy = mu * (uy + vx), txz = mu * (uz + wx), tyz = mu * (vz + wy);
  const double u = val[0], v = val[1], w = val[2];
  const double bx = u * txx + v * txy + w * txz + kap * Tx;            /* Eq. 7 */
  const double by = u * txy + v * tyy + w * tyz + kap * Ty;
  const double bz = u * txz + v * tyz + w * tzz + kap * Tz;
  const double mx = mh[3 * d], my = mh[3 * d + 1], mz = mh[3 * d + 2]; /* hatted normal metrics */
  Fv[0] = 0.0;                                                         /* Eq. 3, 34 */
  Fv[1] = mx * txx + my * txy + mz * txz;
  Fv[2] = mx * txy + my * tyy + mz * tyz;
  Fv[3] = mx * txz + my * tyz + mz * tzz;
  Fv[4] = mx * bx + my * by + mz * bz;
}

/* ----------------------------------- O2 primitives + ghosts -------------------------------- */
namespace {

void prim_interior(meg6o_grid* G, const double* U) {
  const meg6o_params& p = G->p;
  const int ni = G->n[0], nj = G->n[1], nk = G->n[2];
  const size_t N = (size_t)ni * nj * nk;
  for (int f = 0; f < 6; ++f) G->P[f].init(G->n, GP);
  /* Eq. 5 inverted */
  OMP_FOR
  for (int k = 0; k < nk; ++k)
    for (int j = 0; j < nj; ++j)
      for (int i = 0; i < ni; ++i) {
        const size_t c = ((size_t)k * nj + j) * ni + i;
        const double r = U[c], u = U[N + c] / r, v = U[2 * N + c] / r, w = U[3 * N + c] / r;
        const double pp = (p.gamma - 1.0) * (U[4 * N + c] - 0.5 * r * (u * u + v * v + w * w));
        G->P[0](i, j, k) = r; G->P[1](i, j, k) = u; G->P[2](i, j, k) = v; G->P[3](i, j, k) = w; G->P[4](i, j, k) = pp;
      }
}

/* ghost fill of direction d, after the lower directions: xi over interior (j,k); eta over all filled i; zeta over
 * all (i,j).  With several blocks, direction d is filled in every block before direction d+1 in any. */
void ghost_dir(meg6o_grid* G, int d, bool edges = false) {
  const meg6o_params& p = G->p;
  int lo[3] = {0, 0, 0}, hi[3] = {G->n[0], G->n[1], G->n[2]};
  for (int e = 0; e < d; ++e) { lo[e] = -GP; hi[e] = G->n[e] + GP; }
  /* edges (R28): the second round of a multi-block fill -- the faces linked to a neighbour block only, over the ghost
   * ranges of BOTH transverse directions: an edge ghost cell beyond an interface is the neighbour's own ghost cell
   * there (its boundary rule with ITS face data), also where the other direction is filled after this one */
  if (edges) {
    if (p.periodic[d]) return;
    for (int e = d + 1; e < 3; ++e) { lo[e] = -GP; hi[e] = G->n[e] + GP; }
  }
  {
    const int n = G->n[d];
    int a = (d + 1) % 3, b = (d + 2) % 3;
    if (a > b) std::swap(a, b);   /* a < b: the transverse directions in storage order */
    for (int tb = lo[b]; tb < hi[b]; ++tb)
      for (int ta = lo[a]; ta < hi[a]; ++ta) {
        int ix[3];
        ix[a] = ta; ix[b] = tb;
        auto at = [&](int f, int s) -> double& { ix[d] = s; return G->P[f](ix[0], ix[1], ix[2]); };
        if (p.periodic[d]) {
          for (int q = 1; q <= GP; ++q)
            for (int f = 0; f < 5; ++f) { at(f, -q) = at(f, n - q); at(f, n - 1 + q) = at(f, q - 1); }
          continue;
        }
        for (int side = 0; side < 2; ++side) {
          const int face = 2 * d + side, bc = p.bc[face];
          const int last = side ? n - 1 : 0, sg = side ? 1 : -1;
          if (edges && !(bc == 5 && G->link[face])) continue;
          /* transverse position clamped to the interior for the lookup of face data, and to the range on which the
           * cell-centre metrics exist (five ghost layers) for the metric lookups of the wall and outflow rules: in the
           * ghost columns beyond a block interface those are the neighbour's true metrics (R27, R28) */
          /* (face data in the ghost columns of a PERIODIC transverse direction: the periodic image's, Table 1 periodic
           * column -- a ghost cell is its image cell, boundary data included) */
          const int ca = p.periodic[a] ? (ta % G->n[a] + G->n[a]) % G->n[a] : std::min(std::max(ta, 0), G->n[a] - 1);
          const int cb = p.periodic[b] ? (tb % G->n[b] + G->n[b]) % G->n[b] : std::min(std::max(tb, 0), G->n[b] - 1);
          const int ma = std::min(std::max(ta, -5), G->n[a] + 4), mb = std::min(std::max(tb, -5), G->n[b] + 4);
          if (bc == 5) {
            /* block interface, Table 1 last column, R28: ghost layer q = the q-th interior cell of the
             * neighbour block counted from its opposite face, same transverse index (aligned blocks) */
            const meg6o_grid* nb = G->link[face];
            if (nb) {
              for (int q = 1; q <= GP; ++q) {
                int h[3], m[3];
                h[a] = ta; h[b] = tb; h[d] = last + sg * q;
                for (int e = 0; e < 3; ++e)
                  m[G->lax[face][e]] = G->lsg[face][e] > 0 ? h[e] + G->lsh[face][e] : G->lsh[face][e] - h[e];
                for (int f = 0; f < 5; ++f) at(f, last + sg * q) = nb->P[f](m[0], m[1], m[2]);
              }
            } else {
              /* packed layers of a neighbour that lives elsewhere (meg6o_stage_pack on its side): layer l = 0..5 in
               * the neighbour's own order along d, [field][tb][ta][l] over the padded transverse ranges */
              const double* buf = G->ibuf[face];
              const size_t ea = G->n[a] + 2 * GP, eb = G->n[b] + 2 * GP;
              for (int q = 1; q <= GP; ++q) {
                const int l = side ? q - 1 : GP - q;
                for (int f = 0; f < 5; ++f)
                  at(f, last + sg * q) = buf[((f * eb + (size_t)(tb + GP)) * ea + (size_t)(ta + GP)) * GP + l];
              }
            }
          } else if (bc == 1) {
            /* fixed inflow, Table 1, R20: ghost = 2 P_in - P_mirror */
            const size_t n1 = G->n[a], nf = (size_t)G->n[a] * G->n[b];
            const double* pin = G->inflow[face].data();
            for (int q = 1; q <= GP; ++q)
              for (int f = 0; f < 5; ++f)
                at(f, last + sg * q) = 2.0 * pin[f * nf + (size_t)cb * n1 + ca] - at(f, last - sg * (q - 1));
          } else if (bc == 3 || bc == 4) {
            /* walls, Table 1, R27: ghost layer q takes rho and p of its mirror cell m (the q-th interior
             * cell counted from the face).  Inviscid wall (bc 3): u_ghost = u_m - (2 V ktilde_x)_m and likewise v, w,
             * V = u ktilde_x + v ktilde_y + w ktilde_z, ktilde = the unit vector along the hatted metrics of this
             * direction at cell m (static meshes only: no time metric in V).  Adiabatic wall (bc 4): velocity negated. */
            for (int q = 1; q <= GP; ++q) {
              const int m = last - sg * (q - 1);
              double pv[5];
              for (int f = 0; f < 5; ++f) pv[f] = at(f, m);
              if (bc == 3) {
                int im[3]; im[a] = ma; im[b] = mb; im[d] = m;
                const double mx = G->met[3 * d](im[0], im[1], im[2]), my = G->met[3 * d + 1](im[0], im[1], im[2]),
                             mz = G->met[3 * d + 2](im[0], im[1], im[2]);
                const double gm = std::sqrt(mx * mx + my * my + mz * mz);
                const double kx = mx / gm, ky = my / gm, kz = mz / gm;
                const double V = pv[1] * kx + pv[2] * ky + pv[3] * kz;
                pv[1] = pv[1] - 2.0 * V * kx; pv[2] = pv[2] - 2.0 * V * ky; pv[3] = pv[3] - 2.0 * V * kz;
              } else {
                pv[1] = -pv[1]; pv[2] = -pv[2]; pv[3] = -pv[3];
              }
              for (int f = 0; f < 5; ++f) at(f, last + sg * q) = pv[f];
            }
          } else {
            /* outflow, Table 1, R20: copy of the last interior cell; p = p_out where the outward
             * normal Mach number of that cell is below one */
            double pv[5];
            for (int f = 0; f < 5; ++f) pv[f] = at(f, last);
            int im[3]; im[a] = ma; im[b] = mb; im[d] = last;
            const double mx = G->met[3 * d](im[0], im[1], im[2]), my = G->met[3 * d + 1](im[0], im[1], im[2]),
                         mz = G->met[3 * d + 2](im[0], im[1], im[2]);
            const double gm = std::sqrt(mx * mx + my * my + mz * mz);
            const double cs = std::sqrt(p.gamma * pv[4] / pv[0]);
            const double mn = sg * (mx * pv[1] + my * pv[2] + mz * pv[3]) / (gm * cs);
            if (mn < 1.0) pv[4] = p.p_out;
            for (int q = 1; q <= GP; ++q)
              for (int f = 0; f < 5; ++f) at(f, last + sg * q) = pv[f];
          }
        }
      }
  }
}

void finish_primitives(meg6o_grid* G) {
  const meg6o_params& p = G->p;
  for (int f = 0; f < 5; ++f) G->P[f].valid_all();
  /* T = p / (rho R) everywhere, ghosts included (R18) */
  G->P[5].valid_all();
  for (size_t q = 0; q < G->P[5].d.size(); ++q) G->P[5].d[q] = G->P[4].d[q] / (G->P[0].d[q] * p.r_gas);
}

void fill_primitives(meg6o_grid* G, const double* U) {   /* single block */
  prim_interior(G, U);
  for (int d = 0; d < 3; ++d) ghost_dir(G, d);
  finish_primitives(G);
}

void rhs_from_primitives(meg6o_grid* G, const double* U, double* dUdt);

}  // namespace

/* --------------------------------------- O2-O5 RHS ---------------------------------------- */
void meg6o_rhs_blocks(int nb, meg6o_grid* const* G, const double* const* U, double* const* dUdt) {
  for (int b = 0; b < nb; ++b) {
    if (!G[b]->have_metrics) { fprintf(stderr, "meg6o_rhs before metrics_compute\n"); abort(); }
    for (int f = 0; f < 6; ++f)
      if (!G[b]->p.periodic[f / 2] && G[b]->p.bc[f] == 5 && !G[b]->link[f] && !G[b]->ibuf[f]) { fprintf(stderr, "meg6o_rhs: unlinked block interface\n"); abort(); }
    prim_interior(G[b], U[b]);
  }
  /* rotated links (R29): the neighbour cell behind an edge or corner ghost may itself be a ghost of a direction the
   * neighbour fills later; repeating the fill makes every ghost cell the fixed point of the exchange */
  bool rot = false;
  for (int b = 0; b < nb; ++b) rot = rot || G[b]->rotated;
  for (int pass = 0; pass < (rot ? 3 : 1); ++pass)
    for (int d = 0; d < 3; ++d)
      for (int b = 0; b < nb; ++b) ghost_dir(G[b], d);
  bool linked = false;
  for (int b = 0; b < nb; ++b)
    for (int f = 0; f < 6; ++f) linked = linked || (!G[b]->p.periodic[f / 2] && G[b]->p.bc[f] == 5 && G[b]->link[f]);
  if (linked)
    for (int d = 0; d < 3; ++d)
      for (int b = 0; b < nb; ++b) ghost_dir(G[b], d, true);
  for (int b = 0; b < nb; ++b) finish_primitives(G[b]);
  for (int b = 0; b < nb; ++b) rhs_from_primitives(G[b], U[b], dUdt[b]);
}

void meg6o_rhs(meg6o_grid* G, const double* U, double* dUdt) { meg6o_rhs_blocks(1, &G, &U, &dUdt); }

namespace {
void rhs_from_primitives(meg6o_grid* G, const double* U, double* dUdt) {
  const meg6o_params& p = G->p;
  const int ni = G->n[0], nj = G->n[1], nk = G->n[2];
  const size_t N = (size_t)ni * nj * nk;
  /* O2: first gradients of rho,u,v,w,p (and T if viscous) along the three directions, Eq. 17 */
  const int nf = p.viscous ? 6 : 5;
  for (int d = 0; d < 3; ++d)
    for (int f = 0; f < nf; ++f) grad_dir(G->P[f], d, p.scheme, G->G1[d][f]);

  std::vector<double> res(5 * N, 0.0);
  unsigned long long lim = 0, tst = 0;

  /* O3: inviscid flux differences, directions xi, eta, zeta in this order (R22) */
  for (int d = 0; d < 3; ++d) {
    Arr P2[5];
    for (int f = 0; f < 5; ++f) d2_dir(G->P[f], G->G1[d][f], d, P2[f]);      /* Eq. 19 */
    /* interface fluxes: index s of the flux array = interface between cells s-1 and s along d */
    int fn[3] = {ni, nj, nk};
    fn[d] += 1;
    std::vector<double> flux((size_t)5 * fn[0] * fn[1] * fn[2]);
    const size_t FN = (size_t)fn[0] * fn[1] * fn[2];
    if (G->want_masks) G->mask[d].assign(FN, 0);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) num_threads(g_threads) reduction(+ : lim, tst)
#endif
    for (int k = 0; k < fn[2]; ++k)
      for (int j = 0; j < fn[1]; ++j)
        for (int i = 0; i < fn[0]; ++i) {
          int c0[3] = {i, j, k};
          c0[d] -= 1;   /* cell "i" of the paper (left of the interface) */
          double Pc[4][5], P1[2][5], PP2[4][5], m[4], F[5];
          for (int q = 0; q < 4; ++q) {
            int c[3] = {c0[0], c0[1], c0[2]};
            c[d] += q - 1;
            for (int f = 0; f < 5; ++f) { Pc[q][f] = G->P[f](c[0], c[1], c[2]); PP2[q][f] = P2[f](c[0], c[1], c[2]); }
          }
          for (int q = 0; q < 2; ++q) {
            int c[3] = {c0[0], c0[1], c0[2]};
            c[d] += q;
            for (int f = 0; f < 5; ++f) P1[q][f] = G->G1[d][f](c[0], c[1], c[2]);
          }
          for (int q = 0; q < 3; ++q) m[q] = G->fmet[d][3 * d + q](c0[0], c0[1], c0[2]);
          m[3] = p.moving ? G->fmt[d](c0[0], c0[1], c0[2]) : 0.0;
          FaceStats st;
          inviscid_face_impl(Pc, P1, PP2, m, p.gamma, p.mp_alpha, F, &st);
          lim += st.limited; tst += st.tested;
          const size_t fi = ((size_t)k * fn[1] + j) * fn[0] + i;
          for (int f = 0; f < 5; ++f) flux[f * FN + fi] = F[f];
          if (G->want_masks) G->mask[d][fi] = (unsigned short)st.mask;
        }
    /* Eq. 25, Eq. 8-9: Res_i -= F_{i+1/2} - F_{i-1/2} */
    const size_t fs = (d == 0) ? 1 : (d == 1) ? (size_t)fn[0] : (size_t)fn[0] * fn[1];
    OMP_FOR
    for (int k = 0; k < nk; ++k)
      for (int j = 0; j < nj; ++j)
        for (int i = 0; i < ni; ++i) {
          const size_t c = ((size_t)k * nj + j) * ni + i;
          const size_t fi = ((size_t)k * fn[1] + j) * fn[0] + i;
          for (int f = 0; f < 5; ++f) res[f * N + c] -= flux[f * FN + fi + fs] - flux[f * FN + fi];
        }
  }
  G->n_limited += lim; G->n_tested += tst;

  /* O4: viscous flux differences, Eq. 35 */
  if (p.viscous) {
    for (int d = 0; d < 3; ++d) {
      int fn[3] = {ni, nj, nk};
      fn[d] += 1;
      const size_t FN = (size_t)fn[0] * fn[1] * fn[2];
      std::vector<double> flux((size_t)5 * FN);
      OMP_FOR
      for (int k = 0; k < fn[2]; ++k)
        for (int j = 0; j < fn[1]; ++j)
          for (int i = 0; i < fn[0]; ++i) {
            int c0[3] = {i, j, k};
            c0[d] -= 1;
            double phi[2][4], g[2][3][4], mh[9], Fv[5];
            for (int q = 0; q < 2; ++q) {
              int c[3] = {c0[0], c0[1], c0[2]};
              c[d] += q;
              for (int f = 0; f < 4; ++f) {
                const int pf = (f < 3) ? f + 1 : 5;   /* u,v,w,T */
                phi[q][f] = G->P[pf](c[0], c[1], c[2]);
                for (int e = 0; e < 3; ++e) g[q][e][f] = G->G1[e][pf](c[0], c[1], c[2]);
              }
            }
            for (int q = 0; q < 9; ++q) mh[q] = G->fmet[d][q](c0[0], c0[1], c0[2]);
            const double rj = G->fmet[d][9](c0[0], c0[1], c0[2]);
            meg6o_viscous_face(d, phi, g, mh, rj, &p, Fv);
            const size_t fi = ((size_t)k * fn[1] + j) * fn[0] + i;
            for (int f = 0; f < 5; ++f) flux[f * FN + fi] = Fv[f];
          }
      const size_t fs = (d == 0) ? 1 : (d == 1) ? (size_t)fn[0] : (size_t)fn[0] * fn[1];
      OMP_FOR
      for (int k = 0; k < nk; ++k)
        for (int j = 0; j < nj; ++j)
          for (int i = 0; i < ni; ++i) {
            const size_t c = ((size_t)k * nj + j) * ni + i;
            const size_t fi = ((size_t)k * fn[1] + j) * fn[0] + i;
            for (int f = 0; f < 5; ++f) res[f * N + c] += flux[f * FN + fi + fs] - flux[f * FN + fi];
          }
    }
  }
  /* O5 assembly: dQ/dt = J (Res - (1/J)_t Q) - sigma (Q - Q_ref)   (Eq. 9, 12, 14; sponge R16) */
  const bool sponge = !G->sigma.empty();
  OMP_FOR
  for (int k = 0; k < nk; ++k)
    for (int j = 0; j < nj; ++j)
      for (int i = 0; i < ni; ++i) {
        const size_t c = ((size_t)k * nj + j) * ni + i;
        const double J = 1.0 / G->rj(i, j, k);
        const double rjt = p.moving ? G->rjt(i, j, k) : 0.0;
        for (int f = 0; f < 5; ++f) {
          double v = J * (res[f * N + c] - rjt * U[f * N + c]);
          if (sponge) v -= G->sigma[c] * (U[f * N + c] - G->uref[f * N + c]);
          dUdt[f * N + c] = v;
        }
      }
}
}  // namespace

/* O6: SSP/TVD-RK3, Eq. B.1; stage times t, t+dt, t+dt/2; moving meshes recompute the
 * geometry at each stage time (R17). */
void meg6o_rk3_step_blocks(int nb, meg6o_grid* const* G, double* const* U, double t, double dt) {
  std::vector<std::vector<double>> U0(nb), L(nb);
  std::vector<double*> Lp(nb);
  std::vector<const double*> Uc(nb);
  for (int b = 0; b < nb; ++b) {
    const size_t M = (size_t)5 * G[b]->n[0] * G[b]->n[1] * G[b]->n[2];
    U0[b].assign(U[b], U[b] + M); L[b].resize(M); Lp[b] = L[b].data(); Uc[b] = U[b];
  }
  const double ts[3] = {t, t + dt, t + 0.5 * dt};
  for (int s = 0; s < 3; ++s) {
    if (G[0]->p.moving) meg6o_metrics_compute_blocks(nb, G, ts[s]);
    meg6o_rhs_blocks(nb, G, Uc.data(), Lp.data());
    for (int b = 0; b < nb; ++b) {
      double* u = U[b];
      const double* u0 = U0[b].data();
      const double* l = L[b].data();
      const size_t M = U0[b].size();
      if (s == 0) for (size_t q = 0; q < M; ++q) u[q] = u0[q] + dt * l[q];
      else if (s == 1) for (size_t q = 0; q < M; ++q) u[q] = 3.0 / 4.0 * u0[q] + 1.0 / 4.0 * (u[q] + dt * l[q]);
      else for (size_t q = 0; q < M; ++q) u[q] = 1.0 / 3.0 * u0[q] + 2.0 / 3.0 * (u[q] + dt * l[q]);
    }
  }
}

void meg6o_rk3_step(meg6o_grid* G, double* U, double t, double dt) { meg6o_rk3_step_blocks(1, &G, &U, t, dt); }

/* Staged evaluation for blocks that live in different processes (the caller carries the packed layers). */
size_t meg6o_interface_doubles(const meg6o_grid* G, int face) {
  const int d = face / 2;
  int a = (d + 1) % 3, b = (d + 2) % 3;
  return (size_t)5 * GP * (G->n[a] + 2 * GP) * (G->n[b] + 2 * GP);
}
void meg6o_set_interface_buffer(meg6o_grid* G, int face, const double* layers) {
  G->ibuf[face] = layers;
  if (layers) G->link[face] = nullptr;
}
void meg6o_stage_prim(meg6o_grid* G, const double* U) { prim_interior(G, U); }
void meg6o_stage_ghosts(meg6o_grid* G, int d) { ghost_dir(G, d); }
void meg6o_stage_pack(meg6o_grid* G, int face, double* layers) {
  const int d = face / 2, side = face & 1;
  int a = (d + 1) % 3, b = (d + 2) % 3;
  if (a > b) std::swap(a, b);
  const size_t ea = G->n[a] + 2 * GP, eb = G->n[b] + 2 * GP;
  const int first = side ? G->n[d] - GP : 0;
  for (int f = 0; f < 5; ++f)
    for (int tb = -GP; tb < G->n[b] + GP; ++tb)
      for (int ta = -GP; ta < G->n[a] + GP; ++ta)
        for (int l = 0; l < GP; ++l) {
          int is[3]; is[a] = ta; is[b] = tb; is[d] = first + l;
          layers[((f * eb + (size_t)(tb + GP)) * ea + (size_t)(ta + GP)) * GP + l] = G->P[f].d[G->P[f].idx(is[0], is[1], is[2])];
        }
}
void meg6o_stage_rhs(meg6o_grid* G, const double* U, double* dUdt) {
  finish_primitives(G);
  rhs_from_primitives(G, U, dUdt);
}

/* Block interface (Sec. 6; Table 1 last column): face `face` of `home` (bc 5) takes its ghost cells -- the
 * primitives, and the cell-centre coordinates the metrics are built from -- out of the block `nb`, whose face `nb_face`
 * is the same surface.  "Each block possesses its own coordinate system": the two transverse axes of the home
 * face, in storage order (a < b), run along the neighbour's transverse axes (a' < b') as a -> a', b -> b' (swap = 0) or
 * a -> b', b -> a' (swap = 1), each forwards (flip = 0) or backwards (flip = 1); the cell counts must agree ("the
 * dimensions of the block interface plane should be identical").  off[3] is added to the neighbour's coordinates
 * seen from home (zero; the period vector across a wrap-around link).  Returns 0 on success.  R28, R29. */
int meg6o_link_blocks_oriented(meg6o_grid* home, int face, meg6o_grid* nb, int nb_face, int swap, int flip_a, int flip_b,
                               const double* off) {
  if (!home || !nb || face < 0 || face > 5 || nb_face < 0 || nb_face > 5) return 1;
  const int d = face / 2, dn = nb_face / 2;
  if (home->p.periodic[d] || home->p.bc[face] != 5) return 1;
  if (nb->p.periodic[dn] || nb->n[dn] < GP) return 1;
  int a = (d + 1) % 3, b = (d + 2) % 3, an = (dn + 1) % 3, bn = (dn + 2) % 3;
  if (a > b) std::swap(a, b);
  if (an > bn) std::swap(an, bn);
  const int ta = swap ? bn : an, tb = swap ? an : bn;     /* images of the home axes a, b */
  if (nb->n[ta] != home->n[a] || nb->n[tb] != home->n[b]) return 1;
  int* ax = home->lax[face]; int* sg = home->lsg[face]; int* sh = home->lsh[face];
  ax[a] = ta; sg[a] = flip_a ? -1 : 1; sh[a] = flip_a ? home->n[a] - 1 : 0;
  ax[b] = tb; sg[b] = flip_b ? -1 : 1; sh[b] = flip_b ? home->n[b] - 1 : 0;
  /* along the normal: ghost layer q of home = the q-th interior cell of the neighbour counted from nb_face */
  const int n = home->n[d], nn = nb->n[dn], hs = face & 1, ns = nb_face & 1;
  ax[d] = dn;
  if (hs && !ns) { sg[d] = 1; sh[d] = -n; }
  else if (hs && ns) { sg[d] = -1; sh[d] = nn - 1 + n; }
  else if (!hs && ns) { sg[d] = 1; sh[d] = nn; }
  else { sg[d] = -1; sh[d] = -1; }
  for (int c = 0; c < 3; ++c) home->loff[face][c] = off ? off[c] : 0.0;
  home->link[face] = nb;
  home->ibuf[face] = nullptr; home->gbuf[face] = nullptr;
  const bool aligned = ax[0] == 0 && ax[1] == 1 && ax[2] == 2 && sg[0] > 0 && sg[1] > 0 && sg[2] > 0;
  if (!aligned) { home->rotated = true; nb->rotated = true; }
  if (nn < GX) home->thin_nb = true;
  return 0;
}

/* aligned blocks: same orientation of the three computational axes, nb's opposite face */
int meg6o_link_blocks(meg6o_grid* home, int face, meg6o_grid* nb) {
  if (!home || !nb || face < 0 || face > 5) return 1;
  const int d = face / 2;
  for (int e = 0; e < 3; ++e)
    if (e != d && nb->p.periodic[e] != home->p.periodic[e]) return 1;
  return meg6o_link_blocks_oriented(home, face, nb, face ^ 1, 0, 0, 0, nullptr);
}

/* Eq. B.2 / B.3: un-hatted metrics = hatted * J; viscous alpha read as alpha^D = 4 (R25) */
double meg6o_cfl_dt(meg6o_grid* G, const double* U, double cfl) {
  const meg6o_params& p = G->p;
  const int ni = G->n[0], nj = G->n[1], nk = G->n[2];
  const size_t N = (size_t)ni * nj * nk;
  double inv_min = std::numeric_limits<double>::infinity(), vis_min = std::numeric_limits<double>::infinity();
  for (int k = 0; k < nk; ++k)
    for (int j = 0; j < nj; ++j)
      for (int i = 0; i < ni; ++i) {
        const size_t c = ((size_t)k * nj + j) * ni + i;
        const double r = U[c], u = U[N + c] / r, v = U[2 * N + c] / r, w = U[3 * N + c] / r;
        const double pp = (p.gamma - 1.0) * (U[4 * N + c] - 0.5 * r * (u * u + v * v + w * w));
        const double cs = std::sqrt(p.gamma * pp / r), J = 1.0 / G->rj(i, j, k);
        const double mu = p.viscous ? meg6o_sutherland(&p, pp / (r * p.r_gas)) : 0.0;
        for (int d = 0; d < 3; ++d) {
          const double mx = J * G->met[3 * d](i, j, k), my = J * G->met[3 * d + 1](i, j, k), mz = J * G->met[3 * d + 2](i, j, k);
          const double mtt = p.moving ? J * G->mt[d](i, j, k) : 0.0;
          const double gn = std::sqrt(mx * mx + my * my + mz * mz);
          inv_min = std::min(inv_min, 1.0 / (std::fabs(mtt + mx * u + my * v + mz * w) + cs * gn));
          if (p.viscous) vis_min = std::min(vis_min, 1.0 / (mu * gn * gn));
        }
      }
  double dt = inv_min;
  if (p.viscous) dt = std::min(dt, vis_min / 4.0);
  return cfl * dt;
}

/* Volume-averaged kinetic energy and enstrophy, the integrals of Eq. 54 written for three dimensions and
 * curvilinear cells (dV = 1/J), the vorticity from the SHARED first gradients of the primitives through the
 * chain rule with the cell-centre metrics (Eq. 32 form):  out = { E_k, enstrophy, volume }. */
void meg6o_diagnostics(meg6o_grid* G, const double* U, double* out) {
  const meg6o_params& p = G->p;
  const int ni = G->n[0], nj = G->n[1], nk = G->n[2];
  fill_primitives(G, U);
  Arr g[3][3];   /* g[d][c] = gradient along direction d of velocity component c */
  for (int d = 0; d < 3; ++d)
    for (int c = 0; c < 3; ++c) grad_dir(G->P[1 + c], d, p.scheme, g[d][c]);
  double ke = 0.0, en = 0.0, vol = 0.0;
  for (int k = 0; k < nk; ++k)
    for (int j = 0; j < nj; ++j)
      for (int i = 0; i < ni; ++i) {
        const double rj = G->rj(i, j, k), J = 1.0 / rj;
        double dv[3][3];   /* dv[c][x] = d(velocity c)/d(coordinate x) */
        for (int c = 0; c < 3; ++c)
          for (int x = 0; x < 3; ++x)
            dv[c][x] = J * (G->met[x](i, j, k) * g[0][c](i, j, k) + G->met[3 + x](i, j, k) * g[1][c](i, j, k) +
                            G->met[6 + x](i, j, k) * g[2][c](i, j, k));
        const double ox = dv[2][1] - dv[1][2], oy = dv[0][2] - dv[2][0], oz = dv[1][0] - dv[0][1];
        const double r = G->P[0](i, j, k), u = G->P[1](i, j, k), v = G->P[2](i, j, k), w = G->P[3](i, j, k);
        ke += r * 0.5 * (u * u + v * v + w * w) * rj;
        en += r * 0.5 * (ox * ox + oy * oy + oz * oz) * rj;
        vol += rj;
      }
  out[0] = ke / vol; out[1] = en / vol; out[2] = vol;
}

void meg6o_limiter_stats(meg6o_grid* G, unsigned long long* n_limited, unsigned long long* n_tested) {
  *n_limited = G->n_limited; *n_tested = G->n_tested;
}

void meg6o_branch_masks_enable(meg6o_grid* G, int on) {
  G->want_masks = on != 0;
  if (!on) for (int d = 0; d < 3; ++d) std::vector<unsigned short>().swap(G->mask[d]);
}
size_t meg6o_get_branch_mask(meg6o_grid* G, int d, unsigned short* out) {
  if (d < 0 || d > 2) return 0;
  if (out) std::copy(G->mask[d].begin(), G->mask[d].end(), out);
  return G->mask[d].size();
}

/* -------------------------------------- inspection ---------------------------------------- */
void meg6o_get_cell(meg6o_grid* G, int which, double* out) {
  if (which < 9) interior_copy(G->met[which], out);
  else if (which == 9) interior_copy(G->rj, out);
  else if (which < 13) interior_copy(G->mt[which - 10], out);
  else if (which == 13) interior_copy(G->rjt, out);
  else interior_copy(G->xc[which - 14], out);
}

void meg6o_get_face(meg6o_grid* G, int d, int q, double* out) {
  const Arr& a = (q < 10) ? G->fmet[d][q] : G->fmt[d];
  int lo[3] = {0, 0, 0};
  lo[d] = -1;
  size_t m = 0;
  for (int k = lo[2]; k < G->n[2]; ++k)
    for (int j = lo[1]; j < G->n[1]; ++j)
      for (int i = lo[0]; i < G->n[0]; ++i) out[m++] = a(i, j, k);
}

void meg6o_get_prim(meg6o_grid* G, int field, double* out) { interior_copy(G->P[field], out); }
void meg6o_get_grad(meg6o_grid* G, int d, int field, double* out) { interior_copy(G->G1[d][field], out); }

void meg6o_line_op(int op, int n, const double* f, double* out) {
  const int nn[3] = {n, 1, 1};
  Arr a(nn, 0), r;
  for (int i = 0; i < n; ++i) a(i, 0, 0) = f[i];
  Arr f1, f2;
  switch (op) {
    case 0: grad_dir(a, 0, 0, r); break;
    case 1: grad_dir(a, 0, 0, f1); d2_dir(a, f1, 0, r); break;
    case 2: case 3: {
      grad_dir(a, 0, 0, f1); d2_dir(a, f1, 0, f2);
      r.init(nn, 0); r.lo[0] = f2.lo[0]; r.hi[0] = f2.hi[0];
      for (int i = r.lo[0]; i < r.hi[0]; ++i)
        r(i, 0, 0) = (op == 2) ? op_Lft(a(i, 0, 0), f1(i, 0, 0), f2(i, 0, 0)) : op_Rgt(a(i, 0, 0), f1(i, 0, 0), f2(i, 0, 0));
      break;
    }
    case 4: H_dir(a, 0, 0, false, r); break;
    case 5: delta_dir(a, 0, 0, r); break;
    case 6: {
      /* Eq. 29-31 with alpha^D = 4, beta^D = 0, at i+1/2 */
      grad_dir(a, 0, 0, f1);
      r.init(nn, 0); r.lo[0] = f1.lo[0]; r.hi[0] = f1.hi[0] - 1;
      for (int i = r.lo[0]; i < r.hi[0]; ++i) {
        const double uL = a(i, 0, 0) + 0.5 * f1(i, 0, 0), uR = a(i + 1, 0, 0) - 0.5 * f1(i + 1, 0, 0);
        r(i, 0, 0) = 0.5 * (f1(i, 0, 0) + f1(i + 1, 0, 0)) + 4.0 / 2.0 * (uR - uL);
      }
      break;
    }
    case 7: grad_c4(a, 0, r); break;
    case 8: grad_dir(a, 0, 1, r); break;                       /* IG4 */
    case 9: delta_dir(a, 0, 1, r); break;                      /* consistent derivative with IG4 gradients */
    case 10: H_dir(a, 0, 1, false, r); break;
    default: r.init(nn, 0); r.lo[0] = r.hi[0] = 0;
  }
  for (int i = 0; i < n; ++i)
    out[i] = (i >= r.lo[0] && i < r.hi[0]) ? r(i, 0, 0) : std::numeric_limits<double>::quiet_NaN();
}

}  // extern "C"
