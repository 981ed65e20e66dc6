// meg6_geom.cu -- metric / Jacobian kernels and their launcher.  Compiled with -fmad=false (see meg6_geom.cuh).
#include <cstdlib>
#include <cstring>
#include <math.h>
#include "meg6_geom.cuh"
#include "meg6_ig4.cuh"

namespace meg6 {

static inline unsigned nblk(long long n, int t) { return (unsigned)((n + t - 1) / t); }

static GeomIn geom_in(meg6_grid* g, double t) {
  GeomIn gi;
  for (int q = 0; q < 3; ++q) { gi.node[q] = g->nodes[q]; gi.mode[q] = g->modes[q]; }
  const double ph = 2.0 * M_PI * g->p.omega * t;
  gi.s = g->p.moving ? sin(ph) : 0.0;
  gi.sd = g->p.moving ? 2.0 * M_PI * g->p.omega * cos(ph) : 0.0;
  gi.tp = g->tp_cur;   // set while a graph of meg6_rk3_steps is being captured: the two numbers come from device memory
  return gi;
}

// stage 1 of the geometry: cell centres (and grid velocities) of the interior cells
cudaError_t geom_centres(meg6_grid* g, double t) {
  const Consts& c = g->c;
  P3 xc, xt;
  for (int q = 0; q < 3; ++q) { xc.p[q] = g->xc[q]; xt.p[q] = g->xt[q]; }
  k_centres<<<nblk(c.LC.n, 256), 256, 0, g->stream>>>(c, geom_in(g, t), xc, xt);
  ++g->geom_launches;
  return cudaGetLastError();
}

// stage 2, once per direction (xi, then eta over the xi-extended array, then zeta): ghost layers of direction d.  With
// several blocks, direction d is extended in every block before direction d+1 in any (block-interface faces read the
// neighbour's array, ghosts of the lower directions included)
cudaError_t geom_extend(meg6_grid* g, int d) {
  const Consts& c = g->c;
  P3 xc, xt;
  for (int q = 0; q < 3; ++q) { xc.p[q] = g->xc[q]; xt.p[q] = g->xt[q]; }
  if (c.periodic[0] && c.periodic[1] && c.periodic[2]) {   // all wraps: the three passes as one launch, at d == 0
    if (d != 0) return cudaSuccess;
    const long long e0 = c.n[0] + 2 * GX, e1 = c.n[1] + 2 * GX;
    const long long nthr = e0 * e1 * 2 * GX + e0 * 2 * GX * c.n[2] + 2LL * GX * c.n[1] * c.n[2];
    k_extend_periodic<<<nblk(nthr, 256), 256, 0, g->stream>>>(c, xc, xt);
    ++g->geom_launches;
    return cudaGetLastError();
  }
  ExtIn in;
  memset(&in, 0, sizeof(in));
  for (int side = 0; side < 2; ++side) {
    const int face = 2 * d + side;
    if (c.periodic[d] || c.bc[face] != 5) continue;
    const meg6_grid* nb = g->link[face];
    if (nb) {
      for (int q = 0; q < 3; ++q) { in.nbx[side][q] = nb->xc[q]; in.nbv[side][q] = nb->xt[q]; in.off[side][q] = g->loff[face][q]; }
      in.nbL[side] = nb->c.LX;
      for (int e = 0; e < 3; ++e) { in.nax[side][e] = g->lax[face][e]; in.nsg[side][e] = g->lsg[face][e]; in.nsh[side][e] = g->lsh[face][e]; }
    } else if (g->gbuf[face]) {   // packed layers of a remote neighbour: a block ten cells thick, aligned
      const Lay LQ = geom_pack_lay(c.LX, d);
      for (int q = 0; q < 3; ++q) {
        in.nbx[side][q] = g->gbuf[face] + q * LQ.n;
        in.nbv[side][q] = g->p.moving ? g->gbuf[face] + (3 + q) * LQ.n : nullptr;
        in.off[side][q] = g->goff[face][q];
      }
      in.nbL[side] = LQ;
      for (int e = 0; e < 3; ++e) { in.nax[side][e] = e; in.nsg[side][e] = 1; in.nsh[side][e] = 0; }
      in.nsh[side][d] = side ? -c.n[d] : GX;
    }
  }
  int a = (d + 1) % 3, b = (d + 2) % 3;
  if (a > b) { int t = a; a = b; b = t; }
  const long long ea = c.n[a] + ((a < d) ? 2 * GX : 0), eb = c.n[b] + ((b < d) ? 2 * GX : 0);
  k_extend<<<nblk(ea * eb * 2 * GX, 256), 256, 0, g->stream>>>(c, d, xc, xt, in);
  ++g->geom_launches;
  return cudaGetLastError();
}

cudaError_t geom_pack(meg6_grid* g, int face, double* layers) {
  const int d = face / 2;
  const Lay LQ = geom_pack_lay(g->c.LX, d);
  const int first = (face & 1) ? g->c.n[d] - GX : 0;
  P6c src;
  for (int q = 0; q < 3; ++q) { src.p[q] = g->xc[q]; src.p[3 + q] = g->xt[q]; }
  k_pack_geom<<<nblk(LQ.n, 256), 256, 0, g->stream>>>(g->c.LX, LQ, d, first, g->p.moving ? 6 : 3, src, layers);
  return cudaGetLastError();
}

// ---- MIG4 (scheme 1): the geometry as whole-array passes, each the operation the discretisation names ----
static Box box_all(const Consts& c) {
  Box b;
  for (int a = 0; a < 3; ++a) { b.lo[a] = -GX; b.hi[a] = c.n[a] + GX; }
  return b;
}
static Box box_and(const Box& a, const Box& b) {
  Box r;
  for (int q = 0; q < 3; ++q) { r.lo[q] = a.lo[q] > b.lo[q] ? a.lo[q] : b.lo[q]; r.hi[q] = a.hi[q] < b.hi[q] ? a.hi[q] : b.hi[q]; }
  return r;
}
static long long box_n(const Box& b) { return (long long)(b.hi[0] - b.lo[0]) * (b.hi[1] - b.lo[1]) * (b.hi[2] - b.lo[2]); }

// IG4 gradient of f (valid on fb) along dir into out; returns the valid box of out.  Lay L: layout of both arrays.
Box launch_ig4_batch(meg6_grid* g, const Lay& L, const double* f, const Box& fb, int dir, double* out, int nfields,
                     long long fs_in, long long fs_out) {
  Box ob = fb;
  ob.lo[dir] += 2; ob.hi[dir] -= 2;
  const int a1 = (dir == 0) ? 1 : 0, a2 = (dir == 2) ? 1 : 2;
  const long long lines = (long long)(ob.hi[a1] - ob.lo[a1]) * (ob.hi[a2] - ob.lo[a2]);
  const dim3 grid((unsigned)nblk(lines, 128), (unsigned)nfields);
  if (dir == 0) k_ig4x<<<grid, 128, 0, g->stream>>>(L, f, out, ob, g->ig4_cc, g->ig4_den, fs_in, fs_out);
  else if (dir == 1) k_ig4<1><<<grid, 128, 0, g->stream>>>(L, f, out, ob, g->ig4_cc, g->ig4_den, fs_in, fs_out);
  else k_ig4<2><<<grid, 128, 0, g->stream>>>(L, f, out, ob, g->ig4_cc, g->ig4_den, fs_in, fs_out);
  ++g->geom_launches;
  return ob;
}

Box launch_ig4(meg6_grid* g, const Lay& L, const double* f, const Box& fb, int dir, double* out) {
  return launch_ig4_batch(g, L, f, fb, dir, out, 1, 0, 0);
}

// Flow gradients only (rounding order differs from the plain Thomas loop at segment boundaries): the segmented
// two-pass solve along eta / zeta where the line fits, the plain kernels otherwise and along xi.
Box launch_ig4_flow(meg6_grid* g, const Lay& L, const double* f, const Box& fb, int dir, double* out, int nfields,
                    long long fs_in, long long fs_out) {
  const int m = fb.hi[dir] - fb.lo[dir] - 4;
  if (m - 2 > IG4S_NSEG * IG4S_SEGMAX || m < 3)
    return launch_ig4_batch(g, L, f, fb, dir, out, nfields, fs_in, fs_out);
  Box ob = fb;
  ob.lo[dir] += 2; ob.hi[dir] -= 2;
  if (dir == 0) {
    // lanes of a warp = segments of one xi line, or of several short lines
    const int spl = (m - 2 + IG4S_SEGMAX - 1) / IG4S_SEGMAX;        // segments per line (<= 32)
    const int lpw = 32 / spl;                                        // lines per warp
    if ((long long)lpw * (m + 4) > IG4SX_TILE) return launch_ig4_batch(g, L, f, fb, dir, out, nfields, fs_in, fs_out);
    const long long lines = (long long)(ob.hi[1] - ob.lo[1]) * (ob.hi[2] - ob.lo[2]);
    const dim3 grid((unsigned)nblk(lines, (long long)IG4SX_WARPS * lpw), (unsigned)nfields);
    k_ig4sx<<<grid, 32 * IG4SX_WARPS, 0, g->stream>>>(L, f, out, ob, g->ig4_cc, fs_in, fs_out, spl, lpw);
    return ob;
  }
  const int od = (dir == 1) ? 2 : 1;
  const dim3 grid((unsigned)nblk(ob.hi[0] - ob.lo[0], IG4S_LANES), (unsigned)(ob.hi[od] - ob.lo[od]), (unsigned)nfields);
  const int nseg = (m - 2 + IG4S_SEGMAX - 1) / IG4S_SEGMAX;   // segments of (nearly) full length, fewer threads for short lines
  const int nthr = IG4S_LANES * ((nseg + 1) / 2 * 2);        // whole warps
  if (dir == 1) k_ig4s<1><<<grid, nthr, 0, g->stream>>>(L, f, out, ob, g->ig4_cc, fs_in, fs_out);
  else k_ig4s<2><<<grid, nthr, 0, g->stream>>>(L, f, out, ob, g->ig4_cc, fs_in, fs_out);
  return ob;
}

// H of f along dir into a cell-layout array (index i = interface i+1/2); returns its valid box
static Box H_pass(meg6_grid* g, const double* f, const Box& fb, int dir, double* f1, double* H) {
  const Lay& L = g->c.LX;
  const Box gb = launch_ig4(g, L, f, fb, dir, f1);
  Box hb = gb;
  hb.lo[dir] += 1; hb.hi[dir] -= 2;
  k_H_from<<<nblk(box_n(hb), 256), 256, 0, g->stream>>>(L, L, dir, 0, f, f1, H, hb);
  ++g->geom_launches;
  return hb;
}
// consistent derivative Eq. 37 of f along dir into out
static Box delta_pass(meg6_grid* g, const double* f, const Box& fb, int dir, double* f1, double* H, double* out) {
  const Box hb = H_pass(g, f, fb, dir, f1, H);
  Box db = hb;
  db.lo[dir] += 1;
  k_point<<<nblk(box_n(db), 256), 256, 0, g->stream>>>(g->c.LX, 0, dir, H, nullptr, out, db);
  ++g->geom_launches;
  return db;
}

static cudaError_t launch_geometry_ig4(meg6_grid* g) {
  const Consts& c = g->c;
  const Lay& L = c.LX;
  double* f1 = g->scr[0]; double* H = g->scr[1]; double* t1 = g->scr[2]; double* t2 = g->scr[3];
  double* d1 = g->scr[4]; double* d2 = g->scr[5];
  const Box all = box_all(c);
  Box cdb[9];
  for (int cc = 0; cc < 3; ++cc)
    for (int d = 0; d < 3; ++d) cdb[3 * cc + d] = delta_pass(g, g->xc[cc], all, d, f1, H, g->cd[3 * cc + d]);
  // Thomas-Lombard conservative metrics, Eq. 10: m = delta_b(delta_a(q) s) - delta_a(delta_b(q) s)
  Box mb[9];
  for (int r = 0; r < 3; ++r) {
    const int a = (r + 1) % 3, b = (r + 2) % 3;
    for (int cc = 0; cc < 3; ++cc) {
      const int q = (cc + 1) % 3, s = (cc + 2) % 3;
      const Box b1 = box_and(cdb[3 * q + a], all), b2 = box_and(cdb[3 * q + b], all);
      k_point<<<nblk(box_n(b1), 256), 256, 0, g->stream>>>(L, 1, 0, g->cd[3 * q + a], g->xc[s], t1, b1);
      k_point<<<nblk(box_n(b2), 256), 256, 0, g->stream>>>(L, 1, 0, g->cd[3 * q + b], g->xc[s], t2, b2);
      const Box e1 = delta_pass(g, t1, b1, b, f1, H, d1);
      const Box e2 = delta_pass(g, t2, b2, a, f1, H, d2);
      mb[3 * r + cc] = box_and(e1, e2);
      k_point<<<nblk(box_n(mb[3 * r + cc]), 256), 256, 0, g->stream>>>(L, 2, 0, d1, d2, g->met[3 * r + cc], mb[3 * r + cc]);
      g->geom_launches += 3;
    }
  }
  Box rjb = all;
  for (int q = 0; q < 9; ++q) rjb = box_and(rjb, cdb[q]);
  {
    P9c cd;
    for (int q = 0; q < 9; ++q) cd.p[q] = g->cd[q];
    k_rj_box<<<nblk(box_n(rjb), 256), 256, 0, g->stream>>>(L, cd, g->rj, rjb);
    ++g->geom_launches;
  }
  Box mtb[3];
  if (g->p.moving) {
    // the line systems end where the valid range ends (R26): every array keeps exactly the box the passes give it
    P3c vt;
    for (int q = 0; q < 3; ++q) vt.p[q] = g->xt[q];
    for (int r = 0; r < 3; ++r) {
      mtb[r] = mb[3 * r];
      k_mt_box<<<nblk(box_n(mtb[r]), 256), 256, 0, g->stream>>>(L, vt, g->met[3 * r], g->met[3 * r + 1], g->met[3 * r + 2],
                                                                 g->mt[r], mtb[r]);
      ++g->geom_launches;
    }
  }
  // interface metrics: each hatted quantity interpolated as a whole, Eq. 38
  for (int d = 0; d < 3; ++d) {
    Box fb;   // interfaces 0..n_d of family d <-> H index -1..n_d-1
    for (int a = 0; a < 3; ++a) { fb.lo[a] = 0; fb.hi[a] = c.n[a]; }
    fb.lo[d] = -1;
    for (int q = 0; q < 11; ++q) {
      const double* src; Box sb; double* dst;
      if (q < 9) { src = g->met[q]; sb = mb[q]; dst = g->fmet[d][q]; }
      else if (q == 9) { src = g->rj; sb = rjb; dst = g->fmet[d][9]; }
      else { if (!g->p.moving) continue; src = g->mt[d]; sb = mtb[d]; dst = g->fmt[d]; }
      if (!dst) continue;
      const Box gb = launch_ig4(g, L, src, sb, d, f1);
      Box hb = gb;
      hb.lo[d] += 1; hb.hi[d] -= 2;
      for (int a = 0; a < 3; ++a)
        if (hb.lo[a] > fb.lo[a] || hb.hi[a] < fb.hi[a]) return cudaErrorInvalidValue;   // ghost depth too small
      k_H_from<<<nblk(box_n(fb), 256), 256, 0, g->stream>>>(L, c.LF[d], d, 1, src, f1, dst, fb);
      ++g->geom_launches;
    }
  }
  if (g->p.moving) { k_rjt<<<nblk(c.LC.n, 256), 256, 0, g->stream>>>(c, g->fmt[0], g->fmt[1], g->fmt[2], g->rjt); ++g->geom_launches; }
  return cudaGetLastError();
}

// stage 3: everything after the ghost coordinates (derivatives, metrics, 1/J, time metrics, interface values, GCL)
cudaError_t geom_rest(meg6_grid* g) {
  const Consts& c = g->c;
  P3 xc, xt, mt; P9 cd, met;
  for (int q = 0; q < 3; ++q) { xc.p[q] = g->xc[q]; xt.p[q] = g->xt[q]; mt.p[q] = g->mt[q]; }
  for (int q = 0; q < 9; ++q) { cd.p[q] = g->cd[q]; met.p[q] = g->met[q]; }
  if (g->p.scheme == 1) return launch_geometry_ig4(g);
  const int T = 256;
  // blocking along the grid line trades threads for shared intermediates: it pays once the grid fills the GPU several
  // times over (256^3: -7 % per call), not on config 2's 64^3 (+3 %)
  // MEG6_GEOM_BLOCKED=0/1 in the environment at grid_create forces the choice (the parity tests run both forms on the
  // same small grids)
  const bool blocked = g->geom_blocked >= 0 ? (g->geom_blocked == 1) : (c.LC.n >= (1LL << 21));
  g->geom_launches += 1 + 3 + (blocked ? 3 : 1) + (g->p.moving ? 1 : 0);   // coordinate derivatives, metric sweeps, interface families, GCL
  if (blocked) k_coord_deriv_blk<CD_KB><<<nblk((long long)c.LX.pi * c.LX.pj * nblk(c.n[2] + 2 * GX, CD_KB), T), T, 0, g->stream>>>(c, xc, cd, g->rj);
  else
  k_coord_deriv<<<nblk(c.LX.n, T), T, 0, g->stream>>>(c, xc, cd, g->rj);
  {
    const int e0 = c.n[0] + 10, e1 = c.n[1] + 10, e2 = c.n[2] + 10;
    k_met_dir<0><<<dim3(nblk(e0, MetCfg<0>::TS), nblk(e1, MetCfg<0>::TW), e2), 256, 0, g->stream>>>(c, xc, xt, cd, met, mt);
    k_met_dir<1><<<dim3(nblk(e0, MetCfg<1>::TW), nblk(e1, MetCfg<1>::TS), e2), 256, 0, g->stream>>>(c, xc, xt, cd, met, mt);
    k_met_dir<2><<<dim3(nblk(e0, MetCfg<2>::TW), nblk(e2, MetCfg<2>::TS), e1), 256, 0, g->stream>>>(c, xc, xt, cd, met, mt);
  }
  FaceJob3 jobs;
  for (int d = 0; d < 3; ++d) {
    FaceJob& job = jobs.job[d];
    job.n = 0;
    for (int q = 0; q < 10; ++q)
      if (g->fmet[d][q]) { job.src[job.n] = (q < 9) ? g->met[q] : g->rj; job.dst[job.n] = g->fmet[d][q]; ++job.n; }
    if (g->p.moving) { job.src[job.n] = g->mt[d]; job.dst[job.n] = g->fmt[d]; ++job.n; }
  }
  if (!blocked) {
    long long nmax = c.LF[0].n;
    for (int d = 1; d < 3; ++d) nmax = c.LF[d].n > nmax ? c.LF[d].n : nmax;
    k_face_metrics3<<<dim3(nblk(nmax, T), 3), T, 0, g->stream>>>(c, jobs);
  }
  for (int d = 0; d < 3 && blocked; ++d) {
    const FaceJob& job = jobs.job[d];
    if (d == 0) k_face_metrics<<<nblk(c.LF[d].n, T), T, 0, g->stream>>>(c, d, job);
    else {
      const Lay& LF = c.LF[d];
      const long long nthr = (long long)LF.pi * nblk(d == 1 ? LF.pj : LF.pk, FACE_KB) * (d == 1 ? LF.pk : LF.pj);
      k_face_metrics_blk<FACE_KB><<<nblk(nthr, T), T, 0, g->stream>>>(c, d, job);
    }
  }
  if (g->p.moving) k_rjt<<<nblk(c.LC.n, T), T, 0, g->stream>>>(c, g->fmt[0], g->fmt[1], g->fmt[2], g->rjt);
  return cudaGetLastError();
}

}  // namespace meg6
