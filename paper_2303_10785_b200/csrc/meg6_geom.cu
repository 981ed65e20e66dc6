// meg6_geom.cu -- metric / Jacobian kernels and their launcher.  Compiled with -fmad=false (see meg6_geom.cuh).
#include <math.h>
#include "meg6_geom.cuh"

namespace meg6 {

static inline unsigned nblk(long long n, int t) { return (unsigned)((n + t - 1) / t); }

cudaError_t launch_geometry(meg6_grid* g, double t) {
  const Consts& c = g->c;
  GeomIn gi;
  for (int q = 0; q < 3; ++q) { gi.node[q] = g->nodes[q]; gi.mode[q] = g->modes[q]; }
  const double ph = 2.0 * M_PI * g->p.omega * t;
  gi.s = g->p.moving ? sin(ph) : 0.0;
  gi.sd = g->p.moving ? 2.0 * M_PI * g->p.omega * cos(ph) : 0.0;
  P3 xc, xt, mt; P9 cd, met;
  for (int q = 0; q < 3; ++q) { xc.p[q] = g->xc[q]; xt.p[q] = g->xt[q]; mt.p[q] = g->mt[q]; }
  for (int q = 0; q < 9; ++q) { cd.p[q] = g->cd[q]; met.p[q] = g->met[q]; }
  const int T = 256;
  k_centres<<<nblk(c.LX.n, T), T, 0, g->stream>>>(c, gi, xc, xt);
  k_coord_deriv<<<nblk(c.LX.n, T), T, 0, g->stream>>>(c, xc, cd);
  const long long nm = (long long)(c.n[0] + 10) * (c.n[1] + 10) * (c.n[2] + 10);
  k_metrics<<<nblk(nm, 128), 128, 0, g->stream>>>(c, xc, xt, cd, met, g->rj, mt);
  for (int d = 0; d < 3; ++d) {
    FaceJob job;
    job.n = 0;
    for (int q = 0; q < 10; ++q)
      if (g->fmet[d][q]) { job.src[job.n] = (q < 9) ? g->met[q] : g->rj; job.dst[job.n] = g->fmet[d][q]; ++job.n; }
    if (g->p.moving) { job.src[job.n] = g->mt[d]; job.dst[job.n] = g->fmt[d]; ++job.n; }
    k_face_metrics<<<nblk(c.LF[d].n, T), T, 0, g->stream>>>(c, d, job);
  }
  if (g->p.moving) k_rjt<<<nblk(c.LC.n, T), T, 0, g->stream>>>(c, g->fmt[0], g->fmt[1], g->fmt[2], g->rjt);
  return cudaGetLastError();
}

}  // namespace meg6
