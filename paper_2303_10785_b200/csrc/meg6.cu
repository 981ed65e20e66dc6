// meg6.cu -- host side of the C ABI declared in include/meg6.h: workspace carving, kernel launches.
// Single translation unit of libmeg6.so (sm_100a).  No CPU fallback; shares nothing with oracle/.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <mutex>
#include <new>

#include "meg6_common.cuh"
#include "meg6_flow.cuh"
#include "meg6_flux3.cuh"
#include "meg6_probe.cuh"
#include <stdlib.h>

using namespace meg6;

static thread_local char g_err[512] = "";

static meg6_status fail(meg6_status s, const char* fmt, const char* a = "") {
  snprintf(g_err, sizeof(g_err), fmt, a);
  return s;
}
#define CUDA_OK(call)                                                              \
  do {                                                                             \
    cudaError_t e_ = (call);                                                       \
    if (e_ != cudaSuccess) return fail(MEG6_ECUDA, #call ": %s", cudaGetErrorString(e_)); \
  } while (0)

static bool params_ok(const meg6_params* p) {
  if (!p) return false;
  if (p->ni < 10 || p->nj < 10 || p->nk < 10) return false;
  if (p->scheme != 0 && p->scheme != 1) return false;
  if (!(p->gamma > 1.0) || !(p->r_gas > 0.0)) return false;
  for (int d = 0; d < 3; ++d)
    if (!p->periodic[d])
      for (int s = 0; s < 2; ++s)
      {
        const int bc = p->bc[2 * d + s];
        if (bc < 1 || bc > 5) return false;
        if (bc >= 3 && p->moving) return false;   // Table 1 gives the wall rules without a wall velocity (R27)
      }
  if (p->viscous && !(p->prandtl > 0.0)) return false;
  return true;
}

static Consts make_consts(const meg6_params* p) {
  Consts c;
  memset(&c, 0, sizeof(c));
  c.n[0] = p->ni; c.n[1] = p->nj; c.n[2] = p->nk;
  for (int d = 0; d < 3; ++d) {
    c.periodic[d] = p->periodic[d] ? 1 : 0;
    for (int q = 0; q < 3; ++q) c.period[d][q] = p->period[d][q];
  }
  c.viscous = p->viscous ? 1 : 0;
  c.moving = p->moving ? 1 : 0;
  for (int f = 0; f < 6; ++f) c.bc[f] = p->bc[f];
  c.gamma = p->gamma; c.r_gas = p->r_gas; c.prandtl = p->prandtl;
  c.mu_ref = p->mu_ref; c.t_ref = p->t_ref; c.s_suth = p->s_suth;
  c.mp_alpha = p->mp_alpha; c.p_out = p->p_out;
  c.kappa_fac = p->viscous ? p->gamma * p->r_gas / ((p->gamma - 1.0) * p->prandtl) : 0.0;
  c.igm1 = 1.0 / (p->gamma - 1.0);
  c.suth_c = (p->viscous && p->s_suth >= 0.0) ? p->mu_ref * (p->t_ref + p->s_suth) / (p->t_ref * sqrt(p->t_ref)) : 0.0;
  c.LX = make_lay(p->ni, p->nj, p->nk, GX, GX, GX);
  // row pitches are even so that every TMA global stride is a multiple of 16 bytes
  c.LP = make_lay(p->ni, p->nj, p->nk, GPI, GPJ, GPK, 2);
  c.LG = make_lay(p->ni, p->nj, p->nk, GGI, GGJ, GGK, 2);
  c.LC = make_lay(p->ni, p->nj, p->nk, 0, 0, 0);
  c.LR = make_lay(p->ni, p->nj, p->nk, 0, 0, 0, 2);
  c.LF[0] = make_lay(p->ni + 1, p->nj, p->nk, 0, 0, 0, 2);
  c.LF[1] = make_lay(p->ni, p->nj + 1, p->nk, 0, 0, 0, 2);
  c.LF[2] = make_lay(p->ni, p->nj, p->nk + 1, 0, 0, 0, 2);
  auto fs = [](long long n) { return (long long)(((size_t)n * 8 + 255) / 256 * 256 / 8); };
  c.fsP = fs(c.LP.n); c.fsG = fs(c.LG.n); c.fsR = fs(c.LR.n);
  for (int d = 0; d < 3; ++d) c.fsM[d] = fs(c.LF[d].n);
  return c;
}

// Carves the workspace; with g == nullptr only sizes it.
static size_t carve(const meg6_params* p, const Consts& c, meg6_grid* g, char* base) {
  size_t off = 0;
  auto take = [&](long long n_doubles) -> double* {
    double* ptr = base ? (double*)(base + off) : nullptr;
    off += ((size_t)n_doubles * sizeof(double) + 255) / 256 * 256;
    return ptr;
  };
  const long long nn = (long long)(p->ni + 1) * (p->nj + 1) * (p->nk + 1);
  meg6_grid tmp = meg6_grid();
  meg6_grid* G = g ? g : &tmp;
  for (int q = 0; q < 3; ++q) G->nodes[q] = take(nn);
  for (int q = 0; q < 3; ++q) G->modes[q] = p->moving ? take(nn) : nullptr;
  for (int q = 0; q < 3; ++q) G->xc[q] = take(c.LX.n);
  for (int q = 0; q < 3; ++q) G->xt[q] = p->moving ? take(c.LX.n) : nullptr;
  for (int q = 0; q < 9; ++q) G->cd[q] = take(c.LX.n);
  for (int q = 0; q < 9; ++q) G->met[q] = take(c.LX.n);
  G->rj = take(c.LX.n);
  for (int q = 0; q < 3; ++q) G->mt[q] = p->moving ? take(c.LX.n) : nullptr;
  for (int d = 0; d < 3; ++d) {
    for (int q = 0; q < 10; ++q) {
      const bool own = (q >= 3 * d && q < 3 * d + 3);
      G->fmet[d][q] = (own || p->viscous) ? take(c.LF[d].n) : nullptr;
    }
    G->fmt[d] = p->moving ? take(c.LF[d].n) : nullptr;
  }
  G->rjt = p->moving ? take(c.LC.n) : nullptr;
  for (int q = 0; q < 6; ++q) G->scr[q] = (p->scheme == 1) ? take(c.LX.n) : nullptr;
  for (int d = 0; d < 3; ++d)
    for (int f = 0; f < 6; ++f) G->Gi[d][f] = (p->scheme == 1) ? take(c.LP.n) : nullptr;
  {
    const int mx = (p->ni > p->nj ? (p->ni > p->nk ? p->ni : p->nk) : (p->nj > p->nk ? p->nj : p->nk)) + 2 * GX;
    G->ig4_cc = (p->scheme == 1) ? take(mx) : nullptr;
    G->ig4_den = (p->scheme == 1) ? take(mx) : nullptr;
  }
  for (int f = 0; f < 6; ++f) G->P[f] = take(c.LP.n);
  for (int f = 0; f < 6; ++f) G->Pb[f] = take(c.LP.n);   // ping-pong partner written by the fused last sweep
  for (int e = 0; e < 3; ++e)
    for (int f = 0; f < 4; ++f) G->G[e][f] = (p->viscous && p->scheme == 0) ? take(c.LG.n) : nullptr;
  G->res = take(c.LR.n);
  for (int f = 1; f < 5; ++f) take(c.LR.n);   // fields c.fsR apart
  G->U0 = take(5 * c.LC.n);
  for (int f = 0; f < 6; ++f) {
    const int d = f / 2;
    G->inflow[f] = nullptr;
    G->link[f] = nullptr;
    G->ibuf[f] = nullptr;
    if (!p->periodic[d] && p->bc[f] == 1) {
      int a = (d + 1) % 3, b = (d + 2) % 3;
      G->inflow[f] = take(5LL * c.n[a] * c.n[b]);
    }
  }
  G->stats = (unsigned long long*)take(2);
  G->red = take(4 * CFL_BLOCKS);
  G->tp = take(16);
  return off;
}

static inline unsigned nblk(long long n, int t) { return (unsigned)((n + t - 1) / t); }
namespace meg6 {
cudaError_t geom_centres(meg6_grid* g, double t);
cudaError_t geom_extend(meg6_grid* g, int d);
cudaError_t geom_rest(meg6_grid* g);
cudaError_t geom_pack(meg6_grid* g, int face, double* layers);
Box launch_ig4(meg6_grid* g, const Lay& L, const double* f, const Box& fb, int dir, double* out);
Box launch_ig4_batch(meg6_grid* g, const Lay& L, const double* f, const Box& fb, int dir, double* out, int nfields,
                     long long fs_in, long long fs_out);
Box launch_ig4_flow(meg6_grid* g, const Lay& L, const double* f, const Box& fb, int dir, double* out, int nfields,
                    long long fs_in, long long fs_out);
}

// ---- TMA descriptors (cuTensorMapEncodeTiled through the runtime's driver entry point: no libcuda link) ----
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static bool make_map4(EncodeTiledFn fn, CUtensorMap* tm, const double* base, const Lay& L, long long fs, int nfields,
                      const int box[4]) {
  cuuint64_t dims[4] = {(cuuint64_t)L.pi, (cuuint64_t)L.pj, (cuuint64_t)L.pk, (cuuint64_t)nfields};
  cuuint64_t strides[3] = {(cuuint64_t)L.sj * 8, (cuuint64_t)L.sk * 8, (cuuint64_t)fs * 8};
  cuuint32_t bx[4] = {(cuuint32_t)box[0], (cuuint32_t)box[1], (cuuint32_t)box[2], (cuuint32_t)box[3]};
  cuuint32_t es[4] = {1, 1, 1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void*)base, dims, strides, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int DIR, bool VISC>
static bool make_maps3_dir(EncodeTiledFn fn, meg6_grid* g, int buf) {
  if (g->p.scheme == 1) {
    // MIG4: same tiles, gradients from the line-solve arrays Gi (layout of the primitives)
    using C = Cfg3<DIR, VISC, true>;
    const Consts& c = g->c;
    TmaMaps& t = g->tmaps3[buf][DIR];
    auto box = [](int sweep, int trans, int nf, int out[4]) {
      if (DIR == 0) { out[0] = sweep; out[1] = trans; out[2] = 1; }
      else if (DIR == 1) { out[0] = trans; out[1] = sweep; out[2] = 1; }
      else { out[0] = trans; out[1] = 1; out[2] = sweep; }
      out[3] = nf;
    };
    int b[4];
    bool ok = true;
    box(C::LPT, C::TT, C::NF, b);
    ok = ok && make_map4(fn, &t.P, buf ? g->Pb[0] : g->P[0], c.LP, c.fsP, 6, b);
    box(C::LF, C::TT, C::NM, b);
    ok = ok && make_map4(fn, &t.M, VISC ? g->fmet[DIR][0] : g->fmet[DIR][3 * DIR], c.LF[DIR], c.fsM[DIR], C::NM, b);
    if (g->p.moving) {
      box(C::LF, C::TT, 1, b);
      ok = ok && make_map4(fn, &t.Mt, g->fmt[DIR], c.LF[DIR], c.fsM[DIR], 1, b);
    }
    box(C::LQ, C::TT, C::NF, b);
    ok = ok && make_map4(fn, &t.Q, g->Gi[DIR][0], c.LP, c.fsP, 6, b);
    if (VISC) {
      int slot = 0;
      for (int e = 0; e < 3; ++e) {
        if (e == DIR) continue;
        box(C::LG, C::TT, 5, b);
        ok = ok && make_map4(fn, &t.G3[slot], g->Gi[e][0], c.LP, c.fsP, 6, b);
        ++slot;
      }
    }
    return ok;
  }
  using C = Cfg3<DIR, VISC>;
  const Consts& c = g->c;
  TmaMaps& t = g->tmaps3[buf][DIR];
  auto box = [](int sweep, int trans, int nf, int out[4]) {
    if (DIR == 0) { out[0] = sweep; out[1] = trans; out[2] = 1; }
    else if (DIR == 1) { out[0] = trans; out[1] = sweep; out[2] = 1; }
    else { out[0] = trans; out[1] = 1; out[2] = sweep; }
    out[3] = nf;
  };
  int b[4];
  bool ok = true;
  box(C::LPT, C::TT, C::NF, b);
  ok = ok && make_map4(fn, &t.P, buf ? g->Pb[0] : g->P[0], c.LP, c.fsP, 6, b);
  box(C::LF, C::TT, C::NM, b);
  ok = ok && make_map4(fn, &t.M, VISC ? g->fmet[DIR][0] : g->fmet[DIR][3 * DIR], c.LF[DIR], c.fsM[DIR], C::NM, b);
  if (g->p.moving) {
    box(C::LF, C::TT, 1, b);
    ok = ok && make_map4(fn, &t.Mt, g->fmt[DIR], c.LF[DIR], c.fsM[DIR], 1, b);
  }
  if (VISC) {
    box(C::LG, C::TT, 4, b);
    ok = ok && make_map4(fn, &t.G, g->G[0][0], c.LG, c.fsG, 12, b);
  }
  if (C::nR) {   // running residual of the tile, read by the second sweep
    box(C::TS, C::TT, 5, b);
    ok = ok && make_map4(fn, &t.R, g->res, c.LR, c.fsR, 5, b);
  }
  return ok;
}

static cudaError_t setup_tma(meg6_grid* g) {
  void* fp = nullptr;
  cudaDriverEntryPointQueryResult qr;
  cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fp, cudaEnableDefault, &qr);
  if (e != cudaSuccess) return e;
  if (!fp || qr != cudaDriverEntryPointSuccess) return cudaErrorNotSupported;
  EncodeTiledFn fn = (EncodeTiledFn)fp;
  bool ok = true;
  for (int buf = 0; buf < 2 && ok; ++buf) {
    if (g->p.viscous) ok = make_maps3_dir<0, true>(fn, g, buf) && make_maps3_dir<1, true>(fn, g, buf) && make_maps3_dir<2, true>(fn, g, buf);
    else ok = make_maps3_dir<0, false>(fn, g, buf) && make_maps3_dir<1, false>(fn, g, buf) && make_maps3_dir<2, false>(fn, g, buf);
  }
  if (!ok) return cudaErrorInvalidValue;
  // final phase of the fused xi sweep (MEG6): U^n and 1/J tiles; sigma and the caller's U are encoded when they are known
  g->encode_fn = (void*)fn;
  g->mapU_ptr = nullptr; g->mapSg_ptr = nullptr;
  g->tail_ok = g->p.scheme == 0 && (g->c.n[0] % 2 == 0) && Cfg3<0, true>::nU > 0;
  if (g->tail_ok) {
    const int b5[4] = {Cfg3<0, true>::TS, Cfg3<0, true>::TT, 1, 5}, b1[4] = {Cfg3<0, true>::TS, Cfg3<0, true>::TT, 1, 1};
    g->tail_ok = make_map4(fn, &g->mapU0, g->U0, g->c.LC, g->c.LC.n, 5, b5) &&
                 make_map4(fn, &g->mapJ, g->rj, g->c.LX, g->c.LX.n, 1, b1);
  }
  // opt in to the dynamic shared memory the flux kernels need
#define SET_SMEM3(D, V, F)                                                                                  \
  if ((e = cudaFuncSetAttribute(k_flux3<D, V, F>, cudaFuncAttributeMaxDynamicSharedMemorySize,              \
                                Cfg3<D, V>::SMEM_BYTES)) != cudaSuccess) return e;
  SET_SMEM3(0, false, true) SET_SMEM3(1, false, false) SET_SMEM3(2, false, false)
  SET_SMEM3(0, true, true) SET_SMEM3(1, true, false) SET_SMEM3(2, true, false)
#undef SET_SMEM3
#define SET_SMEM3I(D, V, F)                                                                                 \
  if ((e = cudaFuncSetAttribute(k_flux3<D, V, F, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,        \
                                Cfg3<D, V, true>::SMEM_BYTES)) != cudaSuccess) return e;
  if (g->p.scheme == 1) {
    SET_SMEM3I(0, false, true) SET_SMEM3I(1, false, false) SET_SMEM3I(2, false, false)
    SET_SMEM3I(0, true, true) SET_SMEM3I(1, true, false) SET_SMEM3I(2, true, false)
  }
#undef SET_SMEM3I
  return cudaSuccess;
}

// ---- per-kernel timing: one event pair per launch (or launch group) while profiling is enabled ----
struct ProfScope {
  meg6_grid* g; size_t rec;
  ProfScope(meg6_grid* g_, int kind, int launches) : g(g_), rec((size_t)-1) {
    if (!g->prof_on) return;
    while (g->prof_pool.size() < g->prof_used + 2) {
      cudaEvent_t e;
      if (cudaEventCreate(&e) != cudaSuccess) return;
      g->prof_pool.push_back(e);
    }
    meg6_grid::ProfRec r;
    r.kind = kind; r.launches = launches; r.e0 = g->prof_used; r.e1 = g->prof_used + 1;
    g->prof_used += 2;
    cudaEventRecord(g->prof_pool[r.e0], g->stream);
    g->prof_recs.push_back(r);
    rec = g->prof_recs.size() - 1;
  }
  void set_launches(int n) { if (rec != (size_t)-1) g->prof_recs[rec].launches = n; }
  ~ProfScope() {
    if (rec != (size_t)-1) cudaEventRecord(g->prof_pool[g->prof_recs[rec].e1], g->stream);
  }
};

// ---- meg6_cfl_dt_noalloc: the time-step reduction with its scratch in a static device array (include/meg6.h) ----
// One partial minimum pair per block of NOALLOC_CPB consecutive cells; the array holds NOALLOC_MAX_BLOCKS pairs, i.e.
// grids of up to NOALLOC_MAX_CELLS cells.  256 KiB of device memory on every GPU that loads the library, until exit.
// In HOST code the name g_noalloc_scratch is a stand-in for the symbol, not a device address: the address the kernels
// get comes from cudaGetSymbolAddress, taken once per device at grid creation with that device current.
constexpr int NOALLOC_CPB = 1024;                                   // cells per block (256 threads x 4)
constexpr long long NOALLOC_MAX_CELLS = 1LL << 24;                  // 16 777 216 cells (config 4: 12.8 M; 256^3)
constexpr int NOALLOC_MAX_BLOCKS = (int)(NOALLOC_MAX_CELLS / NOALLOC_CPB);
static __device__ __align__(256) double g_noalloc_scratch[2 * NOALLOC_MAX_BLOCKS];

// Eq. B.2 / B.3 per cell as in k_cfl; block b reduces cells [b CPB, (b+1) CPB) and writes its pair
__global__ void __launch_bounds__(256) k_cfl_part(Consts c, const double* __restrict__ U, CflIn in, double* __restrict__ part) {
  const long long N = c.LC.n;
  double inv_min = INFINITY, vis_min = INFINITY;
  const long long first = (long long)blockIdx.x * NOALLOC_CPB;
  for (int q = 0; q < NOALLOC_CPB / 256; ++q) {
    const long long tid = first + q * 256 + threadIdx.x;
    if (tid >= N) break;
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
  if (threadIdx.x == 0) { part[2 * blockIdx.x] = sa[0]; part[2 * blockIdx.x + 1] = sb[0]; }
}

// the nb pairs of THIS call (the array keeps older calls' pairs beyond nb: they are not read) -> dt in device memory
__global__ void __launch_bounds__(256) k_cfl_fin(const double* __restrict__ part, int nb, double cfl, int viscous,
                                                 double* __restrict__ dt) {
  double a = INFINITY, b = INFINITY;
  for (int q = threadIdx.x; q < nb; q += 256) { a = fmin(a, part[2 * q]); b = fmin(b, part[2 * q + 1]); }
  __shared__ double sa[256], sb[256];
  sa[threadIdx.x] = a; sb[threadIdx.x] = b;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      sa[threadIdx.x] = fmin(sa[threadIdx.x], sa[threadIdx.x + o]);
      sb[threadIdx.x] = fmin(sb[threadIdx.x], sb[threadIdx.x + o]);
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double r = sa[0];
    if (viscous) r = fmin(r, sb[0] / 4.0);   // R25: the alpha of Eq. B.3 read as alpha^D = 4
    *dt = cfl * r;
  }
}

// device address of the static scratch array on the CURRENT device, resolved once per device (set-up time)
static cudaError_t noalloc_scratch_address(double** out) {
  static double* addr[64] = {nullptr};
  static std::mutex mu;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= 64) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  if (!addr[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    addr[dev] = ptr;
  }
  *out = addr[dev];
  return cudaSuccess;
}

extern "C" {

meg6_status meg6_profile_enable(meg6_grid* g, int on) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  g->prof_on = on ? 1 : 0;
  return MEG6_OK;
}

meg6_status meg6_profile_read(meg6_grid* g, double* ms, unsigned long long* launches) {
  if (!g || !ms || !launches) return fail(MEG6_EINVAL, "profile_read: null pointer%s");
  CUDA_OK(cudaStreamSynchronize(g->stream));
  for (int k = 0; k < 16; ++k) { ms[k] = 0.0; launches[k] = 0; }
  for (const meg6_grid::ProfRec& r : g->prof_recs) {
    float t = 0.f;
    CUDA_OK(cudaEventElapsedTime(&t, g->prof_pool[r.e0], g->prof_pool[r.e1]));
    ms[r.kind] += t; launches[r.kind] += r.launches;
  }
  g->prof_recs.clear(); g->prof_used = 0;
  return MEG6_OK;
}

int meg6_version(void) { return 1000; }
const char* meg6_last_error(void) { return g_err; }

size_t meg6_workspace_bytes(const meg6_params* p) {
  if (!params_ok(p)) { fail(MEG6_EINVAL, "invalid params%s"); return 0; }
  Consts c = make_consts(p);
  return carve(p, c, nullptr, nullptr);
}

meg6_status meg6_grid_create(const meg6_params* p, const double* x, const double* y, const double* z,
                             const double* dxm, const double* dym, const double* dzm, void* workspace,
                             size_t workspace_bytes, void* cuda_stream, meg6_grid** out) {
  if (!params_ok(p)) return fail(MEG6_EINVAL, "invalid params%s");
  if (!x || !y || !z || !workspace || !out) return fail(MEG6_EINVAL, "null pointer%s");
  if (p->moving && (!dxm || !dym || !dzm)) return fail(MEG6_EINVAL, "moving mesh needs displacement modes%s");
  if (((uintptr_t)workspace & 255) != 0) return fail(MEG6_EINVAL, "workspace must be 256-byte aligned%s");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return fail(MEG6_ECUDA, "no CUDA device%s");
  meg6_grid* g = new (std::nothrow) meg6_grid();   // value-initialised: all pointers null, flags zero
  if (!g) return fail(MEG6_ENOMEM, "host allocation failed%s");
  g->p = *p;
  g->c = make_consts(p);
  g->stream = (cudaStream_t)cuda_stream;
  g->ws = (char*)workspace; g->ws_bytes = workspace_bytes;
  {
    const char* forced = getenv("MEG6_GEOM_BLOCKED");   // read once, here: which form of the geometry kernels (tests)
    g->geom_blocked = forced ? (forced[0] == '1' ? 1 : 0) : -1;
  }
  const size_t need = carve(p, g->c, g, g->ws);
  if (need > workspace_bytes) { delete g; return fail(MEG6_ENOMEM, "workspace too small%s"); }
  const size_t nn = (size_t)(p->ni + 1) * (p->nj + 1) * (p->nk + 1) * sizeof(double);
  const double* src[3] = {x, y, z};
  const double* msrc[3] = {dxm, dym, dzm};
  cudaError_t e = cudaMemsetAsync(g->ws, 0, need, g->stream);
  for (int q = 0; q < 3 && e == cudaSuccess; ++q) {
    e = cudaMemcpyAsync(g->nodes[q], src[q], nn, cudaMemcpyDeviceToDevice, g->stream);
    if (e == cudaSuccess && p->moving) e = cudaMemcpyAsync(g->modes[q], msrc[q], nn, cudaMemcpyDeviceToDevice, g->stream);
  }
  if (e == cudaSuccess && p->scheme == 1) {
    // Thomas elimination coefficients of the IG4 systems (position-only; R26): den_q = 1 - alpha c_{q-1}, c_q = alpha/den_q
    const int mx = (p->ni > p->nj ? (p->ni > p->nk ? p->ni : p->nk) : (p->nj > p->nk ? p->nj : p->nk)) + 2 * GX;
    std::vector<double> cc(mx, 0.0), den(mx, 1.0);
    const double al = 5.0 / 14.0;
    for (int q = 1; q < mx; ++q) { den[q] = 1.0 - al * cc[q - 1]; cc[q] = al / den[q]; }
    e = cudaMemcpyAsync(g->ig4_cc, cc.data(), sizeof(double) * mx, cudaMemcpyHostToDevice, g->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g->ig4_den, den.data(), sizeof(double) * mx, cudaMemcpyHostToDevice, g->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(g->stream);   // the host vectors go out of scope
  }
  if (e == cudaSuccess) e = setup_tma(g);
  if (e == cudaSuccess) e = noalloc_scratch_address(&g->noalloc_scratch);   // set-up: this grid's device is current
  if (e != cudaSuccess) { delete g; return fail(MEG6_ECUDA, "grid_create: %s", cudaGetErrorString(e)); }
  *out = g;
  return MEG6_OK;
}

void meg6_grid_destroy(meg6_grid* g) {
  if (!g) return;
  for (cudaEvent_t e : g->prof_pool) cudaEventDestroy(e);
  if (g->steps_graph) cudaGraphExecDestroy(g->steps_graph);
  delete g;
}

static bool links_ok(const meg6_grid* g, bool single);

// Geometry of n linked blocks together: cell centres of all, then the ghost coordinates direction by direction over all
// blocks (repeated where a link is rotated, R29), then each block's metrics.
meg6_status meg6_metrics_compute_blocks(int n, meg6_grid* const* g, double t) {
  if (n < 1 || !g) return fail(MEG6_EINVAL, "metrics_compute_blocks: no blocks%s");
  bool todo = false, rot = false;
  for (int b = 0; b < n; ++b) {
    if (!g[b]) return fail(MEG6_EINVAL, "metrics_compute_blocks: null grid%s");
    if (!links_ok(g[b], false)) return fail(MEG6_ESTATE, "metrics_compute: block-interface face without a link%s");
    for (int f = 0; f < 6; ++f) {   // every neighbour must be in the list: its cell centres are read
      const meg6_grid* nb = g[b]->link[f];
      bool found = nb == nullptr;
      for (int q = 0; q < n && !found; ++q) found = g[q] == nb;
      if (!found) return fail(MEG6_ESTATE, "metrics_compute: a linked neighbour block is not in the call (use meg6_metrics_compute_blocks)%s");
    }
    todo = todo || !g[b]->have_metrics || g[b]->p.moving;
    rot = rot || g[b]->rotated;
  }
  if (!todo) return MEG6_OK;   // static: idempotent
  cudaError_t e = cudaSuccess;
  std::vector<ProfScope*> scopes;
  for (int b = 0; b < n; ++b) g[b]->geom_launches = 0;
  {
    // one timing scope over the whole call, charged to the first block
    ProfScope ps(g[0], 0, 0);
    for (int b = 0; b < n && e == cudaSuccess; ++b) e = meg6::geom_centres(g[b], t);
    for (int pass = 0; pass < (rot ? 3 : 1); ++pass)
      for (int d = 0; d < 3; ++d)
        for (int b = 0; b < n && e == cudaSuccess; ++b) e = meg6::geom_extend(g[b], d);
    for (int b = 0; b < n && e == cudaSuccess; ++b) e = meg6::geom_rest(g[b]);   // meg6_geom.cu (-fmad=false)
    int nl = 0;
    for (int b = 0; b < n; ++b) nl += g[b]->geom_launches;
    ps.set_launches(nl);
  }
  if (e != cudaSuccess) return fail(MEG6_ECUDA, "metrics_compute: %s", cudaGetErrorString(e));
  for (int b = 0; b < n; ++b) g[b]->have_metrics = true;
  return MEG6_OK;
}

meg6_status meg6_metrics_compute(meg6_grid* g, double t) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  return meg6_metrics_compute_blocks(1, &g, t);
}

// ---- staged geometry (blocks on different devices): centres -> for d: [pack / deliver] extend(d) -> finish ----
size_t meg6_geom_interface_doubles(const meg6_grid* g, int face) {
  if (!g || face < 0 || face > 5) return 0;
  const int d = face / 2;
  const int e1 = (d == 0) ? 1 : 0, e2 = (d == 2) ? 1 : 2;
  return (size_t)(g->p.moving ? 6 : 3) * GX * (size_t)(g->c.n[e1] + 2 * GX) * (size_t)(g->c.n[e2] + 2 * GX);
}

meg6_status meg6_set_geom_interface_buffer(meg6_grid* g, int face, const double* layers, const double* off) {
  if (!g || face < 0 || face > 5) return fail(MEG6_EINVAL, "set_geom_interface_buffer: bad argument%s");
  if (g->p.periodic[face / 2] || g->p.bc[face] != 5) return fail(MEG6_EINVAL, "set_geom_interface_buffer: face is not a block-interface face (bc 5)%s");
  g->gbuf[face] = layers;
  for (int q = 0; q < 3; ++q) g->goff[face][q] = off ? off[q] : 0.0;
  return MEG6_OK;
}

meg6_status meg6_stage_geom_centres(meg6_grid* g, double t) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  g->geom_launches = 0;
  CUDA_OK(meg6::geom_centres(g, t));
  return MEG6_OK;
}

meg6_status meg6_stage_geom_pack(meg6_grid* g, int face, double* layers) {
  if (!g || !layers || face < 0 || face > 5) return fail(MEG6_EINVAL, "stage_geom_pack: bad argument%s");
  CUDA_OK(meg6::geom_pack(g, face, layers));
  return MEG6_OK;
}

meg6_status meg6_stage_geom_extend(meg6_grid* g, int d) {
  if (!g || d < 0 || d > 2) return fail(MEG6_EINVAL, "stage_geom_extend: bad argument%s");
  for (int side = 0; side < 2; ++side) {
    const int f = 2 * d + side;
    if (!g->p.periodic[d] && g->p.bc[f] == 5 && !g->link[f] && !g->gbuf[f])
      return fail(MEG6_ESTATE, "stage_geom_extend: block-interface face without a link or a coordinate buffer%s");
  }
  CUDA_OK(meg6::geom_extend(g, d));
  return MEG6_OK;
}

meg6_status meg6_stage_geom_finish(meg6_grid* g) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  {
    ProfScope ps(g, 0, 0);
    const cudaError_t e = meg6::geom_rest(g);
    ps.set_launches(g->geom_launches);
    if (e != cudaSuccess) return fail(MEG6_ECUDA, "stage_geom_finish: %s", cudaGetErrorString(e));
  }
  g->have_metrics = true;
  return MEG6_OK;
}

meg6_status meg6_set_inflow(meg6_grid* g, int face, const double* P_in) {
  if (!g || !P_in || face < 0 || face > 5) return fail(MEG6_EINVAL, "set_inflow: bad argument%s");
  if (!g->inflow[face]) return fail(MEG6_EINVAL, "set_inflow: face is not a fixed-inflow face%s");
  const int d = face / 2, a = (d + 1) % 3, b = (d + 2) % 3;
  CUDA_OK(cudaMemcpyAsync(g->inflow[face], P_in, sizeof(double) * 5 * (size_t)g->c.n[a] * g->c.n[b],
                          cudaMemcpyDeviceToDevice, g->stream));
  return MEG6_OK;
}

meg6_status meg6_set_sponge(meg6_grid* g, const double* sigma, const double* U_ref) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  if ((sigma == nullptr) != (U_ref == nullptr)) return fail(MEG6_EINVAL, "set_sponge: both or neither%s");
  g->sigma = sigma; g->uref = U_ref;
  return MEG6_OK;
}

// ghost layers of direction d in primitive buffer `buf` (the lower directions are filled already).  Block interfaces
// read the SAME buffer of the neighbour block: with several blocks, direction d is filled in every block before
// direction d+1 in any (edge and corner ghosts then arrive from the diagonal neighbours in two steps).
static cudaError_t fill_ghosts_dir(meg6_grid* g, int buf, int d, bool edges = false) {
  const Consts& c = g->c;
  if (edges && (c.periodic[d] || (!g->link[2 * d] && !g->link[2 * d + 1]))) return cudaSuccess;
  double* const* Pc = buf ? g->Pb : g->P;
  P6 P;
  for (int f = 0; f < 6; ++f) P.p[f] = Pc[f];
  int a = (d + 1) % 3, b = (d + 2) % 3;
  if (a > b) { int t = a; a = b; b = t; }
  const long long ea = c.n[a] + ((a < d || edges) ? 12 : 0), eb = c.n[b] + ((b < d || edges) ? 12 : 0);
  GhostIn gin;
  memset(&gin, 0, sizeof(gin));
  gin.edges = edges ? 1 : 0;
  for (int side = 0; side < 2; ++side) gin.edge[side] = (c.bc[2 * d + side] == 5 && g->link[2 * d + side]) ? 1 : 0;
  gin.inflow[0] = g->inflow[2 * d]; gin.inflow[1] = g->inflow[2 * d + 1];
  gin.mx = g->met[3 * d]; gin.my = g->met[3 * d + 1]; gin.mz = g->met[3 * d + 2];
  for (int side = 0; side < 2; ++side) {
    const meg6_grid* nb = g->link[2 * d + side];
    if (nb) {
      gin.nbP[side] = buf ? nb->Pb[0] : nb->P[0];
      gin.nbL[side] = nb->c.LP; gin.nbfs[side] = nb->c.fsP;
      for (int e = 0; e < 3; ++e) { gin.nax[side][e] = g->lax[2 * d + side][e]; gin.nsg[side][e] = g->lsg[2 * d + side][e]; gin.nsh[side][e] = g->lsh[2 * d + side][e]; }
    } else if (g->ibuf[2 * d + side]) {   // packed layers of a remote neighbour: a block six cells thick, aligned
      gin.nbP[side] = g->ibuf[2 * d + side];
      gin.nbL[side] = pack_lay(c.LP, d); gin.nbfs[side] = gin.nbL[side].n;
      for (int e = 0; e < 3; ++e) { gin.nax[side][e] = e; gin.nsg[side][e] = 1; gin.nsh[side][e] = 0; }
      gin.nsh[side][d] = side ? -c.n[d] : 6;
    }
  }
  ProfScope ps(g, 2, 1);
  k_ghost<<<nblk(ea * eb * 12, 256), 256, 0, g->stream>>>(c, d, P, gin);
  return cudaGetLastError();
}

static cudaError_t fill_ghosts(meg6_grid* g, int buf) {
  const Consts& c = g->c;
  if (c.periodic[0] && c.periodic[1] && c.periodic[2]) {   // all wraps: one launch (k_ghost_periodic)
    P6 P;
    for (int f = 0; f < 6; ++f) P.p[f] = buf ? g->Pb[f] : g->P[f];
    const long long e0 = c.n[0] + 12, e1 = c.n[1] + 12;
    const long long nthr = e0 * e1 * 12 + e0 * 12 * c.n[2] + 12LL * c.n[1] * c.n[2];
    ProfScope ps(g, 2, 1);
    k_ghost_periodic<<<nblk(nthr, 256), 256, 0, g->stream>>>(c, P);
    return cudaGetLastError();
  }
  for (int pass = 0; pass < (g->rotated ? 3 : 1); ++pass)
    for (int d = 0; d < 3; ++d) {
      const cudaError_t e = fill_ghosts_dir(g, buf, d);
      if (e != cudaSuccess) return e;
    }
  for (int d = 0; d < 3; ++d) {   // edge round (R28): a block linked to itself
    const cudaError_t e = fill_ghosts_dir(g, buf, d, true);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

static bool links_ok(const meg6_grid* g, bool single) {
  for (int f = 0; f < 6; ++f)
    if (!g->p.periodic[f / 2] && g->p.bc[f] == 5) {
      if (!g->link[f] && !g->ibuf[f]) return false;
      if (single && g->link[f] != g) return false;   // a single-grid call may only see itself across an interface
    }
  return true;
}

// One RK stage (or one dQ/dt evaluation) for the state whose primitives are in buffer `buf` (ghosts filled):
// stored gradients, eta and zeta sweeps into g->res, xi sweep fused with the residual
// assembly, the stage update and the primitive conversion of the new state (into the other buffer).
static meg6_status stage_sweeps(meg6_grid* g, int buf, const Fuse3& fu) {
  const Consts& c = g->c;
  double* const* Pc = buf ? g->Pb : g->P;
  P6 P;
  for (int f = 0; f < 6; ++f) P.p[f] = Pc[f];
  const bool IG = g->p.scheme == 1;
  if (IG) {
    // MIG4: implicit gradients of every staged field along the three directions (Eq. 18), whole grid lines
    ProfScope ps(g, 3, 3);
    meg6::Box pb;
    for (int a = 0; a < 3; ++a) { pb.lo[a] = -6; pb.hi[a] = c.n[a] + 6; }
    // the fields of P and of Gi[d] are fsP doubles apart: one launch per direction for all of them
    for (int d = 0; d < 3; ++d) meg6::launch_ig4_flow(g, c.LP, Pc[0], pb, d, g->Gi[d][0], g->p.viscous ? 6 : 5, c.fsP, c.fsP);
  } else if (g->p.viscous) {
    P12 G;
    for (int e = 0; e < 3; ++e)
      for (int f = 0; f < 4; ++f) G.p[4 * e + f] = g->G[e][f];
    ProfScope ps(g, 3, 1);
    k_grad<<<dim3(nblk(c.LG.pi / 2, 32), nblk(c.n[1] + 2, 8), nblk(c.n[2] + 2, GRAD_KB)), dim3(32, 8, 1), 0, g->stream>>>(c, P, G, 1);
  }
  CUDA_OK(cudaGetLastError());
  FluxIn3 i3;
  i3.res = g->res; i3.stats = g->stats_on ? g->stats : nullptr; i3.moving = g->p.moving ? 1 : 0; i3.mask = nullptr;
  i3.gown = (g->p.viscous && !IG) ? g->G[1][0] : nullptr; i3.gfs = c.fsG;
  const bool V = g->p.viscous != 0;
  TmaMaps tm[3] = {g->tmaps3[buf][0], g->tmaps3[buf][1], g->tmaps3[buf][2]};
  if (fu.tail_tma) { tm[0].U = g->mapU; tm[0].U0 = g->mapU0; tm[0].J = g->mapJ; if (g->sigma) tm[0].Sg = g->mapSg; }
#define LAUNCH3(D, VV, FF, GRID)                                                                                        \
  do {                                                                                                                  \
    if (IG) k_flux3<D, VV, FF, true><<<GRID, Cfg3<D, VV, true>::NT, Cfg3<D, VV, true>::SMEM_BYTES, g->stream>>>(c, i3, tm[D], fu); \
    else k_flux3<D, VV, FF><<<GRID, Cfg3<D, VV>::NT, Cfg3<D, VV>::SMEM_BYTES, g->stream>>>(c, i3, tm[D], fu);           \
  } while (0)
  // sweep order eta, zeta, xi: the fused final phase then works on rows that are contiguous along xi
  {
    ProfScope ps(g, 5, 1);
    i3.first = 1; i3.mask = g->bmask[1];
    dim3 grid(nblk(c.n[0], Cfg3<1, false>::TT), nblk(c.n[1], Cfg3<1, false>::TS * (IG ? 1 : Cfg3<1, false>::NSUB)), c.n[2]);
    if (V) LAUNCH3(1, true, false, grid); else LAUNCH3(1, false, false, grid);
  }
  {
    ProfScope ps(g, 6, 1);
    i3.first = 0; i3.mask = g->bmask[2];
    dim3 grid(nblk(c.n[0], Cfg3<2, false>::TT), nblk(c.n[2], Cfg3<2, false>::TS * (IG ? 1 : Cfg3<2, false>::NSUB)), c.n[1]);
    if (V) LAUNCH3(2, true, false, grid); else LAUNCH3(2, false, false, grid);
  }
  {
    ProfScope ps(g, 4, 1);
    i3.mask = g->bmask[0];
    dim3 grid(nblk(c.n[0], Cfg3<0, false>::TS), nblk(c.n[1], Cfg3<0, false>::TT), c.n[2]);
    if (V) LAUNCH3(0, true, true, grid); else LAUNCH3(0, false, true, grid);
  }
#undef LAUNCH3
  CUDA_OK(cudaGetLastError());
  return MEG6_OK;
}

static meg6_status stage(meg6_grid* g, int buf, const Fuse3& fu) {
  CUDA_OK(fill_ghosts(g, buf));
  return stage_sweeps(g, buf, fu);
}

static cudaError_t launch_prim(meg6_grid* g, const double* U) {
  P6 P;
  for (int f = 0; f < 6; ++f) P.p[f] = g->P[f];
  ProfScope ps(g, 1, 1);
  k_prim<<<nblk(g->c.LC.n, 256), 256, 0, g->stream>>>(g->c, U, P);
  return cudaGetLastError();
}

static Fuse3 make_fuse(meg6_grid* g, const double* U, double* out) {
  Fuse3 fu;
  memset(&fu, 0, sizeof(fu));
  fu.U = U; fu.out = out; fu.U0 = g->U0;
  fu.rj = g->rj; fu.rjt = g->p.moving ? g->rjt : nullptr;
  fu.sigma = g->sigma; fu.uref = g->uref;
  // tensor maps of the caller's arrays, re-encoded only when a pointer changes
  fu.tail_tma = 0;
  if (g->tail_ok && (reinterpret_cast<uintptr_t>(U) & 15) == 0 && (!g->sigma || (reinterpret_cast<uintptr_t>(g->sigma) & 15) == 0)) {
    EncodeTiledFn fn = (EncodeTiledFn)g->encode_fn;
    const int b5[4] = {Cfg3<0, true>::TS, Cfg3<0, true>::TT, 1, 5}, b1[4] = {Cfg3<0, true>::TS, Cfg3<0, true>::TT, 1, 1};
    bool ok = true;
    if (g->mapU_ptr != U) { ok = make_map4(fn, &g->mapU, U, g->c.LC, g->c.LC.n, 5, b5); g->mapU_ptr = ok ? U : nullptr; }
    if (ok && g->sigma && g->mapSg_ptr != g->sigma) {
      ok = make_map4(fn, &g->mapSg, g->sigma, g->c.LC, g->c.LC.n, 1, b1); g->mapSg_ptr = ok ? g->sigma : nullptr;
    }
    fu.tail_tma = ok ? 1 : 0;
  }
  return fu;
}

meg6_status meg6_rhs(meg6_grid* g, const double* U, double* dUdt) {
  if (!g || !U || !dUdt) return fail(MEG6_EINVAL, "rhs: null pointer%s");
  if (!g->have_metrics) return fail(MEG6_ESTATE, "rhs called before metrics_compute%s");
  if (!links_ok(g, true)) return fail(MEG6_ESTATE, "rhs: block-interface face without a link, or linked to another block (use meg6_rhs_blocks)%s");
  CUDA_OK(launch_prim(g, U));
  Fuse3 fu = make_fuse(g, U, dUdt);
  fu.mode = 0;
  return stage(g, 0, fu);
}

static const double RK_A[3] = {0.0, 3.0 / 4.0, 1.0 / 3.0}, RK_B[3] = {1.0, 1.0 / 4.0, 2.0 / 3.0};

// stage s of a step whose primitives are in buffer `buf`; more: another stage follows that may use the primitives of the
// state this one produces (always within a step; across steps only inside meg6_rk3_steps, where nobody touches U)
static Fuse3 make_fuse_rk(meg6_grid* g, double* U, int s, double dt, int buf = -1, bool more = false) {
  if (buf < 0) buf = s & 1;
  Fuse3 fu = make_fuse(g, U, U);
  fu.mode = 1; fu.a = RK_A[s]; fu.b = RK_B[s]; fu.dt = dt;
  fu.U0w = (s == 0) ? g->U0 : nullptr;                                // stage 1 saves U^n on the way
  fu.Pn = (s < 2 || more) ? (buf ? g->P[0] : g->Pb[0]) : nullptr;     // primitives of the next stage's state
  return fu;
}

meg6_status meg6_rk3_step(meg6_grid* g, double* U, double t, double dt) {
  if (!g || !U) return fail(MEG6_EINVAL, "rk3_step: null pointer%s");
  if (!g->have_metrics && !g->p.moving) return fail(MEG6_ESTATE, "rk3_step called before metrics_compute%s");
  if (!links_ok(g, true)) return fail(MEG6_ESTATE, "rk3_step: block-interface face without a link, or linked to another block (use meg6_rk3_step_blocks)%s");
  const double ts[3] = {t, t + dt, t + 0.5 * dt};
  CUDA_OK(launch_prim(g, U));   // the caller owns U: its primitives are recomputed at every step
  for (int s = 0; s < 3; ++s) {
    meg6_status st;
    if (g->p.moving && (st = meg6_metrics_compute(g, ts[s])) != MEG6_OK) return st;
    if ((st = stage(g, s & 1, make_fuse_rk(g, U, s, dt))) != MEG6_OK) return st;
  }
  return MEG6_OK;
}

// n steps of constant dt in one call: the time loop stays in the library (nothing leaves the device between
// steps), so the primitives of U^{n+1} that the last sweep of a step can write on its way are those of the next step's
// first stage -- the separate conversion kernel runs once per call instead of once per step.
meg6_status meg6_rk3_steps(meg6_grid* g, double* U, double t, double dt, int nsteps) {
  if (!g || !U || nsteps < 0) return fail(MEG6_EINVAL, "rk3_steps: bad argument%s");
  if (nsteps == 0) return MEG6_OK;
  if (!g->have_metrics && !g->p.moving) return fail(MEG6_ESTATE, "rk3_steps called before metrics_compute%s");
  if (!links_ok(g, true)) return fail(MEG6_ESTATE, "rk3_steps: block-interface face without a link, or linked to another block%s");
  CUDA_OK(launch_prim(g, U));
  int buf = 0, n0 = 0;
  // (stream capture is not available on the legacy default stream: callers that want the graph pass their own stream)
  if (!g->prof_on && nsteps >= 2 && g->stream != nullptr && g->stream != cudaStreamLegacy &&
      g->stream != cudaStreamPerThread) {
    // two steps (six stages: the primitive buffers swap roles every stage) as one CUDA graph.  Small grids are bound by the
    // launch rate of the host (config 1: 18 launches of ~5 us of work each per step; config 2: 54 with the geometry)
    meg6_grid::GraphKey key;
    memset(&key, 0, sizeof(key));
    key.U = U; key.dt = dt; key.sigma = g->sigma; key.uref = g->uref; key.stats_on = g->stats_on;
    for (int d = 0; d < 3; ++d) key.bm[d] = g->bmask[d];
    if (!g->steps_graph || memcmp(&key, &g->steps_key, sizeof(key)) != 0) {
      if (g->steps_graph) { cudaGraphExecDestroy(g->steps_graph); g->steps_graph = nullptr; }
      (void)make_fuse(g, U, U);   // tensor maps of the caller's arrays encoded before the capture
      cudaGraph_t graph = nullptr;
      CUDA_OK(cudaStreamBeginCapture(g->stream, cudaStreamCaptureModeThreadLocal));
      meg6_status st = MEG6_OK;
      int b = 0;
      for (int q = 0; q < 6 && st == MEG6_OK; ++q, b ^= 1) {
        if (g->p.moving) {   // the geometry of stage q at ITS time: the two time factors are read from g->tp at replay
          g->tp_cur = g->tp + 2 * q;
          st = meg6_metrics_compute(g, 0.0);
          g->tp_cur = nullptr;
        }
        if (st == MEG6_OK) st = stage(g, b, make_fuse_rk(g, U, q % 3, dt, b, true));
      }
      const cudaError_t ec = cudaStreamEndCapture(g->stream, &graph);
      if (st != MEG6_OK) { if (graph) cudaGraphDestroy(graph); return st; }
      CUDA_OK(ec);
      const cudaError_t ei = cudaGraphInstantiate(&g->steps_graph, graph, 0);
      cudaGraphDestroy(graph);
      CUDA_OK(ei);
      g->steps_key = key;
    }
    for (; n0 + 2 <= nsteps; n0 += 2) {
      if (g->p.moving) {
        // moving mesh: the stage times of these two steps, as the factors meg6_metrics_compute(t) forms on the host
        // (same expressions, same bits); the copy is ordered after the previous replay on the stream
        double tp[12];
        for (int q = 0; q < 6; ++q) {
          const double tn = t + (n0 + q / 3) * dt;
          const double ts = (q % 3 == 0) ? tn : (q % 3 == 1) ? tn + dt : tn + 0.5 * dt;
          const double ph = 2.0 * M_PI * g->p.omega * ts;
          tp[2 * q] = sin(ph); tp[2 * q + 1] = 2.0 * M_PI * g->p.omega * cos(ph);
        }
        CUDA_OK(cudaMemcpyAsync(g->tp, tp, sizeof(tp), cudaMemcpyHostToDevice, g->stream));
      }
      CUDA_OK(cudaGraphLaunch(g->steps_graph, g->stream));
    }
  }
  for (int n = n0; n < nsteps; ++n) {
    const double tn = t + n * dt;
    const double ts[3] = {tn, tn + dt, tn + 0.5 * dt};
    for (int s = 0; s < 3; ++s) {
      meg6_status st;
      if (g->p.moving && (st = meg6_metrics_compute(g, ts[s])) != MEG6_OK) return st;
      if ((st = stage(g, buf, make_fuse_rk(g, U, s, dt, buf, n + 1 < nsteps))) != MEG6_OK) return st;
      buf ^= 1;
    }
  }
  return MEG6_OK;
}

// ---- multi-block (Sec. 6; Table 1 last column; R28) ----
meg6_status meg6_link_blocks_oriented(meg6_grid* home, int face, meg6_grid* nb, int nb_face, int swap, int flip_a, int flip_b,
                                      const double* off) {
  if (!home || !nb || face < 0 || face > 5 || nb_face < 0 || nb_face > 5) return fail(MEG6_EINVAL, "link_blocks: bad argument%s");
  const int d = face / 2, dn = nb_face / 2;
  if (home->p.periodic[d] || home->p.bc[face] != 5) return fail(MEG6_EINVAL, "link_blocks: face is not a block-interface face (bc 5)%s");
  if (nb->p.periodic[dn]) return fail(MEG6_EINVAL, "link_blocks: the neighbour is periodic in that direction%s");
  int a = (d + 1) % 3, b = (d + 2) % 3, an = (dn + 1) % 3, bn = (dn + 2) % 3;
  if (a > b) { int t = a; a = b; b = t; }
  if (an > bn) { int t = an; an = bn; bn = t; }
  const int ta = swap ? bn : an, tb = swap ? an : bn;   // images of the home axes a, b
  if (nb->c.n[ta] != home->c.n[a] || nb->c.n[tb] != home->c.n[b])
    return fail(MEG6_EINVAL, "link_blocks: the interface planes of the two blocks have different cell counts%s");
  if (nb->stream != home->stream) return fail(MEG6_EINVAL, "link_blocks: the blocks must share one stream%s");
  if (nb->p.moving != home->p.moving || nb->p.scheme != home->p.scheme || nb->p.viscous != home->p.viscous)
    return fail(MEG6_EINVAL, "link_blocks: the blocks differ in scheme, viscous or moving%s");
  int* ax = home->lax[face]; int* sg = home->lsg[face]; int* sh = home->lsh[face];
  ax[a] = ta; sg[a] = flip_a ? -1 : 1; sh[a] = flip_a ? home->c.n[a] - 1 : 0;
  ax[b] = tb; sg[b] = flip_b ? -1 : 1; sh[b] = flip_b ? home->c.n[b] - 1 : 0;
  // along the normal: ghost layer q of home = the q-th interior cell of the neighbour counted from nb_face
  const int n = home->c.n[d], nn = nb->c.n[dn], hs = face & 1, ns = nb_face & 1;
  ax[d] = dn;
  if (hs && !ns) { sg[d] = 1; sh[d] = -n; }
  else if (hs && ns) { sg[d] = -1; sh[d] = nn - 1 + n; }
  else if (!hs && ns) { sg[d] = 1; sh[d] = nn; }
  else { sg[d] = -1; sh[d] = -1; }
  for (int q = 0; q < 3; ++q) home->loff[face][q] = off ? off[q] : 0.0;
  home->link[face] = nb;
  home->ibuf[face] = nullptr; home->gbuf[face] = nullptr;
  const bool aligned = ax[0] == 0 && ax[1] == 1 && ax[2] == 2 && sg[0] > 0 && sg[1] > 0 && sg[2] > 0;
  if (!aligned) { home->rotated = true; nb->rotated = true; }
  home->have_metrics = false;   // the ghost coordinates of this face change with the link
  return MEG6_OK;
}

meg6_status meg6_link_blocks(meg6_grid* home, int face, meg6_grid* nb) {
  if (!home || !nb || face < 0 || face > 5) return fail(MEG6_EINVAL, "link_blocks: bad argument%s");
  const int d = face / 2;
  for (int e = 0; e < 3; ++e)
    if (e != d && nb->c.periodic[e] != home->c.periodic[e])
      return fail(MEG6_EINVAL, "link_blocks: transverse sizes or periodicity differ%s");
  return meg6_link_blocks_oriented(home, face, nb, face ^ 1, 0, 0, 0, nullptr);
}

// rotated links (R29): the neighbour cell behind an edge or corner ghost may itself be a ghost of a direction the
// neighbour fills later; repeating the fill makes every ghost cell the fixed point of the exchange
static int ghost_passes(int n, meg6_grid* const* g) {
  for (int b = 0; b < n; ++b)
    if (g[b]->rotated) return 3;
  return 1;
}

static meg6_status blocks_ok(int n, meg6_grid* const* g, const char* who) {
  if (n < 1 || !g) return fail(MEG6_EINVAL, "%s: no blocks", who);
  for (int b = 0; b < n; ++b) {
    if (!g[b]) return fail(MEG6_EINVAL, "%s: null grid", who);
    if (g[b]->stream != g[0]->stream) return fail(MEG6_EINVAL, "%s: the blocks must share one stream", who);
    if (!links_ok(g[b], false)) return fail(MEG6_ESTATE, "%s: block-interface face without a link", who);
    for (int f = 0; f < 6; ++f) {   // every neighbour must be advanced by the same call
      const meg6_grid* nb = g[b]->link[f];
      bool found = nb == nullptr;
      for (int q = 0; q < n && !found; ++q) found = g[q] == nb;
      if (!found) return fail(MEG6_EINVAL, "%s: a linked neighbour is not in the block list", who);
    }
  }
  return MEG6_OK;
}

meg6_status meg6_rhs_blocks(int n, meg6_grid* const* g, const double* const* U, double* const* dUdt) {
  meg6_status st = blocks_ok(n, g, "rhs_blocks");
  if (st != MEG6_OK) return st;
  if (!U || !dUdt) return fail(MEG6_EINVAL, "rhs_blocks: null pointer%s");
  for (int b = 0; b < n; ++b) {
    if (!U[b] || !dUdt[b]) return fail(MEG6_EINVAL, "rhs_blocks: null pointer%s");
    if (!g[b]->have_metrics) return fail(MEG6_ESTATE, "rhs_blocks called before metrics_compute%s");
    CUDA_OK(launch_prim(g[b], U[b]));
  }
  for (int pass = 0; pass < ghost_passes(n, g); ++pass)
    for (int d = 0; d < 3; ++d)
      for (int b = 0; b < n; ++b) CUDA_OK(fill_ghosts_dir(g[b], 0, d));
  for (int d = 0; d < 3; ++d)   // edge round (R28; nothing is launched for a block without linked faces along d)
    for (int b = 0; b < n; ++b) CUDA_OK(fill_ghosts_dir(g[b], 0, d, true));
  for (int b = 0; b < n; ++b) {
    Fuse3 fu = make_fuse(g[b], U[b], dUdt[b]);
    fu.mode = 0;
    if ((st = stage_sweeps(g[b], 0, fu)) != MEG6_OK) return st;
  }
  return MEG6_OK;
}

meg6_status meg6_rk3_step_blocks(int n, meg6_grid* const* g, double* const* U, double t, double dt) {
  meg6_status st = blocks_ok(n, g, "rk3_step_blocks");
  if (st != MEG6_OK) return st;
  if (!U) return fail(MEG6_EINVAL, "rk3_step_blocks: null pointer%s");
  for (int b = 0; b < n; ++b) {
    if (!U[b]) return fail(MEG6_EINVAL, "rk3_step_blocks: null pointer%s");
    if (!g[b]->have_metrics && !g[b]->p.moving) return fail(MEG6_ESTATE, "rk3_step_blocks called before metrics_compute%s");
    CUDA_OK(launch_prim(g[b], U[b]));
  }
  const double ts[3] = {t, t + dt, t + 0.5 * dt};
  for (int s = 0; s < 3; ++s) {
    // every block writes the primitives of its new state into the buffer NOT read by this stage, so the ghost
    // exchange of the next stage finds all neighbours' interiors complete
    if (g[0]->p.moving && (st = meg6_metrics_compute_blocks(n, g, ts[s])) != MEG6_OK) return st;
    for (int pass = 0; pass < ghost_passes(n, g); ++pass)
      for (int d = 0; d < 3; ++d)
        for (int b = 0; b < n; ++b) CUDA_OK(fill_ghosts_dir(g[b], s & 1, d));
    for (int d = 0; d < 3; ++d)
      for (int b = 0; b < n; ++b) CUDA_OK(fill_ghosts_dir(g[b], s & 1, d, true));
    for (int b = 0; b < n; ++b)
      if ((st = stage_sweeps(g[b], s & 1, make_fuse_rk(g[b], U[b], s, dt))) != MEG6_OK) return st;
  }
  return MEG6_OK;
}

// ---- staged stepping: the pieces of one RK stage as separate calls, for callers that exchange interface layers
// themselves between the ghost fill of one direction and the next (blocks on other devices) ----
size_t meg6_interface_doubles(const meg6_grid* g, int face) {
  if (!g || face < 0 || face > 5) return 0;
  return (size_t)(6 * pack_lay(g->c.LP, face / 2).n);
}

meg6_status meg6_set_interface_buffer(meg6_grid* g, int face, const double* layers) {
  if (!g || face < 0 || face > 5) return fail(MEG6_EINVAL, "set_interface_buffer: bad argument%s");
  if (g->p.periodic[face / 2] || g->p.bc[face] != 5) return fail(MEG6_EINVAL, "set_interface_buffer: face is not a block-interface face (bc 5)%s");
  g->ibuf[face] = layers;
  if (layers) g->link[face] = nullptr;
  return MEG6_OK;
}

static bool staged_ok(const meg6_grid* g) {
  for (int f = 0; f < 6; ++f)
    if (!g->p.periodic[f / 2] && g->p.bc[f] == 5 && !g->link[f] && !g->ibuf[f]) return false;
  return true;
}

meg6_status meg6_stage_prim(meg6_grid* g, const double* U) {
  if (!g || !U) return fail(MEG6_EINVAL, "stage_prim: null pointer%s");
  CUDA_OK(launch_prim(g, U));
  return MEG6_OK;
}

meg6_status meg6_stage_ghosts(meg6_grid* g, int s, int d) {
  if (!g || s < 0 || s > 2 || d < 0 || d > 2) return fail(MEG6_EINVAL, "stage_ghosts: bad argument%s");
  if (!g->have_metrics) return fail(MEG6_ESTATE, "stage_ghosts called before metrics_compute%s");
  if (!staged_ok(g)) return fail(MEG6_ESTATE, "stage_ghosts: block-interface face without a link or a buffer%s");
  CUDA_OK(fill_ghosts_dir(g, s & 1, d));
  return MEG6_OK;
}

meg6_status meg6_stage_pack(meg6_grid* g, int s, int face, double* layers) {
  if (!g || !layers || s < 0 || s > 2 || face < 0 || face > 5) return fail(MEG6_EINVAL, "stage_pack: bad argument%s");
  const int d = face / 2;
  const Lay LQ = pack_lay(g->c.LP, d);
  const int first = (face & 1) ? g->c.n[d] - 6 : 0;   // the layers a neighbour beyond this face needs
  ProfScope ps(g, 2, 1);
  k_pack<<<nblk(LQ.n, 256), 256, 0, g->stream>>>(g->c.LP, LQ, d, first, g->c.fsP, (s & 1) ? g->Pb[0] : g->P[0], layers);
  CUDA_OK(cudaGetLastError());
  return MEG6_OK;
}

meg6_status meg6_stage_sweeps(meg6_grid* g, double* U, double* dUdt, int s, double dt) {
  if (!g || !U || s < 0 || s > 2) return fail(MEG6_EINVAL, "stage_sweeps: bad argument%s");
  if (!g->have_metrics) return fail(MEG6_ESTATE, "stage_sweeps called before metrics_compute%s");
  if (dUdt) {   // plain right-hand side of the state whose primitives are in buffer 0
    if (s != 0) return fail(MEG6_EINVAL, "stage_sweeps: dUdt is written at s == 0 only%s");
    Fuse3 fu = make_fuse(g, U, dUdt);
    fu.mode = 0;
    return stage_sweeps(g, 0, fu);
  }
  return stage_sweeps(g, s & 1, make_fuse_rk(g, U, s, dt));
}

meg6_status meg6_cfl_dt(meg6_grid* g, const double* U, double cfl, double* dt) {
  if (!g || !U || !dt) return fail(MEG6_EINVAL, "cfl_dt: null pointer%s");
  if (!g->have_metrics) return fail(MEG6_ESTATE, "cfl_dt called before metrics_compute%s");
  CflIn in;
  for (int q = 0; q < 9; ++q) in.met[q] = g->met[q];
  for (int q = 0; q < 3; ++q) in.mt[q] = g->mt[q];
  in.rj = g->rj;
  const int nb = (int)((g->c.LC.n + 255) / 256 < CFL_BLOCKS ? (g->c.LC.n + 255) / 256 : CFL_BLOCKS);
  { ProfScope ps(g, 9, 1); k_cfl<<<nb, 256, 0, g->stream>>>(g->c, U, in, g->red); }
  static thread_local double host[2 * CFL_BLOCKS];
  CUDA_OK(cudaMemcpyAsync(host, g->red, sizeof(double) * 2 * nb, cudaMemcpyDeviceToHost, g->stream));
  CUDA_OK(cudaStreamSynchronize(g->stream));
  double a = INFINITY, b = INFINITY;
  for (int q = 0; q < nb; ++q) { a = fmin(a, host[2 * q]); b = fmin(b, host[2 * q + 1]); }
  double r = a;
  if (g->p.viscous) r = fmin(r, b / 4.0);   // R25: the alpha of Eq. B.3 read as alpha^D = 4
  *dt = cfl * r;
  return MEG6_OK;
}

meg6_status meg6_cfl_dt_noalloc(meg6_grid* g, const double* U, double cfl, double* dt_device) {
  if (!g || !U || !dt_device) return fail(MEG6_EINVAL, "cfl_dt_noalloc: null pointer%s");
  if (g->c.LC.n > NOALLOC_MAX_CELLS)
    return fail(MEG6_EINVAL, "cfl_dt_noalloc: the grid has more cells than the static scratch array holds (maximum 16777216 = 2^24 cells; use meg6_cfl_dt)%s");
  if (!g->have_metrics) return fail(MEG6_ESTATE, "cfl_dt_noalloc called before metrics_compute%s");
  if (!g->noalloc_scratch) return fail(MEG6_ESTATE, "cfl_dt_noalloc: scratch address not resolved%s");
  CflIn in;
  for (int q = 0; q < 9; ++q) in.met[q] = g->met[q];
  for (int q = 0; q < 3; ++q) in.mt[q] = g->mt[q];
  in.rj = g->rj;
  const int nb = (int)((g->c.LC.n + NOALLOC_CPB - 1) / NOALLOC_CPB);
  k_cfl_part<<<nb, 256, 0, g->stream>>>(g->c, U, in, g->noalloc_scratch);
  k_cfl_fin<<<1, 256, 0, g->stream>>>(g->noalloc_scratch, nb, cfl, g->p.viscous ? 1 : 0, dt_device);
  CUDA_OK(cudaGetLastError());
  return MEG6_OK;
}

meg6_status meg6_diagnostics(meg6_grid* g, const double* U, double* out) {
  if (!g || !U || !out) return fail(MEG6_EINVAL, "diagnostics: null pointer%s");
  if (!g->have_metrics) return fail(MEG6_ESTATE, "diagnostics called before metrics_compute%s");
  const Consts& c = g->c;
  CUDA_OK(launch_prim(g, U));
  CUDA_OK(fill_ghosts(g, 0));
  DiagIn in;
  memset(&in, 0, sizeof(in));
  for (int q = 0; q < 9; ++q) in.met[q] = g->met[q];
  in.rj = g->rj;
  for (int f = 0; f < 4; ++f) in.P[f] = g->P[f];
  in.ig4 = g->p.scheme == 1;
  if (in.ig4) {
    meg6::Box pb;
    for (int a = 0; a < 3; ++a) { pb.lo[a] = -6; pb.hi[a] = c.n[a] + 6; }
    for (int d = 0; d < 3; ++d)
      for (int cc = 0; cc < 3; ++cc) {
        meg6::launch_ig4(g, c.LP, g->P[1 + cc], pb, d, g->Gi[d][1 + cc]);
        in.g[3 * d + cc] = g->Gi[d][1 + cc];
      }
  }
  const int nb = (int)((c.LC.n + 255) / 256 < CFL_BLOCKS ? (c.LC.n + 255) / 256 : CFL_BLOCKS);
  k_diag<<<nb, 256, 0, g->stream>>>(c, in, g->red);
  CUDA_OK(cudaGetLastError());
  static thread_local double host[3 * CFL_BLOCKS];
  CUDA_OK(cudaMemcpyAsync(host, g->red, sizeof(double) * 3 * nb, cudaMemcpyDeviceToHost, g->stream));
  CUDA_OK(cudaStreamSynchronize(g->stream));
  double ke = 0.0, en = 0.0, vol = 0.0;
  for (int q = 0; q < nb; ++q) { ke += host[3 * q]; en += host[3 * q + 1]; vol += host[3 * q + 2]; }
  out[0] = ke / vol; out[1] = en / vol; out[2] = vol;
  return MEG6_OK;
}

meg6_status meg6_fp64_peak(void* cuda_stream, double* scratch, double* dfma_per_second) {
  if (!scratch || !dfma_per_second) return fail(MEG6_EINVAL, "fp64_peak: null pointer%s");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0, nsm = 0;
  CUDA_OK(cudaGetDevice(&dev));
  CUDA_OK(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = nsm * 8 * 4;   // four waves of eight 256-thread CTAs per SM
  cudaEvent_t e0, e1;
  CUDA_OK(cudaEventCreate(&e0));
  CUDA_OK(cudaEventCreate(&e1));
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {   // the first repetition warms up
    cudaEventRecord(e0, st);
    k_dfma_probe<<<blocks, PROBE_THREADS, 0, st>>>(1.0000001, 1e-9, scratch);
    cudaEventRecord(e1, st);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); cudaEventDestroy(e1); return fail(MEG6_ECUDA, "fp64_peak: %s", cudaGetErrorString(e)); }
    const double rate = (double)blocks * PROBE_THREADS * PROBE_CHAINS * PROBE_ITERS / (ms * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  *dfma_per_second = best;
  return MEG6_OK;
}

meg6_status meg6_limiter_stats_enable(meg6_grid* g, int on) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  g->stats_on = on ? 1 : 0;
  return MEG6_OK;
}

meg6_status meg6_set_branch_masks(meg6_grid* g, unsigned short* xi, unsigned short* eta, unsigned short* zeta) {
  if (!g) return fail(MEG6_EINVAL, "null grid%s");
  g->bmask[0] = xi; g->bmask[1] = eta; g->bmask[2] = zeta;
  return MEG6_OK;
}

meg6_status meg6_limiter_stats(meg6_grid* g, unsigned long long* n_limited, unsigned long long* n_tested) {
  if (!g || !n_limited || !n_tested) return fail(MEG6_EINVAL, "limiter_stats: null pointer%s");
  unsigned long long h[2];
  CUDA_OK(cudaMemcpyAsync(h, g->stats, sizeof(h), cudaMemcpyDeviceToHost, g->stream));
  CUDA_OK(cudaStreamSynchronize(g->stream));
  *n_limited = h[0]; *n_tested = h[1];
  return MEG6_OK;
}

meg6_status meg6_get_array(meg6_grid* g, int kind, int which, double* out) {
  if (!g || !out) return fail(MEG6_EINVAL, "get_array: null pointer%s");
  const Consts& c = g->c;
  const double* src = nullptr;
  Lay L = c.LX;
  int ext[3] = {c.n[0], c.n[1], c.n[2]};
  if (kind == 0) {
    if (which >= 0 && which < 9) src = g->met[which];
    else if (which == 9) src = g->rj;
    else if (which >= 10 && which < 13) src = g->mt[which - 10];
    else if (which == 13) { src = g->rjt; L = c.LC; }
    else if (which >= 14 && which < 17) src = g->xc[which - 14];
  } else if (kind == 1) {
    const int d = which / 16, q = which % 16;
    if (d >= 0 && d < 3 && q >= 0 && q <= 10) { src = (q < 10) ? g->fmet[d][q] : g->fmt[d]; L = c.LF[d]; ext[d] += 1; }
  } else if (kind == 2) {
    if (which >= 0 && which < 6) { src = g->P[which]; L = c.LP; }
  }
  if (!src) return fail(MEG6_EINVAL, "get_array: no such array%s");
  // strided device-to-host copy of the interior box
  cudaMemcpy3DParms p3;
  memset(&p3, 0, sizeof(p3));
  p3.srcPtr = make_cudaPitchedPtr((void*)src, (size_t)L.pi * sizeof(double), L.pi, L.pj);
  p3.srcPos = make_cudaPos((size_t)L.gi * sizeof(double), L.gj, L.gk);
  p3.dstPtr = make_cudaPitchedPtr(out, (size_t)ext[0] * sizeof(double), ext[0], ext[1]);
  p3.extent = make_cudaExtent((size_t)ext[0] * sizeof(double), ext[1], ext[2]);
  p3.kind = cudaMemcpyDeviceToHost;
  CUDA_OK(cudaMemcpy3DAsync(&p3, g->stream));
  CUDA_OK(cudaStreamSynchronize(g->stream));
  return MEG6_OK;
}

}  // extern "C"
