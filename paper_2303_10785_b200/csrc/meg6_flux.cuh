// meg6_flux.cuh -- per-direction flux kernel: E6 gradients + Eq. 19 second derivatives of the tile in shared
// memory, characteristic projection, MP limiter, contravariant HLLC, alpha-damping viscous flux, flux
// difference (SURVEY 8(a) rows R-xi/eta/zeta and V; paper Fig. 3, Fig. 5).
#pragma once
#include "meg6_common.cuh"
#include "meg6_flow.cuh"

namespace meg6 {

__device__ __forceinline__ double minmod(double a, double b) {   // E.2
  const double m = fmin(fabs(a), fabs(b));
  const bool same = ((__double2hiint(a) ^ __double2hiint(b)) >= 0);
  return same ? copysign(m, a) : 0.0;
}

struct Eig { double nx, ny, nz, ra, a2; };

// W = Linv * P (A.6a; R6) for one 5-vector (rho,u,v,w,p)
__device__ __forceinline__ void project(const Eig& e, double r, double u, double v, double w, double p, double W[5]) {
  const double un = fma(e.nz, w, fma(e.ny, v, e.nx * u));
  W[0] = fma(-e.ra, un, p);
  W[4] = fma(e.ra, un, p);
  const double q = fma(e.a2, r, -p);
  W[1] = fma(e.nx, q, fma(e.ny, w, -e.nz * v));
  W[2] = fma(e.nz, q, fma(e.nx, v, -e.ny * u));
  W[3] = fma(-e.ny, q, fma(e.nx, w, -e.nz * u));
}

// P = Rmat * W (A.4b; R6)
__device__ __forceinline__ void backproject(const Eig& e, double ia2, double h_ira, const double W[5], double P[5]) {
  const double sp = W[0] + W[4];
  P[0] = ia2 * fma(0.5, sp, fma(e.nx, W[1], fma(e.nz, W[2], -e.ny * W[3])));
  const double s = h_ira * (W[4] - W[0]);
  P[1] = fma(e.nx, s, -fma(e.ny, W[2], e.nz * W[3]));
  P[2] = fma(e.ny, s, fma(e.nx, W[2], -e.nz * W[1]));
  P[3] = fma(e.nz, s, fma(e.ny, W[1], e.nx * W[3]));
  P[4] = 0.5 * sp;
}

// App. E (R7): full limiting path, returns the limited value (w if `fail` is false).
__device__ __forceinline__ double mp_full(double w, double c0, double cm, double cp, double dnear, double dfar,
                                          double alpha, bool fail) {
  const double d0 = c0 - cm;
  const double wmd = fma(-0.5, dnear, 0.5 * (c0 + cp));
  const double wul = fma(alpha, d0, c0);
  const double wlc = fma(4.0 / 3.0, dfar, 0.5 * (3.0 * c0 - cm));
  const double wmin = fmax(fmin(fmin(c0, cp), wmd), fmin(fmin(c0, wul), wlc));
  const double wmax = fmin(fmax(fmax(c0, cp), wmd), fmax(fmax(c0, wul), wlc));
  const double lim = w + minmod(wmin - w, wmax - w);   // E.4
  return fail ? lim : w;
}

// E.1: true when the unlimited value must be limited
__device__ __forceinline__ bool mp_test(double w, double c0, double cm, double cp, double alpha) {
  const double wmp = c0 + minmod(cp - c0, alpha * (c0 - cm));
  return !((w - c0) * (w - wmp) <= 1e-20);
}

// Contravariant HLLC, Eq. 26-27 with the flux of Eq. 2; energy row R9; cascade R10.
__device__ __forceinline__ void hllc(const double PL[5], const double PR[5], double mx, double my, double mz, double mt,
                                     double g, double g2, double ig2, double gamma, double F[5]) {
  const double igm1 = 1.0 / (gamma - 1.0);
  const double UL = fma(mz, PL[3], fma(my, PL[2], fma(mx, PL[1], mt)));
  const double UR = fma(mz, PR[3], fma(my, PR[2], fma(mx, PR[1], mt)));
  const double cL = sqrt(gamma * PL[4] / PL[0]), cR = sqrt(gamma * PR[4] / PR[0]);
  const double SL = fmin(UL - cL * g, UR - cR * g);
  const double SR = fmax(UL + cL * g, UR + cR * g);
  const double SS = (PR[0] * UR * (SR - UR) - PL[0] * UL * (SL - UL) + (PL[4] - PR[4]) * g2) /
                    (PR[0] * (SR - UR) - PL[0] * (SL - UL));
  const bool left = (SL >= 0.0) || (SS >= 0.0);
  const bool star = !(SL >= 0.0) && ((SS >= 0.0) || (SR >= 0.0));
  const double r = left ? PL[0] : PR[0], u = left ? PL[1] : PR[1], v = left ? PL[2] : PR[2];
  const double w = left ? PL[3] : PR[3], p = left ? PL[4] : PR[4];
  const double UK = left ? UL : UR, SK = left ? SL : SR;
  const double E = fma(p, igm1, 0.5 * r * (u * u + v * v + w * w));
  const double ru = r * UK;
  F[0] = ru;
  F[1] = fma(ru, u, mx * p);
  F[2] = fma(ru, v, my * p);
  F[3] = fma(ru, w, mz * p);
  F[4] = fma(E + p, UK, -mt * p);
  if (star) {
    const double dS = SK - UK;
    const double fac = r * dS / (SK - SS);
    const double dU = (SS - UK) * ig2;
    const double q0 = fac;
    const double q1 = fac * fma(mx, dU, u);
    const double q2 = fac * fma(my, dU, v);
    const double q3 = fac * fma(mz, dU, w);
    const double q4 = fac * (E / r + (SS - UK) * ((SS - mt) * ig2 + p / (r * dS)));
    F[0] = fma(SK, q0 - r, F[0]);
    F[1] = fma(SK, q1 - r * u, F[1]);
    F[2] = fma(SK, q2 - r * v, F[2]);
    F[3] = fma(SK, q3 - r * w, F[3]);
    F[4] = fma(SK, q4 - E, F[4]);
  }
}

// O3 steps 1-8 for one interface (Fig. 3).  pP: field 0 of cell i-1; pP1: P' of cell i; pP2: P'' of
// cell i-1; SS = stride to the next cell along the sweep, FP/F1/F2 = field strides.  Returns the E.1 flags
// (bit r: left state of component r limited, bit 5+r: right state).
template <int SS_, int FP, int F1, int F2>
__device__ __forceinline__ unsigned inviscid_face(const Consts& c, const double* __restrict__ pP, const double* __restrict__ pP1,
                                                  const double* __restrict__ pP2, double mx, double my, double mz, double mt,
                                                  double F[5]) {
  const double g2 = fma(mx, mx, fma(my, my, mz * mz));
  const double g = sqrt(g2), ig = 1.0 / g;
  Eig e;
  e.nx = mx * ig; e.ny = my * ig; e.nz = mz * ig;
  const double rb = 0.5 * (pP[SS_] + pP[2 * SS_]);
  const double pb = 0.5 * (pP[4 * FP + SS_] + pP[4 * FP + 2 * SS_]);
  const double irb = 1.0 / rb;
  e.a2 = c.gamma * pb * irb;
  const double a = sqrt(e.a2), ia = 1.0 / a;
  e.ra = rb * a;
  const double ia2 = ia * ia, h_ira = 0.5 * irb * ia;
  double W[4][5], D1[5], D2[5], WL[5], WR[5];
#pragma unroll
  for (int cidx = 0; cidx < 4; ++cidx)
    project(e, pP[cidx * SS_], pP[FP + cidx * SS_], pP[2 * FP + cidx * SS_], pP[3 * FP + cidx * SS_],
            pP[4 * FP + cidx * SS_], W[cidx]);
  project(e, pP2[SS_], pP2[F2 + SS_], pP2[2 * F2 + SS_], pP2[3 * F2 + SS_], pP2[4 * F2 + SS_], D1);
  project(e, pP2[2 * SS_], pP2[F2 + 2 * SS_], pP2[2 * F2 + 2 * SS_], pP2[3 * F2 + 2 * SS_], pP2[4 * F2 + 2 * SS_], D2);
  {
    double G0[5], G1[5];
    project(e, pP1[0], pP1[F1], pP1[2 * F1], pP1[3 * F1], pP1[4 * F1], G0);
    project(e, pP1[SS_], pP1[F1 + SS_], pP1[2 * F1 + SS_], pP1[3 * F1 + SS_], pP1[4 * F1 + SS_], G1);
#pragma unroll
    for (int r = 0; r < 5; ++r) {   // Eq. 21-22
      WL[r] = W[1][r] + 0.5 * G0[r] + D1[r] / 12.0;
      WR[r] = W[2][r] - 0.5 * G1[r] + D2[r] / 12.0;
    }
  }
  unsigned fl = 0;
#pragma unroll
  for (int r = 0; r < 5; ++r) {
    if (mp_test(WL[r], W[1][r], W[0][r], W[2][r], c.mp_alpha)) fl |= 1u << r;
    if (mp_test(WR[r], W[2][r], W[3][r], W[1][r], c.mp_alpha)) fl |= 32u << r;
  }
  // warp-uniform early accept of test E.1: the full limiting path runs only if some lane needs it
  if (__any_sync(__activemask(), fl != 0)) {
    double D0[5], D3[5];
    project(e, pP2[0], pP2[F2], pP2[2 * F2], pP2[3 * F2], pP2[4 * F2], D0);
    project(e, pP2[3 * SS_], pP2[F2 + 3 * SS_], pP2[2 * F2 + 3 * SS_], pP2[3 * F2 + 3 * SS_], pP2[4 * F2 + 3 * SS_], D3);
#pragma unroll
    for (int r = 0; r < 5; ++r) {
      const double dmid = minmod(D1[r], D2[r]);
      WL[r] = mp_full(WL[r], W[1][r], W[0][r], W[2][r], dmid, minmod(D0[r], D1[r]), c.mp_alpha, (fl >> r) & 1u);
      WR[r] = mp_full(WR[r], W[2][r], W[3][r], W[1][r], dmid, minmod(D2[r], D3[r]), c.mp_alpha, (fl >> (r + 5)) & 1u);
    }
  }
  double PL[5], PR[5];
  backproject(e, ia2, h_ira, WL, PL);
  backproject(e, ia2, h_ira, WR, PR);
  hllc(PL, PR, mx, my, mz, mt, g, g2, ig * ig, c.gamma, F);
  return fl;
}

// O4: alpha-damping viscous flux, Eq. 29-35, subtracted from F (Res = -(F - Fv) differences).
// pP: field 0 of cell L = i; pP1: P' of cell L; getG(e, f, cell) = stored tangential gradient of field f along e
// at cell L (0) / R (1); getM(q) = hatted interface metric q (q = 9: 1/J) for the directions other than DIR.
template <int DIR, int SS_, int FP, int F1, class GetG, class GetM>
__device__ __forceinline__ void viscous_face(const Consts& c, const double* __restrict__ pP, const double* __restrict__ pP1,
                                             double mx, double my, double mz, GetG getG, GetM getM, double F[5]) {
  double val[4], gr[3][4];
#pragma unroll
  for (int f = 0; f < 4; ++f) {
    const int pf = (f < 3) ? f + 1 : 5;
    const double gL = pP1[pf * F1], gR = pP1[pf * F1 + SS_];
    const double phL = fma(0.5, gL, pP[pf * FP]);            // Eq. 30 (beta^D = 0)
    const double phR = fma(-0.5, gR, pP[pf * FP + SS_]);     // Eq. 31
#pragma unroll
    for (int e = 0; e < 3; ++e) {
      if (e == DIR) gr[e][f] = fma(2.0, phR - phL, 0.5 * (gL + gR));   // Eq. 29, alpha^D = 4
      else gr[e][f] = 0.5 * (getG(e, f, 0) + getG(e, f, 1));           // R11
    }
    val[f] = 0.5 * (phL + phR);
  }
  const double mu = sutherland(c, val[3]);
  const double lam = -2.0 / 3.0 * mu, kap = mu * c.kappa_fac;
  const double irj = 1.0 / getM(9);
  double mh[9];
#pragma unroll
  for (int q = 0; q < 9; ++q) mh[q] = (q / 3 == DIR) ? ((q % 3 == 0) ? mx : (q % 3 == 1) ? my : mz) : getM(q);
  double dx[3][4];
#pragma unroll
  for (int cc = 0; cc < 3; ++cc) {
    const double k0 = mh[cc] * irj, k1 = mh[3 + cc] * irj, k2 = mh[6 + cc] * irj;   // R12
#pragma unroll
    for (int f = 0; f < 4; ++f) dx[cc][f] = fma(k2, gr[2][f], fma(k1, gr[1][f], k0 * gr[0][f]));   // Eq. 32
  }
  const double div = dx[0][0] + dx[1][1] + dx[2][2];
  const double txx = fma(2.0 * mu, dx[0][0], lam * div), tyy = fma(2.0 * mu, dx[1][1], lam * div),
               tzz = fma(2.0 * mu, dx[2][2], lam * div);
  const double txy = mu * (dx[1][0] + dx[0][1]), txz = mu * (dx[2][0] + dx[0][2]), tyz = mu * (dx[2][1] + dx[1][2]);
  const double bx = fma(kap, dx[0][3], fma(val[2], txz, fma(val[1], txy, val[0] * txx)));
  const double by = fma(kap, dx[1][3], fma(val[2], tyz, fma(val[1], tyy, val[0] * txy)));
  const double bz = fma(kap, dx[2][3], fma(val[2], tzz, fma(val[1], tyz, val[0] * txz)));
  F[1] -= fma(mz, txz, fma(my, txy, mx * txx));
  F[2] -= fma(mz, tyz, fma(my, tyy, mx * txy));
  F[3] -= fma(mz, tzz, fma(my, tyz, mx * txz));
  F[4] -= fma(mz, bz, fma(my, by, mx * bx));
}

template <int DIR, bool VISC>
struct FluxCfg {
  static constexpr int TS = (DIR == 0) ? 32 : 15;   // cells along the sweep direction per tile
  static constexpr int TT = (DIR == 0) ? 8 : 32;    // transverse extent: rows (xi sweep) or i-lanes (eta/zeta sweep)
  static constexpr int NT = (DIR == 0) ? 288 : 256; // threads
  static constexpr int NF = VISC ? 6 : 5;           // fields staged (T only for the viscous flux)
  static constexpr int LP = TS + 12, L1 = TS + 2, L2 = TS + 4, LF = TS + 1;
  static constexpr int SMEM_DOUBLES = NF * TT * LP + NF * TT * L1 + 5 * TT * L2 + 5 * TT * LF;
};

template <int DIR, int TT>
__device__ __forceinline__ int sidx(int f, int a, int t, int LA) {
  return (DIR == 0) ? (f * TT + t) * LA + a : (f * LA + a) * TT + t;
}

struct FluxIn {
  const double* P[6];
  const double* m[10];    // interface metrics of this family: 9 hatted + 1/J (only own 3 when inviscid)
  const double* mt;       // own time metric (moving) or null
  const double* G[12];    // stored gradients (viscous)
  double* res;            // [5][N]
  unsigned long long* stats;
  int first;              // 1: res = ..., 0: res += ...
};

template <int DIR, bool VISC>
__global__ void __launch_bounds__(FluxCfg<DIR, VISC>::NT) k_flux(Consts c, FluxIn in) {
  using C = FluxCfg<DIR, VISC>;
  constexpr int TS = C::TS, TT = C::TT, NT = C::NT, NF = C::NF, LP = C::LP, L1 = C::L1, L2 = C::L2, LF = C::LF;
  constexpr int SS_ = (DIR == 0) ? 1 : TT;   // shared-memory stride along the sweep direction
  extern __shared__ double smem[];
  double* sP = smem;
  double* sP1 = sP + NF * TT * LP;
  double* sP2 = sP1 + NF * TT * L1;
  double* sF = sP2 + 5 * TT * L2;
  const int tid = threadIdx.x;
  int s0, t0, o;
  if (DIR == 0) { s0 = blockIdx.x * TS; t0 = blockIdx.y * TT; o = blockIdx.z; }
  else if (DIR == 1) { t0 = blockIdx.x * TT; s0 = blockIdx.y * TS; o = blockIdx.z; }
  else { t0 = blockIdx.x * TT; o = blockIdx.y; s0 = blockIdx.z * TS; }
  const int nd = c.n[DIR];
  const int nt = (DIR == 0) ? c.n[1] : c.n[0];

  // ---- stage the primitive tile (halo 6 along the sweep direction) ----
  for (int idx = tid; idx < NF * TT * LP; idx += NT) {
    int f, a, t;
    if (DIR == 0) { a = idx % LP; t = (idx / LP) % TT; f = idx / (LP * TT); }
    else { t = idx % TT; a = (idx / TT) % LP; f = idx / (TT * LP); }
    const int cs = min(s0 + a - 6, nd + 5);
    const int ct = min(t0 + t, nt - 1);
    long long at;
    if (DIR == 0) at = c.LP.at(cs, ct, o);
    else if (DIR == 1) at = c.LP.at(ct, cs, o);
    else at = c.LP.at(ct, o, cs);
    const int ff = (f == 5) ? 5 : f;
    sP[sidx<DIR, TT>(f, a, t, LP)] = __ldg(in.P[ff] + at);
  }
  __syncthreads();
  // ---- E6 first gradients (Eq. 17) on cells -1..TS and Eq. 19 second derivatives on cells -2..TS+1 ----
  for (int idx = tid; idx < NF * TT * L1; idx += NT) {
    int f, a, t;
    if (DIR == 0) { a = idx % L1; t = (idx / L1) % TT; f = idx / (L1 * TT); }
    else { t = idx % TT; a = (idx / TT) % L1; f = idx / (TT * L1); }
    const double* q = sP + sidx<DIR, TT>(f, a + 5, t, LP);
    double r = CE1 * (q[SS_] - q[-SS_]);
    r = fma(CE2, q[2 * SS_] - q[-2 * SS_], r);
    r = fma(CE3, q[3 * SS_] - q[-3 * SS_], r);
    sP1[sidx<DIR, TT>(f, a, t, L1)] = r;
  }
  for (int idx = tid; idx < 5 * TT * L2; idx += NT) {
    int f, a, t;
    if (DIR == 0) { a = idx % L2; t = (idx / L2) % TT; f = idx / (L2 * TT); }
    else { t = idx % TT; a = (idx / TT) % L2; f = idx / (TT * L2); }
    const double* q = sP + sidx<DIR, TT>(f, a + 4, t, LP);
    double r = CS0 * q[0];
    r = fma(CS1, q[SS_] + q[-SS_], r);
    r = fma(CS2, q[2 * SS_] + q[-2 * SS_], r);
    r = fma(CS3, q[3 * SS_] + q[-3 * SS_], r);
    r = fma(CS4, q[4 * SS_] + q[-4 * SS_], r);
    sP2[sidx<DIR, TT>(f, a, t, L2)] = r;
  }
  __syncthreads();

  // ---- one interface per work item ----
  unsigned nlim = 0, ntst = 0;
  for (int item = tid; item < TT * LF; item += NT) {
    int sI, t;
    if (DIR == 0) { sI = item % LF; t = item / LF; }
    else { t = item % TT; sI = item / TT; }
    const int fs = min(s0 + sI, nd);          // interface between cells fs-1 and fs
    const int ct = min(t0 + t, nt - 1);
    const bool valid = (s0 + sI <= nd) && (t0 + t < nt);
    long long af;
    if (DIR == 0) af = c.LF[0].at(fs, ct, o);
    else if (DIR == 1) af = c.LF[1].at(ct, fs, o);
    else af = c.LF[2].at(ct, o, fs);
    const double mx = __ldg(in.m[3 * DIR] + af), my = __ldg(in.m[3 * DIR + 1] + af), mz = __ldg(in.m[3 * DIR + 2] + af);
    const double mt = in.mt ? __ldg(in.mt + af) : 0.0;
    double F[5];
    {
      constexpr int FP = (DIR == 0) ? TT * LP : LP * TT;   // field strides
      constexpr int F1 = (DIR == 0) ? TT * L1 : L1 * TT;
      constexpr int F2 = (DIR == 0) ? TT * L2 : L2 * TT;
      const unsigned fl = inviscid_face<SS_, FP, F1, F2>(c, sP + sidx<DIR, TT>(0, sI + 4, t, LP), sP1 + sidx<DIR, TT>(0, sI, t, L1),
                                                         sP2 + sidx<DIR, TT>(0, sI, t, L2), mx, my, mz, mt, F);
      if (valid && (sI < TS || s0 + sI == nd)) { nlim += __popc(fl); ntst += 10; }   // tile-shared faces once
    }
    if (VISC) {
      constexpr int FP = (DIR == 0) ? TT * LP : LP * TT;
      constexpr int F1 = (DIR == 0) ? TT * L1 : L1 * TT;
      const int cl = fs - 1;
      long long agL, agS;
      if (DIR == 0) { agL = c.LG.at(cl, ct, o); agS = 1; }
      else if (DIR == 1) { agL = c.LG.at(ct, cl, o); agS = c.LG.sj; }
      else { agL = c.LG.at(ct, o, cl); agS = c.LG.sk; }
      auto getG = [&](int e, int f, int cell) { return __ldg(in.G[4 * e + f] + agL + cell * agS); };
      auto getM = [&](int q) { return __ldg(in.m[q] + af); };
      viscous_face<DIR, SS_, FP, F1>(c, sP + sidx<DIR, TT>(0, sI + 5, t, LP), sP1 + sidx<DIR, TT>(0, sI, t, L1),
                                     mx, my, mz, getG, getM, F);
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) sF[sidx<DIR, TT>(f, sI, t, LF)] = F[f];
  }
  if (in.stats) {
    // warp-aggregated counters (diagnostic path only)
    for (int off = 16; off > 0; off >>= 1) {
      nlim += __shfl_down_sync(0xffffffffu, nlim, off);
      ntst += __shfl_down_sync(0xffffffffu, ntst, off);
    }
    if ((tid & 31) == 0 && ntst) { atomicAdd(in.stats, (unsigned long long)nlim); atomicAdd(in.stats + 1, (unsigned long long)ntst); }
  }
  __syncthreads();
  // ---- flux difference, Eq. 25: Res_i -= F_{i+1/2} - F_{i-1/2} ----
  for (int item = tid; item < TT * TS; item += NT) {
    int s, t;
    if (DIR == 0) { s = item % TS; t = item / TS; }
    else { t = item % TT; s = item / TT; }
    if (s0 + s >= nd || t0 + t >= nt) continue;
    long long ac;
    if (DIR == 0) ac = c.LR.at(s0 + s, t0 + t, o);
    else if (DIR == 1) ac = c.LR.at(t0 + t, s0 + s, o);
    else ac = c.LR.at(t0 + t, o, s0 + s);
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      const double dF = sF[sidx<DIR, TT>(f, s + 1, t, LF)] - sF[sidx<DIR, TT>(f, s, t, LF)];
      double* rp = in.res + f * c.fsR + ac;
      *rp = in.first ? -dF : *rp - dF;
    }
  }
}

}  // namespace meg6
