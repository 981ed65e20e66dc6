// meg6_flux3.cuh -- per-direction flux kernel, third generation (sm_100a).
//
// Same method as meg6_flux.cuh (Fig. 3 P:204-262 and Fig. 5), reorganised after the first ncu pass
// (profiles/r1a_*: latency/issue bound at 14 warps per SM, 60 % of the issued instructions not FP64):
//   * the tile computes, per cell, the two one-sided reconstruction offsets of Eq. 16/21-22
//        aL = +1/2 P' + P''/12,   aR = -1/2 P' + P''/12        (P' Eq. 17, P'' Eq. 19)
//     once in shared memory; P'' of a cell is recovered as 6 (aL + aR), P' as aL - aR;
//   * the characteristic step works on DIFFERENCES (c0 - cm, cp - c0, W_unlimited - c0): every formula of
//     App. E is invariant under a shift of all its arguments, and the projection is linear (frozen matrix,
//     Eq. 20), so five projections replace eight and the limited state is P_cell + R (limited offset);
//   * reciprocals are shared (1/(a b) gives 1/a and 1/b), rsqrt replaces sqrt + divide;
//   * shared memory is addressed as shared (LDS with immediate offsets), the flux tile aliases the metric tile,
//     the running residual is read from global memory in the final phase: 5 CTAs of 4 warps per SM.
// Results differ from the step-by-step order of the oracle at round-off level only.
#pragma once
#include <cuda.h>
#include "meg6_common.cuh"

namespace meg6 {

// Build parameters of the sweeps, fixed after the measurements recorded in DESIGN.md section 6 ("tried and rejected"):
// 4 CTAs per SM (128 registers; 5 CTAs at 96-100 registers: -6 % eta/zeta, -10 % all three on C4, r2c), eta/zeta tiles
// of 15 cells x 8 xi-lanes (11, 19, 23, 31 cells and 16 lanes all slower), 5 cells per thread in the offset phase.
constexpr int SWEEP_MINB = 4, TS_Y = 15, TT_Y = 8, BLK_Y = 5, NSUB_Y = 2;

// IG4 = MIG4 variant (scheme 1): the sweep-direction gradients P' are not E6 stencils of the tile but solutions of
// the implicit systems of Eq. 18, computed beforehand for whole grid lines and loaded like the primitives.
template <int DIR, bool VISC, bool IG4 = false>
struct Cfg3 {
  static constexpr int TS = (DIR == 0) ? 30 : TS_Y;     // cells along the sweep per tile
  static constexpr int TT = (DIR == 0) ? 4 : TT_Y; // transverse positions (rows for xi, i-lanes otherwise)
  static constexpr int NI = TS + 1;                          // interfaces per pencil
  static constexpr int NT = (DIR == 0) ? 32 * TT : NI * TT;  // threads: one interface each (xi: one warp per row)
  static constexpr int MINB = SWEEP_MINB;
  static constexpr int NF = VISC ? 6 : 5;                    // staged fields (T only for the viscous flux)
  static constexpr int NM = VISC ? 10 : 3;                   // interface metrics loaded
  static constexpr int NMF = NM > 5 ? NM : 5;                // the metric region later receives the 5 fluxes
  // eta/zeta sweeps (MEG6): a CTA works through NSUB consecutive sub-tiles of TS cells along the sweep out of ONE
  // primitive window of NSUB TS + 12 cells, loaded by one TMA box at the start: the wait for the primitives (DRAM
  // latency at the head of every CTA, 15 % of the warp samples of the one-tile kernel, ncu r2c) is paid once per NSUB
  // sub-tiles, and the 12-cell halo is shared; the metric / gradient / residual boxes of sub-tile h+1 are issued when
  // sub-tile h is finished and arrive while its offsets (phase 1) are formed
  static constexpr int NSUB = (DIR != 0 && !IG4) ? NSUB_Y : 1;
  static constexpr int LP = TS + 12;                         // P of one sub-tile: cells -6 .. TS+5
  static constexpr int LPT = TS * NSUB + 12;                 // the primitive window of the CTA
  static constexpr int LA = TS + 4;                          // aL/aR: cells -2 .. TS+1
  static constexpr int LT = TS + 2;                          // T': cells -1 .. TS
  static constexpr int LF = (DIR == 0) ? TS + 2 : TS + 1;    // interface rows (xi: even length, TMA box bytes % 16)
  static constexpr int LG = (DIR == 0) ? TS + 4 : TS + 2;    // stored gradients: cells -1..TS (xi: box starts at -2)
  static constexpr int GOFF = (DIR == 0) ? 1 : 0;
  static constexpr int LQ = (DIR == 0) ? TS + 8 : TS + 6;    // IG4: P' cells -3..TS+2 (xi: box starts at -4)
  static constexpr int QOFF = (DIR == 0) ? 1 : 0;
  static constexpr int al(int n) { return (n + 15) / 16 * 16; }   // 128-byte granules (TMA destinations)
  // stored tangential gradients: two groups (the two tangential directions).  MEG6: 4 fields (u,v,w,T) each, one
  // box per group out of the 12-field array; MIG4: one 5-field box (u,v,w,p,T of the line-solve arrays) per group,
  // the second group starting on the next 128-byte boundary
  static constexpr int GFLD = IG4 ? 5 : 4, GSLOT = IG4 ? al(5 * LG * TT) : 4 * LG * TT;
  static constexpr int nP = NF * LPT * TT, nA = 10 * LA * TT, nT1 = (VISC && !IG4) ? LT * TT : 0, nM = NMF * LF * TT,
                       nMt = LF * TT, nG = VISC ? GSLOT + GFLD * LG * TT : 0, nGtx = VISC ? 2 * GFLD * LG * TT : 0,
                       nQ = IG4 ? NF * LQ * TT : 0;
  // eta/zeta sweeps, MEG6: the running residual of the tile arrives by TMA with the metrics (it is needed at the very
  // end of the CTA; as plain loads behind an L2 prefetch it cost the second sweep 0.09 ms against the first)
  static constexpr int nR = !IG4 ? 5 * TS * TT : 0;
  // fused xi sweep, MEG6: what the final phase reads besides the residual -- U (5), U^n (5), 1/J, sigma -- as four more
  // boxes on the same barrier (replaces an L2-prefetch loop of 10 % of the kernel's instructions and 12 late loads)
  static constexpr int nU = (DIR == 0 && !IG4) ? 5 * TS * TT : 0, n1 = nU ? TS * TT : 0;
  static constexpr int oP = 0, oM = oP + al(nP), oMt = oM + al(nM), oG = oMt + al(nMt), oQ = oG + al(nG), oA = oQ + al(nQ),
                       oT1 = oA + al(nA), oR = oT1 + al(nT1), oU = oR + al(nR), oU0 = oU + al(nU), oJ = oU0 + al(nU),
                       oSg = oJ + al(n1), oBar = oSg + al(n1);
  static constexpr int SMEM_BYTES = (oBar + 2) * 8;   // two mbarriers
};

template <int DIR, int TT>
__device__ __forceinline__ int sidx3(int f, int a, int t, int LA) {
  return (DIR == 0) ? (f * TT + t) * LA + a : (f * LA + a) * TT + t;
}

struct FluxIn3 {
  double* res;                  // [5] running residual, layout LR, field stride fsR
  unsigned long long* stats;    // limiter counters or null
  unsigned short* mask;         // branch record of this family's interfaces (meg6_set_branch_masks) or null
  double* gown;                 // eta sweep (MEG6, viscous): where it stores the eta gradients of (u,v,w,T) of its cells for
  long long gfs;                // the later sweeps' tangential terms (field 0, layout LG, field stride gfs), or null
  int first, moving;
};

// Residual assembly + SSP-RK3 stage + primitive conversion fused into the final phase of the LAST sweep
// (SURVEY 8(a) rows S, T and the first half of G): the complete residual of a cell is in registers there, so
//   dQ/dt = J (Res - (1/J)_t Q) - sigma (Q - Q_ref)            (Eq. 9, 12, 14; R16)
//   mode 0: out = dQ/dt                                          (meg6_rhs)
//   mode 1: out = a U0 + b (U + dt dQ/dt)  (a = 0: stage 1, which also saves U0 = U)   (Eq. B.1)
// and the primitives of the new state go to the OTHER primitive buffer (the current one is still being read by
// neighbouring tiles), ready for the ghost fill of the next stage.
struct Fuse3 {
  const double* U; const double* U0; double* U0w; double* out;
  const double* rj; const double* rjt; const double* sigma; const double* uref;
  double* Pn;                   // next primitive buffer (field 0; stride fsP) or null
  double a, b, dt;
  int mode;
  int tail_tma;                 // U, U0, 1/J, sigma of the tile come by TMA (maps valid)
};

__device__ __forceinline__ uint32_t smem_u32_3(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void tma4(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32_3(dst)), "l"((uint64_t)tm), "r"(smem_u32_3(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

__device__ __forceinline__ void mbar_wait3(uint64_t* bar, uint32_t parity = 0) {   // phase `parity` of the barrier
  uint32_t done = 0;
  const uint32_t b = smem_u32_3(bar);
  while (!done) {
    asm volatile(
        "{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done) : "r"(b), "r"(parity) : "memory");
  }
}

// shared-memory load the compiler may not merge with an earlier load of the same address: values that are needed
// again long after their first use are re-read instead of being kept in registers across the limiter
__device__ __forceinline__ double lds_again(const double* p) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(smem_u32_3(p)));
  return v;
}

// Reciprocal as its own operation: a/b is written a * rcp3(b) (the reciprocal sequence is shorter than the division
// sequence; C4: -4 % on the sweeps).  Hand-rolled MUFU-seed + Newton versions without the library's special-case
// branches were measured SLOWER in round 1 (more live registers, more spills).
__device__ __forceinline__ double rcp3(double x) { return 1.0 / x; }

// min / max of two doubles as one compare and one select.  The library fmin / fmax carry IEEE NaN handling and compile
// to DSETP + SEL + FSEL + LOP3 + three or four register moves each (sm_100a has no FP64 min/max instruction; SASS of the
// round-1 build: 8 instructions per call, 24 % of the limiting path); a NaN here means the state is lost anyway.  For
// ordered operands the result is the same value bit for bit (the limiter's own +-0 cases select equal magnitudes).
__device__ __forceinline__ double dmin3(double a, double b) { return (a < b) ? a : b; }
__device__ __forceinline__ double dmax3(double a, double b) { return (a > b) ? a : b; }
// The wave-speed bounds of HLLC are the one place where an unordered operand occurs in a run that is otherwise fine: a
// limited state that has left the physical range (negative density: the violent inflow interface of the randomised
// parity case) has a NaN sound speed.  The forms below are those of std::min / std::max -- the FIRST operand comes back
// when the second is a NaN -- which is what the step-by-step CPU restatement of the method does, so such an interface
// takes the same branch of Eq. 26 on both sides (and the left state's flux, which is finite).
__device__ __forceinline__ double hmin3(double a, double b) { return (b < a) ? b : a; }
__device__ __forceinline__ double hmax3(double a, double b) { return (a < b) ? b : a; }

__device__ __forceinline__ double minmod3(double a, double b) {   // E.2
  // same sign: the operand of smaller magnitude IS sign * min(|a|, |b|)
  const double m = (fabs(a) < fabs(b)) ? a : b;
  const bool same = ((__double2hiint(a) ^ __double2hiint(b)) >= 0);
  return same ? m : 0.0;
}

struct Eig3 { double nx, ny, nz, ra, a2; };

// W = Linv * P (A.6a; R6)
__device__ __forceinline__ void project3(const Eig3& e, double r, double u, double v, double w, double p, double W[5]) {
  const double un = fma(e.nz, w, fma(e.ny, v, e.nx * u));
  W[0] = fma(-e.ra, un, p);
  W[4] = fma(e.ra, un, p);
  const double q = fma(e.a2, r, -p);
  W[1] = fma(e.nx, q, fma(e.ny, w, -e.nz * v));
  W[2] = fma(e.nz, q, fma(e.nx, v, -e.ny * u));
  W[3] = fma(-e.ny, q, fma(e.nx, w, -e.nz * u));
}

// P = base + Rmat * W (A.4b; R6)
__device__ __forceinline__ void backproject3(const Eig3& e, double ia2, double h_ira, const double W[5], const double B[5],
                                             double P[5]) {
  const double sp = W[0] + W[4];
  P[0] = fma(ia2, fma(0.5, sp, fma(e.nx, W[1], fma(e.nz, W[2], -e.ny * W[3]))), B[0]);
  const double s = h_ira * (W[4] - W[0]);
  P[1] = B[1] + fma(e.nx, s, -fma(e.ny, W[2], e.nz * W[3]));
  P[2] = B[2] + fma(e.ny, s, fma(e.nx, W[2], -e.nz * W[1]));
  P[3] = B[3] + fma(e.nz, s, fma(e.ny, W[1], e.nx * W[3]));
  P[4] = fma(0.5, sp, B[4]);
}

// App. E (R7) in offset form (all quantities relative to c0):
//   e = W_unlimited - c0, dp = cp - c0, dm = c0 - cm; returns the limited offset.
__device__ __forceinline__ double mp_limit3(double e, double dp, double dm, double dnear, double dfar, double alpha) {
  const double wmd = 0.5 * (dp - dnear);
  const double wul = alpha * dm;
  const double wlc = fma(4.0 / 3.0, dfar, 0.5 * dm);
  const double wmin = dmax3(dmin3(dmin3(0.0, dp), wmd), dmin3(dmin3(0.0, wul), wlc));
  const double wmax = dmin3(dmax3(dmax3(0.0, dp), wmd), dmax3(dmax3(0.0, wul), wlc));
  return e + minmod3(wmin - e, wmax - e);   // E.4
}

// Contravariant HLLC, Eq. 26-27 with the flux of Eq. 2; energy row R9; cascade R10.
// Returns the branch 0..3 of Eq. 26 taken.
__device__ __forceinline__ unsigned hllc3(const double PL[5], const double PR[5], double mx, double my, double mz, double mt,
                                          double g, double g2, double ig2, double gamma, double igm1, double F[5]) {
  const double UL = fma(mz, PL[3], fma(my, PL[2], fma(mx, PL[1], mt)));
  const double UR = fma(mz, PR[3], fma(my, PR[2], fma(mx, PR[1], mt)));
  const double t = rcp3(PL[0] * PR[0]);
  const double irL = PR[0] * t, irR = PL[0] * t;
  const double cL = sqrt(gamma * PL[4] * irL) * g, cR = sqrt(gamma * PR[4] * irR) * g;
  const double SL = hmin3(UL - cL, UR - cR);
  const double SR = hmax3(UL + cL, UR + cR);
  const double mL = PL[0] * (SL - UL), mR = PR[0] * (SR - UR);
  const double SS = (fma(mR, UR, -mL * UL) + (PL[4] - PR[4]) * g2) * rcp3(mR - mL);
  const bool left = (SL >= 0.0) || (SS >= 0.0);
  const bool star = !(SL >= 0.0) && ((SS >= 0.0) || (SR >= 0.0));
  const double r = left ? PL[0] : PR[0], u = left ? PL[1] : PR[1], v = left ? PL[2] : PR[2];
  const double w = left ? PL[3] : PR[3], p = left ? PL[4] : PR[4];
  const double UK = left ? UL : UR, SK = left ? SL : SR;
  const double E = fma(p, igm1, 0.5 * r * fma(u, u, fma(v, v, w * w)));
  const double ru = r * UK;
  F[0] = ru;
  F[1] = fma(ru, u, mx * p);
  F[2] = fma(ru, v, my * p);
  F[3] = fma(ru, w, mz * p);
  F[4] = fma(E + p, UK, -mt * p);
  if (star) {
    const double dK = SK - SS, dSU = SS - UK;
    // Q*_K - Q_K without cancellation: fac - rho_K = rho_K (S* - U_K)/(S_K - S*), and
    // fac (S*-U_K) p/(rho_K (S_K-U_K)) = p (S*-U_K)/(S_K-S*)
    const double idK = rcp3(dK);
    const double k = dSU * idK;              // (S* - U_K)/(S_K - S*)
    const double rk = r * k;                 // fac - rho_K
    const double fd = (r + rk) * dSU * ig2;  // fac (S* - U_K)/g^2
    F[0] = fma(SK, rk, F[0]);
    F[1] = fma(SK, fma(rk, u, fd * mx), F[1]);
    F[2] = fma(SK, fma(rk, v, fd * my), F[2]);
    F[3] = fma(SK, fma(rk, w, fd * mz), F[3]);
    F[4] = fma(SK, fma(k, E + p, fd * (SS - mt)), F[4]);
  }
  return left ? (star ? 1u : 0u) : (star ? 2u : 3u);
}

// One interface: O3 steps 1-8 (inviscid, Fig. 3) and O4 (alpha-damping viscous flux, Fig. 5; subtracted from F).
//   pP   : field 0 (rho) of cell L-1 in the primitive tile        (cells L-1, L, R, R+1 at +0..3 SS)
//   pA   : aL field 0 of cell L-1 in the offset tile              (aR fields are 5 FA further)
//   pT1  : T' of cell L;  pG: stored tangential gradients at cell L;  pM: interface metrics (field stride FM)
// SS = stride between consecutive cells along the sweep; FP/FA/FG/FM = field strides.
// Returns the E.1 flags (bit r: left state of component r limited, bit 5+r: right state) and, in bits 10-11, the
// branch of Eq. 26 the HLLC flux took.
template <int DIR, bool VISC, int SS, int FP, int FA, int FG, int FM, int GSLOT, bool IG4>
__device__ __forceinline__ unsigned face3(const Consts& c, const double* __restrict__ pP, const double* __restrict__ pA,
                                          const double* __restrict__ pT1, const double* __restrict__ pG,
                                          const double* __restrict__ pM, double mt, double F[5]) {
  constexpr int q0 = VISC ? 3 * DIR : 0;
  const double mx = pM[q0 * FM], my = pM[(q0 + 1) * FM], mz = pM[(q0 + 2) * FM];
  const double g2 = fma(mx, mx, fma(my, my, mz * mz));
  const double ig = rsqrt(g2), g = g2 * ig, ig2 = ig * ig;
  Eig3 e;
  e.nx = mx * ig; e.ny = my * ig; e.nz = mz * ig;
  double BL[5], BR[5];   // cell values L, R
#pragma unroll
  for (int f = 0; f < 5; ++f) { BL[f] = pP[f * FP + SS]; BR[f] = pP[f * FP + 2 * SS]; }
  const double rb = 0.5 * (BL[0] + BR[0]), pb = 0.5 * (BL[4] + BR[4]);   // R5
  const double irb = rcp3(rb);
  e.a2 = c.gamma * pb * irb;
  const double ia = rsqrt(e.a2), a = e.a2 * ia;
  e.ra = rb * a;
  const double ia2 = ia * ia, h_ira = 0.5 * irb * ia;
  double Wm[5], W0[5], Wp[5], EL[5], ER[5];
  project3(e, BL[0] - pP[0], BL[1] - pP[FP], BL[2] - pP[2 * FP], BL[3] - pP[3 * FP], BL[4] - pP[4 * FP], Wm);
  project3(e, BR[0] - BL[0], BR[1] - BL[1], BR[2] - BL[2], BR[3] - BL[3], BR[4] - BL[4], W0);
  project3(e, pP[3 * SS] - BR[0], pP[FP + 3 * SS] - BR[1], pP[2 * FP + 3 * SS] - BR[2], pP[3 * FP + 3 * SS] - BR[3],
           pP[4 * FP + 3 * SS] - BR[4], Wp);
  // Eq. 21-22 as offsets from the cell value
  project3(e, pA[SS], pA[FA + SS], pA[2 * FA + SS], pA[3 * FA + SS], pA[4 * FA + SS], EL);
  project3(e, pA[5 * FA + 2 * SS], pA[6 * FA + 2 * SS], pA[7 * FA + 2 * SS], pA[8 * FA + 2 * SS], pA[9 * FA + 2 * SS], ER);
  unsigned fl = 0;
#pragma unroll
  for (int r = 0; r < 5; ++r) {   // E.1: (W - c0)(W - W^MP) <= 1e-20 accepts
    const double mmL = minmod3(W0[r], c.mp_alpha * Wm[r]);
    const double mmR = minmod3(W0[r], c.mp_alpha * Wp[r]);
    if (!(EL[r] * (EL[r] - mmL) <= 1e-20)) fl |= 1u << r;
    if (!(ER[r] * (ER[r] + mmR) <= 1e-20)) fl |= 32u << r;
  }
  // warp-uniform early accept: the full limiting path runs only if some lane needs it
  if (__any_sync(__activemask(), fl != 0)) {
    double Dm[5], DL[5], DR[5], Dp[5];   // projected P'' of cells L-1, L, R, R+1;  P'' = 6 (aL + aR)
#define MEG6_D2(cell, f) (6.0 * (pA[(f) * FA + (cell) * SS] + pA[((f) + 5) * FA + (cell) * SS]))
    project3(e, MEG6_D2(0, 0), MEG6_D2(0, 1), MEG6_D2(0, 2), MEG6_D2(0, 3), MEG6_D2(0, 4), Dm);
    project3(e, MEG6_D2(1, 0), MEG6_D2(1, 1), MEG6_D2(1, 2), MEG6_D2(1, 3), MEG6_D2(1, 4), DL);
    project3(e, MEG6_D2(2, 0), MEG6_D2(2, 1), MEG6_D2(2, 2), MEG6_D2(2, 3), MEG6_D2(2, 4), DR);
    project3(e, MEG6_D2(3, 0), MEG6_D2(3, 1), MEG6_D2(3, 2), MEG6_D2(3, 3), MEG6_D2(3, 4), Dp);
#undef MEG6_D2
    // component by component, side by side: evaluated only where some lane of the warp failed E.1 there (failures
    // cluster at extrema of one characteristic field, so most of the ten evaluations are skipped in smooth flow)
    const unsigned wfl = __reduce_or_sync(__activemask(), fl);
#pragma unroll
    for (int r = 0; r < 5; ++r) {
      if ((wfl >> r) & 33u) {
        const double dnear = minmod3(DL[r], DR[r]);
        if ((wfl >> r) & 1u) {
          const double lL = mp_limit3(EL[r], W0[r], Wm[r], dnear, minmod3(Dm[r], DL[r]), c.mp_alpha);
          EL[r] = ((fl >> r) & 1u) ? lL : EL[r];
        }
        if ((wfl >> r) & 32u) {
          const double lR = mp_limit3(ER[r], -W0[r], -Wp[r], dnear, minmod3(DR[r], Dp[r]), c.mp_alpha);
          ER[r] = ((fl >> (r + 5)) & 1u) ? lR : ER[r];
        }
      }
    }
  }
  double PL[5], PR[5];
#pragma unroll
  for (int f = 0; f < 5; ++f) { BL[f] = lds_again(pP + f * FP + SS); BR[f] = lds_again(pP + f * FP + 2 * SS); }
  backproject3(e, ia2, h_ira, EL, BL, PL);   // Eq. 23
  backproject3(e, ia2, h_ira, ER, BR, PR);
  fl |= hllc3(PL, PR, mx, my, mz, mt, g, g2, ig2, c.gamma, c.igm1, F) << 10;

  if (VISC) {
    // O4: Eq. 29-35.  fields (u,v,w,T); normal gradient with alpha^D = 4, beta^D = 0.
    double val[4], gr[3][4];
#pragma unroll
    for (int f = 0; f < 4; ++f) {
      double cL, cR, gL, gR;
      if (f < 3) {
        cL = lds_again(pP + (f + 1) * FP + SS); cR = lds_again(pP + (f + 1) * FP + 2 * SS);
        gL = pA[(f + 1) * FA + SS] - pA[(f + 6) * FA + SS];           // P' = aL - aR
        gR = pA[(f + 1) * FA + 2 * SS] - pA[(f + 6) * FA + 2 * SS];
      } else {
        cL = pP[5 * FP + SS]; cR = pP[5 * FP + 2 * SS];
        gL = pT1[0]; gR = pT1[SS];
      }
      const double phL = fma(0.5, gL, cL);            // Eq. 30
      const double phR = fma(-0.5, gR, cR);           // Eq. 31
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        if (d == DIR) gr[d][f] = fma(2.0, phR - phL, 0.5 * (gL + gR));   // Eq. 29
        else {
          const int slot = (DIR == 0) ? d - 1 : (DIR == 1) ? (d == 0 ? 0 : 1) : d;   // tangential directions in order
          const int gf = slot * GSLOT + ((IG4 && f == 3) ? 4 : f) * FG;   // MIG4 group: (u,v,w,p,T)
          gr[d][f] = 0.5 * (pG[gf] + pG[gf + SS]);   // R11
        }
      }
      val[f] = 0.5 * (phL + phR);
    }
    // Sutherland (R15) and 1/(1/J) with one division
    const double rjh = pM[9 * FM];
    double mu, irj;
    if (c.s_suth < 0.0) { mu = c.mu_ref; irj = rcp3(rjh); }
    else {
      const double ts = val[3] + c.s_suth;
      const double t = rcp3(rjh * ts);
      irj = ts * t;
      mu = c.suth_c * val[3] * sqrt(val[3]) * (rjh * t);
    }
    const double lam = -2.0 / 3.0 * mu, kap = mu * c.kappa_fac;
    double dx[3][4];
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) {
      double k[3];
#pragma unroll
      for (int d = 0; d < 3; ++d) k[d] = ((d == DIR) ? ((cc == 0) ? mx : (cc == 1) ? my : mz) : pM[(3 * d + cc) * FM]) * irj;   // R12
#pragma unroll
      for (int f = 0; f < 4; ++f) dx[cc][f] = fma(k[2], gr[2][f], fma(k[1], gr[1][f], k[0] * gr[0][f]));   // Eq. 32
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
  return fl;
}

template <int DIR, bool VISC, bool FUSE, bool IG4 = false>
__global__ void __launch_bounds__(Cfg3<DIR, VISC, IG4>::NT, Cfg3<DIR, VISC, IG4>::MINB)
k_flux3(const Consts c, const FluxIn3 in, const __grid_constant__ TmaMaps tm, const Fuse3 fu) {
  using C = Cfg3<DIR, VISC, IG4>;
  constexpr int LQ = C::LQ;
  constexpr int TS = C::TS, TT = C::TT, NT = C::NT, NF = C::NF, LP = C::LP, LA = C::LA, LT = C::LT, LF = C::LF, LG = C::LG;
  constexpr int NSUB = C::NSUB, LPT = C::LPT;          // sub-tiles per CTA, length of the primitive window
  constexpr int SS = (DIR == 0) ? 1 : TT;
  constexpr int FP = (DIR == 0) ? TT * LPT : LPT * TT;   // field strides
  constexpr int FA = (DIR == 0) ? TT * LA : LA * TT;
  constexpr int FM = (DIR == 0) ? TT * LF : LF * TT;
  constexpr int FG = (DIR == 0) ? TT * LG : LG * TT;
  extern __shared__ __align__(1024) double sm3[];
  double* const sP = sm3 + C::oP;
  double* const sM = sm3 + C::oM;
  double* const sMt = sm3 + C::oMt;
  double* const sG = sm3 + C::oG;
  double* const sA = sm3 + C::oA;
  double* const sQ = sm3 + C::oQ;   // IG4: P' of the sweep direction
  double* const sT1 = sm3 + C::oT1;
  uint64_t* const bar = (uint64_t*)(sm3 + C::oBar);
  const int tid = threadIdx.x;
  int s0, t0, o;
  if (DIR == 0) { s0 = blockIdx.x * TS; t0 = blockIdx.y * TT; o = blockIdx.z; }
  else if (DIR == 1) { t0 = blockIdx.x * TT; s0 = blockIdx.y * (TS * NSUB); o = blockIdx.z; }
  else { t0 = blockIdx.x * TT; s0 = blockIdx.y * (TS * NSUB); o = blockIdx.z; }   // chunks of a line run back to back (halo re-use in L2)
  const int nd = c.n[DIR];
  const int nt = (DIR == 0) ? c.n[1] : c.n[0];

  // box coordinates are (i, j, k, field) in the padded layout of each array: sweep start, transverse start, other
  auto coords = [](int s, int t, int oo, int gi, int gj, int gk, int& c0, int& c1, int& c2) {
    if (DIR == 0) { c0 = s + gi; c1 = t + gj; c2 = oo + gk; }
    else if (DIR == 1) { c0 = t + gi; c1 = s + gj; c2 = oo + gk; }
    else { c0 = t + gi; c1 = oo + gj; c2 = s + gk; }
  };
  // what a sub-tile starting at cell s needs besides the primitives, on the second barrier (thread 0 only)
  auto issue_tile = [&](int s) {
    uint32_t bytes1 = (C::NM * LF * TT + C::nGtx) * 8;
    if (in.moving) bytes1 += C::nMt * 8;
    if (C::nR && !in.first) bytes1 += C::nR * 8;
    const bool ttma = C::nU && FUSE && fu.tail_tma;
    if (ttma) bytes1 += (C::nU + C::n1 + ((fu.mode == 1 && fu.a != 0.0) ? C::nU : 0) + (fu.sigma ? C::n1 : 0)) * 8;
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32_3(bar + 1)), "r"(bytes1) : "memory");
    constexpr int G0 = (DIR == 0) ? 4 : 0, G1 = (DIR == 2) ? 4 : 8;      // the two tangential gradient groups
    constexpr int GS = (DIR == 0) ? -2 : -1;                             // first stored-gradient cell of the box
    int c0, c1, c2;
    coords(s, t0, o, 0, 0, 0, c0, c1, c2);
    tma4(sM, &tm.M, bar + 1, c0, c1, c2, 0);
    if (in.moving) tma4(sMt, &tm.Mt, bar + 1, c0, c1, c2, 0);
    if (C::nR && !in.first) tma4(sm3 + C::oR, &tm.R, bar + 1, c0, c1, c2, 0);   // LR has no ghosts: same coordinates
    if (ttma) {
      tma4(sm3 + C::oU, &tm.U, bar + 1, c0, c1, c2, 0);
      if (fu.mode == 1 && fu.a != 0.0) tma4(sm3 + C::oU0, &tm.U0, bar + 1, c0, c1, c2, 0);
      if (fu.sigma) tma4(sm3 + C::oSg, &tm.Sg, bar + 1, c0, c1, c2, 0);
      tma4(sm3 + C::oJ, &tm.J, bar + 1, c0 + GX, c1 + GX, c2 + GX, 0);
    }
    if (VISC) {
      coords(s + GS, t0, o, GGI, GGJ, GGK, c0, c1, c2);
      if (!IG4) {
        tma4(sG, &tm.G, bar + 1, c0, c1, c2, G0);
        tma4(sG + 4 * FG, &tm.G, bar + 1, c0, c1, c2, G1);
      } else {
        // tangential gradients = the implicit gradients of the two other directions (fields u,v,w and T of each)
        coords(s + GS, t0, o, GPI, GPJ, GPK, c0, c1, c2);
        tma4(sG, &tm.G3[0], bar + 1, c0, c1, c2, 1);
        tma4(sG + C::GSLOT, &tm.G3[1], bar + 1, c0, c1, c2, 1);
      }
    }
  };
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32_3(bar)), "r"(1) : "memory");
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32_3(bar + 1)), "r"(1) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32_3(bar)), "r"((C::nP + C::nQ) * 8) : "memory");
    int c0, c1, c2;
    coords(s0 - 6, t0, o, GPI, GPJ, GPK, c0, c1, c2);
    tma4(sP, &tm.P, bar, c0, c1, c2, 0);   // the whole primitive window of the CTA
    if (IG4) {
      coords(s0 - 3 - C::QOFF, t0, o, GPI, GPJ, GPK, c0, c1, c2);
      tma4(sQ, &tm.Q, bar, c0, c1, c2, 0);
    }
    issue_tile(s0);
  }
  if ((FUSE && !(C::nU && fu.tail_tma)) || (!FUSE && !in.first && !C::nR)) {
    // L2 prefetch of what the final phase will read from global memory (running residual; fused: U, U0, 1/J,
    // sponge): those loads sit at the tail of the CTA with nothing to overlap them
    constexpr int NROW = (DIR == 0) ? TT : TS;                  // tile rows that are contiguous in memory
    constexpr int SEG = (DIR == 0) ? (TS + 15) / 16 + 1 : 1;    // 128-byte lines per row
    constexpr int NARR = FUSE ? 22 : 5;
    const long long N = c.LC.n;
    for (int it = tid; it < NARR * NROW * SEG; it += NT) {
      const int arr = it / (NROW * SEG), rr = (it / SEG) % NROW, sg = it % SEG;
      int ci, cj, ck;
      if (DIR == 0) { ci = s0 + sg * 16; cj = t0 + rr; ck = o; if (sg * 16 >= TS + 15) continue; }
      else if (DIR == 1) { ci = t0; cj = s0 + rr; ck = o; }
      else { ci = t0; cj = o; ck = s0 + rr; }
      if (ci >= c.n[0] || cj >= c.n[1] || ck >= c.n[2]) continue;
      const double* ptr = nullptr;
      if (arr < 5) ptr = (in.first || C::nR) ? nullptr : in.res + arr * c.fsR + c.LR.at(ci, cj, ck);
      else {
        const long long ic = c.LC.at(ci, cj, ck);
        if (arr < 10) ptr = fu.U + (arr - 5) * N + ic;
        else if (arr < 15) ptr = (fu.mode == 1 && fu.a != 0.0) ? fu.U0 + (arr - 10) * N + ic : nullptr;
        else if (arr < 20) ptr = fu.sigma ? fu.uref + (arr - 15) * N + ic : nullptr;
        else if (arr == 20) ptr = fu.sigma ? fu.sigma + ic : nullptr;
        else ptr = fu.rj + c.LX.at(ci, cj, ck);
      }
      if (ptr) asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr));
    }
  }
  __syncthreads();   // the barriers are initialised before anyone polls them
  mbar_wait3(bar);   // primitive window
  int s0h = s0;                 // first cell of the current sub-tile
  const double* sPh = sP;       // its cell -6 in the primitive window

  // ---- per cell: aL = 1/2 P' + P''/12, aR = -1/2 P' + P''/12 (Eq. 16-17, 19) on cells -2..TS+1; T' on -1..TS ----
  // One (cell, lane) position per thread and pass, all five fields; the positions left over after the full
  // passes are spread over the threads as (position, field) items so that no warp runs an extra pass alone.
  auto cell_field = [&](int f, int a, int t) {
    const double* q = sPh + sidx3<DIR, TT>(f, a + 4, t, LPT);
    const double c0 = q[0], p1 = q[SS], m1 = q[-SS], p2 = q[2 * SS], m2 = q[-2 * SS], p3 = q[3 * SS], m3 = q[-3 * SS],
                 p4 = q[4 * SS], m4 = q[-4 * SS];
    double d1 = CE1 * (p1 - m1);
    d1 = fma(CE2, p2 - m2, d1);
    d1 = fma(CE3, p3 - m3, d1);
    double d2 = CS0 * c0;
    d2 = fma(CS1, p1 + m1, d2);
    d2 = fma(CS2, p2 + m2, d2);
    d2 = fma(CS3, p3 + m3, d2);
    d2 = fma(CS4, p4 + m4, d2);
    const double h = 0.5 * d1, d = d2 * (1.0 / 12.0);
    sA[sidx3<DIR, TT>(f, a, t, LA)] = d + h;
    sA[sidx3<DIR, TT>(f + 5, a, t, LA)] = d - h;
  };
  // MIG4: P' comes from the line solves; P'' by Eq. 19 from P and P'
  auto cell_field_ig4 = [&](int f, int a, int t) {
    const double* q = sPh + sidx3<DIR, TT>(f, a + 4, t, LPT);
    const double* g1 = sQ + sidx3<DIR, TT>(f, a + 1 + C::QOFF, t, LQ);
    const double d2 = 2.0 * (q[SS] - 2.0 * q[0] + q[-SS]) - 0.5 * (g1[SS] - g1[-SS]);
    const double h = 0.5 * g1[0], d = d2 * (1.0 / 12.0);
    sA[sidx3<DIR, TT>(f, a, t, LA)] = d + h;
    sA[sidx3<DIR, TT>(f + 5, a, t, LA)] = d - h;
  };
  // ---- the sub-tiles of the CTA, one after the other (NSUB = 1: the body below runs once) ----
#pragma unroll 1
  for (int h = 0; h < NSUB; ++h) {
    if (h > 0) {
      s0h = s0 + h * TS;
      if (s0h >= nd) break;                 // ragged end of the line (uniform over the CTA)
      sPh = sP + h * TS * SS;
      __syncthreads();                      // every thread is through the final phase of the previous sub-tile
      if (tid == 0) {
        // the metric / gradient / residual buffers were read and written through the generic proxy: order those
        // accesses before the asynchronous-proxy writes of the new boxes
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        issue_tile(s0h);
      }
    }
    if (IG4) {
      if (DIR == 0) {
        const int t = tid >> 5, lane = tid & 31;
#pragma unroll
        for (int f = 0; f < 5; ++f) cell_field_ig4(f, lane, t);
        for (int it = lane; it < (LA - 32) * 5; it += 32) cell_field_ig4(it / (LA - 32), 32 + it % (LA - 32), t);
      } else {
        for (int it = tid; it < 5 * LA * TT; it += NT) cell_field_ig4(it / (LA * TT), (it / TT) % LA, it % TT);
      }
    } else if (DIR != 0) {
      // eta/zeta sweeps: the sweep index is the slow one in shared memory, so one thread takes BLK consecutive cells
      // of one lane and field: BLK + 8 loads instead of 9 BLK (shared-memory bandwidth was at 55-60 % of peak, r1c)
      constexpr int BLK = BLK_Y, NQ = (LA + BLK - 1) / BLK;
      for (int it = tid; it < NQ * TT * 5; it += NT) {
        const int t = it % TT, qd = (it / TT) % NQ, f = it / (TT * NQ);
        const int a0 = qd * BLK;
        const double* q = sPh + sidx3<DIR, TT>(f, a0, t, LPT);
        double v[BLK + 8];
#pragma unroll
        for (int m = 0; m < BLK + 8; ++m) v[m] = (a0 + m < LP) ? q[m * SS] : 0.0;
#pragma unroll
        for (int b = 0; b < BLK; ++b) {
          if (a0 + b < LA) {
            const double* w = v + b + 4;
            double d1 = CE1 * (w[1] - w[-1]);
            d1 = fma(CE2, w[2] - w[-2], d1);
            d1 = fma(CE3, w[3] - w[-3], d1);
            double d2 = CS0 * w[0];
            d2 = fma(CS1, w[1] + w[-1], d2);
            d2 = fma(CS2, w[2] + w[-2], d2);
            d2 = fma(CS3, w[3] + w[-3], d2);
            d2 = fma(CS4, w[4] + w[-4], d2);
            const double h = 0.5 * d1, d = d2 * (1.0 / 12.0);
            sA[sidx3<DIR, TT>(f, a0 + b, t, LA)] = d + h;
            sA[sidx3<DIR, TT>(f + 5, a0 + b, t, LA)] = d - h;
          }
        }
      }
    } else {
      // xi sweep: one warp per row, and a row needs nothing from the other rows: the warp fills the offsets of its own
      // row and carries on without a CTA-wide barrier (the warps of a CTA drift apart and overlap each other's tails)
      const int t = tid >> 5, lane = tid & 31;
      for (int a = lane; a < LA; a += 32) {
        if (a < 32) {
#pragma unroll
          for (int f = 0; f < 5; ++f) cell_field(f, a, t);
        }
      }
      for (int it = lane; it < (LA - 32) * 5; it += 32) cell_field(it / (LA - 32), 32 + it % (LA - 32), t);
    }
    if (VISC && !IG4) {
      // T' on cells -1..TS.  xi: lane = cell of the warp's own row; eta/zeta: reversed so that the leftover items go to
      // the last warp
      for (int it = (DIR == 0) ? (tid & 31) : NT - 1 - tid; it < ((DIR == 0) ? LT : LT * TT); it += (DIR == 0) ? 32 : NT) {
        int a, t;
        if (DIR == 0) { a = it; t = tid >> 5; }
        else { t = it % TT; a = it / TT; }
        const double* q = sPh + sidx3<DIR, TT>(5, a + 5, t, LPT);
        double d1 = CE1 * (q[SS] - q[-SS]);
        d1 = fma(CE2, q[2 * SS] - q[-2 * SS], d1);
        d1 = fma(CE3, q[3 * SS] - q[-3 * SS], d1);
        sT1[sidx3<DIR, TT>(0, a, t, LT)] = d1;
      }
    }
    if (DIR == 0) __syncwarp(); else __syncthreads();
    mbar_wait3(bar + 1, (uint32_t)(h & 1));   // interface metrics and stored gradients (issued together with the primitive tile)

    // ---- one interface per thread ----
    int sI, row;
    if (DIR == 0) { sI = tid & 31; row = tid >> 5; }
    else { row = tid % TT; sI = tid / TT; }
    const bool valid = (sI <= TS) && (s0h + sI <= nd) && (t0 + row < nt);
    unsigned nlim = 0, ntst = 0;
    double F[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    if (valid) {
      const double mt = in.moving ? sMt[sidx3<DIR, TT>(0, sI, row, LF)] : 0.0;
      const unsigned fl = face3<DIR, VISC, SS, FP, FA, FG, FM, C::GSLOT, IG4>(
          c, sPh + sidx3<DIR, TT>(0, sI + 4, row, LPT), sA + sidx3<DIR, TT>(0, sI, row, LA),
          IG4 ? sQ + sidx3<DIR, TT>(5, sI + 2 + C::QOFF, row, LQ) : sT1 + sidx3<DIR, TT>(0, sI, row, LT),
          sG + sidx3<DIR, TT>(0, sI + C::GOFF, row, LG),
          sM + sidx3<DIR, TT>(0, sI, row, LF), mt, F);
      if (sI < TS || s0h + sI == nd) {   // tile-shared faces counted once
        nlim = __popc(fl & 1023u); ntst = 10;
        if (in.mask) {   // interface (s0h + sI) of n_d + 1 along the sweep, interior extents along the others, i fastest
          long long im;
          if (DIR == 0) im = ((long long)o * c.n[1] + (t0 + row)) * (c.n[0] + 1) + (s0h + sI);
          else if (DIR == 1) im = ((long long)o * (c.n[1] + 1) + (s0h + sI)) * c.n[0] + (t0 + row);
          else im = ((long long)(s0h + sI) * c.n[1] + o) * c.n[0] + (t0 + row);
          in.mask[im] = (unsigned short)fl;
        }
      }
    }
    if (DIR != 0 && sI <= TS) {
      // the flux tile aliases the metric tile: slot (sI,row) of every metric field is read only by this thread
#pragma unroll
      for (int f = 0; f < 5; ++f) sM[sidx3<DIR, TT>(f, sI, row, LF)] = F[f];
    }
    if (in.stats) {
      for (int off = 16; off > 0; off >>= 1) {
        nlim += __shfl_down_sync(0xffffffffu, nlim, off);
        ntst += __shfl_down_sync(0xffffffffu, ntst, off);
      }
      if ((tid & 31) == 0 && ntst) { atomicAdd(in.stats, (unsigned long long)nlim); atomicAdd(in.stats + 1, (unsigned long long)ntst); }
    }
    // ---- flux difference, Eq. 25: Res_i -= F_{i+1/2} - F_{i-1/2}, then (last sweep) assembly + update ----
    auto finish_cell = [&](int s, int t, const double dF[5]) {
      long long ac;
      if (DIR == 0) ac = c.LR.at(s0h + s, t0 + t, o);
      else if (DIR == 1) ac = c.LR.at(t0 + t, s0h + s, o);
      else ac = c.LR.at(t0 + t, o, s0h + s);
      double old[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
      if (!in.first) {
#pragma unroll
        for (int f = 0; f < 5; ++f) old[f] = C::nR ? (sm3 + C::oR)[sidx3<DIR, TT>(f, s, t, TS)] : in.res[f * c.fsR + ac];
      }
      double R[5];
#pragma unroll
      for (int f = 0; f < 5; ++f) R[f] = old[f] - dF[f];
      if (!FUSE) {
#pragma unroll
        for (int f = 0; f < 5; ++f) in.res[f * c.fsR + ac] = R[f];
        if (DIR == 1 && VISC && !IG4 && in.gown) {
          // The E6 gradients along eta of (u, v, w, T) at this cell exist in the tile (P' = aL - aR, T'): they are the
          // TANGENTIAL gradients of the zeta and xi sweeps that follow in this stage, so the stored-gradient kernel
          // forms them only in the ghost columns no eta tile covers (gradients are shared, not recomputed)
          const long long ag = c.LG.at(t0 + t, s0h + s, o);
#pragma unroll
          for (int f = 0; f < 3; ++f)
            in.gown[f * in.gfs + ag] = sA[sidx3<DIR, TT>(f + 1, s + 2, t, LA)] - sA[sidx3<DIR, TT>(f + 6, s + 2, t, LA)];
          in.gown[3 * in.gfs + ag] = sT1[sidx3<DIR, TT>(0, s + 1, t, LT)];
        }
      } else {
        int ci, cj, ck;
        if (DIR == 0) { ci = s0h + s; cj = t0 + t; ck = o; }
        else if (DIR == 1) { ci = t0 + t; cj = s0h + s; ck = o; }
        else { ci = t0 + t; cj = o; ck = s0h + s; }
        const long long N = c.LC.n, ic = c.LC.at(ci, cj, ck);
        // every load of the phase before its first store: U, U0w and out may be the same memory as far as the compiler
        // knows, so a store between two loads would chain their latencies one after the other
        const bool tt = C::nU && fu.tail_tma;          // DIR == 0 here: the tile row t, cell s
        const int st = (C::nU ? t * TS + s : 0);
        const double rjv = tt ? (sm3 + C::oJ)[st] : fu.rj[c.LX.at(ci, cj, ck)];
        const double rjt = fu.rjt ? fu.rjt[ic] : 0.0;
        const double sg = fu.sigma ? (tt ? (sm3 + C::oSg)[st] : fu.sigma[ic]) : 0.0;
        const bool blend = fu.mode == 1 && fu.a != 0.0;
        double uu[5], ur[5], u0[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) uu[f] = tt ? (sm3 + C::oU)[f * TT * TS + st] : fu.U[f * N + ic];
#pragma unroll
        for (int f = 0; f < 5; ++f) u0[f] = blend ? (tt ? (sm3 + C::oU0)[f * TT * TS + st] : fu.U0[f * N + ic]) : 0.0;
#pragma unroll
        for (int f = 0; f < 5; ++f) ur[f] = (sg != 0.0) ? fu.uref[f * N + ic] : 0.0;   // sigma = 0 outside the sponge: Q_ref is not read there
        const double J = 1.0 / rjv;
        double Q[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) {
          const double u = uu[f];
          double L = J * (R[f] - rjt * u);
          if (sg != 0.0) L -= sg * (u - ur[f]);
          if (fu.mode == 0) Q[f] = L;
          else {
            double v = u + fu.dt * L;
            if (fu.a != 0.0) v = fu.a * u0[f] + fu.b * v;
            Q[f] = v;
          }
        }
        if (fu.mode == 1 && fu.a == 0.0 && fu.U0w) {
#pragma unroll
          for (int f = 0; f < 5; ++f) fu.U0w[f * N + ic] = uu[f];
        }
#pragma unroll
        for (int f = 0; f < 5; ++f) fu.out[f * N + ic] = Q[f];
        if (fu.Pn) {   // Q -> P of the new state (Eq. 5, P:83 inverted; T = p/(rho R)), as k_prim
          const double r = Q[0], ir = 1.0 / r;
          const double u = Q[1] * ir, v = Q[2] * ir, w = Q[3] * ir;
          const double p = (c.gamma - 1.0) * (Q[4] - 0.5 * r * (u * u + v * v + w * w));
          double* pn = fu.Pn + c.LP.at(ci, cj, ck);
          pn[0] = r; pn[c.fsP] = u; pn[2 * c.fsP] = v; pn[3 * c.fsP] = w; pn[4 * c.fsP] = p;
          pn[5 * c.fsP] = p / (r * c.r_gas);
        }
      }
    };
    if (DIR == 0) {
      // the right-hand interface of cell `lane` belongs to the next lane of the same warp: no shared memory, no barrier
      double dF[5];
#pragma unroll
      for (int f = 0; f < 5; ++f) dF[f] = __shfl_down_sync(0xffffffffu, F[f], 1) - F[f];
      if (sI < TS && s0h + sI < nd && t0 + row < nt) finish_cell(sI, row, dF);
    } else {
      __syncthreads();
      for (int it = tid; it < TS * TT; it += NT) {
        const int t = it % TT, s = it / TT;
        if (s0h + s >= nd || t0 + t >= nt) continue;
        double dF[5];
#pragma unroll
        for (int f = 0; f < 5; ++f) dF[f] = sM[sidx3<DIR, TT>(f, s + 1, t, LF)] - sM[sidx3<DIR, TT>(f, s, t, LF)];
        finish_cell(s, t, dF);
      }
    }
  }
}

}  // namespace meg6
