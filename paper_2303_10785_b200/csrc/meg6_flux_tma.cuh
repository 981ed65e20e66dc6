// meg6_flux_tma.cuh -- per-direction flux kernel with TMA staging (sm_100a).
//
// One CTA owns a tile of TS cells along the sweep direction times TT transverse positions.  A single elected
// thread issues 4-D tensor copies (cp.async.bulk.tensor, UTMALDG in SASS) that land the primitive pencil tile
// with its 6-cell halo (all fields in one box), the interface metrics, the stored tangential gradients and the
// running residual in shared memory; completion is signalled on one mbarrier.  Out-of-range box elements are
// zero-filled by the hardware, so ragged tiles need no index clamping.  The arithmetic is that of
// meg6_flux.cuh (inviscid_face / viscous_face).
#pragma once
#include <cuda.h>
#include "meg6_flux.cuh"

namespace meg6 {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE;\n"
      "bra WAIT_LOOP;\n"
      "DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"((uint64_t)tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}

// Tile shape (tunable at build time).  Several small CTAs per SM: while one waits on its TMA boxes the others compute.
#ifndef MEG6_TT_X
#define MEG6_TT_X 4     // xi sweep: rows (j) per tile
#endif
#ifndef MEG6_TT_Y
#define MEG6_TT_Y 8     // eta/zeta sweep: i-lanes per tile
#endif
#ifndef MEG6_MINB_X
#define MEG6_MINB_X 3
#endif
#ifndef MEG6_MINB_Y
#define MEG6_MINB_Y 4
#endif

template <int DIR, bool VISC>
struct TmaCfg {
  static constexpr int TS = (DIR == 0) ? 32 : 15;
  static constexpr int TT = (DIR == 0) ? MEG6_TT_X : MEG6_TT_Y;
  static constexpr int NT = (DIR == 0) ? 36 * MEG6_TT_X : 16 * MEG6_TT_Y;
  static constexpr int MINB = (DIR == 0) ? MEG6_MINB_X : MEG6_MINB_Y;
  static constexpr int NF = VISC ? 6 : 5;
  static constexpr int NM = VISC ? 10 : 3;
  static constexpr int LP = TS + 12, L1 = TS + 2, L2 = TS + 4;
  // interface rows: TS+1; for the xi sweep the box row is widened to an even length (inner box bytes % 16 == 0)
  static constexpr int LF = (DIR == 0) ? TS + 2 : TS + 1;
  // stored-gradient rows: cells -1..TS; the xi-sweep box starts one cell earlier so that the box origin stays
  // 16-byte aligned in global memory (an 8-byte-aligned origin faults with an illegal-instruction error)
  static constexpr int LG = (DIR == 0) ? TS + 4 : TS + 2;
  static constexpr int GOFF = (DIR == 0) ? 1 : 0;
  static constexpr int nP = NF * LP * TT, nM = NM * LF * TT, nMt = LF * TT, nG = VISC ? 8 * LG * TT : 0,
                       nR = 5 * TS * TT, nP1 = NF * L1 * TT, nP2 = 5 * L2 * TT, nF = 5 * LF * TT;
  static constexpr int al(int n) { return (n + 15) / 16 * 16; }   // 128-byte granules
  static constexpr int oP = 0, oM = oP + al(nP), oMt = oM + al(nM), oG = oMt + al(nMt), oR = oG + al(nG),
                       oP1 = oR + al(nR), oP2 = oP1 + al(nP1), oF = oP2 + al(nP2), oBar = oF + al(nF);
  static constexpr int SMEM_BYTES = (oBar + 16) * 8 + 128;   // + slack for the 128-byte alignment of the base
};

struct FluxIn2 {
  double* res;
  unsigned long long* stats;
  int first, moving, dbg;
};

template <int DIR, bool VISC>
__global__ void __launch_bounds__(TmaCfg<DIR, VISC>::NT, TmaCfg<DIR, VISC>::MINB) k_flux_tma(const Consts c, const FluxIn2 in,
                                                                    const __grid_constant__ TmaMaps tm) {
  using C = TmaCfg<DIR, VISC>;
  constexpr int TS = C::TS, TT = C::TT, NF = C::NF, NM = C::NM, LP = C::LP, L1 = C::L1, L2 = C::L2, LF = C::LF,
                LG = C::LG;
  constexpr int SS_ = (DIR == 0) ? 1 : TT;
  extern __shared__ unsigned char smem_raw[];
  double* sm = (double*)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
  double* sP = sm + C::oP; double* sM = sm + C::oM; double* sMt = sm + C::oMt; double* sG = sm + C::oG;
  double* sR = sm + C::oR; double* sP1 = sm + C::oP1; double* sP2 = sm + C::oP2; double* sF = sm + C::oF;
  uint64_t* bar = (uint64_t*)(sm + C::oBar);
  const int tid = threadIdx.x;
  int s0, t0, o;
  if (DIR == 0) { s0 = blockIdx.x * TS; t0 = blockIdx.y * TT; o = blockIdx.z; }
  else if (DIR == 1) { t0 = blockIdx.x * TT; s0 = blockIdx.y * TS; o = blockIdx.z; }
  else { t0 = blockIdx.x * TT; o = blockIdx.y; s0 = blockIdx.z * TS; }
  const int nd = c.n[DIR];
  const int nt = (DIR == 0) ? c.n[1] : c.n[0];

  if (tid == 0) {
    mbar_init(bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (tid == 0) {
    uint32_t bytes = (C::nP + C::nM) * 8;
    if (!(in.dbg & 1)) bytes += C::nG * 8;
    if (in.moving) bytes += C::nMt * 8;
    if (!in.first) bytes += C::nR * 8;
    mbar_expect_tx(bar, bytes);
    // coordinates are (i, j, k, field) in the padded layout of each array
    if (DIR == 0) {
      tma_load_4d(sP, &tm.P, bar, s0 - 6 + GPI, t0 + GPJ, o + GPK, 0);
      tma_load_4d(sM, &tm.M, bar, s0, t0, o, 0);
      if (in.moving) tma_load_4d(sMt, &tm.Mt, bar, s0, t0, o, 0);
      if (VISC && !(in.dbg & 1)) {
        tma_load_4d(sG, &tm.G, bar, s0 - 2 + GGI, t0 + GGJ, o + GGK, 4);
        tma_load_4d(sG + 4 * LG * TT, &tm.G, bar, s0 - 2 + GGI, t0 + GGJ, o + GGK, 8);
      }
      if (!in.first) tma_load_4d(sR, &tm.R, bar, s0, t0, o, 0);
    } else if (DIR == 1) {
      tma_load_4d(sP, &tm.P, bar, t0 + GPI, s0 - 6 + GPJ, o + GPK, 0);
      tma_load_4d(sM, &tm.M, bar, t0, s0, o, 0);
      if (in.moving) tma_load_4d(sMt, &tm.Mt, bar, t0, s0, o, 0);
      if (VISC && !(in.dbg & 1)) {
        tma_load_4d(sG, &tm.G, bar, t0 + GGI, s0 - 1 + GGJ, o + GGK, 0);
        tma_load_4d(sG + 4 * LG * TT, &tm.G, bar, t0 + GGI, s0 - 1 + GGJ, o + GGK, 8);
      }
      if (!in.first) tma_load_4d(sR, &tm.R, bar, t0, s0, o, 0);
    } else {
      tma_load_4d(sP, &tm.P, bar, t0 + GPI, o + GPJ, s0 - 6 + GPK, 0);
      tma_load_4d(sM, &tm.M, bar, t0, o, s0, 0);
      if (in.moving) tma_load_4d(sMt, &tm.Mt, bar, t0, o, s0, 0);
      if (VISC && !(in.dbg & 1)) {
        tma_load_4d(sG, &tm.G, bar, t0 + GGI, o + GGJ, s0 - 1 + GGK, 0);
        tma_load_4d(sG + 4 * LG * TT, &tm.G, bar, t0 + GGI, o + GGJ, s0 - 1 + GGK, 4);
      }
      if (!in.first) tma_load_4d(sR, &tm.R, bar, t0, o, s0, 0);
    }
  }
  mbar_wait(bar, 0);

  // thread -> (sweep position, transverse position) without runtime divisions
  int col, row, nrow_step;
  if (DIR == 0) { col = tid % 36; row = tid / 36; nrow_step = 0; }   // TT rows x 36 sweep positions
  else { row = tid % TT; col = tid / TT; nrow_step = C::NT / TT; }    // TT lanes x NT/TT sweep positions

  // ---- E6 first gradients (Eq. 17) on cells -1..TS, Eq. 19 second derivatives on cells -2..TS+1 ----
  for (int a = col; a < L2; a += (DIR == 0 ? 36 : nrow_step)) {
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      if (a < L1) {
        const double* q = sP + sidx<DIR, TT>(f, a + 5, row, LP);
        double r = CE1 * (q[SS_] - q[-SS_]);
        r = fma(CE2, q[2 * SS_] - q[-2 * SS_], r);
        r = fma(CE3, q[3 * SS_] - q[-3 * SS_], r);
        sP1[sidx<DIR, TT>(f, a, row, L1)] = r;
      }
      if (f < 5) {
        const double* q = sP + sidx<DIR, TT>(f, a + 4, row, LP);
        double r = CS0 * q[0];
        r = fma(CS1, q[SS_] + q[-SS_], r);
        r = fma(CS2, q[2 * SS_] + q[-2 * SS_], r);
        r = fma(CS3, q[3 * SS_] + q[-3 * SS_], r);
        r = fma(CS4, q[4 * SS_] + q[-4 * SS_], r);
        sP2[sidx<DIR, TT>(f, a, row, L2)] = r;
      }
    }
  }
  __syncthreads();

  // ---- one interface per (thread, pass) ----
  unsigned nlim = 0, ntst = 0;
  constexpr int FP = (DIR == 0) ? TT * LP : LP * TT;
  constexpr int F1 = (DIR == 0) ? TT * L1 : L1 * TT;
  constexpr int F2 = (DIR == 0) ? TT * L2 : L2 * TT;
  constexpr int FM = (DIR == 0) ? TT * LF : LF * TT;
  constexpr int FG = (DIR == 0) ? TT * LG : LG * TT;
  for (int sI = col; sI <= TS; sI += (DIR == 0 ? 36 : nrow_step)) {
    const bool valid = (s0 + sI <= nd) && (t0 + row < nt);
    const double* pM = sM + sidx<DIR, TT>(0, sI, row, LF);
    const int q0 = VISC ? 3 * DIR : 0;
    const double mx = pM[q0 * FM], my = pM[(q0 + 1) * FM], mz = pM[(q0 + 2) * FM];
    const double mt = in.moving ? sMt[sidx<DIR, TT>(0, sI, row, LF)] : 0.0;
    double F[5];
    if (valid) {
      const unsigned fl = inviscid_face<SS_, FP, F1, F2>(c, sP + sidx<DIR, TT>(0, sI + 4, row, LP),
                                                         sP1 + sidx<DIR, TT>(0, sI, row, L1),
                                                         sP2 + sidx<DIR, TT>(0, sI, row, L2), mx, my, mz, mt, F);
      if (sI < TS || s0 + sI == nd) { nlim += __popc(fl); ntst += 10; }
      if (VISC && !(in.dbg & 2)) {
        const double* pG = sG + sidx<DIR, TT>(0, sI + C::GOFF, row, LG);   // cell L = sI-1
        auto getG = [&](int e, int f, int cell) {
          // tangential directions in increasing order: slot 0 = first e != DIR, slot 1 = second
          const int slot = (DIR == 0) ? e - 1 : (DIR == 1) ? (e == 0 ? 0 : 1) : e;
          return pG[(4 * slot + f) * FG + cell * SS_];
        };
        auto getM = [&](int q) { return pM[q * FM]; };
        viscous_face<DIR, SS_, FP, F1>(c, sP + sidx<DIR, TT>(0, sI + 5, row, LP), sP1 + sidx<DIR, TT>(0, sI, row, L1),
                                       mx, my, mz, getG, getM, F);
      }
    } else {
#pragma unroll
      for (int f = 0; f < 5; ++f) F[f] = 0.0;
    }
#pragma unroll
    for (int f = 0; f < 5; ++f) sF[sidx<DIR, TT>(f, sI, row, LF)] = F[f];
  }
  if (in.stats) {
    for (int off = 16; off > 0; off >>= 1) {
      nlim += __shfl_down_sync(0xffffffffu, nlim, off);
      ntst += __shfl_down_sync(0xffffffffu, ntst, off);
    }
    if ((tid & 31) == 0 && ntst) { atomicAdd(in.stats, (unsigned long long)nlim); atomicAdd(in.stats + 1, (unsigned long long)ntst); }
  }
  __syncthreads();
  // ---- flux difference, Eq. 25: Res_i -= F_{i+1/2} - F_{i-1/2} ----
  for (int s = col; s < TS; s += (DIR == 0 ? 36 : nrow_step)) {
    if (s0 + s >= nd || t0 + row >= nt) continue;
    long long ac;
    if (DIR == 0) ac = c.LR.at(s0 + s, t0 + row, o);
    else if (DIR == 1) ac = c.LR.at(t0 + row, s0 + s, o);
    else ac = c.LR.at(t0 + row, o, s0 + s);
#pragma unroll
    for (int f = 0; f < 5; ++f) {
      const double dF = sF[sidx<DIR, TT>(f, s + 1, row, LF)] - sF[sidx<DIR, TT>(f, s, row, LF)];
      const double old = in.first ? 0.0 : sR[sidx<DIR, TT>(f, s, row, TS)];
      in.res[f * c.fsR + ac] = in.first ? -dF : old - dF;
    }
  }
}

}  // namespace meg6
