// meg6_ig4.cuh -- MIG4 variant (scheme = 1): implicit fourth-order gradients IG4, Eq. 18 (R2), and the
// pass-based geometry that uses them wherever MEG6 uses E6.
//
// Reading R26: a tridiagonal system spans every cell of the padded grid line whose right-hand side
// exists and is closed at both ends with the explicit fourth-order difference of Eq. D.2.  One thread solves one
// line with the Thomas algorithm; the elimination coefficients depend on the position only and come from the host.
// Part of meg6_geom.cu (compiled with -fmad=false): the operation order is the one the discretisation states, and
// the geometry arrays are compared bit for bit with the oracle's.
#pragma once
#include "meg6_common.cuh"

namespace meg6 {

__device__ __forceinline__ double c4_op(const double* __restrict__ f, long long s) {   // Eq. D.2
  return 2.0 / 3.0 * (f[s] - f[-s]) - 1.0 / 12.0 * (f[2 * s] - f[-2 * s]);
}

// out = IG4 gradient of f along DIR on `ob` (= the box of f shrunk by 2 at both ends of DIR).
template <int DIR>
__global__ void __launch_bounds__(128) k_ig4(Lay L, const double* __restrict__ f, double* __restrict__ out, Box ob,
                                             const double* __restrict__ cc, const double* __restrict__ den,
                                             long long fs_in, long long fs_out) {
  // blockIdx.y = field of a batch (arrays fs_in / fs_out doubles apart): one launch for all fields keeps the grid many
  // waves deep -- a thread lives as long as its whole line, so a launch of ~2 waves wastes most of its last one
  f += blockIdx.y * fs_in; out += blockIdx.y * fs_out;
  constexpr int A1 = (DIR == 0) ? 1 : 0, A2 = (DIR == 2) ? 1 : 2;   // transverse directions, lower index fastest
  const int n1 = ob.hi[A1] - ob.lo[A1], n2 = ob.hi[A2] - ob.lo[A2];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)n1 * n2) return;
  int ix[3];
  ix[A1] = ob.lo[A1] + (int)(tid % n1); ix[A2] = ob.lo[A2] + (int)(tid / n1); ix[DIR] = ob.lo[DIR];
  const int m = ob.hi[DIR] - ob.lo[DIR];
  const long long at = L.at(ix[0], ix[1], ix[2]), s = L.stride(DIR);
  const double* pf = f + at;
  double* px = out + at;
  const double al = 5.0 / 14.0, ca = (2.0 + al) / 3.0, cb = (4.0 * al - 1.0) / 12.0;
  // The recurrences are serial, the loads are not: each chunk of CH cells first gathers its window of f (CH + 4
  // independent loads in flight instead of one cache miss per step), then runs the chain.  Same operations, same
  // order per cell as the plain loop.  Indices are clamped to the valid range of f (cells -2 .. m+1 relative to the
  // first unknown), so the ragged last chunk reads nothing it should not.
  constexpr int CH = 16;
  double prev = c4_op(pf, s);                       // first unknown: explicit
  px[0] = prev;
  for (int q0 = 1; q0 < m - 1; q0 += CH) {
    double w[CH + 4], dn[CH];
#pragma unroll
    for (int u = 0; u < CH + 4; ++u) w[u] = pf[(long long)min(q0 - 2 + u, m + 1) * s];
#pragma unroll
    for (int u = 0; u < CH; ++u) dn[u] = den[min(q0 + u, m - 1)];
#pragma unroll
    for (int u = 0; u < CH; ++u) {
      const int q = q0 + u;
      if (q < m - 1) {
        const double r = ca * (w[u + 3] - w[u + 1]) + cb * (w[u + 4] - w[u]);
        prev = (r - al * prev) / dn[u];
        px[(long long)q * s] = prev;
      }
    }
  }
  double nxt = c4_op(pf + (long long)(m - 1) * s, s);   // last unknown: explicit
  px[(long long)(m - 1) * s] = nxt;
  for (int q0 = m - 2; q0 >= 1; q0 -= CH) {
    double d[CH], cq[CH];
#pragma unroll
    for (int u = 0; u < CH; ++u) {
      const int q = max(q0 - u, 1);
      d[u] = px[(long long)q * s]; cq[u] = cc[q];
    }
#pragma unroll
    for (int u = 0; u < CH; ++u) {
      const int q = q0 - u;
      if (q >= 1) {
        nxt = d[u] - cq[u] * nxt;
        px[(long long)q * s] = nxt;
      }
    }
  }
}

// The same solve for lines along xi (unit stride): a thread walking along its own row would touch 32 different rows
// per warp instruction.  Here a warp owns 32 rows and moves along xi in chunks of 32 columns: the chunk is loaded
// row by row with full-width coalesced accesses into a shared-memory tile, every lane runs the recurrence of its own
// row out of the tile (row pitch 37: conflict-free), and the results leave the same way.  Operations and their order
// per cell are those of k_ig4.
__global__ void __launch_bounds__(128) k_ig4x(Lay L, const double* __restrict__ f, double* out, Box ob,
                                              const double* __restrict__ cc, const double* __restrict__ den,
                                              long long fs_in, long long fs_out) {
  f += blockIdx.y * fs_in; out += blockIdx.y * fs_out;
  __shared__ double tile[4][32][37];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double (*T)[37] = tile[warp];
  const int n1 = ob.hi[1] - ob.lo[1], n2 = ob.hi[2] - ob.lo[2];
  const long long nl = (long long)n1 * n2, lid = ((long long)blockIdx.x * 4 + warp) * 32 + lane;
  const bool active = lid < nl;
  const long long lc = active ? lid : 0;
  const long long at = L.at(ob.lo[0], ob.lo[1] + (int)(lc % n1), ob.lo[2] + (int)(lc / n1));
  const int m = ob.hi[0] - ob.lo[0];
  const double al = 5.0 / 14.0, ca = (2.0 + al) / 3.0, cb = (4.0 * al - 1.0) / 12.0;
  double prev = c4_op(f + at, 1);                   // first unknown: explicit
  if (active) out[at] = prev;
  for (int q0 = 1; q0 < m - 1; q0 += 32) {
    for (int r = 0; r < 32; ++r) {                  // window columns q0-2 .. q0+33 of row r
      const long long ar = __shfl_sync(0xffffffffu, at, r);
      T[r][lane] = f[ar + min(q0 - 2 + lane, m + 1)];
      if (lane < 4) T[r][32 + lane] = f[ar + min(q0 + 30 + lane, m + 1)];
    }
    __syncwarp();
    for (int u = 0; u < 32; ++u) {
      const int q = q0 + u;
      if (q < m - 1) {
        const double r = ca * (T[lane][u + 3] - T[lane][u + 1]) + cb * (T[lane][u + 4] - T[lane][u]);
        prev = (r - al * prev) / den[q];
        T[lane][u] = prev;                          // column u is not read again
      }
    }
    __syncwarp();
    for (int r = 0; r < 32; ++r) {
      const long long ar = __shfl_sync(0xffffffffu, at, r);
      const bool actr = __shfl_sync(0xffffffffu, (int)active, r) != 0;
      if (actr && q0 + lane < m - 1) out[ar + q0 + lane] = T[r][lane];
    }
    __syncwarp();
  }
  double nxt = c4_op(f + at + (m - 1), 1);          // last unknown: explicit
  if (active) out[at + (m - 1)] = nxt;
  __syncwarp();
  for (int q0 = m - 2; q0 >= 1; q0 -= 32) {
    const int lo = q0 - 31;                         // chunk columns lo .. q0
    for (int r = 0; r < 32; ++r) {
      const long long ar = __shfl_sync(0xffffffffu, at, r);
      T[r][lane] = out[ar + max(lo + lane, 1)];
    }
    __syncwarp();
    for (int u = 0; u < 32; ++u) {
      const int q = q0 - u;
      if (q >= 1) {
        nxt = T[lane][q - lo] - cc[q] * nxt;
        T[lane][q - lo] = nxt;
      }
    }
    __syncwarp();
    for (int r = 0; r < 32; ++r) {
      const long long ar = __shfl_sync(0xffffffffu, at, r);
      const bool actr = __shfl_sync(0xffffffffu, (int)active, r) != 0;
      if (actr && lo + lane >= 1) out[ar + lo + lane] = T[r][lane];
    }
    __syncwarp();
  }
}

// Segmented solve for the FLOW gradients along eta / zeta (not for the geometry: the rounding order differs from the
// plain Thomas loop at the segment boundaries).  The two sweeps of the Thomas algorithm are first-order linear
// recurrences, d_q = (r_q - alpha d_{q-1}) / den_q and x_q = d_q - c_q x_{q+1}: a line is cut into NSEG segments, each
// thread runs its segment once with a zero inflow value (which gives the affine map inflow -> outflow, slope = product
// of the -c_q, ~0.4^length), the maps are chained through shared memory, and the segment is run again from its true
// inflow value.  Everything between the two passes stays in registers: f is read once and the gradient written once
// (the one-thread-per-line kernel writes d and reads it back: four array passes instead of two).
// CTA = 16 xi-lanes (128-byte rows) x NSEG segments, two CTAs per SM; a line has at most NSEG * SEGMAX + 2 unknowns.
constexpr int IG4S_NSEG = 32, IG4S_SEGMAX = 13, IG4S_LANES = 16;
template <int DIR>
__global__ void __launch_bounds__(IG4S_LANES * IG4S_NSEG, 2) k_ig4s(Lay L, const double* __restrict__ f, double* __restrict__ out,
                                                                  Box ob, const double* __restrict__ cc, long long fs_in,
                                                                  long long fs_out) {
  constexpr int NSEG = IG4S_NSEG, SMAX = IG4S_SEGMAX, NL = IG4S_LANES;
  constexpr int OD = (DIR == 1) ? 2 : 1;            // the other transverse direction (xi is the lane direction)
  __shared__ double sA[NSEG][NL], sB[NSEG][NL], sX[2][NL];
  f += blockIdx.z * fs_in; out += blockIdx.z * fs_out;
  const int lane = threadIdx.x % NL, seg = threadIdx.x / NL;
  const int n0 = ob.hi[0] - ob.lo[0];
  const int i = blockIdx.x * NL + lane;
  const bool act = i < n0;
  int ix[3];
  ix[0] = ob.lo[0] + (act ? i : 0); ix[OD] = ob.lo[OD] + blockIdx.y; ix[DIR] = ob.lo[DIR];
  const int m = ob.hi[DIR] - ob.lo[DIR];            // unknowns 0 .. m-1; 0 and m-1 explicit
  const long long at = L.at(ix[0], ix[1], ix[2]), s = L.stride(DIR);
  const double* pf = f + at;
  double* px = out + at;
  const double al = 5.0 / 14.0, ial = 14.0 / 5.0, ca = (2.0 + al) / 3.0, cb = (4.0 * al - 1.0) / 12.0;
  const int nseg = blockDim.x / NL;                 // segments of this launch (<= NSEG)
  const int len = (m - 2 + nseg - 1) / nseg;        // interior unknowns per segment (<= SMAX)
  // a segment multiplies its inflow value by the product of its c_q (< 0.42 each): beyond `reach` segments the
  // contribution is below 0.42^48 = 1e-18 of the value and is not summed
  const int reach = (48 + len - 1) / len;
  const int q0 = 1 + seg * len;                     // first unknown of this segment
  const int nq = max(0, min(len, m - 1 - q0));      // its unknowns
  const bool last = nq > 0 && q0 + nq == m - 1;     // the segment next to the explicit last unknown
  double r[SMAX];
  {
    double w[SMAX + 4];
    const double* pw = pf + (long long)(q0 - 2) * s;   // running pointer: one 64-bit add per load instead of a multiply
#pragma unroll
    for (int u = 0; u < SMAX + 4; ++u) { w[u] = (nq > 0 && u < nq + 4) ? *pw : 0.0; pw += s; }
#pragma unroll
    for (int u = 0; u < SMAX; ++u) r[u] = fma(cb, w[u + 4] - w[u], ca * (w[u + 3] - w[u + 1]));
  }
  if (seg == 0) sX[0][lane] = c4_op(pf, s);                              // first unknown: explicit (R26)
  if (last) sX[1][lane] = c4_op(pf + (long long)(m - 1) * s, s);         // last unknown: explicit
  const double* __restrict__ cs = cc + q0;                               // c_q = alpha / den_q, position only
  // ---- forward sweep: d_q = (r_q - alpha d_{q-1}) / den_q, 1/den_q = c_q / alpha ----
  {
    double a = 0.0, b = 1.0;
#pragma unroll
    for (int u = 0; u < SMAX; ++u)
      if (u < nq) { const double c = __ldg(cs + u); a = fma(-al, a, r[u]) * (c * ial); b = -c * b; }
    sA[seg][lane] = a; sB[seg][lane] = b;
  }
  __syncthreads();
  double din = (seg <= reach) ? sX[0][lane] : 0.0;
  for (int t = max(0, seg - reach); t < seg; ++t) din = fma(sB[t][lane], din, sA[t][lane]);
#pragma unroll
  for (int u = 0; u < SMAX; ++u)
    if (u < nq) { din = fma(-al, din, r[u]) * (__ldg(cs + u) * ial); r[u] = din; }
  __syncthreads();
  // ---- backward sweep: x_q = d_q - c_q x_{q+1} ----
  {
    double a = 0.0, b = 1.0;
#pragma unroll
    for (int u = SMAX - 1; u >= 0; --u)
      if (u < nq) { const double c = __ldg(cs + u); a = fma(-c, a, r[u]); b = -c * b; }
    sA[seg][lane] = a; sB[seg][lane] = b;
  }
  __syncthreads();
  double xin = (seg + reach >= nseg - 1) ? sX[1][lane] : 0.0;
  for (int t = min(nseg - 1, seg + reach); t > seg; --t) xin = fma(sB[t][lane], xin, sA[t][lane]);
  if (!act) return;
  double* po = px + (long long)(q0 + SMAX - 1) * s;
#pragma unroll
  for (int u = SMAX - 1; u >= 0; --u) {
    if (u < nq) { xin = fma(-__ldg(cs + u), xin, r[u]); *po = xin; }
    po -= s;
  }
  if (seg == 0) px[0] = sX[0][lane];
  if (last) px[(long long)(m - 1) * s] = sX[1][lane];
}

// The segmented solve for lines along xi (flow gradients only, like k_ig4s).  A xi line is contiguous in memory, so the
// lanes of a warp are the segments of one line (or of several short lines: LPW lines of SPL segments each): the warp
// copies its lines into shared memory with full-width coalesced loads, every lane takes its SEG-cell window from
// there (lane stride 13 doubles: conflict-free), the affine maps of the two Thomas sweeps are chained with warp shuffles,
// and the gradients leave through the same tile.  f is read once and the gradient written once (k_ig4x: four passes).
constexpr int IG4SX_WARPS = 4, IG4SX_TILE = 32 * IG4S_SEGMAX + 8;
__global__ void __launch_bounds__(32 * IG4SX_WARPS) k_ig4sx(Lay L, const double* __restrict__ f, double* __restrict__ out, Box ob,
                                                            const double* __restrict__ cc, long long fs_in, long long fs_out,
                                                            int spl, int lpw) {
  constexpr int SMAX = IG4S_SEGMAX;
  __shared__ double tile[IG4SX_WARPS][IG4SX_TILE];
  f += blockIdx.y * fs_in; out += blockIdx.y * fs_out;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  double* T = tile[warp];
  const int n1 = ob.hi[1] - ob.lo[1], n2 = ob.hi[2] - ob.lo[2];
  const long long nl = (long long)n1 * n2;
  const int m = ob.hi[0] - ob.lo[0];                // unknowns 0 .. m-1 of a line; 0 and m-1 explicit (R26)
  const int W = m + 4;                              // f window of a line: cells -2 .. m+1 relative to the first unknown
  const long long line0 = ((long long)blockIdx.x * IG4SX_WARPS + warp) * lpw;   // first line of this warp
  const double al = 5.0 / 14.0, ial = 14.0 / 5.0, ca = (2.0 + al) / 3.0, cb = (4.0 * al - 1.0) / 12.0;
  // ---- stage the windows of the warp's lines ----
  for (int l = 0; l < lpw; ++l) {
    const long long lid = line0 + l;
    if (lid >= nl) break;
    const double* pf = f + L.at(ob.lo[0], ob.lo[1] + (int)(lid % n1), ob.lo[2] + (int)(lid / n1)) - 2;
    for (int q = lane; q < W; q += 32) T[l * W + q] = pf[q];
  }
  __syncwarp();
  const int ln = lane / spl, seg = lane % spl;      // this lane: segment `seg` of the warp's line `ln`
  const long long lid = line0 + ln;
  const bool act = ln < lpw && lid < nl;
  const int len = (m - 2 + spl - 1) / spl;          // interior unknowns per segment (<= SMAX)
  const int reach = (48 + len - 1) / len;           // see k_ig4s
  const int q0 = 1 + seg * len;
  const int nq = act ? max(0, min(len, m - 1 - q0)) : 0;
  const double* Tl = T + (act ? ln : 0) * W + 2;    // Tl[q] = f at unknown q of this lane's line
  double r[SMAX];
#pragma unroll
  for (int u = 0; u < SMAX; ++u) {
    const double* w = Tl + q0 + u;
    r[u] = (u < nq) ? fma(cb, w[2] - w[-2], ca * (w[1] - w[-1])) : 0.0;
  }
  const double x0 = 2.0 / 3.0 * (Tl[1] - Tl[-1]) - 1.0 / 12.0 * (Tl[2] - Tl[-2]);                    // Eq. D.2 at unknown 0
  const double xm = 2.0 / 3.0 * (Tl[m] - Tl[m - 2]) - 1.0 / 12.0 * (Tl[m + 1] - Tl[m - 3]);          // ... and at m-1
  const double* __restrict__ cs = cc + q0;
  const unsigned full = 0xffffffffu;
  // ---- forward sweep ----
  double a = 0.0, b = 1.0;
#pragma unroll
  for (int u = 0; u < SMAX; ++u)
    if (u < nq) { const double c = __ldg(cs + u); a = fma(-al, a, r[u]) * (c * ial); b = -c * b; }
  double din = (seg <= reach) ? x0 : 0.0;
  for (int k = reach; k >= 1; --k) {                // maps of the segments seg-k .. seg-1 of the same line, in order
    const double at = __shfl_up_sync(full, a, k), bt = __shfl_up_sync(full, b, k);
    if (seg - k >= 0) din = fma(bt, din, at);
  }
#pragma unroll
  for (int u = 0; u < SMAX; ++u)
    if (u < nq) { din = fma(-al, din, r[u]) * (__ldg(cs + u) * ial); r[u] = din; }
  // ---- backward sweep ----
  a = 0.0; b = 1.0;
#pragma unroll
  for (int u = SMAX - 1; u >= 0; --u)
    if (u < nq) { const double c = __ldg(cs + u); a = fma(-c, a, r[u]); b = -c * b; }
  const int nsg = (m - 2 + len - 1) / len;          // segments that hold unknowns
  double xin = (seg + reach >= nsg - 1) ? xm : 0.0;
  for (int k = reach; k >= 1; --k) {                // maps of the segments seg+k .. seg+1
    const double at = __shfl_down_sync(full, a, k), bt = __shfl_down_sync(full, b, k);
    if (seg + k <= nsg - 1 && seg + k < spl) xin = fma(bt, xin, at);
  }
  __syncwarp();                                     // every lane has read its window: the tile now takes the results
#pragma unroll
  for (int u = SMAX - 1; u >= 0; --u)
    if (u < nq) { xin = fma(-__ldg(cs + u), xin, r[u]); T[ln * W + 2 + q0 + u] = xin; }
  if (act && seg == 0) { T[ln * W + 2] = x0; T[ln * W + 2 + m - 1] = xm; }
  __syncwarp();
  for (int l = 0; l < lpw; ++l) {
    const long long lo = line0 + l;
    if (lo >= nl) break;
    double* po = out + L.at(ob.lo[0], ob.lo[1] + (int)(lo % n1), ob.lo[2] + (int)(lo / n1));
    for (int q = lane; q < m; q += 32) po[q] = T[l * W + 2 + q];
  }
}

// Central interface value Eq. 36/38 from f and its gradient f1: index i of `out` = interface between
// cells i and i+1 along dir.  The second derivative is Eq. 19.  `out` may have another layout (interface
// arrays): LO, and an index shift `sh` along dir (interface arrays number the face between cells i-1 and i as i).
__global__ void __launch_bounds__(256) k_H_from(Lay L, Lay LO, int dir, int sh, const double* __restrict__ f,
                                                const double* __restrict__ f1, double* __restrict__ out, Box ob) {
  const int n0 = ob.hi[0] - ob.lo[0], n1 = ob.hi[1] - ob.lo[1], n2 = ob.hi[2] - ob.lo[2];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)n0 * n1 * n2) return;
  int ix[3] = {ob.lo[0] + (int)(tid % n0), ob.lo[1] + (int)((tid / n0) % n1), ob.lo[2] + (int)(tid / ((long long)n0 * n1))};
  const long long c = L.at(ix[0], ix[1], ix[2]), s = L.stride(dir);
  const double* pf = f + c;
  const double* p1 = f1 + c;
  const double f2a = 2.0 * (pf[s] - 2.0 * pf[0] + pf[-s]) - 0.5 * (p1[s] - p1[-s]);
  const double f2b = 2.0 * (pf[2 * s] - 2.0 * pf[s] + pf[0]) - 0.5 * (p1[2 * s] - p1[0]);
  const double Lv = pf[0] + 0.5 * p1[0] + f2a / 12.0;
  const double Rv = pf[s] - 0.5 * p1[s] + f2b / 12.0;
  ix[dir] += sh;
  out[LO.at(ix[0], ix[1], ix[2])] = 0.5 * (Lv + Rv);
}

// mode 0: out_i = a_i - a_{i-1 along dir} (Eq. 37);  mode 1: out = a * b;  mode 2: out = a - b
__global__ void __launch_bounds__(256) k_point(Lay L, int mode, int dir, const double* __restrict__ a,
                                               const double* __restrict__ b, double* __restrict__ out, Box ob) {
  const int n0 = ob.hi[0] - ob.lo[0], n1 = ob.hi[1] - ob.lo[1], n2 = ob.hi[2] - ob.lo[2];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)n0 * n1 * n2) return;
  const int i = ob.lo[0] + (int)(tid % n0), j = ob.lo[1] + (int)((tid / n0) % n1), k = ob.lo[2] + (int)(tid / ((long long)n0 * n1));
  const long long c = L.at(i, j, k);
  if (mode == 0) out[c] = a[c] - a[c - L.stride(dir)];
  else if (mode == 1) out[c] = a[c] * b[c];
  else out[c] = a[c] - b[c];
}

struct P9c { const double* p[9]; };
struct P3c { const double* p[3]; };
struct P3w { double* p[3]; };

// 1/J = det of the coordinate derivatives, Eq. 13
__global__ void __launch_bounds__(256) k_rj_box(Lay L, P9c cd, double* __restrict__ rj, Box ob) {
  const int n0 = ob.hi[0] - ob.lo[0], n1 = ob.hi[1] - ob.lo[1], n2 = ob.hi[2] - ob.lo[2];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)n0 * n1 * n2) return;
  const long long at = L.at(ob.lo[0] + (int)(tid % n0), ob.lo[1] + (int)((tid / n0) % n1), ob.lo[2] + (int)(tid / ((long long)n0 * n1)));
  const double xx = cd.p[0][at], xe = cd.p[1][at], xz = cd.p[2][at];
  const double yx = cd.p[3][at], ye = cd.p[4][at], yz = cd.p[5][at];
  const double zx = cd.p[6][at], ze = cd.p[7][at], zz = cd.p[8][at];
  rj[at] = xx * (ye * zz - ze * yz) - yx * (xe * zz - ze * xz) + zx * (xe * yz - ye * xz);
}

// hatted time metric of direction r, Eq. 11, on the box of that direction's metrics
__global__ void __launch_bounds__(256) k_mt_box(Lay L, P3c xt, const double* __restrict__ mx, const double* __restrict__ my,
                                                const double* __restrict__ mz, double* __restrict__ mt, Box ob) {
  const int n0 = ob.hi[0] - ob.lo[0], n1 = ob.hi[1] - ob.lo[1], n2 = ob.hi[2] - ob.lo[2];
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (tid >= (long long)n0 * n1 * n2) return;
  const long long at = L.at(ob.lo[0] + (int)(tid % n0), ob.lo[1] + (int)((tid / n0) % n1), ob.lo[2] + (int)(tid / ((long long)n0 * n1)));
  mt[at] = -(xt.p[0][at] * mx[at] + xt.p[1][at] * my[at] + xt.p[2][at] * mz[at]);
}

}  // namespace meg6
