// The fused propagate-times-operator chain kernel.
//
// One *work unit* = (surviving string, panel of <= W carried columns).  A team of warps owns a unit for the whole
// chain: the carried panel X (d x W, stored column-wise with the contraction index contiguous) lives in shared memory
// in two ping-pong buffers, each step computes
//        X' = 2^-k * diag(exp(-Delta (E - Emin))) * F_alpha(q) * X
// on the FP64 tensor cores (mma.sync m8n8k4, SASS DMMA.8x8x4).  The operator block streams from the device store
// (L2 / HBM) straight into A fragments (each element is needed by exactly one warp, so staging it in shared memory would
// buy no reuse), the propagator is applied in the epilogue of the same step (never as a separate pass) as a mantissa in
// [1, 2) per row plus an integer row exponent; the largest exponent over non-zero rows is reduced with warp shuffles, goes
// into the running exponent, and the rows are brought to it by exact powers of two (so neither long chains nor
// Delta (E - Emin) >> 745 can overflow or underflow).  The last step is followed by the diagonal sum (trace) or the
// sum of squares (Frobenius norm of a segment).
// Work units are independent, so there is no inter-CTA communication: a persistent grid pulls units from an atomic
// counter, heaviest first.
#pragma once
#include <climits>

#include "common.cuh"

namespace ctqmc {

struct ChainParams {
  DevImp imp;
  BatchView bv;
  const StringRec* strings;
  const int2* units;
  Counters* cnt;
  Slot* slots;
  int ldx;          // leading dimension of a panel column in elements
  int mode;         // 0 trace, 1 Frobenius^2 of segments
  int segment_len;  // mode 1
};

template <int TEAM_WARPS>
__device__ __forceinline__ void team_sync(int team) {
  if constexpr (TEAM_WARPS == 1) {
    __syncwarp();
  } else if constexpr (TEAM_WARPS == kCtaWarps) {
    __syncthreads();
  } else {
    asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "r"(TEAM_WARPS * 32) : "memory");
  }
}

template <bool CPLX, int NT, int TEAM_WARPS>
__global__ void __launch_bounds__(kCtaThreads) chain_kernel(ChainParams P) {
  constexpr int ES = CPLX ? 2 : 1;
  constexpr int W = 8 * NT;
  constexpr int TEAMS = kCtaWarps / TEAM_WARPS;
  constexpr int TT = TEAM_WARPS * 32;
  constexpr int KS = CPLX ? 4 : 8;   // contraction indices consumed per 128-bit fragment load
  constexpr int U = 4;               // fragment loads kept in flight per lane

  extern __shared__ __align__(16) double smem[];
  __shared__ unsigned long long s_unit[TEAMS];
  __shared__ double s_red[TEAMS][TEAM_WARPS];
  __shared__ int s_exp[2][TEAMS][TEAM_WARPS];

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int team = warp / TEAM_WARPS, tw = warp % TEAM_WARPS;
  const int g = lane >> 2, t = lane & 3;
  const int tt = tw * 32 + lane;
  const int Q = P.imp.Q;
  const int ldx = P.ldx;
  const size_t xsz = (size_t)W * ldx * ES;
  double* Xbuf0 = smem + (size_t)team * 2 * xsz;
  double* Xbuf1 = Xbuf0 + xsz;

  for (;;) {
    if (tt == 0) s_unit[team] = atomicAdd(&P.cnt->next_unit, 1ull);
    team_sync<TEAM_WARPS>(team);
    const unsigned long long u = s_unit[team];
    team_sync<TEAM_WARPS>(team);
    if (u >= P.cnt->n_slots) break;

    const int2 un = P.units[u];
    const StringRec sr = P.strings[un.x];
    const long long b = un.x / Q;
    const long long base = P.bv.offset[b];
    const int L = (int)(P.bv.offset[b + 1] - base);
    const int* sym = P.bv.symbol + base;
    const double* tau = P.bv.tau + base;

    // ---- decode the unit: first operator, number of steps, start sector, column window
    int q = sr.q_start, i0 = sr.r, nsteps = L, c0, ncols;
    if (P.mode == 0) {
      c0 = un.y * W;
      ncols = min(W, sr.c - c0);
    } else {
      int rem = un.y, i = 0;
      for (;;) {
        int np = (P.imp.dim[q] + W - 1) / W;
        if (rem < np) break;
        rem -= np;
        int stop = min(L, i + P.segment_len);
        for (; i < stop; ++i) q = P.imp.blks[P.imp.blk_of[sym[i] * Q + q]].dst;
      }
      i0 = i;
      nsteps = min(P.segment_len, L - i0);
      c0 = rem * W;
      ncols = min(W, P.imp.dim[q] - c0);
    }
    const int ntu = (ncols + 7) >> 3;
    int d = P.imp.dim[q];

    // ---- X_0 = columns [c0, c0 + ncols) of the identity
    {
      const int kp = round_up(d, 8);
      for (int idx = tt; idx < W * kp; idx += TT) {
        int n = idx / kp, k = idx - n * kp;
        double v = (n < ncols && k == c0 + n) ? 1.0 : 0.0;
        if constexpr (CPLX) {
          *reinterpret_cast<double2*>(Xbuf0 + ((size_t)n * ldx + k) * 2) = make_double2(v, 0.0);
        } else {
          Xbuf0[(size_t)n * ldx + k] = v;
        }
      }
    }
    team_sync<TEAM_WARPS>(team);

    double* X = Xbuf0;
    double* Xn = Xbuf1;
    long long e2 = 0;
    bool dead = false;

    for (int j = 0; j < nsteps; ++j) {
      int i = i0 + j;
      if (i >= L) i -= L;
      const int blk = P.imp.blk_of[sym[i] * Q + q];
      const BlkDesc bd = P.imp.blks[blk];
      const int qn = bd.dst, dn = bd.rows;
      const double delta = (i + 1 < L) ? (tau[i + 1] - tau[i]) : (P.bv.beta - tau[i] + tau[0]);
      const double* E = P.imp.energy + P.imp.e_off[qn];
      const double emin = P.imp.e_min[qn];
      const int MT = (dn + 7) >> 3;
      const int nk = round_up(d, KS) / KS;
      int wexp = INT_MIN;

      for (int mt = tw; mt < MT; mt += TEAM_WARPS) {
        const int row = mt * 8 + g;
        const double* Ar = P.imp.store + bd.off + (size_t)row * bd.ld * ES + t * 2;
        const double* Xr = X + (size_t)g * ldx * ES + t * 2;
        double acc[NT][CPLX ? 4 : 2];
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int x = 0; x < (CPLX ? 4 : 2); ++x) acc[nt][x] = 0.0;

        double2 a_cur[U], a_nxt[U];
#pragma unroll
        for (int uu = 0; uu < U; ++uu)
          a_cur[uu] = (uu < nk) ? __ldg(reinterpret_cast<const double2*>(Ar + uu * 8)) : make_double2(0.0, 0.0);

        for (int kb = 0; kb < nk; kb += U) {
#pragma unroll
          for (int uu = 0; uu < U; ++uu) {
            int kk = kb + U + uu;
            a_nxt[uu] = (kk < nk) ? __ldg(reinterpret_cast<const double2*>(Ar + kk * 8)) : make_double2(0.0, 0.0);
          }
#pragma unroll
          for (int uu = 0; uu < U; ++uu) {
            if (kb + uu < nk) {
              const double2 a = a_cur[uu];
              const double* Xk = Xr + (kb + uu) * 8;
              if constexpr (CPLX) {
                const double na = -a.y;
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                  if (nt < ntu) {
                    const double2 bb = *reinterpret_cast<const double2*>(Xk + (size_t)nt * 8 * ldx * 2);
                    dmma884(acc[nt][0], acc[nt][1], a.x, bb.x);
                    dmma884(acc[nt][0], acc[nt][1], na, bb.y);
                    dmma884(acc[nt][2], acc[nt][3], a.x, bb.y);
                    dmma884(acc[nt][2], acc[nt][3], a.y, bb.x);
                  }
                }
              } else {
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) {
                  if (nt < ntu) {
                    const double2 bb = *reinterpret_cast<const double2*>(Xk + (size_t)nt * 8 * ldx);
                    dmma884(acc[nt][0], acc[nt][1], a.x, bb.x);
                    dmma884(acc[nt][0], acc[nt][1], a.y, bb.y);
                  }
                }
              }
            }
          }
#pragma unroll
          for (int uu = 0; uu < U; ++uu) a_cur[uu] = a_nxt[uu];
        }

        // epilogue, phase 1: the propagator exp(-Delta (E_row - Emin)) = 2^x is split into the mantissa 2^(x - floor x),
        // multiplied in here, and the integer floor(x), which only enters the row's binary exponent (so no row can
        // underflow, whatever Delta (E - Emin) is); track the largest exponent of a non-zero row.
        double mr = 0.0;
        int kr = 0;
        if (row < dn) {
          const double x = prop_x(delta, E[row], emin);
          const double kf = floor(x);
          mr = exp2(__dsub_rn(x, kf));
          kr = row_exp(x);
        }
        double rmax = 0.0;
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) {
          if (nt < ntu) {
            const int n = nt * 8 + 2 * t;
            if constexpr (CPLX) {
              const double2 v0 = make_double2(acc[nt][0] * mr, acc[nt][2] * mr);
              const double2 v1 = make_double2(acc[nt][1] * mr, acc[nt][3] * mr);
              *reinterpret_cast<double2*>(Xn + ((size_t)n * ldx + row) * 2) = v0;
              *reinterpret_cast<double2*>(Xn + ((size_t)(n + 1) * ldx + row) * 2) = v1;
              rmax = fmax(fmax(rmax, fmax(fabs(v0.x), fabs(v0.y))), fmax(fabs(v1.x), fabs(v1.y)));
            } else {
              const double v0 = acc[nt][0] * mr, v1 = acc[nt][1] * mr;
              Xn[(size_t)n * ldx + row] = v0;
              Xn[(size_t)(n + 1) * ldx + row] = v1;
              rmax = fmax(rmax, fmax(fabs(v0), fabs(v1)));
            }
          }
        }
        rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, 1));
        rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, 2));
        if (rmax > 0.0) wexp = max(wexp, kr + ilogb(rmax));
      }

      // running exponent: largest row exponent over the team
      wexp = __reduce_max_sync(0xffffffffu, wexp);
      if (lane == 0) s_exp[j & 1][team][tw] = wexp;
      team_sync<TEAM_WARPS>(team);
      int kmax = INT_MIN;
#pragma unroll
      for (int w = 0; w < TEAM_WARPS; ++w) kmax = max(kmax, s_exp[j & 1][team][w]);
      if (kmax == INT_MIN) { dead = true; break; }
      e2 += kmax;

      // epilogue, phase 2: every thread brings the elements it wrote to the common exponent (exact power of two;
      // rows more than 2^-1022 below the largest flush to zero)
      for (int mt = tw; mt < MT; mt += TEAM_WARPS) {
        const int row = mt * 8 + g;
        if (row < dn) {
          const double x = prop_x(delta, E[row], emin);
          const int sh = row_exp(x) - kmax;
          const bool slow = sh > 1022;
          const double f = (sh < -1022) ? 0.0 : pow2i(min(sh, 1022));
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            if (nt < ntu) {
              const int n = nt * 8 + 2 * t;
              if constexpr (CPLX) {
                double2* p0 = reinterpret_cast<double2*>(Xn + ((size_t)n * ldx + row) * 2);
                double2* p1 = reinterpret_cast<double2*>(Xn + ((size_t)(n + 1) * ldx + row) * 2);
                double2 v0 = *p0, v1 = *p1;
                if (slow) { v0.x = scalbn(v0.x, sh); v0.y = scalbn(v0.y, sh); v1.x = scalbn(v1.x, sh); v1.y = scalbn(v1.y, sh); }
                else { v0.x *= f; v0.y *= f; v1.x *= f; v1.y *= f; }
                *p0 = v0; *p1 = v1;
              } else {
                double* p0 = Xn + (size_t)n * ldx + row;
                double* p1 = Xn + (size_t)(n + 1) * ldx + row;
                if (slow) { *p0 = scalbn(*p0, sh); *p1 = scalbn(*p1, sh); }
                else { *p0 *= f; *p1 *= f; }
              }
            }
          }
        }
      }
      team_sync<TEAM_WARPS>(team);
      double* tmp = X; X = Xn; Xn = tmp;
      q = qn;
      d = dn;
    }

    // ---- reduction of the final panel
    if (P.mode == 0) {
      if (tt == 0) {
        Slot out; out.re = 0.0; out.im = 0.0; out.e2 = 0; out.pad = 0;
        if (!dead) {
          double re = 0.0, im = 0.0;
          if (L == 0) {   // empty configuration: Tr P_beta(q0), the partition-function term (reading A7)
            const double* E0 = P.imp.energy + P.imp.e_off[q];
            const double em0 = P.imp.e_min[q];
            for (int n = 0; n < ncols; ++n) re += exp(-P.bv.beta * (E0[c0 + n] - em0));
          } else
          for (int n = 0; n < ncols; ++n) {
            if constexpr (CPLX) {
              const double2 v = *reinterpret_cast<const double2*>(X + ((size_t)n * ldx + c0 + n) * 2);
              re += v.x; im += v.y;
            } else {
              re += X[(size_t)n * ldx + c0 + n];
            }
          }
          out.re = re; out.im = im; out.e2 = e2;
        }
        P.slots[sr.slot + un.y] = out;
      }
    } else {
      double ss = 0.0;
      if (!dead) {
        for (int idx = tt; idx < ncols * d; idx += TT) {
          int n = idx / d, k = idx - n * d;
          if constexpr (CPLX) {
            const double2 v = *reinterpret_cast<const double2*>(X + ((size_t)n * ldx + k) * 2);
            ss += v.x * v.x + v.y * v.y;
          } else {
            const double v = X[(size_t)n * ldx + k];
            ss += v * v;
          }
        }
      }
      ss = warp_sum(ss);
      team_sync<TEAM_WARPS>(team);
      if (lane == 0) s_red[team][tw] = ss;
      team_sync<TEAM_WARPS>(team);
      if (tt == 0) {
        double tot = 0.0;
        for (int w = 0; w < TEAM_WARPS; ++w) tot += s_red[team][w];
        Slot out; out.re = tot; out.im = 0.0; out.e2 = dead ? 0 : e2; out.pad = 0;
        P.slots[sr.slot + un.y] = out;
      }
    }
    team_sync<TEAM_WARPS>(team);
  }
}

}  // namespace ctqmc
