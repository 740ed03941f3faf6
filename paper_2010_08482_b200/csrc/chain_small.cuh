// Small-sector path (all sectors of dimension <= 16, e.g. the Kanamori impurities): the WHOLE hot path of a configuration
// -- validation, sector routing (a2), the fused propagate x operator chain with running exponent (a3, a4), the trace and
// the exponent-aligned sector sum (a5) -- in ONE kernel launch (PAPER.md:529 Eq. 65, :532-534, :521).
//
// The complete operator store (a few KB once packed without padding), the eigenvalues and the routing table are copied
// into shared memory once per CTA ("packed many-per-CTA in shared memory"); a group of G lanes (a sub-warp) owns one
// configuration: its lanes first walk the sector map for all start sectors in parallel (one q0 per lane), then multiply
// the chains of the surviving start sectors, one output element per lane, carried matrix in shared memory.  Nothing but
// the operator string (12 B per operator, coalesced, read twice) and the results (24 B + Q per configuration) touches
// HBM.  These matrices are far too small for the tensor cores (d <= 16, carried width usually 1..3): plain FP64 FMAs.
#pragma once
#include <climits>

#include "common.cuh"

namespace ctqmc {

struct SmallParams {
  DevImp imp;
  BatchView bv;
  const double* pack;       // unpadded row-major blocks (ES doubles per element)
  const int4* pblk;         // per block {offset into pack (elements), rows, cols, dst}
  int n_blocks, pack_len, n_energy;
  int literal;
  double* mant; long long* exp2; uint8_t* survive; int* status;
  Counters* cnt;
  int dmax;
};

// ilogb of a finite non-zero double on the integer pipe (subnormals take the library path)
__device__ __forceinline__ int ilogb_fast(double v) {
  const int ex = (__double2hiint(v) >> 20) & 0x7ff;
  return ex ? ex - 1023 : ilogb(v);
}

template <int G>
__device__ __forceinline__ unsigned group_mask(int lane) {
  if constexpr (G == 32) return 0xffffffffu;
  else return ((1u << G) - 1u) << (lane & ~(G - 1));
}

__host__ __device__ inline size_t small_group_bytes(int Q, int dmax, int es) {
  // X ping-pong + per-q0 terms (re, im, lg as doubles; e as long long) + per-q0 ints (c, r, qstart)
  size_t b = (size_t)2 * dmax * dmax * es * 8 + (size_t)Q * (8 * 4) + (size_t)Q * 4 * 3;
  return (b + 15) / 16 * 16;
}
__host__ __device__ inline size_t small_common_bytes(int Q, int A, int nb, int pack_len, int n_energy, int es) {
  size_t b = ((size_t)pack_len * es * 8 + (size_t)n_energy * 8 + (size_t)Q * 8 + 15) / 16 * 16;   // doubles, then 16-byte aligned
  b += (size_t)nb * 16 + (size_t)Q * 4 * 2 + (size_t)A * Q * 2;
  return (b + 15) / 16 * 16;
}

template <bool CPLX, int G>
__global__ void __launch_bounds__(256) small_trace_kernel(SmallParams P) {
  constexpr int ES = CPLX ? 2 : 1;
  extern __shared__ __align__(16) unsigned char ssm[];
  const int Q = P.imp.Q, A = P.imp.A;
  // ---- shared copies of the impurity
  double* s_pack = reinterpret_cast<double*>(ssm);
  double* s_energy = s_pack + (size_t)P.pack_len * ES;
  double* s_emin = s_energy + P.n_energy;
  int4* s_blk = reinterpret_cast<int4*>(ssm + ((size_t)(P.pack_len * ES + P.n_energy + Q) * 8 + 15) / 16 * 16);
  int* s_dim = reinterpret_cast<int*>(s_blk + P.n_blocks);
  int* s_eoff = s_dim + Q;
  short* s_blkof = reinterpret_cast<short*>(s_eoff + Q);
  unsigned char* s_groups = ssm + small_common_bytes(Q, A, P.n_blocks, P.pack_len, P.n_energy, ES);
  for (int i = threadIdx.x; i < P.pack_len * ES; i += blockDim.x) s_pack[i] = P.pack[i];
  for (int i = threadIdx.x; i < P.n_energy; i += blockDim.x) s_energy[i] = P.imp.energy[i];
  for (int i = threadIdx.x; i < Q; i += blockDim.x) { s_emin[i] = P.imp.e_min[i]; s_dim[i] = P.imp.dim[i]; s_eoff[i] = (int)P.imp.e_off[i]; }
  for (int i = threadIdx.x; i < P.n_blocks; i += blockDim.x) s_blk[i] = P.pblk[i];
  for (int i = threadIdx.x; i < A * Q; i += blockDim.x) s_blkof[i] = (short)P.imp.blk_of[i];
  __syncthreads();

  const int lane = threadIdx.x & 31, lg = lane & (G - 1);
  const unsigned mask = group_mask<G>(lane);
  const int grp_in_cta = threadIdx.x / G;
  const size_t gbytes = small_group_bytes(Q, P.dmax, ES);
  double* Xa = reinterpret_cast<double*>(s_groups + (size_t)grp_in_cta * gbytes);
  double* Xb = Xa + (size_t)P.dmax * P.dmax * ES;
  double* t_re = Xb + (size_t)P.dmax * P.dmax * ES;
  double* t_im = t_re + Q;
  double* t_lg = t_im + Q;
  long long* t_e = reinterpret_cast<long long*>(t_lg + Q);
  int* s_c = reinterpret_cast<int*>(t_e + Q);   // columns carried, 0 = no chain to multiply, -1 = does not survive
  int* s_r = s_c + Q;
  int* s_qs = s_r + Q;

  const long long n_groups = (long long)gridDim.x * (blockDim.x / G);
  unsigned long long st_strings = 0, st_flops = 0, st_exp = 0;
  for (long long b = (long long)blockIdx.x * (blockDim.x / G) + grp_in_cta; b < P.bv.B; b += n_groups) {
    const long long lo = P.bv.offset[b];
    const long long hi_off = P.bv.offset[b + 1];
    const bool off_ok = lo >= 0 && hi_off >= lo && hi_off <= P.bv.n_ops && hi_off - lo <= (long long)P.bv.max_len;
    const int L = off_ok ? (int)(hi_off - lo) : 0;   // corrupt offsets: status 2, and no read through them
    const int* sym = P.bv.symbol + lo;
    const double* tau = P.bv.tau + lo;
    const double beta = P.bv.beta;

    // ---- validation (reading A7): symbols in range, tau non-decreasing in [0, beta)
    bool ok = off_ok;
    for (int i = lg; i < L; i += G) {
      const int a = sym[i];
      const double t = tau[i];
      const double prev = i ? tau[i - 1] : 0.0;
      ok = ok && (a >= 0) && (a < A) && (t >= prev) && (t < beta);
    }
    ok = __all_sync(mask, ok);
    if (!ok) {
      if (lg == 0) {
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        P.mant[2 * b] = nan; P.mant[2 * b + 1] = nan; P.exp2[b] = 0; P.status[b] = 2;
      }
      if (P.survive) for (int q0 = lg; q0 < Q; q0 += G) P.survive[b * Q + q0] = 0;
      continue;
    }

    // ---- routing (a2): one start sector per lane
    bool any_surv = false;
    for (int q0 = lg; q0 < Q; q0 += G) {
      int q = q0, d = s_dim[q0], dmin = d, rpos = 0, qmin = q0;
      double lgv = 0.0;
      bool alive = true;
      const double t0 = L ? tau[0] : 0.0;
      double tcur = t0;
      for (int i = 0; i < L; ++i) {
        const int blk = s_blkof[sym[i] * Q + q];
        if (blk < 0) { alive = false; break; }
        const int qn = s_blk[blk].w;
        const int dn = s_dim[qn];
        const double tnext = (i + 1 < L) ? tau[i + 1] : beta + t0;
        lgv -= (tnext - tcur) * s_emin[qn] * kLog2e;
        tcur = tnext;
        if (i + 1 < L && dn < dmin) { dmin = dn; rpos = i + 1; qmin = qn; }
        q = qn;
      }
      if (L == 0) lgv = -beta * s_emin[q0] * kLog2e;
      int c = -1;
      if (alive) {
        c = 0;
        if (q == q0) {   // a survivor that does not return to q0 contributes nothing (:532)
          if (P.literal) { c = s_dim[q0]; s_r[q0] = 0; s_qs[q0] = q0; }
          else { c = dmin; s_r[q0] = rpos; s_qs[q0] = qmin; }
        }
      }
      s_c[q0] = c; t_lg[q0] = lgv;
      t_re[q0] = 0.0; t_im[q0] = 0.0; t_e[q0] = 0;
      if (P.survive) P.survive[b * Q + q0] = alive ? 1 : 0;
      any_surv = any_surv || alive;
    }
    any_surv = __any_sync(mask, any_surv);
    __syncwarp(mask);

    // ---- chains of the surviving start sectors (a3, a4, a5)
    for (int q0 = 0; q0 < Q; ++q0) {
      const int c = s_c[q0];
      if (c <= 0) continue;
      int q = s_qs[q0];
      const int r = s_r[q0];
      double* X = Xa;
      double* Xn = Xb;
      double re = 0.0, im = 0.0;
      long long e2 = 0;
      bool dead = false;
      if (L == 0) {   // empty configuration: Tr P_beta(q0) (reading A7)
        for (int n = lg; n < c; n += G) re += exp(-beta * (s_energy[s_eoff[q] + n] - s_emin[q]));
      } else {
        for (int e = lg; e < c * c; e += G) {
          const int m = e / c, n = e - m * c;
          X[e * ES] = (m == n) ? 1.0 : 0.0;
          if constexpr (CPLX) X[e * ES + 1] = 0.0;
        }
        __syncwarp(mask);
        int d = c;
        unsigned long long macs = 0, nexp = 0;
        const int m_first = lg / c, n_first = lg - m_first * c;   // c is fixed along the chain
        for (int j = 0; j < L; ++j) {
          int i = r + j;
          if (i >= L) i -= L;
          const int4 bd = s_blk[s_blkof[__ldg(sym + i) * Q + q]];
          const int dn = bd.y, qn = bd.w;
          const double delta = (i + 1 < L) ? (__ldg(tau + i + 1) - __ldg(tau + i)) : (beta - __ldg(tau + i) + __ldg(tau));
          const double* F = s_pack + (size_t)bd.x * ES;
          const double* E = s_energy + s_eoff[qn];
          const double emin = s_emin[qn];
          const int nel = dn * c;
          int wexp = INT_MIN, kr0 = 0;
          for (int e = lg; e < nel; e += G) {
            int m = m_first, n = n_first;
            if (e != lg) { m = e / c; n = e - m * c; }
            const double x = prop_x(delta, E[m], emin);
            const double kf = floor(x);
            const double mr = exp2(__dsub_rn(x, kf));
            const int kr = row_exp(x);
            if (e == lg) kr0 = kr;
            const double* Fr = F + (size_t)m * d * ES;
            if constexpr (CPLX) {
              double ar = 0.0, ai = 0.0;
              for (int k = 0; k < d; ++k) {
                const double fr = Fr[2 * k], fi = Fr[2 * k + 1];
                const double xr = X[(k * c + n) * 2], xi = X[(k * c + n) * 2 + 1];
                ar = fma(fr, xr, ar); ar = fma(-fi, xi, ar);
                ai = fma(fr, xi, ai); ai = fma(fi, xr, ai);
              }
              ar *= mr; ai *= mr;
              Xn[e * 2] = ar; Xn[e * 2 + 1] = ai;
              const double mx = fmax(fabs(ar), fabs(ai));
              if (mx > 0.0) wexp = max(wexp, kr + ilogb_fast(mx));
            } else {
              double acc = 0.0;
              const double* Xc = X + n;
#pragma unroll 3
              for (int k = 0; k < d; ++k) acc = fma(Fr[k], Xc[k * c], acc);
              acc *= mr;
              Xn[e] = acc;
              if (acc != 0.0) wexp = max(wexp, kr + ilogb_fast(acc));
            }
          }
          const int kmax = __reduce_max_sync(mask, wexp);
          if (kmax == INT_MIN) { dead = true; break; }
          e2 += kmax;
          for (int e = lg; e < nel; e += G) {
            const int sh = ((e == lg) ? kr0 : row_exp(prop_x(delta, E[e / c], emin))) - kmax;
            if (sh > 1022 || sh < -1022) {
              Xn[e * ES] = scalbn(Xn[e * ES], max(sh, -2200));
              if constexpr (CPLX) Xn[e * ES + 1] = scalbn(Xn[e * ES + 1], max(sh, -2200));
            } else {
              const double f = pow2i(sh);
              Xn[e * ES] *= f;
              if constexpr (CPLX) Xn[e * ES + 1] *= f;
            }
          }
          __syncwarp(mask);
          double* tmp = X; X = Xn; Xn = tmp;
          macs += (unsigned long long)dn * d;
          nexp += (unsigned long long)dn;
          q = qn; d = dn;
        }
        if (!dead)
          for (int n = lg; n < c; n += G) { re += X[(n * c + n) * ES]; if constexpr (CPLX) im += X[(n * c + n) * ES + 1]; }
        if (lg == 0) { st_strings += 1; st_flops += macs * (unsigned long long)c * (CPLX ? 8ull : 2ull); st_exp += nexp; }
        __syncwarp(mask);
      }
#pragma unroll
      for (int o = G / 2; o > 0; o >>= 1) { re += __shfl_xor_sync(mask, re, o); im += __shfl_xor_sync(mask, im, o); }
      if (lg == 0) { t_re[q0] = dead ? 0.0 : re; t_im[q0] = dead ? 0.0 : im; t_e[q0] = dead ? 0 : e2; }
    }
    __syncwarp(mask);

    // ---- sector sum with exponent alignment (a5): q0 ascending, Neumaier-compensated, normalised to [1, 2)
    if (lg == 0) {
      bool any_nz = false;
      long long emax = 0;
      for (int q0 = 0; q0 < Q; ++q0) {
        if (s_c[q0] <= 0) continue;
        const double kf = floor(t_lg[q0]);
        const double f = exp2(t_lg[q0] - kf);
        const double mx = fmax(fabs(t_re[q0]), fabs(t_im[q0])) * f;
        if (mx > 0.0) {
          const long long e = t_e[q0] + (long long)kf + ilogb(mx);
          emax = any_nz ? max(emax, e) : e;
          any_nz = true;
        }
      }
      double re = 0.0, im = 0.0, cre = 0.0, cim = 0.0;
      if (any_nz) {
        for (int q0 = 0; q0 < Q; ++q0) {
          if (s_c[q0] <= 0) continue;
          const double kf = floor(t_lg[q0]);
          const double f = exp2(t_lg[q0] - kf);
          long long sh = t_e[q0] + (long long)kf - emax;
          double xr = 0.0, xi = 0.0;
          if (sh >= -1100) { if (sh > 1000) sh = 1000; xr = scalbn(t_re[q0] * f, (int)sh); xi = scalbn(t_im[q0] * f, (int)sh); }
          const double tr = re + xr; cre += (fabs(re) >= fabs(xr)) ? (re - tr) + xr : (xr - tr) + re; re = tr;
          const double ti = im + xi; cim += (fabs(im) >= fabs(xi)) ? (im - ti) + xi : (xi - ti) + im; im = ti;
        }
        re += cre; im += cim;
      }
      const double mx = fmax(fabs(re), fabs(im));
      if (mx > 0.0) {
        const int k = ilogb(mx);
        P.mant[2 * b] = scalbn(re, -k); P.mant[2 * b + 1] = scalbn(im, -k); P.exp2[b] = emax + k;
      } else {
        P.mant[2 * b] = 0.0; P.mant[2 * b + 1] = 0.0; P.exp2[b] = 0;
      }
      P.status[b] = any_surv ? 0 : 1;
    }
    __syncwarp(mask);
  }
  if (lg == 0 && st_strings) {
    atomicAdd(&P.cnt->n_strings, st_strings);
    atomicAdd(&P.cnt->n_slots, st_strings);
    atomicAdd(&P.cnt->alg_flops, st_flops);
    atomicAdd(&P.cnt->macs, st_flops / 2);
    atomicAdd(&P.cnt->n_exp, st_exp);
  }
}

}  // namespace ctqmc
