// Lazy-trace bounds with segment length 1 for small real impurities, in ONE launch (PAPER.md:542-548
// "it is typically much faster to compute these bounds"): validation, routing and, per surviving start sector, the product
// of the factor norms from tables held in shared memory -- no matrix is ever multiplied:
//   Frobenius  ||P_Delta(q') F||_F^2 = sum_m p_m^2 r_m,  r_m = sum_k |F_mk|^2 (row-norm table), p_m = exp(-Delta (E_m - Emin))
//   spectral   ||P_Delta(q') F||_2  <= exp(-Delta Emin(q')) sigma_max(F)
// Same lane layout as chain_small2.cuh (DP lanes per configuration, lane = row), same formulas as bound_s1_kernel.
#pragma once
#include "chain_small2.cuh"
#include "reduce.cuh"

namespace ctqmc {

struct Small2BoundParams {
  DevImp imp;
  BatchView bv;
  const int2* binfo;        // [n_blocks] {dst sector, rows << 16 | cols}
  int n_blocks;
  int norm_kind;
  double* bound_mant; long long* bound_exp2;
  double* sector_mant; long long* sector_exp2;   // [B][Q] or null
  int* status;
};

__host__ __device__ inline size_t small2b_common_bytes(int Q, int A, int nb, int DP) {
  size_t b = ((size_t)nb * DP * 8 + (size_t)nb * 8 + (size_t)Q * DP * 8 + (size_t)Q * 8 + 15) / 16 * 16;
  b += (size_t)nb * 8 + (size_t)Q * 4 + (size_t)A * Q * 2;
  return (b + 15) / 16 * 16;
}
__host__ __device__ inline size_t small2b_group_bytes(int Q, int DP) {
  size_t b = (size_t)2 * DP * 8 + (size_t)Q * (8 * 3) + (size_t)Q * 4 * 2 + 16;
  return (b + 15) / 16 * 16;
}

template <int DP>
__global__ void __launch_bounds__(512) small2_bound_kernel(Small2BoundParams P) {
  constexpr int GPW = 32 / DP;
  extern __shared__ __align__(16) unsigned char ssb[];
  const int Q = P.imp.Q, A = P.imp.A, nb = P.n_blocks;
  double* s_rn = reinterpret_cast<double*>(ssb);        // [nb][DP] row-norm^2, zero on padded rows
  double* s_sigma = s_rn + (size_t)nb * DP;             // [nb]
  double* s_de = s_sigma + nb;                          // [Q][DP]
  double* s_emin = s_de + (size_t)Q * DP;
  int2* s_binfo = reinterpret_cast<int2*>(ssb + ((size_t)(nb * DP + nb + Q * DP + Q) * 8 + 15) / 16 * 16);
  int* s_dim = reinterpret_cast<int*>(s_binfo + nb);
  short* s_blkof = reinterpret_cast<short*>(s_dim + Q);
  unsigned char* s_groups = ssb + small2b_common_bytes(Q, A, nb, DP);
  for (int i = threadIdx.x; i < nb * DP; i += blockDim.x) {
    const int b = i / DP, m = i - b * DP;
    const BlkDesc bd = P.imp.blks[b];
    s_rn[i] = (m < bd.rows) ? P.imp.rownorm2[bd.rn_off + m] : 0.0;
  }
  for (int i = threadIdx.x; i < nb; i += blockDim.x) { s_sigma[i] = P.imp.sigma[i]; s_binfo[i] = P.binfo[i]; }
  for (int i = threadIdx.x; i < Q * DP; i += blockDim.x) {
    const int q = i / DP, r = i - q * DP;
    s_de[i] = (r < P.imp.dim[q]) ? __dsub_rn(P.imp.energy[P.imp.e_off[q] + r], P.imp.e_min[q]) : 0.0;
  }
  for (int i = threadIdx.x; i < Q; i += blockDim.x) { s_emin[i] = P.imp.e_min[i]; s_dim[i] = P.imp.dim[i]; }
  for (int i = threadIdx.x; i < A * Q; i += blockDim.x) s_blkof[i] = (short)P.imp.blk_of[i];
  __syncthreads();

  const int lane = threadIdx.x & 31, grp = lane / DP;
  if (grp >= GPW) return;
  const int lg = lane - grp * DP;
  const unsigned mask = ((1u << DP) - 1u) << (grp * DP);
  const int grp_in_cta = (threadIdx.x >> 5) * GPW + grp;
  const int groups_per_cta = (blockDim.x >> 5) * GPW;
  unsigned char* gb = s_groups + (size_t)grp_in_cta * small2b_group_bytes(Q, DP);
  double* scr_a = reinterpret_cast<double*>(gb);        // [DP] per-row scratch (max pass)
  double* scr_b = scr_a + DP;                           // [DP] per-row scratch (sum pass)
  double* t_m = scr_b + DP;                             // [Q] per-sector bound mantissa
  double* t_lg = t_m + Q;                               // [Q] real exponent from routing
  long long* t_e = reinterpret_cast<long long*>(t_lg + Q);
  int* s_dmin = reinterpret_cast<int*>(t_e + Q);        // [Q] smallest dimension along the string, 0 = does not survive
  int* s_sv = s_dmin + Q;                               // [Q + 1] survivors, count

  const long long n_groups = (long long)gridDim.x * groups_per_cta;
  for (long long b = (long long)blockIdx.x * groups_per_cta + grp_in_cta; b < P.bv.B; b += n_groups) {
    const long long lo = P.bv.offset[b];
    const long long hi_off = P.bv.offset[b + 1];
    const bool off_ok = lo >= 0 && hi_off >= lo && hi_off <= P.bv.n_ops && hi_off - lo <= (long long)P.bv.max_len;
    const int L = off_ok ? (int)(hi_off - lo) : 0;   // corrupt offsets: status 2, and no read through them
    const int* sym = P.bv.symbol + lo;
    const double* tau = P.bv.tau + lo;
    const double beta = P.bv.beta;
    const double nan = __longlong_as_double(0x7ff8000000000000LL);

    bool ok = off_ok;
    for (int i = lg; i < L; i += DP) {
      const int a = __ldg(sym + i);
      const double t = __ldg(tau + i);
      const double prev = i ? __ldg(tau + i - 1) : 0.0;
      ok = ok && (a >= 0) && (a < A) && (t >= prev) && (t < beta);
    }
    ok = __all_sync(mask, ok);
    if (!ok) {
      if (lg == 0) { P.bound_mant[b] = nan; P.bound_exp2[b] = 0; P.status[b] = 2; }
      if (P.sector_mant) for (int q0 = lg; q0 < Q; q0 += DP) { P.sector_mant[b * Q + q0] = nan; P.sector_exp2[b * Q + q0] = 0; }
      continue;
    }

    // ---- routing: survive, d_min, real exponent lg = -sum_i Delta_i Emin(q_i) log2 e (cyclic time differences)
    for (int q0 = lg; q0 < Q; q0 += DP) {
      int q = q0, dmin = s_dim[q0];
      double lgv = 0.0;
      bool alive = true;
      const double t0 = L ? __ldg(tau) : 0.0;
      double tcur = t0;
      int sym_nx = L ? __ldg(sym) : 0;
      double tau_nx = (L > 1) ? __ldg(tau + 1) : 0.0;
      for (int i = 0; i < L; ++i) {
        const int sym_c = sym_nx;
        const double tau_c1 = tau_nx;
        if (i + 1 < L) sym_nx = __ldg(sym + i + 1);
        if (i + 2 < L) tau_nx = __ldg(tau + i + 2);
        const int blk = s_blkof[sym_c * Q + q];
        if (blk < 0) { alive = false; break; }
        const int qn = s_binfo[blk].x;
        const double tnext = (i + 1 < L) ? tau_c1 : beta + t0;
        lgv -= (tnext - tcur) * s_emin[qn] * kLog2e;
        tcur = tnext;
        if (i + 1 < L) dmin = min(dmin, s_dim[qn]);
        q = qn;
      }
      if (L == 0) lgv = -beta * s_emin[q0] * kLog2e;
      s_dmin[q0] = alive ? dmin : 0;
      t_lg[q0] = lgv; t_m[q0] = 0.0; t_e[q0] = 0;
    }
    __syncwarp(mask);
    if (lg == 0) {
      int ns = 0;
      for (int q0 = 0; q0 < Q; ++q0) if (s_dmin[q0] > 0) s_sv[ns++] = q0;
      s_sv[Q] = ns;
    }
    __syncwarp(mask);
    const int n_surv = s_sv[Q];

    // ---- per surviving start sector: product of the factor norms (lane = row of the destination sector)
    for (int si = 0; si < n_surv; ++si) {
      const int q0 = s_sv[si];
      const int dmin = s_dmin[q0];
      double val = P.norm_kind == 0 ? sqrt((double)dmin) : (double)dmin;
      long long e = 0;
      double lgx = 0.0;
      int q = q0;
      if (L == 0) {
        if (P.norm_kind == 0) {
          const double p = (lg < s_dim[q0]) ? exp(-beta * s_de[q0 * DP + lg]) : 0.0;
          scr_b[lg] = p * p;
          __syncwarp(mask);
          double ss = 0.0;
#pragma unroll
          for (int m = 0; m < DP; ++m) ss += scr_b[m];
          val *= sqrt(ss);
          __syncwarp(mask);
        }
      } else {
        int sym_nx = __ldg(sym);
        double ta_nx = __ldg(tau), tb_nx = __ldg(tau + ((1 < L) ? 1 : 0));
        for (int i = 0; i < L; ++i) {
          const int sym_c = sym_nx;
          const double ta = ta_nx, tb = tb_nx;
          const bool wrap = i + 1 >= L;
          const int i2 = wrap ? 0 : i + 1;
          sym_nx = __ldg(sym + i2);
          ta_nx = __ldg(tau + i2); tb_nx = __ldg(tau + ((i2 + 1 < L) ? i2 + 1 : 0));
          const int blk = s_blkof[sym_c * Q + q];
          const int qn = s_binfo[blk].x;
          if (P.norm_kind == 1) {
            val *= s_sigma[blk];
          } else {
            const double delta = wrap ? (beta - ta + tb) : (tb - ta);
            const double rn = s_rn[blk * DP + lg];
            const double x = __dmul_rn(__dmul_rn(-delta, s_de[qn * DP + lg]), kLog2e);
            scr_a[lg] = (rn > 0.0) ? x : -INFINITY;
            __syncwarp(mask);
            double xmax = -INFINITY;
#pragma unroll
            for (int m = 0; m < DP; ++m) xmax = fmax(xmax, scr_a[m]);
            if (xmax == -INFINITY) {
              val = 0.0;
            } else {
              scr_b[lg] = (rn > 0.0) ? exp2(2.0 * (x - xmax)) * rn : 0.0;
              __syncwarp(mask);
              double ss = 0.0;
#pragma unroll
              for (int m = 0; m < DP; ++m) ss += scr_b[m];
              val *= sqrt(ss);
              lgx += xmax;
            }
            __syncwarp(mask);
          }
          if (val != 0.0) { const int k = ilogb(val); val = scalbn(val, -k); e += k; }
          q = qn;
        }
      }
      if (lg == 0) {
        const Scaled sb = finish_sector_bound(val, e, t_lg[q0] + lgx);
        t_m[q0] = sb.m; t_e[q0] = sb.e;
      }
    }
    __syncwarp(mask);

    // ---- sum over start sectors with exponent alignment, rounded outward (same as bound_reduce_kernel)
    if (P.sector_mant)
      for (int q0 = lg; q0 < Q; q0 += DP) { P.sector_mant[b * Q + q0] = t_m[q0]; P.sector_exp2[b * Q + q0] = t_e[q0]; }
    if (lg == 0) {
      bool any_nz = false;
      long long emax = 0;
      for (int q0 = 0; q0 < Q; ++q0)
        if (s_dmin[q0] > 0 && t_m[q0] > 0.0) { emax = any_nz ? max(emax, t_e[q0]) : t_e[q0]; any_nz = true; }
      double sum = 0.0;
      if (any_nz)
        for (int q0 = 0; q0 < Q; ++q0)
          if (s_dmin[q0] > 0) sum += shift_clamped(t_m[q0], t_e[q0] - emax);
      sum *= (1.0 + 2.220446049250313e-16 * 2.0 * Q);
      const Scaled r = normalize(sum, emax);
      P.bound_mant[b] = (sum > 0.0) ? r.m : 0.0;
      P.bound_exp2[b] = (sum > 0.0) ? r.e : 0;
      P.status[b] = n_surv > 0 ? 0 : 1;
    }
    __syncwarp(mask);
  }
}

}  // namespace ctqmc
