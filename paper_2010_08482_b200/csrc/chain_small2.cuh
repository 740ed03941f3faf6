// Small-sector path, uniform variant (real impurities, all sectors <= 16 states): same single-launch fusion as
// chain_small.cuh (validation, routing a2, chain a3/a4, trace and sector sum a5), but instruction-lean:
//   * every sector is padded to DP states (DP = 2, 4, 6, 9, 12 or 16 >= d_max) and every operator block to DP x DP with
//     zeros, stored TRANSPOSED in shared memory, so a chain step is the same fully unrolled DP-term dot product for every
//     string whatever sectors it is in -- no data-dependent loop bounds, no index arithmetic;
//   * a group of DP lanes owns one configuration (lane = row of the carried matrix), 32/DP configurations per warp.
//   * small batches (P.split): the whole warp owns ONE configuration -- its 32/DP groups share validation and routing (start
//     sectors dealt over all lanes) and take the surviving start sectors' chains round-robin, so the latency of a launch is that of
//     a third (DP = 9) or an eighth (DP = 4) of one configuration's chains instead of all of them.
// Padded rows carry exact zeros (their operator rows are zero), so results are those of the unpadded product.
#pragma once
#include <climits>

#include "chain_large.cuh"
#include "chain_small.cuh"

namespace ctqmc {

// 2^f for f in [0, 1] as sqrt(2) exp((f - 1/2) ln 2), Taylor to degree 14 (|(f - 1/2) ln 2| <= 0.347: remainder 5e-18), Horner with
// the coefficients as constant-bank operands: 16 FP64 instructions.  The library's exp2 costs 45 on this path (range reduction
// for arbitrary arguments, 22 UMOV re-materialising its constants every step, a special-case branch).
__constant__ double kExp2Taylor[15] = {1.0, 0.6931471805599453, 0.24022650695910072, 0.05550410866482158, 0.009618129107628477,
                                       0.0013333558146428443, 0.0001540353039338161, 1.5252733804059841e-05, 1.321548679014431e-06,
                                       1.01780860092397e-07, 7.054911620801123e-09, 4.4455382718708116e-10, 2.5678435993488206e-11,
                                       1.3691488853904128e-12, 6.778726354822545e-14};
__device__ __forceinline__ double exp2_unit(double f) {
  const double t = f - 0.5;
  double p = kExp2Taylor[14];
#pragma unroll
  for (int k = 13; k >= 0; --k) p = fma(p, t, kExp2Taylor[k]);
  return p * 1.4142135623730951;
}

struct Small2Params {
  DevImp imp;
  BatchView bv;
  const double* ftpad;      // [n_blocks][DP][DP]: ftpad[b][k][r] = F_b[r][k], zero padded
  const int2* binfo;        // [n_blocks] {dst sector, rows << 16 | cols}
  int n_blocks;
  int literal;
  int split;                // 1: one warp per configuration (small batches), 0: one group of DP lanes per configuration
  double* mant; long long* exp2; uint8_t* survive; int* status;
  Counters* cnt;
};

__host__ __device__ inline size_t small2_common_bytes(int Q, int A, int nb, int DP) {
  size_t b = ((size_t)nb * DP * DP * 8 + (size_t)Q * DP * 8 + (size_t)Q * 8 + 15) / 16 * 16;
  b += (size_t)nb * 8 + (size_t)Q * 4 + (size_t)A * Q * 2;
  return (b + 15) / 16 * 16;
}
__host__ __device__ inline size_t small2_group_bytes(int Q, int DP) {
  size_t b = (size_t)2 * DP * DP * 8 + (size_t)Q * (8 * 3) + (size_t)Q * 4 * 4 + 16;
  return (b + 15) / 16 * 16;
}

// split mode: per warp, the carried matrices of its 32/DP groups and ONE set of per-configuration tables
__host__ __device__ inline size_t small2_warp_bytes(int Q, int DP) {
  size_t b = (size_t)(32 / DP) * 2 * DP * DP * 8 + (size_t)Q * (8 * 3) + (size_t)Q * 4 * 4 + 16;
  return (b + 15) / 16 * 16;
}

template <int DP>
__global__ void __launch_bounds__(512) small2_trace_kernel(Small2Params P) {
  constexpr int GPW = 32 / DP;                       // groups (configurations) per warp
  extern __shared__ __align__(16) unsigned char ssm2[];
  const int Q = P.imp.Q, A = P.imp.A, nb = P.n_blocks;
  double* s_ft = reinterpret_cast<double*>(ssm2);
  double* s_de = s_ft + (size_t)nb * DP * DP;        // [Q][DP]  E - Emin (0 on padded rows)
  double* s_emin = s_de + (size_t)Q * DP;
  int2* s_binfo = reinterpret_cast<int2*>(ssm2 + ((size_t)(nb * DP * DP + Q * DP + Q) * 8 + 15) / 16 * 16);
  int* s_dim = reinterpret_cast<int*>(s_binfo + nb);
  short* s_blkof = reinterpret_cast<short*>(s_dim + Q);
  unsigned char* s_groups = ssm2 + small2_common_bytes(Q, A, nb, DP);
  // operator store -> shared memory with 1-D bulk copies (cp.async.bulk) issued by one thread and awaited on an mbarrier: a plain
  // copy loop waits for every load before the next one (90 us of a 64-thread CTA's launch on config 2 with a cold L2; 8 loads in
  // flight per thread still left 23 us).  The odd last double, if any, is copied by hand.
  __shared__ __align__(8) unsigned long long fill_bar;
  const unsigned ft_bytes = (unsigned)((size_t)nb * DP * DP * 8), ft_bulk = ft_bytes & ~15u;
  if (threadIdx.x == 0) {
    mbar_init(&fill_bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    if (ft_bulk) {
      mbar_expect_tx(&fill_bar, ft_bulk);
      for (unsigned o = 0; o < ft_bulk; o += 32768u) {
        const unsigned n = ft_bulk - o < 32768u ? ft_bulk - o : 32768u;
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"(smem_u32(reinterpret_cast<unsigned char*>(s_ft) + o)), "l"(reinterpret_cast<const unsigned char*>(P.ftpad) + o), "r"(n),
                       "r"(smem_u32(&fill_bar)) : "memory");
      }
    }
    if (ft_bulk != ft_bytes) s_ft[nb * DP * DP - 1] = P.ftpad[nb * DP * DP - 1];
  }
  for (int i = threadIdx.x; i < Q * DP; i += blockDim.x) {
    const int q = i / DP, r = i - q * DP;
    s_de[i] = (r < P.imp.dim[q]) ? __dsub_rn(P.imp.energy[P.imp.e_off[q] + r], P.imp.e_min[q]) : 0.0;
  }
  for (int i = threadIdx.x; i < Q; i += blockDim.x) { s_emin[i] = P.imp.e_min[i]; s_dim[i] = P.imp.dim[i]; }
  for (int i = threadIdx.x; i < nb; i += blockDim.x) s_binfo[i] = P.binfo[i];
  for (int i = threadIdx.x; i < A * Q; i += blockDim.x) s_blkof[i] = (short)P.imp.blk_of[i];
  __syncthreads();                                   // fill_bar is initialised for everyone
  if (ft_bulk) mbar_wait(&fill_bar, 0);
  __syncthreads();

  const int lane = threadIdx.x & 31, grp = lane / DP;
  if (grp >= GPW) return;                            // spare lanes of the warp (32 is not a multiple of DP)
  const int lg = lane - grp * DP;
  const unsigned mask = (DP == 32 ? 0xffffffffu : ((1u << DP) - 1u)) << (grp * DP);
  const int grp_in_cta = (threadIdx.x >> 5) * GPW + grp;
  const size_t gbytes = small2_group_bytes(Q, DP);
  const bool split = P.split != 0;
  const size_t wbytes = small2_warp_bytes(Q, DP);
  double* Xa = split ? reinterpret_cast<double*>(s_groups + (size_t)(threadIdx.x >> 5) * wbytes) + (size_t)grp * 2 * DP * DP
                     : reinterpret_cast<double*>(s_groups + (size_t)grp_in_cta * gbytes);
  double* Xb = Xa + DP * DP;
  // the lanes that share a configuration: this group, or (split) every group of the warp; the per-configuration tables then live
  // once per warp (small2_warp_bytes)
  const int sub = split ? grp : 0, nsub = split ? GPW : 1;
  const int cl = sub * DP + lg, ncl = nsub * DP;
  const unsigned cmask = split ? ((GPW * DP == 32) ? 0xffffffffu : ((1u << (GPW * DP)) - 1u)) : mask;
  const int slot_in_cta = split ? (int)(threadIdx.x >> 5) : grp_in_cta;
  const int groups_per_cta = split ? (int)(blockDim.x >> 5) : (int)(blockDim.x >> 5) * GPW;      // configurations in flight per CTA
  double* t_re = split ? reinterpret_cast<double*>(s_groups + (size_t)(threadIdx.x >> 5) * wbytes) + (size_t)GPW * 2 * DP * DP
                       : reinterpret_cast<double*>(s_groups + (size_t)grp_in_cta * gbytes) + 2 * DP * DP;
  double* t_lg = t_re + Q;
  long long* t_e = reinterpret_cast<long long*>(t_lg + Q);
  int* s_c = reinterpret_cast<int*>(t_e + Q);
  int* s_r = s_c + Q;
  int* s_qs = s_r + Q;
  int* s_sv = s_qs + Q;   // [Q + 1]: start sectors with a chain to multiply, then their count

  const long long n_groups = (long long)gridDim.x * groups_per_cta;
  unsigned long long st_strings = 0, st_flops = 0, st_exp = 0, st_pmacs = 0;
  for (long long b = (long long)blockIdx.x * groups_per_cta + slot_in_cta; b < P.bv.B; b += n_groups) {
    const long long lo = P.bv.offset[b];
    const long long hi_off = P.bv.offset[b + 1];
    const bool off_ok = lo >= 0 && hi_off >= lo && hi_off <= P.bv.n_ops && hi_off - lo <= (long long)P.bv.max_len;
    const int L = off_ok ? (int)(hi_off - lo) : 0;   // corrupt offsets: status 2, and no read through them
    const int* sym = P.bv.symbol + lo;
    const double* tau = P.bv.tau + lo;
    const double beta = P.bv.beta;

    // ---- validation (reading A7)
    bool ok = off_ok;
    for (int i = cl; i < L; i += ncl) {
      const int a = __ldg(sym + i);
      const double t = __ldg(tau + i);
      const double prev = i ? __ldg(tau + i - 1) : 0.0;
      ok = ok && (a >= 0) && (a < A) && (t >= prev) && (t < beta);
    }
    ok = __all_sync(cmask, ok);
    if (!ok) {
      if (cl == 0) {
        const double nan = __longlong_as_double(0x7ff8000000000000LL);
        P.mant[2 * b] = nan; P.mant[2 * b + 1] = nan; P.exp2[b] = 0; P.status[b] = 2;
      }
      if (P.survive) for (int q0 = cl; q0 < Q; q0 += ncl) P.survive[b * Q + q0] = 0;
      continue;
    }

    // ---- routing (a2): start sectors dealt to the lanes that share the configuration, two independent walks per lane and pass
    //      (integer only: the exponent of exp(-Delta Emin) is summed by the chain pass, for the strings that have a chain)
    bool any_surv = false;
    for (int qa0 = cl; qa0 < Q; qa0 += 2 * ncl) {
      const int qb0 = qa0 + ncl;
      const bool has_b = qb0 < Q;
      int qa = qa0, qb = has_b ? qb0 : 0;
      int dmin_a = s_dim[qa0], dmin_b = s_dim[qb], rpos_a = 0, rpos_b = 0, qmin_a = qa0, qmin_b = qb;
      bool alive_a = true, alive_b = has_b;
      int sym_nx = L ? __ldg(sym) : 0;
      for (int i = 0; i < L; ++i) {
        const int sym_c = sym_nx;
        if (i + 1 < L) sym_nx = __ldg(sym + i + 1);
        if (alive_a) {
          const int blk = s_blkof[sym_c * Q + qa];
          if (blk < 0) alive_a = false;
          else {
            const int2 bi = s_binfo[blk];
            const int dn = bi.y >> 16;                        // rows of the block = dimension of its target sector
            if (i + 1 < L && dn < dmin_a) { dmin_a = dn; rpos_a = i + 1; qmin_a = bi.x; }
            qa = bi.x;
          }
        }
        if (alive_b) {
          const int blk = s_blkof[sym_c * Q + qb];
          if (blk < 0) alive_b = false;
          else {
            const int2 bi = s_binfo[blk];
            const int dn = bi.y >> 16;
            if (i + 1 < L && dn < dmin_b) { dmin_b = dn; rpos_b = i + 1; qmin_b = bi.x; }
            qb = bi.x;
          }
        }
        if (!alive_a && !alive_b) break;
      }
#pragma unroll
      for (int w = 0; w < 2; ++w) {
        if (w == 1 && !has_b) break;
        const int q0 = w ? qb0 : qa0, q = w ? qb : qa;
        const bool alive = w ? alive_b : alive_a;
        int c = -1;
        if (alive) {
          c = 0;
          if (q == q0) {
            if (P.literal) { c = s_dim[q0]; s_r[q0] = 0; s_qs[q0] = q0; }
            else { c = w ? dmin_b : dmin_a; s_r[q0] = w ? rpos_b : rpos_a; s_qs[q0] = w ? qmin_b : qmin_a; }
          }
        }
        s_c[q0] = c; t_lg[q0] = 0.0; t_re[q0] = 0.0; t_e[q0] = 0;
        if (P.survive) P.survive[b * Q + q0] = alive ? 1 : 0;
        any_surv = any_surv || alive;
      }
    }
    any_surv = __any_sync(cmask, any_surv);
    __syncwarp(cmask);
    if (cl == 0) {   // compact list of the start sectors that have a chain: every group of the warp then runs its
      int ns = 0;    // si-th chain at the same time (a `continue` over q0 would serialise the groups of a warp)
      for (int q0 = 0; q0 < Q; ++q0) if (s_c[q0] > 0) s_sv[ns++] = q0;
      s_sv[Q] = ns;
    }
    __syncwarp(cmask);
    const int n_chain = s_sv[Q];

    // ---- chains of the surviving start sectors (a3, a4, a5)
    for (int si = sub; si < n_chain; si += nsub) {
      const int q0 = s_sv[si];
      const int c = s_c[q0];
      int q = s_qs[q0];
      const int r = s_r[q0];
      double* X = Xa;      // X[n * DP + k]: column n of the carried matrix, padded rows are zero
      double* Xn = Xb;
      double tr = 0.0, lgv = 0.0;
      long long e2 = 0;
      bool dead = false;
      if (L == 0) {        // empty configuration: Tr P_beta(q0) (reading A7)
        if (lg == 0) for (int n = 0; n < c; ++n) tr += exp(-beta * s_de[q * DP + n]);
        lgv = -beta * s_emin[q0] * kLog2e;
      } else {
        for (int n = 0; n < c; ++n) X[n * DP + lg] = (lg == n) ? 1.0 : 0.0;
        __syncwarp(mask);
        unsigned long long macs = 0, nexp = 0;
        // One column (the string passes through a one-state sector: most strings of configs 1 and 2) has a loop of its own -- this
        // lane's entry stays in a register between the product and the rescale, 32-bit counters, one new tau per step -- taken when
        // every group that is at this point of the warp together with this one has one column too: groups on different loops would
        // run one after the other.  Both loops do the same arithmetic in the same order, so the choice never changes a result.
        const unsigned together = __activemask();
        if (__all_sync(together, c == 1)) {
          unsigned macs32 = 0, nexp32 = 0;
          int cur = r, nx = (r + 1 >= L) ? 0 : r + 1;         // this step's operator and the next one (cyclically)
          int sym_c = __ldg(sym + cur);
          double ta = __ldg(tau + cur), tb = __ldg(tau + nx);
          for (int j = 0; j < L; ++j) {
            const bool wrap = cur + 1 >= L;
            const double delta = wrap ? (beta - ta + tb) : (tb - ta);
            const int nn = (nx + 1 >= L) ? 0 : nx + 1;
            const int sym_n = __ldg(sym + nx);               // next step's operator, in flight during this step
            const double tb_n = __ldg(tau + nn);
            const int blk = s_blkof[sym_c * Q + q];
            const int2 bi = s_binfo[blk];
            const int qn = bi.x;
            lgv -= delta * s_emin[qn] * kLog2e;
            const double* ft = s_ft + (size_t)blk * (DP * DP) + lg;
            double a0 = 0.0, a1 = 0.0;
#pragma unroll
            for (int k = 0; k + 1 < DP; k += 2) { a0 = fma(ft[k * DP], X[k], a0); a1 = fma(ft[(k + 1) * DP], X[k + 1], a1); }
            if (DP & 1) a0 = fma(ft[(DP - 1) * DP], X[DP - 1], a0);
            const double x = __dmul_rn(__dmul_rn(-delta, s_de[qn * DP + lg]), kLog2e);
            const int kr = row_exp(x);
            double v = (a0 + a1) * exp2_unit(__dsub_rn(x, floor(x)));
            const int kmax = __reduce_max_sync(mask, v != 0.0 ? kr + ilogb_fast(v) : INT_MIN);
            if (kmax == INT_MIN) { dead = true; break; }
            e2 += kmax;
            const int sh = kr - kmax;
            v = (sh > 1022 || sh < -1022) ? scalbn(v, max(sh, -2200)) : v * pow2i(sh);
            Xn[lg] = v;
            __syncwarp(mask);
            double* tmp = X; X = Xn; Xn = tmp;
            macs32 += (unsigned)(bi.y >> 16) * (unsigned)(bi.y & 0xffff);
            nexp32 += (unsigned)(bi.y >> 16);
            q = qn;
            cur = nx; nx = nn; sym_c = sym_n; ta = tb; tb = tb_n;
          }
          macs = macs32; nexp = nexp32;
        } else {
          int i = r;
          int sym_nx = __ldg(sym + i);
          double ta_nx = __ldg(tau + i), tb_nx = __ldg(tau + ((i + 1 < L) ? i + 1 : 0));
          for (int j = 0; j < L; ++j) {
            const int sym_c = sym_nx;
            const double ta = ta_nx, tb = tb_nx;
            const bool wrap = i + 1 >= L;
            i = wrap ? 0 : i + 1;
            sym_nx = __ldg(sym + i);                     // next step's operator, in flight during this step
            ta_nx = __ldg(tau + i); tb_nx = __ldg(tau + ((i + 1 < L) ? i + 1 : 0));
            const int blk = s_blkof[sym_c * Q + q];
            const int2 bi = s_binfo[blk];
            const int qn = bi.x;
            const double delta = wrap ? (beta - ta + tb) : (tb - ta);
            lgv -= delta * s_emin[qn] * kLog2e;
            // this lane's row of F (transposed store: consecutive lanes read consecutive doubles)
            const double* ft = s_ft + (size_t)blk * (DP * DP) + lg;
            double f[DP];
  #pragma unroll
            for (int k = 0; k < DP; ++k) f[k] = ft[k * DP];
            // propagator of this row: 2^x = mantissa in [1, 2) times 2^kr  (prop_x with the pre-subtracted energy)
            const double x = __dmul_rn(__dmul_rn(-delta, s_de[qn * DP + lg]), kLog2e);
            const double mr = exp2_unit(__dsub_rn(x, floor(x)));
            const int kr = row_exp(x);
            int wexp = INT_MIN;
            for (int n = 0; n < c; ++n) {
              const double* xs = X + n * DP;
              double a0 = 0.0, a1 = 0.0;
  #pragma unroll
              for (int k = 0; k + 1 < DP; k += 2) { a0 = fma(f[k], xs[k], a0); a1 = fma(f[k + 1], xs[k + 1], a1); }
              if (DP & 1) a0 = fma(f[DP - 1], xs[DP - 1], a0);
              const double v = (a0 + a1) * mr;
              Xn[n * DP + lg] = v;
              if (v != 0.0) wexp = max(wexp, kr + ilogb_fast(v));
            }
            const int kmax = __reduce_max_sync(mask, wexp);
            if (kmax == INT_MIN) { dead = true; break; }
            e2 += kmax;
            const int sh = kr - kmax;
            if (sh > 1022 || sh < -1022) {
              for (int n = 0; n < c; ++n) Xn[n * DP + lg] = scalbn(Xn[n * DP + lg], max(sh, -2200));
            } else {
              const double sc = pow2i(sh);
              for (int n = 0; n < c; ++n) Xn[n * DP + lg] *= sc;
            }
            __syncwarp(mask);
            double* tmp = X; X = Xn; Xn = tmp;
            macs += (unsigned long long)(bi.y >> 16) * (unsigned long long)(bi.y & 0xffff);
            nexp += (unsigned long long)(bi.y >> 16);
            q = qn;
          }
        }
        if (lg == 0) {
          if (!dead) for (int n = 0; n < c; ++n) tr += X[n * DP + n];
          st_strings += 1; st_flops += macs * (unsigned long long)c * 2ull; st_exp += nexp;
          st_pmacs += (unsigned long long)L * (unsigned long long)(DP * DP * c);   // executed: every step multiplies the padded DP x DP block
        }
        __syncwarp(mask);
      }
      if (lg == 0) { t_re[q0] = dead ? 0.0 : tr; t_e[q0] = dead ? 0 : e2; t_lg[q0] = lgv; }
    }
    __syncwarp(cmask);

    // ---- sector sum with exponent alignment (a5): q0 ascending, Neumaier-compensated, normalised to [1, 2)
    if (cl == 0) {
      bool any_nz = false;
      long long emax = 0;
      for (int q0 = 0; q0 < Q; ++q0) {
        if (s_c[q0] <= 0) continue;
        const double kf = floor(t_lg[q0]);
        const double mx = fabs(t_re[q0]) * exp2(t_lg[q0] - kf);
        if (mx > 0.0) {
          const long long e = t_e[q0] + (long long)kf + ilogb(mx);
          emax = any_nz ? max(emax, e) : e;
          any_nz = true;
        }
      }
      double re = 0.0, cre = 0.0;
      if (any_nz) {
        for (int q0 = 0; q0 < Q; ++q0) {
          if (s_c[q0] <= 0) continue;
          const double kf = floor(t_lg[q0]);
          long long sh = t_e[q0] + (long long)kf - emax;
          double xr = 0.0;
          if (sh >= -1100) { if (sh > 1000) sh = 1000; xr = scalbn(t_re[q0] * exp2(t_lg[q0] - kf), (int)sh); }
          const double t2 = re + xr; cre += (fabs(re) >= fabs(xr)) ? (re - t2) + xr : (xr - t2) + re; re = t2;
        }
        re += cre;
      }
      if (re != 0.0) {
        const int k = ilogb(re);
        P.mant[2 * b] = scalbn(re, -k); P.mant[2 * b + 1] = 0.0; P.exp2[b] = emax + k;
      } else {
        P.mant[2 * b] = 0.0; P.mant[2 * b + 1] = 0.0; P.exp2[b] = 0;
      }
      P.status[b] = any_surv ? 0 : 1;
    }
    __syncwarp(cmask);
  }
  if (lg == 0 && st_strings) {
    atomicAdd(&P.cnt->n_strings, st_strings);
    atomicAdd(&P.cnt->n_slots, st_strings);
    atomicAdd(&P.cnt->alg_flops, st_flops);
    atomicAdd(&P.cnt->macs, st_pmacs);
    atomicAdd(&P.cnt->n_exp, st_exp);
  }
}

}  // namespace ctqmc
