// Accumulation of the reduced density matrix of the impurity over a batch of configurations (
// PAPER.md:254 Eq. 27 with the tau integral done analytically, :572 "matrix addition" kernel):
//
//     rho_uv += weight_b / beta * int_0^beta w_loc(C_b, |v><u|(tau)) / w_loc(C_b) dtau          for every configuration b.
//
// Per surviving closed string (start sector q0), with the cyclic factors A_i = P_{Delta_i}(q_i) F_i (reading A2):
//     G_i = F_i A_{i-1} ... A_1 (forward sweep, every G_i kept),   Y_i = A_L ... A_{i+1} (backward sweep),
//     rho(q_i)_uv += K_i(u, v) (G_i Y_i)_uv / (beta w_loc),   K_i(u, v) = int_0^Delta_i exp(-s E_u - (Delta_i - s) E_v) ds
//                                                                    = Delta exp(-Delta min(E_u, E_v)) phi(Delta |E_u - E_v|).
// One persistent CTA per scratch slot walks the strings it is dealt; products run on the FP64 tensor cores through the node-
// product tile of lazy.cuh (bounds-guarded, any sector dimension up to 512); exponents as everywhere else (mantissa / row
// exponent split of the propagator, running integer exponents of X and Y, real exponent lg for exp(-Delta Emin)).  The sum
// into rho is the paper's matrix addition: atomicAdd, several strings may hit the same block.
#pragma once
#include "lazy.cuh"

namespace ctqmc {

constexpr int kDnMaxQ = 1024;      // sectors the hand-out order is built for (more: configuration-major order)

struct DensityParams {
  DevImp imp;
  BatchView bv;
  const double* w_mant; const long long* w_exp2; const int* status;   // of the same batch, from ctqmc_trace_batch
  const double* weight;          // [B] or null
  double* rho;                   // sum_q dim_q^2 elements, sector q at rho_off[q], column-major (u + v dim_q)
  const long long* rho_off;      // [Q]
  double* scratch;               // per CTA: slot_doubles
  long long slot_doubles;
  int ldm;                       // leading dimension of every scratch matrix (= d_max)
  int Lcap;                      // steps a slot can hold (= max_len)
  int* work;                     // next (configuration, start sector) candidate to hand out; zeroed before the launch
};

__host__ __device__ inline long long density_slot_doubles(int dmax, int Lcap, int es) {
  const long long mat = (long long)dmax * dmax * es;
  return (long long)Lcap * mat + 5 * mat + 2LL * (Lcap + 2);      // G_i, X ping-pong, Y ping-pong, C, exponents + sectors
}

// dst = diag(2^x) src brought to a common exponent (reading A5); returns that exponent (INT_MIN: src vanishes).  The mantissa and
// the exponent of every row's propagator factor are computed once per row into `rowm` / `rowk` (shared memory, >= rows entries:
// the kernel lends the operand stage of its product tile), and the scaling pass keeps four loads in flight per thread (a
// load-scale-store loop is serialised by the possible aliasing of its stores with the next load).
template <bool CPLX>
__device__ int dn_propagate(const double* src, double* dst, int ld, int rows, int cols, double delta, const double* E, double emin,
                            int* redi, double* rowm, int* rowk) {
  constexpr int ES = CPLX ? 2 : 1;
  const int n = rows * cols;
  if (n <= (int)blockDim.x) {          // small impurities: one element per thread, nothing to amortise
    const int r = threadIdx.x % rows, c = threadIdx.x / rows;
    const bool on = (int)threadIdx.x < n;
    double vr = 0.0, vi = 0.0, m = 1.0;
    int kr = 0, km = INT_MIN;
    if (on) {
      const double* p = src + ((long long)c * ld + r) * ES;
      vr = p[0]; if (CPLX) vi = p[1];
      const double x = prop_x(delta, E[r], emin);
      m = exp2(__dsub_rn(x, floor(x))); kr = row_exp(x);
      const double mx = CPLX ? fmax(fabs(vr), fabs(vi)) : fabs(vr);
      if (mx > 0.0) km = kr + ilogb(mx * m);
    }
    km = lz_block_max(km, redi);
    const int k = km == INT_MIN ? 0 : km;
    if (on) {
      double* o = dst + ((long long)c * ld + r) * ES;
      o[0] = lz_scale(vr * m, kr - k);
      if (CPLX) o[1] = lz_scale(vi * m, kr - k);
    }
    __syncthreads();
    return km;
  }
  __syncthreads();
  for (int r = threadIdx.x; r < rows; r += blockDim.x) {
    const double x = prop_x(delta, E[r], emin);
    rowm[r] = exp2(__dsub_rn(x, floor(x))); rowk[r] = row_exp(x);
  }
  __syncthreads();
  int km = INT_MIN;
  for (int idx = threadIdx.x; idx < n; idx += blockDim.x) {
    const int r = idx % rows, c = idx / rows;
    const double* p = src + ((long long)c * ld + r) * ES;
    const double mx = CPLX ? fmax(fabs(p[0]), fabs(p[1])) : fabs(p[0]);
    if (mx > 0.0) km = max(km, rowk[r] + ilogb(mx * rowm[r]));
  }
  km = lz_block_max(km, redi);
  const int k = km == INT_MIN ? 0 : km;
  constexpr int kBatch = 4;
  for (int idx0 = threadIdx.x; idx0 < n; idx0 += kBatch * blockDim.x) {
    double vr[kBatch], vi[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = idx0 + u * blockDim.x;
      vr[u] = 0.0; vi[u] = 0.0;
      if (idx < n) {
        const double* p = src + ((long long)(idx / rows) * ld + idx % rows) * ES;
        vr[u] = p[0]; if (CPLX) vi[u] = p[1];
      }
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = idx0 + u * blockDim.x;
      if (idx < n) {
        const int r = idx % rows;
        const int sh = rowk[r] - k;
        double* o = dst + ((long long)(idx / rows) * ld + r) * ES;
        o[0] = lz_scale(vr[u] * rowm[r], sh);
        if (CPLX) o[1] = lz_scale(vi[u] * rowm[r], sh);
      }
    }
  }
  __syncthreads();
  return km;
}

// in place: M <- M 2^-k
template <bool CPLX>
__device__ void dn_rescale(double* Mx, int ld, int rows, int cols, int k) {
  constexpr int ES = CPLX ? 2 : 1;
  const int n = rows * cols;
  constexpr int kBatch = 4;
  for (int idx0 = threadIdx.x; idx0 < n; idx0 += kBatch * blockDim.x) {
    double vr[kBatch], vi[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = idx0 + u * blockDim.x;
      vr[u] = 0.0; vi[u] = 0.0;
      if (idx < n) { const double* p = Mx + ((long long)(idx / rows) * ld + idx % rows) * ES; vr[u] = p[0]; if (CPLX) vi[u] = p[1]; }
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int idx = idx0 + u * blockDim.x;
      if (idx < n) {
        double* p = Mx + ((long long)(idx / rows) * ld + idx % rows) * ES;
        p[0] = lz_scale(vr[u], -k);
        if (CPLX) p[1] = lz_scale(vi[u], -k);
      }
    }
  }
  __syncthreads();
}

// C (M x N) = A B over all tiles of the CTA; *s_k receives the largest binary exponent of the result (INT_MIN: zero)
template <bool CPLX>
__device__ void dn_gemm(LzSmem<CPLX>& S, int M, int N, int K, const double* A, long long a_rs, long long a_cs, const double* B, int ldb, int b_ks,
                        double* Cm, int ldc, int* s_k) {
  if (threadIdx.x == 0) *s_k = INT_MIN;
  __syncthreads();
  LzDiag dg; dg.delta = 0.0; dg.E = nullptr; dg.emin = 0.0; dg.kmax = 0;
  LzRowScale rs; rs.on = 0; rs.delta = 0.0; rs.E = nullptr; rs.emin = 0.0;
  for (int m0 = 0; m0 < M; m0 += kLzTile)
    for (int n0 = 0; n0 < N; n0 += kLzTile) {
      lz_gemm_tile<CPLX>(S, m0, n0, M, N, K, A, a_rs, a_cs, B, ldb, dg, Cm, ldc, rs, s_k, b_ks);
      __syncthreads();
    }
  __threadfence_block();
  __syncthreads();
}

template <bool CPLX>
__global__ void __launch_bounds__(kLzThreads) density_kernel(DensityParams P) {
  constexpr int ES = CPLX ? 2 : 1;
  __shared__ LzSmem<CPLX> S;
  __shared__ int s_k, s_ok, redi[32];
  // per-row propagator factors of dn_propagate live in the operand stage of the product tile (idle between products):
  // kLzMaxDim doubles + kLzMaxDim ints = 6 KB of its 10 KB
  static_assert(sizeof(S.A[0]) >= kLzMaxDim * (sizeof(double) + sizeof(int)), "row table does not fit the operand stage");
  double* rowm = &S.A[0][0][0];
  int* rowk = reinterpret_cast<int*>(rowm + kLzMaxDim);
  const int Q = P.imp.Q, ld = P.ldm;
  const long long mat = (long long)ld * ld * ES;
  double* base = P.scratch + (size_t)blockIdx.x * P.slot_doubles;
  double* Gs = base;                                   // [Lcap] matrices G_i
  double* Xa = Gs + (long long)P.Lcap * mat; double* Xb = Xa + mat;
  double* Ya = Xb + mat; double* Yb = Ya + mat;
  double* Cb = Yb + mat;
  long long* eG = reinterpret_cast<long long*>(Cb + mat);          // [Lcap + 1]
  int* qs = reinterpret_cast<int*>(eG + P.Lcap + 1);               // [Lcap + 1] sectors q_0 .. q_L
  const long long nS = P.bv.B * Q;
  __shared__ int s_next;
  // start sectors in order of decreasing dimension (the cost of a string grows with the square of it): the heavy strings are
  // handed out first, the tail of the launch is made of light ones
  __shared__ short s_qord[kDnMaxQ];
  const bool ordered = Q <= kDnMaxQ;
  if (ordered) {
    for (int q = threadIdx.x; q < Q; q += blockDim.x) {
      const int d = P.imp.dim[q];
      int rank = 0;
      for (int p = 0; p < Q; ++p) { const int dp = P.imp.dim[p]; rank += (dp > d) || (dp == d && p < q); }
      s_qord[rank] = (short)q;
    }
  }
  // candidates are handed out one by one: few of them survive and close, and the survivors differ in length by an order of
  // magnitude -- with a fixed stride the SMs were busy a third of the launch (config 4, profiles/r02_density.md)
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) s_next = atomicAdd(P.work, 1);
    __syncthreads();
    const long long s = s_next;
    if (s >= nS) break;
    const long long b = ordered ? s % P.bv.B : s / Q;
    const int q0 = ordered ? (int)s_qord[s / P.bv.B] : (int)(s - b * Q);
    if (P.status[b] != 0) continue;
    const double wr = P.w_mant[2 * b], wi = P.w_mant[2 * b + 1];
    if ((wr == 0.0 && wi == 0.0) || !isfinite(wr) || !isfinite(wi)) continue;
    const long long we = P.w_exp2[b];
    const long long lo = P.bv.offset[b];
    const int L = (int)(P.bv.offset[b + 1] - lo);
    if (L > P.Lcap) continue;                                        // cannot happen for status 0 (max_len is checked by the trace call)
    const int* sym = P.bv.symbol + lo;
    const double* tau = P.bv.tau + lo;
    const double beta = P.bv.beta;
    const double wgt = (P.weight ? P.weight[b] : 1.0) / beta;
    const double wn = wr * wr + wi * wi;
    __syncthreads();
    if (threadIdx.x == 0) {                                          // sector walk (a2): the string must survive and close
      int q = q0, ok = 1;
      qs[0] = q0;
      for (int i = 0; i < L && ok; ++i) {
        const int blk = P.imp.blk_of[sym[i] * Q + q];
        if (blk < 0) ok = 0; else { q = P.imp.blks[blk].dst; qs[i + 1] = q; }
      }
      s_ok = ok && q == q0;
    }
    __syncthreads();
    if (!s_ok) continue;
    const int d0 = P.imp.dim[q0];
    double* rho0 = P.rho + P.rho_off[q0] * ES;
    if (L == 0) {                                                    // thermal state: rho_uu = exp(-beta E_u) / Z
      const double* E = P.imp.energy + P.imp.e_off[q0];
      const double emin = P.imp.e_min[q0];
      const LzC z = lz_apply_lg(1.0, 0.0, 0, -beta * emin * kLog2e);
      const double sc = lz_scale(z.re, (int)max(min(z.e - we, 2000LL), -2200LL)) * wgt * beta;
      for (int u = threadIdx.x; u < d0; u += blockDim.x) {
        const double v = exp(-beta * (E[u] - emin)) * sc;
        atomicAdd(rho0 + ((long long)u * d0 + u) * ES, v * wr / wn);
        if (CPLX) atomicAdd(rho0 + ((long long)u * d0 + u) * ES + 1, -v * wi / wn);
      }
      continue;
    }
    // ---- forward sweep: G_i = F_i X_{i-1} kept, X_i = P_{Delta_i} G_i
    for (int idx = threadIdx.x; idx < d0 * d0; idx += blockDim.x) {
      const int r = idx % d0, c = idx / d0;
      Xa[((long long)c * ld + r) * ES] = r == c ? 1.0 : 0.0;
      if (CPLX) Xa[((long long)c * ld + r) * ES + 1] = 0.0;
    }
    __syncthreads();
    double* X = Xa; double* Xn = Xb;
    long long ex = 0;
    double lg = 0.0;
    bool dead = false;
    for (int i = 0; i < L; ++i) {
      const BlkDesc bd = P.imp.blks[P.imp.blk_of[sym[i] * Q + qs[i]]];
      const int qn = bd.dst;
      const double delta = (i + 1 < L) ? (tau[i + 1] - tau[i]) : (beta - tau[i] + tau[0]);
      double* Gi = Gs + (long long)i * mat;
      dn_gemm<CPLX>(S, bd.rows, d0, bd.cols, P.imp.store + bd.off, bd.ld, 1, X, ld, 1, Gi, ld, &s_k);
      if (threadIdx.x == 0) eG[i] = ex;
      const int k = dn_propagate<CPLX>(Gi, Xn, ld, bd.rows, d0, delta, P.imp.energy + P.imp.e_off[qn], P.imp.e_min[qn], redi, rowm, rowk);
      if (k == INT_MIN) { dead = true; break; }
      ex += k;
      lg += -delta * P.imp.e_min[qn] * kLog2e;
      double* t = X; X = Xn; Xn = t;
    }
    if (dead) continue;
    // ---- backward sweep on Y^T (dim q_i x dim q_0): accumulate interval i, then Y_{i-1}^T = F_i^T (P_{Delta_i} Y_i^T)
    for (int idx = threadIdx.x; idx < d0 * d0; idx += blockDim.x) {
      const int r = idx % d0, c = idx / d0;
      Ya[((long long)c * ld + r) * ES] = r == c ? 1.0 : 0.0;
      if (CPLX) Ya[((long long)c * ld + r) * ES + 1] = 0.0;
    }
    __syncthreads();
    double* Y = Ya; double* Yn = Yb;
    long long ey = 0;
    for (int i = L - 1; i >= 0; --i) {
      const BlkDesc bd = P.imp.blks[P.imp.blk_of[sym[i] * Q + qs[i]]];
      const int qn = bd.dst, dn = bd.rows;
      const double delta = (i + 1 < L) ? (tau[i + 1] - tau[i]) : (beta - tau[i] + tau[0]);
      const double* E = P.imp.energy + P.imp.e_off[qn];
      const double emin = P.imp.e_min[qn];
      const double* Gi = Gs + (long long)i * mat;
      // C = G_i Y_i = G_i (Y^T)^T  (dim q_i x dim q_i)
      dn_gemm<CPLX>(S, dn, dn, d0, Gi, 1, ld, Y, 1, ld, Cb, ld, &s_k);
      const LzC z = lz_apply_lg(1.0, 0.0, eG[i] + ey, lg);
      const double sc = lz_scale(z.re, (int)max(min(z.e - we, 2000LL), -2200LL)) * wgt;
      double* rq = P.rho + P.rho_off[qn] * ES;
      for (int idx = threadIdx.x; idx < dn * dn; idx += blockDim.x) {
        const int u = idx % dn, v = idx / dn;
        const double du = E[u] - emin, dv = E[v] - emin;
        const double x = delta * fabs(du - dv);
        const double kf = delta * exp(-delta * fmin(du, dv)) * (x > 0.0 ? -expm1(-x) / x : 1.0) * sc;
        const double cr = Cb[((long long)v * ld + u) * ES] * kf, ci = CPLX ? Cb[((long long)v * ld + u) * ES + 1] * kf : 0.0;
        // divide by w_loc (complex)
        const double rr = (cr * wr + ci * wi) / wn, ri = (ci * wr - cr * wi) / wn;
        if (rr != 0.0) atomicAdd(rq + ((long long)v * dn + u) * ES, rr);
        if (CPLX && ri != 0.0) atomicAdd(rq + ((long long)v * dn + u) * ES + 1, ri);
      }
      __syncthreads();
      if (i == 0) break;
      const int k1 = dn_propagate<CPLX>(Y, Y, ld, dn, d0, delta, E, emin, redi, rowm, rowk);
      if (k1 == INT_MIN) break;                                     // nothing left to carry back
      ey += k1;
      // Y_{i-1}^T = F_i^T Y': F_i is row-major (dim q_i x dim q_{i-1}), its transpose has row stride 1 and column stride ld
      dn_gemm<CPLX>(S, bd.cols, d0, dn, P.imp.store + bd.off, 1, bd.ld, Y, ld, 1, Yn, ld, &s_k);
      const int k2 = s_k;
      __syncthreads();
      if (k2 == INT_MIN) break;
      dn_rescale<CPLX>(Yn, ld, bd.cols, d0, k2);
      ey += k2;
      double* t = Y; Y = Yn; Yn = t;
    }
  }
}

}  // namespace ctqmc
