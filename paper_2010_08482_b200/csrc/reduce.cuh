// Trace reduction with exponent alignment and the norm-product bounds (a6).
#pragma once
#include "common.cuh"

namespace ctqmc {

struct Scaled {   // value = m * 2^e
  double m;
  long long e;
};

__device__ __forceinline__ Scaled normalize(double m, long long e) {
  Scaled r;
  if (m == 0.0 || !isfinite(m)) { r.m = m; r.e = 0; return r; }
  int k = ilogb(m);
  r.m = scalbn(m, -k);
  r.e = e + k;
  return r;
}

__device__ __forceinline__ double shift_clamped(double v, long long sh) {
  if (sh < -1100) return 0.0;
  if (sh > 1000) sh = 1000;
  return scalbn(v, (int)sh);
}

struct TraceReduceParams {
  long long B;
  int Q;
  const int* status_in;
  const uint8_t* survive;
  const StringRec* strings;
  const Slot* slots;
  double* mant;        // [B][2]
  long long* exp2;     // [B]
  int* status;         // [B]
};

// One thread per configuration: w = sum over surviving start sectors and their panels of (re + i im) 2^(e2 + lg),
// aligned to the largest term, summed in a fixed order (q0 ascending, panels ascending) with Neumaier compensation,
// then normalised so that max(|re|, |im|) is in [1, 2).
__global__ void trace_reduce_kernel(TraceReduceParams P) {
  long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (b >= P.B) return;
  if (P.status_in[b] == 2) {
    P.mant[2 * b] = __longlong_as_double(0x7ff8000000000000LL);
    P.mant[2 * b + 1] = __longlong_as_double(0x7ff8000000000000LL);
    P.exp2[b] = 0;
    P.status[b] = 2;
    return;
  }
  bool any_surv = false, any_nz = false;
  long long emax = 0;
  for (int q0 = 0; q0 < P.Q; ++q0) {
    long long s = b * P.Q + q0;
    if (!P.survive[s]) continue;
    any_surv = true;
    const StringRec rec = P.strings[s];
    const double kf = floor(rec.lg);
    const double f = exp2(rec.lg - kf);
    for (int p = 0; p < rec.n_units; ++p) {
      const Slot sl = P.slots[rec.slot + p];
      const double mx = fmax(fabs(sl.re), fabs(sl.im)) * f;
      if (mx > 0.0) {
        long long e = sl.e2 + (long long)kf + ilogb(mx);
        emax = any_nz ? max(emax, e) : e;
        any_nz = true;
      }
    }
  }
  double re = 0.0, im = 0.0, cre = 0.0, cim = 0.0;
  if (any_nz) {
    for (int q0 = 0; q0 < P.Q; ++q0) {
      long long s = b * P.Q + q0;
      if (!P.survive[s]) continue;
      const StringRec rec = P.strings[s];
      const double kf = floor(rec.lg);
      const double f = exp2(rec.lg - kf);
      for (int p = 0; p < rec.n_units; ++p) {
        const Slot sl = P.slots[rec.slot + p];
        const long long sh = sl.e2 + (long long)kf - emax;
        const double xr = shift_clamped(sl.re * f, sh), xi = shift_clamped(sl.im * f, sh);
        double tr = re + xr; cre += (fabs(re) >= fabs(xr)) ? (re - tr) + xr : (xr - tr) + re; re = tr;
        double ti = im + xi; cim += (fabs(im) >= fabs(xi)) ? (im - ti) + xi : (xi - ti) + im; im = ti;
      }
    }
    re += cre; im += cim;
  }
  const double mx = fmax(fabs(re), fabs(im));
  if (mx > 0.0) {
    int k = ilogb(mx);
    P.mant[2 * b] = scalbn(re, -k);
    P.mant[2 * b + 1] = scalbn(im, -k);
    P.exp2[b] = emax + k;
  } else {
    P.mant[2 * b] = 0.0; P.mant[2 * b + 1] = 0.0; P.exp2[b] = 0;
  }
  P.status[b] = any_surv ? 0 : 1;
}

struct BoundParams {
  DevImp imp;
  BatchView bv;
  const uint8_t* survive;
  const StringRec* strings;
  const Slot* slots;     // segment mode
  Scaled* sector;        // [B*Q] per-string bound (already inflated, lg applied)
  int norm_kind;
  int segment_len;
  int W;
};

__device__ __forceinline__ Scaled finish_sector_bound(double val, long long e, double lg) {
  const double kf = floor(lg);
  return normalize(val * kBoundInflation * exp2(lg - kf), e + (long long)kf);
}

// segment_len == 1: one warp per string, tables only (DESIGN.md pin P-B3):
//   Frobenius  ||diag(p) F||_F^2 = sum_m p_m^2 r_m,  r_m = sum_k |F_mk|^2 precomputed at load,  p_m = exp(-Delta (E_m - Emin))
//   spectral   exp(-Delta Emin) sigma_max(F); the exponential part is already in lg.
__global__ void bound_s1_kernel(BoundParams P) {
  const int Q = P.imp.Q;
  const int lane = threadIdx.x & 31;
  long long s = (blockIdx.x * (long long)blockDim.x + threadIdx.x) >> 5;
  if (s >= P.bv.B * Q) return;
  if (!P.survive[s]) { if (lane == 0) { P.sector[s].m = 0.0; P.sector[s].e = 0; } return; }
  const long long b = s / Q;
  const int q0 = (int)(s - b * Q);
  const StringRec rec = P.strings[s];
  const long long lo = P.bv.offset[b];
  const int L = (int)(P.bv.offset[b + 1] - lo);
  double val = P.norm_kind == 0 ? sqrt((double)rec.dmin) : (double)rec.dmin;
  long long e = 0;
  double lgx = 0.0;
  int q = q0;
  if (L == 0) {
    if (P.norm_kind == 0) {
      const double* E = P.imp.energy + P.imp.e_off[q0];
      const double emin = P.imp.e_min[q0];
      double ss = 0.0;
      for (int m = lane; m < P.imp.dim[q0]; m += 32) { double p = exp(-P.bv.beta * (E[m] - emin)); ss += p * p; }
      val *= sqrt(warp_sum(ss));
    }
  }
  for (int i = 0; i < L; ++i) {
    const int blk = P.imp.blk_of[P.bv.symbol[lo + i] * Q + q];
    const BlkDesc bd = P.imp.blks[blk];
    if (P.norm_kind == 1) {
      val *= P.imp.sigma[blk];
    } else {
      const double delta = (i + 1 < L) ? (P.bv.tau[lo + i + 1] - P.bv.tau[lo + i]) : (P.bv.beta - P.bv.tau[lo + i] + P.bv.tau[lo]);
      const double* E = P.imp.energy + P.imp.e_off[bd.dst];
      const double emin = P.imp.e_min[bd.dst];
      const double* rn = P.imp.rownorm2 + bd.rn_off;
      // ||diag(2^x) F||_F^2 = sum_m 4^x_m r_m relative to the largest x_m of a non-zero row (cannot underflow)
      double xmax = -INFINITY;
      for (int m = lane; m < bd.rows; m += 32)
        if (rn[m] > 0.0) xmax = fmax(xmax, (-delta * (E[m] - emin)) * kLog2e);
      xmax = warp_max(xmax);
      if (xmax == -INFINITY) { val = 0.0; }
      else {
        double ss = 0.0;
        for (int m = lane; m < bd.rows; m += 32)
          if (rn[m] > 0.0) ss += exp2(2.0 * ((-delta * (E[m] - emin)) * kLog2e - xmax)) * rn[m];
        val *= sqrt(warp_sum(ss));
        lgx += xmax;
      }
    }
    if (val != 0.0) { int k = ilogb(val); val = scalbn(val, -k); e += k; }
    q = bd.dst;
  }
  if (lane == 0) P.sector[s] = finish_sector_bound(val, e, rec.lg + lgx);
}

// segment_len != 1: the chain kernel (mode 1) left sum |X|^2 per (segment, panel) in the slots; combine panels of a segment
// at a common exponent, take the root, multiply the segments.  One thread per string.
// norm_kind 0: B = sqrt(d_min) prod_j ||G_j||_F.   norm_kind 1 ("spectral norm"): B = d_min prod_j u_j with
// u_j = min(||G_j||_F, prod_{i in segment j} sigma_max(F_i)), both rigorous upper estimates of ||G_j||_2 (the propagator
// part exp(-Delta (E - Emin)) <= 1 never increases a spectral norm; exp(-Delta Emin) is in lg): an iterative estimate of
// ||G_j||_2 itself approaches it from below and cannot be certified, so it is not used (reading A1).
__global__ void bound_segments_kernel(BoundParams P) {
  const int Q = P.imp.Q;
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s >= P.bv.B * Q) return;
  if (!P.survive[s]) { P.sector[s].m = 0.0; P.sector[s].e = 0; return; }
  const long long b = s / Q;
  const int q0 = (int)(s - b * Q);
  const StringRec rec = P.strings[s];
  const long long lo = P.bv.offset[b];
  const int L = (int)(P.bv.offset[b + 1] - lo);
  double val = P.norm_kind == 0 ? sqrt((double)rec.dmin) : (double)rec.dmin;
  long long e = 0;
  if (L == 0 && P.norm_kind == 0) {
    const double* E = P.imp.energy + P.imp.e_off[q0];
    const double emin = P.imp.e_min[q0];
    double ss = 0.0;
    for (int m = 0; m < P.imp.dim[q0]; ++m) { double p = exp(-P.bv.beta * (E[m] - emin)); ss += p * p; }
    val *= sqrt(ss);
  }
  int q = q0, slot = rec.slot;
  for (int i = 0; i < L;) {
    const int np = (P.imp.dim[q] + P.W - 1) / P.W;
    long long emax = 0; bool any = false;
    for (int p = 0; p < np; ++p) {
      const Slot sl = P.slots[slot + p];
      if (sl.re > 0.0) { long long ee = 2 * sl.e2 + ilogb(sl.re); emax = any ? max(emax, ee) : ee; any = true; }
    }
    double ss = 0.0;
    if (any) {
      if (emax & 1) emax += 1;   // keep the exponent even so that the root is exact in the exponent
      for (int p = 0; p < np; ++p) {
        const Slot sl = P.slots[slot + p];
        ss += shift_clamped(sl.re, 2 * sl.e2 - emax);
      }
    }
    const double fro = sqrt(ss);
    const int stop = min(L, i + P.segment_len);
    double sprod = 1.0;
    for (; i < stop; ++i) { const int blk = P.imp.blk_of[P.bv.symbol[lo + i] * Q + q]; sprod *= P.imp.sigma[blk]; q = P.imp.blks[blk].dst; }
    if (P.norm_kind == 0 || fro == 0.0 || log2(fro) + (double)(emax / 2) <= log2(sprod)) { val *= fro; e += emax / 2; }
    else val *= sprod;
    if (val != 0.0) { int k = ilogb(val); val = scalbn(val, -k); e += k; } else { e = 0; }
    slot += np;
  }
  P.sector[s] = finish_sector_bound(val, e, rec.lg);
}

struct BoundReduceParams {
  long long B;
  int Q;
  const int* status_in;
  const uint8_t* survive;
  const Scaled* sector;
  double* bound_mant; long long* bound_exp2;
  double* sector_mant; long long* sector_exp2;   // may be null
  int* status;
};

__global__ void bound_reduce_kernel(BoundReduceParams P) {
  long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (b >= P.B) return;
  const double nan = __longlong_as_double(0x7ff8000000000000LL);
  if (P.status_in[b] == 2) {
    P.bound_mant[b] = nan; P.bound_exp2[b] = 0; P.status[b] = 2;
    if (P.sector_mant) for (int q = 0; q < P.Q; ++q) { P.sector_mant[b * P.Q + q] = nan; P.sector_exp2[b * P.Q + q] = 0; }
    return;
  }
  bool any_surv = false, any_nz = false;
  long long emax = 0;
  for (int q = 0; q < P.Q; ++q) {
    long long s = b * P.Q + q;
    Scaled v; v.m = 0.0; v.e = 0;
    if (P.survive[s]) { any_surv = true; v = P.sector[s]; }
    if (P.sector_mant) { P.sector_mant[s] = v.m; P.sector_exp2[s] = v.e; }
    if (v.m > 0.0) { emax = any_nz ? max(emax, v.e) : v.e; any_nz = true; }
  }
  double sum = 0.0;
  if (any_nz)
    for (int q = 0; q < P.Q; ++q) {
      long long s = b * P.Q + q;
      if (P.survive[s]) sum += shift_clamped(P.sector[s].m, P.sector[s].e - emax);
    }
  sum *= (1.0 + 2.220446049250313e-16 * 2.0 * P.Q);   // summation rounding, outward
  Scaled r = normalize(sum, emax);
  P.bound_mant[b] = (sum > 0.0) ? r.m : 0.0;
  P.bound_exp2[b] = (sum > 0.0) ? r.e : 0;
  P.status[b] = any_surv ? 0 : 1;
}

}  // namespace ctqmc
