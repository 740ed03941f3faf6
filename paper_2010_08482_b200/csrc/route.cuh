// Sector routing: integer-only walk of the sector map s_alpha(q) for every
// (configuration, start sector), input validation, and construction of the work-unit list for the chain kernel.
#pragma once
#include "common.cuh"

namespace ctqmc {

// DESIGN.md reading A7: symbols in [0, A), tau finite, non-decreasing, in [0, beta).  One thread per configuration.
__global__ void validate_kernel(BatchView bv, int A, int* __restrict__ status) {
  long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (b >= bv.B) return;
  long long lo = bv.offset[b], hi = bv.offset[b + 1];
  // a corrupt offset array must give status 2, not an out-of-bounds read
  bool ok = lo >= 0 && hi >= lo && hi <= bv.n_ops && hi - lo <= (long long)bv.max_len;
  double prev = 0.0;
  for (long long i = lo; ok && i < hi; ++i) {
    int a = bv.symbol[i];
    double t = bv.tau[i];
    ok = (a >= 0) && (a < A) && (t >= prev) && (t < bv.beta);  // NaN fails both comparisons
    prev = t;
  }
  status[b] = ok ? 0 : 2;
}

struct RouteParams {
  DevImp imp;
  BatchView bv;
  const int* status;
  uint8_t* survive;       // [B*Q] internal
  uint8_t* survive_out;   // [B*Q] caller's, or nullptr
  StringRec* strings;     // [B*Q]
  Counters* cnt;
  int W;                  // panel width (columns per work unit)
  int kstep;              // K padding granularity of the chain kernel (8 real, 4 complex)
  int literal;            // CTQMC_SCHEDULE_LITERAL
  int flops_per_mac;      // 2 real, 8 complex
  int mode;               // 0 trace, 1 bound by segments
  int segment_len;        // mode 1: S >= 1 (S == L handled as "whole chain" by the caller passing a huge S)
};

// One thread per (configuration b, start sector q0).  Follows q_i = s_alpha_i(q_{i-1}); a string that reaches the zero
// sector does not survive.  For survivors it records where the visited sector is smallest (thin start:
// the trace is invariant under cyclic rotation, so the chain may start there and carry only d_min columns), the real
// exponent lg = -sum_i Delta_i Emin(q_i) log2 e with the cyclic time differences Delta_i, and reserves result slots.
__global__ void route_kernel(RouteParams P) {
  const int Q = P.imp.Q;
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s >= P.bv.B * Q) return;
  long long b = s / Q;
  int q0 = (int)(s - b * Q);
  StringRec rec;
  rec.lg = 0.0; rec.q_start = q0; rec.r = 0; rec.c = 0; rec.slot = 0; rec.n_units = 0; rec.dmin = 0; rec.cls = 0;
  uint8_t alive = 0;
  if (P.status[b] == 0) {
    long long lo = P.bv.offset[b];
    int L = (int)(P.bv.offset[b + 1] - lo);
    int q = q0, d = P.imp.dim[q0];
    int dmin = d, rpos = 0, qmin = q0;
    double lg = 0.0;
    unsigned long long cost = 0, alg = 0;   // per carried column
    unsigned long long seg_units = 0;       // mode 1: sum over segments of panels
    bool ok = true;
    double t0 = L ? P.bv.tau[lo] : 0.0, tcur = t0;
    if (P.mode == 1 && L > 0) seg_units = (unsigned)((d + P.W - 1) / P.W);
    for (int i = 0; i < L; ++i) {
      int blk = P.imp.blk_of[P.bv.symbol[lo + i] * Q + q];
      if (blk < 0) { ok = false; break; }
      int qn = P.imp.blks[blk].dst;
      int dn = P.imp.dim[qn];
      double tnext = (i + 1 < L) ? P.bv.tau[lo + i + 1] : P.bv.beta + t0;
      lg -= (tnext - tcur) * P.imp.e_min[qn] * kLog2e;
      tcur = tnext;
      cost += (unsigned long long)round_up(dn, 8) * (unsigned long long)round_up(d, P.kstep);
      alg += (unsigned long long)dn * (unsigned long long)d;
      if (i + 1 < L && dn < dmin) { dmin = dn; rpos = i + 1; qmin = qn; }
      if (P.mode == 1 && i + 1 < L && (i + 1) % P.segment_len == 0) seg_units += (unsigned)((dn + P.W - 1) / P.W);
      q = qn; d = dn;
    }
    if (L == 0) lg = -P.bv.beta * P.imp.e_min[q0] * kLog2e;
    if (ok) {
      alive = 1;
      rec.lg = lg;
      rec.dmin = dmin;
      if (P.mode == 0) {
        if (q == q0) {   // a survivor that does not return to q0 is an off-diagonal block: contributes nothing (:532)
          if (P.literal) { rec.q_start = q0; rec.r = 0; rec.c = P.imp.dim[q0]; }
          else { rec.q_start = qmin; rec.r = rpos; rec.c = dmin; }
          rec.n_units = (rec.c + P.W - 1) / P.W;
        }
      } else {
        rec.q_start = q0; rec.r = 0; rec.c = P.imp.dim[q0];
        rec.n_units = (L == 0) ? 0 : (int)seg_units;
        if (L > 0) { cost = cost / (unsigned long long)((L + P.segment_len - 1) / P.segment_len) + 1; }
      }
      if (rec.n_units > 0) {
        int wc = P.mode == 0 ? min(P.W, rec.c) : P.W;
        unsigned long long ucost = cost * (unsigned long long)wc + 1ull;
        rec.cls = 63 - __clzll((long long)ucost);
        rec.slot = (int)atomicAdd(&P.cnt->n_slots, (unsigned long long)rec.n_units);
        atomicAdd(&P.cnt->class_count[rec.cls], (unsigned)rec.n_units);
        atomicAdd(&P.cnt->n_strings, 1ull);
        atomicMax(&P.cnt->max_len, (unsigned)L);
        atomicMax(&P.cnt->max_c, (unsigned)rec.c);
        atomicAdd(&P.cnt->sum_c, (unsigned long long)rec.c);
        if (P.mode == 0) {
          atomicAdd(&P.cnt->macs, cost * (unsigned long long)(round_up(rec.c, 8)) * (unsigned long long)(P.flops_per_mac / 2));
          atomicAdd(&P.cnt->alg_flops, alg * (unsigned long long)rec.c * (unsigned long long)P.flops_per_mac);
        }
      }
    }
  }
  P.survive[s] = alive;
  if (P.survive_out) P.survive_out[s] = alive;
  P.strings[s] = rec;
}

// Adds one round's counters to the call's totals (a call is cut into rounds of configurations when its scratch would not
// fit the arena; ctqmc_last_stats reports the totals).
__global__ void accumulate_counters_kernel(const Counters* __restrict__ c, Counters* __restrict__ tot) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  tot->n_strings += c->n_strings; tot->n_slots += c->n_slots; tot->macs += c->macs; tot->alg_flops += c->alg_flops;
  tot->sum_c += c->sum_c; tot->n_exp += c->n_exp;
  tot->max_len = max(tot->max_len, c->max_len); tot->max_c = max(tot->max_c, c->max_c);
}

// Heaviest cost class first (longest-processing-time order for the persistent chain kernel).
__global__ void class_scan_kernel(Counters* cnt) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    unsigned run = 0;
    for (int c = kCostClasses - 1; c >= 0; --c) {
      cnt->class_base[c] = run;
      run += cnt->class_count[c];
      cnt->class_cursor[c] = 0;
    }
  }
}

__global__ void unit_scatter_kernel(const StringRec* __restrict__ strings, long long n_strings_total, Counters* cnt,
                                    int2* __restrict__ units) {
  long long s = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (s >= n_strings_total) return;
  int n = strings[s].n_units;
  if (n <= 0) return;
  int cls = strings[s].cls;
  unsigned pos = cnt->class_base[cls] + atomicAdd(&cnt->class_cursor[cls], (unsigned)n);
  for (int p = 0; p < n; ++p) units[pos + p] = make_int2((int)s, p);
}

}  // namespace ctqmc
