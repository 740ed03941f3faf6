// Shared device-side types and helpers of libctqmc_b200 (sm_100a only).
// Notation follows the paper: q sectors, alpha symbols, F_alpha(q) blocks, P_tau(q) propagators.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ctqmc {

constexpr double kLog2e = 1.4426950408889634;
constexpr double kBoundInflation = 1.0 + 9.094947017729282e-13;  // 1 + 2^-40, reading A9
constexpr int kCtaThreads = 256;
constexpr int kCtaWarps = 8;
constexpr int kCostClasses = 64;

// One sector-to-sector block F_alpha(q) in the device operator store: row-major, rows = destination
// states, padded with zeros to rows_pad (multiple of 8) x ld (multiple of 8 real / 4 complex elements) so that the
// MMA loops need no bounds checks.  Offsets are in doubles.
struct BlkDesc {
  long long off;     // into store
  long long rn_off;  // into rownorm2 (rows entries)
  int ld;            // leading dimension in elements (element = 1 double real, 2 doubles complex)
  int rows, cols;    // dim[dst], dim[src]
  int dst, src;
  int pad;
};

struct DevImp {
  int Q, A, cplx, dmax;
  const int* dim;            // [Q]
  const long long* e_off;    // [Q] offset of the sector's eigenvalues in energy
  const double* energy;      // [sum dim]
  const double* e_min;       // [Q]
  const int* blk_of;         // [A*Q] block index of (alpha, q) or -1 (the zero sector)
  const BlkDesc* blks;
  const double* store;       // operator store
  const double* rownorm2;    // per block row: sum_k |F_mk|^2
  const double* sigma;       // [n_blocks] spectral norm
  const int* blk_order;      // [n_blocks] block indices, heaviest (rows x cols) first: tile order of the grouped path
};

struct BatchView {
  long long B;
  const long long* offset;
  const int* symbol;
  const double* tau;
  double beta;
  long long n_ops;   // length of symbol / tau as stated by the caller: every offset is checked against it
  int max_len;       // longest configuration the caller vouches for (sizes the step loops); longer ones are invalid
};

// One surviving (configuration, start sector) string, written by the routing kernel.
struct StringRec {
  double lg;      // -sum_i Delta_i Emin(q_i) log2(e): real exponent factored out of the propagators
  int q_start;    // sector the (cyclically rotated) chain starts in
  int r;          // rotation: the chain starts after operator r (0 = literal order)
  int c;          // columns carried: dim(q_start)
  int slot;       // first result slot of this string's work units
  int n_units;
  int dmin;       // smallest sector dimension along the string
  int cls;        // cost class (log2 of the estimated MACs of one unit)
  int pad;
};

// Result of one work unit: value = (re + i im) * 2^e2.
struct Slot {
  double re, im;
  long long e2;
  long long pad;
};

struct Counters {
  unsigned long long n_strings;
  unsigned long long n_slots;
  unsigned long long next_unit;
  unsigned long long macs;        // real MACs executed (padded)
  unsigned long long alg_flops;   // algorithmic flops of the executed schedule
  unsigned int max_len;           // longest chain among strings with work (large-sector path: number of step launches)
  unsigned int max_c;             // widest carried matrix among them
  unsigned long long sum_c;       // total carried columns (grouped path: columns per chain position)
  unsigned long long n_exp;       // propagator exponentials evaluated (small path: sum over steps of dim(q_i))
  unsigned int class_count[kCostClasses];
  unsigned int class_base[kCostClasses];
  unsigned int class_cursor[kCostClasses];
};

__device__ __forceinline__ int round_up(int x, int m) { return (x + m - 1) / m * m; }

__device__ __forceinline__ double warp_max(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// x = -Delta (E - Emin) log2(e) with every operation rounded on its own (no FMA contraction): the producer of a row
// exponent floor(x) and its consumers (the rescale, the next step's load) must see bit-identical x.
__device__ __forceinline__ double prop_x(double delta, double e, double emin) {
  return __dmul_rn(__dmul_rn(-delta, __dsub_rn(e, emin)), kLog2e);
}

// integer part of the row exponent, floor(x), saturated; one instruction (cvt.rmi.s32.f64).  Every producer and consumer of
// a row exponent uses this function so that they agree bit for bit.
__device__ __forceinline__ int row_exp(double x) { return max(__double2int_rd(x), -(1 << 30)); }

// exact 2^k for |k| <= 1022
__device__ __forceinline__ double pow2i(int k) { return __longlong_as_double((long long)(k + 1023) << 52); }

// Native FP64 tensor-core op on sm_100a: D(8x8) += A(8x4, row) * B(4x8, col).  SASS: DMMA.8x8x4.
// Fragments (g = lane/4, t = lane%4): a = A[g][t], b = B[t][g], c0/c1 = C[g][2t], C[g][2t+1].
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1},{%2},{%3},{%0,%1};"
               : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

}  // namespace ctqmc
