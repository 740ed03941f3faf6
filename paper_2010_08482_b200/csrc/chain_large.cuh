// Large-sector chain path (SURVEY.md §8(a) a3-a5 for sectors whose carried matrix does not fit in shared memory, e.g. the
// 1001 / 2002 / 3003-state sectors of the low-symmetry f-shell; PAPER.md:554 "858", :572 "matrix multiplication ... kernels").
//
// Here one chain step   X' = diag(exp(-Delta (E - Emin))) * F_alpha(q) * X   is a real dense contraction (hundreds of flop
// per byte), so it runs as a tiled GEMM on the FP64 tensor cores: CTA tile 128 x 64, 8 warps of 32 x 32, operands staged
// global -> shared by a 4-deep cp.async pipeline of 128-byte rows (XOR-swizzled so the 128-bit fragment loads are
// bank-conflict free), mma.sync m8n8k4 f64 (SASS DMMA.8x8x4), complex as four real products on interleaved (re, im) storage.
// All surviving strings of the batch advance together: one launch per chain position, grid = (tiles, strings).
//
// Fusion.  The propagator is never a separate pass (PAPER.md:572 has a separate "time evolution" kernel): its mantissa
// 2^(x - floor x), x = -Delta (E_row - Emin) log2 e, is multiplied into the accumulators in the epilogue; its integer
// part floor(x) stays a per-row binary exponent that the *next* step applies, together with the running-exponent
// rescale, as one exact power-of-two factor per contraction index while it loads its B fragments (SURVEY a4 "applied
// lazily in the next step's load").  The largest row exponent of a step is found with warp shuffles plus one atomicMax
// per warp.  Only a shift of more than 2^1022 between a row and the largest row is clamped (flushes to zero / cannot
// occur for operators with O(1) entries).
#pragma once
#include <climits>
#include <cuda.h>

#include "chain.cuh"

namespace ctqmc {

constexpr int kLBM = 128, kLBN = 64, kLStages = 4;
constexpr int kLStageBytes = (kLBM + kLBN) * 128;

struct LargeParams {
  DevImp imp;
  BatchView bv;
  const StringRec* strings;
  const int2* units;      // unit u -> (string index, 0)
  const Counters* cnt;    // cnt->n_slots = units that exist (device-side: the host only knows an upper bound)
  long long u0;           // first unit of this group
  int n_group;            // unit slots in this group (host-side upper bound; slots beyond cnt->n_slots stay idle)
  int Lmax;               // plan stride
  int ldx;                // leading dimension (elements) of an X column
  long long sum_d;        // sum of all sector dimensions (mode 0: column slab of one configuration, per parity)
  double* X;              // carried matrices: columns of ldx elements; unit s owns columns [u_x[s], u_x[s] + 2 u_w[s])
  long long* u_x;         // [n_group] first column of the unit's two parity buffers
  int* u_w;               // [n_group] columns per parity buffer
  int* plan_blk;          // [n_group][Lmax]
  double* plan_delta;     // [n_group][Lmax]
  int* kmax;              // [n_group][Lmax]
  int* u_q;               // [n_group] sector the unit's chain starts in
  int* u_n;               // [n_group] chain positions to multiply
  int* u_c;               // [n_group] columns carried
  int mode;               // 0 trace of the whole (rotated) chain, 1 Frobenius norm^2 of one segment per unit
  int segment_len;        // mode 1
  const CUtensorMap* amaps;   // [n_blocks] tensor maps of the operator blocks (TMA variant)
  Slot* slots;
};

// One thread per string of the group: the sector walk in the (rotated) order the chain will be multiplied in.
__global__ void large_plan_kernel(LargeParams P) {
  const int s = blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= P.n_group) return;
  if ((unsigned long long)(P.u0 + s) >= P.cnt->n_slots) {   // idle slot: every later kernel skips it
    P.u_q[s] = 0; P.u_n[s] = -1; P.u_c[s] = 0; P.u_x[s] = 0; P.u_w[s] = 0;
    return;
  }
  const int2 un = P.units[P.u0 + s];
  const StringRec sr = P.strings[un.x];
  const int Q = P.imp.Q;
  const long long b = un.x / Q;
  const long long base = P.bv.offset[b];
  const int L = (int)(P.bv.offset[b + 1] - base);
  const int* sym = P.bv.symbol + base;
  const double* tau = P.bv.tau + base;
  int q = sr.q_start, i0 = sr.r, n = L, c = sr.c;
  if (P.mode == 1) {   // unit = segment un.y of the literal chain: starts from the identity of the sector it begins in
    i0 = un.y * P.segment_len;
    for (int i = 0; i < i0; ++i) q = P.imp.blks[P.imp.blk_of[sym[i] * Q + q]].dst;
    n = min(P.segment_len, L - i0);
    c = P.imp.dim[q];
  }
  P.u_q[s] = q; P.u_n[s] = n; P.u_c[s] = c;
  if (P.mode == 1) { P.u_w[s] = P.imp.dmax; P.u_x[s] = (long long)s * 2 * P.imp.dmax; }
  else {   // string (b, q0) of the round owns dim(q0) >= c columns per parity at a position the host can compute
    const int q0 = un.x - (int)(b * Q);
    P.u_w[s] = P.imp.dim[q0];
    P.u_x[s] = 2 * (b * P.sum_d + P.imp.e_off[q0]);
  }
  for (int j = 0; j < n; ++j) {
    int i = i0 + j;
    if (i >= L) i -= L;
    const int blk = P.imp.blk_of[sym[i] * Q + q];
    P.plan_blk[(size_t)s * P.Lmax + j] = blk;
    P.plan_delta[(size_t)s * P.Lmax + j] = (i + 1 < L) ? (tau[i + 1] - tau[i]) : (P.bv.beta - tau[i] + tau[0]);
    P.kmax[(size_t)s * P.Lmax + j] = INT_MIN;
    q = P.imp.blks[blk].dst;
  }
}

// X_0 = identity (c x c, c = dim of the start sector); grid (column blocks, strings).  Whole columns (ldx rows) of BOTH parity
// buffers are written: rows beyond the current sector's dimension are read by later steps (multiplied by an exact 0), so they
// must hold finite numbers, and the arena they live in is shared with integer tables of earlier calls.
template <bool CPLX>
__global__ void large_init_kernel(LargeParams P) {
  const int s = blockIdx.y;
  const int c = P.u_c[s];
  if (P.u_n[s] < 0) return;
  constexpr int ES = CPLX ? 2 : 1;
  double* X0 = P.X + (size_t)P.u_x[s] * P.ldx * ES;
  double* X1 = X0 + (size_t)P.u_w[s] * P.ldx * ES;
  for (int col = blockIdx.x; col < c; col += gridDim.x)
    for (int k = threadIdx.x; k < P.ldx; k += blockDim.x) {
      const double v = (k == col) ? 1.0 : 0.0;
      if constexpr (CPLX) {
        *reinterpret_cast<double2*>(X0 + ((size_t)col * P.ldx + k) * 2) = make_double2(v, 0.0);
        *reinterpret_cast<double2*>(X1 + ((size_t)col * P.ldx + k) * 2) = make_double2(0.0, 0.0);
      } else {
        X0[(size_t)col * P.ldx + k] = v;
        X1[(size_t)col * P.ldx + k] = 0.0;
      }
    }
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem, bool valid) {
  const unsigned sa = (unsigned)__cvta_generic_to_shared(smem);
  const int sz = valid ? 16 : 0;
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(gmem), "r"(sz) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// ---- TMA (cp.async.bulk.tensor) + mbarrier primitives: the Blackwell-native way to stage the operand tiles.  One elected
// thread arms the stage's barrier with the byte count and issues four 2-D box copies (two k-halves of F rows and of X
// columns); the copy engine writes shared memory and completes the transaction on the barrier; all threads wait on it.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// all earlier cp.async of this thread arrive on `bar` when they have landed (the barrier's count includes this arrival)
__device__ __forceinline__ void cp_async_arrive(unsigned long long* bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}"
      ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, unsigned long long* bar, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(smem_u32(bar)) : "memory");
}

// One chain position for every string of the group.  blockIdx.x = mt * NTmax + nt (nt fastest: CTAs that share rows of
// F run together and hit L2), blockIdx.y = string.
// `xmap`: ONE tensor map over the whole carried-matrix region (2-D: ldx elements x all columns), passed by value; a unit
// addresses its matrix by its global column index, so no per-string maps have to be built or copied.
template <bool CPLX, bool TMA>
__global__ void __launch_bounds__(256, 1) large_step_kernel(const __grid_constant__ CUtensorMap xmap_all, LargeParams P, int j, int NTmax) {
  constexpr int ES = CPLX ? 2 : 1;
  constexpr int BKE = CPLX ? 8 : 16;       // contraction indices per stage (128-byte rows)
  extern __shared__ __align__(128) unsigned char lsm[];
  __shared__ __align__(8) unsigned long long full_bar[kLStages], empty_bar[kLStages];
  double* sscale = reinterpret_cast<double*>(lsm + kLStages * kLStageBytes);

  const int s = blockIdx.y;
  if (j >= P.u_n[s]) return;
  const int blk = P.plan_blk[(size_t)s * P.Lmax + j];
  const BlkDesc bd = P.imp.blks[blk];
  const int dn = bd.rows, d = bd.cols, c = P.u_c[s];
  const int mt0 = blockIdx.x / NTmax, nt0 = blockIdx.x - mt0 * NTmax;
  const int m0 = mt0 * kLBM, n0 = nt0 * kLBN;
  if (m0 >= dn || n0 >= c) return;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp >> 1, wn = warp & 1;
  const long long xcol_in = P.u_x[s] + (long long)(j & 1) * P.u_w[s], xcol_out = P.u_x[s] + (long long)((j + 1) & 1) * P.u_w[s];
  const double* Xin = P.X + (size_t)xcol_in * P.ldx * ES;
  double* Xout = P.X + (size_t)xcol_out * P.ldx * ES;
  const int nkt = (d + BKE - 1) / BKE;

  // exact power-of-two factor per contraction index: row exponent of the previous step minus its largest (a4)
  {
    int kprev = 0;
    double dprev = 0.0;
    if (j > 0) { kprev = P.kmax[(size_t)s * P.Lmax + j - 1]; dprev = P.plan_delta[(size_t)s * P.Lmax + j - 1]; }
    const double* Eq = P.imp.energy + P.imp.e_off[bd.src];
    const double emin = P.imp.e_min[bd.src];
    for (int k = tid; k < nkt * BKE; k += 256) {
      double f = 0.0;
      if (k < d && kprev != INT_MIN) {
        if (j == 0) f = 1.0;
        else {
          const double x = prop_x(dprev, Eq[k], emin);
          const long long sh = (long long)row_exp(x) - (long long)kprev;
          f = (sh < -1022) ? 0.0 : pow2i((int)min(sh, 1022LL));
        }
      }
      sscale[k] = f;
    }
  }

  const unsigned char* Ag = reinterpret_cast<const unsigned char*>(P.imp.store + bd.off);
  const unsigned char* Bg = reinterpret_cast<const unsigned char*>(Xin);
  const int rows_pad = round_up(dn, 8);
  const size_t a_row_bytes = (size_t)bd.ld * ES * 8, b_col_bytes = (size_t)P.ldx * ES * 8;
  const int ld_chunks = bd.ld * ES / 2;          // 16-byte chunks per row of F (padded with zeros)
  const int x_chunks = CPLX ? d : (d + 1) / 2;   // 16-byte chunks of an X column that hold data
  const CUtensorMap* amap = P.amaps + blk;
  const CUtensorMap* xmap = &xmap_all;
  const int xcol0 = (int)xcol_in + n0;

  // cp.async variant: 128-byte rows, 16-byte chunks XOR-swizzled by the row parity.
  // TMA variant: per k-half a dense box of 64-byte rows (two adjacent rows = one 128-byte line, so the 128-bit fragment loads
  // of a quarter warp are conflict free without any swizzle); out-of-range rows / k are zero-filled by the copy engine.
  auto load_stage = [&](int kt, int stage) {
    unsigned char* As = lsm + stage * kLStageBytes;
    if constexpr (TMA) {
      if (tid == 0) {
        mbar_expect_tx(&full_bar[stage], kLStageBytes);
#pragma unroll
        for (int sub = 0; sub < 2; ++sub) {
          tma_load_2d(As + sub * (kLBM * 64), amap, &full_bar[stage], kt * 16 + sub * 8, m0);
          tma_load_2d(As + 2 * (kLBM * 64) + sub * (kLBN * 64), xmap, &full_bar[stage], kt * 16 + sub * 8, xcol0);
        }
      }
    } else {
      unsigned char* Bs = As + kLBM * 128;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const int idx = tid + i * 256, r = idx >> 3, ch = idx & 7;
        const int row = m0 + r, gch = kt * 8 + ch;
        const bool ok = row < rows_pad && gch < ld_chunks;
        cp_async16(As + r * 128 + ((ch ^ ((r & 1) << 2)) << 4), ok ? Ag + (size_t)row * a_row_bytes + (size_t)gch * 16 : Ag, ok);
      }
#pragma unroll
      for (int i = 0; i < 2; ++i) {
        const int idx = tid + i * 256, r = idx >> 3, ch = idx & 7;
        const int col = n0 + r, gch = kt * 8 + ch;
        const bool ok = col < c && gch < x_chunks;
        cp_async16(Bs + r * 128 + ((ch ^ ((r & 1) << 2)) << 4), ok ? Bg + (size_t)col * b_col_bytes + (size_t)gch * 16 : Bg, ok);
      }
    }
  };

  double acc[4][4][CPLX ? 4 : 2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
      for (int x = 0; x < (CPLX ? 4 : 2); ++x) acc[a][b][x] = 0.0;

  if constexpr (TMA) {
    if (tid == 0) {
#pragma unroll
      for (int st = 0; st < kLStages; ++st) { mbar_init(&full_bar[st], 1); mbar_init(&empty_bar[st], 8); }
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
  }
  // TMA variant: full/empty barrier ring, no CTA-wide barrier in the loop.  The producer (thread 0) refills the slot that was
  // consumed TWO iterations ago, so a warp may run a whole k-tile ahead of the slowest one before anybody waits.
  constexpr int kAhead = TMA ? kLStages - 2 : kLStages - 1;
#pragma unroll
  for (int st = 0; st < kAhead; ++st) {
    if (st < nkt) load_stage(st, st);
    if constexpr (!TMA) cp_async_commit();
  }

  const int swz = (g & 1) << 2;
  for (int kt = 0; kt < nkt; ++kt) {
    if constexpr (TMA) {
      const int nx = kt + kAhead;
      if (nx < nkt) {
        if (tid == 0 && nx >= kLStages) mbar_wait(&empty_bar[nx % kLStages], ((nx / kLStages) - 1) & 1);
        load_stage(nx, nx % kLStages);
      }
      mbar_wait(&full_bar[kt % kLStages], (kt / kLStages) & 1);
    } else {
      cp_async_wait<kLStages - 2>();
      __syncthreads();
      const int nx = kt + kLStages - 1;
      if (nx < nkt) load_stage(nx, nx % kLStages);
      cp_async_commit();
    }
    const unsigned char* As = lsm + (kt % kLStages) * kLStageBytes;
#pragma unroll
    for (int sub = 0; sub < 2; ++sub) {
      const int ch = sub * 4 + t;
      double2 a[4], b[4];
      if constexpr (TMA) {
        const unsigned char* Ah = As + sub * (kLBM * 64) + t * 16;
        const unsigned char* Bh = As + 2 * (kLBM * 64) + sub * (kLBN * 64) + t * 16;
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) a[mt] = *reinterpret_cast<const double2*>(Ah + (wm * 32 + mt * 8 + g) * 64);
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) b[nt] = *reinterpret_cast<const double2*>(Bh + (wn * 32 + nt * 8 + g) * 64);
      } else {
        const unsigned char* Bs = As + kLBM * 128;
        const int so = ((ch ^ swz) << 4);
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) a[mt] = *reinterpret_cast<const double2*>(As + (wm * 32 + mt * 8 + g) * 128 + so);
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) b[nt] = *reinterpret_cast<const double2*>(Bs + (wn * 32 + nt * 8 + g) * 128 + so);
      }
      if constexpr (CPLX) {
        const double f = sscale[kt * 8 + ch];
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) { b[nt].x *= f; b[nt].y *= f; }
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) {
            dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt].x, b[nt].x);
            dmma884(acc[mt][nt][2], acc[mt][nt][3], a[mt].x, b[nt].y);
          }
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
          const double na = -a[mt].y;
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) {
            dmma884(acc[mt][nt][0], acc[mt][nt][1], na, b[nt].y);
            dmma884(acc[mt][nt][2], acc[mt][nt][3], a[mt].y, b[nt].x);
          }
        }
      } else {
        const double2 f = *reinterpret_cast<const double2*>(sscale + kt * 16 + ch * 2);
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) { b[nt].x *= f.x; b[nt].y *= f.y; }
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt].x, b[nt].x);
#pragma unroll
        for (int mt = 0; mt < 4; ++mt)
#pragma unroll
          for (int nt = 0; nt < 4; ++nt) dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt].y, b[nt].y);
      }
    }
    if constexpr (TMA) {   // this warp is done reading the slot
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty_bar[kt % kLStages]);
    }
  }
  if constexpr (!TMA) cp_async_wait<0>();

  // ---- epilogue: propagator mantissa, store, largest row exponent
  const double delta = P.plan_delta[(size_t)s * P.Lmax + j];
  const double* E = P.imp.energy + P.imp.e_off[bd.dst];
  const double emin = P.imp.e_min[bd.dst];
  int wexp = INT_MIN;
#pragma unroll
  for (int mt = 0; mt < 4; ++mt) {
    const int row = m0 + wm * 32 + mt * 8 + g;
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
    for (int nt = 0; nt < 4; ++nt) {
      const int col = n0 + wn * 32 + nt * 8 + 2 * t;
      if constexpr (CPLX) {
        const double2 v0 = make_double2(acc[mt][nt][0] * mr, acc[mt][nt][2] * mr);
        const double2 v1 = make_double2(acc[mt][nt][1] * mr, acc[mt][nt][3] * mr);
        if (row < dn && col < c) {
          *reinterpret_cast<double2*>(Xout + ((size_t)col * P.ldx + row) * 2) = v0;
          rmax = fmax(rmax, fmax(fabs(v0.x), fabs(v0.y)));
        }
        if (row < dn && col + 1 < c) {
          *reinterpret_cast<double2*>(Xout + ((size_t)(col + 1) * P.ldx + row) * 2) = v1;
          rmax = fmax(rmax, fmax(fabs(v1.x), fabs(v1.y)));
        }
      } else {
        const double v0 = acc[mt][nt][0] * mr, v1 = acc[mt][nt][1] * mr;
        if (row < dn && col < c) { Xout[(size_t)col * P.ldx + row] = v0; rmax = fmax(rmax, fabs(v0)); }
        if (row < dn && col + 1 < c) { Xout[(size_t)(col + 1) * P.ldx + row] = v1; rmax = fmax(rmax, fabs(v1)); }
      }
    }
    rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, 1));
    rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, 2));
    if (rmax > 0.0) wexp = max(wexp, kr + ilogb(rmax));
  }
  wexp = __reduce_max_sync(0xffffffffu, wexp);
  if (lane == 0 && wexp != INT_MIN) atomicMax(&P.kmax[(size_t)s * P.Lmax + j], wexp);
}

// Mode 0: trace of the final matrix (a5): sum_n X[n][n] 2^(row exponent - largest).  Mode 1: squared Frobenius norm of the
// segment product (a6).  Running exponent = sum of the steps' largest row exponents.
template <bool CPLX>
__global__ void large_finish_kernel(LargeParams P) {
  constexpr int ES = CPLX ? 2 : 1;
  __shared__ double red[2][8];
  const int s = blockIdx.x;
  if (P.u_n[s] < 0) return;   // idle slot
  const int2 un = P.units[P.u0 + s];
  const StringRec sr = P.strings[un.x];
  const int n_steps = P.u_n[s], c = P.u_c[s];
  double re = 0.0, im = 0.0;
  long long e2 = 0;
  bool dead = false;
  if (n_steps == 0) {   // empty configuration, trace mode only: Tr P_beta(q0)
    const int q = P.u_q[s];
    const double* E = P.imp.energy + P.imp.e_off[q];
    const double emin = P.imp.e_min[q];
    for (int n = threadIdx.x; n < c; n += blockDim.x) re += exp(-P.bv.beta * (E[n] - emin));
  } else {
    for (int j = 0; j < n_steps; ++j) {
      const int k = P.kmax[(size_t)s * P.Lmax + j];
      if (k == INT_MIN) { dead = true; break; }
      e2 += k;
    }
    if (!dead) {
      const BlkDesc bl = P.imp.blks[P.plan_blk[(size_t)s * P.Lmax + n_steps - 1]];
      const double* E = P.imp.energy + P.imp.e_off[bl.dst];
      const double emin = P.imp.e_min[bl.dst];
      const int klast = P.kmax[(size_t)s * P.Lmax + n_steps - 1];
      const double dlast = P.plan_delta[(size_t)s * P.Lmax + n_steps - 1];
      const double* X = P.X + (size_t)(P.u_x[s] + (long long)(n_steps & 1) * P.u_w[s]) * P.ldx * ES;
      if (P.mode == 0) {
        for (int n = threadIdx.x; n < c; n += blockDim.x) {
          const long long sh = (long long)row_exp(prop_x(dlast, E[n], emin)) - (long long)klast;
          const double f = (sh < -1022) ? 0.0 : pow2i((int)min(sh, 1022LL));
          if constexpr (CPLX) {
            const double2 v = *reinterpret_cast<const double2*>(X + ((size_t)n * P.ldx + n) * 2);
            re += v.x * f; im += v.y * f;
          } else {
            re += X[(size_t)n * P.ldx + n] * f;
          }
        }
      } else {
        const int rows = bl.rows;
        for (long long idx = threadIdx.x; idx < (long long)rows * c; idx += blockDim.x) {
          const int col = (int)(idx / rows), row = (int)(idx - (long long)col * rows);
          const long long sh = (long long)row_exp(prop_x(dlast, E[row], emin)) - (long long)klast;
          const double f = (sh < -1022) ? 0.0 : pow2i((int)min(sh, 1022LL));
          if constexpr (CPLX) {
            const double2 v = *reinterpret_cast<const double2*>(X + ((size_t)col * P.ldx + row) * 2);
            re += (v.x * f) * (v.x * f) + (v.y * f) * (v.y * f);
          } else {
            const double v = X[(size_t)col * P.ldx + row] * f;
            re += v * v;
          }
        }
      }
    }
  }
  re = warp_sum(re); im = warp_sum(im);
  if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = re; red[1][threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tr = 0.0, ti = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { tr += red[0][w]; ti += red[1][w]; }
    Slot out; out.re = dead ? 0.0 : tr; out.im = dead ? 0.0 : ti; out.e2 = dead ? 0 : e2; out.pad = 0;
    P.slots[sr.slot + (P.mode == 1 ? un.y : 0)] = out;
  }
}

inline size_t large_smem_bytes(int dmax) {
  return (size_t)kLStages * kLStageBytes + (size_t)((dmax + 15) / 16 * 16 + 16) * sizeof(double);
}

}  // namespace ctqmc
