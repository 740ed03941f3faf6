// Split-precision (Ozaki-type) evaluation of the large-sector chain step on the 5th-generation tensor cores
// ("in the future we hope to achieve an even more dramatic acceleration in the hardest
// problems by using a mixed-precision matrix-multiplication kernel").
//
// B200's FP64 tensor pipe is at its ceiling on config 5 (0.90 of 37 TFLOP/s, profiles/r02_cfg5_large_step_full.md); its
// int8 tensor pipe is two orders of magnitude faster.  A complex FP64 product C = F X is evaluated EXACTLY up to the
// truncation of its operands to 7 S - 1 bits below the largest entry of each row of F / column of X:
//     a_ik = 2^(eA_i) sum_t q^A_t 2^(-7 (t + 1)),   b_kj = 2^(eB_j) sum_u q^B_u 2^(-7 (u + 1)),   |q| <= 64  (int8 slices),
//     C_ij = 2^(eA_i + eB_j - 14) sum_{dg < S} 2^(-7 dg) D_dg,     D_dg = sum_{t + u = dg} sum_k q^A_t,ik q^B_u,kj   (int32, exact),
// complex as [Cr; Ci] = [Fr Xr + Fi (-Xi); Fi Xr + Fr Xi] (the minus sign lives in a third set of X planes).  Every D_dg is one
// accumulation chain of tcgen05.mma.kind::i8 (M = 128, N = 128, K = 32) into TMEM; |D_dg| <= 7 * 2 * 3003 * 64 * 64 < 2^31.
// A CTA owns one 128 x 128 tile of Cr or Ci: warp 0 feeds a 5-stage shared-memory ring with TMA (128-byte swizzled boxes of
// the K-major slice planes), one thread of warp 1 issues the MMAs and commits stages / accumulators to mbarriers, warps 2-9
// drain the double-buffered TMEM accumulator with tcgen05.ld, weight the diagonals in FP64 registers, and finish the step exactly
// like large_step_kernel (propagator mantissa per row, store, largest row exponent by atomicMax).
#pragma once
#include <cuda.h>

#include "chain_large.cuh"
#include "lazy.cuh"

namespace ctqmc {

constexpr int kSpM = 128, kSpN = 128, kSpKB = 128;        // tile, bytes of K per stage row (= 128 int8 = 4 MMAs of K = 32)
constexpr int kSpStages = 5;
constexpr int kSpStageBytes = (kSpM + kSpN) * kSpKB;      // 32 KB
constexpr int kSpThreads = 320;                           // producer warp, MMA warp, 8 epilogue warps
constexpr int kSpMaxSlices = 8;
constexpr size_t kSpSmemBytes = (size_t)kSpStages * kSpStageBytes + 1024;   // + alignment slack

// ---- tcgen05 / TMEM primitives (inline PTX; sm_100a)
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_alloc(unsigned* dst_smem, int cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned taddr, int cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
// D[tmem] (+)= A[smem] B[smem], int8 x int8 -> int32, issued by ONE thread
__device__ __forceinline__ void tc_mma_i8(unsigned tmem_d, unsigned long long adesc, unsigned long long bdesc, unsigned idesc, unsigned accumulate) {
  asm volatile(
      "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}"
      ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// all MMAs issued so far by this thread arrive on `bar` when they have completed (implies fence::before_thread_sync)
__device__ __forceinline__ void tc_commit(unsigned long long* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// this thread's TMEM lane, 32 consecutive 32-bit columns
__device__ __forceinline__ void tmem_ld32(unsigned taddr, int (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,"
      "%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]),
        "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]),
        "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]),
        "=r"(v[31])
      : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// shared-memory matrix descriptor: K-major operand, 128-byte swizzle, rows of 128 bytes, 8-row groups 1024 bytes apart
__device__ __forceinline__ unsigned long long sp_smem_desc(unsigned saddr) {
  return (unsigned long long)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((unsigned long long)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor: S32 accumulate, signed 8-bit A and B, both K-major, N = 128, M = 128
constexpr unsigned kSpIdesc = (2u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(kSpN >> 3) << 17) | ((unsigned)(kSpM >> 4) << 24);

// ---- slicing: one vector (a row of F, or a column of X with the deferred row scaling of the previous step) per CTA.
// v_k = 2^e sum_t q_t[k] 2^(-7 (t + 1)), e = exponent of the largest |re| / |im| of the vector + 2, |q_t| <= 64.
struct SliceOut {
  signed char* re; signed char* im; signed char* nim;   // plane bases of THIS vector's row for slice 0 (nim may be null)
  long long slice_stride;                               // bytes between consecutive slices of a plane
  int kpad;                                             // bytes to fill (zero beyond the vector's length)
};
template <class Scale>
__device__ __forceinline__ void sp_slice_vector(const double* src, long long stride /*doubles between elements*/, int len, Scale kscale,
                                                int S, const SliceOut& o, int* e_out, int* redi) {
  double mx = 0.0;
  for (int k = threadIdx.x; k < len; k += blockDim.x) {
    const double f = kscale(k);
    mx = fmax(mx, fmax(fabs(src[k * stride] * f), fabs(src[k * stride + 1] * f)));
  }
  int ex = mx > 0.0 ? ilogb(mx) : INT_MIN;
  ex = lz_block_max(ex, redi);
  const int e = ex == INT_MIN ? 0 : ex + 2;
  if (threadIdx.x == 0) *e_out = e;
  for (int k = threadIdx.x; k < o.kpad; k += blockDim.x) {
    double rr = 0.0, ri = 0.0;
    if (k < len) {
      const double f = kscale(k);
      rr = scalbn(src[k * stride] * f, -e); ri = scalbn(src[k * stride + 1] * f, -e);
    }
    for (int t = 0; t < S; ++t) {
      rr *= 128.0; ri *= 128.0;
      const double qr = rint(rr), qi = rint(ri);
      rr -= qr; ri -= qi;
      o.re[t * o.slice_stride + k] = (signed char)(int)qr;
      o.im[t * o.slice_stride + k] = (signed char)(int)qi;
      if (o.nim) o.nim[t * o.slice_stride + k] = (signed char)(-(int)qi);
    }
  }
}

struct SplitStore {          // int8 slice planes of the operator store, built at load
  signed char* planes;       // block b at a_off[b]: [2 (re, im)][S][Mpad_b][Kpad_b]
  const long long* a_off;    // [n_blocks]
  int* ea;                   // row exponents, block b at ea_off[b] (Mpad_b entries)
  const long long* ea_off;
  int S;
};
__host__ __device__ inline int sp_pad(int x) { return (x + 127) / 128 * 128; }

// grid (Mpad, n_blocks): rows beyond the block stay zero (the planes are zeroed once)
__global__ void split_slice_store_kernel(DevImp imp, SplitStore st) {
  __shared__ int redi[32];
  const BlkDesc bd = imp.blks[blockIdx.y];
  const int i = blockIdx.x;
  if (i >= bd.rows) return;
  const int Mp = sp_pad(bd.rows), Kp = sp_pad(bd.cols);
  signed char* base = st.planes + st.a_off[blockIdx.y];
  SliceOut o;
  o.slice_stride = (long long)Mp * Kp;
  o.re = base + (long long)i * Kp; o.im = base + (long long)st.S * o.slice_stride + (long long)i * Kp; o.nim = nullptr; o.kpad = Kp;
  sp_slice_vector(imp.store + bd.off + (long long)i * bd.ld * 2, 2, bd.cols, [](int) { return 1.0; }, st.S, o, st.ea + st.ea_off[blockIdx.y] + i, redi);
}

struct SplitStepParams {
  SplitStore st;
  signed char* bplanes;      // per unit: [3 (Xr, Xi, -Xi)][S][Npad][Kpad]
  int* eb;                   // [units][Npad] column exponents
  int Npad, Kpad;            // sp_pad(widest carried matrix), sp_pad(d_max)
  const CUtensorMap* amaps8; // [n_blocks] uint8 maps of the slice planes (inner Kpad_b bytes, outer 2 S Mpad_b rows)
};

// columns of the carried matrix of every unit -> int8 slice planes, with the exact power-of-two row factor of the previous
// step (row exponent minus its largest, a4) folded in, as large_step_kernel does while loading its B fragments
__global__ void split_slice_x_kernel(LargeParams P, SplitStepParams Q, int j) {
  __shared__ int redi[32];
  const int s = blockIdx.y, n = blockIdx.x;
  if (j >= P.u_n[s] || n >= P.u_c[s]) return;
  const int blk = P.plan_blk[(size_t)s * P.Lmax + j];
  const BlkDesc bd = P.imp.blks[blk];
  const int d = bd.cols;
  const long long xcol_in = P.u_x[s] + (long long)(j & 1) * P.u_w[s];
  const double* col = P.X + ((size_t)(xcol_in + n) * P.ldx) * 2;
  int kprev = 0;
  double dprev = 0.0;
  if (j > 0) { kprev = P.kmax[(size_t)s * P.Lmax + j - 1]; dprev = P.plan_delta[(size_t)s * P.Lmax + j - 1]; }
  const double* Eq = P.imp.energy + P.imp.e_off[bd.src];
  const double emin = P.imp.e_min[bd.src];
  auto scale = [&](int k) {
    if (kprev == INT_MIN) return 0.0;
    if (j == 0) return 1.0;
    const long long sh = (long long)row_exp(prop_x(dprev, Eq[k], emin)) - (long long)kprev;
    return (sh < -1022) ? 0.0 : pow2i((int)min(sh, 1022LL));
  };
  const long long row_bytes = Q.Kpad, plane = (long long)Q.st.S * Q.Npad * row_bytes;
  signed char* base = Q.bplanes + (long long)s * 3 * plane + (long long)n * row_bytes;
  SliceOut o;
  o.slice_stride = (long long)Q.Npad * row_bytes;
  o.re = base; o.im = base + plane; o.nim = base + 2 * plane; o.kpad = sp_pad(d);
  sp_slice_vector(col, 2, d, scale, Q.st.S, o, Q.eb + (size_t)s * Q.Npad + n, redi);
}

// One chain position of every unit on the int8 tensor pipe.  blockIdx.x = (mt * NTmax + nt) * 2 + part (0: real, 1: imaginary
// part of the result tile), blockIdx.y = unit.
__global__ void __launch_bounds__(kSpThreads, 1) split_step_kernel(const __grid_constant__ CUtensorMap bmap, LargeParams P, SplitStepParams Q, int j, int NTmax) {
  extern __shared__ unsigned char sp_raw[];
  __shared__ __align__(8) unsigned long long full_bar[kSpStages], empty_bar[kSpStages], tfull_bar[2], tempty_bar[2];
  __shared__ unsigned s_tmem;
  const int s = blockIdx.y;
  if (j >= P.u_n[s]) return;
  const int blk = P.plan_blk[(size_t)s * P.Lmax + j];
  const BlkDesc bd = P.imp.blks[blk];
  const int dn = bd.rows, d = bd.cols, c = P.u_c[s];
  const int part = blockIdx.x & 1, tile = blockIdx.x >> 1;
  const int mt0 = tile / NTmax, nt0 = tile - mt0 * NTmax;
  const int m0 = mt0 * kSpM, n0 = nt0 * kSpN;
  if (m0 >= dn || n0 >= c) return;
  unsigned char* smem = reinterpret_cast<unsigned char*>(((uintptr_t)sp_raw + 1023) & ~(uintptr_t)1023);   // 128-byte swizzle atoms are 1024-byte aligned
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int S = Q.st.S;
  const int Mp = sp_pad(dn), nkc = sp_pad(d) / kSpKB;

  if (tid == 0) {
    for (int i = 0; i < kSpStages; ++i) { mbar_init(&full_bar[i], 1); mbar_init(&empty_bar[i], 1); }
    for (int i = 0; i < 2; ++i) { mbar_init(&tfull_bar[i], 1); mbar_init(&tempty_bar[i], 8); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(&s_tmem, 256);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = s_tmem;

  // sub-products of this part: real = Fr Xr + Fi (-Xi), imaginary = Fi Xr + Fr Xi   (A planes: 0 re, 1 im; B planes: 0 Xr, 1 Xi, 2 -Xi)
  const int pa[2] = {part == 0 ? 0 : 1, part == 0 ? 1 : 0};
  const int pb[2] = {0, part == 0 ? 2 : 1};

  if (warp == 0) {
    if (lane == 0) {            // ===== TMA producer
      const CUtensorMap* amap = Q.amaps8 + blk;
      int stage = 0, phase = 0;
      for (int dg = 0; dg < S; ++dg)
        for (int t = 0; t <= dg; ++t)
          for (int sub = 0; sub < 2; ++sub) {
            const int arow = (pa[sub] * S + t) * Mp + m0;
            const int brow = ((s * 3 + pb[sub]) * S + (dg - t)) * Q.Npad + n0;
            for (int kc = 0; kc < nkc; ++kc) {
              mbar_wait(&empty_bar[stage], phase ^ 1);
              unsigned char* As = smem + stage * kSpStageBytes;
              mbar_expect_tx(&full_bar[stage], kSpStageBytes);
              tma_load_2d(As, amap, &full_bar[stage], kc * kSpKB, arow);
              tma_load_2d(As + kSpM * kSpKB, &bmap, &full_bar[stage], kc * kSpKB, brow);
              if (++stage == kSpStages) { stage = 0; phase ^= 1; }
            }
          }
    }
  } else if (warp == 1) {
    if (lane == 0) {            // ===== MMA issuer
      int stage = 0, phase = 0;
      for (int dg = 0; dg < S; ++dg) {
        const int buf = dg & 1;
        mbar_wait(&tempty_bar[buf], ((dg >> 1) & 1) ^ 1);      // the epilogue has drained this accumulator
        tc_fence_after();
        unsigned acc = 0;
        for (int t = 0; t <= dg; ++t)
          for (int sub = 0; sub < 2; ++sub)
            for (int kc = 0; kc < nkc; ++kc) {
              mbar_wait(&full_bar[stage], phase);
              tc_fence_after();
              const unsigned sa = smem_u32(smem + stage * kSpStageBytes);
              const unsigned long long ad = sp_smem_desc(sa), bdsc = sp_smem_desc(sa + kSpM * kSpKB);
#pragma unroll
              for (int k = 0; k < kSpKB / 32; ++k) {
                tc_mma_i8(tmem + buf * kSpN, ad + (unsigned long long)(k * 2), bdsc + (unsigned long long)(k * 2), kSpIdesc, acc);
                acc = 1;
              }
              tc_commit(&empty_bar[stage]);                   // the slot is free once these MMAs have read it
              if (++stage == kSpStages) { stage = 0; phase ^= 1; }
            }
        tc_commit(&tfull_bar[buf]);                           // diagonal dg is complete in TMEM
      }
    }
  } else {
    // ===== epilogue warps: TMEM lane quarter = warp % 4, column half = (warp - 2) / 4
    const int quarter = warp & 3, half = (warp - 2) >> 2;
    const int row = m0 + quarter * 32 + lane;
    double accd[64];
#pragma unroll
    for (int i = 0; i < 64; ++i) accd[i] = 0.0;
    double w = 1.0;
    for (int dg = 0; dg < S; ++dg) {
      const int buf = dg & 1;
      mbar_wait(&tfull_bar[buf], (dg >> 1) & 1);
      tc_fence_after();
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        int v[32];
        tmem_ld32(tmem + ((unsigned)(quarter * 32) << 16) + (unsigned)(buf * kSpN + half * 64 + h * 32), v);
#pragma unroll
        for (int i = 0; i < 32; ++i) accd[h * 32 + i] = fma((double)v[i], w, accd[h * 32 + i]);
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty_bar[buf]);
      w *= 0.0078125;                                         // 2^-7 per diagonal
    }
    // finish as large_step_kernel: exponents of the slices, propagator mantissa of the row, store, largest row exponent
    const double delta = P.plan_delta[(size_t)s * P.Lmax + j];
    const double* E = P.imp.energy + P.imp.e_off[bd.dst];
    const double emin = P.imp.e_min[bd.dst];
    const long long xcol_out = P.u_x[s] + (long long)((j + 1) & 1) * P.u_w[s];
    double* Xout = P.X + (size_t)xcol_out * P.ldx * 2;
    int wexp = INT_MIN;
    if (row < dn) {
      const double x = prop_x(delta, E[row], emin);
      const double mr = exp2(__dsub_rn(x, floor(x)));
      const int kr = row_exp(x);
      const int ea = Q.st.ea[Q.st.ea_off[blk] + row];
      const int* eb = Q.eb + (size_t)s * Q.Npad + n0 + half * 64;
      double rmax = 0.0;
#pragma unroll
      for (int i = 0; i < 64; ++i) {
        const int col = n0 + half * 64 + i;
        if (col < c) {
          const double v = scalbn(accd[i], ea + eb[i] - 14) * mr;
          Xout[((size_t)col * P.ldx + row) * 2 + part] = v;
          rmax = fmax(rmax, fabs(v));
        }
      }
      if (rmax > 0.0) wexp = kr + ilogb(rmax);
    }
    wexp = __reduce_max_sync(0xffffffffu, wexp);
    if (lane == 0 && wexp != INT_MIN) atomicMax(&P.kmax[(size_t)s * P.Lmax + j], wexp);
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 256);
}

}  // namespace ctqmc
