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
// Work is cut into items of one 128-row tile x one group of up to four diagonals x one 128-column tile of [Cr; Ci]; the items of a
// chain position are listed heaviest first (split_list_kernel) and persistent CTAs (one per SM) take them from an atomic counter
// through a four-deep queue.  Per item and 32-byte K chunk ONE 1-D bulk copy per operand brings all slices the group needs into a
// shared-memory stage (the planes are stored as the tensor core's shared-memory image, 32-byte swizzle pre-applied, so the copies
// move whole 128-byte lines); warp 0 fetches items and copies X slices, warp 10 copies F slices, one thread of warp 1 issues the
// MMAs as straight-line code (compile-time (t, u) pattern, neighbouring X slices paired into N = 256) and commits stages /
// accumulators to mbarriers, warps 2-9 drain the TMEM accumulators (4 diagonals side by side = 512 columns) with tcgen05.ld,
// weight the diagonals in FP64 registers, and finish the step exactly like large_step_kernel (propagator mantissa per row,
// store, largest row exponent by atomicMax).  History and measurements: profiles/r02_split_step.md.
#pragma once
#include <cuda.h>

#include "chain_large.cuh"
#include "lazy.cuh"

namespace ctqmc {

constexpr int kSpM = 128, kSpN = 128;                     // output tile of one MMA accumulator
constexpr int kSpThreads = 352;                           // B-producer warp, MMA warp, 8 epilogue warps, A-producer warp
constexpr int kSpMaxSlices = 8;

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
// instruction descriptor: S32 accumulate, signed 8-bit A and B, both K-major, N = 128, M = 128
constexpr unsigned kSpIdesc = (2u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(kSpN >> 3) << 17) | ((unsigned)(kSpM >> 4) << 24);
constexpr unsigned kSpIdesc256 = (2u << 4) | (1u << 7) | (1u << 10) | ((unsigned)(256 >> 3) << 17) | ((unsigned)(kSpM >> 4) << 24);   // N = 256

// ---- slicing: one vector (a row of F, or a column of X with the deferred row scaling of the previous step) per CTA.
// v_k = 2^e sum_t q_t[k] 2^(-7 (t + 1)), e = exponent of the largest |re| / |im| of the vector + 2, |q_t| <= 64.
// Plane layout = the shared-memory image the tensor core reads, tile by tile: [128-row tile][K chunk of 32 bytes][slice][4 KB], the
// 4 KB being 128 rows x 32 bytes with the 32-byte swizzle applied (16-byte halves of a row exchanged when bit 2 of the row is set).
// All slices of one (row tile, K chunk) are contiguous, so a stage is filled by ONE 1-D bulk copy per operand, in whole 128-byte lines.
struct SliceOut {
  signed char* re; signed char* im; signed char* nim;   // plane bases (nim may be null)
  int S, nkc;                                           // slices, K chunks per row of the plane
  int row;                                              // this vector's row in the plane
  int kpad;                                             // bytes to fill (zero beyond the vector's length)
};
__device__ __forceinline__ long long sp_image_index(int k, int row, int t, int S, int nkc) {
  const int r = row & 127;
  return ((((long long)(row >> 7) * nkc + (k >> 5)) * S + t) << 12) + r * 32 + ((((k >> 4) & 1) ^ ((r >> 2) & 1)) << 4) + (k & 15);
}
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
      const long long at = sp_image_index(k, o.row, t, o.S, o.nkc);
      o.re[at] = (signed char)(int)qr;
      o.im[at] = (signed char)(int)qi;
      if (o.nim) o.nim[at] = (signed char)(-(int)qi);
    }
  }
}

struct SplitStore {          // int8 slice planes of the operator store, built at load
  signed char* planes;       // block b at a_off[b]: [2 (re, im)] images of S * Mpad_b * Kpad_b bytes (sp_image_index)
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
  o.re = base; o.im = base + (long long)st.S * Mp * Kp; o.nim = nullptr; o.kpad = Kp; o.S = st.S; o.nkc = Kp / 32; o.row = i;
  sp_slice_vector(imp.store + bd.off + (long long)i * bd.ld * 2, 2, bd.cols, [](int) { return 1.0; }, st.S, o, st.ea + st.ea_off[blockIdx.y] + i, redi);
}

struct SplitStepParams {
  SplitStore st;
  signed char* bplanes;      // per unit: [3 (Xr, Xi, -Xi)] images of S * Npad * Kpad bytes (sp_image_index)
  int* eb;                   // [units][Npad] column exponents
  int Npad, Kpad;            // sp_pad(widest carried matrix), sp_pad(d_max)
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
  signed char* base = Q.bplanes + (long long)s * 3 * plane;
  SliceOut o;
  o.re = base; o.im = base + plane; o.nim = base + 2 * plane; o.kpad = sp_pad(d); o.S = Q.st.S; o.nkc = Q.Kpad / 32; o.row = n;
  sp_slice_vector(col, 2, d, scale, Q.st.S, o, Q.eb + (size_t)s * Q.Npad + n, redi);
}

// One chain position of every unit on the int8 tensor pipe; a work item is (unit, 128 x 128 tile, real | imaginary part).
//
// Operand traffic decides this kernel: with one (A slice, B slice) pair fetched per product the ring pulls 17 TB/s out of L2 and
// the tensor pipe waits (57 % busy, profiles/r02_split_step.md).  So the diagonals are evaluated in GROUPS of up to four that are
// accumulated side by side in TMEM (4 x 128 columns): per 32-byte K chunk every slice of both operands the group needs is loaded
// ONCE into one stage and all their pairs t + u in the group's range are issued from shared memory.  The accumulators of a group
// are drained by the epilogue warps before the next group starts.
constexpr int kSpKC = 32;                                  // bytes of K per chunk: one MMA K step, 32-byte swizzle
constexpr int kSpTile = kSpM * kSpKC;                      // 4 KB: one operand tile of one slice
constexpr size_t kSpSmemMax = 226 * 1024;
__host__ __device__ constexpr int sp_stages(int S) { return (int)((kSpSmemMax - 1024) / ((size_t)2 * S * kSpTile)) < 6 ? (int)((kSpSmemMax - 1024) / ((size_t)2 * S * kSpTile)) : 6; }
// the epilogue warps wait for a whole group of diagonals: back off instead of spinning on the issue slots
__device__ __forceinline__ void mbar_wait_sleep(unsigned long long* bar, unsigned parity) {
  unsigned ok = 0;
  while (!ok) {
    asm volatile("{\n.reg .pred P1;\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%1], %2;\nselp.u32 %0, 1, 0, P1;\n}" : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity) : "memory");
    if (!ok) __nanosleep(500);
  }
}
// shared-memory matrix descriptor: K-major, 32-byte swizzle, rows of 32 bytes, 8-row groups 256 bytes apart
__device__ __forceinline__ unsigned long long sp_smem_desc32(unsigned saddr) {
  return (unsigned long long)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | ((unsigned long long)(256 >> 4) << 32) | (1ull << 46) | (6ull << 61);
}
__device__ __forceinline__ void bulk_load(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

struct SpTile { int ok, s, blk, dn, d, c, m0, n0, part, Mp, nch; };
__device__ __forceinline__ SpTile sp_decode(const LargeParams& P, long long w, int tiles_per_unit, int NTmax, int j) {
  SpTile T; T.ok = 0;
  T.s = (int)(w / tiles_per_unit);
  const int r = (int)(w - (long long)T.s * tiles_per_unit);
  if (j >= P.u_n[T.s]) return T;
  T.blk = P.plan_blk[(size_t)T.s * P.Lmax + j];
  const BlkDesc bd = P.imp.blks[T.blk];
  T.dn = bd.rows; T.d = bd.cols; T.c = P.u_c[T.s];
  T.part = r & 1;
  const int tile = r >> 1, mt0 = tile / NTmax, nt0 = tile - mt0 * NTmax;
  T.m0 = mt0 * kSpM; T.n0 = nt0 * kSpN;
  if (T.m0 >= T.dn || T.n0 >= T.c) return T;
  T.Mp = sp_pad(T.dn); T.nch = 2 * (sp_pad(T.d) / kSpKC);            // chunks: both sub-products, one after the other
  T.ok = 1;
  return T;
}

// Work list of one chain position: the (unit, tile, part) items that exist, heaviest (longest contraction) first.  The host only
// knows upper bounds, and launching one CTA per CANDIDATE cost more than the products themselves (a CTA that needs all of an SM's
// shared memory occupies the SM's only slot even if it exits at once: 1.6 ms of a 3.4 ms launch).  One CTA, three passes.
struct SplitList { int* items; int* ctr; };     // items[n], ctr[0] = n, ctr[1] = next item to hand out
__global__ void split_list_kernel(LargeParams P, SplitList W, int j, int tiles_per_unit, int NTmax, long long total) {
  __shared__ int cnt[4], base[4];
  if (threadIdx.x < 4) cnt[threadIdx.x] = 0;
  __syncthreads();
  for (long long w = threadIdx.x; w < total; w += blockDim.x) {
    const SpTile T = sp_decode(P, w, tiles_per_unit, NTmax, j);
    if (T.ok) atomicAdd(&cnt[min(3, (T.nch - 1) / 32)], 1);          // contraction length class (chunks of both sub-products): <= 32, <= 64, <= 96, more
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    int b = 0;
    for (int k = 3; k >= 0; --k) { base[k] = b; b += cnt[k]; cnt[k] = 0; }
    W.ctr[0] = b; W.ctr[1] = 0;
  }
  __syncthreads();
  for (long long w = threadIdx.x; w < total; w += blockDim.x) {
    const SpTile T = sp_decode(P, w, tiles_per_unit, NTmax, j);
    if (T.ok) { const int k = min(3, (T.nch - 1) / 32); W.items[base[k] + atomicAdd(&cnt[k], 1)] = (int)w; }
  }
}

// The MMAs of one K chunk of one group of diagonals: compile-time (t, u) pattern, two neighbouring B slices as one N = 256 operand
// feeding two neighbouring accumulators wherever a slice has a neighbour left.  Straight-line code: the single issuing thread has
// ~100 cycles per instruction (a microbenchmark of the same instruction with ~50 scalar instructions of bookkeeping per product
// ran at a third of the pipe's rate).
template <int S, int G>
__device__ __forceinline__ void sp_issue_chunk(unsigned tmem, unsigned long long a_set, unsigned long long b_set, unsigned accum) {
  constexpr int dg0 = 4 * G, dg1 = (S < dg0 + 4 ? S : dg0 + 4) - 1;
#pragma unroll
  for (int t = 0; t <= dg1; ++t) {
    const unsigned long long ad = a_set + (unsigned long long)(t * (kSpTile >> 4));
    const int ulo = dg0 - t > 0 ? dg0 - t : 0, uhi = dg1 - t;
    const unsigned acc_t = (t == 0) ? accum : 1u;            // t = 0 touches every accumulator of the group first
#pragma unroll
    for (int u = ulo; u <= uhi; u += 2) {
      const unsigned long long bdsc = b_set + (unsigned long long)(u * (kSpTile >> 4));
      const unsigned dst = tmem + (unsigned)((t + u - dg0) * kSpN);
      if (u + 1 <= uhi) tc_mma_i8(dst, ad, bdsc, kSpIdesc256, acc_t);
      else              tc_mma_i8(dst, ad, bdsc, kSpIdesc, acc_t);
    }
  }
}

template <int S>
__global__ void __launch_bounds__(kSpThreads, 1) split_step_kernel(LargeParams P, SplitStepParams Q, int j, int NTmax, int tiles_per_unit, SplitList W) {
  constexpr int NST = sp_stages(S);                            // stages: every stage holds all slices of both operands for one K chunk
  constexpr int n_groups = (S + 3) / 4;
  extern __shared__ unsigned char sp_raw[];
  __shared__ __align__(8) unsigned long long full[NST], empty[NST], tfull_bar, tempty_bar;
  __shared__ __align__(8) unsigned long long qfull[4], qempty[4];
  __shared__ int q_item[4];
  __shared__ unsigned s_tmem;
  // Persistent: one CTA per SM takes items off the work list (atomic counter); the B producer fetches them and hands them to the A
  // producer, the MMA thread and the epilogue warps through a four-deep queue, so barriers, the TMEM allocation and the ring / phase
  // counters live across items and the epilogue's final store of one item overlaps the next item's first products.
  unsigned char* smem = reinterpret_cast<unsigned char*>(((uintptr_t)sp_raw + 1023) & ~(uintptr_t)1023);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  unsigned char* sA = smem;                                        // [NST][S] tiles
  unsigned char* sB = smem + NST * S * kSpTile;                    // [NST][S] tiles

  if (tid == 0) {
    for (int i = 0; i < NST; ++i) { mbar_init(&full[i], 2); mbar_init(&empty[i], 1); }      // both producers arm a stage; one commit frees it
    mbar_init(&tfull_bar, 1); mbar_init(&tempty_bar, 8);
    for (int i = 0; i < 4; ++i) { mbar_init(&qfull[i], 1); mbar_init(&qempty[i], 10); }    // consumers: A producer, MMA thread, 8 epilogue warps
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) tmem_alloc(&s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const unsigned tmem = s_tmem;

  if (warp == 0) {
    if (lane == 0) {            // ===== work-item fetch + producer of the B slices (one bulk copy per K chunk: all slices of the group)
      int stage = 0, phase = 0;
      const int n_items = W.ctr[0];
      for (int qn = 0;; ++qn) {
        mbar_wait(&qempty[qn & 3], ((qn >> 2) & 1) ^ 1);
        const int it = atomicAdd(&W.ctr[1], 1);
        const int wi = it < n_items ? W.items[it] : -1;
        q_item[qn & 3] = wi;
        mbar_arrive(&qfull[qn & 3]);
        if (wi < 0) break;
        const SpTile T = sp_decode(P, wi, tiles_per_unit, NTmax, j);
        const int half_ch = T.nch >> 1;
        // sub-products of this part: real = Fr Xr + Fi (-Xi), imaginary = Fi Xr + Fr Xi   (A planes: 0 re, 1 im; B planes: 0 Xr, 1 Xi, 2 -Xi)
        const int pb[2] = {0, T.part == 0 ? 2 : 1};
        for (int g = 0; g < n_groups; ++g) {
          const int ns = g == 0 ? (S < 4 ? S : 4) : S;             // slices 0 .. ns-1 of both operands feed this group's diagonals
          const int nkc = Q.Kpad / kSpKC;
          for (int ch = 0; ch < T.nch; ++ch) {
            const int sub = ch >= half_ch, kc = sub ? ch - half_ch : ch;
            const signed char* src = Q.bplanes + ((long long)(T.s * 3 + pb[sub]) * Q.Npad * Q.Kpad) * S + ((((long long)(T.n0 >> 7) * nkc + kc) * S) << 12);
            mbar_wait(&empty[stage], phase ^ 1);
            mbar_expect_tx(&full[stage], (unsigned)(ns * kSpTile));
            bulk_load(sB + stage * S * kSpTile, src, (unsigned)(ns * kSpTile), &full[stage]);
            if (++stage == NST) { stage = 0; phase ^= 1; }
          }
        }
      }
    }
  } else if (warp == 10) {
    if (lane == 0) {            // ===== producer of the A slices (its own thread: the two operand streams never wait for each other)
      int stage = 0, phase = 0;
      for (int qn = 0;; ++qn) {
        mbar_wait(&qfull[qn & 3], (qn >> 2) & 1);
        const int wi = q_item[qn & 3];
        mbar_arrive(&qempty[qn & 3]);
        if (wi < 0) break;
        const SpTile T = sp_decode(P, wi, tiles_per_unit, NTmax, j);
        const int half_ch = T.nch >> 1;
        const int pa[2] = {T.part == 0 ? 0 : 1, T.part == 0 ? 1 : 0};
        for (int g = 0; g < n_groups; ++g) {
          const int ns = g == 0 ? (S < 4 ? S : 4) : S;
          const int nkc = sp_pad(T.d) / kSpKC;
          const signed char* ablk = Q.st.planes + Q.st.a_off[T.blk];
          for (int ch = 0; ch < T.nch; ++ch) {
            const int sub = ch >= half_ch, kc = sub ? ch - half_ch : ch;
            const signed char* src = ablk + (long long)pa[sub] * S * T.Mp * sp_pad(T.d) + ((((long long)(T.m0 >> 7) * nkc + kc) * S) << 12);
            mbar_wait(&empty[stage], phase ^ 1);
            mbar_expect_tx(&full[stage], (unsigned)(ns * kSpTile));
            bulk_load(sA + stage * S * kSpTile, src, (unsigned)(ns * kSpTile), &full[stage]);
            if (++stage == NST) { stage = 0; phase ^= 1; }
          }
        }
      }
    }
  } else if (warp == 1) {
    if (lane == 0) {            // ===== MMA issuer
      int stage = 0, phase = 0, gcount = 0;
      const unsigned long long a_base = sp_smem_desc32(smem_u32(sA)), b_base = sp_smem_desc32(smem_u32(sB));
      for (int qn = 0;; ++qn) {
        mbar_wait(&qfull[qn & 3], (qn >> 2) & 1);
        const int wi = q_item[qn & 3];
        mbar_arrive(&qempty[qn & 3]);
        if (wi < 0) break;
        const SpTile T = sp_decode(P, wi, tiles_per_unit, NTmax, j);
        const int nch = T.nch;
#pragma unroll
        for (int g = 0; g < n_groups; ++g, ++gcount) {
          mbar_wait(&tempty_bar, (gcount & 1) ^ 1);                // the epilogue has drained the previous group's accumulators
          tc_fence_after();
          for (int ch = 0; ch < nch; ++ch) {
            mbar_wait(&full[stage], phase);
            tc_fence_after();
            const unsigned long long off = (unsigned long long)(stage * S * (kSpTile >> 4));
            if (g == 0) sp_issue_chunk<S, 0>(tmem, a_base + off, b_base + off, ch > 0 ? 1u : 0u);
            else        sp_issue_chunk<S, 1>(tmem, a_base + off, b_base + off, ch > 0 ? 1u : 0u);
            tc_commit(&empty[stage]);                             // the stage is free once these MMAs have read it
            if (++stage == NST) { stage = 0; phase ^= 1; }
          }
          tc_commit(&tfull_bar);                                   // the group's diagonals are complete in TMEM
        }
      }
    }
  } else if (warp >= 2) {
    // ===== epilogue warps: TMEM lane quarter = warp % 4, column half = (warp - 2) / 4
    const int quarter = warp & 3, half = (warp - 2) >> 2;
    int gcount = 0;
    for (int qn = 0;; ++qn) {
    mbar_wait_sleep(&qfull[qn & 3], (qn >> 2) & 1);
    const int wi = q_item[qn & 3];
    __syncwarp();
    if (lane == 0) mbar_arrive(&qempty[qn & 3]);
    if (wi < 0) break;
    const SpTile T = sp_decode(P, wi, tiles_per_unit, NTmax, j);
    const int s = T.s, blk = T.blk, dn = T.dn, c = T.c, m0 = T.m0, n0 = T.n0, part = T.part;
    const BlkDesc bd = P.imp.blks[blk];
    const int row = m0 + quarter * 32 + lane;
    double accd[64];
#pragma unroll
    for (int i = 0; i < 64; ++i) accd[i] = 0.0;
    double wgt = 1.0;
    for (int g = 0; g < n_groups; ++g, ++gcount) {
      const int dg0 = 4 * g, dg1 = min(S, dg0 + 4) - 1;
      mbar_wait_sleep(&tfull_bar, gcount & 1);
      tc_fence_after();
      for (int a = 0; a <= dg1 - dg0; ++a) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          int v[32];
          tmem_ld32(tmem + ((unsigned)(quarter * 32) << 16) + (unsigned)(a * kSpN + half * 64 + h * 32), v);
#pragma unroll
          for (int i = 0; i < 32; ++i) accd[h * 32 + i] = fma((double)v[i], wgt, accd[h * 32 + i]);
        }
        wgt *= 0.0078125;                                            // 2^-7 per diagonal
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(&tempty_bar);
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
          const int sh = ea + eb[i] - 14;
          const double v = ((sh >= -1000 && sh <= 1000) ? accd[i] * pow2i(sh) : scalbn(accd[i], sh)) * mr;
          Xout[((size_t)col * P.ldx + row) * 2 + part] = v;
          rmax = fmax(rmax, fabs(v));
        }
      }
      if (rmax > 0.0) wexp = kr + ilogb(rmax);
    }
    wexp = __reduce_max_sync(0xffffffffu, wexp);
    if (lane == 0 && wexp != INT_MIN) atomicMax(&P.kmax[(size_t)s * P.Lmax + j], wexp);
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem, 512);
}

}  // namespace ctqmc
