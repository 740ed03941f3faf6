// Incremental, lazy local trace for many Markov chains at once (PAPER.md:540 stored sub-products in a
// balanced tree, :542-548 lazy trace, :560-574 many chains in flight on one device with a pre-allocated block).
//
// Every chain owns a complete binary tree over a fixed dyadic partition of [0, beta) (readings F1-F4): node
// (l, i) stores, for every sector q that survives it, the evolution operator across its interval as a dense matrix
// U(q) (dim[tgt] x dim[q], column-major) with an integer exponent e, a real exponent lg, the target sector and the Frobenius
// norm.  A proposal (operators to insert / remove) dirties the leaves that contain its times and their ancestors; their new
// contents are built in SHADOW slots taken from the chain's free list, so a rejected proposal costs nothing to undo and an
// accepted one is committed by swapping slot indices.  All chains advance in lock-step through the same launches (the
// B200 recast of the paper's stream-per-chain round robin): a launch covers (tile, chain x dirty node, sector) and CTAs whose
// chain has nothing to do at that point exit at once, so nothing is ever read back by the host.
#pragma once
#include <climits>

#include "common.cuh"
#include "reduce.cuh"

namespace ctqmc {

constexpr int kLzTile = 64;      // CTA tile of the node products
constexpr int kLzKC = 16;        // contraction chunk staged in shared memory
constexpr int kLzThreads = 256;
constexpr int kLzMaxDim = 512;   // sector dimensions beyond this do not fit the per-chain node storage anyway

struct LazyView {
  DevImp imp;
  double beta;
  int nC;                 // chains
  int D, nleaf, nnode;    // depth, 2^D leaves, 2^(D+1) - 1 nodes (heap order: children of n are 2n+1, 2n+2)
  int cap;                // operators a leaf can hold
  int emax;               // edits per proposal
  int smax;               // shadow slots per chain = emax * (D + 1)
  int NN;                 // physical slots per chain = nnode + smax + emax (the last emax: leaf ping-pong scratch)
  int ldm;                // leading dimension of every stored matrix (elements)
  long long node_elems;   // doubles per slot = n_energy * ldm * (1 | 2)
  // configuration: operators of every leaf, time-ordered
  int* leaf_n; double* leaf_tau; int* leaf_sym;
  // tree
  int* slot_of;           // [nC][nnode] physical slot of each node
  int* free_slot;         // [nC][smax + emax]
  // entries [nC][NN][Q]
  int* ent_tgt; int* ent_valid; int* ent_k; long long* ent_e; double* ent_lg; double* ent_nrm;
  double* mats;
  // proposal state
  int* p_status; int* p_ndirty; int* p_nleaf; int* p_node;   // p_node [nC][smax]: dirty nodes, leaves first, then level by level
  int* sh_n; double* sh_tau; int* sh_sym;                    // [nC][emax](x cap) shadow leaves
  double* sb_m; long long* sb_e; int* order; int* n_alive;   // [nC][Q] sector bounds, evaluation order
  int* decided; int* decided_by; int* n_eval;                // 0 undecided / 1 accept / 2 reject;  0 bound / 1 partial / 2 full
  double* term_re; double* term_im; long long* term_e;       // [nC][Q] exact sector terms in evaluation order
  double* thr;
  int* p_accept;                                             // accept flags of the last proposal (commit's default mask)
  unsigned long long* n_products;
  int* p_lvl_start; int* p_lvl_cnt;                          // [nC][D]: where the dirty ancestors of a level sit in p_node
  // Work lists, built on the device (the host only knows bounds): what is launched per step is a fixed number of persistent
  // CTAs that walk a compact list, so a step in which few chains (or none) have work costs a few microseconds instead of one
  // CTA per candidate.  Leaf lists rotate over three buffers (step j reads j % 3, the fix of step j fills (j + 1) % 3, the
  // step kernel clears (j + 2) % 3), node lists over two (parity of the host's launch sequence number).
  int* w_cnt;                                                // [0..2] leaf tasks, [3..5] leaf tiles, [6..7] node tasks, [8..9] node tiles,
                                                             // [10..12] / [13..14] next tile to hand out (leaf / node product kernels)
  int4* w_ltask; int4* w_ltile; int4* w_ntask; int4* w_ntile;
  int* w_larr; int* w_narr; double* w_part;                  // tiles of a task that have been rescaled; their partial sums of squares
  long long w_task_cap, w_tile_cap;                          // entries per buffer
};

struct LazyEdits {
  const long long* offset; const double* tau; const int* sym; const int* kind; long long n_edits;
};

// 64 x 64 tiles of an M x N result appended to a tile list (one thread)
__device__ __forceinline__ void lz_push_tiles(int* cnt, int4* tiles, int task, int M, int N) {
  const int tm = (M + kLzTile - 1) / kLzTile, tn = (N + kLzTile - 1) / kLzTile;
  const int base = atomicAdd(cnt, tm * tn);
  for (int i = 0; i < tm * tn; ++i) tiles[base + i] = make_int4(task, (i / tn) * kLzTile, (i % tn) * kLzTile, i);
}

// ------------------------------------------------------------------------------------------------ small helpers
__device__ __forceinline__ int lz_level(int node) { return 31 - __clz(node + 1); }

__device__ __forceinline__ int lz_leaf_of(const LazyView& V, double t) {
  int l = (int)(t / V.beta * (double)V.nleaf);
  return l < V.nleaf - 1 ? l : V.nleaf - 1;
}
__device__ __forceinline__ double lz_edge(const LazyView& V, int i) { return (double)i * V.beta / (double)V.nleaf; }

__device__ __forceinline__ int lz_dirty_index(const LazyView& V, int c, int node) {
  const int n = V.p_ndirty[c];
  const int* pn = V.p_node + (size_t)c * V.smax;
  for (int i = 0; i < n; ++i) if (pn[i] == node) return i;
  return -1;
}
// physical slot of `node` as the current proposal sees it (its shadow if dirty)
__device__ __forceinline__ int lz_slot(const LazyView& V, int c, int node) {
  const int di = lz_dirty_index(V, c, node);
  return di >= 0 ? V.free_slot[(size_t)c * (V.smax + V.emax) + di] : V.slot_of[(size_t)c * V.nnode + node];
}
__device__ __forceinline__ size_t lz_ent(const LazyView& V, int c, int slot, int q) { return ((size_t)c * V.NN + slot) * V.imp.Q + q; }
__device__ __forceinline__ double* lz_mat(const LazyView& V, int c, int slot, int q) {
  return V.mats + ((size_t)c * V.NN + slot) * V.node_elems + (size_t)V.imp.e_off[q] * V.ldm * (V.imp.cplx ? 2 : 1);
}

__device__ __forceinline__ double lz_scale(double v, int sh) {
  if (sh >= -1022 && sh <= 1022) return v * pow2i(sh);
  return scalbn(v, max(sh, -2200));
}

// sum of z_s 2^e_s aligned to the largest exponent (Neumaier), normalised so that max(|re|, |im|) is in [1, 2)
struct LzC { double re, im; long long e; };
__device__ inline LzC lz_norm(double re, double im, long long e) {
  LzC r; r.re = re; r.im = im; r.e = 0;
  const double mx = fmax(fabs(re), fabs(im));
  if (mx == 0.0 || !isfinite(mx)) return r;
  const int k = ilogb(mx);
  r.re = scalbn(re, -k); r.im = scalbn(im, -k); r.e = e + k;
  return r;
}
__device__ inline LzC lz_apply_lg(double re, double im, long long e, double lg) {
  const double kf = floor(lg), f = exp2(lg - kf);
  return lz_norm(re * f, im * f, e + (long long)kf);
}
template <class F>
__device__ inline LzC lz_sum(int n, F item) {
  bool any = false; long long emax = 0;
  for (int i = 0; i < n; ++i) { const LzC z = item(i); if (z.re != 0.0 || z.im != 0.0) { emax = any ? max(emax, z.e) : z.e; any = true; } }
  if (!any) { LzC r; r.re = 0.0; r.im = 0.0; r.e = 0; return r; }
  double re = 0.0, im = 0.0, cr = 0.0, ci = 0.0;
  for (int i = 0; i < n; ++i) {
    const LzC z = item(i);
    if (z.re == 0.0 && z.im == 0.0) continue;
    const double xr = shift_clamped(z.re, z.e - emax), xi = shift_clamped(z.im, z.e - emax);
    const double tr = re + xr; cr += (fabs(re) >= fabs(xr)) ? (re - tr) + xr : (xr - tr) + re; re = tr;
    const double ti = im + xi; ci += (fabs(im) >= fabs(xi)) ? (im - ti) + xi : (xi - ti) + im; im = ti;
  }
  return lz_norm(re + cr, im + ci, emax);
}
__device__ inline double lz_log2(double m, long long e) { return m == 0.0 ? -INFINITY : log2(fabs(m)) + (double)e; }

__device__ inline double lz_block_sum(double v, double* red) {
  v = warp_sum(v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  double t = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
  return t;
}
__device__ inline int lz_block_max(int v, int* red) {
  v = __reduce_max_sync(0xffffffffu, v);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  int t = INT_MIN;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t = max(t, red[w]);
  return t;
}

// ------------------------------------------------------------------------------------------------ node product tile
// C (M x N, column-major ldc) = [diag(2^x mantissas)] A (M x K, element (r, k) at A[(r a_rs + k a_cs) ES]) B (K x N, column-
// major ldb with contraction stride b_ks, or -- B == nullptr -- the diagonal propagator P_delta of a sector).  64 x 64 tile per CTA, 8 warps of 16 x 32,
// FP64 tensor-core mma (DMMA m8n8k4), operands staged in shared memory with bounds guards (sector dimensions are arbitrary).
// The largest binary exponent of the tile's non-zero results (plus the row exponent of the propagator) goes to *kmax_out.
template <bool CPLX>
struct LzSmem {
  double A[CPLX ? 2 : 1][kLzTile][kLzKC + 4];   // row stride 20 doubles: the 16 lanes of a half-warp (rows g..g+3, k..k+3) hit 16 different banks
  double B[CPLX ? 2 : 1][kLzTile][kLzKC + 4];
  double rowm[kLzTile];
  int rowk[kLzTile];
};

struct LzDiag { double delta; const double* E; double emin; int kmax; };
struct LzRowScale { int on; double delta; const double* E; double emin; };

__device__ __forceinline__ double lz_diag_value(const LzDiag& d, int n) {
  const double x = prop_x(d.delta, d.E[n], d.emin);
  const int sh = row_exp(x) - d.kmax;
  return sh < -1022 ? 0.0 : exp2(__dsub_rn(x, floor(x))) * pow2i(min(sh, 0));
}

template <bool CPLX>
__device__ void lz_gemm_tile(LzSmem<CPLX>& S, int m0, int n0, int M, int N, int K, const double* __restrict__ A, long long a_rs,
                             long long a_cs, const double* __restrict__ B, int ldb, LzDiag dg, double* __restrict__ Cm, int ldc,
                             LzRowScale rs, int* kmax_out, int b_ks = 1) {
  constexpr int ES = CPLX ? 2 : 1;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int wm = warp & 3, wn = warp >> 2, g = lane >> 2, t = lane & 3;
  if (tid < kLzTile) {
    double mr = 1.0; int kr = 0;
    if (rs.on && m0 + tid < M) {
      const double x = prop_x(rs.delta, rs.E[m0 + tid], rs.emin);
      mr = exp2(__dsub_rn(x, floor(x))); kr = row_exp(x);
    }
    S.rowm[tid] = mr; S.rowk[tid] = kr;
  }
  double acc[2][4][CPLX ? 4 : 2];
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int x = 0; x < (CPLX ? 4 : 2); ++x) acc[mi][ni][x] = 0.0;

  // the next K chunk travels from global memory to registers while the tensor cores work on the current one
  constexpr int kPer = kLzTile * kLzKC / kLzThreads;      // staged values per thread, operand and chunk
  double pa[kPer], pai[kPer], pb[kPer], pbi[kPer];
  auto fetch = [&](int k0) {
#pragma unroll
    for (int u = 0; u < kPer; ++u) {
      const int idx = tid + u * kLzThreads;
      int r, kk;
      if (a_cs == 1) { r = idx / kLzKC; kk = idx % kLzKC; } else { r = idx % kLzTile; kk = idx / kLzTile; }
      double vr = 0.0, vi = 0.0;
      if (m0 + r < M && k0 + kk < K) {
        const double* p = A + ((long long)(m0 + r) * a_rs + (long long)(k0 + kk) * a_cs) * ES;
        vr = p[0]; if (CPLX) vi = p[1];
      }
      pa[u] = vr; pai[u] = vi;
      const int kb = idx % kLzKC, nn = idx / kLzKC;
      vr = 0.0; vi = 0.0;
      if (n0 + nn < N && k0 + kb < K) {
        if (B) { const double* p = B + ((long long)(n0 + nn) * ldb + (long long)(k0 + kb) * b_ks) * ES; vr = p[0]; if (CPLX) vi = p[1]; }
        else if (n0 + nn == k0 + kb) vr = lz_diag_value(dg, n0 + nn);
      }
      pb[u] = vr; pbi[u] = vi;
    }
  };
  fetch(0);
  for (int k0 = 0; k0 < K; k0 += kLzKC) {
    __syncthreads();
#pragma unroll
    for (int u = 0; u < kPer; ++u) {
      const int idx = tid + u * kLzThreads;
      int r, kk;
      if (a_cs == 1) { r = idx / kLzKC; kk = idx % kLzKC; } else { r = idx % kLzTile; kk = idx / kLzTile; }
      S.A[0][r][kk] = pa[u]; if (CPLX) S.A[CPLX ? 1 : 0][r][kk] = pai[u];
      S.B[0][idx / kLzKC][idx % kLzKC] = pb[u]; if (CPLX) S.B[CPLX ? 1 : 0][idx / kLzKC][idx % kLzKC] = pbi[u];
    }
    if (k0 + kLzKC < K) fetch(k0 + kLzKC);
    __syncthreads();
#pragma unroll
    for (int ks = 0; ks < kLzKC; ks += 4) {
      double ar[2], ai[2], br[4], bi[4];
#pragma unroll
      for (int mi = 0; mi < 2; ++mi) { ar[mi] = S.A[0][wm * 16 + mi * 8 + g][ks + t]; ai[mi] = CPLX ? S.A[CPLX ? 1 : 0][wm * 16 + mi * 8 + g][ks + t] : 0.0; }
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) { br[ni] = S.B[0][wn * 32 + ni * 8 + g][ks + t]; bi[ni] = CPLX ? S.B[CPLX ? 1 : 0][wn * 32 + ni * 8 + g][ks + t] : 0.0; }
#pragma unroll
      for (int mi = 0; mi < 2; ++mi)
#pragma unroll
        for (int ni = 0; ni < 4; ++ni) {
          dmma884(acc[mi][ni][0], acc[mi][ni][1], ar[mi], br[ni]);
          if constexpr (CPLX) {
            dmma884(acc[mi][ni][0], acc[mi][ni][1], -ai[mi], bi[ni]);
            dmma884(acc[mi][ni][2], acc[mi][ni][3], ar[mi], bi[ni]);
            dmma884(acc[mi][ni][2], acc[mi][ni][3], ai[mi], br[ni]);
          }
        }
    }
  }
  int wexp = INT_MIN;
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int x = 0; x < 2; ++x) {
        const int rl = wm * 16 + mi * 8 + g, row = m0 + rl, col = n0 + wn * 32 + ni * 8 + 2 * t + x;
        if (row < M && col < N) {
          const double mr = S.rowm[rl];
          const double vr = acc[mi][ni][x] * mr, vi = CPLX ? acc[mi][ni][2 + x] * mr : 0.0;
          double* p = Cm + ((long long)col * ldc + row) * ES;
          p[0] = vr; if (CPLX) p[1] = vi;
          const double mx = fmax(fabs(vr), fabs(vi));
          if (mx > 0.0) wexp = max(wexp, S.rowk[rl] + ilogb(mx));
        }
      }
  wexp = __reduce_max_sync(0xffffffffu, wexp);
  if (lane == 0 && wexp != INT_MIN) atomicMax(kmax_out, wexp);
}

// Brings a freshly multiplied entry to its common exponent k (rows of a propagated product additionally by their own row
// exponent) and returns the sum of squares of the result (thread 0 .. all threads: block-reduced).
template <bool CPLX>
__device__ double lz_fix_entry(double* Mx, int ld, int rows, int cols, int k, LzRowScale rs, double* red) {
  constexpr int ES = CPLX ? 2 : 1;
  double ss = 0.0;
  for (int idx = threadIdx.x; idx < rows * cols; idx += blockDim.x) {
    const int r = idx % rows, c = idx / rows;
    const int sh = (rs.on ? row_exp(prop_x(rs.delta, rs.E[r], rs.emin)) : 0) - k;
    double* p = Mx + ((long long)c * ld + r) * ES;
    const double vr = lz_scale(p[0], sh); p[0] = vr; ss += vr * vr;
    if (CPLX) { const double vi = lz_scale(p[1], sh); p[1] = vi; ss += vi * vi; }
  }
  return lz_block_sum(ss, red);
}

// The same, one 64 x 64 tile per CTA (the rescale of a 295 x 295 product by one CTA was a third of a config-4 round).
template <bool CPLX>
__device__ double lz_fix_tile(double* Mx, int ld, int rows, int cols, int m0, int n0, int k, LzRowScale rs, double* red) {
  constexpr int ES = CPLX ? 2 : 1;
  double ss = 0.0;
  // blockDim.x is a multiple of the tile height: a thread stays on one row, whose shift is computed once
  const int r_fixed = m0 + (threadIdx.x & (kLzTile - 1));
  const int sh_fixed = ((rs.on && r_fixed < rows) ? row_exp(prop_x(rs.delta, rs.E[r_fixed], rs.emin)) : 0) - k;
  // eight loads in flight per thread (a load-scale-store loop waits for every load: the stores may alias the next load)
  constexpr int kBatch = 8;
  const int r = r_fixed;
  for (int c0 = n0 + (int)(threadIdx.x / kLzTile); c0 < n0 + kLzTile; c0 += kBatch * (int)(blockDim.x / kLzTile)) {
    double vr[kBatch], vi[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int c = c0 + u * (int)(blockDim.x / kLzTile);
      vr[u] = 0.0; vi[u] = 0.0;
      if (r < rows && c < cols && c < n0 + kLzTile) {
        const double* p = Mx + ((long long)c * ld + r) * ES;
        if (CPLX) { const double2 z = *reinterpret_cast<const double2*>(p); vr[u] = z.x; vi[u] = z.y; } else vr[u] = p[0];
      }
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const int c = c0 + u * (int)(blockDim.x / kLzTile);
      if (r < rows && c < cols && c < n0 + kLzTile) {
        double* p = Mx + ((long long)c * ld + r) * ES;
        const double xr = lz_scale(vr[u], sh_fixed);
        ss += xr * xr;
        if (CPLX) {
          const double xi = lz_scale(vi[u], sh_fixed);
          ss += xi * xi;
          *reinterpret_cast<double2*>(p) = make_double2(xr, xi);
        } else p[0] = xr;
      }
    }
  }
  return lz_block_sum(ss, red);
}
// Thread 0 of a CTA reports its tile (position `it` of the tile list, `ordinal` within its task).  The CTA that completes the
// task gets the task's sum of squares, the partial sums added in tile order (so the norm does not depend on the schedule);
// every other caller gets -1.
__device__ __forceinline__ double lz_fix_arrive(double* part, int* arrived, int it, int ordinal, int ntiles, double ss) {
  part[it] = ss;
  __threadfence();
  if (atomicAdd(arrived, 1) != ntiles - 1) return -1.0;
  __threadfence();
  double t = 0.0;
  for (int i = 0; i < ntiles; ++i) t += ((volatile double*)part)[it - ordinal + i];
  return t;
}

// ------------------------------------------------------------------------------------------------ creation
__global__ void lazy_reset_kernel(LazyView V) {
  const long long n = (long long)V.nC * V.NN * V.imp.Q;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const int q = (int)(i % V.imp.Q);
    V.ent_tgt[i] = q; V.ent_valid[i] = 0; V.ent_k[i] = INT_MIN; V.ent_e[i] = 0; V.ent_lg[i] = 0.0; V.ent_nrm[i] = 0.0;
  }
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < (long long)V.nC * V.nnode; i += (long long)gridDim.x * blockDim.x)
    V.slot_of[i] = (int)(i % V.nnode);
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < (long long)V.nC * (V.smax + V.emax); i += (long long)gridDim.x * blockDim.x)
    V.free_slot[i] = V.nnode + (int)(i % (V.smax + V.emax));
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < (long long)V.nC * V.nleaf; i += (long long)gridDim.x * blockDim.x)
    V.leaf_n[i] = 0;
  if (blockIdx.x == 0 && threadIdx.x < 16) V.w_cnt[threadIdx.x] = 0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < (long long)V.nC * V.D; i += (long long)gridDim.x * blockDim.x) {
    V.p_lvl_start[i] = 0; V.p_lvl_cnt[i] = 0;
  }
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < (long long)V.nC; i += (long long)gridDim.x * blockDim.x) {
    V.p_status[i] = 0; V.p_ndirty[i] = 0; V.p_nleaf[i] = 0; V.decided[i] = 2; V.decided_by[i] = 0; V.n_eval[i] = 0; V.n_alive[i] = 0;
  }
}

// Diagonal propagator of an operator-free interval written as a dense entry: U(q) = P_delta(q).
template <bool CPLX>
__device__ void lz_write_diag_entry(const LazyView& V, int c, int slot, int q, double delta, double* red, int* redi) {
  constexpr int ES = CPLX ? 2 : 1;
  const int d = V.imp.dim[q];
  const double* E = V.imp.energy + V.imp.e_off[q];
  const double emin = V.imp.e_min[q];
  int km = INT_MIN;
  for (int r = threadIdx.x; r < d; r += blockDim.x) km = max(km, row_exp(prop_x(delta, E[r], emin)));
  km = lz_block_max(km, redi);
  double* Mx = lz_mat(V, c, slot, q);
  LzDiag dg; dg.delta = delta; dg.E = E; dg.emin = emin; dg.kmax = km;
  double ss = 0.0;
  for (int idx = threadIdx.x; idx < d * d; idx += blockDim.x) {
    const int r = idx % d, cc = idx / d;
    const double v = (r == cc) ? lz_diag_value(dg, r) : 0.0;
    double* p = Mx + ((long long)cc * V.ldm + r) * ES;
    p[0] = v; if (CPLX) p[1] = 0.0;
    ss += v * v;
  }
  ss = lz_block_sum(ss, red);
  if (threadIdx.x == 0) {
    const size_t en = lz_ent(V, c, slot, q);
    V.ent_e[en] = km; V.ent_lg[en] = -delta * emin * kLog2e; V.ent_nrm[en] = sqrt(ss); V.ent_tgt[en] = q; V.ent_valid[en] = 1;
  }
}

// chain 0, empty configuration: every leaf is the propagator across its interval
template <bool CPLX>
__global__ void lazy_build_leaves_kernel(LazyView V) {
  __shared__ double red[32]; __shared__ int redi[32];
  const int leaf = blockIdx.x, q = blockIdx.y;
  lz_write_diag_entry<CPLX>(V, 0, V.nleaf - 1 + leaf, q, lz_edge(V, leaf + 1) - lz_edge(V, leaf), red, redi);
}

// chain 0 -> every other chain (stored nodes only)
__global__ void lazy_replicate_kernel(LazyView V) {
  const long long per_mat = (long long)V.nnode * V.node_elems, per_ent = (long long)V.nnode * V.imp.Q;
  const long long stride = (long long)gridDim.x * blockDim.x, t0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  for (int c = 1; c < V.nC; ++c) {
    double* dm = V.mats + (size_t)c * V.NN * V.node_elems;
    for (long long i = t0; i < per_mat; i += stride) dm[i] = V.mats[i];
    const size_t eo = (size_t)c * V.NN * V.imp.Q;
    for (long long i = t0; i < per_ent; i += stride) {
      V.ent_tgt[eo + i] = V.ent_tgt[i]; V.ent_valid[eo + i] = V.ent_valid[i]; V.ent_e[eo + i] = V.ent_e[i];
      V.ent_lg[eo + i] = V.ent_lg[i]; V.ent_nrm[eo + i] = V.ent_nrm[i];
    }
  }
}

// ------------------------------------------------------------------------------------------------ proposal: integer part
// One warp per chain.  Lane 0 validates the edits and builds the shadow leaves' operator lists and the dirty-node list (leaves
// first, then their ancestors level by level); then the lanes share the sectors for the sector maps of every shadow entry.
__global__ void lazy_prepare_kernel(LazyView V, LazyEdits E, const double* log2_thr) {
  const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (c >= V.nC) return;
  const int Q = V.imp.Q, A = V.imp.A, cap = V.cap;
  int status = 0, n = 0;
  long long lo = 0;
  int* pn = V.p_node + (size_t)c * V.smax;
  int nl = 0, total = 0;
  if (lane == 0) {
    if (E.offset) {
      lo = E.offset[c];
      const long long hi = E.offset[c + 1];
      if (lo < 0 || hi < lo || hi > E.n_edits || hi - lo > V.emax) status = 2; else n = (int)(hi - lo);
    }
    for (int e = 0; e < n && status == 0; ++e) {
      const double t = E.tau[lo + e];
      const int a = E.sym[lo + e], k = E.kind[lo + e];
      if (!(t >= 0.0 && t < V.beta) || a < 0 || a >= A || (k != 1 && k != -1)) { status = 2; break; }
      const int leaf = lz_leaf_of(V, t);
      int pos = 0;
      while (pos < nl && pn[pos] < leaf) ++pos;
      if (pos < nl && pn[pos] == leaf) continue;
      for (int i = nl; i > pos; --i) pn[i] = pn[i - 1];
      pn[pos] = leaf; ++nl;
    }
    // shadow operator lists: removals first (first match in time order), then insertions after every operator with tau <= t
    for (int k = 0; k < nl && status == 0; ++k) {
      const int leaf = pn[k];
      double* st = V.sh_tau + ((size_t)c * V.emax + k) * cap;
      int* ss = V.sh_sym + ((size_t)c * V.emax + k) * cap;
      int cnt = V.leaf_n[(size_t)c * V.nleaf + leaf];
      for (int i = 0; i < cnt; ++i) { st[i] = V.leaf_tau[((size_t)c * V.nleaf + leaf) * cap + i]; ss[i] = V.leaf_sym[((size_t)c * V.nleaf + leaf) * cap + i]; }
      for (int e = 0; e < n && status == 0; ++e) {
        if (E.kind[lo + e] != -1 || lz_leaf_of(V, E.tau[lo + e]) != leaf) continue;
        int i = 0;
        while (i < cnt && !(st[i] == E.tau[lo + e] && ss[i] == E.sym[lo + e])) ++i;
        if (i == cnt) { status = 3; break; }
        for (; i + 1 < cnt; ++i) { st[i] = st[i + 1]; ss[i] = ss[i + 1]; }
        --cnt;
      }
      for (int e = 0; e < n && status == 0; ++e) {
        if (E.kind[lo + e] != 1 || lz_leaf_of(V, E.tau[lo + e]) != leaf) continue;
        if (cnt == cap) { status = 4; break; }
        int pos = 0;
        while (pos < cnt && st[pos] <= E.tau[lo + e]) ++pos;
        for (int i = cnt; i > pos; --i) { st[i] = st[i - 1]; ss[i] = ss[i - 1]; }
        st[pos] = E.tau[lo + e]; ss[pos] = E.sym[lo + e]; ++cnt;
      }
      V.sh_n[(size_t)c * V.emax + k] = cnt;
    }
    if (status != 0) nl = 0;
    if (c == 0) for (int i = 0; i < 6; ++i) { V.w_cnt[i] = 0; if (i < 3) V.w_cnt[10 + i] = 0; }      // leaf work lists of this proposal start empty
    total = nl;
    for (int i = 0; i < nl; ++i) pn[i] += V.nleaf - 1;
    {
      int start = 0, cnt = nl;
      for (int level = V.D - 1; level >= 0; --level) {
        int prev = -1, nc = 0;
        for (int i = start; i < start + cnt; ++i) { const int p = (pn[i] - 1) >> 1; if (p != prev) { pn[total + nc++] = p; prev = p; } }
        V.p_lvl_start[(size_t)c * V.D + level] = total; V.p_lvl_cnt[(size_t)c * V.D + level] = nc;
        start = total; total += nc; cnt = nc;
      }
    }
    V.p_status[c] = status; V.p_nleaf[c] = nl; V.p_ndirty[c] = total;
    V.decided[c] = status ? 2 : 0; V.decided_by[c] = 0; V.n_eval[c] = 0; V.n_alive[c] = 0;
    V.thr[c] = log2_thr ? log2_thr[c] : -INFINITY;
  }
  __syncwarp();
  nl = __shfl_sync(0xffffffffu, nl, 0); total = __shfl_sync(0xffffffffu, total, 0);
  // sector maps of the shadow entries (children come earlier in the list: a warp barrier after every entry)
  const int* fs = V.free_slot + (size_t)c * (V.smax + V.emax);
  for (int i = 0; i < total; ++i) {
    const int slot = fs[i], node = pn[i];
    int sl = 0, sr = 0;
    if (i >= nl) {
      const int left = 2 * node + 1, right = left + 1;
      sl = V.slot_of[(size_t)c * V.nnode + left]; sr = V.slot_of[(size_t)c * V.nnode + right];
      for (int j = 0; j < i; ++j) { if (pn[j] == left) sl = fs[j]; if (pn[j] == right) sr = fs[j]; }
    }
    for (int q = lane; q < Q; q += 32) {
      int tq = q;
      if (i < nl) {
        const int cnt = V.sh_n[(size_t)c * V.emax + i];
        const int* ss = V.sh_sym + ((size_t)c * V.emax + i) * cap;
        for (int j = 0; j < cnt && tq >= 0; ++j) { const int b = V.imp.blk_of[ss[j] * Q + tq]; tq = b < 0 ? -1 : V.imp.blks[b].dst; }
      } else {
        const int m = V.ent_tgt[lz_ent(V, c, sl, q)];
        tq = m < 0 ? -1 : V.ent_tgt[lz_ent(V, c, sr, m)];
      }
      const size_t en = lz_ent(V, c, slot, q);
      V.ent_tgt[en] = tq; V.ent_valid[en] = 0; V.ent_k[en] = INT_MIN; V.ent_e[en] = 0; V.ent_lg[en] = 0.0; V.ent_nrm[en] = 0.0;
    }
    __syncwarp();
  }
}

// ------------------------------------------------------------------------------------------------ proposal: shadow leaves
struct LzLeafTask {
  int ok, c, k, q0, slot, n, leaf;
  double a, b;
};
__device__ __forceinline__ LzLeafTask lz_leaf_task(const LazyView& V, int y, int q0) {
  LzLeafTask T; T.ok = 0;
  T.c = y / V.emax; T.k = y % V.emax; T.q0 = q0;
  if (T.k >= V.p_nleaf[T.c]) return T;
  T.slot = V.free_slot[(size_t)T.c * (V.smax + V.emax) + T.k];
  if (V.ent_tgt[lz_ent(V, T.c, T.slot, q0)] < 0) return T;
  T.leaf = V.p_node[(size_t)T.c * V.smax + T.k] - (V.nleaf - 1);
  T.a = lz_edge(V, T.leaf); T.b = lz_edge(V, T.leaf + 1);
  T.n = V.sh_n[(size_t)T.c * V.emax + T.k];
  T.ok = 1;
  return T;
}

// first propagation P_{t1 - a}(q0): exponent bookkeeping, and the whole entry when the shadow leaf holds no operator;
// a leaf with operators becomes a task of step 0 (grid: (chain, leaf) x start sector -- the one launch with a CTA per candidate)
template <bool CPLX>
__global__ void lazy_leaf_init_kernel(LazyView V) {
  __shared__ double red[32]; __shared__ int redi[32];
  const LzLeafTask T = lz_leaf_task(V, blockIdx.x, blockIdx.y);
  if (!T.ok) return;
  if (T.n == 0) { lz_write_diag_entry<CPLX>(V, T.c, T.slot, T.q0, T.b - T.a, red, redi); return; }
  const double delta = V.sh_tau[((size_t)T.c * V.emax + T.k) * V.cap] - T.a;
  const int d = V.imp.dim[T.q0];
  const double* E = V.imp.energy + V.imp.e_off[T.q0];
  const double emin = V.imp.e_min[T.q0];
  int km = INT_MIN;
  for (int r = threadIdx.x; r < d; r += blockDim.x) km = max(km, row_exp(prop_x(delta, E[r], emin)));
  km = lz_block_max(km, redi);
  if (threadIdx.x == 0) {
    const size_t en = lz_ent(V, T.c, T.slot, T.q0); V.ent_e[en] = km; V.ent_lg[en] = -delta * emin * kLog2e;
    const int ti = atomicAdd(&V.w_cnt[0], 1);
    V.w_ltask[ti] = make_int4((int)blockIdx.x, T.q0, T.q0, 0); V.w_larr[ti] = 0;
    const int blk = V.imp.blk_of[V.sh_sym[((size_t)T.c * V.emax + T.k) * V.cap] * V.imp.Q + T.q0];
    lz_push_tiles(&V.w_cnt[3], V.w_ltile, ti, V.imp.blks[blk].rows, d);
  }
}

// operator j of the shadow leaf of a task {y = chain * emax + leaf index, start sector, sector the chain has reached}
struct LzLeafStep { int c, k, q0, n, blk, qn; size_t en; double delta; double* in; double* out; };
__device__ __forceinline__ LzLeafStep lz_leaf_step(const LazyView& V, int4 task, int j) {
  LzLeafStep S;
  S.c = task.x / V.emax; S.k = task.x % V.emax; S.q0 = task.y;
  const int* ss = V.sh_sym + (size_t)task.x * V.cap;
  const double* st = V.sh_tau + (size_t)task.x * V.cap;
  S.n = V.sh_n[task.x];
  S.blk = V.imp.blk_of[ss[j] * V.imp.Q + task.z]; S.qn = V.imp.blks[S.blk].dst;
  const int leaf = V.p_node[(size_t)S.c * V.smax + S.k] - (V.nleaf - 1);
  S.delta = ((j + 1 < S.n) ? st[j + 1] : lz_edge(V, leaf + 1)) - st[j];
  const int* fs = V.free_slot + (size_t)S.c * (V.smax + V.emax);
  const int slot = fs[S.k];
  S.en = lz_ent(V, S.c, slot, S.q0);
  double* ent = lz_mat(V, S.c, slot, S.q0);
  double* tmp = lz_mat(V, S.c, fs[V.smax + S.k], S.q0);
  S.out = ((S.n - 1 - j) & 1) ? tmp : ent;     // the last step lands in the entry
  S.in = ((S.n - 1 - j) & 1) ? ent : tmp;
  return S;
}

// operator j of every shadow leaf that has one: M <- P_{Delta_j}(q_{j+1}) F_j M   (persistent CTAs over the tile list of step j)
template <bool CPLX>
__global__ void __launch_bounds__(kLzThreads) lazy_leaf_step_kernel(LazyView V, int j) {
  __shared__ LzSmem<CPLX> S;
  const int cur = j % 3, nxt2 = (j + 2) % 3;
  __shared__ int s_it;
  if (blockIdx.x == 0 && threadIdx.x == 0) { V.w_cnt[nxt2] = 0; V.w_cnt[3 + nxt2] = 0; V.w_cnt[10 + nxt2] = 0; }
  const int n_items = V.w_cnt[3 + cur];
  const int4* tiles = V.w_ltile + (size_t)cur * V.w_tile_cap;
  const int4* tasks = V.w_ltask + (size_t)cur * V.w_task_cap;
  for (;;) {                                                   // tiles differ in contraction length: handed out one by one
    if (threadIdx.x == 0) s_it = atomicAdd(&V.w_cnt[10 + cur], 1);
    __syncthreads();
    const int it = s_it;
    if (it >= n_items) break;
    const int4 tl = tiles[it];
    const LzLeafStep st = lz_leaf_step(V, tasks[tl.x], j);
    const BlkDesc bd = V.imp.blks[st.blk];
    LzDiag dg; dg.delta = 0.0; dg.E = nullptr; dg.emin = 0.0; dg.kmax = 0;
    if (j == 0) {
      const int leaf = V.p_node[(size_t)st.c * V.smax + st.k] - (V.nleaf - 1);
      dg.delta = V.sh_tau[((size_t)st.c * V.emax + st.k) * V.cap] - lz_edge(V, leaf);
      dg.E = V.imp.energy + V.imp.e_off[st.q0]; dg.emin = V.imp.e_min[st.q0]; dg.kmax = (int)V.ent_e[st.en];
    }
    LzRowScale rs; rs.on = 1; rs.delta = st.delta; rs.E = V.imp.energy + V.imp.e_off[st.qn]; rs.emin = V.imp.e_min[st.qn];
    lz_gemm_tile<CPLX>(S, tl.y, tl.z, bd.rows, V.imp.dim[st.q0], bd.cols, V.imp.store + bd.off, bd.ld, 1, j == 0 ? nullptr : st.in, V.ldm, dg,
                       st.out, V.ldm, rs, &V.ent_k[st.en]);
    __syncthreads();
  }
}

// common exponent and norm of the product of step j, tile by tile (persistent CTAs over the tile list); the CTA that finishes a
// task's last tile closes the step and moves the task on to step j + 1
template <bool CPLX>
__global__ void lazy_leaf_fix_kernel(LazyView V, int j) {
  __shared__ double red[32];
  const int cur = j % 3, nxt = (j + 1) % 3;
  const int n_items = V.w_cnt[3 + cur];
  const int4* tiles = V.w_ltile + (size_t)cur * V.w_tile_cap;
  const int4* tasks = V.w_ltask + (size_t)cur * V.w_task_cap;
  for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
    const int4 tl = tiles[it];
    const int4 task = tasks[tl.x];
    const LzLeafStep st = lz_leaf_step(V, task, j);
    int k = V.ent_k[st.en];
    if (k == INT_MIN) k = 0;
    LzRowScale rs; rs.on = 1; rs.delta = st.delta; rs.E = V.imp.energy + V.imp.e_off[st.qn]; rs.emin = V.imp.e_min[st.qn];
    const int rows = V.imp.dim[st.qn], cols = V.imp.dim[st.q0];
    const double part = lz_fix_tile<CPLX>(st.out, V.ldm, rows, cols, tl.y, tl.z, k, rs, red);
    if (threadIdx.x == 0) {
      const int nt = ((rows + kLzTile - 1) / kLzTile) * ((cols + kLzTile - 1) / kLzTile);
      const double ss = lz_fix_arrive(V.w_part, &V.w_larr[(size_t)cur * V.w_task_cap + tl.x], it, tl.w, nt, part);
      if (ss >= 0.0) {
        V.ent_e[st.en] += k; V.ent_lg[st.en] += -st.delta * rs.emin * kLog2e; V.ent_k[st.en] = INT_MIN;
        if (j == st.n - 1) { V.ent_nrm[st.en] = sqrt(ss); V.ent_valid[st.en] = 1; }
        else {
          const int t2 = atomicAdd(&V.w_cnt[nxt], 1);
          V.w_ltask[(size_t)nxt * V.w_task_cap + t2] = make_int4(task.x, task.y, st.qn, 0);
          V.w_larr[(size_t)nxt * V.w_task_cap + t2] = 0;
          const int blk = V.imp.blk_of[V.sh_sym[(size_t)task.x * V.cap + j + 1] * V.imp.Q + st.qn];
          lz_push_tiles(&V.w_cnt[3 + nxt], V.w_ltile + (size_t)nxt * V.w_tile_cap, t2, V.imp.blks[blk].rows, cols);
        }
        atomicAdd(V.n_products, 1ull);
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------ proposal: bounds
// One warp per chain.  Cover of the time axis = dirty leaves + maximal clean subtrees, left to right (reading F3):
// B(q0) = sqrt(r) prod ||U_node||_F rounded outward; the sum decides "reject by bound"; the start sectors are ordered by
// decreasing bound for the lazy evaluation (reading F4).
__global__ void lazy_bound_kernel(LazyView V, double* bound_mant, long long* bound_exp2) {
  const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (c >= V.nC) return;
  const int Q = V.imp.Q;
  if (V.p_status[c] != 0) {
    if (lane == 0) { bound_mant[c] = __longlong_as_double(0x7ff8000000000000LL); bound_exp2[c] = 0; }
    return;
  }
  for (int q0 = lane; q0 < Q; q0 += 32) {
    int q = q0, dmin = V.imp.dim[q0];
    double val = 1.0, lg = 0.0; long long e = 0; bool alive = true;
    int stack[40]; int sp = 0; stack[sp++] = 0;
    while (sp > 0 && alive) {
      const int node = stack[--sp];
      const int di = lz_dirty_index(V, c, node);
      if (di >= 0 && lz_level(node) < V.D) { stack[sp++] = 2 * node + 2; stack[sp++] = 2 * node + 1; continue; }
      const int slot = di >= 0 ? V.free_slot[(size_t)c * (V.smax + V.emax) + di] : V.slot_of[(size_t)c * V.nnode + node];
      const size_t en = lz_ent(V, c, slot, q);
      const int tq = V.ent_tgt[en];
      if (tq < 0) { alive = false; break; }
      val *= V.ent_nrm[en]; e += V.ent_e[en]; lg += V.ent_lg[en]; q = tq;
      dmin = min(dmin, V.imp.dim[q]);
      if (val != 0.0) { const int k = ilogb(val); val = scalbn(val, -k); e += k; }
    }
    Scaled b; b.m = 0.0; b.e = 0;
    if (alive) b = finish_sector_bound(sqrt((double)dmin) * val, e, lg);
    V.sb_m[(size_t)c * Q + q0] = alive ? b.m : -1.0;      // -1: the string dies (no bound, not in the order)
    V.sb_e[(size_t)c * Q + q0] = b.e;
  }
  __syncwarp();
  if (lane != 0) return;
  const double* sm = V.sb_m + (size_t)c * Q; const long long* se = V.sb_e + (size_t)c * Q;
  const LzC tot = lz_sum(Q, [&](int i) { LzC z; z.re = sm[i] > 0.0 ? sm[i] : 0.0; z.im = 0.0; z.e = se[i]; return z; });
  bound_mant[c] = tot.re; bound_exp2[c] = tot.e;
  int* ord = V.order + (size_t)c * Q;
  int na = 0;
  for (int q0 = 0; q0 < Q; ++q0) {     // stable insertion sort by decreasing log2 of the bound
    if (sm[q0] < 0.0) continue;
    const double key = lz_log2(sm[q0], se[q0]);
    int pos = na;
    while (pos > 0 && lz_log2(sm[ord[pos - 1]], se[ord[pos - 1]]) < key) { ord[pos] = ord[pos - 1]; --pos; }
    ord[pos] = q0; ++na;
  }
  V.n_alive[c] = na;
  if (lz_log2(tot.re, tot.e) <= V.thr[c]) { V.decided[c] = 2; V.decided_by[c] = 0; }
}

// ------------------------------------------------------------------------------------------------ dirty ancestors
// mode 0: lazy round r -- only the entry that start sector order[r] needs at this node;  mode 1: every missing entry of the
// node (completion of an accepted / undecided proposal, or -- gate = mask -- of a commit).
// Plan of one (level, mode, r) step: one thread per candidate (chain, dirty ancestor of the level, sector) decides whether the
// entry has to be multiplied now and appends it (two int4: {chain, slot, start sector, left slot}, {right slot, middle sector,
// target sector, 0}) and its tiles to the node lists of parity `par`.
__device__ __forceinline__ bool lz_node_candidate(const LazyView& V, int level, int mode, int r, const int* gate, int gate_commit,
                                                  long long idx, int4& t0, int4& t1) {
  const int nsec = mode == 0 ? 1 : V.imp.Q;
  if (idx >= (long long)V.nC * V.emax * nsec) return false;
  const int z = (int)(idx % nsec), i = (int)((idx / nsec) % V.emax), c = (int)(idx / ((long long)nsec * V.emax));
  if (V.p_status[c] != 0 || i >= V.p_lvl_cnt[(size_t)c * V.D + level]) return false;
  const int di = V.p_lvl_start[(size_t)c * V.D + level] + i;
  if (di >= V.p_ndirty[c]) return false;                       // nothing proposed since the last commit
  if (gate_commit ? (gate[c] == 0) : (V.decided[c] == 2)) return false;
  const int node = V.p_node[(size_t)c * V.smax + di];
  int qin = z;
  if (mode == 0) {
    if (r >= V.n_alive[c]) return false;
    qin = V.order[(size_t)c * V.imp.Q + r];
    int cur = 0;
    for (int l = 0; l < level; ++l) {                          // walk from the root down to `node`
      const int anc = (((node + 1) >> (level - l - 1)) - 1);   // ancestor of `node` at level l + 1
      const int left = 2 * cur + 1;
      if (anc != left) { qin = V.ent_tgt[lz_ent(V, c, lz_slot(V, c, left), qin)]; if (qin < 0) return false; }
      cur = anc;
    }
  }
  const int slot = V.free_slot[(size_t)c * (V.smax + V.emax) + di];
  const size_t en = lz_ent(V, c, slot, qin);
  if (V.ent_tgt[en] < 0 || V.ent_valid[en]) return false;
  const int sl = lz_slot(V, c, 2 * node + 1), sr = lz_slot(V, c, 2 * node + 2);
  const int mid = V.ent_tgt[lz_ent(V, c, sl, qin)];
  if (mid < 0) return false;
  if (!V.ent_valid[lz_ent(V, c, sl, qin)] || !V.ent_valid[lz_ent(V, c, sr, mid)]) return false;
  t0 = make_int4(c, slot, qin, sl); t1 = make_int4(sr, mid, V.ent_tgt[lz_ent(V, c, sr, mid)], 0);
  return true;
}
__global__ void lazy_node_plan_kernel(LazyView V, int level, int mode, int r, const int* gate, int gate_commit, int par) {
  int4 t0, t1;
  if (!lz_node_candidate(V, level, mode, r, gate, gate_commit, blockIdx.x * (long long)blockDim.x + threadIdx.x, t0, t1)) return;
  const int ti = atomicAdd(&V.w_cnt[6 + par], 1);
  int4* nt = V.w_ntask + ((size_t)par * V.w_task_cap + ti) * 2;
  nt[0] = t0; nt[1] = t1; V.w_narr[(size_t)par * V.w_task_cap + ti] = 0;
  lz_push_tiles(&V.w_cnt[8 + par], V.w_ntile + (size_t)par * V.w_tile_cap, ti, V.imp.dim[t1.z], V.imp.dim[t0.z]);
}

template <bool CPLX>
__global__ void __launch_bounds__(kLzThreads) lazy_node_gemm_kernel(LazyView V, int par) {
  __shared__ LzSmem<CPLX> S;
  __shared__ int s_it;
  if (blockIdx.x == 0 && threadIdx.x == 0) { V.w_cnt[6 + (par ^ 1)] = 0; V.w_cnt[8 + (par ^ 1)] = 0; V.w_cnt[13 + (par ^ 1)] = 0; }
  const int n_items = V.w_cnt[8 + par];
  const int4* tiles = V.w_ntile + (size_t)par * V.w_tile_cap;
  const int4* tasks = V.w_ntask + (size_t)par * V.w_task_cap * 2;
  LzDiag dg; dg.delta = 0.0; dg.E = nullptr; dg.emin = 0.0; dg.kmax = 0;
  LzRowScale rs; rs.on = 0; rs.delta = 0.0; rs.E = nullptr; rs.emin = 0.0;
  for (;;) {
    if (threadIdx.x == 0) s_it = atomicAdd(&V.w_cnt[13 + par], 1);
    __syncthreads();
    const int it = s_it;
    if (it >= n_items) break;
    const int4 tl = tiles[it];
    const int4 t0 = tasks[2 * tl.x], t1 = tasks[2 * tl.x + 1];      // {c, slot, qin, sl}, {sr, mid, tq}
    lz_gemm_tile<CPLX>(S, tl.y, tl.z, V.imp.dim[t1.z], V.imp.dim[t0.z], V.imp.dim[t1.y], lz_mat(V, t0.x, t1.x, t1.y), 1, V.ldm,
                       lz_mat(V, t0.x, t0.w, t0.z), V.ldm, dg, lz_mat(V, t0.x, t0.y, t0.z), V.ldm, rs, &V.ent_k[lz_ent(V, t0.x, t0.y, t0.z)]);
    __syncthreads();
  }
}

template <bool CPLX>
__global__ void lazy_node_fix_kernel(LazyView V, int par) {
  __shared__ double red[32];
  const int n_items = V.w_cnt[8 + par];
  const int4* tiles = V.w_ntile + (size_t)par * V.w_tile_cap;
  const int4* tasks = V.w_ntask + (size_t)par * V.w_task_cap * 2;
  LzRowScale rs; rs.on = 0; rs.delta = 0.0; rs.E = nullptr; rs.emin = 0.0;
  for (int it = blockIdx.x; it < n_items; it += gridDim.x) {
    const int4 tl = tiles[it];
    const int4 t0 = tasks[2 * tl.x], t1 = tasks[2 * tl.x + 1];
    const size_t en = lz_ent(V, t0.x, t0.y, t0.z), el = lz_ent(V, t0.x, t0.w, t0.z), er = lz_ent(V, t0.x, t1.x, t1.y);
    int k = V.ent_k[en];
    if (k == INT_MIN) k = 0;
    const int rows = V.imp.dim[t1.z], cols = V.imp.dim[t0.z];
    const double part = lz_fix_tile<CPLX>(lz_mat(V, t0.x, t0.y, t0.z), V.ldm, rows, cols, tl.y, tl.z, k, rs, red);
    if (threadIdx.x == 0) {
      const int nt = ((rows + kLzTile - 1) / kLzTile) * ((cols + kLzTile - 1) / kLzTile);
      const double ss = lz_fix_arrive(V.w_part, &V.w_narr[(size_t)par * V.w_task_cap + tl.x], it, tl.w, nt, part);
      if (ss >= 0.0) {
        V.ent_e[en] = V.ent_e[el] + V.ent_e[er] + k; V.ent_lg[en] = V.ent_lg[el] + V.ent_lg[er];
        V.ent_nrm[en] = sqrt(ss); V.ent_k[en] = INT_MIN;
        __threadfence();
        V.ent_valid[en] = 1;
        atomicAdd(V.n_products, 1ull);
      }
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------ small impurities
// Sector dimensions <= 16 (configs 1 and 2): a 64 x 64 tensor-core tile would be all padding and a launch per operator all
// latency.  One WARP owns a task and keeps both operands in shared memory (A k-major, B column-major, leading dimension 16);
// lane l holds result elements l, l + 32, ... (row = e % M, column = e / M).  A shadow leaf is rebuilt in ONE launch (the warp
// walks its operators), a dirty level in one launch (candidate test, product, common exponent and norm fused).  The arithmetic
// is that of lz_gemm_tile + lz_fix_entry element by element; only the order of the contraction sum differs.
constexpr int kLzSmall = 16;
constexpr int kLzSmallWarps = 4;
__host__ __device__ constexpr int lz_node_small_warps(bool cplx) { return cplx ? 4 : 8; }   // 32 KB of operands per CTA either way
template <bool CPLX>
struct LzSmallSmem { double A[CPLX ? 2 : 1][kLzSmall * kLzSmall]; double B[CPLX ? 2 : 1][kLzSmall * kLzSmall]; };

template <bool CPLX>
__device__ __forceinline__ void lz_small_product(const LzSmallSmem<CPLX>& S, int M, int N, int K, int lane, double (&cr)[8], double (&ci)[8]) {
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    cr[u] = 0.0; ci[u] = 0.0;
    const int e = lane + 32 * u;
    if (e < M * N) {
      const int r = e % M, col = e / M;
      for (int k = 0; k < K; ++k) {
        const double ar = S.A[0][k * kLzSmall + r], br = S.B[0][col * kLzSmall + k];
        cr[u] = fma(ar, br, cr[u]);
        if (CPLX) {
          const double ai = S.A[CPLX ? 1 : 0][k * kLzSmall + r], bi = S.B[CPLX ? 1 : 0][col * kLzSmall + k];
          cr[u] = fma(-ai, bi, cr[u]);
          ci[u] = fma(ar, bi, ci[u]); ci[u] = fma(ai, br, ci[u]);
        }
      }
    }
  }
}

// every shadow leaf of every chain, start to end: grid = ceil(chains * emax * Q / 4) CTAs of 4 warps
template <bool CPLX>
__global__ void __launch_bounds__(32 * kLzSmallWarps) lazy_leaf_small_kernel(LazyView V) {
  constexpr int ES = CPLX ? 2 : 1;
  __shared__ LzSmallSmem<CPLX> Sm[kLzSmallWarps];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const long long id = blockIdx.x * (long long)kLzSmallWarps + warp;
  const int Q = V.imp.Q;
  if (id >= (long long)V.nC * V.emax * Q) return;
  const int y = (int)(id / Q), q0 = (int)(id % Q);
  const LzLeafTask T = lz_leaf_task(V, y, q0);
  if (!T.ok) return;
  LzSmallSmem<CPLX>& S = Sm[warp];
  const int d0 = V.imp.dim[q0];
  const double* st = V.sh_tau + (size_t)y * V.cap;
  const int* ss = V.sh_sym + (size_t)y * V.cap;
  // first propagation P_{t1 - a}(q0) as the right operand
  const double delta0 = (T.n ? st[0] : T.b) - T.a;
  LzDiag dg; dg.delta = delta0; dg.E = V.imp.energy + V.imp.e_off[q0]; dg.emin = V.imp.e_min[q0];
  int km = lane < d0 ? row_exp(prop_x(delta0, dg.E[lane], dg.emin)) : INT_MIN;
  km = __reduce_max_sync(0xffffffffu, km);
  dg.kmax = km;
  for (int e = lane; e < kLzSmall * kLzSmall; e += 32) { S.B[0][e] = 0.0; if (CPLX) S.B[CPLX ? 1 : 0][e] = 0.0; }
  __syncwarp();
  double cr[8], ci[8];
#pragma unroll
  for (int u = 0; u < 8; ++u) { cr[u] = 0.0; ci[u] = 0.0; }
  if (lane < d0) S.B[0][lane * kLzSmall + lane] = lz_diag_value(dg, lane);
  __syncwarp();
  long long e_acc = km;
  double lg = -delta0 * dg.emin * kLog2e;
  int q = q0, M = d0;                                     // rows of the current product
  if (T.n == 0) {
#pragma unroll
    for (int u = 0; u < 8; ++u) { const int e = lane + 32 * u; if (e < d0 * d0) cr[u] = S.B[0][(e / d0) * kLzSmall + e % d0]; }
  }
  for (int j = 0; j < T.n; ++j) {
    const BlkDesc bd = V.imp.blks[V.imp.blk_of[ss[j] * Q + q]];
    const int qn = bd.dst, K = bd.cols;
    M = bd.rows;
    const double delta = ((j + 1 < T.n) ? st[j + 1] : T.b) - st[j];
    const double* F = V.imp.store + bd.off;
    for (int e = lane; e < M * K; e += 32) {
      const int r = e / K, k = e % K;
      const double* p = F + ((long long)r * bd.ld + k) * ES;
      S.A[0][k * kLzSmall + r] = p[0]; if (CPLX) S.A[CPLX ? 1 : 0][k * kLzSmall + r] = p[1];
    }
    __syncwarp();
    lz_small_product<CPLX>(S, M, d0, K, lane, cr, ci);
    const double* En = V.imp.energy + V.imp.e_off[qn];
    const double eminn = V.imp.e_min[qn];
    int kr[8], wexp = INT_MIN;
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int e = lane + 32 * u;
      kr[u] = 0;
      if (e < M * d0) {
        const double x = prop_x(delta, En[e % M], eminn);
        const double mr = exp2(__dsub_rn(x, floor(x)));
        kr[u] = row_exp(x);
        cr[u] *= mr; if (CPLX) ci[u] *= mr;
        const double mx = fmax(fabs(cr[u]), fabs(ci[u]));
        if (mx > 0.0) wexp = max(wexp, kr[u] + ilogb(mx));
      }
    }
    wexp = __reduce_max_sync(0xffffffffu, wexp);
    const int k = wexp == INT_MIN ? 0 : wexp;
    __syncwarp();
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      const int e = lane + 32 * u;
      if (e < M * d0) {
        cr[u] = lz_scale(cr[u], kr[u] - k); if (CPLX) ci[u] = lz_scale(ci[u], kr[u] - k);
        S.B[0][(e / M) * kLzSmall + e % M] = cr[u]; if (CPLX) S.B[CPLX ? 1 : 0][(e / M) * kLzSmall + e % M] = ci[u];
      }
    }
    __syncwarp();
    e_acc += k; lg += -delta * eminn * kLog2e; q = qn;
  }
  double* Mx = lz_mat(V, T.c, T.slot, q0);
  double sq = 0.0;
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const int e = lane + 32 * u;
    if (e < M * d0) {
      double* p = Mx + ((long long)(e / M) * V.ldm + e % M) * ES;
      p[0] = cr[u]; sq += cr[u] * cr[u];
      if (CPLX) { p[1] = ci[u]; sq += ci[u] * ci[u]; }
    }
  }
  sq = warp_sum(sq);
  if (lane == 0) {
    const size_t en = lz_ent(V, T.c, T.slot, q0);
    V.ent_e[en] = e_acc; V.ent_lg[en] = lg; V.ent_nrm[en] = sqrt(sq); V.ent_valid[en] = 1;
    if (T.n) atomicAdd(V.n_products, (unsigned long long)T.n);
  }
}

// the dirty ancestors of one chain, bottom-up (one CTA per chain; a level depends only on the chain's own lower levels, so a
// CTA-wide barrier separates them): candidate test, product of the two children, common exponent, norm (one warp per candidate)
template <bool CPLX>
__device__ __forceinline__ void lz_node_small(const LazyView& V, LzSmallSmem<CPLX>& S, int4 t0, int4 t1, int lane);

template <bool CPLX>
__global__ void __launch_bounds__(32 * lz_node_small_warps(CPLX)) lazy_node_small_kernel(LazyView V, int mode, int r, const int* gate, int gate_commit) {
  constexpr int kLzSmallWarps = lz_node_small_warps(CPLX);
  __shared__ LzSmallSmem<CPLX> Sm[kLzSmallWarps];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, c = blockIdx.x;
  const int nsec = mode == 0 ? 1 : V.imp.Q;
  if (V.p_status[c] != 0 || V.p_ndirty[c] == 0) return;
  if (gate_commit ? (gate[c] == 0) : (V.decided[c] == 2)) return;
  for (int level = V.D - 1; level >= 0; --level) {
    const int n_cand = V.p_lvl_cnt[(size_t)c * V.D + level] * nsec;
    for (int cand = warp; cand < n_cand; cand += kLzSmallWarps) {
      int4 t0, t1;                                           // {c, slot, qin, sl}, {sr, mid, tq}
      if (lz_node_candidate(V, level, mode, r, gate, gate_commit, ((long long)c * V.emax + cand / nsec) * nsec + cand % nsec, t0, t1))
        lz_node_small<CPLX>(V, Sm[warp], t0, t1, lane);
      __syncwarp();
    }
    __syncthreads();
  }
}

template <bool CPLX>
__device__ __forceinline__ void lz_node_small(const LazyView& V, LzSmallSmem<CPLX>& S, int4 t0, int4 t1, int lane) {
  constexpr int ES = CPLX ? 2 : 1;
  const int M = V.imp.dim[t1.z], K = V.imp.dim[t1.y], N = V.imp.dim[t0.z];
  const double* R = lz_mat(V, t0.x, t1.x, t1.y);
  const double* L = lz_mat(V, t0.x, t0.w, t0.z);
  for (int e = lane; e < M * K; e += 32) {
    const double* p = R + ((long long)(e / M) * V.ldm + e % M) * ES;
    S.A[0][(e / M) * kLzSmall + e % M] = p[0]; if (CPLX) S.A[CPLX ? 1 : 0][(e / M) * kLzSmall + e % M] = p[1];
  }
  for (int e = lane; e < K * N; e += 32) {
    const double* p = L + ((long long)(e / K) * V.ldm + e % K) * ES;
    S.B[0][(e / K) * kLzSmall + e % K] = p[0]; if (CPLX) S.B[CPLX ? 1 : 0][(e / K) * kLzSmall + e % K] = p[1];
  }
  __syncwarp();
  double cr[8], ci[8];
  lz_small_product<CPLX>(S, M, N, K, lane, cr, ci);
  int wexp = INT_MIN;
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const double mx = fmax(fabs(cr[u]), fabs(ci[u]));
    if (mx > 0.0) wexp = max(wexp, ilogb(mx));
  }
  wexp = __reduce_max_sync(0xffffffffu, wexp);
  const int k = wexp == INT_MIN ? 0 : wexp;
  double* Mx = lz_mat(V, t0.x, t0.y, t0.z);
  double sq = 0.0;
#pragma unroll
  for (int u = 0; u < 8; ++u) {
    const int e = lane + 32 * u;
    if (e < M * N) {
      const double vr = lz_scale(cr[u], -k), vi = CPLX ? lz_scale(ci[u], -k) : 0.0;
      double* p = Mx + ((long long)(e / M) * V.ldm + e % M) * ES;
      p[0] = vr; sq += vr * vr;
      if (CPLX) { p[1] = vi; sq += vi * vi; }
    }
  }
  sq = warp_sum(sq);
  if (lane == 0) {
    const size_t en = lz_ent(V, t0.x, t0.y, t0.z), el = lz_ent(V, t0.x, t0.w, t0.z), er = lz_ent(V, t0.x, t1.x, t1.y);
    V.ent_e[en] = V.ent_e[el] + V.ent_e[er] + k; V.ent_lg[en] = V.ent_lg[el] + V.ent_lg[er];
    V.ent_nrm[en] = sqrt(sq); V.ent_k[en] = INT_MIN;
    __threadfence();
    V.ent_valid[en] = 1;
    atomicAdd(V.n_products, 1ull);
  }
}

// chain 0 at creation: every node of `level`, every sector (children are stored nodes)
template <bool CPLX>
__global__ void __launch_bounds__(kLzThreads) lazy_build_gemm_kernel(LazyView V, int level, int NT) {
  __shared__ LzSmem<CPLX> S;
  const int node = (1 << level) - 1 + blockIdx.x, q = blockIdx.z;
  const int d = V.imp.dim[q];
  const int m0 = (blockIdx.y / NT) * kLzTile, n0 = (blockIdx.y % NT) * kLzTile;
  if (m0 >= d || n0 >= d) return;
  LzDiag dg; dg.delta = 0.0; dg.E = nullptr; dg.emin = 0.0; dg.kmax = 0;
  LzRowScale rs; rs.on = 0; rs.delta = 0.0; rs.E = nullptr; rs.emin = 0.0;
  lz_gemm_tile<CPLX>(S, m0, n0, d, d, d, lz_mat(V, 0, 2 * node + 2, q), 1, V.ldm, lz_mat(V, 0, 2 * node + 1, q), V.ldm, dg,
                     lz_mat(V, 0, node, q), V.ldm, rs, &V.ent_k[lz_ent(V, 0, node, q)]);
}
template <bool CPLX>
__global__ void lazy_build_fix_kernel(LazyView V, int level) {
  __shared__ double red[32];
  const int node = (1 << level) - 1 + blockIdx.x, q = blockIdx.y;
  const size_t en = lz_ent(V, 0, node, q), el = lz_ent(V, 0, 2 * node + 1, q), er = lz_ent(V, 0, 2 * node + 2, q);
  int k = V.ent_k[en];
  if (k == INT_MIN) k = 0;
  LzRowScale rs; rs.on = 0; rs.delta = 0.0; rs.E = nullptr; rs.emin = 0.0;
  const int d = V.imp.dim[q];
  const double ss = lz_fix_entry<CPLX>(lz_mat(V, 0, node, q), V.ldm, d, d, k, rs, red);
  if (threadIdx.x == 0) {
    V.ent_e[en] = V.ent_e[el] + V.ent_e[er] + k; V.ent_lg[en] = V.ent_lg[el] + V.ent_lg[er];
    V.ent_nrm[en] = sqrt(ss); V.ent_k[en] = INT_MIN; V.ent_tgt[en] = q; V.ent_valid[en] = 1;
  }
}

// ------------------------------------------------------------------------------------------------ decision (reading F4)
// One warp per chain: takes the exact terms of the start sectors order[r_lo .. r_hi) from the (shadow) root, and replays the
// bracketing of the pre-drawn threshold: |S| - R > T accepts, |S| + R <= T rejects, with S the sum of the exact terms so far
// and R the sum of the bounds of the sectors not yet evaluated.  `last`: the outputs are final after this call.
template <bool CPLX>
__global__ void lazy_decide_kernel(LazyView V, int r_lo, int r_hi, int last, int* accept, int* decided_by, int* n_eval, double* trace_mant,
                                   long long* trace_exp2, int* status) {
  constexpr int ES = CPLX ? 2 : 1;
  const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (c >= V.nC) return;
  const int Q = V.imp.Q;
  const int na = V.n_alive[c];
  int dec = V.decided[c], by = V.decided_by[c], ne = V.n_eval[c];
  if (V.p_status[c] == 0 && dec != 2) {
    const int rslot = lz_slot(V, c, 0);
    const int* ord = V.order + (size_t)c * Q;
    double* tre = V.term_re + (size_t)c * Q; double* tim = V.term_im + (size_t)c * Q; long long* te = V.term_e + (size_t)c * Q;
    const double* sm = V.sb_m + (size_t)c * Q; const long long* se = V.sb_e + (size_t)c * Q;
    for (int r = r_lo; r < r_hi && r < na; ++r) {
      const int q0 = ord[r];
      const size_t en = lz_ent(V, c, rslot, q0);
      double zr = 0.0, zi = 0.0;
      if (V.ent_tgt[en] == q0 && V.ent_valid[en]) {
        const double* Mx = lz_mat(V, c, rslot, q0);
        const int d = V.imp.dim[q0];
        for (int i = lane; i < d; i += 32) { zr += Mx[((long long)i * V.ldm + i) * ES]; if (CPLX) zi += Mx[((long long)i * V.ldm + i) * ES + 1]; }
        zr = warp_sum(zr); zi = warp_sum(zi);
      }
      if (lane == 0) {
        const LzC t = lz_apply_lg(zr, zi, V.ent_e[en], V.ent_lg[en]);
        tre[r] = t.re; tim[r] = t.im; te[r] = t.e;
        ne = r + 1;
        if (dec == 0) {
          const LzC S = lz_sum(r + 1, [&](int i) { LzC z; z.re = tre[i]; z.im = tim[i]; z.e = te[i]; return z; });
          const LzC R = lz_sum(na - r - 1, [&](int i) { LzC z; z.re = sm[ord[r + 1 + i]]; z.im = 0.0; z.e = se[ord[r + 1 + i]]; return z; });
          const double aS = hypot(S.re, S.im);
          // |S| - R and |S| + R at a common exponent
          double lo_m; long long lo_e;
          if (R.re == 0.0) { lo_m = aS; lo_e = S.e; }
          else if (aS == 0.0) { lo_m = -R.re; lo_e = R.e; }
          else { lo_e = max(S.e, R.e); lo_m = shift_clamped(aS, S.e - lo_e) - shift_clamped(R.re, R.e - lo_e); }
          const LzC hi = lz_sum(2, [&](int i) { LzC z; z.re = i ? R.re : aS; z.im = 0.0; z.e = i ? R.e : S.e; return z; });
          const bool rest = r + 1 < na;
          if (lo_m > 0.0 && lz_log2(lo_m, lo_e) > V.thr[c]) { dec = 1; by = rest ? 1 : 2; }
          else if (lz_log2(hi.re, hi.e) <= V.thr[c]) { dec = 2; by = rest ? 1 : 2; }
        }
      }
      dec = __shfl_sync(0xffffffffu, dec, 0);
      if (dec == 2) break;
    }
    if (lane == 0) {
      if (dec == 0 && r_hi >= na) { dec = 2; by = 2; }     // cannot happen (R = 0 makes the bracket a point); kept as the oracle has it
      V.decided[c] = dec; V.decided_by[c] = by; V.n_eval[c] = ne;
    }
  }
  if (last && lane == 0) {
    dec = V.decided[c];
    accept[c] = dec == 1; V.p_accept[c] = dec == 1; decided_by[c] = V.decided_by[c]; n_eval[c] = V.n_eval[c]; status[c] = V.p_status[c];
    LzC w; w.re = 0.0; w.im = 0.0; w.e = 0;
    if (dec == 1) {
      const double* tre = V.term_re + (size_t)c * Q; const double* tim = V.term_im + (size_t)c * Q; const long long* te = V.term_e + (size_t)c * Q;
      w = lz_sum(na, [&](int i) { LzC z; z.re = tre[i]; z.im = tim[i]; z.e = te[i]; return z; });
    }
    trace_mant[2 * c] = w.re; trace_mant[2 * c + 1] = w.im; trace_exp2[c] = w.e;
  }
}

// ------------------------------------------------------------------------------------------------ commit / trace
__global__ void lazy_commit_kernel(LazyView V, const int* mask) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= V.nC) return;
  if (mask[c] == 0 || V.p_status[c] != 0) return;
  const int nl = V.p_nleaf[c], total = V.p_ndirty[c];
  const int* pn = V.p_node + (size_t)c * V.smax;
  for (int k = 0; k < nl; ++k) {
    const int leaf = pn[k] - (V.nleaf - 1), cnt = V.sh_n[(size_t)c * V.emax + k];
    V.leaf_n[(size_t)c * V.nleaf + leaf] = cnt;
    for (int i = 0; i < cnt; ++i) {
      V.leaf_tau[((size_t)c * V.nleaf + leaf) * V.cap + i] = V.sh_tau[((size_t)c * V.emax + k) * V.cap + i];
      V.leaf_sym[((size_t)c * V.nleaf + leaf) * V.cap + i] = V.sh_sym[((size_t)c * V.emax + k) * V.cap + i];
    }
  }
  int* fs = V.free_slot + (size_t)c * (V.smax + V.emax);
  for (int i = 0; i < total; ++i) {
    const int old = V.slot_of[(size_t)c * V.nnode + pn[i]];
    V.slot_of[(size_t)c * V.nnode + pn[i]] = fs[i]; fs[i] = old;
  }
  V.p_ndirty[c] = 0; V.p_nleaf[c] = 0; V.decided[c] = 2;
}

// current trace of every chain from its stored root (one warp per chain)
template <bool CPLX>
__global__ void lazy_trace_kernel(LazyView V, double* mant, long long* exp2) {
  constexpr int ES = CPLX ? 2 : 1;
  const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (c >= V.nC) return;
  const int Q = V.imp.Q, rslot = V.slot_of[(size_t)c * V.nnode];
  double* tre = V.term_re + (size_t)c * Q; double* tim = V.term_im + (size_t)c * Q; long long* te = V.term_e + (size_t)c * Q;
  for (int q0 = 0; q0 < Q; ++q0) {
    const size_t en = lz_ent(V, c, rslot, q0);
    double zr = 0.0, zi = 0.0;
    if (V.ent_tgt[en] == q0) {
      const double* Mx = lz_mat(V, c, rslot, q0);
      const int d = V.imp.dim[q0];
      for (int i = lane; i < d; i += 32) { zr += Mx[((long long)i * V.ldm + i) * ES]; if (CPLX) zi += Mx[((long long)i * V.ldm + i) * ES + 1]; }
      zr = warp_sum(zr); zi = warp_sum(zi);
    }
    if (lane == 0) { const LzC t = lz_apply_lg(zr, zi, V.ent_e[en], V.ent_lg[en]); tre[q0] = t.re; tim[q0] = t.im; te[q0] = t.e; }
  }
  if (lane == 0) {
    const LzC w = lz_sum(Q, [&](int i) { LzC z; z.re = tre[i]; z.im = tim[i]; z.e = te[i]; return z; });
    mant[2 * c] = w.re; mant[2 * c + 1] = w.im; exp2[c] = w.e;
  }
}

}  // namespace ctqmc
