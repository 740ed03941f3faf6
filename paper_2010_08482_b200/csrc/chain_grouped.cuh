// Step-synchronous grouped path (SURVEY.md §8(a) a3-a5 for the "many moderate-sized matrices" regime, PAPER.md:31, :71:
// configs 3-4, sector dimensions 1..295, thousands of strings in flight).
//
// All surviving strings of the batch advance one chain position per launch.  At a given position many strings apply the
// SAME operator block F_alpha(q) (there are only a few hundred blocks), so their carried matrices are concatenated column-
// wise and multiplied by F in one GEMM per block:   [X'_s1 | X'_s2 | ...] = F * [X_s1 | X_s2 | ...].
// F is then read once per group instead of once per string, the N dimension is filled with real columns instead of the
// 1..30 columns a single thin-start string carries, and the work is a dense contraction on the FP64 tensor cores
// (mma.sync m8n8k4 f64, 64 x 64 CTA tiles, 8 warps of 32 x 16 -- small warp tiles keep the kernel at 128 registers so that
// 16 warps per SM hide the per-tile latencies --, cp.async pipeline of swizzled 128-byte rows).
// The schedule (which string sits in which column of which tile at which chain position) is a pure function of the
// routing result and is built once per call by three small kernels.
//
// Fusion (a3/a4): each column belongs to a string with its own time difference, so the propagator mantissa
// 2^(x - floor x), x = -Delta_s (E_row - Emin) log2 e, is applied per (row, string) in the epilogue, the integer row
// exponents floor(x) stay implicit and are re-derived bit-exactly (prop_x) by the next step, which folds "row exponent
// minus the string's largest" into the B fragments as an exact power of two.  The largest exponent per string and step
// is reduced with shared-memory atomics per tile and one global atomicMax per string run.
#pragma once
#include <climits>
#include <type_traits>

#include "chain_large.cuh"
#include "chain_small.cuh"

namespace ctqmc {

#ifndef CTQMC_GROUPED_WN
#define CTQMC_GROUPED_WN 4
#endif
// CTA tile 64 x 64; warps: 2 along M x kGWN along N; a warp owns 4 row blocks x kGNT column blocks of 8 x 8
constexpr int kGBM = 64, kGBN = 64, kGStages = 4, kGWN = CTQMC_GROUPED_WN, kGNT = 8 / kGWN, kGThreads = 64 * kGWN;
constexpr int kGStageBytes = (kGBM + kGBN) * 128;

// 2^(e - 1023) for a biased exponent e, built on the integer pipe: e <= 0 gives exactly 0.0 (the row is more than 2^1022
// below the string's largest), e is capped at 2045 (= 2^1022).  Same values as `sh < -1022 ? 0 : pow2i(min(sh, 1022))`.
__device__ __forceinline__ double pow2_biased(int e) { return __hiloint2double(min(max(e, 0), 2045) << 20, 0); }

struct GroupedParams {
  DevImp imp;
  BatchView bv;
  const StringRec* strings;
  const int2* units;
  const Counters* cnt;       // cnt->n_slots = number of units (device-side; the host sizes everything by upper bounds)
  int Lmax, ldx, nb;
  long long xtot;            // elements per parity buffer
  double* X;                 // [2][xtot] elements
  long long* xoff;           // [n_units] element offset of the unit's carried matrix
  int* plan_blk;             // [n_units][Lmax]
  double* plan_delta;        // [n_units][Lmax]
  int* kmax;                 // [n_units][Lmax]
  int* coff;                 // [n_units][Lmax] first column of the unit inside its block group
  int* ulen;                 // [n_units] chain length
  int* ucols;                // [n_units] columns carried
  int* colcnt;               // [Lmax][nb]
  int* colbase;              // [Lmax][nb]
  int4* tiles;               // [Lmax][tile_cap] {block, first column, columns, -}
  int* ntiles;               // [Lmax]
  int* tilecur;              // [Lmax] next (tile, row slab) of the step: the persistent step kernel's work counter
  int2* colmap;              // [Lmax][col_cap] (unit, column of the unit)
  int tile_cap;
  long long col_cap;
  Slot* slots;
};

// One thread per unit: sector walk in multiplication order, per-unit sizes.
__global__ void grouped_plan_kernel(GroupedParams P) {
  const int u = blockIdx.x * blockDim.x + threadIdx.x;
  if (u >= (int)P.cnt->n_slots) return;
  const int2 un = P.units[u];
  const StringRec sr = P.strings[un.x];
  const int Q = P.imp.Q;
  const long long b = un.x / Q;
  const long long base = P.bv.offset[b];
  const int L = (int)(P.bv.offset[b + 1] - base);
  const int* sym = P.bv.symbol + base;
  const double* tau = P.bv.tau + base;
  P.ulen[u] = L;
  P.ucols[u] = sr.c;
  int q = sr.q_start;
  for (int j = 0; j < L; ++j) {
    int i = sr.r + j;
    if (i >= L) i -= L;
    const int blk = P.imp.blk_of[sym[i] * Q + q];
    P.plan_blk[(size_t)u * P.Lmax + j] = blk;
    P.plan_delta[(size_t)u * P.Lmax + j] = (i + 1 < L) ? (tau[i + 1] - tau[i]) : (P.bv.beta - tau[i] + tau[0]);
    P.kmax[(size_t)u * P.Lmax + j] = INT_MIN;
    q = P.imp.blks[blk].dst;
  }
}

// Exclusive prefix sum of ucols * ldx -> xoff (one CTA; n_units is at most a few hundred thousand on this path).
__global__ void grouped_xoff_kernel(GroupedParams P) {
  __shared__ long long s_part[1024];
  __shared__ long long s_run;
  const int n_units = (int)P.cnt->n_slots;
  if (threadIdx.x == 0) s_run = 0;
  __syncthreads();
  for (int base = 0; base < n_units; base += 1024) {
    const int u = base + threadIdx.x;
    const long long v = (u < n_units) ? (long long)P.ucols[u] * P.ldx : 0;
    s_part[threadIdx.x] = v;
    __syncthreads();
    for (int o = 1; o < 1024; o <<= 1) {
      long long add = (threadIdx.x >= o) ? s_part[threadIdx.x - o] : 0;
      __syncthreads();
      s_part[threadIdx.x] += add;
      __syncthreads();
    }
    if (u < n_units) P.xoff[u] = s_run + s_part[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == 0) s_run += s_part[1023];
    __syncthreads();
  }
}

// Schedule, pass 1: columns per (chain position, block); each unit reserves its column range inside the group.
__global__ void grouped_count_kernel(GroupedParams P) {
  const long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= (long long)P.cnt->n_slots * P.Lmax) return;
  const int u = (int)(idx / P.Lmax), j = (int)(idx - (long long)u * P.Lmax);
  if (j >= P.ulen[u]) return;
  const int blk = P.plan_blk[idx];
  P.coff[idx] = atomicAdd(&P.colcnt[(size_t)j * P.nb + blk], P.ucols[u]);
}

// Schedule, pass 2: one CTA per chain position; block groups -> column bases and the tile list.
__global__ void grouped_tiles_kernel(GroupedParams P) {
  const int j = blockIdx.x;
  if (threadIdx.x != 0) return;
  int col = 0, nt = 0;
  for (int o = 0; o < P.nb; ++o) {   // heaviest blocks first: the launch's tail is made of short tiles
    const int blk = P.imp.blk_order[o];
    const int cnt = P.colcnt[(size_t)j * P.nb + blk];
    P.colbase[(size_t)j * P.nb + blk] = col;
    for (int c0 = 0; c0 < cnt; c0 += kGBN) {
      if (nt < P.tile_cap) P.tiles[(size_t)j * P.tile_cap + nt] = make_int4(blk, col + c0, min(kGBN, cnt - c0), 0);
      ++nt;
    }
    col += cnt;
  }
  P.ntiles[j] = min(nt, P.tile_cap);
}

// Schedule, pass 3: column -> (unit, column of the unit).
__global__ void grouped_fill_kernel(GroupedParams P) {
  const long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= (long long)P.cnt->n_slots * P.Lmax) return;
  const int u = (int)(idx / P.Lmax), j = (int)(idx - (long long)u * P.Lmax);
  if (j >= P.ulen[u]) return;
  const int blk = P.plan_blk[idx];
  const int c = P.ucols[u];
  int2* dst = P.colmap + (size_t)j * P.col_cap + P.colbase[(size_t)j * P.nb + blk] + P.coff[idx];
  for (int i = 0; i < c; ++i) dst[i] = make_int2(u, i);
}

// X_0 = identity for every unit (grid: units).
template <bool CPLX>
__global__ void grouped_init_kernel(GroupedParams P) {
  constexpr int ES = CPLX ? 2 : 1;
  const int n_units = (int)P.cnt->n_slots;
  // whole columns (ldx rows) of BOTH parity buffers: rows beyond the current sector's dimension are read (and multiplied by
  // an exact 0 or by zero padding of F) by later steps, so they must be finite whatever the shared arena held before
  for (int u = blockIdx.x; u < n_units; u += gridDim.x) {
    const int c = P.ucols[u];
    double* X0 = P.X + P.xoff[u] * ES;
    double* X1 = X0 + P.xtot * ES;
    for (int idx = threadIdx.x; idx < c * P.ldx; idx += blockDim.x) {
      const int col = idx / P.ldx, k = idx - col * P.ldx;
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
}

// One chain position for every string.  Work item = (tile of the step's tile list, 64-row slab of F); the number of items is
// known on the device only (the host sizes the launch by an upper bound and never reads a counter back), so the grid is
// persistent: a few CTAs per SM pull items from an atomic counter, heaviest tiles first.
template <bool CPLX>
__global__ void __launch_bounds__(kGThreads, (kGWN == 2 && !CPLX) ? 3 : 2) grouped_step_kernel(GroupedParams P, int j, int MTmax) {
  constexpr int ES = CPLX ? 2 : 1;
  constexpr int BKE = CPLX ? 8 : 16;
  extern __shared__ __align__(128) unsigned char gsm[];
  __shared__ const unsigned char* s_xin[kGBN];
  __shared__ double* s_xout[kGBN];
  __shared__ double s_dprev[kGBN], s_delta[kGBN];
  __shared__ int s_kprev[kGBN], s_u[kGBN], s_kmax[kGBN];
  __shared__ __align__(8) unsigned long long g_full[kGStages], g_empty[kGStages];
  __shared__ int s_item;
  double* sde = reinterpret_cast<double*>(gsm + kGStages * kGStageBytes);   // E[k] - Emin of the source sector

  // Programmatic dependent launch: the next chain position's grid may start as soon as every CTA of this one is resident, so
  // its CTAs fill the SM slots this launch's tail leaves empty and run their prologue (tile list, column map, barrier
  // set-up: nothing a previous step writes) there; they wait (griddepcontrol.wait, below) before touching the carried matrices.
  asm volatile("griddepcontrol.launch_dependents;");
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int g = lane >> 2, t = lane & 3;
  const int wm = warp / kGWN, wn = warp % kGWN;
  if (tid == 0) {
#pragma unroll
    for (int st = 0; st < kGStages; ++st) { mbar_init(&g_full[st], kGThreads); mbar_init(&g_empty[st], kGThreads / 32); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  const int n_items = P.ntiles[j] * MTmax;
  unsigned gk = 0;          // k-tiles this CTA has pushed through the ring so far: slot = gk % stages, phase = (gk / stages) & 1
  bool waited = false;
  for (;;) {
  __syncthreads();          // everybody is done with the previous item's shared arrays
  if (tid == 0) s_item = atomicAdd(&P.tilecur[j], 1);
  __syncthreads();
  const int item = s_item;
  if (item >= n_items) break;
  const int tile_id = item / MTmax, slab = item - tile_id * MTmax;   // slabs of a tile are neighbours: F rows stay in L2
  const int4 tl = P.tiles[(size_t)j * P.tile_cap + tile_id];
  const BlkDesc bd = P.imp.blks[tl.x];
  const int dn = bd.rows, d = bd.cols, ncols = tl.z;
  const int m0 = slab * kGBM;
  if (m0 >= dn) continue;
  const int nkt = (d + BKE - 1) / BKE;
  // 8-row / 8-column blocks are dealt to the warps round-robin, and blocks that are all padding are skipped: the tensor
  // work is quantised to 8 x 8 although the CTA stages 64 x 64 tiles
  const int mtu = ((min(kGBM, dn - m0) + 7) / 8 - wm + 1) / 2;
  const int ntu = ((ncols + 7) / 8 - wn + kGWN - 1) / kGWN;
  const size_t par_in = (size_t)(j & 1) * P.xtot, par_out = (size_t)((j + 1) & 1) * P.xtot;

  {   // source-sector energies: static data, still before the wait
    const double* Eq = P.imp.energy + P.imp.e_off[bd.src];
    const double emin = P.imp.e_min[bd.src];
    for (int k = tid; k < nkt * BKE; k += kGThreads) sde[k] = (k < d) ? __dsub_rn(Eq[k], emin) : 0.0;
  }
  if (!waited) { asm volatile("griddepcontrol.wait;" ::: "memory"); waited = true; }   // the previous chain position is complete and its writes are visible
  if (tid < kGBN) {
    const int n = tid;
    if (n < ncols) {
      const int2 ui = P.colmap[(size_t)j * P.col_cap + tl.y + n];
      const size_t idx = (size_t)ui.x * P.Lmax + j;
      const size_t col = (size_t)P.xoff[ui.x] + (size_t)ui.y * P.ldx;
      s_xin[n] = reinterpret_cast<const unsigned char*>(P.X + (par_in + col) * ES);
      s_xout[n] = P.X + (par_out + col) * ES;
      s_delta[n] = P.plan_delta[idx];
      int kp = 0;
      double dp = 0.0;               // j == 0: x = 0, shift 0, factor 1 (X_0 is the identity)
      if (j > 0) { kp = P.kmax[idx - 1]; dp = P.plan_delta[idx - 1]; }
      s_kprev[n] = (kp == INT_MIN) ? (1 << 29) : kp;   // a dead string keeps multiplying zeros
      s_dprev[n] = dp;
      s_u[n] = ui.x;
    } else {
      s_xin[n] = nullptr; s_xout[n] = nullptr; s_delta[n] = 0.0; s_dprev[n] = 0.0; s_kprev[n] = 1 << 29; s_u[n] = -1;
    }
    s_kmax[n] = INT_MIN;
  }
  __syncthreads();

  const unsigned char* Ag = reinterpret_cast<const unsigned char*>(P.imp.store + bd.off);
  const int rows_pad = round_up(dn, 8);
  const size_t a_row_bytes = (size_t)bd.ld * ES * 8;
  const int ld_chunks = bd.ld * ES / 2;
  const int x_chunks = CPLX ? d : (d + 1) / 2;

  auto load_stage = [&](int kt, int stage) {
    unsigned char* As = gsm + stage * kGStageBytes;
    unsigned char* Bs = As + kGBM * 128;
#pragma unroll
    for (int i = 0; i < kGBM * 8 / kGThreads; ++i) {
      const int idx = tid + i * kGThreads, r = idx >> 3, ch = idx & 7;
      const int row = m0 + r, gch = kt * 8 + ch;
      const bool ok = row < rows_pad && gch < ld_chunks;
      cp_async16(As + r * 128 + ((ch ^ ((r & 1) << 2)) << 4), ok ? Ag + (size_t)row * a_row_bytes + (size_t)gch * 16 : Ag, ok);
    }
#pragma unroll
    for (int i = 0; i < kGBN * 8 / kGThreads; ++i) {
      const int idx = tid + i * kGThreads, r = idx >> 3, ch = idx & 7;
      const int gch = kt * 8 + ch;
      const unsigned char* src = s_xin[r];
      const bool ok = src != nullptr && gch < x_chunks;
      cp_async16(Bs + r * 128 + ((ch ^ ((r & 1) << 2)) << 4), ok ? src + (size_t)gch * 16 : Ag, ok);
    }
  };

  double acc[4][kGNT][CPLX ? 4 : 2];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < kGNT; ++b)
#pragma unroll
      for (int x = 0; x < (CPLX ? 4 : 2); ++x) acc[a][b][x] = 0.0;

  // this lane's B-fragment columns: n = wn*32 + nt*8 + g
  double ndp[kGNT];
  int kpv[kGNT];
#pragma unroll
  for (int nt = 0; nt < kGNT; ++nt) { ndp[nt] = -s_dprev[(nt * kGWN + wn) * 8 + g]; kpv[nt] = s_kprev[(nt * kGWN + wn) * 8 + g] - 1023; }   // biased

  // the main loop is instantiated for every (row blocks, column blocks) count of a warp, so partial tiles issue only the
  // DMMAs they need and the loops stay fully unrolled
  auto mainloop = [&](auto mtc, auto ntc) {
    constexpr int MTU = decltype(mtc)::value, NTU = decltype(ntc)::value;
    // full/empty mbarrier ring (as in the large-sector kernel), fed by cp.async: a thread's copies of a stage arrive on the
    // stage's "full" barrier when they land (cp.async.mbarrier.arrive.noinc), a warp releases a slot on its "empty" barrier;
    // the slot consumed two k-tiles ago is refilled, so there is no CTA-wide barrier in the loop
    constexpr int kAhead = kGStages - 2;
  #pragma unroll
    for (int st = 0; st < kAhead; ++st)
      if (st < nkt) {
        const unsigned n = gk + st;
        if (n >= kGStages) mbar_wait(&g_empty[n % kGStages], ((n / kGStages) - 1) & 1);
        load_stage(st, n % kGStages);
        cp_async_arrive(&g_full[n % kGStages]);
      }
    const int swz = (g & 1) << 2;
    for (int kt = 0; kt < nkt; ++kt) {
      {
        const int nx = kt + kAhead;
        if (nx < nkt) {
          const unsigned n = gk + nx;
          if (n >= kGStages) mbar_wait(&g_empty[n % kGStages], ((n / kGStages) - 1) & 1);
          load_stage(nx, n % kGStages);
          cp_async_arrive(&g_full[n % kGStages]);
        }
      }
      const unsigned nc = gk + kt;
      mbar_wait(&g_full[nc % kGStages], (nc / kGStages) & 1);
      const unsigned char* As = gsm + (nc % kGStages) * kGStageBytes;
      const unsigned char* Bs = As + kGBM * 128;
  #pragma unroll
      for (int sub = 0; sub < 2; ++sub) {
        const int ch = sub * 4 + t;
        const int so = ((ch ^ swz) << 4);
        double2 a[MTU > 0 ? MTU : 1], b[NTU > 0 ? NTU : 1];
  #pragma unroll
        for (int mt = 0; mt < MTU; ++mt) a[mt] = *reinterpret_cast<const double2*>(As + ((mt * 2 + wm) * 8 + g) * 128 + so);
  #pragma unroll
        for (int nt = 0; nt < NTU; ++nt) b[nt] = *reinterpret_cast<const double2*>(Bs + ((nt * kGWN + wn) * 8 + g) * 128 + so);
        if constexpr (CPLX) {
          const double de = sde[kt * 8 + ch];
  #pragma unroll
          for (int nt = 0; nt < NTU; ++nt) {
            const double f = pow2_biased(__double2int_rd(__dmul_rn(__dmul_rn(ndp[nt], de), kLog2e)) - kpv[nt]);
            b[nt].x *= f; b[nt].y *= f;
          }
  #pragma unroll
          for (int mt = 0; mt < MTU; ++mt)
  #pragma unroll
            for (int nt = 0; nt < NTU; ++nt)
              {
                dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt].x, b[nt].x);
                dmma884(acc[mt][nt][2], acc[mt][nt][3], a[mt].x, b[nt].y);
              }
  #pragma unroll
          for (int mt = 0; mt < MTU; ++mt) {
            const double na = -a[mt].y;
  #pragma unroll
            for (int nt = 0; nt < NTU; ++nt)
              {
                dmma884(acc[mt][nt][0], acc[mt][nt][1], na, b[nt].y);
                dmma884(acc[mt][nt][2], acc[mt][nt][3], a[mt].y, b[nt].x);
              }
          }
        } else {
          const double2 de = *reinterpret_cast<const double2*>(sde + kt * 16 + ch * 2);
  #pragma unroll
          for (int nt = 0; nt < NTU; ++nt) {
            b[nt].x *= pow2_biased(__double2int_rd(__dmul_rn(__dmul_rn(ndp[nt], de.x), kLog2e)) - kpv[nt]);
            b[nt].y *= pow2_biased(__double2int_rd(__dmul_rn(__dmul_rn(ndp[nt], de.y), kLog2e)) - kpv[nt]);
          }
  #pragma unroll
          for (int mt = 0; mt < MTU; ++mt)
  #pragma unroll
            for (int nt = 0; nt < NTU; ++nt)
              dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt].x, b[nt].x);
  #pragma unroll
          for (int mt = 0; mt < MTU; ++mt)
  #pragma unroll
            for (int nt = 0; nt < NTU; ++nt)
              dmma884(acc[mt][nt][0], acc[mt][nt][1], a[mt].y, b[nt].y);
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&g_empty[nc % kGStages]);
    }
  };
#define CTQMC_GD(M, N) case (M) * 8 + (N): mainloop(std::integral_constant<int, M>{}, std::integral_constant<int, N>{}); break;
  switch ((mtu > 0 && ntu > 0) ? mtu * 8 + ntu : 0) {
    CTQMC_GD(1, 1) CTQMC_GD(2, 1) CTQMC_GD(3, 1) CTQMC_GD(4, 1)
#if CTQMC_GROUPED_WN <= 4
    CTQMC_GD(1, 2) CTQMC_GD(2, 2) CTQMC_GD(3, 2) CTQMC_GD(4, 2)
#endif
#if CTQMC_GROUPED_WN <= 2
    CTQMC_GD(1, 3) CTQMC_GD(1, 4) CTQMC_GD(2, 3) CTQMC_GD(2, 4) CTQMC_GD(3, 3) CTQMC_GD(3, 4) CTQMC_GD(4, 3) CTQMC_GD(4, 4)
#endif
    default: mainloop(std::integral_constant<int, 0>{}, std::integral_constant<int, 0>{}); break;
  }
#undef CTQMC_GD
  gk += nkt;

  // ---- epilogue: per (row, string) propagator mantissa, scatter to the strings' matrices, largest exponent per column
  const double* E = P.imp.energy + P.imp.e_off[bd.dst];
  const double emin = P.imp.e_min[bd.dst];
  double er[4];
#pragma unroll
  for (int mt = 0; mt < 4; ++mt) {
    const int row = m0 + (mt * 2 + wm) * 8 + g;
    er[mt] = (row < dn) ? E[row] : emin;
  }
  int cur_u = -2;
  double mr[4];
  int kr[4];
#pragma unroll
  for (int nt = 0; nt < kGNT; ++nt) {
#pragma unroll
    for (int half = 0; half < 2; ++half) {
      const int n = (nt * kGWN + wn) * 8 + 2 * t + half;
      const int u = s_u[n];
      if (u < 0) continue;
      if (u != cur_u) {   // columns of one string are adjacent: its row factors are computed once
        cur_u = u;
        const double delta = s_delta[n];
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
          const double x = prop_x(delta, er[mt], emin);
          const double kf = floor(x);
          mr[mt] = exp2(__dsub_rn(x, kf));
          kr[mt] = row_exp(x);
        }
      }
      double* xo = s_xout[n];
      int cexp = INT_MIN;
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) {
        const int row = m0 + (mt * 2 + wm) * 8 + g;
        if (row < dn) {
          if constexpr (CPLX) {
            const double2 v = make_double2(acc[mt][nt][half] * mr[mt], acc[mt][nt][2 + half] * mr[mt]);
            *reinterpret_cast<double2*>(xo + (size_t)row * 2) = v;
            const double mx = fmax(fabs(v.x), fabs(v.y));
            if (mx > 0.0) cexp = max(cexp, kr[mt] + ilogb_fast(mx));
          } else {
            const double v = acc[mt][nt][half] * mr[mt];
            xo[row] = v;
            if (v != 0.0) cexp = max(cexp, kr[mt] + ilogb_fast(v));
          }
        } else if (!CPLX && row == dn && (dn & 1)) {
          xo[row] = 0.0;   // real matrices are read in 16-byte chunks of two rows: the pad row of an odd sector must hold an
                           // exact zero, not whatever an earlier string left in the arena (it is scaled by 2^-kprev on load)
        }
      }
      if (cexp != INT_MIN) atomicMax(&s_kmax[n], cexp);
    }
  }
  __syncthreads();
  if (tid < ncols) {
    const int u = s_u[tid];
    if (tid == 0 || s_u[tid - 1] != u) {   // leader of a run of columns of the same string
      int k = INT_MIN;
      for (int n = tid; n < ncols && s_u[n] == u; ++n) k = max(k, s_kmax[n]);
      if (k != INT_MIN) atomicMax(&P.kmax[(size_t)u * P.Lmax + j], k);
    }
  }
  }   // item loop
}

// Trace of each string's final matrix (a5); one CTA per unit.
template <bool CPLX>
__global__ void grouped_finish_kernel(GroupedParams P) {
  constexpr int ES = CPLX ? 2 : 1;
  __shared__ double red[2][8];
  const int u = blockIdx.x;
  if (u >= (int)P.cnt->n_slots) return;
  const int2 un = P.units[u];
  const StringRec sr = P.strings[un.x];
  const int L = P.ulen[u], c = sr.c, q = sr.q_start;
  const double* E = P.imp.energy + P.imp.e_off[q];
  const double emin = P.imp.e_min[q];
  double re = 0.0, im = 0.0;
  long long e2 = 0;
  bool dead = false;
  if (L == 0) {
    for (int n = threadIdx.x; n < c; n += blockDim.x) re += exp(-P.bv.beta * (E[n] - emin));
  } else {
    for (int j = 0; j < L; ++j) {
      const int k = P.kmax[(size_t)u * P.Lmax + j];
      if (k == INT_MIN) { dead = true; break; }
      e2 += k;
    }
    if (!dead) {
      const int klast = P.kmax[(size_t)u * P.Lmax + L - 1];
      const double dlast = P.plan_delta[(size_t)u * P.Lmax + L - 1];
      const double* X = P.X + ((size_t)(L & 1) * P.xtot + P.xoff[u]) * ES;
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
    }
  }
  re = warp_sum(re); im = warp_sum(im);
  if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = re; red[1][threadIdx.x >> 5] = im; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double tr = 0.0, ti = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) { tr += red[0][w]; ti += red[1][w]; }
    Slot out; out.re = dead ? 0.0 : tr; out.im = dead ? 0.0 : ti; out.e2 = dead ? 0 : e2; out.pad = 0;
    P.slots[sr.slot] = out;
  }
}

inline size_t grouped_smem_bytes(int dmax) {
  return (size_t)kGStages * kGStageBytes + (size_t)((dmax + 15) / 16 * 16 + 16) * sizeof(double);
}

}  // namespace ctqmc
