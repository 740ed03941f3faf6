// C ABI of libctqmc_b200 (include/ctqmc.h): host-side validation, device store construction, scratch arena and the
// kernel sequence of ctqmc_trace_batch / ctqmc_bound_batch.  sm_100a only; there is no CPU fallback anywhere.
#include "../../include/ctqmc.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "chain.cuh"
#include "chain_grouped.cuh"
#include "chain_large.cuh"
#include "chain_small.cuh"
#include "chain_small2.cuh"
#include "bound_small2.cuh"
#include "common.cuh"
#include "peak.cuh"
#include "reduce.cuh"
#include "route.cuh"
#include "store.cuh"
#include "split_gemm.cuh"

using namespace ctqmc;

namespace {

thread_local std::string g_err;

int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  g_err = buf;
  return code;
}

#define CU(call)                                                                                   \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return fail(e_ == cudaErrorMemoryAllocation ? CTQMC_ERR_OOM : CTQMC_ERR_CUDA, "%s: %s (%s:%d)", #call, \
                  cudaGetErrorString(e_), __FILE__, __LINE__);                                     \
  } while (0)

template <class T>
int upload(T** dst, const std::vector<T>& v) {
  *dst = nullptr;
  size_t bytes = (v.size() ? v.size() : 1) * sizeof(T);
  CU(cudaMalloc((void**)dst, bytes));
  if (!v.empty()) CU(cudaMemcpy(*dst, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  return 0;
}

struct Arena {
  // ONE device block, allocated between calls (at the first call that needs it, when a later call needs more and growth is
  // allowed, or by ctqmc_set_option(CTQMC_OPT_ARENA_BYTES)) and carved up on the host from upper bounds the host knows (B, Q,
  // n_ops, max_len, sector dimensions): nothing is sized from a device counter, so a batch call never waits for the device
  // ("only asynchronous CUDA functions ... pre-allocate ... our own memory allocator").
  char* base = nullptr;
  size_t cap = 0;
  size_t fixed_bytes = 0;            // > 0: size set by the caller, never grown
  Counters* cnt = nullptr;           // counters of the current round
  Counters* cnt_total = nullptr;     // summed over the rounds of the last call (ctqmc_last_stats)
  // host-variant staging
  void* h_stage = nullptr; size_t h_stage_bytes = 0;
  void* d_stage = nullptr; size_t d_stage_bytes = 0;
};

enum RoundKind { K_PANEL = 0, K_GROUPED = 1, K_LARGE = 2, K_TABLES = 3 };

// Pointers of one round's scratch inside the arena block.
struct RoundBuf {
  int* status; uint8_t* survive; StringRec* strings; Scaled* sector; int2* units; Slot* slots;
  long long n_units_cap;
  // large-sector path
  signed char* sp_b; int* sp_eb; int sp_npad, sp_kpad; int* sp_items; int* sp_ctr;
  double* lx; long long lx_cols; int* plan_blk; double* plan_delta; int* lkmax; int* lunit; long long* lux; long long G; int lstride;
  // grouped path
  double* gx; long long sum_c_cap; long long* gxoff; int* gplan_blk; double* gplan_delta; int* gkmax; int* gcoff; int* gulen; int* gucols;
  int* gcolcnt; int* gcolbase; int4* gtiles; int* gntiles; int* gtilecur; int2* gcolmap; int tile_cap;
};

struct Bump {
  char* base; size_t off = 0;
  template <class T> T* take(size_t n) {
    off = (off + 255) / 256 * 256;
    T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
    off += (n ? n : 1) * sizeof(T);
    return p;
  }
};

}  // namespace

struct ctqmc_impurity {
  int device = 0;
  int sm_count = 0;
  DevImp dev{};
  int n_blocks = 0;
  // owned device arrays
  int* d_dim = nullptr; long long* d_eoff = nullptr; double* d_energy = nullptr; double* d_emin = nullptr;
  int* d_blkof = nullptr; BlkDesc* d_blks = nullptr; double* d_store = nullptr; double* d_rownorm2 = nullptr;
  double* d_sigma = nullptr;
  int* d_blkorder = nullptr;
  // split-precision large-sector path (split_gemm.cuh): int8 slice planes of the operator store, their tensor maps
  int split = 0, split_slices = 7;
  signed char* d_sp_planes = nullptr; long long* d_sp_aoff = nullptr; int* d_sp_ea = nullptr; long long* d_sp_eaoff = nullptr;
  long long* d_rho_off = nullptr;     // [Q] offset of sector q's block in the reduced density matrix (sum of dim^2)
  long long rho_len = 0;
  std::vector<BlkDesc> h_blks;        // host copy (tensor-map construction)
  CUtensorMap* d_amaps = nullptr;     // large path, TMA variant: one tensor map per operator block
  int use_tma = 1;
  double* d_pack = nullptr; int4* d_pblk = nullptr;   // small-sector path: unpadded store
  int pack_len = 0, n_energy = 0;
  int small_ok = 0, small = 0, small_g = 32, small_grid_max = 0;
  double* d_ftpad = nullptr; int2* d_binfo = nullptr;   // uniform small-sector variant (real): padded transposed blocks
  int small2 = 0, small2_dp = 0, small2_threads = 512;
  int small2_occ[17] = {0};
  size_t small2_smem = 0;
  size_t small_smem = 0;
  // schedule
  int schedule = CTQMC_SCHEDULE_THIN;
  int path = CTQMC_PATH_AUTO;
  long long scratch_limit = 0;   // bytes the grouped path may use for its schedule and carried matrices (0 = no limit)
  int nt = 0, team_warps = 8, ldx = 0, large = 0, grouped = 0, grouped_ok = 0, grouped_now = 0, last_path = 0;
  size_t grouped_smem = 0;
  int grouped_ctas_per_sm = 2;
  size_t smem_bytes = 0;
  int grid = 0;
  Arena arena;
  cudaStream_t last_stream = nullptr;
  long long last_launches = 0;
  int keep_totals = 0;                         // host form, chunked: later chunks add to the first chunk's counters
  int timing = 0, timing_valid = 0;
  cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
  cudaStream_t copy_stream = nullptr;          // host form, pinned inputs: H2D of chunk k+1 overlaps the kernel of chunk k
  cudaEvent_t ev_chunk[9] = {nullptr};
};

namespace {

constexpr long long kGroupedMinBatch = 64;   // measured crossover: the panel kernel wins at 32 configurations, the grouped path at 128

using KernelFn = void (*)(ChainParams);

KernelFn pick_kernel(int cplx, int nt, int tw) {
#define PICK(C, N, T) if (cplx == C && nt == N && tw == T) return chain_kernel<(C != 0), N, T>;
  PICK(0, 1, 1) PICK(0, 2, 1) PICK(1, 1, 1) PICK(1, 2, 1)
  PICK(0, 1, 8) PICK(0, 2, 8) PICK(0, 4, 8)
  PICK(1, 1, 8) PICK(1, 2, 8) PICK(1, 4, 8)
#undef PICK
  return nullptr;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// 2-D FP64 tensor map: `inner` doubles contiguous, `outer` rows of `stride_bytes`; box = 8 doubles (64 B) x box_outer rows,
// no swizzle, out-of-range elements read as zero.
int encode_2d(CUtensorMap* m, const void* base, unsigned long long inner, unsigned long long outer, unsigned long long stride_bytes,
              unsigned box_outer) {
  EncodeTiledFn fn = encode_tiled_fn();
  if (!fn) return fail(CTQMC_ERR_CUDA, "cuTensorMapEncodeTiled is not available from this driver");
  const cuuint64_t dims[2] = {inner, outer}, strides[1] = {stride_bytes};
  const cuuint32_t box[2] = {8, box_outer}, estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(CTQMC_ERR_CUDA, "cuTensorMapEncodeTiled failed (%d): inner %llu outer %llu stride %llu", (int)r, inner, outer, stride_bytes);
  return 0;
}

using SplitStepFn = void (*)(LargeParams, SplitStepParams, int, int, int, SplitList);
SplitStepFn pick_split(int S) {
  switch (S) { case 5: return split_step_kernel<5>; case 6: return split_step_kernel<6>; case 7: return split_step_kernel<7>; case 8: return split_step_kernel<8>; }
  return nullptr;
}
size_t split_smem(int S) { return (size_t)sp_stages(S) * 2 * S * kSpTile + 1024; }

// Builds (once) the int8 slice planes of the operator store for the split-precision path.
int split_prepare(ctqmc_impurity* h) {
  if (h->d_sp_planes) return 0;
  const int nb = h->n_blocks, S = h->split_slices;
  std::vector<long long> aoff(nb), eaoff(nb);
  long long bytes = 0, rows = 0;
  int mpmax = 0;
  for (int b = 0; b < nb; ++b) {
    const BlkDesc& bd = h->h_blks[b];
    const long long Mp = sp_pad(bd.rows), Kp = sp_pad(bd.cols);
    aoff[b] = bytes; eaoff[b] = rows;
    bytes += 2LL * S * Mp * Kp; rows += Mp;
    if (Mp > mpmax) mpmax = (int)Mp;
  }
  CU(cudaMalloc((void**)&h->d_sp_planes, (size_t)(bytes ? bytes : 1)));
  CU(cudaMemset(h->d_sp_planes, 0, (size_t)(bytes ? bytes : 1)));
  CU(cudaMalloc((void**)&h->d_sp_ea, (size_t)(rows ? rows : 1) * sizeof(int)));
  CU(cudaMemset(h->d_sp_ea, 0, (size_t)(rows ? rows : 1) * sizeof(int)));
  int rc = upload(&h->d_sp_aoff, aoff); if (rc) return rc;
  rc = upload(&h->d_sp_eaoff, eaoff); if (rc) return rc;
  SplitStore st; st.planes = h->d_sp_planes; st.a_off = h->d_sp_aoff; st.ea = h->d_sp_ea; st.ea_off = h->d_sp_eaoff; st.S = S;
  if (nb > 0) split_slice_store_kernel<<<dim3((unsigned)mpmax, (unsigned)nb), 128>>>(h->dev, st);
  CU(cudaGetLastError());
  CU(cudaFuncSetAttribute(pick_split(S), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)split_smem(S)));
  CU(cudaDeviceSynchronize());
  return 0;
}

using SmallFn = void (*)(SmallParams);
SmallFn pick_small(int cplx, int g) {
  if (cplx) return g == 8 ? small_trace_kernel<true, 8> : g == 16 ? small_trace_kernel<true, 16> : small_trace_kernel<true, 32>;
  return g == 8 ? small_trace_kernel<false, 8> : g == 16 ? small_trace_kernel<false, 16> : small_trace_kernel<false, 32>;
}

using Small2Fn = void (*)(Small2Params);
Small2Fn pick_small2(int dp) {
  switch (dp) {
    case 2: return small2_trace_kernel<2>;   case 4: return small2_trace_kernel<4>;   case 6: return small2_trace_kernel<6>;
    case 9: return small2_trace_kernel<9>;   case 12: return small2_trace_kernel<12>; case 16: return small2_trace_kernel<16>;
  }
  return nullptr;
}
using Small2BoundFn = void (*)(Small2BoundParams);
Small2BoundFn pick_small2_bound(int dp) {
  switch (dp) {
    case 2: return small2_bound_kernel<2>;   case 4: return small2_bound_kernel<4>;   case 6: return small2_bound_kernel<6>;
    case 9: return small2_bound_kernel<9>;   case 12: return small2_bound_kernel<12>; case 16: return small2_bound_kernel<16>;
  }
  return nullptr;
}
int small2_dp_for(int dmax) { const int c[6] = {2, 4, 6, 9, 12, 16}; for (int v : c) if (v >= dmax) return v; return 0; }

int pick_ldx(int cplx, int dmax) {
  int l = (dmax + 7) / 8 * 8;
  if (cplx) { while (l % 8 != 4) ++l; }       // 16-byte elements: conflict-free 128-bit fragment loads need ldx = 4 mod 8
  else      { while (l % 16 != 8) ++l; }      // 8-byte elements, two per load: ldx = 8 mod 16
  return l;
}

// Choose panel width / team size for this impurity and set up the persistent grid.
int configure(ctqmc_impurity* h, int want_w) {
  const int cplx = h->dev.cplx, es = cplx ? 2 : 1;
  const size_t smem_max = 227 * 1024 - 2048;
  h->small = 0;
  if (h->path == CTQMC_PATH_SMALL && !h->small_ok)
    return fail(CTQMC_ERR_UNSUPPORTED, "the small-sector kernel needs all sectors <= 16 states and a store that fits in shared memory");
  if (h->small_ok && (h->path == CTQMC_PATH_AUTO || h->path == CTQMC_PATH_SMALL)) {
    int g = h->dev.dmax <= 2 ? 8 : h->dev.dmax <= 4 ? 16 : 32;
    if (const char* e = getenv("CTQMC_SMALL_G")) { int v = atoi(e); if (v == 8 || v == 16 || v == 32) g = v; }
    h->small_g = g;
    h->small_smem = small_common_bytes(h->dev.Q, h->dev.A, h->n_blocks, h->pack_len, h->n_energy, es) +
                    (size_t)(kCtaThreads / g) * small_group_bytes(h->dev.Q, h->dev.dmax, es);
    if (h->small_smem <= smem_max) {
      SmallFn fn = pick_small(cplx, g);
      CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->small_smem));
      int occ = 0;
      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kCtaThreads, h->small_smem));
      if (occ >= 1) { h->small = 1; h->small_grid_max = occ * h->sm_count; }
    }
    if (!h->small && h->path == CTQMC_PATH_SMALL) return fail(CTQMC_ERR_UNSUPPORTED, "small-sector kernel does not fit in shared memory");
    // uniform variant for real impurities (chain_small2.cuh) unless CTQMC_SMALL_V1=1
    h->small2 = 0;
    const char* v1 = getenv("CTQMC_SMALL_V1");
    if (h->small && h->d_ftpad && !(v1 && atoi(v1))) {
      const int dp = h->small2_dp;
      Small2Fn fn = pick_small2(dp);
      for (int threads : {512, 256}) {
        const size_t bytes = small2_common_bytes(h->dev.Q, h->dev.A, h->n_blocks, dp) +
                             (size_t)(threads / 32) * (32 / dp) * small2_group_bytes(h->dev.Q, dp);
        if (fn && bytes <= smem_max) {
          CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
          int occ = 0;
          CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, bytes));
          if (occ >= 1) { h->small2 = 1; h->small2_threads = threads; h->small2_smem = bytes; h->small_grid_max = occ * h->sm_count; break; }
        }
      }
    }
  }
  h->ldx = pick_ldx(cplx, h->dev.dmax);
  h->team_warps = h->dev.dmax <= 16 ? 1 : 8;
  const int teams = kCtaWarps / h->team_warps;
  int nt_try[3] = {4, 2, 1};
  h->nt = 0;
  h->large = 0;
  for (int i = 0; i < 3 && h->path != CTQMC_PATH_LARGE && h->path != CTQMC_PATH_SPLIT; ++i) {
    int nt = nt_try[i];
    if (want_w && nt * 8 != want_w) continue;
    if (!pick_kernel(cplx, nt, h->team_warps)) continue;
    size_t bytes = (size_t)teams * 2 * (8 * nt) * h->ldx * es * sizeof(double);
    if (bytes <= smem_max) { h->nt = nt; h->smem_bytes = bytes; break; }
  }
  if (h->path == CTQMC_PATH_PANEL && h->nt == 0)
    return fail(CTQMC_ERR_UNSUPPORTED, "the shared-memory panel kernel cannot hold sectors of dimension %d", h->dev.dmax);
  h->grouped = 0; h->grouped_ok = 0;
  if (h->path == CTQMC_PATH_GROUPED || (h->path == CTQMC_PATH_AUTO && h->nt != 0 && !h->small)) {
    h->grouped_smem = grouped_smem_bytes(h->dev.dmax);
    if (h->grouped_smem <= smem_max) {
      if (cplx) CU(cudaFuncSetAttribute(grouped_step_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->grouped_smem));
      else      CU(cudaFuncSetAttribute(grouped_step_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->grouped_smem));
      int occ = 0;
      if (cplx) CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, grouped_step_kernel<true>, kGThreads, h->grouped_smem));
      else      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, grouped_step_kernel<false>, kGThreads, h->grouped_smem));
      h->grouped_ctas_per_sm = occ > 0 ? occ : 1;
      h->grouped_ok = 1;
    }
    if (h->path == CTQMC_PATH_GROUPED) {
      if (!h->grouped_ok) return fail(CTQMC_ERR_UNSUPPORTED, "sector dimension %d exceeds the grouped kernel's limit", h->dev.dmax);
      h->grouped = 1;
    }
  }
  h->split = (h->path == CTQMC_PATH_SPLIT);
  if (h->split && !cplx) return fail(CTQMC_ERR_UNSUPPORTED, "the split-precision path is built for complex impurities");
  h->large = (h->nt == 0 || h->path == CTQMC_PATH_LARGE || h->split);
  if (h->large) {
    h->nt = 0;
    h->ldx = (h->dev.dmax + 7) / 8 * 8;
    h->smem_bytes = large_smem_bytes(h->dev.dmax);
    if (h->smem_bytes > smem_max) return fail(CTQMC_ERR_UNSUPPORTED, "sector dimension %d exceeds the large-sector kernel's limit", h->dev.dmax);
    if (const char* e = getenv("CTQMC_LARGE_TMA")) h->use_tma = atoi(e) != 0;
    if (cplx) {
      CU(cudaFuncSetAttribute(large_step_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_bytes));
      CU(cudaFuncSetAttribute(large_step_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_bytes));
    } else {
      CU(cudaFuncSetAttribute(large_step_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_bytes));
      CU(cudaFuncSetAttribute(large_step_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_bytes));
    }
    if (h->use_tma && !h->d_amaps && h->n_blocks > 0) {   // tensor maps of the operator blocks, once
      std::vector<CUtensorMap> maps(h->n_blocks);
      for (int b = 0; b < h->n_blocks; ++b) {
        const BlkDesc& bd = h->h_blks[b];
        int rc = encode_2d(&maps[b], h->d_store + bd.off, (unsigned long long)bd.ld * es, (unsigned long long)((bd.rows + 7) / 8 * 8),
                           (unsigned long long)bd.ld * es * 8, kLBM);
        if (rc) return rc;
      }
      CU(cudaMalloc((void**)&h->d_amaps, maps.size() * sizeof(CUtensorMap)));
      CU(cudaMemcpy(h->d_amaps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice));
    }
    h->grid = 0;
    if (h->split) { int rc = split_prepare(h); if (rc) return rc; }
    return 0;
  }
  KernelFn fn = pick_kernel(cplx, h->nt, h->team_warps);
  CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)h->smem_bytes));
  int occ = 0;
  CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, kCtaThreads, h->smem_bytes));
  if (occ < 1) return fail(CTQMC_ERR_CUDA, "chain kernel does not fit on an SM (smem %zu)", h->smem_bytes);
  h->grid = occ * h->sm_count;
  return 0;
}

long long unit_bound(const ctqmc_impurity* h, int kind, int mode, long long Bs, int Lmax, int S) {
  const long long nS = Bs * h->dev.Q;
  if (mode == 2 || kind == K_TABLES) return nS;
  const long long panels = kind == K_PANEL ? (h->dev.dmax + 8 * h->nt - 1) / (8 * h->nt) : 1;
  if (mode == 0) return nS * panels;
  const long long segs = (S >= Lmax) ? 1 : (long long)Lmax / S + 1;   // ceil(L / S) <= Lmax / S + 1 for every L <= Lmax
  return nS * panels * segs;
}

// Carves one round's scratch out of `base` (nullptr: size computation only) and returns the bytes used.  Every size is an
// upper bound computed from host-known numbers; the kernels learn the actual counts from the device-side counters.
size_t layout_round(const ctqmc_impurity* h, int kind, int mode, long long Bs, int Lmax, int S, long long G, char* base, RoundBuf* rb) {
  Bump bp{base};
  RoundBuf r{};
  const long long Q = h->dev.Q, nS = Bs * Q, nU = unit_bound(h, kind, mode, Bs, Lmax, S);
  const int es = h->dev.cplx ? 2 : 1;
  r.status = bp.take<int>(Bs);
  r.survive = bp.take<uint8_t>(nS);
  r.strings = bp.take<StringRec>(nS);
  r.sector = bp.take<Scaled>(nS);
  r.units = bp.take<int2>(nU);
  r.slots = bp.take<Slot>(nU);
  r.n_units_cap = nU;
  if (kind == K_LARGE) {
    r.G = mode == 1 ? G : nU;
    r.lstride = mode == 1 ? (S < Lmax ? S : Lmax) : Lmax;
    if (r.lstride < 1) r.lstride = 1;
    r.lx_cols = mode == 1 ? 2 * r.G * h->dev.dmax : 2 * Bs * (long long)h->n_energy;
    r.lx = bp.take<double>((size_t)r.lx_cols * h->ldx * es);
    r.plan_blk = bp.take<int>((size_t)r.G * r.lstride);
    r.plan_delta = bp.take<double>((size_t)r.G * r.lstride);
    r.lkmax = bp.take<int>((size_t)r.G * r.lstride);
    r.lunit = bp.take<int>((size_t)4 * r.G);
    r.lux = bp.take<long long>((size_t)r.G);
    if (h->split && mode == 0) {   // int8 slice planes of every unit's carried matrix (split_gemm.cuh)
      r.sp_npad = sp_pad(h->dev.dmax); r.sp_kpad = sp_pad(h->dev.dmax);
      r.sp_eb = bp.take<int>((size_t)r.G * r.sp_npad);
      r.sp_ctr = bp.take<int>(4);
      r.sp_items = bp.take<int>((size_t)r.G * 2 * ((h->dev.dmax + kSpM - 1) / kSpM) * ((h->dev.dmax + kSpN - 1) / kSpN));
      r.sp_b = bp.take<signed char>((size_t)r.G * 3 * h->split_slices * r.sp_npad * r.sp_kpad);
    }
  } else if (kind == K_GROUPED) {
    const int ldx = (h->dev.dmax + 7) / 8 * 8, nb = h->n_blocks;
    const size_t L = (size_t)(Lmax > 0 ? Lmax : 1), nul = (size_t)nU * L;
    r.sum_c_cap = Bs * (long long)h->n_energy;          // every start sector q0 carries at most dim(q0) columns
    r.tile_cap = (int)(r.sum_c_cap / kGBN + (nU < nb ? nU : nb) + 1);
    r.gx = bp.take<double>((size_t)2 * r.sum_c_cap * ldx * es);
    r.gxoff = bp.take<long long>(nU);
    r.gplan_blk = bp.take<int>(nul); r.gplan_delta = bp.take<double>(nul); r.gkmax = bp.take<int>(nul); r.gcoff = bp.take<int>(nul);
    r.gulen = bp.take<int>(nU); r.gucols = bp.take<int>(nU);
    r.gcolcnt = bp.take<int>(L * nb); r.gcolbase = bp.take<int>(L * nb);
    r.gtiles = bp.take<int4>(L * r.tile_cap);
    r.gntiles = bp.take<int>(L); r.gtilecur = bp.take<int>(L);
    r.gcolmap = bp.take<int2>(L * (size_t)r.sum_c_cap);
  }
  if (rb) *rb = r;
  return bp.off + 256;
}

bool round_ok(const ctqmc_impurity* h, int kind, int mode, long long Bs, int Lmax, int S) {
  // int indexing inside the kernels
  const long long nU = unit_bound(h, kind, mode, Bs, Lmax, S);
  if (nU > 2000000000LL) return false;
  if (kind == K_GROUPED && (nU * (long long)(Lmax > 0 ? Lmax : 1) > 2000000000LL || Bs * (long long)h->n_energy > 1000000000LL)) return false;
  if (kind == K_LARGE && mode == 0 && (2 * Bs * (long long)h->n_energy > 2000000000LL || nU > 65535)) return false;   // grid.y
  return true;
}

// Decides how the batch is cut into rounds of `*Bs` configurations (and, large-sector bounds, groups of `*G` units) so that
// one round's scratch fits the arena; grows the arena first when that is allowed.  Everything here is host arithmetic plus,
// at most, one cudaFree / cudaMalloc BEFORE anything of this call is enqueued.  CTQMC_ERR_OOM: not even one configuration fits.
int plan_rounds(ctqmc_impurity* h, int kind, int mode, long long B, int Lmax, int S, long long* Bs_out, long long* G_out) {
  Arena& a = h->arena;
  long long Bs = B;
  while (Bs > 1 && !round_ok(h, kind, mode, Bs, Lmax, S)) Bs = (Bs + 1) / 2;
  if (!round_ok(h, kind, mode, Bs, Lmax, S)) return fail(CTQMC_ERR_ARG, "one configuration exceeds the library's index range (max_len %d)", Lmax);
  const bool var_g = (kind == K_LARGE && mode == 1);
  auto need = [&](long long bs, long long g) { return layout_round(h, kind, mode, bs, Lmax, S, g, nullptr, nullptr); };
  const size_t want = need(Bs, var_g ? unit_bound(h, kind, mode, Bs, Lmax, S) : 0);
  if (want > a.cap && a.fixed_bytes == 0) {
    size_t free_b = 0, total_b = 0;
    CU(cudaMemGetInfo(&free_b, &total_b));
    size_t limit = (size_t)(0.8 * (double)(free_b + a.cap));
    if (h->scratch_limit > 0 && (size_t)h->scratch_limit < limit) limit = (size_t)h->scratch_limit;
    size_t target = want < limit ? want : limit;
    if (target > a.cap) {
      // growing synchronises the device (cudaFree): it happens before this call enqueues anything, and only when a call is
      // larger than every earlier one; a caller that must never stall fixes the size once with CTQMC_OPT_ARENA_BYTES
      target += target / 16;
      if (target > limit) target = limit;
      CU(cudaDeviceSynchronize());
      cudaFree(a.base); a.base = nullptr; a.cap = 0;
      cudaError_t e = cudaMalloc((void**)&a.base, target);
      if (e != cudaSuccess) { cudaGetLastError(); return fail(CTQMC_ERR_OOM, "cannot allocate a scratch arena of %zu bytes", target); }
      a.cap = target;
      CU(cudaMemset(a.base, 0, a.cap));
    }
  }
  if (need(Bs, var_g ? 1 : 0) > a.cap) {   // rounds: largest Bs whose round fits
    long long lo = 0, hi = Bs;             // need(lo) fits (lo = 0: nothing), need(hi) does not
    while (hi - lo > 1) {
      const long long mid = (lo + hi) / 2;
      if (need(mid, var_g ? 1 : 0) <= a.cap) lo = mid; else hi = mid;
    }
    if (lo < 1) return fail(CTQMC_ERR_OOM, "the scratch arena (%zu bytes) cannot hold one configuration of this batch (%zu bytes needed)%s",
                            a.cap, need(1, var_g ? 1 : 0), a.fixed_bytes ? "; raise CTQMC_OPT_ARENA_BYTES" : "");
    Bs = lo;
  }
  long long G = 0;
  if (var_g) {
    const long long nU = unit_bound(h, kind, mode, Bs, Lmax, S);
    const size_t base_need = need(Bs, 1), per = need(Bs, 2) - base_need;
    G = 1 + (long long)((a.cap - base_need) / (per ? per : 1));
    if (G > nU) G = nU;
    if (G > 65535) G = 65535;
    while (G > 1 && need(Bs, G) > a.cap) --G;
  }
  *Bs_out = Bs; *G_out = G;
  return 0;
}

inline void mark(ctqmc_impurity* h, int i, cudaStream_t st) {
  if (h->timing) cudaEventRecord(h->ev[i], st);
}

int check_batch_args(const ctqmc_impurity* h, double beta, const ctqmc_batch* batch) {
  if (!h || !batch) return fail(CTQMC_ERR_ARG, "null impurity or batch");
  if (!(beta > 0.0) || !std::isfinite(beta)) return fail(CTQMC_ERR_ARG, "beta must be positive and finite");
  if (batch->n_configs < 0) return fail(CTQMC_ERR_ARG, "n_configs < 0");
  if (batch->n_configs > 0 && (!batch->offset)) return fail(CTQMC_ERR_ARG, "batch.offset is null");
  if (batch->n_ops < 0) return fail(CTQMC_ERR_ARG, "batch.n_ops < 0");
  if (batch->n_ops > 0 && (!batch->symbol || !batch->tau)) return fail(CTQMC_ERR_ARG, "batch.symbol / batch.tau is null");
  if (batch->max_len < 0) return fail(CTQMC_ERR_ARG, "batch.max_len < 0");
  if (batch->n_configs * (long long)h->dev.Q > 2000000000LL) return fail(CTQMC_ERR_ARG, "n_configs * n_sectors exceeds 2^31");
  return 0;
}

// Longest configuration the step loops are sized for: the caller's max_len, or -- when the caller does not know it -- the
// only bound the host has, n_ops (correct, but one launch per operator of the whole batch: callers should state max_len).
int effective_max_len(const ctqmc_batch* batch) {
  long long m = batch->max_len > 0 ? (long long)batch->max_len : batch->n_ops;
  if (m > batch->n_ops) m = batch->n_ops;
  if (m > 0x3fffffff) m = 0x3fffffff;
  return (int)m;
}

BatchView make_view(const ctqmc_batch* batch, double beta, long long b0, long long Bs, int Lmax) {
  BatchView bv;
  bv.B = Bs; bv.offset = (const long long*)batch->offset + b0; bv.symbol = batch->symbol; bv.tau = batch->tau; bv.beta = beta;
  bv.n_ops = batch->n_ops; bv.max_len = Lmax;
  return bv;
}

// validate -> route -> class scan -> unit scatter; leaves strings / units / counters of the round ready.
int enqueue_routing(ctqmc_impurity* h, const BatchView& bv, const RoundBuf& rb, uint8_t* survive_out, int mode, int segment_len,
                    bool whole_matrix_units, cudaStream_t st) {
  Arena& a = h->arena;
  const long long B = bv.B, nS = B * h->dev.Q;
  CU(cudaMemsetAsync(a.cnt, 0, sizeof(Counters), st));
  validate_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(bv, h->dev.A, rb.status);
  RouteParams rp;
  rp.imp = h->dev; rp.bv = bv; rp.status = rb.status; rp.survive = rb.survive; rp.survive_out = survive_out;
  rp.strings = rb.strings; rp.cnt = a.cnt; rp.W = whole_matrix_units ? (1 << 20) : 8 * h->nt; rp.kstep = h->dev.cplx ? 4 : 8;
  rp.literal = (h->schedule == CTQMC_SCHEDULE_LITERAL); rp.flops_per_mac = h->dev.cplx ? 8 : 2;
  rp.mode = mode; rp.segment_len = segment_len;
  route_kernel<<<(unsigned)((nS + 255) / 256), 256, 0, st>>>(rp);
  h->last_launches += 2;
  if (mode != 2) {
    class_scan_kernel<<<1, 32, 0, st>>>(a.cnt);
    unit_scatter_kernel<<<(unsigned)((nS + 255) / 256), 256, 0, st>>>(rb.strings, nS, a.cnt, rb.units);
    h->last_launches += 2;
  }
  CU(cudaGetLastError());
  return 0;
}

int enqueue_chain(ctqmc_impurity* h, const BatchView& bv, const RoundBuf& rb, int mode, int segment_len, cudaStream_t st) {
  ChainParams cp;
  cp.imp = h->dev; cp.bv = bv; cp.strings = rb.strings; cp.units = rb.units; cp.cnt = h->arena.cnt; cp.slots = rb.slots;
  cp.ldx = h->ldx; cp.mode = mode; cp.segment_len = segment_len;
  KernelFn fn = pick_kernel(h->dev.cplx, h->nt, h->team_warps);
  fn<<<h->grid, kCtaThreads, h->smem_bytes, st>>>(cp);
  h->last_launches += 1;
  CU(cudaGetLastError());
  return 0;
}

// Grouped path (chain_grouped.cuh): schedule for all chain positions, then one persistent GEMM launch per position.  The
// number of units, columns and tiles is known on the device only; buffers and the step loop are sized by host-known bounds
// (configurations x sectors, sum of sector dimensions, max_len), so nothing is read back.
int enqueue_grouped(ctqmc_impurity* h, const BatchView& bv, const RoundBuf& rb, int Lmax, cudaStream_t st) {
  if (Lmax < 1) Lmax = 1;
  const int nb = h->n_blocks;
  const int ldx = (h->dev.dmax + 7) / 8 * 8;
  const long long nU = rb.n_units_cap;
  const size_t nul = (size_t)nU * Lmax;
  GroupedParams gp;
  gp.imp = h->dev; gp.bv = bv; gp.strings = rb.strings; gp.units = rb.units; gp.cnt = h->arena.cnt; gp.Lmax = Lmax; gp.ldx = ldx;
  gp.nb = nb; gp.xtot = rb.sum_c_cap * ldx; gp.X = rb.gx; gp.xoff = rb.gxoff; gp.plan_blk = rb.gplan_blk;
  gp.plan_delta = rb.gplan_delta; gp.kmax = rb.gkmax; gp.coff = rb.gcoff; gp.ulen = rb.gulen;
  gp.ucols = rb.gucols; gp.colcnt = rb.gcolcnt; gp.colbase = rb.gcolbase; gp.tiles = rb.gtiles;
  gp.ntiles = rb.gntiles; gp.tilecur = rb.gtilecur; gp.colmap = rb.gcolmap; gp.tile_cap = rb.tile_cap; gp.col_cap = rb.sum_c_cap; gp.slots = rb.slots;
  CU(cudaMemsetAsync(gp.colcnt, 0, (size_t)Lmax * nb * sizeof(int), st));
  CU(cudaMemsetAsync(gp.tilecur, 0, (size_t)Lmax * sizeof(int), st));
  const unsigned g_ul = (unsigned)((nul + 255) / 256);
  const unsigned g_units = (unsigned)(nU < 4LL * h->sm_count * 8 ? nU : 4LL * h->sm_count * 8);
  grouped_plan_kernel<<<(unsigned)((nU + 127) / 128), 128, 0, st>>>(gp);
  grouped_xoff_kernel<<<1, 1024, 0, st>>>(gp);
  grouped_count_kernel<<<g_ul, 256, 0, st>>>(gp);
  grouped_tiles_kernel<<<Lmax, 32, 0, st>>>(gp);
  grouped_fill_kernel<<<g_ul, 256, 0, st>>>(gp);
  const int MTmax = (h->dev.dmax + kGBM - 1) / kGBM;
  // persistent step grid: as many CTAs as the SMs hold (never more than the item bound); the next position's CTAs start
  // under programmatic stream serialization as this one's run out of items
  long long sg = (long long)h->grouped_ctas_per_sm * h->sm_count;
  const long long item_bound = (long long)rb.tile_cap * MTmax;
  if (sg > item_bound) sg = item_bound;
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3((unsigned)sg); lc.blockDim = dim3(kGThreads); lc.dynamicSmemBytes = h->grouped_smem; lc.stream = st;
  cudaLaunchAttribute lattr[1];
  lattr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  lattr[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = lattr; lc.numAttrs = 1;
  if (h->dev.cplx) {
    grouped_init_kernel<true><<<g_units ? g_units : 1, 128, 0, st>>>(gp);
    for (int j = 0; j < Lmax; ++j) CU(cudaLaunchKernelEx(&lc, grouped_step_kernel<true>, gp, j, MTmax));
    grouped_finish_kernel<true><<<(unsigned)(nU ? nU : 1), 256, 0, st>>>(gp);
  } else {
    grouped_init_kernel<false><<<g_units ? g_units : 1, 128, 0, st>>>(gp);
    for (int j = 0; j < Lmax; ++j) CU(cudaLaunchKernelEx(&lc, grouped_step_kernel<false>, gp, j, MTmax));
    grouped_finish_kernel<false><<<(unsigned)(nU ? nU : 1), 256, 0, st>>>(gp);
  }
  h->last_launches += 7 + Lmax;
  CU(cudaGetLastError());
  return 0;
}

// Large-sector path (chain_large.cuh): one launch per chain position over all unit slots of a group.  Unit slots, the step
// loop and the carried matrices are sized by host-known bounds; idle slots and steps beyond a string's length exit at once.
int enqueue_large(ctqmc_impurity* h, const BatchView& bv, const RoundBuf& rb, int mode, int segment_len, int Lmax, cudaStream_t st) {
  const long long nU = rb.n_units_cap, G = rb.G;
  if (G < 1) return 0;
  const int n_launch = mode == 1 ? rb.lstride : (Lmax > 0 ? Lmax : 0);
  const int es = h->dev.cplx ? 2 : 1;
  LargeParams lp;
  lp.u_q = rb.lunit; lp.u_n = lp.u_q + G; lp.u_c = lp.u_n + G; lp.u_w = lp.u_c + G; lp.u_x = rb.lux; lp.mode = mode; lp.segment_len = segment_len;
  lp.imp = h->dev; lp.bv = bv; lp.strings = rb.strings; lp.units = rb.units; lp.cnt = h->arena.cnt; lp.Lmax = rb.lstride; lp.ldx = h->ldx;
  lp.sum_d = h->n_energy; lp.X = rb.lx; lp.plan_blk = rb.plan_blk; lp.plan_delta = rb.plan_delta; lp.kmax = rb.lkmax; lp.slots = rb.slots;
  lp.amaps = h->d_amaps;
  const bool tma = h->use_tma && h->d_amaps;
  CUtensorMap xmap;
  memset(&xmap, 0, sizeof xmap);
  if (tma) {   // one map over the whole carried-matrix region, passed to the kernel by value: no per-string maps, no copy
    int rc = encode_2d(&xmap, rb.lx, (unsigned long long)h->ldx * es, (unsigned long long)rb.lx_cols, (unsigned long long)h->ldx * es * 8, kLBN);
    if (rc) return rc;
  }
  const int cw = h->dev.dmax;   // widest carried matrix the host can promise
  const int MTmax = (h->dev.dmax + kLBM - 1) / kLBM, NTmax = (cw + kLBN - 1) / kLBN;
  for (long long u0 = 0; u0 < nU; u0 += G) {
    lp.u0 = u0; lp.n_group = (int)((nU - u0 < G) ? (nU - u0) : G);
    large_plan_kernel<<<(lp.n_group + 127) / 128, 128, 0, st>>>(lp);
    dim3 ig((unsigned)((cw < 256) ? cw : 256), (unsigned)lp.n_group);
    dim3 sg((unsigned)(MTmax * NTmax), (unsigned)lp.n_group);
    if (h->split && mode == 0) {
      // split-precision step (split_gemm.cuh): slice the carried matrices, then the int8 tensor-core product
      SplitStepParams sq;
      sq.st.planes = h->d_sp_planes; sq.st.a_off = h->d_sp_aoff; sq.st.ea = h->d_sp_ea; sq.st.ea_off = h->d_sp_eaoff; sq.st.S = h->split_slices;
      sq.bplanes = rb.sp_b; sq.eb = rb.sp_eb; sq.Npad = rb.sp_npad; sq.Kpad = rb.sp_kpad;
      const int Ssl = h->split_slices;
      CU(cudaMemsetAsync(rb.sp_b, 0, (size_t)G * 3 * h->split_slices * rb.sp_npad * rb.sp_kpad, st));
      const int MT8 = (h->dev.dmax + kSpM - 1) / kSpM, NT8 = (cw + kSpN - 1) / kSpN;
      const int tiles_per_unit = MT8 * NT8 * 2;
      const long long total8 = (long long)tiles_per_unit * lp.n_group;
      dim3 xg((unsigned)cw, (unsigned)lp.n_group), gg((unsigned)(total8 < h->sm_count ? total8 : h->sm_count));
      SplitList wl; wl.items = rb.sp_items; wl.ctr = rb.sp_ctr;
      large_init_kernel<true><<<ig, 256, 0, st>>>(lp);
      for (int j = 0; j < n_launch; ++j) {
        split_slice_x_kernel<<<xg, 128, 0, st>>>(lp, sq, j);
        split_list_kernel<<<1, 1024, 0, st>>>(lp, wl, j, tiles_per_unit, NT8, total8);
        pick_split(Ssl)<<<gg, kSpThreads, split_smem(Ssl), st>>>(lp, sq, j, NT8, tiles_per_unit, wl);
      }
      large_finish_kernel<true><<<lp.n_group, 256, 0, st>>>(lp);
      h->last_launches += 2 * n_launch;
    } else if (h->dev.cplx) {
      large_init_kernel<true><<<ig, 256, 0, st>>>(lp);
      for (int j = 0; j < n_launch; ++j) {
        if (tma) large_step_kernel<true, true><<<sg, 256, h->smem_bytes, st>>>(xmap, lp, j, NTmax);
        else     large_step_kernel<true, false><<<sg, 256, h->smem_bytes, st>>>(xmap, lp, j, NTmax);
      }
      large_finish_kernel<true><<<lp.n_group, 256, 0, st>>>(lp);
    } else {
      large_init_kernel<false><<<ig, 256, 0, st>>>(lp);
      for (int j = 0; j < n_launch; ++j) {
        if (tma) large_step_kernel<false, true><<<sg, 256, h->smem_bytes, st>>>(xmap, lp, j, NTmax);
        else     large_step_kernel<false, false><<<sg, 256, h->smem_bytes, st>>>(xmap, lp, j, NTmax);
      }
      large_finish_kernel<false><<<lp.n_group, 256, 0, st>>>(lp);
    }
    h->last_launches += 3 + n_launch;
  }
  CU(cudaGetLastError());
  return 0;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ load / free
extern "C" int ctqmc_load_impurity(const ctqmc_impurity_desc* desc, int device, ctqmc_impurity** out) {
  if (!desc || !out) return fail(CTQMC_ERR_ARG, "null desc or out");
  *out = nullptr;
  const int Q = desc->n_sectors, A = desc->n_symbols;
  if (Q < 1 || A < 1 || !desc->dim || !desc->energy) return fail(CTQMC_ERR_ARG, "need n_sectors >= 1, n_symbols >= 1, dim, energy");
  if (desc->n_blocks < 0 || desc->n_blocks > 65535) return fail(CTQMC_ERR_ARG, "n_blocks out of range [0, 65535]");
  if (desc->n_blocks > 0 && (!desc->blk_symbol || !desc->blk_src || !desc->blk_dst || !desc->blk_offset || !desc->blk_data))
    return fail(CTQMC_ERR_ARG, "null block arrays");
  const int cplx = desc->is_complex ? 1 : 0, es = cplx ? 2 : 1;
  std::vector<int> dim(desc->dim, desc->dim + Q);
  std::vector<long long> eoff(Q);
  long long ne = 0;
  int dmax = 0;
  for (int q = 0; q < Q; ++q) {
    if (dim[q] < 1) return fail(CTQMC_ERR_ARG, "dim[%d] = %d < 1", q, dim[q]);
    eoff[q] = ne; ne += dim[q];
    if (dim[q] > dmax) dmax = dim[q];
  }
  std::vector<double> energy(desc->energy, desc->energy + ne), emin(Q);
  for (int q = 0; q < Q; ++q) {
    double m = INFINITY;
    for (int n = 0; n < dim[q]; ++n) {
      double e = energy[eoff[q] + n];
      if (!std::isfinite(e)) return fail(CTQMC_ERR_ARG, "non-finite eigenvalue in sector %d", q);
      if (e < m) m = e;
    }
    emin[q] = m;
  }
  const int nb = (int)desc->n_blocks;
  std::vector<int> blkof((size_t)A * Q, -1);
  std::vector<BlkDesc> blks(nb);
  std::vector<long long> raw_off(nb), v_off(nb);
  long long store_len = 0, rn_len = 0, v_len = 0, raw_len = 0;
  int max_rows = 1, max_cols = 1;
  for (int b = 0; b < nb; ++b) {
    int a = desc->blk_symbol[b], s = desc->blk_src[b], d = desc->blk_dst[b];
    if (a < 0 || a >= A || s < 0 || s >= Q || d < 0 || d >= Q) return fail(CTQMC_ERR_ARG, "block %d: symbol/src/dst out of range", b);
    if (blkof[(size_t)a * Q + s] != -1) return fail(CTQMC_ERR_ARG, "block %d duplicates (symbol %d, src %d)", b, a, s);
    if (desc->blk_offset[b] < 0) return fail(CTQMC_ERR_ARG, "block %d: negative offset", b);
    blkof[(size_t)a * Q + s] = b;
    BlkDesc& bd = blks[b];
    bd.rows = dim[d]; bd.cols = dim[s]; bd.dst = d; bd.src = s; bd.pad = 0;
    bd.ld = (bd.cols + (cplx ? 3 : 7)) / (cplx ? 4 : 8) * (cplx ? 4 : 8);
    bd.off = store_len;
    bd.rn_off = rn_len;
    const long long rows_pad = (bd.rows + 7) / 8 * 8;
    store_len += rows_pad * bd.ld * es;
    rn_len += rows_pad;
    v_off[b] = v_len; v_len += bd.ld;
    raw_off[b] = desc->blk_offset[b];
    long long end = desc->blk_offset[b] + (long long)bd.rows * bd.cols;
    if (end > raw_len) raw_len = end;
    if (bd.rows > max_rows) max_rows = bd.rows;
    if (bd.cols > max_cols) max_cols = bd.cols;
  }

  // small-sector path: the same blocks, row-major and unpadded (a few KB; lives in shared memory at run time)
  std::vector<double> pack;
  std::vector<int4> pblk(nb);
  const bool small_ok = dmax <= 16 && nb <= 32767 && nb > 0;
  if (small_ok) {
    const double* raw = (const double*)desc->blk_data;
    for (int b = 0; b < nb; ++b) {
      const BlkDesc& bd = blks[b];
      pblk[b] = make_int4((int)(pack.size() / es), bd.rows, bd.cols, bd.dst);
      for (int m = 0; m < bd.rows; ++m)
        for (int k = 0; k < bd.cols; ++k)
          for (int c = 0; c < es; ++c) pack.push_back(raw[((size_t)raw_off[b] + (size_t)k * bd.rows + m) * es + c]);
    }
  }

  std::vector<double> ftpad;
  std::vector<int2> binfo(nb);
  const int dp2 = (small_ok && !cplx) ? small2_dp_for(dmax) : 0;
  if (dp2) {
    const double* raw = (const double*)desc->blk_data;
    ftpad.assign((size_t)nb * dp2 * dp2, 0.0);
    for (int b = 0; b < nb; ++b) {
      const BlkDesc& bd = blks[b];
      binfo[b] = make_int2(bd.dst, (bd.rows << 16) | bd.cols);
      for (int m = 0; m < bd.rows; ++m)
        for (int k = 0; k < bd.cols; ++k)
          ftpad[((size_t)b * dp2 + k) * dp2 + m] = raw[(size_t)raw_off[b] + (size_t)k * bd.rows + m];
    }
  }

  CU(cudaSetDevice(device));
  ctqmc_impurity* h = new (std::nothrow) ctqmc_impurity();
  if (!h) return fail(CTQMC_ERR_OOM, "host allocation failed");
  h->device = device;
  cudaDeviceProp prop;
  cudaError_t pe = cudaGetDeviceProperties(&prop, device);
  if (pe != cudaSuccess) { delete h; return fail(CTQMC_ERR_CUDA, "cudaGetDeviceProperties: %s", cudaGetErrorString(pe)); }
  if (prop.major != 10) { delete h; return fail(CTQMC_ERR_UNSUPPORTED, "device is sm_%d%d; this library is built for sm_100a only", prop.major, prop.minor); }
  h->sm_count = prop.multiProcessorCount;
  h->n_blocks = nb;
  h->h_blks = blks;

  int rc = 0;
  double* d_raw = nullptr; long long* d_rawoff = nullptr; long long* d_voff = nullptr; double* d_v = nullptr; double* d_u = nullptr;
  double* d_w = nullptr; int* d_need = nullptr;
  auto cleanup_tmp = [&]() { cudaFree(d_raw); cudaFree(d_rawoff); cudaFree(d_voff); cudaFree(d_v); cudaFree(d_u); cudaFree(d_w); cudaFree(d_need); };
#define TRY(x) do { rc = (x); if (rc) { cleanup_tmp(); ctqmc_free_impurity(h); return rc; } } while (0)
#define TRYCU(x) do { cudaError_t e_ = (x); if (e_ != cudaSuccess) { rc = fail(e_ == cudaErrorMemoryAllocation ? CTQMC_ERR_OOM : CTQMC_ERR_CUDA, "%s: %s", #x, cudaGetErrorString(e_)); cleanup_tmp(); ctqmc_free_impurity(h); return rc; } } while (0)
  TRY(upload(&h->d_dim, dim));
  TRY(upload(&h->d_eoff, eoff));
  TRY(upload(&h->d_energy, energy));
  TRY(upload(&h->d_emin, emin));
  TRY(upload(&h->d_blkof, blkof));
  TRY(upload(&h->d_blks, blks));
  {
    std::vector<int> order(nb);
    for (int b = 0; b < nb; ++b) order[b] = b;
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) {
      return (long long)blks[x].rows * blks[x].cols > (long long)blks[y].rows * blks[y].cols; });
    TRY(upload(&h->d_blkorder, order));
  }
  TRY(upload(&d_rawoff, raw_off));
  if (small_ok) {
    TRY(upload(&h->d_pack, pack));
    TRY(upload(&h->d_pblk, pblk));
    h->pack_len = (int)(pack.size() / es); h->small_ok = 1;
  }
  if (dp2) {
    TRY(upload(&h->d_ftpad, ftpad));
    TRY(upload(&h->d_binfo, binfo));
    h->small2_dp = dp2;
  }
  h->n_energy = (int)ne;
  {
    std::vector<long long> roff(Q);
    long long acc = 0;
    for (int q = 0; q < Q; ++q) { roff[q] = acc; acc += (long long)dim[q] * dim[q]; }
    h->rho_len = acc;
    TRY(upload(&h->d_rho_off, roff));
  }
  TRY(upload(&d_voff, v_off));
  TRYCU(cudaMalloc((void**)&h->d_store, (size_t)(store_len ? store_len : 1) * sizeof(double)));
  TRYCU(cudaMemset(h->d_store, 0, (size_t)(store_len ? store_len : 1) * sizeof(double)));
  TRYCU(cudaMalloc((void**)&h->d_rownorm2, (size_t)(rn_len ? rn_len : 1) * sizeof(double)));
  TRYCU(cudaMemset(h->d_rownorm2, 0, (size_t)(rn_len ? rn_len : 1) * sizeof(double)));
  TRYCU(cudaMalloc((void**)&h->d_sigma, (size_t)(nb ? nb : 1) * sizeof(double)));
  if (nb > 0) {
    TRYCU(cudaMalloc((void**)&d_raw, (size_t)raw_len * es * sizeof(double)));
    TRYCU(cudaMemcpy(d_raw, desc->blk_data, (size_t)raw_len * es * sizeof(double), cudaMemcpyHostToDevice));
    TRYCU(cudaMalloc((void**)&d_v, (size_t)v_len * es * sizeof(double)));
    TRYCU(cudaMalloc((void**)&d_u, (size_t)rn_len * es * sizeof(double)));
    TRYCU(cudaMalloc((void**)&d_w, (size_t)v_len * es * sizeof(double)));
    TRYCU(cudaMalloc((void**)&d_need, (size_t)nb * sizeof(int)));
    dim3 tb(32, 8), tg((unsigned)std::min((max_cols + 31) / 32, 64), (unsigned)std::min((max_rows + 31) / 32, 64), (unsigned)nb);
    dim3 rg((unsigned)std::min((max_rows + 7) / 8, 512), (unsigned)nb);
    dim3 cg((unsigned)std::min((max_cols + 127) / 128, 64), (unsigned)nb);
    const int iters = 16;
    if (cplx) {
      relayout_kernel<2><<<tg, tb>>>(d_raw, d_rawoff, h->d_blks, h->d_store);
      rownorm_kernel<2><<<rg, 256>>>(h->d_blks, h->d_store, h->d_rownorm2);
      pi_init_kernel<2><<<nb, 128>>>(h->d_blks, d_voff, d_v);
      pi_norm_kernel<<<nb, 256>>>(h->d_blks, d_voff, 0, 2, d_v, 1, nullptr);
      for (int it = 0; it < iters; ++it) {
        pi_fv_kernel<2><<<rg, 256>>>(h->d_blks, h->d_store, d_voff, d_v, d_u);
        pi_fhu_kernel<2><<<cg, 128>>>(h->d_blks, h->d_store, d_voff, d_u, d_v);
        pi_norm_kernel<<<nb, 256>>>(h->d_blks, d_voff, 0, 2, d_v, 1, nullptr);
      }
      pi_fv_kernel<2><<<rg, 256>>>(h->d_blks, h->d_store, d_voff, d_v, d_u);
      pi_norm_kernel<<<nb, 256>>>(h->d_blks, d_voff, 1, 2, d_u, 0, h->d_sigma);
      pi_fhu_kernel<2><<<cg, 128>>>(h->d_blks, h->d_store, d_voff, d_u, d_w);
      sigma_check_kernel<2><<<nb, 256>>>(h->d_blks, d_voff, d_v, d_w, h->d_sigma, d_need);
      sigma_upper_kernel<2><<<nb, 256>>>(h->d_blks, h->d_store, h->d_rownorm2, d_need, h->d_sigma);
    } else {
      relayout_kernel<1><<<tg, tb>>>(d_raw, d_rawoff, h->d_blks, h->d_store);
      rownorm_kernel<1><<<rg, 256>>>(h->d_blks, h->d_store, h->d_rownorm2);
      pi_init_kernel<1><<<nb, 128>>>(h->d_blks, d_voff, d_v);
      pi_norm_kernel<<<nb, 256>>>(h->d_blks, d_voff, 0, 1, d_v, 1, nullptr);
      for (int it = 0; it < iters; ++it) {
        pi_fv_kernel<1><<<rg, 256>>>(h->d_blks, h->d_store, d_voff, d_v, d_u);
        pi_fhu_kernel<1><<<cg, 128>>>(h->d_blks, h->d_store, d_voff, d_u, d_v);
        pi_norm_kernel<<<nb, 256>>>(h->d_blks, d_voff, 0, 1, d_v, 1, nullptr);
      }
      pi_fv_kernel<1><<<rg, 256>>>(h->d_blks, h->d_store, d_voff, d_v, d_u);
      pi_norm_kernel<<<nb, 256>>>(h->d_blks, d_voff, 1, 1, d_u, 0, h->d_sigma);
      pi_fhu_kernel<1><<<cg, 128>>>(h->d_blks, h->d_store, d_voff, d_u, d_w);
      sigma_check_kernel<1><<<nb, 256>>>(h->d_blks, d_voff, d_v, d_w, h->d_sigma, d_need);
      sigma_upper_kernel<1><<<nb, 256>>>(h->d_blks, h->d_store, h->d_rownorm2, d_need, h->d_sigma);
    }
    TRYCU(cudaGetLastError());
    TRYCU(cudaDeviceSynchronize());
  }
  cleanup_tmp();
  d_raw = nullptr; d_rawoff = nullptr; d_voff = nullptr; d_v = nullptr; d_u = nullptr; d_w = nullptr; d_need = nullptr;

  TRYCU(cudaMalloc((void**)&h->arena.cnt, sizeof(Counters)));
  TRYCU(cudaMalloc((void**)&h->arena.cnt_total, sizeof(Counters)));
  TRYCU(cudaMemset(h->arena.cnt, 0, sizeof(Counters)));
  TRYCU(cudaMemset(h->arena.cnt_total, 0, sizeof(Counters)));
  h->dev.Q = Q; h->dev.A = A; h->dev.cplx = cplx; h->dev.dmax = dmax;
  h->dev.dim = h->d_dim; h->dev.e_off = h->d_eoff; h->dev.energy = h->d_energy; h->dev.e_min = h->d_emin;
  h->dev.blk_of = h->d_blkof; h->dev.blks = h->d_blks; h->dev.store = h->d_store; h->dev.rownorm2 = h->d_rownorm2;
  h->dev.sigma = h->d_sigma; h->dev.blk_order = h->d_blkorder;
  TRY(configure(h, 0));
#undef TRY
#undef TRYCU
  *out = h;
  return 0;
}

extern "C" void ctqmc_free_impurity(ctqmc_impurity* h) {
  if (!h) return;
  cudaSetDevice(h->device);
  cudaFree(h->d_dim); cudaFree(h->d_eoff); cudaFree(h->d_energy); cudaFree(h->d_emin); cudaFree(h->d_blkof);
  cudaFree(h->d_ftpad); cudaFree(h->d_binfo);
  cudaFree(h->d_pack); cudaFree(h->d_pblk); cudaFree(h->d_blkorder); cudaFree(h->d_rho_off);
  cudaFree(h->d_sp_planes); cudaFree(h->d_sp_aoff); cudaFree(h->d_sp_ea); cudaFree(h->d_sp_eaoff);
  cudaFree(h->d_blks); cudaFree(h->d_store); cudaFree(h->d_rownorm2); cudaFree(h->d_sigma);
  Arena& a = h->arena;
  cudaFree(a.base); cudaFree(a.cnt); cudaFree(a.cnt_total); cudaFree(h->d_amaps); cudaFree(a.d_stage);
  if (a.h_stage) cudaFreeHost(a.h_stage);
  for (int i = 0; i < 4; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  for (int i = 0; i < 9; ++i) if (h->ev_chunk[i]) cudaEventDestroy(h->ev_chunk[i]);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  delete h;
}

extern "C" int ctqmc_set_option(ctqmc_impurity* h, int option, int64_t value) {
  if (!h) return fail(CTQMC_ERR_ARG, "null impurity");
  CU(cudaSetDevice(h->device));
  if (option == CTQMC_OPT_SCHEDULE) {
    if (value != CTQMC_SCHEDULE_THIN && value != CTQMC_SCHEDULE_LITERAL) return fail(CTQMC_ERR_ARG, "unknown schedule %lld", (long long)value);
    h->schedule = (int)value;
    return 0;
  }
  if (option == CTQMC_OPT_PANEL_WIDTH) {
    if (value != 0 && value != 8 && value != 16 && value != 32) return fail(CTQMC_ERR_ARG, "panel width must be 0, 8, 16 or 32");
    if (h->large) return 0;
    int rc = configure(h, (int)value);
    if (rc || h->large) {   // restore the whole schedule state (configure() touches the small / grouped flags as well)
      std::string msg = g_err;
      configure(h, 0);
      g_err = msg;
      return rc ? rc : fail(CTQMC_ERR_UNSUPPORTED, "panel width %lld does not fit in shared memory for this impurity", (long long)value);
    }
    return 0;
  }
  if (option == CTQMC_OPT_PATH) {
    if (value != CTQMC_PATH_AUTO && value != CTQMC_PATH_PANEL && value != CTQMC_PATH_LARGE && value != CTQMC_PATH_SMALL && value != CTQMC_PATH_GROUPED && value != CTQMC_PATH_SPLIT) return fail(CTQMC_ERR_ARG, "unknown path %lld", (long long)value);
    const int old = h->path;
    h->path = (int)value;
    int rc = configure(h, 0);
    if (rc) { h->path = old; configure(h, 0); }
    return rc;
  }
  if (option == CTQMC_OPT_SCRATCH_LIMIT) {
    if (value < 0) return fail(CTQMC_ERR_ARG, "scratch limit must be >= 0");
    h->scratch_limit = (long long)value;
    Arena& a = h->arena;
    if (value > 0 && a.fixed_bytes == 0 && a.cap > (size_t)value) {   // an arena already larger than the new limit is released
      CU(cudaDeviceSynchronize());
      cudaFree(a.base); a.base = nullptr; a.cap = 0;
    }
    return 0;
  }
  if (option == CTQMC_OPT_SPLIT_SLICES) {
    if (value < 5 || value > kSpMaxSlices) return fail(CTQMC_ERR_ARG, "split slices must be 5 .. %d", kSpMaxSlices);
    if (h->d_sp_planes && value != h->split_slices) return fail(CTQMC_ERR_ARG, "the slice planes are already built with %d slices", h->split_slices);
    h->split_slices = (int)value;
    return 0;
  }
  if (option == CTQMC_OPT_ARENA_BYTES) {
    // pre-allocate the whole scratch arena now; from here on no batch call allocates or frees device memory
    if (value < 0) return fail(CTQMC_ERR_ARG, "arena size must be >= 0");
    Arena& a = h->arena;
    CU(cudaDeviceSynchronize());
    cudaFree(a.base); a.base = nullptr; a.cap = 0; a.fixed_bytes = 0;
    if (value > 0) {
      cudaError_t e = cudaMalloc((void**)&a.base, (size_t)value);
      if (e != cudaSuccess) { cudaGetLastError(); return fail(CTQMC_ERR_OOM, "cannot allocate a scratch arena of %lld bytes", (long long)value); }
      a.cap = (size_t)value; a.fixed_bytes = (size_t)value;
      CU(cudaMemset(a.base, 0, a.cap));
    }
    return 0;
  }
  if (option == CTQMC_OPT_TIMING) {
    if (value && !h->ev[0])
      for (int i = 0; i < 4; ++i) CU(cudaEventCreate(&h->ev[i]));
    h->timing = value ? 1 : 0;
    h->timing_valid = 0;
    return 0;
  }
  return fail(CTQMC_ERR_ARG, "unknown option %d", option);
}

namespace {

// One round of ctqmc_trace_batch on a sub-batch (panel / grouped / large kernel families).
int trace_round(ctqmc_impurity* h, int kind, const BatchView& bv, const RoundBuf& rb, int Lmax, double* mant, int64_t* exp2,
                uint8_t* survive, int32_t* status, cudaStream_t st) {
  mark(h, 0, st);
  int rc = enqueue_routing(h, bv, rb, survive, 0, 0, kind != K_PANEL, st);
  if (rc) return rc;
  mark(h, 1, st);
  rc = kind == K_GROUPED ? enqueue_grouped(h, bv, rb, Lmax, st) : kind == K_LARGE ? enqueue_large(h, bv, rb, 0, 0, Lmax, st)
                                                                                 : enqueue_chain(h, bv, rb, 0, 0, st);
  if (rc) return rc;
  mark(h, 2, st);
  TraceReduceParams tp;
  tp.B = bv.B; tp.Q = h->dev.Q; tp.status_in = rb.status; tp.survive = rb.survive; tp.strings = rb.strings;
  tp.slots = rb.slots; tp.mant = mant; tp.exp2 = (long long*)exp2; tp.status = status;
  trace_reduce_kernel<<<(unsigned)((bv.B + 127) / 128), 128, 0, st>>>(tp);
  accumulate_counters_kernel<<<1, 1, 0, st>>>(h->arena.cnt, h->arena.cnt_total);
  h->last_launches += 2;
  mark(h, 3, st);
  CU(cudaGetLastError());
  return 0;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ batch calls
extern "C" int ctqmc_trace_batch(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, double* mant, int64_t* exp2,
                                 uint8_t* survive, int32_t* status, void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!mant || !exp2 || !status) return fail(CTQMC_ERR_ARG, "null output (mant, exp2 and status are required)");
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int Lmax = effective_max_len(batch);
  // AUTO: batches of at least kGroupedMinBatch configurations take the step-synchronous grouped path (one launch per chain
  // position pays off once many strings share blocks); smaller ones the persistent panel kernel
  h->grouped_now = h->grouped || (h->path == CTQMC_PATH_AUTO && h->grouped_ok && !h->small && !h->large && B >= kGroupedMinBatch);
  h->last_path = h->small ? CTQMC_PATH_SMALL : h->grouped_now ? CTQMC_PATH_GROUPED : h->split ? CTQMC_PATH_SPLIT : h->large ? CTQMC_PATH_LARGE : CTQMC_PATH_PANEL;
  h->last_stream = st;
  if (!h->keep_totals) { h->last_launches = 0; CU(cudaMemsetAsync(h->arena.cnt_total, 0, sizeof(Counters), st)); }
  h->timing_valid = 0;
  if (h->small) {
    // everything (validation, routing, chain, trace, sector sum) in one launch: chain_small.cuh
    Arena& a = h->arena;
    const BatchView bv = make_view(batch, beta, 0, B, Lmax);
    mark(h, 0, st);
    mark(h, 1, st);
    SmallParams sp;   // the one launch adds its counters straight into the call's totals (zeroed above)
    sp.imp = h->dev; sp.bv = bv; sp.pack = h->d_pack; sp.pblk = h->d_pblk; sp.n_blocks = h->n_blocks; sp.pack_len = h->pack_len;
    sp.n_energy = h->n_energy; sp.literal = (h->schedule == CTQMC_SCHEDULE_LITERAL); sp.mant = mant; sp.exp2 = (long long*)exp2;
    sp.survive = survive; sp.status = status; sp.cnt = a.cnt_total; sp.dmax = h->dev.dmax;
    if (h->small2) {
      Small2Params s2;
      s2.imp = h->dev; s2.bv = bv; s2.ftpad = h->d_ftpad; s2.binfo = h->d_binfo; s2.n_blocks = h->n_blocks; s2.literal = sp.literal;
      s2.mant = mant; s2.exp2 = (long long*)exp2; s2.survive = survive; s2.status = status; s2.cnt = a.cnt_total;
      // CTA size: small batches are latency-bound, so they are spread over all SMs in ONE wave: warps per CTA =
      // ceil(configurations per SM / configurations per warp), at most the configured maximum
      // small batches: one WARP per configuration (its groups share the start sectors) while every configuration still gets a
      // resident warp of its own (with two rounds of warps the gain is gone: measured on config 2 at 4096, 0.273 against 0.227 ms)
      const int max_warps = h->small2_threads / 32;
      s2.split = (32 / h->small2_dp > 1 && B <= (long long)h->sm_count * max_warps) ? 1 : 0;
      const int gpw = s2.split ? 1 : 32 / h->small2_dp;
      long long per_sm = (B + h->sm_count - 1) / h->sm_count;
      int warps = (int)((per_sm + gpw - 1) / gpw);
      if (warps < 2) warps = 2;
      if (warps > max_warps) warps = max_warps;
      const int threads = 32 * warps;
      const long long gpc = (long long)warps * gpw;
      const size_t smem = small2_common_bytes(h->dev.Q, h->dev.A, h->n_blocks, h->small2_dp) +
                          (s2.split ? (size_t)warps * small2_warp_bytes(h->dev.Q, h->small2_dp)
                                    : (size_t)warps * (32 / h->small2_dp) * small2_group_bytes(h->dev.Q, h->small2_dp));
      if (h->small2_occ[warps] == 0) {
        int occ = 0;
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, pick_small2(h->small2_dp), threads, smem));
        h->small2_occ[warps] = occ > 0 ? occ : 1;
      }
      long long grid = (B + gpc - 1) / gpc;
      const long long grid_max = (long long)h->small2_occ[warps] * h->sm_count;
      if (grid > grid_max) grid = grid_max;
      pick_small2(h->small2_dp)<<<(unsigned)grid, threads, smem, st>>>(s2);
    } else {
      const long long gpc = kCtaThreads / h->small_g;
      long long grid = (B + gpc - 1) / gpc;
      if (grid > h->small_grid_max) grid = h->small_grid_max;
      pick_small(h->dev.cplx, h->small_g)<<<(unsigned)grid, kCtaThreads, h->small_smem, st>>>(sp);
    }
    h->last_launches += 1;
    mark(h, 2, st);
    mark(h, 3, st);
    h->timing_valid = h->timing;
    CU(cudaGetLastError());
    return 0;
  }
  int kind = h->grouped_now ? K_GROUPED : h->large ? K_LARGE : K_PANEL;
  long long Bs = 0, G = 0;
  rc = plan_rounds(h, kind, 0, B, Lmax, 0, &Bs, &G);
  if (rc == CTQMC_ERR_OOM && kind == K_GROUPED && h->path == CTQMC_PATH_AUTO) {
    // the grouped path's schedule (one column map per chain position) does not fit: AUTO falls back to the persistent panel
    // kernel, which needs no per-position scratch
    h->grouped_now = 0; h->last_path = CTQMC_PATH_PANEL; kind = K_PANEL;
    rc = plan_rounds(h, kind, 0, B, Lmax, 0, &Bs, &G);
  }
  if (rc) return rc;
  for (long long b0 = 0; b0 < B; b0 += Bs) {
    const long long bs = (B - b0 < Bs) ? (B - b0) : Bs;
    RoundBuf rb;
    layout_round(h, kind, 0, bs, Lmax, 0, G, h->arena.base, &rb);
    const BatchView bv = make_view(batch, beta, b0, bs, Lmax);
    rc = trace_round(h, kind, bv, rb, Lmax, mant + 2 * b0, exp2 + b0, survive ? survive + b0 * h->dev.Q : nullptr, status + b0, st);
    if (rc) return rc;
  }
  h->timing_valid = h->timing;
  return 0;
}

extern "C" int ctqmc_bound_batch(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, int norm_kind, int segment_len,
                                 double* bound_mant, int64_t* bound_exp2, double* sector_bound_mant,
                                 int64_t* sector_bound_exp2, int32_t* status, void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  if (norm_kind != 0 && norm_kind != 1) return fail(CTQMC_ERR_ARG, "norm_kind must be 0 (Frobenius) or 1 (spectral)");
  if (segment_len < 0) return fail(CTQMC_ERR_ARG, "segment_len < 0");
  if ((sector_bound_mant == nullptr) != (sector_bound_exp2 == nullptr)) return fail(CTQMC_ERR_ARG, "sector_bound_mant / _exp2 must both be given or both be null");
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!bound_mant || !bound_exp2 || !status) return fail(CTQMC_ERR_ARG, "null output");
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int Lmax = effective_max_len(batch);
  const int W = h->large ? (1 << 20) : 8 * h->nt;
  const long long Q = h->dev.Q;
  h->last_stream = st; h->last_launches = 0;
  CU(cudaMemsetAsync(h->arena.cnt_total, 0, sizeof(Counters), st));
  h->timing_valid = 0;
  h->grouped_now = 0; h->last_path = h->large ? CTQMC_PATH_LARGE : CTQMC_PATH_PANEL;
  if (segment_len == 1 && h->small2) {
    // small real impurities: validation, routing, norm products and the sector sum in one launch (bound_small2.cuh)
    const BatchView bv = make_view(batch, beta, 0, B, Lmax);
    const int dp = h->small2_dp, gpw = 32 / dp;
    long long per_sm = (B + h->sm_count - 1) / h->sm_count;
    int warps = (int)((per_sm + gpw - 1) / gpw);
    if (warps < 2) warps = 2;
    if (warps > 16) warps = 16;
    const long long gpc = (long long)warps * gpw;
    const size_t smem = small2b_common_bytes(h->dev.Q, h->dev.A, h->n_blocks, dp) + (size_t)gpc * small2b_group_bytes(h->dev.Q, dp);
    Small2BoundFn fn = pick_small2_bound(dp);
    if (fn && smem <= 227 * 1024 - 2048) {
      CU(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      Small2BoundParams sb;
      sb.imp = h->dev; sb.bv = bv; sb.binfo = h->d_binfo; sb.n_blocks = h->n_blocks; sb.norm_kind = norm_kind;
      sb.bound_mant = bound_mant; sb.bound_exp2 = (long long*)bound_exp2; sb.sector_mant = sector_bound_mant;
      sb.sector_exp2 = (long long*)sector_bound_exp2; sb.status = status;
      long long grid = (B + gpc - 1) / gpc;
      if (grid > 8LL * h->sm_count) grid = 8LL * h->sm_count;
      mark(h, 0, st); mark(h, 1, st);
      fn<<<(unsigned)grid, 32 * warps, smem, st>>>(sb);
      h->last_launches += 1; h->last_path = CTQMC_PATH_SMALL;
      mark(h, 2, st); mark(h, 3, st);
      h->timing_valid = h->timing;
      CU(cudaGetLastError());
      return 0;
    }
  }
  // segment_len 1: norms come from the load-time tables; otherwise the chain kernels multiply every segment.  The number of
  // segments per string is bounded on the host by max_len / S + 1, so nothing is read back from the device.
  const int mode = segment_len == 1 ? 2 : 1;
  const int S = segment_len == 0 ? (1 << 30) : segment_len;
  const int kind = mode == 2 ? K_TABLES : h->large ? K_LARGE : K_PANEL;
  long long Bs = 0, G = 0;
  rc = plan_rounds(h, kind, mode, B, Lmax, S, &Bs, &G);
  if (rc) return rc;
  for (long long b0 = 0; b0 < B; b0 += Bs) {
    const long long bs = (B - b0 < Bs) ? (B - b0) : Bs, nS = bs * Q;
    RoundBuf rb;
    layout_round(h, kind, mode, bs, Lmax, S, G, h->arena.base, &rb);
    const BatchView bv = make_view(batch, beta, b0, bs, Lmax);
    BoundParams bp;
    mark(h, 0, st);
    rc = enqueue_routing(h, bv, rb, nullptr, mode, mode == 2 ? 1 : S, h->large, st);
    if (rc) return rc;
    mark(h, 1, st);
    bp.imp = h->dev; bp.bv = bv; bp.survive = rb.survive; bp.strings = rb.strings; bp.slots = rb.slots;
    bp.sector = rb.sector; bp.W = W;
    if (mode == 2) {
      bp.norm_kind = norm_kind; bp.segment_len = 1;
      bound_s1_kernel<<<(unsigned)((nS * 32 + 255) / 256), 256, 0, st>>>(bp);
    } else {
      rc = h->large ? enqueue_large(h, bv, rb, 1, S, Lmax, st) : enqueue_chain(h, bv, rb, 1, S, st);
      if (rc) return rc;
      bp.norm_kind = norm_kind; bp.segment_len = S;
      bound_segments_kernel<<<(unsigned)((nS + 127) / 128), 128, 0, st>>>(bp);
    }
    mark(h, 2, st);
    BoundReduceParams rp;
    rp.B = bs; rp.Q = h->dev.Q; rp.status_in = rb.status; rp.survive = rb.survive; rp.sector = rb.sector;
    rp.bound_mant = bound_mant + b0; rp.bound_exp2 = (long long*)bound_exp2 + b0;
    rp.sector_mant = sector_bound_mant ? sector_bound_mant + b0 * Q : nullptr;
    rp.sector_exp2 = sector_bound_exp2 ? (long long*)sector_bound_exp2 + b0 * Q : nullptr; rp.status = status + b0;
    bound_reduce_kernel<<<(unsigned)((bs + 127) / 128), 128, 0, st>>>(rp);
    accumulate_counters_kernel<<<1, 1, 0, st>>>(h->arena.cnt, h->arena.cnt_total);
    h->last_launches += 3;
    mark(h, 3, st);
    CU(cudaGetLastError());
  }
  h->timing_valid = h->timing;
  return 0;
}

// ------------------------------------------------------------------------------------------------ host-buffer forms
namespace {

struct Staged {
  ctqmc_batch dev_batch;
  char* d_out = nullptr;   // device outputs region
  char* h_out = nullptr;   // pinned mirror
};

size_t align_up(size_t x) { return (x + 255) / 256 * 256; }

// Host forms: the offsets are host memory, so the library derives n_ops and max_len itself (and rejects offsets that would
// make it read outside the caller's symbol / tau arrays before anything is copied).
int host_batch_shape(const ctqmc_batch* hb, long long* n_ops, int* max_len) {
  const long long B = hb->n_configs;
  if (!hb->offset) return fail(CTQMC_ERR_ARG, "batch.offset is null");
  if (hb->offset[0] != 0) return fail(CTQMC_ERR_ARG, "batch.offset[0] must be 0");
  long long mx = 0;
  for (long long b = 0; b < B; ++b) {
    const long long l = hb->offset[b + 1] - hb->offset[b];
    if (l < 0) return fail(CTQMC_ERR_ARG, "batch.offset is decreasing at configuration %lld", b);
    if (l > mx) mx = l;
  }
  if (mx > 0x3fffffff) return fail(CTQMC_ERR_ARG, "configuration longer than 2^30 operators");
  *n_ops = hb->offset[B]; *max_len = (int)mx;
  if (hb->n_ops != 0 && hb->n_ops < *n_ops) return fail(CTQMC_ERR_ARG, "batch.n_ops (%lld) < offset[B] (%lld)", (long long)hb->n_ops, *n_ops);
  if (*n_ops > 0 && (!hb->symbol || !hb->tau)) return fail(CTQMC_ERR_ARG, "null symbol / tau");
  return 0;
}

int stage_in(ctqmc_impurity* h, const ctqmc_batch* hb, size_t out_bytes, Staged* sg, cudaStream_t st) {
  const long long B = hb->n_configs;
  long long n_ops = 0; int max_len = 0;
  { int rc = host_batch_shape(hb, &n_ops, &max_len); if (rc) return rc; }
  const size_t b_off = align_up((size_t)(B + 1) * 8), b_sym = align_up((size_t)n_ops * 4), b_tau = align_up((size_t)n_ops * 8);
  const size_t total = b_off + b_sym + b_tau + align_up(out_bytes);
  Arena& a = h->arena;
  if (total > a.d_stage_bytes) {
    cudaFree(a.d_stage); a.d_stage = nullptr; a.d_stage_bytes = 0;
    if (a.h_stage) cudaFreeHost(a.h_stage);
    a.h_stage = nullptr; a.h_stage_bytes = 0;
    CU(cudaMalloc(&a.d_stage, total));
    CU(cudaMallocHost(&a.h_stage, total));
    a.d_stage_bytes = total; a.h_stage_bytes = total;
  }
  char* hs = (char*)a.h_stage; char* ds = (char*)a.d_stage;
  memcpy(hs, hb->offset, (size_t)(B + 1) * 8);
  if (n_ops) { memcpy(hs + b_off, hb->symbol, (size_t)n_ops * 4); memcpy(hs + b_off + b_sym, hb->tau, (size_t)n_ops * 8); }
  CU(cudaMemcpyAsync(ds, hs, b_off + b_sym + b_tau, cudaMemcpyHostToDevice, st));
  sg->dev_batch.n_configs = B;
  sg->dev_batch.n_ops = n_ops; sg->dev_batch.max_len = max_len;
  sg->dev_batch.offset = (const int64_t*)ds;
  sg->dev_batch.symbol = (const int32_t*)(ds + b_off);
  sg->dev_batch.tau = (const double*)(ds + b_off + b_sym);
  sg->d_out = ds + b_off + b_sym + b_tau;
  sg->h_out = hs + b_off + b_sym + b_tau;
  return 0;
}

bool is_pinned(const void* p) {
  if (!p) return false;
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeHost;
}

// Host form, fast path: the caller's buffers are page-locked, so the library copies straight from / to them (no staging
// memcpy), and -- on the single-launch small-sector path -- cuts the batch into chunks whose host-to-device copies run on a
// second stream while the previous chunk's kernel runs.
int trace_host_pinned(ctqmc_impurity* h, double beta, const ctqmc_batch* hb, double* mant, int64_t* exp2, uint8_t* survive,
                      int32_t* status, cudaStream_t st) {
  const long long B = hb->n_configs;
  long long n_ops = 0; int max_len = 0;
  { int rc = host_batch_shape(hb, &n_ops, &max_len); if (rc) return rc; }
  const size_t Q = h->dev.Q;
  const size_t b_off = align_up((size_t)(B + 1) * 8), b_sym = align_up((size_t)n_ops * 4), b_tau = align_up((size_t)n_ops * 8);
  const size_t o_mant = 0, o_exp = align_up(B * 16), o_stat = o_exp + align_up(B * 8), o_surv = o_stat + align_up(B * 4);
  const size_t out_bytes = o_surv + align_up(B * Q);
  const size_t total = b_off + b_sym + b_tau + out_bytes;
  Arena& a = h->arena;
  if (total > a.d_stage_bytes) {
    cudaFree(a.d_stage); a.d_stage = nullptr; a.d_stage_bytes = 0;
    if (a.h_stage) cudaFreeHost(a.h_stage);
    a.h_stage = nullptr; a.h_stage_bytes = 0;
    CU(cudaMalloc(&a.d_stage, total));
    CU(cudaMallocHost(&a.h_stage, total));
    a.d_stage_bytes = total; a.h_stage_bytes = total;
  }
  char* ds = (char*)a.d_stage;
  long long* d_off = (long long*)ds;
  int* d_sym = (int*)(ds + b_off);
  double* d_tau = (double*)(ds + b_off + b_sym);
  char* d_out = ds + b_off + b_sym + b_tau;
  // chunking pays only when the kernel is throughput-bound; below ~3e4 configurations its duration is one configuration's
  // dependency chain whatever the batch size, and chunks would just serialise that latency
  const int n_chunk = (h->small && B >= 32768) ? 4 : 1;
  if (n_chunk > 1 && !h->copy_stream) {
    CU(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < 9; ++i) CU(cudaEventCreateWithFlags(&h->ev_chunk[i], cudaEventDisableTiming));
  }
  cudaStream_t cs = n_chunk > 1 ? h->copy_stream : st;
  if (n_chunk > 1) {   // the copy stream starts after everything already enqueued on the caller's stream
    CU(cudaEventRecord(h->ev_chunk[8], st));
    CU(cudaStreamWaitEvent(cs, h->ev_chunk[8], 0));
  }
  for (int k = 0; k < n_chunk; ++k) {
    const long long b0 = B * k / n_chunk, b1 = B * (k + 1) / n_chunk;
    const long long p0 = hb->offset[b0], p1 = hb->offset[b1];
    CU(cudaMemcpyAsync(d_off + b0, hb->offset + b0, (size_t)(b1 - b0 + 1) * 8, cudaMemcpyHostToDevice, cs));
    if (p1 > p0) {
      CU(cudaMemcpyAsync(d_sym + p0, hb->symbol + p0, (size_t)(p1 - p0) * 4, cudaMemcpyHostToDevice, cs));
      CU(cudaMemcpyAsync(d_tau + p0, hb->tau + p0, (size_t)(p1 - p0) * 8, cudaMemcpyHostToDevice, cs));
    }
    if (n_chunk > 1) {
      CU(cudaEventRecord(h->ev_chunk[k], cs));
      CU(cudaStreamWaitEvent(st, h->ev_chunk[k], 0));
    }
    ctqmc_batch sub;
    sub.n_configs = b1 - b0; sub.offset = (const int64_t*)(d_off + b0); sub.symbol = d_sym; sub.tau = d_tau;
    sub.n_ops = n_ops; sub.max_len = max_len;
    h->keep_totals = k > 0;   // ctqmc_last_stats reports the whole batch, not the last chunk
    int rc = ctqmc_trace_batch(h, beta, &sub, (double*)(d_out + o_mant) + 2 * b0, (int64_t*)(d_out + o_exp) + b0,
                               survive ? (uint8_t*)(d_out + o_surv) + b0 * Q : nullptr, (int32_t*)(d_out + o_stat) + b0, st);
    h->keep_totals = 0;
    if (rc) return rc;
  }
  CU(cudaMemcpyAsync(mant, d_out + o_mant, B * 16, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(exp2, d_out + o_exp, B * 8, cudaMemcpyDeviceToHost, st));
  CU(cudaMemcpyAsync(status, d_out + o_stat, B * 4, cudaMemcpyDeviceToHost, st));
  if (survive) CU(cudaMemcpyAsync(survive, d_out + o_surv, B * Q, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  return 0;
}

}  // namespace

extern "C" int ctqmc_trace_batch_host(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, double* mant, int64_t* exp2,
                                      uint8_t* survive, int32_t* status, void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!mant || !exp2 || !status) return fail(CTQMC_ERR_ARG, "null output (mant, exp2 and status are required)");
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t Q = h->dev.Q;
  if (batch->offset && is_pinned(batch->offset) && (batch->offset[B] == 0 || (is_pinned(batch->symbol) && is_pinned(batch->tau))) &&
      is_pinned(mant) && is_pinned(exp2) && is_pinned(status) && (!survive || is_pinned(survive)))
    return trace_host_pinned(h, beta, batch, mant, exp2, survive, status, st);
  const size_t o_mant = 0, o_exp = align_up(B * 16), o_stat = o_exp + align_up(B * 8), o_surv = o_stat + align_up(B * 4);
  const size_t out_bytes = o_surv + align_up(B * Q);
  Staged sg;
  rc = stage_in(h, batch, out_bytes, &sg, st);
  if (rc) return rc;
  rc = ctqmc_trace_batch(h, beta, &sg.dev_batch, (double*)(sg.d_out + o_mant), (int64_t*)(sg.d_out + o_exp),
                         survive ? (uint8_t*)(sg.d_out + o_surv) : nullptr, (int32_t*)(sg.d_out + o_stat), cuda_stream);
  if (rc) return rc;
  CU(cudaMemcpyAsync(sg.h_out, sg.d_out, survive ? out_bytes : o_surv, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  memcpy(mant, sg.h_out + o_mant, B * 16);
  memcpy(exp2, sg.h_out + o_exp, B * 8);
  memcpy(status, sg.h_out + o_stat, B * 4);
  if (survive) memcpy(survive, sg.h_out + o_surv, B * Q);
  return 0;
}

extern "C" int ctqmc_bound_batch_host(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, int norm_kind, int segment_len,
                                      double* bound_mant, int64_t* bound_exp2, double* sector_bound_mant,
                                      int64_t* sector_bound_exp2, int32_t* status, void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!bound_mant || !bound_exp2 || !status) return fail(CTQMC_ERR_ARG, "null output");
  if ((sector_bound_mant == nullptr) != (sector_bound_exp2 == nullptr)) return fail(CTQMC_ERR_ARG, "sector_bound_mant / _exp2 must both be given or both be null");
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t Q = h->dev.Q;
  const bool sec = sector_bound_mant != nullptr;
  const size_t o_m = 0, o_e = align_up(B * 8), o_stat = o_e + align_up(B * 8), o_sm = o_stat + align_up(B * 4),
               o_se = o_sm + align_up(B * Q * 8);
  const size_t out_bytes = o_se + align_up(B * Q * 8);
  Staged sg;
  rc = stage_in(h, batch, out_bytes, &sg, st);
  if (rc) return rc;
  rc = ctqmc_bound_batch(h, beta, &sg.dev_batch, norm_kind, segment_len, (double*)(sg.d_out + o_m), (int64_t*)(sg.d_out + o_e),
                         sec ? (double*)(sg.d_out + o_sm) : nullptr, sec ? (int64_t*)(sg.d_out + o_se) : nullptr,
                         (int32_t*)(sg.d_out + o_stat), cuda_stream);
  if (rc) return rc;
  CU(cudaMemcpyAsync(sg.h_out, sg.d_out, sec ? out_bytes : o_sm, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  memcpy(bound_mant, sg.h_out + o_m, B * 8);
  memcpy(bound_exp2, sg.h_out + o_e, B * 8);
  memcpy(status, sg.h_out + o_stat, B * 4);
  if (sec) { memcpy(sector_bound_mant, sg.h_out + o_sm, B * Q * 8); memcpy(sector_bound_exp2, sg.h_out + o_se, B * Q * 8); }
  return 0;
}

extern "C" int ctqmc_last_stats(ctqmc_impurity* h, int64_t stats[10]) {
  if (!h || !stats) return fail(CTQMC_ERR_ARG, "null argument");
  for (int i = 0; i < 10; ++i) stats[i] = 0;
  stats[5] = h->small ? (h->small2 ? h->small2_dp : h->small_g) : h->nt * 8; stats[6] = h->team_warps; stats[7] = h->last_path ? h->last_path : (h->small ? 3 : h->grouped ? 4 : h->large ? 2 : 1);
  stats[9] = (int64_t)h->arena.cap;
  if (!h->arena.cnt_total) return 0;
  CU(cudaSetDevice(h->device));
  Counters c;
  CU(cudaStreamSynchronize(h->last_stream));
  CU(cudaMemcpy(&c, h->arena.cnt_total, sizeof c, cudaMemcpyDeviceToHost));
  stats[0] = (int64_t)c.n_strings; stats[1] = (int64_t)c.n_slots; stats[2] = h->last_launches;
  stats[3] = (int64_t)c.macs; stats[4] = (int64_t)c.alg_flops; stats[8] = (int64_t)c.n_exp;
  return 0;
}

extern "C" int ctqmc_last_timing(ctqmc_impurity* h, double ms[4]) {
  if (!h || !ms) return fail(CTQMC_ERR_ARG, "null argument");
  if (!h->timing_valid) return fail(CTQMC_ERR_ARG, "no timed batch call on this handle (set CTQMC_OPT_TIMING first)");
  CU(cudaSetDevice(h->device));
  CU(cudaEventSynchronize(h->ev[3]));
  for (int i = 0; i < 3; ++i) {
    float f = 0.f;
    CU(cudaEventElapsedTime(&f, h->ev[i], h->ev[i + 1]));
    ms[i] = f;
  }
  float f = 0.f;
  CU(cudaEventElapsedTime(&f, h->ev[0], h->ev[3]));
  ms[3] = f;
  return 0;
}

extern "C" int ctqmc_measure_fp64_peak(int device, double* tflops_dmma, double* tflops_dfma) {
  if (!tflops_dmma || !tflops_dfma) return fail(CTQMC_ERR_ARG, "null output");
  CU(cudaSetDevice(device));
  cudaDeviceProp prop;
  CU(cudaGetDeviceProperties(&prop, device));
  double* sink = nullptr;
  CU(cudaMalloc((void**)&sink, 8));
  cudaEvent_t e0, e1;
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  const int grid = prop.multiProcessorCount * 2, iters = 1 << 16;
  double best[2] = {0.0, 0.0};
  for (int which = 0; which < 2; ++which)
    for (int rep = 0; rep < 4; ++rep) {
      CU(cudaEventRecord(e0));
      if (which == 0) peak_dmma_kernel<<<grid, 256>>>(iters, sink); else peak_dfma_kernel<<<grid, 256>>>(iters, sink);
      CU(cudaEventRecord(e1));
      CU(cudaEventSynchronize(e1));
      float ms = 0.f;
      CU(cudaEventElapsedTime(&ms, e0, e1));
      // DMMA.8x8x4 = 256 FMA per warp instruction, 8 per iteration; DFMA: 32 lanes x 16 per iteration
      const double flop = (double)grid * 8 * iters * (which == 0 ? 8.0 * 256 * 2 : 16.0 * 32 * 2);
      const double tf = flop / (ms * 1e-3) / 1e12;
      if (rep > 0 && tf > best[which]) best[which] = tf;
    }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  CU(cudaGetLastError());
  *tflops_dmma = best[0]; *tflops_dfma = best[1];
  return 0;
}

extern "C" const char* ctqmc_last_error(void) { return g_err.c_str(); }

#include "lazy_api.cuh"
#include "density_api.cuh"
#include "density_static_api.cuh"
