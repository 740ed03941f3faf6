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

struct DevBuf {   // grow-only device buffer
  void* p = nullptr;
  size_t cap = 0;
  bool grew = false;
};

struct Arena {
  long long cap_strings = 0, cap_units = 0, cap_configs = 0;
  int* status = nullptr;
  uint8_t* survive = nullptr;
  StringRec* strings = nullptr;
  int2* units = nullptr;
  Slot* slots = nullptr;
  Scaled* sector = nullptr;
  Counters* cnt = nullptr;
  // large-sector path: carried matrices (two per string), step plan, per-step largest exponents
  double* lx = nullptr; size_t lx_bytes = 0;
  int* plan_blk = nullptr; double* plan_delta = nullptr; int* lkmax = nullptr; size_t plan_cap = 0;
  DevBuf lunit;   // u_q, u_n, u_c
  DevBuf xmaps; const void* xmaps_base = nullptr; long long xmaps_g = 0, xmaps_slab = 0; int xmaps_cmax = 0;
  // grouped path
  DevBuf gx, gxoff, gplan_blk, gplan_delta, gkmax, gcoff, gulen, gucols, gcolcnt, gcolbase, gtiles, gntiles, gcolmap;
  // host-variant staging
  void* h_stage = nullptr; size_t h_stage_bytes = 0;
  void* d_stage = nullptr; size_t d_stage_bytes = 0;
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
  size_t smem_bytes = 0;
  int grid = 0;
  Arena arena;
  cudaStream_t last_stream = nullptr;
  long long last_launches = 0;
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
  for (int i = 0; i < 3 && h->path != CTQMC_PATH_LARGE; ++i) {
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
      h->grouped_ok = 1;
    }
    if (h->path == CTQMC_PATH_GROUPED) {
      if (!h->grouped_ok) return fail(CTQMC_ERR_UNSUPPORTED, "sector dimension %d exceeds the grouped kernel's limit", h->dev.dmax);
      h->grouped = 1;
    }
  }
  h->large = (h->nt == 0 || h->path == CTQMC_PATH_LARGE);
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

int ensure_arena(ctqmc_impurity* h, long long B, long long units_per_string) {
  Arena& a = h->arena;
  const long long n_strings = B * h->dev.Q;
  const long long n_units = n_strings * units_per_string;
  if (!a.cnt) CU(cudaMalloc((void**)&a.cnt, sizeof(Counters)));
  if (B > a.cap_configs) {
    cudaFree(a.status);
    CU(cudaMalloc((void**)&a.status, (size_t)(B ? B : 1) * sizeof(int)));
    a.cap_configs = B;
  }
  if (n_strings > a.cap_strings) {
    cudaFree(a.survive); cudaFree(a.strings); cudaFree(a.sector);
    a.survive = nullptr; a.strings = nullptr; a.sector = nullptr; a.cap_strings = 0;
    size_t n = (size_t)(n_strings ? n_strings : 1);
    CU(cudaMalloc((void**)&a.survive, n));
    CU(cudaMalloc((void**)&a.strings, n * sizeof(StringRec)));
    CU(cudaMalloc((void**)&a.sector, n * sizeof(Scaled)));
    a.cap_strings = n_strings;
  }
  if (n_units > a.cap_units) {
    cudaFree(a.units); cudaFree(a.slots);
    a.units = nullptr; a.slots = nullptr; a.cap_units = 0;
    size_t n = (size_t)(n_units ? n_units : 1);
    CU(cudaMalloc((void**)&a.units, n * sizeof(int2)));
    CU(cudaMalloc((void**)&a.slots, n * sizeof(Slot)));
    a.cap_units = n_units;
  }
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
  if (batch->n_configs * (long long)h->dev.Q > 2000000000LL) return fail(CTQMC_ERR_ARG, "n_configs * n_sectors exceeds 2^31");
  return 0;
}

// validate -> route -> class scan -> unit scatter; leaves strings / units / counters ready.
int enqueue_routing(ctqmc_impurity* h, const BatchView& bv, uint8_t* survive_out, int mode, int segment_len, cudaStream_t st) {
  Arena& a = h->arena;
  const long long B = bv.B, nS = B * h->dev.Q;
  CU(cudaMemsetAsync(a.cnt, 0, sizeof(Counters), st));
  validate_kernel<<<(unsigned)((B + 255) / 256), 256, 0, st>>>(bv, h->dev.A, a.status);
  RouteParams rp;
  rp.imp = h->dev; rp.bv = bv; rp.status = a.status; rp.survive = a.survive; rp.survive_out = survive_out;
  rp.strings = a.strings; rp.cnt = a.cnt; rp.W = (h->large || (h->grouped_now && mode == 0)) ? (1 << 20) : 8 * h->nt; rp.kstep = h->dev.cplx ? 4 : 8;
  rp.literal = (h->schedule == CTQMC_SCHEDULE_LITERAL); rp.flops_per_mac = h->dev.cplx ? 8 : 2;
  rp.mode = mode; rp.segment_len = segment_len;
  route_kernel<<<(unsigned)((nS + 255) / 256), 256, 0, st>>>(rp);
  h->last_launches += 2;
  if (mode != 2) {
    class_scan_kernel<<<1, 32, 0, st>>>(a.cnt);
    unit_scatter_kernel<<<(unsigned)((nS + 255) / 256), 256, 0, st>>>(a.strings, nS, a.cnt, a.units);
    h->last_launches += 2;
  }
  CU(cudaGetLastError());
  return 0;
}

int enqueue_chain(ctqmc_impurity* h, const BatchView& bv, int mode, int segment_len, cudaStream_t st) {
  Arena& a = h->arena;
  ChainParams cp;
  cp.imp = h->dev; cp.bv = bv; cp.strings = a.strings; cp.units = a.units; cp.cnt = a.cnt; cp.slots = a.slots;
  cp.ldx = h->ldx; cp.mode = mode; cp.segment_len = segment_len;
  if (h->large) {
    return fail(CTQMC_ERR_UNSUPPORTED, "internal: large-sector path is driven by enqueue_large");
  } else {
    KernelFn fn = pick_kernel(h->dev.cplx, h->nt, h->team_warps);
    fn<<<h->grid, kCtaThreads, h->smem_bytes, st>>>(cp);
  }
  h->last_launches += 1;
  CU(cudaGetLastError());
  return 0;
}


int grow(DevBuf& b, size_t bytes) {
  b.grew = false;
  if (bytes <= b.cap) return 0;
  cudaFree(b.p); b.p = nullptr; b.cap = 0;
  const size_t want = bytes + bytes / 8;
  CU(cudaMalloc(&b.p, want));
  b.cap = want; b.grew = true;
  return 0;
}

// Grouped path (chain_grouped.cuh): schedule for all chain positions, then one GEMM launch per position.  Like the
// large path it reads the routing counters back once to size its buffers and the step loop.
int enqueue_grouped(ctqmc_impurity* h, const BatchView& bv, cudaStream_t st) {
  Arena& a = h->arena;
  Counters c;
  CU(cudaMemcpyAsync(&c, a.cnt, sizeof c, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  const long long n_units = (long long)c.n_slots;
  if (n_units == 0) return 0;
  if (n_units > 2000000000LL / ((long long)c.max_len + 1)) return fail(CTQMC_ERR_OOM, "batch too large for the grouped path's per-position schedule");   // AUTO falls back to the panel kernel
  const int Lmax = (int)c.max_len > 0 ? (int)c.max_len : 1;
  const long long sum_c = (long long)c.sum_c > 0 ? (long long)c.sum_c : 1;
  const int es = h->dev.cplx ? 2 : 1, nb = h->n_blocks;
  const int ldx = (h->dev.dmax + 7) / 8 * 8;
  const long long xtot = sum_c * ldx;
  const int tile_cap = (int)(sum_c / kGBN + (n_units < nb ? n_units : nb) + 1);
  const size_t nul = (size_t)n_units * Lmax;
  int rc;
  {
    const double need = 2.0 * (double)xtot * es * 8.0 + (double)Lmax * (double)sum_c * 8.0 + (double)nul * 20.0;
    if (h->scratch_limit > 0 && need > (double)h->scratch_limit)
      return fail(CTQMC_ERR_OOM, "grouped path needs %.0f bytes of scratch, limit is %lld", need, h->scratch_limit);
  }
  if ((rc = grow(a.gx, (size_t)2 * xtot * es * sizeof(double)))) return rc;
  if (a.gx.grew) CU(cudaMemsetAsync(a.gx.p, 0, a.gx.cap, st));
  if ((rc = grow(a.gxoff, n_units * sizeof(long long))) || (rc = grow(a.gplan_blk, nul * sizeof(int))) ||
      (rc = grow(a.gplan_delta, nul * sizeof(double))) || (rc = grow(a.gkmax, nul * sizeof(int))) ||
      (rc = grow(a.gcoff, nul * sizeof(int))) || (rc = grow(a.gulen, n_units * sizeof(int))) ||
      (rc = grow(a.gucols, n_units * sizeof(int))) || (rc = grow(a.gcolcnt, (size_t)Lmax * nb * sizeof(int))) ||
      (rc = grow(a.gcolbase, (size_t)Lmax * nb * sizeof(int))) || (rc = grow(a.gtiles, (size_t)Lmax * tile_cap * sizeof(int4))) ||
      (rc = grow(a.gntiles, (size_t)Lmax * sizeof(int))) || (rc = grow(a.gcolmap, (size_t)Lmax * sum_c * sizeof(int2))))
    return rc;
  GroupedParams gp;
  gp.imp = h->dev; gp.bv = bv; gp.strings = a.strings; gp.units = a.units; gp.n_units = (int)n_units; gp.Lmax = Lmax; gp.ldx = ldx;
  gp.nb = nb; gp.xtot = xtot; gp.X = (double*)a.gx.p; gp.xoff = (long long*)a.gxoff.p; gp.plan_blk = (int*)a.gplan_blk.p;
  gp.plan_delta = (double*)a.gplan_delta.p; gp.kmax = (int*)a.gkmax.p; gp.coff = (int*)a.gcoff.p; gp.ulen = (int*)a.gulen.p;
  gp.ucols = (int*)a.gucols.p; gp.colcnt = (int*)a.gcolcnt.p; gp.colbase = (int*)a.gcolbase.p; gp.tiles = (int4*)a.gtiles.p;
  gp.ntiles = (int*)a.gntiles.p; gp.colmap = (int2*)a.gcolmap.p; gp.tile_cap = tile_cap; gp.col_cap = sum_c; gp.slots = a.slots;
  CU(cudaMemsetAsync(gp.colcnt, 0, (size_t)Lmax * nb * sizeof(int), st));
  const unsigned g_ul = (unsigned)((nul + 255) / 256);
  grouped_plan_kernel<<<(unsigned)((n_units + 127) / 128), 128, 0, st>>>(gp);
  grouped_xoff_kernel<<<1, 1024, 0, st>>>(gp);
  grouped_count_kernel<<<g_ul, 256, 0, st>>>(gp);
  grouped_tiles_kernel<<<Lmax, 32, 0, st>>>(gp);
  grouped_fill_kernel<<<g_ul, 256, 0, st>>>(gp);
  const int MTmax = (h->dev.dmax + kGBM - 1) / kGBM;
  const unsigned sg = (unsigned)tile_cap * (unsigned)MTmax;
  // step launches use programmatic stream serialization (see the kernel): launch gaps and tails overlap the next step's prologue
  cudaLaunchConfig_t lc = {};
  lc.gridDim = dim3(sg); lc.blockDim = dim3(kGThreads); lc.dynamicSmemBytes = h->grouped_smem; lc.stream = st;
  cudaLaunchAttribute lattr[1];
  lattr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  lattr[0].val.programmaticStreamSerializationAllowed = 1;
  lc.attrs = lattr; lc.numAttrs = 1;
  if (h->dev.cplx) {
    grouped_init_kernel<true><<<(unsigned)n_units, 128, 0, st>>>(gp);
    for (int j = 0; j < Lmax; ++j) CU(cudaLaunchKernelEx(&lc, grouped_step_kernel<true>, gp, j, MTmax));
    grouped_finish_kernel<true><<<(unsigned)n_units, 256, 0, st>>>(gp);
  } else {
    grouped_init_kernel<false><<<(unsigned)n_units, 128, 0, st>>>(gp);
    for (int j = 0; j < Lmax; ++j) CU(cudaLaunchKernelEx(&lc, grouped_step_kernel<false>, gp, j, MTmax));
    grouped_finish_kernel<false><<<(unsigned)n_units, 256, 0, st>>>(gp);
  }
  h->last_launches += 7 + Lmax;
  CU(cudaGetLastError());
  return 0;
}

// Large-sector path: one launch per chain position over all strings of a group (chain_large.cuh).  Reads back three
// integers (strings with work, longest chain, widest carried matrix) to size the step loop and the carried matrices:
// the one host synchronisation of this path.
int enqueue_large(ctqmc_impurity* h, const BatchView& bv, int mode, int segment_len, cudaStream_t st) {
  Arena& a = h->arena;
  Counters c;
  CU(cudaMemcpyAsync(&c, a.cnt, sizeof c, cudaMemcpyDeviceToHost, st));
  CU(cudaStreamSynchronize(st));
  const long long n_units = (long long)c.n_slots;
  if (n_units == 0) return 0;
  const int Lmax = (int)c.max_len > 0 ? (int)c.max_len : 1;
  const int cmax = mode == 1 ? h->dev.dmax : ((int)c.max_c > 0 ? (int)c.max_c : 1);   // segments start from full identities
  const int n_launch = mode == 1 ? (segment_len < Lmax ? segment_len : Lmax) : Lmax;
  const int es = h->dev.cplx ? 2 : 1;
  const long long xslab = (long long)cmax * h->ldx;
  const size_t per_string = (size_t)2 * xslab * es * sizeof(double);
  size_t free_b = 0, total_b = 0;
  CU(cudaMemGetInfo(&free_b, &total_b));
  const size_t budget = a.lx_bytes + (size_t)(0.7 * (double)free_b);
  long long G = (long long)(budget / per_string);
  if (G < 1) return fail(CTQMC_ERR_OOM, "not enough device memory for one carried matrix pair (%zu bytes)", per_string);
  if (G > n_units) G = n_units;
  if (G > 65535) G = 65535;
  if ((size_t)G * per_string > a.lx_bytes) {
    cudaFree(a.lx); a.lx = nullptr; a.lx_bytes = 0;
    CU(cudaMalloc((void**)&a.lx, (size_t)G * per_string));
    a.lx_bytes = (size_t)G * per_string;
    CU(cudaMemsetAsync(a.lx, 0, a.lx_bytes, st));
  }
  if ((size_t)G * Lmax > a.plan_cap) {
    cudaFree(a.plan_blk); cudaFree(a.plan_delta); cudaFree(a.lkmax);
    a.plan_blk = nullptr; a.plan_delta = nullptr; a.lkmax = nullptr; a.plan_cap = 0;
    const size_t n = (size_t)G * Lmax;
    CU(cudaMalloc((void**)&a.plan_blk, n * sizeof(int)));
    CU(cudaMalloc((void**)&a.plan_delta, n * sizeof(double)));
    CU(cudaMalloc((void**)&a.lkmax, n * sizeof(int)));
    a.plan_cap = n;
  }
  { int rc = grow(a.lunit, (size_t)3 * G * sizeof(int)); if (rc) return rc; }
  LargeParams lp;
  lp.u_q = (int*)a.lunit.p; lp.u_n = lp.u_q + G; lp.u_c = lp.u_n + G; lp.mode = mode; lp.segment_len = segment_len;
  lp.imp = h->dev; lp.bv = bv; lp.strings = a.strings; lp.units = a.units; lp.Lmax = Lmax; lp.ldx = h->ldx;
  lp.xslab = xslab; lp.X = a.lx; lp.plan_blk = a.plan_blk; lp.plan_delta = a.plan_delta; lp.kmax = a.lkmax; lp.slots = a.slots;
  lp.amaps = h->d_amaps; lp.xmaps = nullptr;
  const bool tma = h->use_tma && h->d_amaps;
  if (tma) {   // tensor maps of the carried matrices (two per string slot); rebuilt only when the arena changed
    if (a.xmaps_base != a.lx || a.xmaps_g < G || a.xmaps_slab != xslab || a.xmaps_cmax != cmax) {
      std::vector<CUtensorMap> maps((size_t)2 * G);
      for (long long i = 0; i < 2 * G; ++i) {
        int rc = encode_2d(&maps[i], a.lx + (size_t)i * xslab * es, (unsigned long long)h->ldx * es, (unsigned long long)cmax,
                           (unsigned long long)h->ldx * es * 8, kLBN);
        if (rc) return rc;
      }
      { int rc = grow(a.xmaps, maps.size() * sizeof(CUtensorMap)); if (rc) return rc; }
      CU(cudaMemcpyAsync(a.xmaps.p, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, st));
      CU(cudaStreamSynchronize(st));   // `maps` is a pageable host vector
      a.xmaps_base = a.lx; a.xmaps_g = G; a.xmaps_slab = xslab; a.xmaps_cmax = cmax;
    }
    lp.xmaps = (const CUtensorMap*)a.xmaps.p;
  }
  const int MTmax = (h->dev.dmax + kLBM - 1) / kLBM, NTmax = (cmax + kLBN - 1) / kLBN;
  for (long long u0 = 0; u0 < n_units; u0 += G) {
    lp.u0 = u0; lp.n_group = (int)((n_units - u0 < G) ? (n_units - u0) : G);
    large_plan_kernel<<<(lp.n_group + 127) / 128, 128, 0, st>>>(lp);
    dim3 ig((unsigned)((cmax < 1024) ? cmax : 1024), (unsigned)lp.n_group);
    dim3 sg((unsigned)(MTmax * NTmax), (unsigned)lp.n_group);
    if (h->dev.cplx) {
      large_init_kernel<true><<<ig, 256, 0, st>>>(lp);
      for (int j = 0; j < n_launch; ++j) {
        if (tma) large_step_kernel<true, true><<<sg, 256, h->smem_bytes, st>>>(lp, j, NTmax);
        else     large_step_kernel<true, false><<<sg, 256, h->smem_bytes, st>>>(lp, j, NTmax);
      }
      large_finish_kernel<true><<<lp.n_group, 256, 0, st>>>(lp);
    } else {
      large_init_kernel<false><<<ig, 256, 0, st>>>(lp);
      for (int j = 0; j < n_launch; ++j) {
        if (tma) large_step_kernel<false, true><<<sg, 256, h->smem_bytes, st>>>(lp, j, NTmax);
        else     large_step_kernel<false, false><<<sg, 256, h->smem_bytes, st>>>(lp, j, NTmax);
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
  cudaFree(h->d_pack); cudaFree(h->d_pblk); cudaFree(h->d_blkorder);
  cudaFree(h->d_blks); cudaFree(h->d_store); cudaFree(h->d_rownorm2); cudaFree(h->d_sigma);
  Arena& a = h->arena;
  cudaFree(a.status); cudaFree(a.survive); cudaFree(a.strings); cudaFree(a.units); cudaFree(a.slots); cudaFree(a.sector);
  for (DevBuf* b : {&a.gx, &a.gxoff, &a.gplan_blk, &a.gplan_delta, &a.gkmax, &a.gcoff, &a.gulen, &a.gucols, &a.gcolcnt, &a.gcolbase,
                     &a.gtiles, &a.gntiles, &a.gcolmap}) cudaFree(b->p);
  cudaFree(a.lunit.p); cudaFree(a.xmaps.p); cudaFree(h->d_amaps); cudaFree(a.cnt); cudaFree(a.lx); cudaFree(a.plan_blk); cudaFree(a.plan_delta); cudaFree(a.lkmax); cudaFree(a.d_stage);
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
    int nt = h->nt, tw = h->team_warps, ldx = h->ldx, grid = h->grid; size_t sm = h->smem_bytes;
    int rc = configure(h, (int)value);
    if (rc || h->large) { h->nt = nt; h->team_warps = tw; h->ldx = ldx; h->grid = grid; h->smem_bytes = sm; h->large = 0;
                          return rc ? rc : fail(CTQMC_ERR_UNSUPPORTED, "panel width %lld does not fit in shared memory for this impurity", (long long)value); }
    return 0;
  }
  if (option == CTQMC_OPT_PATH) {
    if (value != CTQMC_PATH_AUTO && value != CTQMC_PATH_PANEL && value != CTQMC_PATH_LARGE && value != CTQMC_PATH_SMALL && value != CTQMC_PATH_GROUPED) return fail(CTQMC_ERR_ARG, "unknown path %lld", (long long)value);
    const int old = h->path;
    h->path = (int)value;
    int rc = configure(h, 0);
    if (rc) { h->path = old; configure(h, 0); }
    return rc;
  }
  if (option == CTQMC_OPT_SCRATCH_LIMIT) {
    if (value < 0) return fail(CTQMC_ERR_ARG, "scratch limit must be >= 0");
    h->scratch_limit = (long long)value;
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
  // AUTO: batches of at least kGroupedMinBatch configurations take the step-synchronous grouped path (one launch per chain
  // position pays off once many strings share blocks); smaller ones the persistent panel kernel
  h->grouped_now = h->grouped || (h->path == CTQMC_PATH_AUTO && h->grouped_ok && !h->small && !h->large && B >= kGroupedMinBatch);
  h->last_path = h->small ? CTQMC_PATH_SMALL : h->grouped_now ? CTQMC_PATH_GROUPED : h->large ? CTQMC_PATH_LARGE : CTQMC_PATH_PANEL;
  const int W = (h->large || h->grouped_now) ? (1 << 20) : 8 * h->nt;
  if (h->small) { if (!h->arena.cnt) CU(cudaMalloc((void**)&h->arena.cnt, sizeof(Counters))); }
  else { rc = ensure_arena(h, B, (h->dev.dmax + W - 1) / W); if (rc) return rc; }
  h->last_stream = st; h->last_launches = 0;
  BatchView bv; bv.B = B; bv.offset = (const long long*)batch->offset; bv.symbol = batch->symbol; bv.tau = batch->tau; bv.beta = beta;
  h->timing_valid = 0;
  if (h->small) {
    // everything (validation, routing, chain, trace, sector sum) in one launch: chain_small.cuh
    Arena& a = h->arena;
    mark(h, 0, st);
    CU(cudaMemsetAsync(a.cnt, 0, sizeof(Counters), st));
    mark(h, 1, st);
    SmallParams sp;
    sp.imp = h->dev; sp.bv = bv; sp.pack = h->d_pack; sp.pblk = h->d_pblk; sp.n_blocks = h->n_blocks; sp.pack_len = h->pack_len;
    sp.n_energy = h->n_energy; sp.literal = (h->schedule == CTQMC_SCHEDULE_LITERAL); sp.mant = mant; sp.exp2 = (long long*)exp2;
    sp.survive = survive; sp.status = status; sp.cnt = a.cnt; sp.dmax = h->dev.dmax;
    if (h->small2) {
      Small2Params s2;
      s2.imp = h->dev; s2.bv = bv; s2.ftpad = h->d_ftpad; s2.binfo = h->d_binfo; s2.n_blocks = h->n_blocks; s2.literal = sp.literal;
      s2.mant = mant; s2.exp2 = (long long*)exp2; s2.survive = survive; s2.status = status; s2.cnt = a.cnt;
      // CTA size: small batches are latency-bound, so they are spread over all SMs in ONE wave: warps per CTA =
      // ceil(configurations per SM / configurations per warp), at most the configured maximum
      const int gpw = 32 / h->small2_dp, max_warps = h->small2_threads / 32;
      long long per_sm = (B + h->sm_count - 1) / h->sm_count;
      int warps = (int)((per_sm + gpw - 1) / gpw);
      if (warps < 2) warps = 2;
      if (warps > max_warps) warps = max_warps;
      const int threads = 32 * warps;
      const long long gpc = (long long)warps * gpw;
      const size_t smem = small2_common_bytes(h->dev.Q, h->dev.A, h->n_blocks, h->small2_dp) + (size_t)gpc * small2_group_bytes(h->dev.Q, h->small2_dp);
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
  mark(h, 0, st);
  rc = enqueue_routing(h, bv, survive, 0, 0, st);
  if (rc) return rc;
  mark(h, 1, st);
  rc = h->grouped_now ? enqueue_grouped(h, bv, st) : h->large ? enqueue_large(h, bv, 0, 0, st) : enqueue_chain(h, bv, 0, 0, st);
  if (rc == CTQMC_ERR_OOM && h->grouped_now && h->path == CTQMC_PATH_AUTO && !h->large) {
    // the grouped path's schedule (one column map per chain position) did not fit: AUTO falls back to the persistent
    // panel kernel, which needs no per-position scratch.  Routing is redone with panel-sized work units.
    cudaGetLastError();
    h->grouped_now = 0; h->last_path = CTQMC_PATH_PANEL; h->last_launches = 0;
    const int Wp = 8 * h->nt;
    rc = ensure_arena(h, B, (h->dev.dmax + Wp - 1) / Wp);
    if (rc) return rc;
    rc = enqueue_routing(h, bv, survive, 0, 0, st);
    if (rc) return rc;
    rc = enqueue_chain(h, bv, 0, 0, st);
  }
  if (rc) return rc;
  mark(h, 2, st);
  TraceReduceParams tp;
  tp.B = B; tp.Q = h->dev.Q; tp.status_in = h->arena.status; tp.survive = h->arena.survive; tp.strings = h->arena.strings;
  tp.slots = h->arena.slots; tp.mant = mant; tp.exp2 = (long long*)exp2; tp.status = status;
  trace_reduce_kernel<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(tp);
  h->last_launches += 1;
  mark(h, 3, st);
  h->timing_valid = h->timing;
  CU(cudaGetLastError());
  return 0;
}

extern "C" int ctqmc_bound_batch(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, int norm_kind, int segment_len,
                                 double* bound_mant, int64_t* bound_exp2, double* sector_bound_mant,
                                 int64_t* sector_bound_exp2, int32_t* status, void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  if (norm_kind != 0 && norm_kind != 1) return fail(CTQMC_ERR_ARG, "norm_kind must be 0 (Frobenius) or 1 (spectral)");
  if (segment_len < 0) return fail(CTQMC_ERR_ARG, "segment_len < 0");
  if (norm_kind == 1 && segment_len != 1)
    return fail(CTQMC_ERR_UNSUPPORTED, "spectral norm is implemented for segment_len = 1 only");
  if ((sector_bound_mant == nullptr) != (sector_bound_exp2 == nullptr)) return fail(CTQMC_ERR_ARG, "sector_bound_mant / _exp2 must both be given or both be null");
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!bound_mant || !bound_exp2 || !status) return fail(CTQMC_ERR_ARG, "null output");
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int W = h->large ? (1 << 20) : 8 * h->nt;
  const long long nS = B * h->dev.Q;
  BatchView bv; bv.B = B; bv.offset = (const long long*)batch->offset; bv.symbol = batch->symbol; bv.tau = batch->tau; bv.beta = beta;
  h->last_stream = st; h->last_launches = 0;
  h->timing_valid = 0;
  h->grouped_now = 0; h->last_path = h->large ? CTQMC_PATH_LARGE : CTQMC_PATH_PANEL;
  BoundParams bp;
  if (segment_len == 1 && h->small2) {
    // small real impurities: validation, routing, norm products and the sector sum in one launch (bound_small2.cuh)
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
  if (segment_len == 1) {
    rc = ensure_arena(h, B, 1);
    if (rc) return rc;
    mark(h, 0, st);
    rc = enqueue_routing(h, bv, nullptr, 2, 1, st);
    if (rc) return rc;
    mark(h, 1, st);
    bp.imp = h->dev; bp.bv = bv; bp.survive = h->arena.survive; bp.strings = h->arena.strings; bp.slots = h->arena.slots;
    bp.sector = h->arena.sector; bp.norm_kind = norm_kind; bp.segment_len = 1; bp.W = W;
    bound_s1_kernel<<<(unsigned)((nS * 32 + 255) / 256), 256, 0, st>>>(bp);
    h->last_launches += 1;
  } else {
    // units per string depend on the chain lengths, which live on the device: one small read-back of the total
    // operator count sizes the arena (the only host synchronisation in the library's device-pointer API).
    long long n_ops = 0;
    CU(cudaMemcpyAsync(&n_ops, batch->offset + B, sizeof(long long), cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));
    const int S = segment_len == 0 ? 1 << 30 : segment_len;
    const long long panels = (h->dev.dmax + W - 1) / W;
    long long max_units_per_string = (segment_len == 0) ? panels : ((n_ops / S) / (B ? 1 : 1) + 1) * panels;
    // worst case: one configuration holds every operator
    rc = ensure_arena(h, B, 1);
    if (rc) return rc;
    {
      // exact sizing would need the per-configuration lengths; bound it by sum over configurations instead:
      // sum_b Q * (L_b / S + 1) * panels <= Q * panels * (n_ops / S + B)
      long long need = (long long)h->dev.Q * panels * ((segment_len == 0 ? 0 : n_ops / S) + B);
      Arena& a = h->arena;
      if (need > a.cap_units) {
        cudaFree(a.units); cudaFree(a.slots); a.units = nullptr; a.slots = nullptr; a.cap_units = 0;
        CU(cudaMalloc((void**)&a.units, (size_t)need * sizeof(int2)));
        CU(cudaMalloc((void**)&a.slots, (size_t)need * sizeof(Slot)));
        a.cap_units = need;
      }
      (void)max_units_per_string;
    }
    mark(h, 0, st);
    rc = enqueue_routing(h, bv, nullptr, 1, S, st);
    if (rc) return rc;
    mark(h, 1, st);
    rc = h->large ? enqueue_large(h, bv, 1, S, st) : enqueue_chain(h, bv, 1, S, st);
    if (rc) return rc;
    bp.imp = h->dev; bp.bv = bv; bp.survive = h->arena.survive; bp.strings = h->arena.strings; bp.slots = h->arena.slots;
    bp.sector = h->arena.sector; bp.norm_kind = 0; bp.segment_len = S; bp.W = W;
    bound_segments_kernel<<<(unsigned)((nS + 127) / 128), 128, 0, st>>>(bp);
    h->last_launches += 1;
  }
  mark(h, 2, st);
  BoundReduceParams rp;
  rp.B = B; rp.Q = h->dev.Q; rp.status_in = h->arena.status; rp.survive = h->arena.survive; rp.sector = h->arena.sector;
  rp.bound_mant = bound_mant; rp.bound_exp2 = (long long*)bound_exp2; rp.sector_mant = sector_bound_mant;
  rp.sector_exp2 = (long long*)sector_bound_exp2; rp.status = status;
  bound_reduce_kernel<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(rp);
  h->last_launches += 1;
  mark(h, 3, st);
  h->timing_valid = h->timing;
  CU(cudaGetLastError());
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

int stage_in(ctqmc_impurity* h, const ctqmc_batch* hb, size_t out_bytes, Staged* sg, cudaStream_t st) {
  const long long B = hb->n_configs;
  if (!hb->offset) return fail(CTQMC_ERR_ARG, "batch.offset is null");
  const long long n_ops = hb->offset[B];
  if (n_ops < 0) return fail(CTQMC_ERR_ARG, "negative operator count");
  if (n_ops > 0 && (!hb->symbol || !hb->tau)) return fail(CTQMC_ERR_ARG, "null symbol / tau");
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
  const long long n_ops = hb->offset[B];
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
    int rc = ctqmc_trace_batch(h, beta, &sub, (double*)(d_out + o_mant) + 2 * b0, (int64_t*)(d_out + o_exp) + b0,
                               survive ? (uint8_t*)(d_out + o_surv) + b0 * Q : nullptr, (int32_t*)(d_out + o_stat) + b0, st);
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
  if (batch->offset && batch->offset[B] >= 0 && (batch->offset[B] == 0 || (batch->symbol && batch->tau)) &&
      is_pinned(batch->offset) && (batch->offset[B] == 0 || (is_pinned(batch->symbol) && is_pinned(batch->tau))) &&
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

extern "C" int ctqmc_last_stats(ctqmc_impurity* h, int64_t stats[8]) {
  if (!h || !stats) return fail(CTQMC_ERR_ARG, "null argument");
  for (int i = 0; i < 8; ++i) stats[i] = 0;
  stats[5] = h->small ? (h->small2 ? h->small2_dp : h->small_g) : h->nt * 8; stats[6] = h->team_warps; stats[7] = h->last_path ? h->last_path : (h->small ? 3 : h->grouped ? 4 : h->large ? 2 : 1);
  if (!h->arena.cnt) return 0;
  CU(cudaSetDevice(h->device));
  Counters c;
  CU(cudaStreamSynchronize(h->last_stream));
  CU(cudaMemcpy(&c, h->arena.cnt, sizeof c, cudaMemcpyDeviceToHost));
  stats[0] = (int64_t)c.n_strings; stats[1] = (int64_t)c.n_slots; stats[2] = h->last_launches;
  stats[3] = (int64_t)c.macs; stats[4] = (int64_t)c.alg_flops;
  if (h->last_path == CTQMC_PATH_SMALL) stats[6] = (int64_t)c.n_exp;
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
