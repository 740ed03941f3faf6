// Host side of the chain-set calls of include/ctqmc.h (ctqmc_chains_*): storage layout and kernel sequences of the
// incremental lazy trace (lazy.cuh).  Included at the end of ctqmc_api.cu (uses its error helpers and the impurity handle).
// Every call only enqueues: launch shapes come from host-known bounds (chains, depth, leaf capacity, edits per proposal,
// sector count and dimensions); which chains still need work is decided on the device, idle CTAs exit at once.
#pragma once
#include "lazy.cuh"

struct ctqmc_chains {
  ctqmc_impurity* imp = nullptr;
  LazyView V{};
  char* block = nullptr;
  size_t bytes = 0;
  int lazy_rounds = 1;
  int NT = 1;                 // tiles per matrix side
  int g_gemm = 1, g_fix = 1;  // persistent CTAs of the list-driven kernels (resident CTAs per SM x SMs)
  int seq = 0;                // node steps enqueued so far: its parity selects the node work lists
  bool small = false;         // every sector dimension <= kLzSmall: warp-per-task kernels (lazy.cuh, "small impurities")
  long long launches = 0;     // kernels enqueued by the most recent call
  cudaStream_t last_stream = nullptr;
};

namespace {

size_t chains_layout(LazyView& V, char* base) {
  Bump bp{base};
  const size_t nC = V.nC, Q = V.imp.Q;
  V.leaf_n = bp.take<int>(nC * V.nleaf);
  V.leaf_tau = bp.take<double>(nC * V.nleaf * V.cap);
  V.leaf_sym = bp.take<int>(nC * V.nleaf * V.cap);
  V.slot_of = bp.take<int>(nC * V.nnode);
  V.free_slot = bp.take<int>(nC * (V.smax + V.emax));
  const size_t ne = nC * V.NN * Q;
  V.ent_tgt = bp.take<int>(ne); V.ent_valid = bp.take<int>(ne); V.ent_k = bp.take<int>(ne);
  V.ent_e = bp.take<long long>(ne); V.ent_lg = bp.take<double>(ne); V.ent_nrm = bp.take<double>(ne);
  V.p_status = bp.take<int>(nC); V.p_ndirty = bp.take<int>(nC); V.p_nleaf = bp.take<int>(nC); V.p_node = bp.take<int>(nC * V.smax);
  V.sh_n = bp.take<int>(nC * V.emax); V.sh_tau = bp.take<double>(nC * V.emax * V.cap); V.sh_sym = bp.take<int>(nC * V.emax * V.cap);
  V.sb_m = bp.take<double>(nC * Q); V.sb_e = bp.take<long long>(nC * Q); V.order = bp.take<int>(nC * Q); V.n_alive = bp.take<int>(nC);
  V.decided = bp.take<int>(nC); V.decided_by = bp.take<int>(nC); V.n_eval = bp.take<int>(nC);
  V.term_re = bp.take<double>(nC * Q); V.term_im = bp.take<double>(nC * Q); V.term_e = bp.take<long long>(nC * Q);
  V.thr = bp.take<double>(nC); V.p_accept = bp.take<int>(nC);
  V.n_products = bp.take<unsigned long long>(1);
  V.p_lvl_start = bp.take<int>(nC * (size_t)(V.D > 0 ? V.D : 1)); V.p_lvl_cnt = bp.take<int>(nC * (size_t)(V.D > 0 ? V.D : 1));
  V.w_cnt = bp.take<int>(16);
  V.w_ltask = bp.take<int4>(3 * (size_t)V.w_task_cap); V.w_ltile = bp.take<int4>(3 * (size_t)V.w_tile_cap);
  V.w_ntask = bp.take<int4>(2 * 2 * (size_t)V.w_task_cap); V.w_ntile = bp.take<int4>(2 * (size_t)V.w_tile_cap);
  V.w_larr = bp.take<int>(3 * (size_t)V.w_task_cap); V.w_narr = bp.take<int>(2 * (size_t)V.w_task_cap); V.w_part = bp.take<double>((size_t)V.w_tile_cap);
  V.mats = bp.take<double>(nC * V.NN * (size_t)V.node_elems);
  return bp.off + 256;
}

// dirty ancestors, bottom-up: mode 0 = the entries start sector order[r] needs, mode 1 = every missing entry
int chains_enqueue_levels(ctqmc_chains* ch, int mode, int r, const int* gate, int gate_commit, cudaStream_t st) {
  const LazyView& V = ch->V;
  const long long cand = (long long)V.nC * V.emax * (mode == 0 ? 1 : V.imp.Q);
  if (ch->small && V.D > 0) {       // all levels in one launch, one CTA per chain
    if (V.imp.cplx) lazy_node_small_kernel<true><<<V.nC, 32 * lz_node_small_warps(true), 0, st>>>(V, mode, r, gate, gate_commit);
    else            lazy_node_small_kernel<false><<<V.nC, 32 * lz_node_small_warps(false), 0, st>>>(V, mode, r, gate, gate_commit);
    ch->launches += 1;
  }
  for (int level = V.D - 1; level >= 0 && !ch->small; --level) {
    const int par = ch->seq++ & 1;
    lazy_node_plan_kernel<<<(unsigned)((cand + 255) / 256), 256, 0, st>>>(V, level, mode, r, gate, gate_commit, par);
    if (V.imp.cplx) {
      lazy_node_gemm_kernel<true><<<ch->g_gemm, kLzThreads, 0, st>>>(V, par);
      lazy_node_fix_kernel<true><<<ch->g_fix, 256, 0, st>>>(V, par);
    } else {
      lazy_node_gemm_kernel<false><<<ch->g_gemm, kLzThreads, 0, st>>>(V, par);
      lazy_node_fix_kernel<false><<<ch->g_fix, 256, 0, st>>>(V, par);
    }
    ch->launches += 3;
  }
  CU(cudaGetLastError());
  return 0;
}

}  // namespace

extern "C" int ctqmc_chains_create(ctqmc_impurity* h, double beta, const ctqmc_chains_desc* desc, void* cuda_stream, ctqmc_chains** out) {
  if (!h || !desc || !out) return fail(CTQMC_ERR_ARG, "null impurity, desc or out");
  *out = nullptr;
  if (!(beta > 0.0) || !std::isfinite(beta)) return fail(CTQMC_ERR_ARG, "beta must be positive and finite");
  if (desc->n_chains < 1 || desc->n_chains > (1 << 20)) return fail(CTQMC_ERR_ARG, "n_chains out of range [1, 2^20]");
  if (desc->depth < 0 || desc->depth > 16) return fail(CTQMC_ERR_ARG, "depth out of range [0, 16]");
  if (desc->leaf_capacity < 1 || desc->leaf_capacity > 64) return fail(CTQMC_ERR_ARG, "leaf_capacity out of range [1, 64]");
  if (desc->max_edits < 1 || desc->max_edits > 16) return fail(CTQMC_ERR_ARG, "max_edits out of range [1, 16]");
  if (desc->lazy_rounds < 0) return fail(CTQMC_ERR_ARG, "lazy_rounds < 0");
  if (h->dev.dmax > kLzMaxDim)
    return fail(CTQMC_ERR_UNSUPPORTED, "chain sets store dense sub-products per tree node: sector dimension %d exceeds %d", h->dev.dmax, kLzMaxDim);
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  ctqmc_chains* ch = new (std::nothrow) ctqmc_chains();
  if (!ch) return fail(CTQMC_ERR_OOM, "host allocation failed");
  ch->imp = h;
  LazyView& V = ch->V;
  V.imp = h->dev; V.beta = beta; V.nC = (int)desc->n_chains; V.D = desc->depth; V.nleaf = 1 << V.D; V.nnode = 2 * V.nleaf - 1;
  V.cap = desc->leaf_capacity; V.emax = desc->max_edits; V.smax = V.emax * (V.D + 1); V.NN = V.nnode + V.smax + V.emax;
  V.ldm = h->dev.dmax; V.node_elems = (long long)h->n_energy * V.ldm * (h->dev.cplx ? 2 : 1);
  ch->lazy_rounds = desc->lazy_rounds < h->dev.Q ? desc->lazy_rounds : h->dev.Q;
  ch->NT = (h->dev.dmax + kLzTile - 1) / kLzTile;
  ch->small = h->dev.dmax <= kLzSmall;
  V.w_task_cap = ch->small ? 1 : (long long)V.nC * V.emax * h->dev.Q;      // small impurities never build work lists
  V.w_tile_cap = V.w_task_cap * ch->NT * ch->NT;
  {
    int occ_g = 1, occ_f = 1, sms = 1;
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->device));
    if (h->dev.cplx) {
      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_g, lazy_node_gemm_kernel<true>, kLzThreads, 0));
      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_f, lazy_node_fix_kernel<true>, 256, 0));
    } else {
      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_g, lazy_node_gemm_kernel<false>, kLzThreads, 0));
      CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_f, lazy_node_fix_kernel<false>, 256, 0));
    }
    ch->g_gemm = sms * (occ_g > 0 ? occ_g : 1); ch->g_fix = sms * (occ_f > 0 ? occ_f : 1);
  }
  if ((long long)V.nC * V.smax > 2000000000LL || V.w_tile_cap > 500000000LL) {
    delete ch; return fail(CTQMC_ERR_ARG, "n_chains * max_edits * (depth + 1), or the work lists of n_chains * max_edits * sectors * tiles, exceed 2^31");
  }
  ch->bytes = chains_layout(V, nullptr);
  cudaError_t e = cudaMalloc((void**)&ch->block, ch->bytes);
  if (e != cudaSuccess) {
    cudaGetLastError();
    const size_t need = ch->bytes;
    delete ch;
    return fail(CTQMC_ERR_OOM, "a chain set of this shape needs %zu bytes of device memory (PAPER.md:574: fewer chains or a shallower tree)", need);
  }
  chains_layout(V, ch->block);
  const int Q = h->dev.Q;
  lazy_reset_kernel<<<1024, 256, 0, st>>>(V);
  CU(cudaMemsetAsync(V.n_products, 0, sizeof(unsigned long long), st));
  // chain 0: leaves, then parents level by level; then replicate (every chain starts from the empty configuration)
  if (h->dev.cplx) lazy_build_leaves_kernel<true><<<dim3(V.nleaf, Q), 256, 0, st>>>(V);
  else             lazy_build_leaves_kernel<false><<<dim3(V.nleaf, Q), 256, 0, st>>>(V);
  for (int level = V.D - 1; level >= 0; --level) {
    dim3 gg(1u << level, (unsigned)(ch->NT * ch->NT), (unsigned)Q), gf(1u << level, (unsigned)Q);
    if (h->dev.cplx) { lazy_build_gemm_kernel<true><<<gg, kLzThreads, 0, st>>>(V, level, ch->NT); lazy_build_fix_kernel<true><<<gf, 256, 0, st>>>(V, level); }
    else             { lazy_build_gemm_kernel<false><<<gg, kLzThreads, 0, st>>>(V, level, ch->NT); lazy_build_fix_kernel<false><<<gf, 256, 0, st>>>(V, level); }
  }
  if (V.nC > 1) lazy_replicate_kernel<<<2048, 256, 0, st>>>(V);
  ch->launches = 3 + 2 * V.D + (V.nC > 1);
  ch->last_stream = st;
  cudaError_t le = cudaGetLastError();
  if (le != cudaSuccess) { cudaFree(ch->block); delete ch; return fail(CTQMC_ERR_CUDA, "chain-set construction: %s", cudaGetErrorString(le)); }
  *out = ch;
  return 0;
}

extern "C" void ctqmc_chains_destroy(ctqmc_chains* ch) {
  if (!ch) return;
  cudaSetDevice(ch->imp->device);
  cudaDeviceSynchronize();
  cudaFree(ch->block);
  delete ch;
}

extern "C" int ctqmc_chains_propose(ctqmc_chains* ch, const ctqmc_edit_batch* edits, const double* log2_threshold, int32_t* accept,
                                    int32_t* decided_by, int32_t* n_sectors_evaluated, double* bound_mant, int64_t* bound_exp2,
                                    double* trace_mant, int64_t* trace_exp2, int32_t* status, void* cuda_stream) {
  if (!ch || !edits) return fail(CTQMC_ERR_ARG, "null chain set or edits");
  if (!accept || !decided_by || !n_sectors_evaluated || !bound_mant || !bound_exp2 || !trace_mant || !trace_exp2 || !status)
    return fail(CTQMC_ERR_ARG, "null output");
  if (edits->n_edits < 0) return fail(CTQMC_ERR_ARG, "n_edits < 0");
  if (edits->n_edits > 0 && (!edits->offset || !edits->tau || !edits->symbol || !edits->kind)) return fail(CTQMC_ERR_ARG, "null edit arrays");
  CU(cudaSetDevice(ch->imp->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const LazyView& V = ch->V;
  const bool cx = V.imp.cplx != 0;
  const int Q = V.imp.Q;
  ch->launches = 0; ch->last_stream = st;
  LazyEdits E;
  E.offset = (const long long*)edits->offset; E.tau = edits->tau; E.sym = edits->symbol; E.kind = edits->kind; E.n_edits = edits->n_edits;
  if (edits->n_edits == 0) E.offset = nullptr;
  lazy_prepare_kernel<<<(unsigned)(((long long)V.nC * 32 + 127) / 128), 128, 0, st>>>(V, E, log2_threshold);
  const unsigned ltasks = (unsigned)((long long)V.nC * V.emax);
  dim3 gl(ltasks, (unsigned)Q);
  if (ch->small) {
    const unsigned g = (unsigned)(((long long)ltasks * Q + kLzSmallWarps - 1) / kLzSmallWarps);
    if (cx) lazy_leaf_small_kernel<true><<<g, 32 * kLzSmallWarps, 0, st>>>(V); else lazy_leaf_small_kernel<false><<<g, 32 * kLzSmallWarps, 0, st>>>(V);
    ch->launches += 1;
  } else if (cx) lazy_leaf_init_kernel<true><<<gl, 256, 0, st>>>(V); else lazy_leaf_init_kernel<false><<<gl, 256, 0, st>>>(V);
  for (int j = 0; j < V.cap && !ch->small; ++j) {
    if (cx) { lazy_leaf_step_kernel<true><<<ch->g_gemm, kLzThreads, 0, st>>>(V, j); lazy_leaf_fix_kernel<true><<<ch->g_fix, 256, 0, st>>>(V, j); }
    else    { lazy_leaf_step_kernel<false><<<ch->g_gemm, kLzThreads, 0, st>>>(V, j); lazy_leaf_fix_kernel<false><<<ch->g_fix, 256, 0, st>>>(V, j); }
  }
  const unsigned wg = (unsigned)(((long long)V.nC * 32 + 255) / 256);
  lazy_bound_kernel<<<wg, 256, 0, st>>>(V, bound_mant, (long long*)bound_exp2);
  ch->launches += ch->small ? 2 : 3 + 2 * V.cap;
  CU(cudaGetLastError());
  // lazy rounds: one start sector each, in order of decreasing bound
  for (int r = 0; r < ch->lazy_rounds; ++r) {
    int rc = chains_enqueue_levels(ch, 0, r, nullptr, 0, st);
    if (rc) return rc;
    if (cx) lazy_decide_kernel<true><<<wg, 256, 0, st>>>(V, r, r + 1, 0, accept, decided_by, n_sectors_evaluated, trace_mant, (long long*)trace_exp2, status);
    else    lazy_decide_kernel<false><<<wg, 256, 0, st>>>(V, r, r + 1, 0, accept, decided_by, n_sectors_evaluated, trace_mant, (long long*)trace_exp2, status);
    ch->launches += 1;
  }
  // whatever is still undecided (or accepted and incomplete): every remaining entry at once
  int rc = chains_enqueue_levels(ch, 1, 0, nullptr, 0, st);
  if (rc) return rc;
  if (cx) lazy_decide_kernel<true><<<wg, 256, 0, st>>>(V, ch->lazy_rounds, Q, 1, accept, decided_by, n_sectors_evaluated, trace_mant, (long long*)trace_exp2, status);
  else    lazy_decide_kernel<false><<<wg, 256, 0, st>>>(V, ch->lazy_rounds, Q, 1, accept, decided_by, n_sectors_evaluated, trace_mant, (long long*)trace_exp2, status);
  ch->launches += 1;
  CU(cudaGetLastError());
  return 0;
}

extern "C" int ctqmc_chains_commit(ctqmc_chains* ch, const int32_t* mask, void* cuda_stream) {
  if (!ch) return fail(CTQMC_ERR_ARG, "null chain set");
  CU(cudaSetDevice(ch->imp->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const LazyView& V = ch->V;
  const int* gate = mask ? (const int*)mask : V.p_accept;
  ch->launches = 0; ch->last_stream = st;
  int rc = chains_enqueue_levels(ch, 1, 0, gate, 1, st);   // entries the lazy evaluation never needed
  if (rc) return rc;
  lazy_commit_kernel<<<(V.nC + 127) / 128, 128, 0, st>>>(V, gate);
  ch->launches += 1;
  CU(cudaGetLastError());
  return 0;
}

extern "C" int ctqmc_chains_trace(ctqmc_chains* ch, double* mant, int64_t* exp2, void* cuda_stream) {
  if (!ch || !mant || !exp2) return fail(CTQMC_ERR_ARG, "null chain set or output");
  CU(cudaSetDevice(ch->imp->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const LazyView& V = ch->V;
  const unsigned wg = (unsigned)(((long long)V.nC * 32 + 255) / 256);
  if (V.imp.cplx) lazy_trace_kernel<true><<<wg, 256, 0, st>>>(V, mant, (long long*)exp2);
  else            lazy_trace_kernel<false><<<wg, 256, 0, st>>>(V, mant, (long long*)exp2);
  ch->launches = 1; ch->last_stream = st;
  CU(cudaGetLastError());
  return 0;
}

extern "C" int ctqmc_chains_stats(ctqmc_chains* ch, int64_t stats[4]) {
  if (!ch || !stats) return fail(CTQMC_ERR_ARG, "null chain set or stats");
  CU(cudaSetDevice(ch->imp->device));
  CU(cudaStreamSynchronize(ch->last_stream));
  unsigned long long np = 0;
  CU(cudaMemcpy(&np, ch->V.n_products, sizeof np, cudaMemcpyDeviceToHost));
  stats[0] = (int64_t)np; stats[1] = (int64_t)ch->bytes; stats[2] = ch->launches; stats[3] = ch->V.NN;
  return 0;
}
