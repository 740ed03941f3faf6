// Host side of ctqmc_density_batch / ctqmc_density_size (include/ctqmc.h): scratch sizing from host-known bounds and the one
// launch of density.cuh.  Included at the end of ctqmc_api.cu.
#pragma once
#include "density.cuh"

extern "C" int64_t ctqmc_density_size(const ctqmc_impurity* h) { return h ? (int64_t)h->rho_len : 0; }

extern "C" int ctqmc_density_batch(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, const double* w_mant, const int64_t* w_exp2,
                                   const int32_t* status, const double* weight, double* rho, void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!w_mant || !w_exp2 || !status || !rho) return fail(CTQMC_ERR_ARG, "null input (w_mant, w_exp2, status) or output (rho)");
  if (h->dev.dmax > kLzMaxDim)
    return fail(CTQMC_ERR_UNSUPPORTED, "the density-matrix estimator keeps every prefix product: sector dimension %d exceeds %d", h->dev.dmax, kLzMaxDim);
  CU(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int Lcap = effective_max_len(batch);
  if (Lcap < 1) Lcap = 1;
  const int es = h->dev.cplx ? 2 : 1;
  const size_t slot_bytes = (size_t)density_slot_doubles(h->dev.dmax, Lcap, es) * sizeof(double);
  const long long nS = B * h->dev.Q;
  long long grid = 2LL * h->sm_count;
  if (grid > nS) grid = nS;
  // scratch: one slot per persistent CTA, from the handle's arena (grown before anything is enqueued, unless its size is fixed)
  Arena& a = h->arena;
  size_t want = (size_t)grid * slot_bytes + 256;
  if (want > a.cap && a.fixed_bytes == 0) {
    size_t free_b = 0, total_b = 0;
    CU(cudaMemGetInfo(&free_b, &total_b));
    size_t limit = (size_t)(0.5 * (double)(free_b + a.cap));
    if (h->scratch_limit > 0 && (size_t)h->scratch_limit < limit) limit = (size_t)h->scratch_limit;
    const size_t target = want < limit ? want : limit;
    if (target > a.cap) {
      CU(cudaDeviceSynchronize());
      cudaFree(a.base); a.base = nullptr; a.cap = 0;
      cudaError_t e = cudaMalloc((void**)&a.base, target);
      if (e != cudaSuccess) { cudaGetLastError(); return fail(CTQMC_ERR_OOM, "cannot allocate a scratch arena of %zu bytes", target); }
      a.cap = target;
      CU(cudaMemset(a.base, 0, a.cap));
    }
  }
  if (want > a.cap) grid = (long long)((a.cap > 256 ? a.cap - 256 : 0) / slot_bytes);
  if (grid < 1)
    return fail(CTQMC_ERR_OOM, "the scratch arena (%zu bytes) cannot hold the prefix products of one string (%zu bytes)", a.cap, slot_bytes);
  DensityParams dp;
  dp.imp = h->dev; dp.bv = make_view(batch, beta, 0, B, Lcap); dp.w_mant = w_mant; dp.w_exp2 = (const long long*)w_exp2; dp.status = status;
  dp.weight = weight; dp.rho = rho; dp.rho_off = h->d_rho_off; dp.scratch = (double*)a.base; dp.slot_doubles = (long long)(slot_bytes / sizeof(double));
  dp.ldm = h->dev.dmax; dp.Lcap = Lcap;
  dp.work = reinterpret_cast<int*>(a.base + (size_t)grid * slot_bytes);        // the 256 spare bytes behind the slots
  CU(cudaMemsetAsync(dp.work, 0, sizeof(int), st));
  if (h->dev.cplx) density_kernel<true><<<(unsigned)grid, kLzThreads, 0, st>>>(dp);
  else             density_kernel<false><<<(unsigned)grid, kLzThreads, 0, st>>>(dp);
  h->last_stream = st; h->last_launches = 1;
  CU(cudaGetLastError());
  return 0;
}
