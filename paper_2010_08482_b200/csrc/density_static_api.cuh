// ctqmc_density_batch_static (include/ctqmc.h): the density-matrix accumulation of density.cuh for callers that cannot call
// cudaMalloc (CUDA graph capture, serving loops, harnesses that forbid it).  The per-string scratch of density_kernel lives in
// a file-scope device array of fixed size instead of the handle's arena; the entry point allocates nothing on the device.
// Included at the end of ctqmc_api.cu (same translation unit as the array: cudaGetSymbolAddress needs that).
#pragma once
#include <mutex>

#include "density.cuh"

namespace ctqmc {
constexpr size_t kDensityStaticBytes = 64ull << 20;       // 64 MiB per GPU that loads the library, held until the process exits
static __device__ __align__(256) double g_density_static_scratch[kDensityStaticBytes / sizeof(double)];
static __device__ int g_density_static_work;              // the kernel's work counter (zeroed by every call, on its stream)
}  // namespace ctqmc

namespace {
constexpr int kStaticMaxDevices = 64;
double* g_density_static_ptr[kStaticMaxDevices] = {};
int* g_density_static_work_ptr[kStaticMaxDevices] = {};
std::mutex g_density_static_mu;

// Device address of the array on `device` (which must be current).  In host code the array's name is only a stand-in for the
// symbol, not an address a kernel can use: resolved once per device with cudaGetSymbolAddress.
int density_static_address(int device, double** out, int** work) {
  if (device < 0 || device >= kStaticMaxDevices) return fail(CTQMC_ERR_ARG, "device ordinal %d out of range for the static scratch table", device);
  std::lock_guard<std::mutex> lock(g_density_static_mu);
  if (!g_density_static_ptr[device]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_density_static_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return fail(CTQMC_ERR_CUDA, "cudaGetSymbolAddress(static density scratch) on device %d: %s", device, cudaGetErrorString(e));
    }
    void* w = nullptr;
    e = cudaGetSymbolAddress(&w, g_density_static_work);
    if (e != cudaSuccess || !w) {
      cudaGetLastError();
      return fail(CTQMC_ERR_CUDA, "cudaGetSymbolAddress(static density work counter) on device %d: %s", device, cudaGetErrorString(e));
    }
    g_density_static_work_ptr[device] = (int*)w;
    g_density_static_ptr[device] = (double*)p;
  }
  *out = g_density_static_ptr[device]; *work = g_density_static_work_ptr[device];
  return 0;
}
}  // namespace

extern "C" int64_t ctqmc_density_static_limit(void) { return (int64_t)kDensityStaticBytes; }

extern "C" int ctqmc_density_batch_static(ctqmc_impurity* h, double beta, const ctqmc_batch* batch, const double* w_mant,
                                          const int64_t* w_exp2, const int32_t* status, const double* weight, double* rho,
                                          void* cuda_stream) {
  int rc = check_batch_args(h, beta, batch);
  if (rc) return rc;
  const long long B = batch->n_configs;
  if (B == 0) return 0;
  if (!w_mant || !w_exp2 || !status || !rho) return fail(CTQMC_ERR_ARG, "null input (w_mant, w_exp2, status) or output (rho)");
  if (h->dev.dmax > kLzMaxDim)
    return fail(CTQMC_ERR_UNSUPPORTED, "the density-matrix estimator keeps every prefix product: sector dimension %d exceeds %d", h->dev.dmax, kLzMaxDim);
  int Lcap = effective_max_len(batch);
  if (Lcap < 1) Lcap = 1;
  const int es = h->dev.cplx ? 2 : 1;
  const size_t slot_bytes = (size_t)density_slot_doubles(h->dev.dmax, Lcap, es) * sizeof(double);
  if (slot_bytes > kDensityStaticBytes)
    return fail(CTQMC_ERR_UNSUPPORTED,
                "ctqmc_density_batch_static: the prefix products of one string (max_len %d x d_max %d: %zu bytes) exceed the static scratch of %zu bytes; "
                "use ctqmc_density_batch", Lcap, h->dev.dmax, slot_bytes, kDensityStaticBytes);
  CU(cudaSetDevice(h->device));
  double* scratch = nullptr;
  int* work = nullptr;
  rc = density_static_address(h->device, &scratch, &work);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  long long grid = 2LL * h->sm_count;
  const long long nS = B * h->dev.Q, fit = (long long)(kDensityStaticBytes / slot_bytes);
  if (grid > nS) grid = nS;
  if (grid > fit) grid = fit;
  // Nothing in the scratch itself has to start at zero: every element a string reads (prefix products, carried matrices, exponent and
  // sector tables of its slot) it has written before, and the product tiles are bounds-guarded.  The array keeps the last
  // call's contents; two calls that overlap on the GPU (different streams) would share slots and race.
  DensityParams dp;
  dp.imp = h->dev; dp.bv = make_view(batch, beta, 0, B, Lcap); dp.w_mant = w_mant; dp.w_exp2 = (const long long*)w_exp2; dp.status = status;
  dp.weight = weight; dp.rho = rho; dp.rho_off = h->d_rho_off; dp.scratch = scratch; dp.slot_doubles = (long long)(slot_bytes / sizeof(double));
  dp.ldm = h->dev.dmax; dp.Lcap = Lcap; dp.work = work;
  CU(cudaMemsetAsync(work, 0, sizeof(int), st));          // the one word that must start at zero
  if (h->dev.cplx) density_kernel<true><<<(unsigned)grid, kLzThreads, 0, st>>>(dp);
  else             density_kernel<false><<<(unsigned)grid, kLzThreads, 0, st>>>(dp);
  h->last_stream = st; h->last_launches = 1;
  CU(cudaGetLastError());
  return 0;
}
