// Device-resident block-sparse operator store ("matrices stay on the GPU").
// Load-time kernels: re-layout of the caller's column-major blocks into the padded row-major store the MMA loops read,
// per-row squared norms (Frobenius tables for the S=1 bound) and the spectral norm of every block by power iteration.
#pragma once
#include "common.cuh"

namespace ctqmc {

// in: column-major rows x cols (ES doubles per element) -> out: row-major, leading dimension ld, zero padding untouched.
template <int ES>
__global__ void relayout_kernel(const double* __restrict__ raw, const long long* __restrict__ raw_off,
                                const BlkDesc* __restrict__ blks, double* __restrict__ store) {
  __shared__ double tile[32][33 * ES];
  const BlkDesc bd = blks[blockIdx.z];
  const double* in = raw + raw_off[blockIdx.z] * ES;
  double* out = store + bd.off;
  for (int m0 = blockIdx.y * 32; m0 < bd.rows; m0 += gridDim.y * 32)
    for (int k0 = blockIdx.x * 32; k0 < bd.cols; k0 += gridDim.x * 32) {
      for (int kk = threadIdx.y; kk < 32; kk += blockDim.y) {
        int m = m0 + threadIdx.x, k = k0 + kk;
        if (m < bd.rows && k < bd.cols)
          for (int c = 0; c < ES; ++c) tile[kk][threadIdx.x * ES + c] = in[((size_t)k * bd.rows + m) * ES + c];
      }
      __syncthreads();
      for (int mm = threadIdx.y; mm < 32; mm += blockDim.y) {
        int m = m0 + mm, k = k0 + threadIdx.x;
        if (m < bd.rows && k < bd.cols)
          for (int c = 0; c < ES; ++c) out[((size_t)m * bd.ld + k) * ES + c] = tile[threadIdx.x][mm * ES + c];
      }
      __syncthreads();
    }
}

// rownorm2[blk][m] = sum_k |F_mk|^2 ; one warp per row.
template <int ES>
__global__ void rownorm_kernel(const BlkDesc* __restrict__ blks, const double* __restrict__ store, double* __restrict__ rownorm2) {
  const BlkDesc bd = blks[blockIdx.y];
  const int lane = threadIdx.x & 31;
  for (int m = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); m < bd.rows; m += gridDim.x * (blockDim.x >> 5)) {
    const double* r = store + bd.off + (size_t)m * bd.ld * ES;
    double ss = 0.0;
    for (int k = lane; k < bd.cols * ES; k += 32) ss += r[k] * r[k];
    ss = warp_sum(ss);
    if (lane == 0) rownorm2[bd.rn_off + m] = ss;
  }
}

// Power iteration on F^H F (spectral norm).  u = F v ; w = F^H u ; v = w / ||w|| ; sigma = ||F v|| at the last pass.
// For c / c^dag blocks F^H F is a projector (all non-zero singular values are 1), so one pass is already exact.
template <int ES>
__global__ void pi_init_kernel(const BlkDesc* __restrict__ blks, const long long* __restrict__ v_off, double* __restrict__ v) {
  const BlkDesc bd = blks[blockIdx.x];
  double* vb = v + v_off[blockIdx.x] * ES;
  for (int k = threadIdx.x; k < bd.cols; k += blockDim.x) {
    vb[k * ES] = 1.0 + 0.5 * sin(0.7 * k + 0.3 * blockIdx.x);
    if (ES == 2) vb[k * ES + 1] = 0.25 * cos(1.3 * k);
  }
}

template <int ES>
__global__ void pi_fv_kernel(const BlkDesc* __restrict__ blks, const double* __restrict__ store,
                             const long long* __restrict__ v_off, const double* __restrict__ v, double* __restrict__ u) {
  const BlkDesc bd = blks[blockIdx.y];
  const int lane = threadIdx.x & 31;
  const double* vb = v + v_off[blockIdx.y] * ES;
  for (int m = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); m < bd.rows; m += gridDim.x * (blockDim.x >> 5)) {
    const double* r = store + bd.off + (size_t)m * bd.ld * ES;
    double sr = 0.0, si = 0.0;
    for (int k = lane; k < bd.cols; k += 32) {
      if (ES == 1) sr += r[k] * vb[k];
      else { double ar = r[2 * k], ai = r[2 * k + 1], br = vb[2 * k], bi = vb[2 * k + 1]; sr += ar * br - ai * bi; si += ar * bi + ai * br; }
    }
    sr = warp_sum(sr); si = warp_sum(si);
    if (lane == 0) { u[(bd.rn_off + m) * ES] = sr; if (ES == 2) u[(bd.rn_off + m) * ES + 1] = si; }
  }
}

template <int ES>
__global__ void pi_fhu_kernel(const BlkDesc* __restrict__ blks, const double* __restrict__ store,
                              const long long* __restrict__ v_off, const double* __restrict__ u, double* __restrict__ v) {
  const BlkDesc bd = blks[blockIdx.y];
  double* vb = v + v_off[blockIdx.y] * ES;
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < bd.cols; k += gridDim.x * blockDim.x) {
    double sr = 0.0, si = 0.0;
    for (int m = 0; m < bd.rows; ++m) {
      const double* e = store + bd.off + ((size_t)m * bd.ld + k) * ES;
      if (ES == 1) sr += e[0] * u[bd.rn_off + m];
      else { double ar = e[0], ai = -e[1], br = u[(bd.rn_off + m) * 2], bi = u[(bd.rn_off + m) * 2 + 1]; sr += ar * br - ai * bi; si += ar * bi + ai * br; }
    }
    vb[k * ES] = sr; if (ES == 2) vb[k * ES + 1] = si;
  }
}

// one CTA per block: nrm = ||x||_2 over n*ES doubles; optionally x /= nrm; optionally out[blk] = nrm
__global__ void pi_norm_kernel(const BlkDesc* __restrict__ blks, const long long* __restrict__ off, int use_rows, int ES,
                               double* __restrict__ x, int do_scale, double* __restrict__ out) {
  __shared__ double red[32];
  __shared__ double s_nrm;
  const BlkDesc bd = blks[blockIdx.x];
  const long long o = (use_rows ? bd.rn_off : off[blockIdx.x]) * ES;
  const int n = (use_rows ? bd.rows : bd.cols) * ES;
  double mx = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) mx = fmax(mx, fabs(x[o + i]));
  mx = warp_max(mx);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
  __syncthreads();
  if (threadIdx.x == 0) { double m = 0.0; for (int w = 0; w < (blockDim.x >> 5); ++w) m = fmax(m, red[w]); s_nrm = m; }
  __syncthreads();
  mx = s_nrm;
  __syncthreads();
  double ss = 0.0;
  if (mx > 0.0) for (int i = threadIdx.x; i < n; i += blockDim.x) { double t = x[o + i] / mx; ss += t * t; }
  ss = warp_sum(ss);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
  __syncthreads();
  if (threadIdx.x == 0) { double s = 0.0; for (int w = 0; w < (blockDim.x >> 5); ++w) s += red[w]; s_nrm = mx * sqrt(s); }
  __syncthreads();
  const double nrm = s_nrm;
  if (do_scale && nrm > 0.0) for (int i = threadIdx.x; i < n; i += blockDim.x) x[o + i] /= nrm;
  if (out && threadIdx.x == 0) out[blockIdx.x] = nrm;
}

}  // namespace ctqmc

namespace ctqmc {

// Spectral-norm guard (reading A1).  Power iteration approaches sigma_max from BELOW; a bound built from an
// under-estimate would not be a bound.  With v the normalised iterate, u = F v, sigma = ||u|| and w = F^H u, the iteration has
// converged iff w = sigma^2 v.  One CTA per block: the iterate is accepted only if the residual r = w - sigma^2 v satisfies
// ||r|| <= 1e-13 sigma^2 (c / c^dag blocks converge exactly after one step: F^H F is a projector, pin P10), and then as
// sqrt(sigma^2 + ||r||), which covers the eigenvalue of F^H F the residual localises.  Everything else -- slow convergence
// (near-degenerate top singular values), or sigma = 0 from a start vector in ker F -- gets need[b] = 1 and the rigorous
// upper estimate of sigma_upper_kernel (which is 0 for an all-zero block).
template <int ES>
__global__ void sigma_check_kernel(const BlkDesc* __restrict__ blks, const long long* __restrict__ v_off,
                                   const double* __restrict__ v, const double* __restrict__ w,
                                   double* __restrict__ sigma, int* __restrict__ need) {
  __shared__ double red[8];
  const BlkDesc bd = blks[blockIdx.x];
  const double s2 = sigma[blockIdx.x] * sigma[blockIdx.x];
  const double* vb = v + v_off[blockIdx.x] * ES;
  const double* wb = w + v_off[blockIdx.x] * ES;
  double r2 = 0.0;
  for (int i = threadIdx.x; i < bd.cols * ES; i += blockDim.x) { const double d = wb[i] - s2 * vb[i]; r2 += d * d; }
  r2 = warp_sum(r2);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = r2;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) t += red[i];
    const double rn = sqrt(t);
    const bool ok = s2 > 0.0 && rn <= 1e-13 * s2;
    need[blockIdx.x] = ok ? 0 : 1;
    if (ok) sigma[blockIdx.x] = sqrt(s2 + rn) * (1.0 + 4e-16);
  }
}

// For blocks whose iteration has not converged: sigma <- max(sigma, min(||F||_F, sqrt(||F||_1 ||F||_inf))), a rigorous upper
// bound of the spectral norm.  One CTA per block; converged blocks return at once.
template <int ES>
__global__ void sigma_upper_kernel(const BlkDesc* __restrict__ blks, const double* __restrict__ store,
                                   const double* __restrict__ rownorm2, const int* __restrict__ need, double* __restrict__ sigma) {
  __shared__ double red[3][8];
  if (!need[blockIdx.x]) return;
  const BlkDesc bd = blks[blockIdx.x];
  const double* F = store + bd.off;
  double fro2 = 0.0, ninf = 0.0, n1 = 0.0;
  for (int m = threadIdx.x; m < bd.rows; m += blockDim.x) {
    fro2 += rownorm2[bd.rn_off + m];
    double s = 0.0;
    for (int k = 0; k < bd.cols; ++k) {
      const double* e = F + ((size_t)m * bd.ld + k) * ES;
      s += (ES == 1) ? fabs(e[0]) : hypot(e[0], e[ES - 1]);
    }
    ninf = fmax(ninf, s);
  }
  for (int k = threadIdx.x; k < bd.cols; k += blockDim.x) {
    double s = 0.0;
    for (int m = 0; m < bd.rows; ++m) {
      const double* e = F + ((size_t)m * bd.ld + k) * ES;
      s += (ES == 1) ? fabs(e[0]) : hypot(e[0], e[ES - 1]);
    }
    n1 = fmax(n1, s);
  }
  fro2 = warp_sum(fro2); ninf = warp_max(ninf); n1 = warp_max(n1);
  if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = fro2; red[1][threadIdx.x >> 5] = ninf; red[2][threadIdx.x >> 5] = n1; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0, c = 0.0;
    for (int i = 0; i < (int)(blockDim.x >> 5); ++i) { a += red[0][i]; b = fmax(b, red[1][i]); c = fmax(c, red[2][i]); }
    const double upper = fmin(sqrt(a), sqrt(b * c)) * (1.0 + 1e-12);
    sigma[blockIdx.x] = fmax(sigma[blockIdx.x], upper);
  }
}

}  // namespace ctqmc
