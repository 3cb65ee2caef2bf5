// lanczos.cuh -- the vector kernels of the k-step Lanczos that supplies the spectral bounds Algorithm 1 takes as inputs
// (PAPER.md:L214 eps_0, eps_ub^uw; L232 "we refer to [30, 31]"; reading #5; SURVEY.md 8(f)-4 "GPU Lanczos bounds").
// Per step j:  w = H v_j  (the library's step kernel on one column),
//              alpha_j = v_j . w,   w <- w - alpha_j v_j - beta_{j-1} v_{j-1},   beta_j = ||w||,   v_{j+1} = w / beta_j
// Scalars never leave the device until the end: every CTA re-sums the same partial sums in the same fixed order, so alpha_j
// and beta_j are deterministic and identical in all CTAs.  Vectors are stored as column 0 of M x 2 row-major panels (even
// leading dimension: the TMA path of the fp64 step kernel needs it).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttdft {

constexpr int LZ_GRID = 592;     // CTAs of the vector kernels = number of partial sums
constexpr int LZ_LD = 2;

__device__ __forceinline__ double lz_block_sum(double x) {       // sum over the 256 threads of a CTA, result in every thread
  __shared__ double s[8];
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  __syncthreads();
  if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = x;
  __syncthreads();
  double t = 0.0;
  for (int i = 0; i < 8; ++i) t += s[i];
  return t;
}
__device__ __forceinline__ double lz_total(const double* __restrict__ part) {   // the LZ_GRID partial sums, fixed order
  double x = 0.0;
  for (int i = threadIdx.x; i < LZ_GRID; i += 256) x += part[i];
  return lz_block_sum(x);
}

// part[cta] = sum over this CTA's rows of a[i] * b[i]   (a == b: squared norm)
__global__ void __launch_bounds__(256) lz_dot_kernel(const double* __restrict__ a, const double* __restrict__ b, int64_t M, double* __restrict__ part) {
  double x = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < M; i += (int64_t)LZ_GRID * 256) x += a[i * LZ_LD] * b[i * LZ_LD];
  x = lz_block_sum(x);
  if (threadIdx.x == 0) part[blockIdx.x] = x;
}

// v = v0 / sqrt(total(part)),  vprev = 0;  status[0] = 1 if the norm is not positive
__global__ void __launch_bounds__(256) lz_start_kernel(const double* __restrict__ v0, int64_t M, const double* __restrict__ part, double* __restrict__ v,
                                                       double* __restrict__ vprev, int32_t* __restrict__ status) {
  const double n2 = lz_total(part);
  if (blockIdx.x == 0 && threadIdx.x == 0) status[0] = (n2 > 0.0) ? 0 : 1;
  const double nrm = sqrt(n2);
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < M; i += (int64_t)LZ_GRID * 256) {
    v[i * LZ_LD] = (n2 > 0.0) ? v0[i] / nrm : 0.0;
    vprev[i * LZ_LD] = 0.0;
  }
}

// alpha_j = total(part);  w <- w - alpha_j v - beta_{j-1} vprev;  part2[cta] = partial sums of w . w
__global__ void __launch_bounds__(256) lz_update_kernel(double* __restrict__ w, const double* __restrict__ v, const double* __restrict__ vprev, int64_t M,
                                                        const double* __restrict__ part, double* __restrict__ alpha, const double* __restrict__ beta,
                                                        int32_t j, double* __restrict__ part2) {
  const double aj = lz_total(part);
  const double bprev = (j > 0) ? beta[j - 1] : 0.0;
  if (blockIdx.x == 0 && threadIdx.x == 0) alpha[j] = aj;
  double x = 0.0;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < M; i += (int64_t)LZ_GRID * 256) {
    const double t = w[i * LZ_LD] - aj * v[i * LZ_LD] - bprev * vprev[i * LZ_LD];
    w[i * LZ_LD] = t;
    x += t * t;
  }
  x = lz_block_sum(x);
  if (threadIdx.x == 0) part2[blockIdx.x] = x;
}

// beta_j = sqrt(total(part2));  vprev <- v;  v <- w / beta_j  (v <- 0 if beta_j == 0: an invariant subspace was found)
__global__ void __launch_bounds__(256) lz_finish_kernel(const double* __restrict__ w, double* __restrict__ v, double* __restrict__ vprev, int64_t M,
                                                        const double* __restrict__ part2, double* __restrict__ beta, int32_t j) {
  const double bj = sqrt(lz_total(part2));
  if (blockIdx.x == 0 && threadIdx.x == 0) beta[j] = bj;
  for (int64_t i = (int64_t)blockIdx.x * 256 + threadIdx.x; i < M; i += (int64_t)LZ_GRID * 256) {
    vprev[i * LZ_LD] = v[i * LZ_LD];
    v[i * LZ_LD] = (bj > 0.0) ? w[i * LZ_LD] / bj : 0.0;
  }
}

}  // namespace ttdft
