// cholesky.cuh -- the small dense fp64 pieces of the Cholesky-QR orthonormalisation (Algorithm 1 step 2,
// PAPER.md:L226 "X_F = Orth(X)", L230 "Gram-Schmidt orthogonalization procedure"):
//   G = X^T X  (ttdft_gram)  ->  G = L L^T  (potrf below)  ->  R^-1 = L^-T  (trinv below)  ->  X_F = X R^-1  (ttdft_rotate)
// For full-rank X the Q of Cholesky-QR is the Q of Gram-Schmidt (R is the unique upper-triangular factor with a
// positive diagonal); the O(M n^2) work runs on the tensor cores, what is left here is O(n^3) on an n x n matrix
// (23 GFLOP at n = 4,096) and is written for clarity, not speed: right-looking blocked Cholesky with 64-wide panels.
// Row-major, lower triangle referenced and overwritten; the strict upper triangle is never touched.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttdft {

constexpr int CH_NB = 64;
constexpr int CH_TILE_BYTES = CH_NB * (CH_NB + 1) * 8;   // one padded 64 x 64 fp64 tile in (dynamic) shared memory
typedef double ch_tile_t[CH_NB][CH_NB + 1];

// Diagonal block: A[k0:k0+nbk, k0:k0+nbk] = L_kk L_kk^T, unblocked, one CTA of 256 threads.
// flag[0] = 1 + (index of the first non-positive pivot) if the matrix is not positive definite.
__global__ void __launch_bounds__(256) ch_potf2_kernel(double* __restrict__ A, int64_t ld, int32_t k0, int32_t nbk, int32_t* __restrict__ flag) {
  __shared__ double s[CH_NB][CH_NB + 1];
  const int tid = threadIdx.x;
  for (int e = tid; e < nbk * nbk; e += 256) {
    const int r = e / nbk, c = e % nbk;
    s[r][c] = (c <= r) ? A[(int64_t)(k0 + r) * ld + k0 + c] : 0.0;
  }
  __syncthreads();
  for (int j = 0; j < nbk; ++j) {
    if (tid == 0) {
      const double d = s[j][j];
      if (!(d > 0.0)) { s[j][j] = 1.0; if (flag[0] == 0) flag[0] = 1 + k0 + j; }
      else s[j][j] = sqrt(d);
    }
    __syncthreads();
    const double ljj = s[j][j];
    for (int r = j + 1 + tid; r < nbk; r += 256) s[r][j] /= ljj;
    __syncthreads();
    // trailing update of the lower triangle: s[r][c] -= s[r][j] * s[c][j], j < c <= r
    const int m = nbk - j - 1;
    for (int e = tid; e < m * m; e += 256) {
      const int r = j + 1 + e / m, c = j + 1 + e % m;
      if (c <= r) s[r][c] -= s[r][j] * s[c][j];
    }
    __syncthreads();
  }
  for (int e = tid; e < nbk * nbk; e += 256) {
    const int r = e / nbk, c = e % nbk;
    if (c <= r) A[(int64_t)(k0 + r) * ld + k0 + c] = s[r][c];
  }
}

// Panel below the diagonal block: A[i, k0:k0+nbk] <- A[i, k0:k0+nbk] L_kk^-T for rows i >= k0+nbk.
// One CTA per 64 rows, one thread per row (forward substitution along the row), L_kk in shared memory.
__global__ void __launch_bounds__(64) ch_trsm_kernel(double* __restrict__ A, int64_t ld, int32_t n, int32_t k0, int32_t nbk) {
  __shared__ double L[CH_NB][CH_NB + 1];
  for (int e = threadIdx.x; e < nbk * nbk; e += 64) {
    const int r = e / nbk, c = e % nbk;
    L[r][c] = (c <= r) ? A[(int64_t)(k0 + r) * ld + k0 + c] : 0.0;
  }
  __syncthreads();
  const int64_t i = (int64_t)k0 + nbk + (int64_t)blockIdx.x * 64 + threadIdx.x;
  if (i >= n) return;
  double* a = A + i * ld + k0;
  double x[CH_NB];
#pragma unroll 1
  for (int c = 0; c < nbk; ++c) {
    double v = a[c];
    for (int t = 0; t < c; ++t) v -= x[t] * L[c][t];
    x[c] = v / L[c][c];
  }
  for (int c = 0; c < nbk; ++c) a[c] = x[c];
}

// Trailing update: A[i, j] -= sum_t P[i, t] P[j, t] for k1 <= j <= i < n (lower triangle), P = A[:, k0:k0+nbk], k1 = k0+nbk.
// grid (tiles, tiles) of 64 x 64 output tiles (upper tiles exit), 256 threads, each a 4 x 4 register tile.
__global__ void __launch_bounds__(256) ch_syrk_kernel(double* __restrict__ A, int64_t ld, int32_t n, int32_t k0, int32_t nbk) {
  if (blockIdx.y > blockIdx.x) return;                       // tile column > tile row: strictly upper
  extern __shared__ double ch_smem[];                        // 2 tiles (dynamic: 2 * CH_TILE_BYTES)
  ch_tile_t& Pi = *reinterpret_cast<ch_tile_t*>(ch_smem);
  ch_tile_t& Pj = *reinterpret_cast<ch_tile_t*>(ch_smem + CH_NB * (CH_NB + 1));
  const int32_t k1 = k0 + nbk;
  const int64_t i0 = (int64_t)k1 + (int64_t)blockIdx.x * 64, j0 = (int64_t)k1 + (int64_t)blockIdx.y * 64;
  for (int e = threadIdx.x; e < 64 * nbk; e += 256) {
    const int r = e / nbk, t = e % nbk;
    Pi[r][t] = (i0 + r < n) ? A[(i0 + r) * ld + k0 + t] : 0.0;
    Pj[r][t] = (j0 + r < n) ? A[(j0 + r) * ld + k0 + t] : 0.0;
  }
  __syncthreads();
  const int tr = (threadIdx.x >> 4) * 4, tc = (threadIdx.x & 15) * 4;
  double acc[4][4] = {};
  for (int t = 0; t < nbk; ++t) {
    double a[4], b[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { a[u] = Pi[tr + u][t]; b[u] = Pj[tc + u][t]; }
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int w = 0; w < 4; ++w) acc[u][w] = fma(a[u], b[w], acc[u][w]);
  }
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int64_t i = i0 + tr + u, j = j0 + tc + w;
      if (i < n && j < n && j <= i) A[i * ld + j] -= acc[u][w];
    }
}

// R^-1 = L^-T, upper triangular, row-major n x n (ldr); the strict lower triangle of Rinv must be zero on entry.
// W = L^-1 is computed by block columns: one CTA (256 threads) per block column k walks down the block rows
//   W_ik = L_ii^-1 (delta_ik I - sum_{j=k}^{i-1} L_ij W_jk)
// and stores W_ik transposed: Rinv[k0 + c, i0 + r] = W_ik[r, c].  Earlier blocks W_jk are re-read from Rinv (L2).
__global__ void __launch_bounds__(256) ch_trinv_kernel(const double* __restrict__ A, int64_t ld, int32_t n, double* __restrict__ Rinv, int64_t ldr) {
  extern __shared__ double ch_smem[];                        // 3 tiles (dynamic: 3 * CH_TILE_BYTES)
  ch_tile_t& T = *reinterpret_cast<ch_tile_t*>(ch_smem);
  ch_tile_t& Lb = *reinterpret_cast<ch_tile_t*>(ch_smem + CH_NB * (CH_NB + 1));
  ch_tile_t& Wb = *reinterpret_cast<ch_tile_t*>(ch_smem + 2 * CH_NB * (CH_NB + 1));
  const int32_t nb = (n + CH_NB - 1) / CH_NB;
  const int32_t k = blockIdx.x, k0 = k * CH_NB, nk = min(CH_NB, n - k0);
  const int tid = threadIdx.x;
  const int tr = (tid >> 4) * 4, tc = (tid & 15) * 4;
  for (int32_t i = k; i < nb; ++i) {
    const int32_t i0 = i * CH_NB, ni = min(CH_NB, n - i0);
    double acc[4][4] = {};
    for (int32_t j = k; j < i; ++j) {
      const int32_t j0 = j * CH_NB;                          // full block (j < i <= nb-1)
      __syncthreads();
      for (int e = tid; e < CH_NB * CH_NB; e += 256) {
        const int r = e / CH_NB, c = e % CH_NB;
        Lb[r][c] = (r < ni) ? A[(int64_t)(i0 + r) * ld + j0 + c] : 0.0;            // L_ij[r][c]
        Wb[r][c] = (c < nk) ? Rinv[(int64_t)(k0 + c) * ldr + j0 + r] : 0.0;        // W_jk[r][c]
      }
      __syncthreads();
      for (int t = 0; t < CH_NB; ++t) {
        double a[4], b[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { a[u] = Lb[tr + u][t]; b[u] = Wb[t][tc + u]; }
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
          for (int w = 0; w < 4; ++w) acc[u][w] = fma(a[u], b[w], acc[u][w]);
      }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int w = 0; w < 4; ++w) T[tr + u][tc + w] = ((i == k && tr + u == tc + w) ? 1.0 : 0.0) - acc[u][w];
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
      const int r = e / CH_NB, c = e % CH_NB;
      Lb[r][c] = (r < ni && c <= r) ? A[(int64_t)(i0 + r) * ld + i0 + c] : ((r == c) ? 1.0 : 0.0);   // L_ii, identity-padded
    }
    __syncthreads();
    if (tid < CH_NB) {                                       // forward substitution, one thread per column of T
      const int c = tid;
      for (int r = 0; r < CH_NB; ++r) {
        double v = T[r][c];
        for (int t = 0; t < r; ++t) v -= Lb[r][t] * T[t][c];
        T[r][c] = v / Lb[r][r];
      }
    }
    __syncthreads();
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
      const int c = e / CH_NB, r = e % CH_NB;                // consecutive threads -> consecutive columns of Rinv
      if (r < ni && c < nk) Rinv[(int64_t)(k0 + c) * ldr + i0 + r] = T[r][c];
    }
    __threadfence_block();
  }
}

// R^-1 of two passes combined is not needed: the second pass rotates the already rotated block.

}  // namespace ttdft
