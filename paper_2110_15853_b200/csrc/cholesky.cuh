// cholesky.cuh -- the small dense fp64 pieces of the Cholesky-QR orthonormalisation (Algorithm 1 step 2,
// PAPER.md:L226 "X_F = Orth(X)", L230 "Gram-Schmidt orthogonalization procedure"):
//   G = X^T X  (ttdft_gram)  ->  G = L L^T  (potf2/panel/syrk below)  ->  R^-1 = L^-T  (level/transpose below)  ->  X_F = X R^-1  (ttdft_rotate)
// For full-rank X the Q of Cholesky-QR is the Q of Gram-Schmidt (R is the unique upper-triangular factor with a
// positive diagonal); the O(M n^2) work runs on the tensor cores, what is left here is O(n^3) on an n x n matrix
// (23 GFLOP at n = 4,096) right-looking blocked Cholesky with 64-wide panels, the block products on the fp64 tensor cores.
// Row-major, lower triangle referenced and overwritten; the strict upper triangle is never touched.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttdft {

constexpr int CH_NB = 64;
constexpr int CH_TILE_BYTES = CH_NB * (CH_NB + 1) * 8;   // one padded 64 x 64 fp64 tile in (dynamic) shared memory
typedef double ch_tile_t[CH_NB][CH_NB + 1];
// The three block products (panel, trailing update, inverse levels) run on the fp64 tensor cores (mma.sync m8n8k4 -> DMMA): one
// 64 x 64 x 64 product per CTA, 8 warps x (16 rows x 32 columns), operands in shared-memory tiles of row stride 68 doubles
// (fragment loads -- lane l reads [l / 4][l % 4] of an 8 x 4 block, or its transpose -- are then bank-conflict free).
// Before: 4 x 4 register tiles on the fp64 ALUs, bound by their shared-memory reads (one load per two FMAs): 5.6 TFLOP/s.
constexpr int CH_LD = CH_NB + 4;
constexpr int CH_GEMM_SMEM = 2 * CH_NB * CH_LD * 8;      // two operand tiles
typedef double ch_gtile_t[CH_NB][CH_LD];
__device__ __forceinline__ void ch_dmma(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// acc += A[wr.., 0..kmax) * B, for this warp's 16 x 32 piece at (wr, wc); BT: B(k, j) = Bs[j][k], else Bs[k][j].  kmax % 4 == 0.
// acc[mi][ni][e]: row wr + 8 mi + lane / 4, column wc + 8 ni + 2 (lane % 4) + e.
template <bool BT>
__device__ __forceinline__ void ch_warp_mma(const ch_gtile_t& As, const ch_gtile_t& Bs, int kmax, int wr, int wc, int lane,
                                            double (&acc)[2][4][2]) {
  const int lr = lane >> 2, lc = lane & 3;
  for (int k = 0; k < kmax; k += 4) {
    double a[2], b[4];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi) a[mi] = As[wr + 8 * mi + lr][k + lc];
#pragma unroll
    for (int ni = 0; ni < 4; ++ni) b[ni] = BT ? Bs[wc + 8 * ni + lr][k + lc] : Bs[k + lc][wc + 8 * ni + lr];
#pragma unroll
    for (int mi = 0; mi < 2; ++mi)
#pragma unroll
      for (int ni = 0; ni < 4; ++ni) ch_dmma(acc[mi][ni][0], acc[mi][ni][1], a[mi], b[ni]);
  }
}

// Diagonal block: A[k0:k0+nbk, k0:k0+nbk] = L_kk L_kk^T, unblocked, one CTA of 256 threads.
// flag[0] = 1 + (index of the first non-positive pivot) if the matrix is not positive definite.
// Also W[k0.., k0..] = L_kk^-1 (lower triangular), which turns the panel solve into a product and seeds the inverse.
__global__ void __launch_bounds__(256) ch_potf2_kernel(double* __restrict__ A, int64_t ld, int32_t k0, int32_t nbk, int32_t* __restrict__ flag,
                                                       double* __restrict__ W, int64_t ldw) {
  extern __shared__ double ch_smem[];                        // 2 tiles (dynamic: 2 * CH_TILE_BYTES): L_kk and its inverse
  ch_tile_t& s = *reinterpret_cast<ch_tile_t*>(ch_smem);
  ch_tile_t& w = *reinterpret_cast<ch_tile_t*>(ch_smem + CH_NB * (CH_NB + 1));
  const int tid = threadIdx.x;
  const int tx = tid & 15, ty = tid >> 4;                    // 16 x 16 threads over the tile (no integer divisions in the loops)
  __shared__ double dg[CH_NB];                               // the diagonal of L_kk
  for (int r = ty; r < nbk; r += 16)
    for (int c = tx; c < nbk; c += 16) s[r][c] = (c <= r) ? A[(int64_t)(k0 + r) * ld + k0 + c] : 0.0;
  __syncthreads();
  for (int j = 0; j < nbk; ++j) {
    // column j: every thread takes the pivot from s[j][j] (not written in this phase), one of them records it
    const double d = s[j][j];
    const bool ok = d > 0.0;
    const double ljj = ok ? sqrt(d) : 1.0;
    if (tid == 0) {
      dg[j] = ljj;
      if (!ok && flag[0] == 0) flag[0] = 1 + k0 + j;
    }
    for (int r = j + 1 + tid; r < nbk; r += 256) s[r][j] /= ljj;
    __syncthreads();
    // trailing update of the lower triangle: s[r][c] -= s[r][j] * s[c][j], j < c <= r
    for (int r = j + 1 + ty; r < nbk; r += 16) {
      const double lrj = s[r][j];
      for (int c = j + 1 + tx; c <= r; c += 16) s[r][c] -= lrj * s[c][j];
    }
    __syncthreads();
  }
  if (tid < nbk) s[tid][tid] = dg[tid];
  __syncthreads();
  for (int r = ty; r < nbk; r += 16)
    for (int c = tx; c <= r && c < nbk; c += 16) A[(int64_t)(k0 + r) * ld + k0 + c] = s[r][c];
  // W_kk = L_kk^-1: forward substitution on the identity, four threads per column (partial sums over t = q mod 4, combined by
  // two shuffles; the four threads of a column sit in one warp, so a warp barrier orders the row just written), then stored
  {
    const int c = tid >> 2, q = tid & 3;                     // 256 threads = 64 columns x 4
    for (int r = 0; r < nbk; ++r) {
      const bool on = (c < nbk && r >= c);
      double v = 0.0;
      if (on)
        for (int t = c + q; t < r; t += 4) v -= s[r][t] * w[t][c];
      v += __shfl_xor_sync(0xffffffffu, v, 1);               // all lanes take part, whatever their column
      v += __shfl_xor_sync(0xffffffffu, v, 2);
      if (on && q == 0) w[r][c] = (v + ((r == c) ? 1.0 : 0.0)) / s[r][r];
      __syncwarp();
    }
  }
  __syncthreads();
  for (int r = ty; r < nbk; r += 16)
    for (int c = tx; c <= r && c < nbk; c += 16) W[(int64_t)(k0 + r) * ldw + k0 + c] = w[r][c];
}

// Panel below the diagonal block: A[i, k0:k0+nbk] <- A[i, k0:k0+nbk] L_kk^-T = A[i, :] W_kk^T for rows i >= k0+nbk.
// One CTA (256 threads, DMMA) per 64 rows; dynamic smem CH_GEMM_SMEM.
__global__ void __launch_bounds__(256) ch_panel_kernel(double* __restrict__ A, int64_t ld, int32_t n, int32_t k0, int32_t nbk,
                                                       const double* __restrict__ W, int64_t ldw) {
  extern __shared__ double ch_smem[];
  ch_gtile_t& As = *reinterpret_cast<ch_gtile_t*>(ch_smem);
  ch_gtile_t& Ws = *reinterpret_cast<ch_gtile_t*>(ch_smem + CH_NB * CH_LD);
  const int64_t i0 = (int64_t)k0 + nbk + (int64_t)blockIdx.x * 64;
  for (int e = threadIdx.x; e < CH_NB * CH_NB; e += 256) {
    const int r = e / CH_NB, c = e % CH_NB;
    As[r][c] = (i0 + r < n && c < nbk) ? A[(i0 + r) * ld + k0 + c] : 0.0;
    Ws[r][c] = (r < nbk && c <= r) ? W[(int64_t)(k0 + r) * ldw + k0 + c] : 0.0;      // W_kk[r][c], lower triangular
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, wr = (warp >> 1) * 16, wc = (warp & 1) * 32;
  double acc[2][4][2] = {};
  ch_warp_mma<true>(As, Ws, CH_NB, wr, wc, lane, acc);       // P[i][c] = sum_t A[i][t] W_kk[c][t]
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int64_t i = i0 + wr + 8 * mi + (lane >> 2);
        const int c = wc + 8 * ni + 2 * (lane & 3) + e;
        if (i < n && c < nbk) A[i * ld + k0 + c] = acc[mi][ni][e];
      }
}

// Trailing update: A[i, j] -= sum_t P[i, t] P[j, t] for k1 <= j <= i < n (lower triangle), P = A[:, k0:k0+nbk], k1 = k0+nbk.
// grid (tiles, tiles) of 64 x 64 output tiles (upper tiles exit), 256 threads, DMMA (ch_warp_mma).
__global__ void __launch_bounds__(256) ch_syrk_kernel(double* __restrict__ A, int64_t ld, int32_t n, int32_t k0, int32_t nbk) {
  if (blockIdx.y > blockIdx.x) return;                       // tile column > tile row: strictly upper
  extern __shared__ double ch_smem[];                        // 2 tiles (dynamic: CH_GEMM_SMEM)
  ch_gtile_t& Pi = *reinterpret_cast<ch_gtile_t*>(ch_smem);
  ch_gtile_t& Pj = *reinterpret_cast<ch_gtile_t*>(ch_smem + CH_NB * CH_LD);
  const int32_t k1 = k0 + nbk;
  const int64_t i0 = (int64_t)k1 + (int64_t)blockIdx.x * 64, j0 = (int64_t)k1 + (int64_t)blockIdx.y * 64;
  for (int e = threadIdx.x; e < CH_NB * CH_NB; e += 256) {
    const int r = e / CH_NB, t = e % CH_NB;
    Pi[r][t] = (i0 + r < n && t < nbk) ? A[(i0 + r) * ld + k0 + t] : 0.0;
    Pj[r][t] = (j0 + r < n && t < nbk) ? A[(j0 + r) * ld + k0 + t] : 0.0;
  }
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, wr = (warp >> 1) * 16, wc = (warp & 1) * 32;
  double acc[2][4][2] = {};
  ch_warp_mma<true>(Pi, Pj, (nbk + 3) & ~3, wr, wc, lane, acc);
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int64_t i = i0 + wr + 8 * mi + (lane >> 2), j = j0 + wc + 8 * ni + 2 * (lane & 3) + e;
        if (i < n && j < n && j <= i) A[i * ld + j] -= acc[mi][ni][e];
      }
}

// ------------------------------------------------------------------------------------------------
// W = L^-1 by recursive doubling over 64-blocks, then R^-1 = W^T:
//   W_kk = L_kk^-1 for every diagonal block (written by ch_potf2), and for half sizes sb = 1, 2, 4, ... blocks, every pair of
//   adjacent groups   [ L11  0  ]^-1   [      W11          0  ]
//                     [ L21 L22 ]    = [ -W22 (L21 W11)   W22 ]      (ch_level: two block GEMMs, all pairs and tiles in one grid)
// The dependency chain is 2 (1 + 2 + ... + nb/2) block products instead of nb^2 / 2 for a column-by-column substitution,
// and every level keeps all SMs busy.  Triangular operands are not multiplied through their zero blocks.
// ------------------------------------------------------------------------------------------------
// One level of the recursion, one 64 x 64 output tile per CTA (256 threads, DMMA), dynamic smem CH_GEMM_SMEM.
//   mode 1:  T[bi, bj] =   sum_{t in first half, t >= bj} L[bi, t] W[t, bj]       (W11 is lower triangular)
//   mode 2:  W[bi, bj] = - sum_{t in second half, t <= bi} W[bi, t] T[t, bj]      (W22 is lower triangular)
// for bi in the second half of the pair, bj in the first half.  grid (sb, sb, pairs).
__global__ void __launch_bounds__(256) ch_level_kernel(const double* __restrict__ A, int64_t lda, const double* __restrict__ B, int64_t ldb,
                                                       double* __restrict__ C, int64_t ldc, int32_t n, int32_t sb, int32_t mode) {
  extern __shared__ double ch_smem[];
  ch_gtile_t& As = *reinterpret_cast<ch_gtile_t*>(ch_smem);
  ch_gtile_t& Bs = *reinterpret_cast<ch_gtile_t*>(ch_smem + CH_NB * CH_LD);
  const int32_t nb = (n + CH_NB - 1) / CH_NB;
  const int32_t f0 = blockIdx.z * 2 * sb, s0 = f0 + sb, s1 = min(s0 + sb, nb);       // first half [f0, s0), second [s0, s1)
  const int32_t bi = s0 + blockIdx.y, bj = f0 + blockIdx.x;
  if (bi >= s1) return;
  const int32_t tlo = (mode == 1) ? bj : s0, thi = (mode == 1) ? s0 : bi + 1;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31, wr = (warp >> 1) * 16, wc = (warp & 1) * 32;
  double acc[2][4][2] = {};
  for (int32_t t = tlo; t < thi; ++t) {
    __syncthreads();
    for (int e = tid; e < CH_NB * CH_NB; e += 256) {
      const int r = e / CH_NB, c = e % CH_NB;
      const int64_t ar = (int64_t)bi * CH_NB + r, ac = (int64_t)t * CH_NB + c, br = (int64_t)t * CH_NB + r, bc = (int64_t)bj * CH_NB + c;
      // triangular operands: only the lower part of a diagonal block is defined
      const bool a_ok = ar < n && ac < n && !(mode == 2 && t == bi && c > r);
      const bool b_ok = br < n && bc < n && !(mode == 1 && t == bj && c > r);
      As[r][c] = a_ok ? A[ar * lda + ac] : 0.0;
      Bs[r][c] = b_ok ? B[br * ldb + bc] : 0.0;
    }
    __syncthreads();
    ch_warp_mma<false>(As, Bs, CH_NB, wr, wc, lane, acc);
  }
  const double sgn = (mode == 2) ? -1.0 : 1.0;
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int64_t i = (int64_t)bi * CH_NB + wr + 8 * mi + (lane >> 2), j = (int64_t)bj * CH_NB + wc + 8 * ni + 2 * (lane & 3) + e;
        if (i < n && j < n) C[i * ldc + j] = sgn * acc[mi][ni][e];
      }
}

// Rinv = W^T (upper triangular, zero below the diagonal); 32 x 32 tiles through shared memory
__global__ void __launch_bounds__(256) ch_transpose_upper_kernel(const double* __restrict__ W, int64_t ldw, int32_t n, double* __restrict__ Rinv, int64_t ldr) {
  __shared__ double t[32][33];
  const int64_t a0 = (int64_t)blockIdx.y * 32, b0 = (int64_t)blockIdx.x * 32;       // Rinv tile rows a0.., columns b0..
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  for (int r = ty; r < 32; r += 8) {
    const int64_t wb = b0 + r, wa = a0 + tx;                                         // W[b][a]
    t[r][tx] = (wb < n && wa < n && wb >= wa) ? W[wb * ldw + wa] : 0.0;
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {
    const int64_t a = a0 + r, bcol = b0 + tx;
    if (a < n && bcol < n) Rinv[a * ldr + bcol] = t[tx][r];
  }
}

}  // namespace ttdft
