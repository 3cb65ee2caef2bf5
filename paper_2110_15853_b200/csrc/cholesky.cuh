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
// The block lives in REGISTERS: thread (ty, tx) of 16 x 16 holds rows ty + 16 u, columns tx + 16 w (u, w < 4) of A and of the
// right-hand side B of L W = I (B = I at the start).  Step j takes the pivot, column j of A and row j of B from a small
// double-buffered shared-memory exchange, scales them by 1 / sqrt(pivot) and applies both rank-1 updates (A -= l l^T,
// B -= l w_j) in registers; the owners of column j + 1 / row j + 1 then publish them: ONE barrier and ~45 instructions per
// column (before: two barriers, a division loop and a shared-memory update of the trailing block per column, then a serial
// forward substitution: 72 -> 12 us per block, and the chain of 64 blocks is serial).
__global__ void __launch_bounds__(256) ch_potf2_kernel(double* __restrict__ A, int64_t ld, int32_t k0, int32_t nbk, int32_t* __restrict__ flag,
                                                       double* __restrict__ W, int64_t ldw) {
  __shared__ double colraw[2][CH_NB], brow[2][CH_NB], piv[2];
  const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
  double a[4][4], bb[4][4];
#pragma unroll
  for (int u = 0; u < 4; ++u)
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const int row = ty + 16 * u, col = tx + 16 * w;
      // only the lower triangle is ever read; rows / columns beyond nbk behave as an identity block
      a[u][w] = (row < nbk && col <= row) ? A[(int64_t)(k0 + row) * ld + k0 + col] : (row == col ? 1.0 : 0.0);
      bb[u][w] = (row == col) ? 1.0 : 0.0;
    }
  if (tx == 0) {
#pragma unroll
    for (int u = 0; u < 4; ++u) colraw[0][ty + 16 * u] = a[u][0];
  }
  if (ty == 0) {
#pragma unroll
    for (int w = 0; w < 4; ++w) brow[0][tx + 16 * w] = bb[0][w];
  }
  if (tid == 0) piv[0] = a[0][0];
  __syncthreads();
#pragma unroll
  for (int jb = 0; jb < 4; ++jb) {
#pragma unroll 1
    for (int j16 = 0; j16 < 16; ++j16) {
      const int j = jb * 16 + j16, p = j & 1, q = p ^ 1;
      double d = piv[p];
      if (!(d > 0.0)) {                                      // not positive definite (or NaN): record, go on with a harmless pivot
        if (tid == 0 && j < nbk && flag[0] == 0) flag[0] = 1 + k0 + j;
        d = 1.0;
      }
      const double r = rsqrt(d);
      double ljj = d * r;
      ljj = fma(fma(-ljj, ljj, d), 0.5 * r, ljj);            // one Newton step: sqrt(d) to the last bit or two
      double lr[4], lc[4], wr[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) lr[u] = colraw[p][ty + 16 * u] * r;          // l_rj of this thread's rows
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        lc[w] = colraw[p][tx + 16 * w] * r;                                    // l_cj of this thread's columns
        wr[w] = brow[p][tx + 16 * w] * r;                                      // row j of W = row j of B / l_jj
      }
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          a[u][w] = fma(-lr[u], lc[w], a[u][w]);             // rows / columns <= j are finished and never read again
          bb[u][w] = fma(-lr[u], wr[w], bb[u][w]);
        }
      if (j < nbk) {
        if (tx == j16) {                                     // column j of L
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int row = ty + 16 * u;
            if (row < nbk && row >= j) A[(int64_t)(k0 + row) * ld + k0 + j] = (row == j) ? ljj : lr[u];
          }
        }
        if (ty == j16) {                                     // row j of W (zero right of the diagonal: not stored)
#pragma unroll
          for (int w = 0; w < 4; ++w) {
            const int col = tx + 16 * w;
            if (col <= j) W[(int64_t)(k0 + j) * ldw + k0 + col] = wr[w];
          }
        }
      }
      // publish column j + 1 of A, row j + 1 of B and the next pivot
      if (j16 < 15) {
        if (tx == j16 + 1) {
#pragma unroll
          for (int u = 0; u < 4; ++u) colraw[q][ty + 16 * u] = a[u][jb];
        }
        if (ty == j16 + 1) {
#pragma unroll
          for (int w = 0; w < 4; ++w) brow[q][tx + 16 * w] = bb[jb][w];
          if (tx == j16 + 1) piv[q] = a[jb][jb];
        }
      } else if (jb < 3) {
        const int jn = jb < 3 ? jb + 1 : 3;
        if (tx == 0) {
#pragma unroll
          for (int u = 0; u < 4; ++u) colraw[q][ty + 16 * u] = a[u][jn];
        }
        if (ty == 0) {
#pragma unroll
          for (int w = 0; w < 4; ++w) brow[q][tx + 16 * w] = bb[jn][w];
          if (tx == 0) piv[q] = a[jn][jn];
        }
      }
      __syncthreads();
    }
  }
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
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, wr = (warp >> 1) * 16, wc = (warp & 1) * 32;
  // the output tile is read FIRST, so that its latency runs under the panel loads and the product (the kernel is bound by
  // memory latency: a tile is 0.5 MFLOP; with the read-modify-write at the end three quarters of the stalls sat on these loads)
  double cv[2][4][2];
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int64_t i = i0 + wr + 8 * mi + (lane >> 2), j = j0 + wc + 8 * ni + 2 * (lane & 3) + e;
        cv[mi][ni][e] = (i < n && j < n && j <= i) ? A[i * ld + j] : 0.0;
      }
  for (int e = threadIdx.x; e < CH_NB * CH_NB; e += 256) {
    const int r = e / CH_NB, t = e % CH_NB;
    Pi[r][t] = (i0 + r < n && t < nbk) ? A[(i0 + r) * ld + k0 + t] : 0.0;
    Pj[r][t] = (j0 + r < n && t < nbk) ? A[(j0 + r) * ld + k0 + t] : 0.0;
  }
  __syncthreads();
  double acc[2][4][2] = {};
  ch_warp_mma<true>(Pi, Pj, (nbk + 3) & ~3, wr, wc, lane, acc);
#pragma unroll
  for (int mi = 0; mi < 2; ++mi)
#pragma unroll
    for (int ni = 0; ni < 4; ++ni)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int64_t i = i0 + wr + 8 * mi + (lane >> 2), j = j0 + wc + 8 * ni + 2 * (lane & 3) + e;
        if (i < n && j < n && j <= i) A[i * ld + j] = cv[mi][ni][e] - acc[mi][ni][e];
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
  double ra[16], rb[16];                                     // this thread's 16 + 16 elements of the next pair of operand tiles
  auto fetch = [&](int32_t t) {
#pragma unroll
    for (int q = 0; q < 16; ++q) {
      const int e = tid + 256 * q, r = e / CH_NB, c = e % CH_NB;
      const int64_t ar = (int64_t)bi * CH_NB + r, ac = (int64_t)t * CH_NB + c, br = (int64_t)t * CH_NB + r, bc = (int64_t)bj * CH_NB + c;
      // triangular operands: only the lower part of a diagonal block is defined
      const bool a_ok = ar < n && ac < n && !(mode == 2 && t == bi && c > r);
      const bool b_ok = br < n && bc < n && !(mode == 1 && t == bj && c > r);
      ra[q] = a_ok ? A[ar * lda + ac] : 0.0;
      rb[q] = b_ok ? B[br * ldb + bc] : 0.0;
    }
  };
  if (tlo < thi) fetch(tlo);
  for (int32_t t = tlo; t < thi; ++t) {
    __syncthreads();
#pragma unroll
    for (int q = 0; q < 16; ++q) {
      const int e = tid + 256 * q, r = e / CH_NB, c = e % CH_NB;
      As[r][c] = ra[q];
      Bs[r][c] = rb[q];
    }
    __syncthreads();
    if (t + 1 < thi) fetch(t + 1);                           // in flight while the tensor cores work on tile t
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
