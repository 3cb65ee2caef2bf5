// generic_spmm.cuh -- fallback kernel K2: one warp per row of H, lanes over columns of X
// (coalesced 8-byte accesses, no alignment requirements), same fused epilogue as K1
// (PAPER.md:L218, L221).  Used for CSR without block structure (BASELINE.json config 5's randomly
// permuted layout), for BSR tile sizes K1 does not cover, and for misaligned X/Y views.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttdft {

constexpr int K2_CPL = 4;                 // columns per lane
constexpr int K2_TN = 32 * K2_CPL;        // columns per warp pass
constexpr int K2_ROWS = 8;                // rows (warps) per CTA

struct K2Params {
  const int32_t* row_ptr;   // CSR: M+1 ; BSR: nb+1
  const int32_t* col;       // CSR: nnz ; BSR: nblocks
  const double* val;
  int64_t M;
  int32_t b;                // BSR tile size (unused for CSR)
  int64_t ncols;
  double alpha, gamma, beta;
  const double* X; int64_t ldx;     // the multiplied block (Y_k)
  const double* Z; int64_t ldz;     // Y_{k-1} / Y, read at the output position if beta != 0
  double* O; int64_t ldo;
  const int32_t* perm;      // BSR handles built from permuted subdomain labels: row r of H is row perm[r] of X/Z/O (else NULL)
  int32_t skip_empty = 0;   // 1: (block) rows without entries are not this handle's: their output rows are left untouched
};

template <bool BSR>
__global__ void __launch_bounds__(32 * K2_ROWS) generic_step_kernel(const K2Params p) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * K2_ROWS + warp;
  if (row >= p.M) return;
  if (p.skip_empty) {
    const int64_t ir = BSR ? row / p.b : row;
    if (p.row_ptr[ir] == p.row_ptr[ir + 1]) return;
  }
  const int64_t urow = (BSR && p.perm) ? p.perm[row] : row;   // the caller's row
  if (urow < 0) return;                                       // a padding row of a subdomain smaller than the tile
  const int64_t c0 = (int64_t)blockIdx.y * K2_TN + lane;
  double acc[K2_CPL];
  bool ok[K2_CPL];
#pragma unroll
  for (int c = 0; c < K2_CPL; ++c) { acc[c] = 0.0; ok[c] = (c0 + 32 * c) < p.ncols; }

  if (p.alpha != 0.0) {
    if (BSR) {
      const int64_t I = row / p.b;
      const int32_t rr = (int32_t)(row - I * p.b);
      for (int32_t q = p.row_ptr[I]; q < p.row_ptr[I + 1]; ++q) {
        const double* tile = p.val + ((size_t)q * p.b + rr) * p.b;
        const int64_t xrow0 = (int64_t)p.col[q] * p.b;
        for (int32_t s = 0; s < p.b; ++s) {
          const double h = __ldg(tile + s);
          const int64_t xrow = p.perm ? (int64_t)p.perm[xrow0 + s] : xrow0 + s;
          if (xrow < 0) continue;                             // padding column (its tile entries are zero)
          const double* xr = p.X + xrow * p.ldx + c0;
#pragma unroll
          for (int c = 0; c < K2_CPL; ++c)
            if (ok[c]) acc[c] = fma(h, __ldg(xr + 32 * c), acc[c]);
        }
      }
    } else {
      const int32_t e0 = p.row_ptr[row], e1 = p.row_ptr[row + 1];
      for (int32_t base = e0; base < e1; base += 32) {
        // one coalesced load of up to 32 (col, val) pairs, then broadcast by shuffle
        const int32_t e = base + lane;
        int32_t jc = 0;
        double hv = 0.0;
        if (e < e1) { jc = __ldg(p.col + e); hv = __ldg(p.val + e); }
        const int n = min(32, e1 - base);
        for (int k = 0; k < n; ++k) {
          const int32_t j = __shfl_sync(0xffffffffu, jc, k);
          const double h = __shfl_sync(0xffffffffu, hv, k);
          const double* xr = p.X + (int64_t)j * p.ldx + c0;
#pragma unroll
          for (int c = 0; c < K2_CPL; ++c)
            if (ok[c]) acc[c] = fma(h, __ldg(xr + 32 * c), acc[c]);
        }
      }
    }
  }
  const bool use_s = (p.gamma != 0.0), use_z = (p.beta != 0.0);
#pragma unroll
  for (int c = 0; c < K2_CPL; ++c) {
    if (!ok[c]) continue;
    const int64_t col = c0 + 32 * c;
    double v = p.alpha * acc[c];
    if (use_s) v = fma(p.gamma, p.X[urow * p.ldx + col], v);
    if (use_z) v = fma(p.beta, p.Z[urow * p.ldz + col], v);
    p.O[urow * p.ldo + col] = v;
  }
}

// K2 for a CSR and a NARROW panel (ncols <= 128 / G): the lanes-over-columns kernel above would keep at most ncols of its 128 column
// slots busy.  Here a warp still owns one row, but works on G (4 or 2) entries of the row at a time: lane = LPG g + l (LPG = 32 / G)
// handles entry group g and the columns l, l + LPG, l + 2 LPG, l + 3 LPG, so one load instruction fetches G pieces of 8 LPG bytes of
// G rows of X; the G partial sums are added by shuffles at the end.  Same fused epilogue.  Config 5's permuted CSR at N = 16:
// 15.7 -> 6.0 ms per product.
template <int G>
__global__ void __launch_bounds__(32 * K2_ROWS) generic_csr_narrow_kernel(const K2Params p) {
  constexpr int LPG = 32 / G;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * K2_ROWS + warp;
  if (row >= p.M) return;
  const int32_t e0 = p.row_ptr[row], e1 = p.row_ptr[row + 1];
  if (p.skip_empty && e0 == e1) return;
  const int g = lane / LPG, l = lane % LPG;
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  bool ok[4];
  const int64_t cb = (int64_t)blockIdx.y * (4 * LPG);     // first column of this CTA's column tile
#pragma unroll
  for (int c = 0; c < 4; ++c) ok[c] = (cb + l + LPG * c) < p.ncols;
  if (p.alpha != 0.0) {
    for (int32_t base = e0; base < e1; base += 32) {
      const int32_t e = base + lane;
      int32_t jc = 0;
      double hv = 0.0;                            // entries beyond the row: value 0 times row 0 of X
      if (e < e1) { jc = __ldg(p.col + e); hv = __ldg(p.val + e); }
      const int n = min(32, e1 - base);
      for (int k = 0; k < n; k += G) {
        const int32_t j = __shfl_sync(0xffffffffu, jc, k + g);
        const double h = __shfl_sync(0xffffffffu, hv, k + g);
        if (k + g < n) {
          const double* xr = p.X + (int64_t)j * p.ldx + cb + l;
#pragma unroll
          for (int c = 0; c < 4; ++c)
            if (ok[c]) acc[c] = fma(h, __ldg(xr + LPG * c), acc[c]);
        }
      }
    }
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (G == 4) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], 8);
    acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], 16);
  }
  if (g != 0) return;
  const bool use_s = (p.gamma != 0.0), use_z = (p.beta != 0.0);
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    if (!ok[c]) continue;
    const int64_t col = cb + l + LPG * c;
    double v = p.alpha * acc[c];
    if (use_s) v = fma(p.gamma, p.X[row * p.ldx + col], v);
    if (use_z) v = fma(p.beta, p.Z[row * p.ldz + col], v);
    p.O[row * p.ldo + col] = v;
  }
}

}  // namespace ttdft
