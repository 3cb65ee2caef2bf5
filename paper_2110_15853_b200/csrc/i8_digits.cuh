// i8_digits.cuh -- exact splitting of fp64 operands into balanced base-256 digits (int8 planes) for the
// integer tensor-core kernel K3 (bsr_i8.cuh).
//
// The product inside every filter step (H x Y_k) is a block-dense fp64
// contraction that is bound by the fp64 pipe.  B200's 5th-generation tensor
// cores have no f64 kind, but they multiply int8 at ~4.5 Pop/s with exact int32 accumulation.  K3
// therefore evaluates the same product as a sum of exact integer products of digit planes:
//
//   row i of H (diagonal entry kept apart in fp64):  h_ik ~= 2^(eH_i-(8S-1)) * sum_p dH_p[i,k] 256^(S-1-p)
//   column j of Y_k:                                 y_kj ~= 2^(eY_j-(8S-1)) * sum_q dY_q[k,j] 256^(S-1-q)
//
// with balanced digits d in [-128,127], 2^e > max|.| of the row/column, S = 6 or 7 planes.  The only
// error is the rounding of each operand to 8S-1 bits below its row/column maximum (2^-47 for S = 6),
// and the omission of digit-pair levels p+q >= S (below that rounding); all accumulation is exact.
// DESIGN.md "Kernel K3" has the error bound.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttdft {

constexpr int I8_EMIN = -960;   // exponent clamp: keeps every scale factor a normal double

// Upper 32 bits of |x| (monotone in |x| for finite x): the currency of the column/row maxima.
__device__ __forceinline__ uint32_t abs_hi(double x) { return (uint32_t)__double2hiint(x) & 0x7fffffffu; }

// Exponent e with max|x| * 2^-e <= 0.9942 (inside the balanced-digit range 127/255*2 = 0.99608), from
// the upper word of the maximum.  The lower word is unknown, hence the margin on the mantissa.
__host__ __device__ __forceinline__ int32_t exp_from_hi(uint32_t hi) {
  int32_t e = (int32_t)(hi >> 20) - 1022;          // 1.f * 2^(E-1023) < 2^(E-1022)
  if ((hi & 0xfffffu) >= 0xfd000u) e += 1;
  if (e < I8_EMIN) e = I8_EMIN;
  return e;
}
// 2^k as a double, k in [-1022, 1023]
__device__ __forceinline__ double pow2i(int32_t k) { return __longlong_as_double((long long)(k + 1023) << 52); }

// Digit planes of FOUR values at once, packed for the k-major operand layout: w[p] = bytes (digit p of x0, x1, x2, x3).
// q + B with B = 0x80...80 (S bytes) has the plain base-256 bytes d_i + 128 of the balanced digits d_i, so
// t = (q + B) ^ B holds every digit as a two's-complement byte -- one 64-bit add and xor instead of a digit loop --
// and a 4 x S byte transpose (PRMT) gathers byte i of the four values.  Byte i of t is the digit of weight 256^i,
// i.e. plane S-1-i.  This is what makes y_digits memory-bound instead of issue-bound at the filter's power-limited clock.
template <int S>
__device__ __forceinline__ void digits4(const double (&x)[4], double scale, uint32_t (&w)[S]) {
  static_assert(S >= 5 && S <= 8, "4 low bytes + up to 4 high bytes");
  constexpr unsigned long long B = 0x8080808080808080ull >> (8 * (8 - S));
  uint32_t lo[4], hi[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const unsigned long long t = ((unsigned long long)__double2ll_rn(x[i] * scale) + B) ^ B;
    lo[i] = (uint32_t)t;
    hi[i] = (uint32_t)(t >> 32);
  }
  uint32_t a = __byte_perm(lo[0], lo[1], 0x5140), b = __byte_perm(lo[2], lo[3], 0x5140);
  uint32_t c = __byte_perm(lo[0], lo[1], 0x7362), d = __byte_perm(lo[2], lo[3], 0x7362);
  w[S - 1] = __byte_perm(a, b, 0x5410);
  w[S - 2] = __byte_perm(a, b, 0x7632);
  w[S - 3] = __byte_perm(c, d, 0x5410);
  w[S - 4] = __byte_perm(c, d, 0x7632);
  a = __byte_perm(hi[0], hi[1], 0x5140); b = __byte_perm(hi[2], hi[3], 0x5140);
  w[S - 5] = __byte_perm(a, b, 0x5410);
  if (S >= 6) w[S - 6] = __byte_perm(a, b, 0x7632);
  if (S >= 7) {
    c = __byte_perm(hi[0], hi[1], 0x7362); d = __byte_perm(hi[2], hi[3], 0x7362);
    w[S - 7] = __byte_perm(c, d, 0x5410);
    if (S >= 8) w[0] = __byte_perm(c, d, 0x7632);
  }
}

// ------------------------------------------------------------------------------------------------
// column maxima of a panel (first step only; later steps get them from K3's epilogue)
// cmax[j] = max_i hi(|Y[i,j]|); cmax must be zero on entry.  grid (ceil(ncols/64), ceil(M/2048)), 256 thr
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) colmax_kernel(const double* __restrict__ Y, int64_t ld, int64_t M, int64_t ncols,
                                                     uint32_t* __restrict__ cmax) {
  const int64_t col = (int64_t)blockIdx.x * 64 + (threadIdx.x & 63);
  const int sub = threadIdx.x >> 6;
  const int64_t r0 = (int64_t)blockIdx.y * 2048;
  const int64_t r1 = min(M, r0 + 2048);
  uint32_t m = 0;
  if (col < ncols)
    for (int64_t r = r0 + sub; r < r1; r += 4) m = max(m, abs_hi(Y[r * ld + col]));
  __shared__ uint32_t sm[4][64];
  sm[sub][threadIdx.x & 63] = m;
  __syncthreads();
  if (sub == 0 && col < ncols) {
    m = max(max(sm[0][threadIdx.x], sm[1][threadIdx.x]), max(sm[2][threadIdx.x], sm[3][threadIdx.x]));
    if (m) atomicMax(&cmax[col], m);
  }
}

// ------------------------------------------------------------------------------------------------
// digit planes of a panel, transposed and tiled:  D[I][ct][q][n][k] = digit q of Y[I*b + k, 64*ct + n]
// (k < 128, n < 64; zero for k >= b and for columns beyond ncols), i.e. the S planes of one (block row,
// 64-column tile) are ONE contiguous S*8 KB piece of HBM -- what one TMA load of K3 fetches.
// One CTA per (block row I, 64-column tile): coalesced fp64 reads along the columns, a shared-memory
// transpose, 128-byte coalesced int8 rows out -- the K-major rows K3's B operand wants.
// e[h]: exponent of column n0 + 32*h + lane (digits are taken of x * 2^(8S-1-e)); sd: S*64*33 words of shared memory.
// ------------------------------------------------------------------------------------------------
template <int S>
__device__ __forceinline__ void y_digits_tile(const double* __restrict__ Y, int64_t ld, int32_t b, int64_t M, int64_t ncols, int64_t I,
                                              int64_t ct, int64_t nct, const int32_t (&e)[2], int8_t* __restrict__ D, uint32_t* sd) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t n0 = ct * 64;
  double scale[2];
  bool cv[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    cv[h] = n0 + 32 * h + lane < ncols;
    scale[h] = pow2i(8 * S - 1 - e[h]);
  }
  const int nquads = b >> 2;
  for (int quad = warp; quad < 32; quad += 8) {
    // all eight loads of this quad of rows (two 32-column halves) are in flight before any digit work
    double x[2][4];
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const double* src = Y + ((int64_t)I * b + 4 * quad) * ld + n0 + 32 * h + lane;
#pragma unroll
      for (int i = 0; i < 4; ++i)   // rows beyond M (ragged last block of the Gram contraction) read as zero
        x[h][i] = (quad < nquads && cv[h] && I * b + 4 * quad + i < M) ? __ldcs(src + (int64_t)i * ld) : 0.0;
    }
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      uint32_t w[S];
      digits4<S>(x[h], scale[h], w);
#pragma unroll
      for (int p = 0; p < S; ++p) sd[(p * 64 + 32 * h + lane) * 33 + quad] = w[p];
    }
  }
  __syncthreads();
  // rows (q, n) of this tile are consecutive 128-byte lines of D
  uint32_t* dst = reinterpret_cast<uint32_t*>(D + (I * nct + ct) * (int64_t)(S * 64 * 128));
  for (int row = warp; row < S * 64; row += 8) dst[row * 32 + lane] = sd[row * 33 + lane];
}

// Digit tiles of a whole panel with the exponent of every column taken from its maximum cmax[j] (upper word).
// Also clears next_cmax (the maxima K3's epilogue will accumulate for the following step) and, if e_out is given, leaves the
// exponents there (K3 reads its column scales from such an array).
// grid (nb, tiles >= ceil(ncols/64)), 256 threads, dynamic smem S*64*33*4 bytes; M = valid rows (<= nb*b)
template <int S>
__global__ void __launch_bounds__(256) y_digits_kernel(const double* __restrict__ Y, int64_t ld, int32_t b, int64_t M, int64_t ncols,
                                                       const uint32_t* __restrict__ cmax, int8_t* __restrict__ D,
                                                       uint32_t* __restrict__ next_cmax, int32_t* __restrict__ e_out) {
  extern __shared__ uint32_t sd[];   // [S][64][33] words: row (q,n) holds 128 k-bytes + 1 pad word
  const int lane = threadIdx.x & 31;
  const int64_t I = blockIdx.x;
  const int64_t n0 = (int64_t)blockIdx.y * 64;
  int32_t e[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int64_t n = n0 + 32 * h + lane;
    e[h] = exp_from_hi(n < ncols ? cmax[n] : 0u);
  }
  if (I == 0 && threadIdx.x < 64 && n0 + threadIdx.x < ncols) {
    if (next_cmax) next_cmax[n0 + threadIdx.x] = 0;
    if (e_out) e_out[n0 + threadIdx.x] = exp_from_hi(cmax[n0 + threadIdx.x]);
  }
  y_digits_tile<S>(Y, ld, b, M, ncols, I, blockIdx.y, gridDim.y, e, D, sd);
}

// ------------------------------------------------------------------------------------------------
// The filter's digit bookkeeping between two steps (K3 "digits from the epilogue").  From step 2 on, K3's epilogue
// writes the digit tiles of the iterate it produces itself, scaled by a PREDICTED exponent per column (the true column maxima are
// only complete when the launch ends).  This kernel runs between two K3 launches and
//   * fixes the exponent every column's digits were really taken with:  e_used[j] = e_pred[j], or -- for the 64-column tiles in
//     which some column outgrew its prediction (flags[ct] != 0, set by K3's epilogue), and for every tile when force != 0 (the
//     filter's first step: no digits exist yet) -- the true exponent from cmax[j]; those tiles' digits are (re)extracted here;
//   * predicts the exponents of the NEXT iterate:  e_pred[j] = e_true[j] + clamp(e_true[j] - e_prev_true[j] + 1, -3, 0) + guard
//     (the iterates of the Chebyshev recurrence shrink or hold their size from step to step, |p_k| <= 1 on the spectrum: a drop of two
//     or more binary orders is followed with one order of slack, the guard bit absorbs a doubling, anything beyond falls back to the
//     path above).  Measured on configs 2 and 3 (m = 20, narrow and wide gap): no tile redone after the first step;
//   * clears next_cmax and next_flags for the coming launch, and the work counters its clusters draw their items from.
// cmax_prev == next_cmax (the two-slot rotation): the previous iterate's maxima are read before they are cleared, by the same thread.
// grid (rows <= nb, tiles), 256 threads, dynamic smem S*64*33*4 bytes: CTA (x, ct) walks the block rows x, x + gridDim.x, ... of
// column tile ct; CTAs of untouched tiles exit at once (the usual case: a small grid keeps that launch at a few microseconds).
// ------------------------------------------------------------------------------------------------
constexpr int I8_GUARD = 1;
__host__ __device__ __forceinline__ int32_t predict_exp(int32_t e_cur, int32_t e_prev, bool have_prev) {
  int32_t d = have_prev ? e_cur - e_prev + 1 : 0;     // a drop by one binary order is jitter across a power of two, not a trend
  d = d > 0 ? 0 : (d < -3 ? -3 : d);
  const int32_t e = e_cur + d + I8_GUARD;
  return e < I8_EMIN ? I8_EMIN : e;
}
template <int S>
__global__ void __launch_bounds__(256) y_digits_fix_kernel(const double* __restrict__ Y, int64_t ld, int32_t b, int64_t M, int64_t ncols,
                                                           int32_t nb, const uint32_t* __restrict__ cmax, int8_t* __restrict__ D,
                                                           const uint32_t* __restrict__ flags, int32_t force, int32_t have_prev,
                                                           int32_t bias, int32_t* __restrict__ e_used, int32_t* __restrict__ e_pred,
                                                           uint32_t* __restrict__ next_cmax, uint32_t* __restrict__ next_flags,
                                                           uint32_t* __restrict__ work_counters) {
  extern __shared__ uint32_t sd[];
  const int lane = threadIdx.x & 31;
  const int64_t n0 = (int64_t)blockIdx.y * 64;
  const bool redo = force || flags[blockIdx.y] != 0;
  if (blockIdx.x == 0 && threadIdx.x < 64) {
    const int64_t n = n0 + threadIdx.x;
    if (n < ncols) {
      const int32_t e_true = exp_from_hi(cmax[n]);
      const int32_t e_prev = have_prev ? exp_from_hi(next_cmax[n]) : 0;     // the slot about to be cleared holds the iterate before
      e_used[n] = redo ? e_true : e_pred[n];
      int32_t ep = predict_exp(e_true, e_prev, have_prev != 0) + bias;      // bias: test hook (TTDFT_K3_PREDICT_BIAS), 0 in normal use
      e_pred[n] = ep < I8_EMIN ? I8_EMIN : ep;
      next_cmax[n] = 0;
    }
    if (threadIdx.x == 0) next_flags[blockIdx.y] = 0;
    if (threadIdx.x == 0 && blockIdx.y == 0) { work_counters[0] = 0; work_counters[1] = 0; }   // the coming K3 launches draw their items from these
  }
  if (!redo) return;
  int32_t e[2];
#pragma unroll
  for (int h = 0; h < 2; ++h) {
    const int64_t n = n0 + 32 * h + lane;
    e[h] = exp_from_hi(n < ncols ? cmax[n] : 0u);
  }
  for (int64_t I = blockIdx.x; I < nb; I += gridDim.x) {
    y_digits_tile<S>(Y, ld, b, M, ncols, I, blockIdx.y, gridDim.y, e, D, sd);
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// H side (builder, A0): row exponents + diagonal, then digit planes of every tile
// ------------------------------------------------------------------------------------------------
// grid nb, 256 threads.  eH[row] from the row maximum over all tiles of the block row, the diagonal
// entry excluded (it is applied in fp64 by K3's epilogue: Kohn-Sham H is diagonally heavy, and keeping
// the diagonal out of the row scale keeps the digits of the couplings at full resolution).
__global__ void __launch_bounds__(256) h_rowscale_kernel(int32_t b, const int32_t* __restrict__ brow_ptr,
                                                         const int32_t* __restrict__ bcol, const double* __restrict__ tiles,
                                                         int32_t* __restrict__ eH, double* __restrict__ hdiag) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int32_t I = blockIdx.x;
  const int32_t p0 = brow_ptr[I], p1 = brow_ptr[I + 1];
  for (int r = warp; r < b; r += 8) {
    uint32_t m = 0;
    double dg = 0.0;
    for (int32_t p = p0; p < p1; ++p) {
      const bool diag_tile = (bcol[p] == I);
      const double* row = tiles + ((size_t)p * b + r) * b;
      for (int k = lane; k < b; k += 32) {
        const double v = row[k];
        if (diag_tile && k == r) dg = v;
        else m = max(m, abs_hi(v));
      }
    }
    m = __reduce_max_sync(0xffffffffu, m);
    // exactly one lane saw the diagonal entry (or none): pass it on by a sum
    for (int o = 16; o > 0; o >>= 1) dg += __shfl_xor_sync(0xffffffffu, dg, o);
    if (lane == 0) {
      eH[(int64_t)I * b + r] = exp_from_hi(m);
      hdiag[(int64_t)I * b + r] = dg;
    }
  }
}

// grid nb, 256 threads: planes Hd[(p*S + q)*b + r][128 bytes] of every tile p of block row I
template <int S>
__global__ void __launch_bounds__(256) h_digits_kernel(int32_t b, const int32_t* __restrict__ brow_ptr,
                                                       const int32_t* __restrict__ bcol, const double* __restrict__ tiles,
                                                       const int32_t* __restrict__ eH, int8_t* __restrict__ Hd) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int32_t I = blockIdx.x;
  const int32_t p0 = brow_ptr[I], p1 = brow_ptr[I + 1];
  for (int32_t p = p0; p < p1; ++p) {
    const bool diag_tile = (bcol[p] == I);
    for (int r = warp; r < b; r += 8) {
      const double scale = pow2i(8 * S - 1 - eH[(int64_t)I * b + r]);
      uint32_t w[S];
      double x[4] = {0.0, 0.0, 0.0, 0.0};      // columns >= b of the 128-byte row stay zero
      if (4 * lane < b) {
        const double* src = tiles + ((size_t)p * b + r) * b + 4 * lane;
#pragma unroll
        for (int i = 0; i < 4; ++i) x[i] = (diag_tile && 4 * lane + i == r) ? 0.0 : src[i];
      }
      digits4<S>(x, scale, w);
#pragma unroll
      for (int q = 0; q < S; ++q)
        reinterpret_cast<uint32_t*>(Hd + (((size_t)p * S + q) * b + r) * 128)[lane] = w[q];
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Row-scaled digit tiles of a dense row-major matrix X (M x K), the A operand of ttdft_rotate (Y = X Q):
//   eX[i] from the maximum of row i;   Dx[(I*nkb + J)*S + q][r][k] = digit q of X[I*128 + r, J*128 + k]
// -- the tile format of the H digit planes with tile (I, J) = rows I*128.., columns J*128.. of X.
// ------------------------------------------------------------------------------------------------
// one warp per row; grid ceil(Mpad/8), 256 threads.  Rows >= M get the smallest exponent.
__global__ void __launch_bounds__(256) x_rowexp_kernel(const double* __restrict__ X, int64_t ld, int64_t M, int64_t Mpad, int64_t K,
                                                       int32_t* __restrict__ eX) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t row = (int64_t)blockIdx.x * 8 + warp;
  if (row >= Mpad) return;
  uint32_t m = 0;
  if (row < M)
    for (int64_t k = lane; k < K; k += 32) m = max(m, abs_hi(X[row * ld + k]));
  m = __reduce_max_sync(0xffffffffu, m);
  if (lane == 0) eX[row] = exp_from_hi(m);
}

// grid (nbm, nkb), 256 threads: thread (r = tid/32 + 8*it, kq = tid%32) converts 4 consecutive k of one row
template <int S>
__global__ void __launch_bounds__(256) x_digits_rows_kernel(const double* __restrict__ X, int64_t ld, int64_t M, int64_t K,
                                                            const int32_t* __restrict__ eX, int8_t* __restrict__ Dx) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t I = blockIdx.x, J = blockIdx.y, nkb = gridDim.y;
  int8_t* tile = Dx + (I * nkb + J) * (int64_t)(S * 128 * 128);
  for (int r = warp; r < 128; r += 8) {
    const int64_t row = I * 128 + r;
    const int64_t k0 = J * 128 + 4 * lane;
    double x[4];
#pragma unroll
    for (int i = 0; i < 4; ++i) x[i] = (row < M && k0 + i < K) ? __ldcs(X + row * ld + k0 + i) : 0.0;
    uint32_t w[S];
    digits4<S>(x, pow2i(8 * S - 1 - eX[row]), w);
#pragma unroll
    for (int q = 0; q < S; ++q) reinterpret_cast<uint32_t*>(tile + ((size_t)q * 128 + r) * 128)[lane] = w[q];
  }
}

// block row pointers / block columns of a dense nbm x nkb grid of tiles
__global__ void dense_tile_index_kernel(int32_t nbm, int32_t nkb, int32_t* __restrict__ brow_ptr, int32_t* __restrict__ bcol) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i <= nbm) brow_ptr[i] = (int32_t)(i * nkb);
  if (i < (int64_t)nbm * nkb) bcol[i] = (int32_t)(i % nkb);
}

}  // namespace ttdft
