// ttdft_oracle.cpp -- CPU ORACLE for the Chebyshev filter of ChFSI (TEST INFRASTRUCTURE ONLY).
//
// This file is test infrastructure.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference legs may build, load or call it.  It shares no code, header,
// table or helper with the CUDA path under paper_2110_15853_b200/ and neither imports the other.
//
// What it is: a plain, slow, obviously-correct fp64 implementation of Algorithm 1, step 1 of
// arXiv 2110.15853, executed literally in the paper's order and notation
// from a CSR matrix, plus the plain definition of Y = alpha*H*X + beta*Y ("the main
// kernel ... is the sparse-dense matrix-matrix multiplication"), a dense brute-force product used
// to pin the sparse code, and a k-step Lanczos that supplies the spectral bounds the paper takes
// as inputs (reading #5 in DESIGN.md).
//
// No blocking, fusion or reordering: each output element is one left-to-right sum over the row's
// stored entries in ascending column order.  OpenMP parallelism is over ROWS only, so every
// element's rounding is independent of the thread count.  Compile with -ffp-contract=off.
//
// Parity pins (tests/test_oracle_pins.py): P1 dense brute force, P2 scalar closed form T_m,
// P3 known eigendecomposition, P4 degenerate matrices, P5 invariants, P6 Lanczos bounds.
// Every function here is pinned by at least one of them; nothing is "parity unpinned".
//
// NEXT-1: oracle_gram is the plain definition of G = X^T W, the second product of the subspace
// projection H_F = X_F^T (H X_F) (Algorithm 1 step 3; Sec. 4.3); the projection itself is
// oracle_spmm_csr followed by oracle_gram.  Pins P7 (tests/test_oracle_pins.py): hand-computed integers
// (tests/golden/gram_pins.txt), numpy's matmul, Q^T H Q = Lambda for a known eigendecomposition, symmetry,
// congruence (XR)^T H (XR) = R^T (X^T H X) R and the trace identity.  oracle_rotate is the plain definition of
// Y = X Q (Algorithm 1 step 5); pins P8: hand-computed integers, numpy's matmul, Q = I and a column
// permutation (exact), and the identity (XQ)^T (XQ) = Q^T (X^T X) Q through oracle_gram.  oracle_orth_gs is Gram-Schmidt
// (Algorithm 1 step 2); pins P9: a hand-computed 2 x 2 case, numpy's QR with the signs of R's diagonal made
// positive, Q^T Q = I, Q^T X upper triangular with positive diagonal, X = Q (Q^T X).
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---------------------------------------------------------------------------------------------
// Dense brute force: Y[i,j] = sum_k Hd[i,k] * X[k,j], triple loop on an M x M row-major array.
// Used only to pin the sparse routines (P1).  Definition of the matrix product.
// ---------------------------------------------------------------------------------------------
void oracle_dense_hx(int64_t M, const double* Hd, const double* X, int64_t ldx, double* Y, int64_t ldy,
                     int64_t ncols) {
  for (int64_t i = 0; i < M; ++i)
    for (int64_t j = 0; j < ncols; ++j) {
      double acc = 0.0;
      for (int64_t k = 0; k < M; ++k) acc += Hd[i * M + k] * X[k * ldx + j];
      Y[i * ldy + j] = acc;
    }
}

// ---------------------------------------------------------------------------------------------
// BSR -> CSR expansion INCLUDING the explicit zeros of every stored block (so a BSR input and its
// CSR expansion define the same sums in the same order).  Blocks are b x b row-major tiles.
// csr_row_ptr: M+1, csr_col / csr_val: nblocks*b*b.
// ---------------------------------------------------------------------------------------------
void oracle_bsr_to_csr(int64_t nb, int32_t b, const int32_t* brow_ptr, const int32_t* bcol,
                       const double* bval, int32_t* csr_row_ptr, int32_t* csr_col, double* csr_val) {
  int64_t o = 0;
  for (int64_t I = 0; I < nb; ++I)
    for (int32_t r = 0; r < b; ++r) {
      csr_row_ptr[I * b + r] = (int32_t)o;
      for (int64_t p = brow_ptr[I]; p < brow_ptr[I + 1]; ++p)
        for (int32_t s = 0; s < b; ++s) {
          csr_col[o] = bcol[p] * b + s;
          csr_val[o] = bval[((size_t)p * b + r) * b + s];
          ++o;
        }
    }
  csr_row_ptr[nb * b] = (int32_t)o;
}

// ---------------------------------------------------------------------------------------------
// Y = alpha * (H X) + beta * Y  (plain definition; beta == 0 does not read Y, BLAS convention).
// H: CSR, 0-based, int32 indices; X, Y row-major M x ncols with leading dimensions ldx, ldy.
// ---------------------------------------------------------------------------------------------
void oracle_spmm_csr(int64_t M, const int32_t* row_ptr, const int32_t* col, const double* val, double alpha,
                     const double* X, int64_t ldx, double beta, double* Y, int64_t ldy, int64_t ncols) {
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < M; ++i)
    for (int64_t j = 0; j < ncols; ++j) {
      double acc = 0.0;
      for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) acc += val[p] * X[(int64_t)col[p] * ldx + j];
      double y = alpha * acc;
      if (beta != 0.0) y = y + beta * Y[i * ldy + j];
      Y[i * ldy + j] = y;
    }
}

// ---------------------------------------------------------------------------------------------
// One recurrence step exactly as written in Algorithm 1 (PAPER.md:L218 with beta absent,
// PAPER.md:L221 otherwise):   Yout = alpha * (H*Yk - c*Yk) + beta * Ykm1
// evaluated per element as  acc = sum_k h[i,k]*Yk[k,j];  t = acc - c*Yk[i,j];
// Yout[i,j] = alpha*t (+ beta*Ykm1[i,j]).   Ykm1 == NULL  <=>  the beta term is absent.
// Yout must not alias Yk.
// ---------------------------------------------------------------------------------------------
void oracle_cheb_step_csr(int64_t M, const int32_t* row_ptr, const int32_t* col, const double* val, double alpha,
                          double c, double beta, const double* Yk, int64_t ldk, const double* Ykm1, int64_t ldm,
                          double* Yout, int64_t ldo, int64_t ncols) {
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < M; ++i)
    for (int64_t j = 0; j < ncols; ++j) {
      double acc = 0.0;
      for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) acc += val[p] * Yk[(int64_t)col[p] * ldk + j];
      double t = acc - c * Yk[i * ldk + j];
      double y = alpha * t;
      if (Ykm1) y = y + beta * Ykm1[i * ldm + j];
      Yout[i * ldo + j] = y;
    }
}

// ---------------------------------------------------------------------------------------------
// Algorithm 1, step 1, literally:
//   e = (eps_ub^uw - eps_ub^w)/2 ; c = (eps_ub^uw + eps_ub^w)/2 ; sigma = e/(eps_0 - c)
//   sigma_1 = sigma ; gamma = 2/sigma_1 ; Xt = (sigma_1/e) (H X - c X)
//   for i = 2:m   sigma_2 = 1/(gamma - sigma)
//                 Xt_new = (2 sigma_2/e)(H Xt - c Xt) - sigma sigma_2 X
//                 X = Xt ; Xt = Xt_new ; sigma = sigma_2
// Arguments follow north_star: a = eps_ub^w, b = eps_ub^uw, a0 = eps_0 (reading #4).
// Output: the newest iterate Xt (reading #1).  m = 0 is defined as Y = X, m = 1 returns the first
// step (reading #3).  Returns 0, or -1 for invalid arguments (m < 0 or not a0 < a < b).
// The three M x ncols iterates are held in private buffers; X is not modified.
// ---------------------------------------------------------------------------------------------
int oracle_cheb_filter_csr(int64_t M, const int32_t* row_ptr, const int32_t* col, const double* val,
                           const double* X, int64_t ldx, double* Y, int64_t ldy, int64_t ncols, int32_t m,
                           double a, double b, double a0) {
  if (m < 0 || !(a0 < a) || !(a < b)) return -1;
  if (m == 0) {
    for (int64_t i = 0; i < M; ++i) std::memcpy(Y + i * ldy, X + i * ldx, (size_t)ncols * sizeof(double));
    return 0;
  }
  const size_t sz = (size_t)M * (size_t)ncols;
  std::vector<double> bufX(sz), bufXt(sz), bufNew(sz);
  double* Xc = bufX.data();     // the paper's X
  double* Xt = bufXt.data();    // the paper's X-tilde
  double* Xn = bufNew.data();   // the paper's X-tilde_new
  for (int64_t i = 0; i < M; ++i) std::memcpy(Xc + i * ncols, X + i * ldx, (size_t)ncols * sizeof(double));

  const double e = 0.5 * (b - a);
  const double c = 0.5 * (b + a);
  double sigma = e / (a0 - c);
  const double sigma1 = sigma;
  const double gamma = 2.0 / sigma1;
  oracle_cheb_step_csr(M, row_ptr, col, val, sigma1 / e, c, 0.0, Xc, ncols, nullptr, 0, Xt, ncols, ncols);
  for (int32_t i = 2; i <= m; ++i) {
    const double sigma2 = 1.0 / (gamma - sigma);
    oracle_cheb_step_csr(M, row_ptr, col, val, 2.0 * sigma2 / e, c, -(sigma * sigma2), Xt, ncols, Xc, ncols, Xn,
                         ncols, ncols);
    double* t = Xc; Xc = Xt; Xt = Xn; Xn = t;   // X = Xt ; Xt = Xt_new
    sigma = sigma2;
  }
  for (int64_t i = 0; i < M; ++i) std::memcpy(Y + i * ldy, Xt + i * ncols, (size_t)ncols * sizeof(double));
  return 0;
}

// Same algorithm with 80-bit long double accumulation and iterates: an error-budget reference that
// tells which of {oracle, GPU} is closer to the exact result when they differ near the tolerance.
int oracle_cheb_filter_csr_ld(int64_t M, const int32_t* row_ptr, const int32_t* col, const double* val,
                              const double* X, int64_t ldx, double* Y, int64_t ldy, int64_t ncols, int32_t m,
                              double a, double b, double a0) {
  if (m < 0 || !(a0 < a) || !(a < b)) return -1;
  const size_t sz = (size_t)M * (size_t)ncols;
  std::vector<long double> A(sz), B(sz), C(sz);
  long double *Xc = A.data(), *Xt = B.data(), *Xn = C.data();
  for (int64_t i = 0; i < M; ++i)
    for (int64_t j = 0; j < ncols; ++j) Xc[i * ncols + j] = X[i * ldx + j];
  if (m == 0) {
    for (int64_t i = 0; i < M; ++i)
      for (int64_t j = 0; j < ncols; ++j) Y[i * ldy + j] = X[i * ldx + j];
    return 0;
  }
  const long double e = 0.5L * ((long double)b - a), c = 0.5L * ((long double)b + a);
  long double sigma = e / ((long double)a0 - c);
  const long double sigma1 = sigma, gamma = 2.0L / sigma1;
  auto step = [&](long double alpha, long double beta, const long double* Yk, const long double* Ykm1,
                  long double* Yo) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < M; ++i)
      for (int64_t j = 0; j < ncols; ++j) {
        long double acc = 0.0L;
        for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) acc += (long double)val[p] * Yk[(int64_t)col[p] * ncols + j];
        long double y = alpha * (acc - c * Yk[i * ncols + j]);
        if (Ykm1) y += beta * Ykm1[i * ncols + j];
        Yo[i * ncols + j] = y;
      }
  };
  step(sigma1 / e, 0.0L, Xc, nullptr, Xt);
  for (int32_t i = 2; i <= m; ++i) {
    const long double sigma2 = 1.0L / (gamma - sigma);
    step(2.0L * sigma2 / e, -(sigma * sigma2), Xt, Xc, Xn);
    long double* t = Xc; Xc = Xt; Xt = Xn; Xn = t;
    sigma = sigma2;
  }
  for (int64_t i = 0; i < M; ++i)
    for (int64_t j = 0; j < ncols; ++j) Y[i * ldy + j] = (double)Xt[i * ncols + j];
  return 0;
}

// ---------------------------------------------------------------------------------------------
// Spectral bounds (harness input; the paper defers to refs [30,31]).  Reading #5:
// k-step Lanczos without reorthogonalisation from start vector v0, eigenpairs (theta, z) of the
// k x k tridiagonal by cyclic Jacobi, residual-corrected Ritz bounds
//     b  = theta_max + |beta_k * z_max[k]| ,   a0 = theta_min - |beta_k * z_min[k]|.
// Outputs: alpha[k], beta[k] (beta[j] couples v_j and v_{j+1}; beta[k-1] is the residual norm),
// theta[k] ascending, zlast[k] = last components of the unit eigenvectors; returns the k used.
// ---------------------------------------------------------------------------------------------
// G = X^T W: G[j,l] = sum_k X[k,j] * W[k,l], k ascending, left to right.
// X, W: M x n row-major (ldx, ldw); G: n x n row-major (ldg).  Parallel over the rows j of G only.
void oracle_gram(int64_t M, int64_t n, const double* X, int64_t ldx, const double* W, int64_t ldw, double* G, int64_t ldg) {
#pragma omp parallel for schedule(static)
  for (int64_t j = 0; j < n; ++j) {
    double* g = G + j * ldg;
    for (int64_t l = 0; l < n; ++l) g[l] = 0.0;
    for (int64_t k = 0; k < M; ++k) {
      const double x = X[k * ldx + j];
      const double* w = W + k * ldw;
      for (int64_t l = 0; l < n; ++l) g[l] = g[l] + x * w[l];
    }
  }
}

// Y = X Q (Algorithm 1 step 5 "Rotate the basis"): Y[i,l] = sum_k X[i,k] * Q[k,l], k ascending.
// X: M x K (ldx), Q: K x n (ldq), Y: M x n (ldy), all row-major.  Parallel over the rows of Y only.
void oracle_rotate(int64_t M, int64_t K, int64_t n, const double* X, int64_t ldx, const double* Q, int64_t ldq, double* Y, int64_t ldy) {
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < M; ++i) {
    double* y = Y + i * ldy;
    for (int64_t l = 0; l < n; ++l) y[l] = 0.0;
    for (int64_t k = 0; k < K; ++k) {
      const double x = X[i * ldx + k];
      const double* q = Q + k * ldq;
      for (int64_t l = 0; l < n; ++l) y[l] = y[l] + x * q[l];
    }
  }
}

// X_F = Orth(X) (Algorithm 1 step 2; L230 "Gram-Schmidt orthogonalization procedure"): Gram-Schmidt column by
// column, the projections removed one at a time (modified Gram-Schmidt) and the whole sweep repeated `sweeps` times
// ("twice is enough": with 2 sweeps the result is orthonormal to rounding level for any X that is numerically full rank):
//   v = x_j;  repeat sweeps times: for i < j: v = v - (q_i . v) q_i;   q_j = v / ||v||_2
// X, Q: M x n row-major.  Returns 1 + j if column j has no component outside the span of the previous ones, else 0.
int oracle_orth_gs(int64_t M, int64_t n, const double* X, int64_t ldx, double* Q, int64_t ldq, int32_t sweeps) {
  std::vector<double> v((size_t)M);
  for (int64_t j = 0; j < n; ++j) {
    for (int64_t k = 0; k < M; ++k) v[(size_t)k] = X[k * ldx + j];
    for (int32_t s = 0; s < sweeps; ++s)
      for (int64_t i = 0; i < j; ++i) {
        double r = 0.0;
        for (int64_t k = 0; k < M; ++k) r = r + Q[k * ldq + i] * v[(size_t)k];
        for (int64_t k = 0; k < M; ++k) v[(size_t)k] = v[(size_t)k] - r * Q[k * ldq + i];
      }
    double nrm2 = 0.0;
    for (int64_t k = 0; k < M; ++k) nrm2 = nrm2 + v[(size_t)k] * v[(size_t)k];
    if (!(nrm2 > 0.0)) return (int)(1 + j);
    const double nrm = std::sqrt(nrm2);
    for (int64_t k = 0; k < M; ++k) Q[k * ldq + j] = v[(size_t)k] / nrm;
  }
  return 0;
}

static void spmv_csr(int64_t M, const int32_t* row_ptr, const int32_t* col, const double* val, const double* x,
                     double* y) {
#pragma omp parallel for schedule(dynamic, 64)
  for (int64_t i = 0; i < M; ++i) {
    double acc = 0.0;
    for (int64_t p = row_ptr[i]; p < row_ptr[i + 1]; ++p) acc += val[p] * x[col[p]];
    y[i] = acc;
  }
}

// cyclic Jacobi on a small dense symmetric matrix A (n x n, destroyed); V gets the eigenvectors (columns)
static void jacobi_eig(int n, std::vector<double>& A, std::vector<double>& V) {
  V.assign((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) V[(size_t)i * n + i] = 1.0;
  for (int sweep = 0; sweep < 100; ++sweep) {
    double off = 0.0;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) off += A[(size_t)p * n + q] * A[(size_t)p * n + q];
    if (off < 1e-300) break;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) {
        double apq = A[(size_t)p * n + q];
        if (apq == 0.0) continue;
        double app = A[(size_t)p * n + p], aqq = A[(size_t)q * n + q];
        double tau = (aqq - app) / (2.0 * apq);
        double t = (tau >= 0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
        double cs = 1.0 / std::sqrt(1.0 + t * t), sn = t * cs;
        for (int k = 0; k < n; ++k) {   // A <- A J  (columns p, q)
          double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
          A[(size_t)k * n + p] = cs * akp - sn * akq;
          A[(size_t)k * n + q] = sn * akp + cs * akq;
        }
        for (int k = 0; k < n; ++k) {   // A <- J^T A  (rows p, q)
          double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
          A[(size_t)p * n + k] = cs * apk - sn * aqk;
          A[(size_t)q * n + k] = sn * apk + cs * aqk;
        }
        for (int k = 0; k < n; ++k) {
          double vkp = V[(size_t)k * n + p], vkq = V[(size_t)k * n + q];
          V[(size_t)k * n + p] = cs * vkp - sn * vkq;
          V[(size_t)k * n + q] = sn * vkp + cs * vkq;
        }
      }
  }
}

int oracle_lanczos_bounds(int64_t M, const int32_t* row_ptr, const int32_t* col, const double* val, int32_t k,
                          const double* v0, double* alpha, double* beta, double* theta, double* zlast,
                          double* a0_out, double* b_out) {
  if (k > M) k = (int32_t)M;
  if (k < 1) return -1;
  std::vector<double> v(M), vprev(M, 0.0), w(M);
  double nrm = 0.0;
  for (int64_t i = 0; i < M; ++i) nrm += v0[i] * v0[i];
  nrm = std::sqrt(nrm);
  if (!(nrm > 0.0)) return -1;
  for (int64_t i = 0; i < M; ++i) v[i] = v0[i] / nrm;
  double bprev = 0.0;
  int kk = k;
  for (int j = 0; j < k; ++j) {
    spmv_csr(M, row_ptr, col, val, v.data(), w.data());
    double aj = 0.0;
    for (int64_t i = 0; i < M; ++i) aj += w[i] * v[i];
    for (int64_t i = 0; i < M; ++i) w[i] = w[i] - aj * v[i] - bprev * vprev[i];
    double bj = 0.0;
    for (int64_t i = 0; i < M; ++i) bj += w[i] * w[i];
    bj = std::sqrt(bj);
    alpha[j] = aj;
    beta[j] = bj;
    if (bj == 0.0) { kk = j + 1; break; }   // invariant subspace found: bounds are exact
    for (int64_t i = 0; i < M; ++i) { vprev[i] = v[i]; v[i] = w[i] / bj; }
    bprev = bj;
  }
  std::vector<double> T((size_t)kk * kk, 0.0), V;
  for (int j = 0; j < kk; ++j) {
    T[(size_t)j * kk + j] = alpha[j];
    if (j + 1 < kk) { T[(size_t)j * kk + j + 1] = beta[j]; T[(size_t)(j + 1) * kk + j] = beta[j]; }
  }
  jacobi_eig(kk, T, V);
  std::vector<int> idx(kk);
  for (int j = 0; j < kk; ++j) idx[j] = j;
  for (int i = 0; i < kk; ++i)   // selection sort, ascending theta
    for (int j = i + 1; j < kk; ++j)
      if (T[(size_t)idx[j] * kk + idx[j]] < T[(size_t)idx[i] * kk + idx[i]]) { int t = idx[i]; idx[i] = idx[j]; idx[j] = t; }
  for (int j = 0; j < kk; ++j) {
    theta[j] = T[(size_t)idx[j] * kk + idx[j]];
    zlast[j] = V[(size_t)(kk - 1) * kk + idx[j]];
  }
  const double res = beta[kk - 1];
  *b_out = theta[kk - 1] + std::fabs(res * zlast[kk - 1]);
  *a0_out = theta[0] - std::fabs(res * zlast[0]);
  return kk;
}

}  // extern "C"
