// recover.cuh -- A0 for a CSR whose rows arrive in arbitrary order WITHOUT subdomain labels (SURVEY.md 8(a) A0 "group rows so
// each subdomain's basis functions are contiguous"; 8(f)-4 "locality recovery for unhinted CSR").  The paper states only the
// structure that makes this possible (the functions of a subdomain overlap each other -- dense diagonal
// blocks -- and those of the neighbouring subdomains); the rule is DESIGN.md reading #18, all in exact integer arithmetic:
//   N(i) = column set of row i;  c_ij = |N(i) & N(j)|,  u_ij = |N(i)| + |N(j)| - c_ij  for j in N(i), j != i   (Jaccard c/u)
//   (1) S(i) = {i} + {j : 5 c_ij u* >= 4 c* u_ij},  (c*, u*) = the row's largest fraction          rc_candidates_kernel
//   (2) V(i) = {j in S(i) : 2 |S(i) & S(j)| >= max(|S(i)|, |S(j)|)}                                 rc_verify_kernel
//   (3) root(i) = smallest row reachable along i -> V(i)                                             rc_propagate_kernel (iterated)
//   (4) roots numbered in ascending order; label(i) = number of root(i)                              rc_number_roots_kernel, rc_label_kernel
// Pure integer / index work: one CTA per row keeps the row's column set as an M-bit map in shared memory and every warp counts
// one neighbour's columns against it (coalesced reads of col_idx, one shared-memory lookup per entry).
#pragma once
#include <cstdint>

namespace ttdft {

constexpr int RC_CAP = 192;             // largest candidate set |S(i)| (the largest tile has 128 rows)
constexpr int RC_MASKW = RC_CAP / 32;   // words of the verified-pair mask of a row
constexpr int RC_T1 = 512;              // threads of rc_candidates_kernel
constexpr int RC_T2 = 256;              // threads of rc_verify_kernel

// out[0] = longest row
__global__ void rc_maxlen_kernel(int64_t M, const int32_t* __restrict__ rp, int32_t* __restrict__ out) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int32_t v = (i < M) ? rp[i + 1] - rp[i] : 0;
  for (int o = 16; o; o >>= 1) v = max(v, __shfl_xor_sync(0xffffffffu, v, o));
  if ((threadIdx.x & 31) == 0 && v > 0) atomicMax(out, v);
}

__device__ __forceinline__ bool rc_frac_greater(int32_t c1, int32_t u1, int32_t c2, int32_t u2) {   // c1/u1 > c2/u2
  return (int64_t)c1 * u2 > (int64_t)c2 * u1;
}

// (1) grid M, RC_T1 threads.  dynamic smem: bitmap[W] | c[maxlen] | u[maxlen].  S: M x RC_CAP, nS: M.  flags[1] |= 1 if a set overflows.
__global__ void __launch_bounds__(RC_T1) rc_candidates_kernel(int64_t M, const int32_t* __restrict__ rp, const int32_t* __restrict__ col,
                                                             int32_t W, int32_t maxlen, int32_t* __restrict__ S, int32_t* __restrict__ nS,
                                                             int32_t* __restrict__ flags) {
  extern __shared__ uint32_t rc_smem[];
  uint32_t* bm = rc_smem;
  int32_t* cc = reinterpret_cast<int32_t*>(rc_smem + W);
  int32_t* uu = cc + maxlen;
  __shared__ int32_t wc[RC_T1 / 32], wu[RC_T1 / 32];
  __shared__ int32_t n_sel, best_c, best_u;
  const int32_t i = (int32_t)blockIdx.x;
  const int32_t s = rp[i], len = rp[i + 1] - s;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int w = tid; w < W; w += RC_T1) bm[w] = 0u;
  if (tid == 0) n_sel = 1;
  __syncthreads();
  for (int t = tid; t < len; t += RC_T1) {
    const int32_t k = col[s + t];
    if ((uint32_t)k < (uint32_t)M) atomicOr(&bm[k >> 5], 1u << (k & 31));      // an out-of-range column (invalid input) is ignored, not a fault
  }
  __syncthreads();
  // one warp per neighbour j: c = number of columns of row j that are columns of row i
  for (int t = warp; t < len; t += RC_T1 / 32) {
    const int32_t j = col[s + t];
    const bool valid = (uint32_t)j < (uint32_t)M && j != i;
    const int32_t sj = valid ? rp[j] : 0, lj = valid ? rp[j + 1] - sj : 0;
    int32_t c = 0;
    for (int q = lane; q < lj; q += 32) {
      const int32_t k = __ldg(col + sj + q);
      if ((uint32_t)k < (uint32_t)M) c += (bm[k >> 5] >> (k & 31)) & 1u;
    }
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) { cc[t] = valid ? c : -1; uu[t] = len + lj - c; }
  }
  __syncthreads();
  // largest fraction of the row
  int32_t bc = 0, bu = 1;
  for (int t = tid; t < len; t += RC_T1)
    if (cc[t] >= 0 && rc_frac_greater(cc[t], uu[t], bc, bu)) { bc = cc[t]; bu = uu[t]; }
  for (int o = 16; o; o >>= 1) {
    const int32_t oc = __shfl_xor_sync(0xffffffffu, bc, o), ou = __shfl_xor_sync(0xffffffffu, bu, o);
    if (rc_frac_greater(oc, ou, bc, bu)) { bc = oc; bu = ou; }
  }
  if (lane == 0) { wc[warp] = bc; wu[warp] = bu; }
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < RC_T1 / 32; ++w)
      if (rc_frac_greater(wc[w], wu[w], bc, bu)) { bc = wc[w]; bu = wu[w]; }
    best_c = bc; best_u = bu;
    S[(int64_t)i * RC_CAP] = i;
  }
  __syncthreads();
  bc = best_c; bu = best_u;
  if (bc > 0)
    for (int t = tid; t < len; t += RC_T1)
      if (cc[t] >= 0 && 5ll * cc[t] * bu >= 4ll * bc * uu[t]) {
        const int pos = atomicAdd(&n_sel, 1);
        if (pos < RC_CAP) S[(int64_t)i * RC_CAP + pos] = col[s + t];
      }
  __syncthreads();
  if (tid == 0) {
    nS[i] = min(n_sel, RC_CAP);
    if (n_sel > RC_CAP) atomicOr(&flags[1], 1);
  }
}

// (2) grid M, RC_T2 threads.  dynamic smem: bitmap[W].  Vm: M x RC_MASKW, bit t of row i <=> S(i)[t] is verified.
// Also the first propagation step: L[i] = smallest verified member.
__global__ void __launch_bounds__(RC_T2) rc_verify_kernel(int64_t M, int32_t W, const int32_t* __restrict__ S, const int32_t* __restrict__ nS,
                                                         uint32_t* __restrict__ Vm, int32_t* __restrict__ L) {
  extern __shared__ uint32_t rc_smem[];
  uint32_t* bm = rc_smem;
  __shared__ int32_t Si[RC_CAP];
  __shared__ uint32_t mask[RC_MASKW];
  __shared__ int32_t lmin;
  const int32_t i = (int32_t)blockIdx.x;
  const int32_t ni = nS[i];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int w = tid; w < W; w += RC_T2) bm[w] = 0u;
  if (tid < RC_MASKW) mask[tid] = 0u;
  if (tid == 0) lmin = i;
  __syncthreads();
  for (int t = tid; t < ni; t += RC_T2) {
    const int32_t k = S[(int64_t)i * RC_CAP + t];
    Si[t] = k;
    atomicOr(&bm[k >> 5], 1u << (k & 31));
  }
  __syncthreads();
  for (int t = warp; t < ni; t += RC_T2 / 32) {
    const int32_t j = Si[t];
    const int32_t nj = nS[j];
    int32_t c = 0;
    for (int q = lane; q < nj; q += 32) {
      const int32_t k = S[(int64_t)j * RC_CAP + q];
      c += (bm[k >> 5] >> (k & 31)) & 1u;
    }
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0 && 2 * c >= max(ni, nj)) {
      atomicOr(&mask[t >> 5], 1u << (t & 31));
      atomicMin(&lmin, j);
    }
  }
  __syncthreads();
  if (tid < RC_MASKW) Vm[(int64_t)i * RC_MASKW + tid] = mask[tid];
  if (tid == 0) L[i] = lmin;
}

// (3) one warp per row: L[i] = min(L[i], L[j] for verified j, L[L[i]]); flags[2] = 1 if anything changed.  Monotone, so the
// unsynchronised reads of other rows' labels are harmless; the host repeats the launch until nothing changes.
__global__ void __launch_bounds__(256) rc_propagate_kernel(int64_t M, const int32_t* __restrict__ S, const int32_t* __restrict__ nS,
                                                           const uint32_t* __restrict__ Vm, int32_t* L, int32_t* __restrict__ flags) {
  const int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= M) return;
  const int32_t ni = nS[i];
  volatile int32_t* Lv = L;
  const int32_t cur = Lv[i];
  int32_t m = cur;
  for (int t = lane; t < ni; t += 32)
    if ((Vm[i * RC_MASKW + (t >> 5)] >> (t & 31)) & 1u) m = min(m, Lv[S[i * RC_CAP + t]]);
  for (int o = 16; o; o >>= 1) m = min(m, __shfl_xor_sync(0xffffffffu, m, o));
  m = min(m, Lv[m]);
  if (lane == 0 && m < cur) { atomicMin(&L[i], m); flags[2] = 1; }
}

// (4a) one CTA of 1024 threads: ids[r] = rank of root r among the roots (L[r] == r) in ascending order; flags[3] = number of roots
__global__ void __launch_bounds__(1024) rc_number_roots_kernel(int64_t M, const int32_t* __restrict__ L, int32_t* __restrict__ ids,
                                                               int32_t* __restrict__ flags) {
  __shared__ int32_t part[1024];
  const int tid = threadIdx.x;
  const int64_t chunk = (M + 1023) / 1024;
  const int64_t lo = min(M, tid * chunk), hi = min(M, lo + chunk);
  int32_t n = 0;
  for (int64_t r = lo; r < hi; ++r) n += (L[r] == (int32_t)r);
  part[tid] = n;
  __syncthreads();
  for (int o = 1; o < 1024; o <<= 1) {                 // inclusive scan
    const int32_t v = (tid >= o) ? part[tid - o] : 0;
    __syncthreads();
    part[tid] += v;
    __syncthreads();
  }
  int32_t k = part[tid] - n;
  for (int64_t r = lo; r < hi; ++r)
    if (L[r] == (int32_t)r) ids[r] = k++;
  if (tid == 1023) flags[3] = part[1023];
}

// (4b) label(i) = number of root(i)
__global__ void rc_label_kernel(int64_t M, const int32_t* __restrict__ L, const int32_t* __restrict__ ids, int32_t* __restrict__ labels) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < M) labels[i] = ids[L[i]];
}

}  // namespace ttdft
