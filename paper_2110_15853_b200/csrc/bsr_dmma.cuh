// bsr_dmma.cuh -- the hot kernel: block-sparse H (b x b fp64 tiles) times a dense column tile of
// Y_k, with the recurrence's scale, shift and axpby fused into the epilogue
// (PAPER.md:L218, L221:  Y_{k+1} = alpha (H Y_k - c Y_k) + beta Y_{k-1};  L236: the SpMM is the kernel).
//
// sm_100a design:
//   * one CTA per (block row I, 128-column tile); 2*WR consumer warps (WR = b/32) + 1 producer warp
//   * the producer streams H_IJ[:, k0:k0+16] (b x 16) and Y_k[J*b+k0 : +16, 128 cols] through a
//     ring of NSTAGE shared-memory stages with TMA (cp.async.bulk.tensor.2d, SWIZZLE_128B) and
//     mbarrier full/empty pairs -- no thread ever computes a global address for operands
//   * consumers contract with fp64 tensor-core MMA (mma.sync.m8n8k4.f64 -> SASS DMMA.8x8x4; sm_100a
//     has no f64 kind in tcgen05), 32 x 64 per warp, accumulators in registers
//   * the k index and the row index inside an MMA are permuted so that every fragment load from the
//     swizzled stages is bank-conflict free (A: LDS.128, B: LDS.64)
//   * epilogue: out = alpha*acc + gamma*Y_k + beta*Y_{k-1} with 128-bit loads/stores
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace ttdft {

constexpr int K1_KS = 16;                  // k-slab per stage (16 doubles = one 128-byte swizzle row)
constexpr int K1_BGRP_BYTES = K1_KS * 128; // one 16-column group of a stage: 16 k-rows x 128 B

struct K1Params {
  const int32_t* brow_ptr;
  const int32_t* bcol;
  int32_t nb;          // block rows
  int32_t b;           // tile size of H (rows of a block row)
  int32_t rs;          // CTAs per block row along the rows: b / (32*WR)
  int32_t nct;         // column tiles = ceil(ncols/TN)
  int32_t cg;          // column tiles per scheduling group (L2 reuse of Y_k across block rows)
  int32_t vec;         // 1: S, Z, O are 16-byte aligned with even leading dimensions
  int32_t skip_empty = 0;   // 1: block rows without tiles are not this handle's: their output rows are left untouched
  int64_t ncols;
  double alpha, gamma, beta;
  const double* S;     // shift source (Y_k), read at the output position; unused if gamma == 0
  int64_t lds;
  const double* Z;     // Y_{k-1} (or Y for spmm), read at the output position; unused if beta == 0
  int64_t ldz;
  double* O;
  int64_t ldo;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int32_t x, int32_t y, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void dmma_8x8x4(double& c0, double& c1, double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}

// WR: row-warps (CTA rows BR = 32*WR); Q: 8-column MMA tiles per warp (CTA columns TN = 16*Q);
// CPS: CTAs resident per SM (2 lets one CTA's epilogue overlap the other's main loop).
template <int WR, int Q, int CPS, int RS = 1>
struct K1Cfg {
  static constexpr int BR = WR * 32;
  static constexpr int TN = 16 * Q;
  static constexpr int NGRP = Q;                       // 16-column groups per stage
  static constexpr int NCW = 2 * WR;                   // consumer warps
  static constexpr int THREADS = 32 * (NCW + 1);
  static constexpr int A_BYTES = BR * 128;
  static constexpr int STAGE_BYTES = A_BYTES + NGRP * K1_BGRP_BYTES;
  static constexpr int BUDGET = (CPS == 1 ? 200 : 100) * 1024;
  static constexpr int NSTAGE_RAW = BUDGET / STAGE_BYTES;
  static constexpr int NSTAGE = NSTAGE_RAW > 8 ? 8 : (NSTAGE_RAW < 3 ? 3 : NSTAGE_RAW);
  static constexpr int BAR_OFFSET = NSTAGE * STAGE_BYTES;
  static constexpr int TOTAL = BAR_OFFSET + 2 * NSTAGE * 8 + 1024;  // + alignment slack
};

// The consumer side of kernel K1 (MMA loop over the ring + fused epilogue), shared with the packed-storage variant
// (bsr_packed.cuh), which fills the A half of every stage by decoding instead of by TMA.
template <int WR, int Q, int CPS, int RS, int NSTG>
__device__ __forceinline__ void k1_consume(const K1Params& prm, uint8_t* smem, uint64_t* full, uint64_t* empty, int32_t I, int32_t rsi,
                                           int32_t col0, int32_t p_begin, int32_t p_end) {
  using SM = K1Cfg<WR, Q, CPS, RS>;
  constexpr int K1_NSTAGE = NSTG;  // stages of the ring (the packed variant runs a shorter one)
  constexpr int K1_TN = SM::TN;
  constexpr int BR = SM::BR;
  constexpr int32_t B = BR * RS;   // tile size of H
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // ================================ consumers: 32 x 64 per warp ================================
  const int wr = warp >> 1, wc = warp & 1;
  const int g = lane >> 2, t = lane & 3;
  const int rho = 4 * (g & 1) + (g >> 1);  // MMA row g  <->  tile row rho (bank-conflict-free LDS.128)

  double acc[4][Q][2];
#pragma unroll
  for (int p = 0; p < 4; ++p)
#pragma unroll
    for (int q = 0; q < Q; ++q) { acc[p][q][0] = 0.0; acc[p][q][1] = 0.0; }

  // per-lane byte offsets inside a stage
  const uint32_t a_row = (uint32_t)(32 * wr + rho) * 128u;
  const uint32_t a_off0 = a_row + (uint32_t)((t ^ rho) << 4);        // k = 2t, 2t+1
  const uint32_t a_off1 = a_row + (uint32_t)(((4 + t) ^ rho) << 4);  // k = 8+2t, 8+2t+1
  // B fragment of MMA tile q, step s: local column nl = wc*8Q + 8q + g -> 16-column group nl>>4, upper
  // half of the group (nl>>3)&1.  For even Q both are compile-time per q; for Q == 1 the half is wc.
  const uint32_t b_base = (uint32_t)SM::A_BYTES + (uint32_t)(2 * t) * 128u + (uint32_t)(g & 1) * 8u +
                          (Q >= 2 ? (uint32_t)(wc * (Q / 2)) * K1_BGRP_BYTES : 0u);
  const uint32_t Lx = ((uint32_t)((g >> 1) ^ (2 * t))) ^ (Q >= 2 ? 0u : 4u * (uint32_t)wc);

  const int nstages_total = (p_end - p_begin) * (B / K1_KS);
  int stage = 0;
  uint32_t phase = 0;
  const uint32_t smem_base = smem_u32(smem);
#pragma unroll 1
  for (int it = 0; it < nstages_total; ++it) {
    mbar_wait(&full[stage], phase);
    const uint32_t sb = smem_base + stage * SM::STAGE_BYTES;
    // A fragments: a[p][s], MMA step s uses k = 2t + (s&1) + 8(s>>1)
    double a[4][4];
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(a[p][0]), "=d"(a[p][1]) : "r"(sb + a_off0 + p * 1024u));
      asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(a[p][2]), "=d"(a[p][3]) : "r"(sb + a_off1 + p * 1024u));
    }
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      double bf[Q];
#pragma unroll
      for (int q = 0; q < Q; ++q) {
        const uint32_t cqs = (uint32_t)((Q >= 2 ? 4 * (q & 1) : 0) ^ (s & 1));
        const uint32_t off = b_base + (uint32_t)(q >> 1) * K1_BGRP_BYTES + (uint32_t)((s & 1) + 8 * (s >> 1)) * 128u + ((Lx ^ cqs) << 4);
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(bf[q]) : "r"(sb + off));
      }
#pragma unroll
      for (int p = 0; p < 4; ++p)
#pragma unroll
        for (int q = 0; q < Q; ++q) dmma_8x8x4(acc[p][q][0], acc[p][q][1], a[p][s], bf[q]);
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[stage]);
    if (++stage == K1_NSTAGE) { stage = 0; phase ^= 1; }
  }

  // ---- fused epilogue: out = alpha*acc + gamma*S + beta*Z at the output position ----
  // Loads are issued in batches of Q (one MMA row block at a time) so that many 128-bit requests are
  // in flight per thread; the producer warp has already pulled both tiles into L2.
  const double alpha = prm.alpha, gamma = prm.gamma, beta = prm.beta;
  const bool use_s = (gamma != 0.0), use_z = (beta != 0.0);
  const int64_t colw = (int64_t)col0 + 8 * Q * wc + 2 * t;   // + 8q
  if (prm.vec && col0 + K1_TN <= prm.ncols) {
    // fast path: whole tile inside the matrix, 16-byte aligned rows
    constexpr int QB = Q > 4 ? 4 : Q;   // loads in flight per operand and thread
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      const int64_t row = (int64_t)I * B + rsi * BR + 32 * wr + 8 * p + rho;
      const double* sp = prm.S + row * prm.lds + colw;
      const double* zp = prm.Z + row * prm.ldz + colw;
      double* op = prm.O + row * prm.ldo + colw;
#pragma unroll
      for (int q0 = 0; q0 < Q; q0 += QB) {
        double2 s2[QB], z2[QB];
        if (use_s) {
#pragma unroll
          for (int q = 0; q < QB; ++q) s2[q] = __ldg(reinterpret_cast<const double2*>(sp + 8 * (q0 + q)));
        }
        if (use_z) {
#pragma unroll
          for (int q = 0; q < QB; ++q) z2[q] = *reinterpret_cast<const double2*>(zp + 8 * (q0 + q));
        }
#pragma unroll
        for (int q = 0; q < QB; ++q) {
          double v0 = alpha * acc[p][q0 + q][0], v1 = alpha * acc[p][q0 + q][1];
          if (use_s) { v0 = fma(gamma, s2[q].x, v0); v1 = fma(gamma, s2[q].y, v1); }
          if (use_z) { v0 = fma(beta, z2[q].x, v0); v1 = fma(beta, z2[q].y, v1); }
          *reinterpret_cast<double2*>(op + 8 * (q0 + q)) = make_double2(v0, v1);
        }
      }
    }
    return;
  }
  // general path: ragged last column tile and/or unaligned views
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    const int64_t row = (int64_t)I * B + rsi * BR + 32 * wr + 8 * p + rho;
#pragma unroll
    for (int q = 0; q < Q; ++q) {
      const int64_t col = colw + 8 * q;
#pragma unroll
      for (int j = 0; j < 2; ++j) {
        if (col + j >= prm.ncols) continue;
        double v = alpha * acc[p][q][j];
        if (use_s) v = fma(gamma, prm.S[row * prm.lds + col + j], v);
        if (use_z) v = fma(beta, prm.Z[row * prm.ldz + col + j], v);
        prm.O[row * prm.ldo + col + j] = v;
      }
    }
  }
}

template <int WR, int Q, int CPS, int RS>
__global__ void __launch_bounds__(32 * (2 * WR + 1), CPS)
bsr_dmma_kernel(const __grid_constant__ CUtensorMap tmH, const __grid_constant__ CUtensorMap tmX, const K1Params prm) {
  using SM = K1Cfg<WR, Q, CPS, RS>;
  constexpr int NCW = SM::NCW;
  constexpr int K1_NSTAGE = SM::NSTAGE;
  constexpr int K1_TN = SM::TN;
  constexpr int K1_NGRP = SM::NGRP;
  constexpr int BR = SM::BR;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + SM::BAR_OFFSET);
  uint64_t* empty = full + K1_NSTAGE;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  // ---- tile decode: column-tile groups outermost, then block rows, column tile fastest ----
  int32_t I, ct, rsi;
  {
    const int64_t per_group = (int64_t)prm.nb * RS * prm.cg;
    const int32_t ngroups = (prm.nct + prm.cg - 1) / prm.cg;
    int32_t g = (int32_t)((int64_t)blockIdx.x / per_group);
    if (g > ngroups - 1) g = ngroups - 1;
    const int64_t rem = (int64_t)blockIdx.x - (int64_t)g * per_group;
    const int32_t width = min(prm.cg, prm.nct - g * prm.cg);
    const int64_t irs = rem / width;
    I = (int32_t)(irs / RS);
    rsi = (int32_t)(irs - (int64_t)I * RS);
    ct = g * prm.cg + (int32_t)(rem % width);
  }
  constexpr int32_t B = BR * RS;   // tile size of H
  const int32_t p_begin = prm.brow_ptr[I], p_end = prm.brow_ptr[I + 1];
  if (prm.skip_empty && p_begin == p_end) return;      // CTA-uniform, before any barrier
  const int32_t col0 = ct * K1_TN;
  const int32_t ngrp_valid = min(K1_NGRP, (int32_t)((prm.ncols - col0 + 15) / 16));

  if (threadIdx.x == 0) {
    for (int s = 0; s < K1_NSTAGE; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], NCW);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  if (warp == NCW) {
    // =========================== TMA producer (one elected lane) ===========================
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmH) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmX) : "memory");
      const uint32_t tx_bytes = SM::A_BYTES + ngrp_valid * K1_BGRP_BYTES;
      int stage = 0;
      uint32_t phase = 0;
      for (int32_t p = p_begin; p < p_end; ++p) {
        const int32_t J = prm.bcol[p];
#pragma unroll 1
        for (int k0 = 0; k0 < B; k0 += K1_KS) {
          mbar_wait(&empty[stage], phase ^ 1);
          uint8_t* As = smem + stage * SM::STAGE_BYTES;
          uint8_t* Bs = As + SM::A_BYTES;
          mbar_expect_tx(&full[stage], tx_bytes);
          tma_load_2d(As, &tmH, k0, p * B + rsi * BR, &full[stage]);
          for (int g = 0; g < ngrp_valid; ++g)
            tma_load_2d(Bs + g * K1_BGRP_BYTES, &tmX, col0 + g * 16, J * B + k0, &full[stage]);
          if (++stage == K1_NSTAGE) { stage = 0; phase ^= 1; }
        }
      }
    }
    __syncwarp();
    // The ring now holds the last NSTAGE slabs of work: use that time to pull the epilogue's operands
    // (Y_k and Y_{k-1} at the output tile) into L2, one 128-byte line per lane and request.
    {
      const int64_t row0 = (int64_t)I * B + rsi * BR;
      const int64_t ncl = min((int64_t)K1_TN, prm.ncols - col0);     // valid columns of this tile
      const int lines_per_row = (int)((ncl * 8 + 127) / 128);
      const int total = BR * lines_per_row;
      for (int idx = lane; idx < total; idx += 32) {
        const int r = idx / lines_per_row, l = idx - r * lines_per_row;
        if (prm.beta != 0.0) {
          const double* zp = prm.Z + (row0 + r) * prm.ldz + col0 + l * 16;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(zp));
        }
        if (prm.gamma != 0.0) {
          const double* sp = prm.S + (row0 + r) * prm.lds + col0 + l * 16;
          asm volatile("prefetch.global.L2 [%0];" ::"l"(sp));
        }
      }
    }
    return;
  }

  k1_consume<WR, Q, CPS, RS, SM::NSTAGE>(prm, smem, full, empty, I, rsi, col0, p_begin, p_end);
}

}  // namespace ttdft
