// bsr_i8t.cuh -- kernel K3T: the filter step of bsr_i8.cuh,  O = alpha*(H*Y_k) + gamma*Y_k + beta*Y_{k-1}  (PAPER.md:L218, L221,
// L236), in the TRANSPOSED formulation  O^T = Y_k^T H^T : the digit planes of Y_k are the A operand of the tensor-core product
// (M = 128 COLUMNS of Y per CTA), the digit planes of the H tile the B operand (N = rows of the tile x digit levels).
//
// Why: K3 puts the rows of a block row on the M = 128 axis of tcgen05.mma.  Tiles narrower than 128 then
// multiply padding rows -- a quarter of the tensor work at b = 96 (BASELINE.json config 4).  Here the tile's rows sit on the N axis,
// which takes any multiple of 16: a CTA works on HR = b/2 rows, N = HR * (S - q) for Y plane q against the concatenation of H planes
// 0..S-1-q (level g = p + q lives at TMEM columns [g*HR, g*HR + HR)), and no padding is multiplied: 2 x 2,016 tensor cycles per
// (96 rows x 128 columns x tile) instead of 2 x 2,688.
//
//   * work item = (block row I, 128-column tile); the two CTAs of a cluster take the two row halves of the block row, so they need
//     the SAME Y digit planes: every plane (128 columns x 128 k-bytes, two adjacent 64-column digit tiles) is fetched half by each
//     CTA and MULTICAST into the same ring slot of both (the mirror image of K3, which multicasts the H planes)
//   * warp 0 (one lane): TMA producer -- per tile (I,J) ONE 3-D load of its half of the H tile (S planes x HR rows x 128 B, double
//     buffered) and S multicast loads of Y planes through a ring of 16 KB slots
//   * warp 1 (one lane): tcgen05.mma.kind::i8 issuer, M = 128, K = 32, N = HR*(S-q) (two nearly equal pieces above 256)
//   * warps 2-9: epilogue.  A TMEM lane is a COLUMN of Y, so lane l of a warp owns column l and its registers hold rows: every
//     load of Y_k / Y_{k-1} and every store is one contiguous 256-byte row segment WITHOUT the register transposition K3 needs;
//     ragged column tiles are plain lane predicates.  Column maxima and the next step's digit planes as in K3.
#pragma once
#include "bsr_i8.cuh"
#include "gram_i8.cuh"   // tma_load_4d, tma_load_4d_mc

namespace ttdft {

constexpr int K3T_NT = 128;      // columns per work item

template <int S, int HR>
struct K3TCfg {
  static constexpr int HBUF = S * HR * 128;               // one half tile of H: S planes x HR rows x 128 k-bytes
  static constexpr int YSLOT = 128 * 128;                 // one digit plane of 128 columns
  static constexpr int NY = (232448 - 4096 - 2 * HBUF) / YSLOT;
  static constexpr int BAR_OFFSET = 2 * HBUF + NY * YSLOT;
  static constexpr int NBAR = 4 + 2 * NY + 2;
  static constexpr int CE_OFFSET = BAR_OFFSET + 8 * ((NBAR + 1) & ~1);   // 128 ints: exponents of the digits of Y_k
  static constexpr int CP_OFFSET = CE_OFFSET + 128 * 4;                  // 128 ints: predicted exponents of the output columns
  static constexpr int CM_OFFSET = CP_OFFSET + 128 * 4;                  // 128 words: column maxima of the output
  static constexpr int RS_OFFSET = CM_OFFSET + 128 * 4;                  // HR doubles: alpha 2^(eH_i - 30)
  static constexpr int GI_OFFSET = RS_OFFSET + 64 * 8;                   // HR doubles: alpha hdiag_i + gamma
  static constexpr int TM_OFFSET = GI_OFFSET + 64 * 8;                   // tmem slot
  static constexpr int Q_OFFSET = TM_OFFSET + 16;                        // work-item queue (K3Queue)
  static constexpr int TOTAL = Q_OFFSET + 192 + 1024;                    // + alignment slack
  static_assert(HR % 16 == 0 && HR <= 64, "rows per CTA: a multiple of 16 (8-row swizzle atoms, 8-row epilogue groups per half)");
  static_assert(S * HR <= 512, "digit levels must fit TMEM");
  static_assert(HBUF % 1024 == 0, "swizzle atoms");
  static_assert(NY >= 3, "Y ring too short");
};

__device__ __forceinline__ void tma_load_4d_mc_hint(void* dst, const CUtensorMap* map, int32_t x, int32_t y, int32_t z, int32_t w,
                                                    uint64_t* bar, uint16_t mask, uint64_t hint) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint [%0], [%1, {%2, %3, %4, %5}], [%6], %7, %8;" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(w), "r"(smem_u32(bar)), "h"(mask), "l"(hint)
      : "memory");
}

// tmH3: 3-D map {128 B, b rows, tiles x stored planes} of the H digit planes, box {128 B, HR rows, S planes};
// tmY4: 4-D map {128 B, 64 columns, S planes, digit tiles} of the Y digit tiles, box {128 B, 64, 1, 1}.
// prm.nct = 64-column digit tiles per block row (EVEN); prm.ct_begin / prm.nctg count 128-column tiles.  Clusters of 2.
template <int S, int HR>
__global__ void __launch_bounds__(K3_THREADS, 1)
bsr_i8t_kernel(const __grid_constant__ CUtensorMap tmH3, const __grid_constant__ CUtensorMap tmY4, const K3Params prm) {
  using Cf = K3TCfg<S, HR>;
  constexpr int NY = Cf::NY;
  constexpr int NR = HR / 2;                     // rows per epilogue warp
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* hbuf = smem;                          // 2 x HBUF
  uint8_t* yring = smem + 2 * Cf::HBUF;           // NY x YSLOT
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cf::BAR_OFFSET);
  uint64_t* hfull = bars;                        // [2]
  uint64_t* hempty = bars + 2;                   // [2]
  uint64_t* yfull = bars + 4;                    // [NY]
  uint64_t* yempty = bars + 4 + NY;              // [NY]
  uint64_t* accfull = bars + 4 + 2 * NY;
  uint64_t* accempty = accfull + 1;
  int32_t* ce_s = reinterpret_cast<int32_t*>(smem + Cf::CE_OFFSET);
  int32_t* cp_s = reinterpret_cast<int32_t*>(smem + Cf::CP_OFFSET);
  uint32_t* cm_s = reinterpret_cast<uint32_t*>(smem + Cf::CM_OFFSET);
  double* rs_s = reinterpret_cast<double*>(smem + Cf::RS_OFFSET);
  double* gi_s = reinterpret_cast<double*>(smem + Cf::GI_OFFSET);
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + Cf::TM_OFFSET);
  K3Queue* wq = reinterpret_cast<K3Queue*>(smem + Cf::Q_OFFSET);          // work items of this cluster (bsr_i8.cuh)

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t nitems = (uint32_t)((int64_t)prm.nb * prm.nctg);   // cluster work items (< 2^32, checked on the host)
  const int32_t crank = (int32_t)cluster_ctarank();           // which half of the block row's rows
  constexpr uint16_t cmask = 3;
  constexpr int C = 2;
  const int32_t b = prm.b;
  const int32_t ksteps = b >> 5;                 // 32-deep int8 MMAs per tile of H

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(&hfull[i], 1); mbar_init(&hempty[i], 1); }
    for (int i = 0; i < NY; ++i) { mbar_init(&yfull[i], 1); mbar_init(&yempty[i], 2); }   // a slot is free once both CTAs have read it
    mbar_init(accfull, 1);
    mbar_init(accempty, 256);
    for (int i = 0; i < K3_NQ; ++i) { mbar_init(&wq->qfull[i], 1); mbar_init(&wq->qempty[i], C * K3_QCONS); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  cluster_sync_all();                            // the peer's barriers are initialised before anything is sent to them
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===================================== TMA producer =====================================
    if (elect_one()) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmH3) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmY4) : "memory");
      int hb = 0, ys = 0;
      uint32_t hph = 0, yph = 0;
      int qs = 0;
      uint32_t qph = 0;
      K3Fetch fetch;
      if (crank == 0)
        for (int i = 0; i < K3_QAHEAD; ++i) k3_q_fetch<C>(wq, fetch, prm.counter, nitems);
      for (;;) {
        const uint32_t u = k3_q_pop(wq, qs, qph, true);
        if (u == K3_NOITEM) break;
        if (crank == 0) k3_q_fetch<C>(wq, fetch, prm.counter, nitems);
        int32_t I, ctg;
        k3_decode(prm, u, I, ctg);
        const int32_t ct = prm.ct_begin + ctg;
        const int32_t p0 = prm.brow_ptr[I], p1 = prm.brow_ptr[I + 1];
        for (int32_t p = p0; p < p1; ++p) {
          const int32_t J = prm.bcol[p];
          mbar_wait(&hempty[hb], hph ^ 1);
          mbar_expect_tx(&hfull[hb], (uint32_t)Cf::HBUF);
          if (prm.l2hints == 1) tma_load_3d_hint(hbuf + hb * Cf::HBUF, &tmH3, 0, crank * HR, p * prm.hplanes, &hfull[hb], L2_EVICT_FIRST);
          else tma_load_3d(hbuf + hb * Cf::HBUF, &tmH3, 0, crank * HR, p * prm.hplanes, &hfull[hb]);
          const int32_t ytile = J * prm.nct + 2 * ct + crank;        // this CTA's half: 64 of the plane's 128 columns
#pragma unroll 1
          for (int q = 0; q < S; ++q) {
            mbar_wait(&yempty[ys], yph ^ 1);       // both CTAs have finished with this slot
            mbar_expect_tx(&yfull[ys], (uint32_t)Cf::YSLOT);
            uint8_t* dst = yring + ys * Cf::YSLOT + crank * 8192;
            if (prm.l2hints) tma_load_4d_mc_hint(dst, &tmY4, 0, 0, q, ytile, &yfull[ys], cmask, L2_EVICT_LAST);
            else tma_load_4d_mc(dst, &tmY4, 0, 0, q, ytile, &yfull[ys], cmask);
            if (++ys == NY) { ys = 0; yph ^= 1; }
          }
          hb ^= 1;
          if (hb == 0) hph ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ====================================== MMA issuer ======================================
    if (elect_one()) {
      int hb = 0, ys = 0;
      uint32_t hph = 0, yph = 0, aph = 0;
      const uint64_t dbase = umma_desc_sw128(0);
      const uint32_t hlo0 = (smem_u32(hbuf) & 0x3ffffu) >> 4, ylo0 = (smem_u32(yring) & 0x3ffffu) >> 4;
      int qs = 0;
      uint32_t qph = 0;
      for (;;) {
        const uint32_t u = k3_q_pop(wq, qs, qph, true);
        if (u == K3_NOITEM) break;
        int32_t I, ctg;
        k3_decode(prm, u, I, ctg);
        const int32_t nJ = prm.brow_ptr[I + 1] - prm.brow_ptr[I];
        if (nJ == 0) continue;
        mbar_wait(accempty, aph ^ 1);            // the epilogue has drained the previous item's accumulators
        asm volatile("tcgen05.fence::after_thread_sync;");
        for (int32_t j = 0; j < nJ; ++j) {
          mbar_wait(&hfull[hb], hph);
          const uint32_t hlo = hlo0 + (uint32_t)hb * (Cf::HBUF >> 4);
#pragma unroll
          for (int q = 0; q < S; ++q) {
            mbar_wait(&yfull[ys], yph);
            asm volatile("tcgen05.fence::after_thread_sync;");
            const uint32_t ylo = ylo0 + (uint32_t)ys * (Cf::YSLOT >> 4);
            const int ntot = (S - q) * HR;          // H planes 0..S-1-q side by side -> levels q..S-1
            const int n1 = ntot > 256 ? ((ntot / 2 + 15) / 16) * 16 : ntot;
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              if (kk < ksteps) {
                const uint64_t da = dbase | (uint64_t)(ylo + kk * 2);    // A: Y plane q, 128 columns of Y x 32 k-bytes
                // plane 0 comes first and spans every level: its first MMA of a work item overwrites the accumulators
                const uint32_t acc = (q > 0 || kk > 0) ? 1u : (j > 0 ? 1u : 0u);
                if (n1 < ntot) {                    // two instructions, A read once (collector fill + lastuse)
                  umma_i8<1>(tmem_base + (uint32_t)(q * HR), da, dbase | (uint64_t)(hlo + kk * 2), umma_idesc_i8(n1), acc);
                  umma_i8<2>(tmem_base + (uint32_t)(q * HR + n1), da, dbase | (uint64_t)(hlo + n1 * 8 + kk * 2), umma_idesc_i8(ntot - n1), acc);
                } else {
                  umma_i8(tmem_base + (uint32_t)(q * HR), da, dbase | (uint64_t)(hlo + kk * 2), umma_idesc_i8(n1), acc);
                }
              }
            }
            umma_commit_mc(&yempty[ys], cmask);     // slot free (in both CTAs) once these MMAs have read it
            if (++ys == NY) { ys = 0; yph ^= 1; }
          }
          umma_commit(&hempty[hb]);
          hb ^= 1;
          if (hb == 0) hph ^= 1;
        }
        umma_commit(accfull);
        aph ^= 1;
      }
    }
  } else {
    // ======================================= epilogue =======================================
    // 8 warps: warp w reads TMEM lane quarter w & 3 (columns 32q..32q+31 of the item's 128) and row half (w - 2) >> 2 of the CTA's
    // HR rows.  Lane l owns one column; its registers run over rows.
    const int quarter = warp & 3;
    const int rh = (warp - 2) >> 2;
    const int et = (warp - 2) * 32 + lane;       // 0..255 among the epilogue threads
    const int cl = quarter * 32 + lane;          // column inside the item
    const double beta = prm.beta;
    const bool use_z = (beta != 0.0);
    const bool use_s = (prm.S != nullptr);
    const bool digits_out = (prm.dO != nullptr);
    uint32_t aph = 0;
    int qs = 0;
    uint32_t qph = 0;
    for (;;) {
      const uint32_t u = k3_q_pop_warp(wq, qs, qph);
      if (u == K3_NOITEM) break;
      int32_t I, ctg;
      k3_decode(prm, u, I, ctg);
      const int32_t ct = prm.ct_begin + ctg;
      const int32_t nJ = prm.brow_ptr[I + 1] - prm.brow_ptr[I];
      if (prm.skip_empty && nJ == 0) continue;           // uniform over the epilogue warps
      const int64_t col = (int64_t)ct * K3T_NT + cl;
      const bool col_ok = col < prm.ncols;
      const int64_t row0 = (int64_t)I * b + crank * HR;        // first row of this CTA
      if (et < 128) {
        const int64_t cj = (int64_t)ct * K3T_NT + et;
        ce_s[et] = cj < prm.ncols ? prm.eS[cj] : I8_EMIN;
        cm_s[et] = 0;
        if (digits_out) cp_s[et] = cj < prm.ncols ? prm.ePredO[cj] : I8_EMIN;
      } else if (et - 128 < HR) {
        const int64_t row = row0 + (et - 128);
        rs_s[et - 128] = prm.alpha * pow2i(prm.eH[row] - 30);   // alpha * 2^(eH_i - 14) / 2^16 (k3_drain returns 2^16 * v)
        gi_s[et - 128] = prm.hdiag ? fma(prm.alpha, prm.hdiag[row], prm.gamma) : prm.gamma;
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");

      double v[NR];
      if (nJ > 0) {
        mbar_wait(accfull, aph);
        aph ^= 1;
        asm volatile("tcgen05.fence::after_thread_sync;");
        k3_drain<S, NR, HR>(tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(rh * NR), v);
        asm volatile("tcgen05.fence::before_thread_sync;");
        mbar_arrive(accempty);                   // TMEM is free for the next work item
      } else {
#pragma unroll
        for (int i = 0; i < NR; ++i) v[i] = 0.0;
      }

      // ---- out = alpha * 2^(eH+eY-30) * v + (alpha*hdiag + gamma) * y + beta * z   (v = 2^16 * Horner) ----
      const int32_t ce = ce_s[cl];
      const int32_t cpred = digits_out ? cp_s[cl] : 0;
      const double dscale = pow2i(8 * S - 1 - cpred);
      const int64_t wrow0 = row0 + rh * NR;                      // first row of this warp
      const double* sw = prm.S + wrow0 * prm.lds + col;
      const double* zw = prm.Z + wrow0 * prm.ldz + col;
      double* ow = prm.O + wrow0 * prm.ldo + col;
      // digit tile of (block row I, 64-column tile 2 ct + quarter / 2), row (plane, column), k bytes of this warp's rows
      uint8_t* dtile = digits_out ? reinterpret_cast<uint8_t*>(prm.dO) +
                                        ((int64_t)I * prm.nct + 2 * ct + (quarter >> 1)) * (int64_t)(S * K3_NT * 128) +
                                        ((quarter & 1) * 32 + lane) * 128 + crank * HR + rh * NR
                                  : nullptr;
      uint32_t cmx = 0;                           // column maximum (upper word) this lane has seen
      // digit words of this lane's column are collected over CH rows (plane q, rows c0 + 4 w .. c0 + 4 w + 3) and stored as few
      // and as wide as the alignment allows: a lane's row is 128 bytes from its neighbour's, so every store instruction costs 32
      // sectors whatever its width
      constexpr int CH = (NR % 16 == 0) ? 16 : NR;
      uint32_t dwd[S][CH / 4];
#pragma unroll
      for (int c0 = 0; c0 < NR; c0 += CH) {
#pragma unroll
      for (int r0 = c0; r0 < c0 + CH; r0 += 8) {
        double y[8], z[8], ov[8];
        if (use_s) {
#pragma unroll
          for (int i = 0; i < 8; ++i) y[i] = col_ok ? __ldcs(sw + (int64_t)(r0 + i) * prm.lds) : 0.0;   // read once: evict first
        }
        if (use_z) {
#pragma unroll
          for (int i = 0; i < 8; ++i) z[i] = col_ok ? __ldcs(zw + (int64_t)(r0 + i) * prm.ldz) : 0.0;
        }
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          double o = scale_pow2(v[r0 + i] * rs_s[rh * NR + r0 + i], ce);
          if (use_s) o = fma(gi_s[rh * NR + r0 + i], y[i], o);
          if (use_z) o = fma(beta, z[i], o);
          if (!col_ok) o = 0.0;                   // columns beyond the panel: nothing stored, zero digits
          ov[i] = o;
          if (col_ok) {
            __stcs(ow + (int64_t)(r0 + i) * prm.ldo, o);
            cmx = max(cmx, abs_hi(o));
          }
        }
        if (digits_out) {
          uint32_t w0[S], w1[S];
          const double x0[4] = {ov[0], ov[1], ov[2], ov[3]}, x1[4] = {ov[4], ov[5], ov[6], ov[7]};
          digits4<S>(x0, dscale, w0);
          digits4<S>(x1, dscale, w1);
#pragma unroll
          for (int q = 0; q < S; ++q) { dwd[q][(r0 - c0) / 4] = w0[q]; dwd[q][(r0 - c0) / 4 + 1] = w1[q]; }
        }
      }
      if (digits_out) {
        const bool lead8 = ((crank * HR + rh * NR + c0) & 8) != 0;   // warp-uniform: the piece starts 8 bytes into a 16-byte unit
#pragma unroll
        for (int q = 0; q < S; ++q) {
          uint8_t* dq = dtile + q * (K3_NT * 128) + c0;
          if (lead8) {
            *reinterpret_cast<uint2*>(dq) = make_uint2(dwd[q][0], dwd[q][1]);
#pragma unroll
            for (int w = 2; w + 4 <= CH / 4; w += 4)
              *reinterpret_cast<uint4*>(dq + 4 * w) = make_uint4(dwd[q][w], dwd[q][w + 1], dwd[q][w + 2], dwd[q][w + 3]);
            if ((CH / 4 - 2) % 4 != 0)
              *reinterpret_cast<uint2*>(dq + CH - 8) = make_uint2(dwd[q][CH / 4 - 2], dwd[q][CH / 4 - 1]);
          } else {
#pragma unroll
            for (int w = 0; w + 4 <= CH / 4; w += 4)
              *reinterpret_cast<uint4*>(dq + 4 * w) = make_uint4(dwd[q][w], dwd[q][w + 1], dwd[q][w + 2], dwd[q][w + 3]);
            if ((CH / 4) % 4 != 0)
              *reinterpret_cast<uint2*>(dq + CH - 8) = make_uint2(dwd[q][CH / 4 - 2], dwd[q][CH / 4 - 1]);
          }
        }
      }
      }
      if (digits_out) {
        // the k bytes beyond the tile's rows (b < 128) stay zero: written by the warp that owns the last rows
        if (crank == 1 && rh == 1) {
          for (int k0 = b; k0 < 128; k0 += 8)
#pragma unroll
            for (int q = 0; q < S; ++q)
              *reinterpret_cast<uint2*>(dtile - (crank * HR + rh * NR) + q * (K3_NT * 128) + k0) = make_uint2(0u, 0u);
        }
        // a column that outgrew its predicted exponent: its digits are invalid, the tile is redone before the next step
        if (col_ok && exp_from_hi(cmx) > cpred) atomicOr(&prm.flagsO[2 * ct + (quarter >> 1)], 1u);
      }
      // ---- column maxima of the new iterate (upper words), for the next step's digit scaling ----
      if (prm.cmaxO) {
        if (cmx) atomicMax(&cm_s[cl], cmx);
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (et < 128 && (int64_t)ct * K3T_NT + et < prm.ncols && cm_s[et]) atomicMax(&prm.cmaxO[(int64_t)ct * K3T_NT + et], cm_s[et]);
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");   // the shared arrays are rewritten by the next item
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  cluster_sync_all();                            // no CTA leaves while the peer may still signal its barriers
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512));
}

}  // namespace ttdft
