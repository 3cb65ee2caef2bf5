// gram_i8.cuh -- kernel K4: G = X^T W for two tall M x N fp64 blocks, the second half of the subspace
// projection H_F = X_F^T (H X_F) (Algorithm 1 step 3; Sec. 4.3: "this matrix is ...
// left-multiplied with X^T").  The paper does this product on the host with PETSc; here it runs on the int8
// tensor cores with the same exact digit-plane arithmetic as K3 (bsr_i8.cuh, i8_digits.cuh):
//
//   G[j,l] = sum_k x_kj w_kl = 2^(eX_j + eW_l - 14) * Horner_g( L_g[j,l] )  (scaled by exponent adds, no fp64 multiply),   L_g = sum_{p+q=g} dX_p^T dW_q   (int32, exact)
//
// Both operands come from y_digits_kernel: D[block][64-column tile][S planes][64 columns][128 k-bytes], i.e.
// K-major rows of 128 contraction indices -- exactly what both tcgen05 operands want.  The A operand of one MMA
// (M = 128) is plane p of TWO adjacent 64-column tiles of X (one 4-D TMA box -> one 16 KB slot), the B operand
// the concatenation of planes 0..S-1-p of one 64-column tile of W, as in K3.
//
// Work item = (128 columns of X = rows of G, 64 columns of W = columns of G, chunk of <= kc 128-row blocks of
// the contraction).  A chunk is short enough for exact int32 accumulation (S * kc * 128 * 2^14 < 2^31) and
// writes its partial tile to P[chunk][.][.]; gram_reduce_kernel then sums the chunks in a fixed order, so the
// result is deterministic (no floating-point atomics).  Clusters of C CTAs along the columns of W share the A
// planes by TMA multicast.
#pragma once
#include "bsr_i8.cuh"

namespace ttdft {

struct K4Params {
  int32_t nbk;                 // 128-row blocks of the contraction = ceil(M / 128)
  int32_t kc, nchunks;         // blocks per chunk, chunks of THIS launch
  int32_t chunk0 = 0;          // first chunk of this launch (a product is launched in groups of a few chunks)
  int32_t nctx;                // 128-column tiles of X (row tiles of G)
  int32_t nctX, nctW;          // 64-column tiles per block in the digit arrays of X (even) and W
  int32_t ctw_begin, nctwg;    // this launch: first 64-column tile of W, groups of C tiles
  int32_t ncols_w;             // columns of W covered by P (panel width, multiple of 64 except at the end)
  int64_t ncols;               // columns of X = rows of G
  double* P; int64_t ldp;      // partial tiles: P[chunk][ncols rows][ldp], column index relative to the panel
  const uint32_t* cmaxX;       // column maxima (upper words) of X  [ncols]
  const uint32_t* cmaxW;       // column maxima of W                [ncols]
  int64_t colw0;               // first column of W of this panel (global), for cmaxW
  int32_t sym;                 // 1: W is X (G = X^T X): tile groups entirely below the diagonal are skipped, the reduction mirrors
};

__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, int32_t x, int32_t y, int32_t z, int32_t w, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(w), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void tma_load_4d_mc(void* dst, const CUtensorMap* map, int32_t x, int32_t y, int32_t z, int32_t w, uint64_t* bar,
                                               uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3, %4, %5}], [%6], %7;" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(w), "r"(smem_u32(bar)), "h"(mask)
      : "memory");
}

// first tile group of row tile ctx that is not entirely below the diagonal of G (symmetric mode; 0 otherwise): group g holds the
// 64-column tiles ctw_begin + g C ... + C - 1, and is needed iff its last column >= the row tile's first row
template <int C>
__device__ __forceinline__ int32_t k4_gmin(const K4Params& prm, int32_t ctx) {
  if (!prm.sym) return 0;
  const int64_t t = (int64_t)ctx * 128 - (K3_NT - 1) - (int64_t)K3_NT * (prm.ctw_begin + C - 1);      // need  g * 64 C >= t
  const int64_t g = t <= 0 ? 0 : (t + K3_NT * C - 1) / (K3_NT * C);
  return (int32_t)min(g, (int64_t)prm.nctwg);
}
// work items of one chunk that are computed at all (symmetric mode skips the groups below the diagonal)
template <int C>
__device__ __forceinline__ int64_t k4_valid_per_chunk(const K4Params& prm) {
  if (!prm.sym) return (int64_t)prm.nctx * prm.nctwg;
  int64_t n = 0;
  for (int32_t ctx = 0; ctx < prm.nctx; ++ctx) n += prm.nctwg - k4_gmin<C>(prm, ctx);
  return n;
}
// cluster work item u -> (chunk, row tile ctx, tile group ctwg).  Chunks outermost; inside a chunk the tiles of G are
// walked in super-tiles of 8 row tiles x 9 tile groups (72 ~ the 74 co-resident 2-CTA clusters), so that the clusters
// running at the same time walk the same blocks of the contraction on few distinct operand tiles: 8 X tile pairs +
// 18 W tiles per block instead of 2-3 X pairs + 64 W tiles, i.e. each W tile is fetched from HBM once per 8 row tiles
// instead of once per row tile.  In symmetric mode ONLY the computed items are numbered (nvalid per chunk): were the
// skipped ones numbered too, a cluster that draws one would move on to the next wave at once, the waves would mix and the
// clusters in flight would no longer share their operand tiles (143 GB of DRAM traffic per launch at config 3's shape).
template <int C>
__device__ __forceinline__ void k4_decode(const K4Params& prm, int64_t u, int64_t nvalid, int32_t& chunk, int32_t& ctx, int32_t& ctwg) {
  constexpr int SX = 8, SW = 9;
  const int32_t lc = (int32_t)(u / nvalid);                    // chunk inside this launch
  chunk = prm.chunk0 + lc;
  int32_t v = (int32_t)(u - (int64_t)lc * nvalid);
  if (!prm.sym) {
    const int32_t sx = v / (SX * prm.nctwg);
    const int32_t hx = min(SX, prm.nctx - sx * SX);            // row tiles in this super row
    const int32_t rem2 = v - sx * SX * prm.nctwg;
    const int32_t sw = rem2 / (hx * SW);
    const int32_t rem3 = rem2 - sw * hx * SW;
    ctx = sx * SX + rem3 % hx;
    ctwg = sw * SW + rem3 / hx;
    return;
  }
  for (int32_t x0 = 0; x0 < prm.nctx; x0 += SX) {
    const int32_t hx = min(SX, prm.nctx - x0);
    int32_t gm[SX];
#pragma unroll
    for (int i = 0; i < SX; ++i) gm[i] = i < hx ? k4_gmin<C>(prm, x0 + i) : prm.nctwg;
    for (int32_t g0 = 0; g0 < prm.nctwg; g0 += SW) {
      const int32_t g1 = min(g0 + SW, prm.nctwg);
      int32_t cnt = 0;
#pragma unroll
      for (int i = 0; i < SX; ++i) cnt += max(0, g1 - max(g0, gm[i]));
      if (v < cnt) {                                           // in this super-tile: same order as above, valid items only
        for (int32_t g = g0; g < g1; ++g)
#pragma unroll
          for (int i = 0; i < SX; ++i)
            if (g >= gm[i]) {
              if (v == 0) { ctx = x0 + i; ctwg = g; return; }
              --v;
            }
      }
      v -= cnt;
    }
  }
  ctx = 0; ctwg = 0;                                           // not reached for u < nchunks * nvalid
}

// a work item is skipped in symmetric mode if even its last 64-column tile lies entirely below the diagonal of G
__device__ __forceinline__ bool k4_skip(const K4Params& prm, int32_t ctx, int32_t ctw_last) {
  return prm.sym && ((int64_t)ctw_last * K3_NT + K3_NT - 1 < (int64_t)ctx * 128);
}

// P[chunk] summed in ascending chunk order:  G[j, colw0 + l] = sum_c P[c][j][l]; in symmetric mode (single panel) the
// entries below the diagonal are the mirror images of the computed ones, so G comes out exactly symmetric
__global__ void __launch_bounds__(256) gram_reduce_kernel(const double* __restrict__ P, int64_t ldp, int64_t rows, int32_t nchunks,
                                                          int64_t ncols_w, double* __restrict__ G, int64_t ldg, int32_t sym) {
  const int64_t j = blockIdx.y;
  const int64_t l = (int64_t)blockIdx.x * 256 + threadIdx.x;
  if (l >= ncols_w) return;
  const int64_t pj = (sym && l < j) ? l : j, pl = (sym && l < j) ? j : l;
  double acc = 0.0;
  for (int32_t c = 0; c < nchunks; ++c) acc += P[((int64_t)c * rows + pj) * ldp + pl];
  G[j * ldg + l] = acc;
}

// tmXd: 4-D map {128 B, 64 columns, S planes, tiles} of the X digit tiles, box {128 B, 64/C columns, 1, 1}: every CTA
//       of a cluster fetches 64/C columns of both tiles of a plane (two boxes) and multicasts them;
// tmWd: 3-D map of the W digit tiles, box S x 64 x 128 B (as K3's Y map).
template <int S, int C>
__global__ void __launch_bounds__(K4_THREADS, 1)
gram_i8_kernel(const __grid_constant__ CUtensorMap tmXd, const __grid_constant__ CUtensorMap tmWd, const K4Params prm) {
  using Cf = K3Cfg<S>;
  constexpr int NH = Cf::NH;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* ybuf = smem;                          // 2 x YBUF: W digit tiles
  uint8_t* hring = smem + 2 * Cf::YBUF;          // NH x HSLOT: X digit planes (128 columns x 128 k-bytes)
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cf::BAR_OFFSET);
  uint64_t* yfull = bars;
  uint64_t* yempty = bars + 2;
  uint64_t* hfull = bars + 4;
  uint64_t* hempty = bars + 4 + NH;
  uint64_t* accfull = bars + 4 + 2 * NH;
  uint64_t* accempty = accfull + 1;
  int32_t* ce_s = reinterpret_cast<int32_t*>(smem + Cf::CS_OFFSET);      // eW_l of the current tile
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(smem + Cf::CM_OFFSET) + 64;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t nvalid = k4_valid_per_chunk<C>(prm);          // computed items per chunk (all of them unless symmetric)
  const int64_t nitems = (int64_t)prm.nchunks * nvalid;
  const int32_t crank = (C > 1) ? (int32_t)cluster_ctarank() : 0;
  const int64_t cluster0 = blockIdx.x / C, nclusters = gridDim.x / C;
  constexpr uint16_t cmask = (uint16_t)((1u << C) - 1u);

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(&yfull[i], 1); mbar_init(&yempty[i], 1); }
    for (int i = 0; i < NH; ++i) { mbar_init(&hfull[i], 1); mbar_init(&hempty[i], C); }
    mbar_init(accfull, 1);
    mbar_init(accempty, 128);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (C > 1) cluster_sync_all();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===================================== TMA producer =====================================
    if (elect_one()) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmXd) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmWd) : "memory");
      int yb = 0, hs = 0;
      uint32_t yph = 0, hph = 0;
      constexpr int ncol = 64 / C;               // columns of each of the two X tiles this CTA fetches per plane
      for (int64_t u = cluster0; u < nitems; u += nclusters) {
        int32_t chunk, ctx, ctwg;
        k4_decode<C>(prm, u, nvalid, chunk, ctx, ctwg);
        const int32_t ctw = prm.ctw_begin + ctwg * C + crank;
        if (k4_skip(prm, ctx, prm.ctw_begin + ctwg * C + C - 1)) continue;
        const int32_t I0 = chunk * prm.kc, I1 = min(prm.nbk, I0 + prm.kc);
        for (int32_t I = I0; I < I1; ++I) {
          mbar_wait(&yempty[yb], yph ^ 1);
          mbar_expect_tx(&yfull[yb], (uint32_t)Cf::YBUF);
          tma_load_3d(ybuf + yb * Cf::YBUF, &tmWd, 0, 0, (I * prm.nctW + ctw) * S, &yfull[yb]);
          const int32_t tx = I * prm.nctX + 2 * ctx;       // first of the two adjacent X tiles
#pragma unroll 1
          for (int q = 0; q < S; ++q) {
            mbar_wait(&hempty[hs], hph ^ 1);
            mbar_expect_tx(&hfull[hs], 128u * 128u);
            uint8_t* slot = hring + hs * Cf::HSLOT;
            if (C > 1) {
              // each CTA fetches 64/C columns of both tiles of the plane and multicasts them to the cluster
              tma_load_4d_mc(slot + crank * ncol * 128, &tmXd, 0, crank * ncol, k3_plane<S>(q), tx, &hfull[hs], cmask);
              tma_load_4d_mc(slot + 8192 + crank * ncol * 128, &tmXd, 0, crank * ncol, k3_plane<S>(q), tx + 1, &hfull[hs], cmask);
            } else {
              tma_load_4d(slot, &tmXd, 0, 0, k3_plane<S>(q), tx, &hfull[hs]);
              tma_load_4d(slot + 8192, &tmXd, 0, 0, k3_plane<S>(q), tx + 1, &hfull[hs]);
            }
            if (++hs == NH) { hs = 0; hph ^= 1; }
          }
          yb ^= 1;
          if (yb == 0) yph ^= 1;
        }
      }
    }
  } else if (warp == 1) {
    // ====================================== MMA issuer ======================================
    if (elect_one()) {
      int yb = 0, hs = 0;
      uint32_t yph = 0, hph = 0, aph = 0;
      const uint64_t dbase = umma_desc_sw128(0);
      const uint32_t ylo0 = (smem_u32(ybuf) & 0x3ffffu) >> 4, hlo0 = (smem_u32(hring) & 0x3ffffu) >> 4;
      for (int64_t u = cluster0; u < nitems; u += nclusters) {
        int32_t chunk, ctx, ctwg;
        k4_decode<C>(prm, u, nvalid, chunk, ctx, ctwg);
        if (k4_skip(prm, ctx, prm.ctw_begin + ctwg * C + C - 1)) continue;
        const int32_t nI = min(prm.nbk, chunk * prm.kc + prm.kc) - chunk * prm.kc;
        mbar_wait(accempty, aph ^ 1);
        asm volatile("tcgen05.fence::after_thread_sync;");
        for (int32_t j = 0; j < nI; ++j) {
          mbar_wait(&yfull[yb], yph);
          const uint32_t ylo = ylo0 + (uint32_t)yb * (Cf::YBUF >> 4);
#pragma unroll
          for (int ip = 0; ip < S; ++ip) {
            const int p = k3_plane<S>(ip);       // wide and narrow products alternate (bsr_i8.cuh)
            mbar_wait(&hfull[hs], hph);
            asm volatile("tcgen05.fence::after_thread_sync;");
            const uint32_t hlo = hlo0 + (uint32_t)hs * (Cf::HSLOT >> 4);
            const int ntot = (S - p) * K3_NT;
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              const uint64_t da = dbase | (uint64_t)(hlo + kk * 2);
              const uint32_t acc = (ip > 0 || kk > 0) ? 1u : (j > 0 ? 1u : 0u);
              if (ntot > 256) {                  // two instructions, A read once (collector fill + lastuse, bsr_i8.cuh)
                umma_i8<1>(tmem_base + (uint32_t)(p * K3_NT), da, dbase | (uint64_t)(ylo + kk * 2), umma_idesc_i8(256), acc);
                umma_i8<2>(tmem_base + (uint32_t)(p * K3_NT + 256), da, dbase | (uint64_t)(ylo + 256 * 8 + kk * 2),
                           umma_idesc_i8(ntot - 256), acc);
              } else {
                umma_i8(tmem_base + (uint32_t)(p * K3_NT), da, dbase | (uint64_t)(ylo + kk * 2), umma_idesc_i8(ntot), acc);
              }
            }
            if (C > 1) umma_commit_mc(&hempty[hs], cmask);
            else umma_commit(&hempty[hs]);
            if (++hs == NH) { hs = 0; hph ^= 1; }
          }
          umma_commit(&yempty[yb]);
          yb ^= 1;
          if (yb == 0) yph ^= 1;
        }
        umma_commit(accfull);
        aph ^= 1;
      }
    }
  } else {
    // ======================================= epilogue =======================================
    const int quarter = warp & 3;
    const int et = (warp - 2) * 32 + lane;
    const int r = quarter * 32 + lane;           // column of X inside the row tile = row of G
    uint32_t aph = 0;
    for (int64_t u = cluster0; u < nitems; u += nclusters) {
      int32_t chunk, ctx, ctwg;
      k4_decode<C>(prm, u, nvalid, chunk, ctx, ctwg);
      const int32_t ctw = prm.ctw_begin + ctwg * C + crank;
      if (k4_skip(prm, ctx, prm.ctw_begin + ctwg * C + C - 1)) continue;
      const int64_t lcol0 = (int64_t)ctw * K3_NT;            // column inside the panel
      const int64_t grow = (int64_t)ctx * 128 + r;           // row of G
      const bool row_ok = grow < prm.ncols;
      if (et < 64) {
        const int64_t cl = prm.colw0 + lcol0 + et;
        ce_s[et] = exp_from_hi((lcol0 + et < prm.ncols_w) ? prm.cmaxW[cl] : 0u);
      }
      const int32_t ex = row_ok ? exp_from_hi(prm.cmaxX[grow]) - 30 : 0;   // 2^(eX_j - 14) / 2^16 (k3_drain returns 2^16 * v)
      asm volatile("bar.sync 1, 128;" ::: "memory");

      double v[K3_NT];
      mbar_wait(accfull, aph);
      aph ^= 1;
      asm volatile("tcgen05.fence::after_thread_sync;");
      const uint32_t trow = tmem_base + ((uint32_t)(quarter * 32) << 16);
      k3_drain<S, K3_NT>(trow, v);
      asm volatile("tcgen05.fence::before_thread_sync;");
      mbar_arrive(accempty);

      if (row_ok) {
        double* pp = prm.P + ((int64_t)chunk * prm.ncols + grow) * prm.ldp + lcol0;
        if (lcol0 + K3_NT <= prm.ncols_w) {
#pragma unroll
          for (int j = 0; j < K3_NT; j += 2)
            *reinterpret_cast<double2*>(pp + j) = make_double2(scale_pow2(v[j], ex + ce_s[j]), scale_pow2(v[j + 1], ex + ce_s[j + 1]));
        } else {
#pragma unroll
          for (int j = 0; j < K3_NT; ++j)
            if (lcol0 + j < prm.ncols_w) pp[j] = scale_pow2(v[j], ex + ce_s[j]);
        }
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");   // cs_s is rewritten by the next item
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (C > 1) cluster_sync_all();
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512));
}

}  // namespace ttdft
