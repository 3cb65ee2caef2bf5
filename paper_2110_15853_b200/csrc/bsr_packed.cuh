// bsr_packed.cuh -- packed tile storage for the HBM-bound regime (N <= 16 columns: BASELINE.json config 5's N = 16 point, the
// one-column products of the Lanczos bounds) and kernel K1P that multiplies from it.
//
// SURVEY.md 7 "Small-N regime", 8(f)-4 "storage variants"; PAPER.md:L250-252 (the tiles of a localized Hamiltonian carry many
// zeros off the diagonal: 30-40 % in BASELINE.json's configs).  For N <= ~20 columns a step is bound by streaming H once, so the
// explicit zeros of dense b x b tiles (5.15 GB at config 3 for 3.18 GB of non-zeros) are what limits it.  Packed format: every
// tile is cut into SLABS of 16 k-columns (the k-slab of kernel K1's pipeline); a slab stores, for its b rows,
//     uint16 rowoff[b]   index of the row's first value inside the slab
//     uint16 mask[b]     bit j set  <=>  H[r, k0 + j] != 0
//     double values[]    the non-zeros in row-major order (count padded to even: 16-byte granules)
// and slab_ptr[] holds the slab offsets in 16-byte units.  3.34 GB at config 3 (0.65x of the dense tiles).
//
// Kernel K1P = kernel K1 (bsr_dmma.cuh) for one 16-column tile with the A operand coming from the packed slabs: the producer
// lane brings a packed slab into a staging ring with ONE bulk copy (cp.async.bulk, 1-D) and the X rows by TMA as before; WR
// decoder warps (one thread per tile row) expand the slab into the stage's A buffer in exactly the layout TMA's SWIZZLE_128B
// would have produced (16-byte chunk c of row r at position c ^ (r & 7)), zeros included; the consumer warps and the fused
// epilogue are K1's own code (k1_consume).  The fp64 tensor pipe still multiplies the zeros -- with 16 columns its floor
// (0.55 ms at config 3) sits just above the HBM time of the packed bytes (0.50 ms), below that of the dense ones (0.79 ms).
#pragma once
#include "bsr_dmma.cuh"

namespace ttdft {

constexpr int PK_NSS = 4;        // staging slots for packed slabs
constexpr int PK_DT = 4;         // decoder threads per tile row (each expands 4 of a slab's 16 k-columns)

__host__ __device__ __forceinline__ uint32_t pk_slab_units(int32_t b, uint32_t nnz) {   // 16-byte units of one packed slab
  return (uint32_t)((4 * b + 8 * ((nnz + 1u) & ~1u)) >> 4);
}

// One warp per slab (tile p, k-slab s).  FILL == false: units[slab + 1] = size of the packed slab in 16-byte units (units[0] = 0;
// an exclusive scan turns the array into slab_ptr).  FILL == true: writes header and values at slab_ptr[slab].
// tiles: dense b x b row-major fp64 tiles.  grid ceil(nslabs / 8), 256 threads.
template <bool FILL>
__global__ void __launch_bounds__(256) pk_slabs_kernel(int32_t b, int64_t nslabs, const double* __restrict__ tiles, uint32_t* __restrict__ units,
                                                       const uint32_t* __restrict__ slab_ptr, uint8_t* __restrict__ pdata) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t slab = (int64_t)blockIdx.x * 8 + warp;
  if (slab >= nslabs) return;
  const int32_t nslab = b >> 4;
  const int64_t p = slab / nslab;
  const int32_t k0 = (int32_t)(slab - p * nslab) << 4;
  uint8_t* dst = FILL ? pdata + (size_t)slab_ptr[slab] * 16 : nullptr;
  uint16_t* rowoff = reinterpret_cast<uint16_t*>(dst);
  uint16_t* maskp = rowoff + b;
  double* vals = reinterpret_cast<double*>(dst + 4 * b);
  uint32_t base = 0;                             // values before this group of 32 rows
  for (int32_t r0 = 0; r0 < b; r0 += 32) {
    const int32_t r = r0 + lane;                 // b is a multiple of 32
    const double* src = tiles + ((size_t)p * b + r) * b + k0;
    double v[16];
    uint32_t m = 0;
#pragma unroll
    for (int j = 0; j < 16; j += 2) {
      const double2 t = *reinterpret_cast<const double2*>(src + j);
      v[j] = t.x; v[j + 1] = t.y;
      m |= (t.x != 0.0 ? 1u : 0u) << j;
      m |= (t.y != 0.0 ? 1u : 0u) << (j + 1);
    }
    const uint32_t cnt = __popc(m);
    uint32_t incl = cnt;                         // inclusive scan over the 32 rows of the group
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    const uint32_t off = base + incl - cnt;
    if (FILL) {
      rowoff[r] = (uint16_t)off;
      maskp[r] = (uint16_t)m;
      uint32_t o = off;
#pragma unroll
      for (int j = 0; j < 16; ++j)
        if (m & (1u << j)) vals[o++] = v[j];
    }
    base += __shfl_sync(0xffffffffu, incl, 31);
  }
  if (!FILL) {
    if (lane == 0) units[slab + 1] = pk_slab_units(b, base);
    if (slab == 0 && lane == 0) units[0] = 0;
  } else if ((base & 1u) && lane == 0) {
    vals[base] = 0.0;                            // the padding value of an odd count
  }
}

// in-place INCLUSIVE scan of a[0..n) (uint32, total < 2^32) by ONE CTA of 1024 threads.  With a[0] = 0 and a[i + 1] = size of
// slab i on entry, a[i] is the offset of slab i on exit and a[n - 1] the total.
__global__ void __launch_bounds__(1024) pk_scan_kernel(uint32_t* __restrict__ a, int64_t n) {
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t carry_s;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  for (int64_t i0 = 0; i0 < n; i0 += 1024) {
    const int64_t i = i0 + threadIdx.x;
    const uint32_t x = i < n ? a[i] : 0u;
    uint32_t incl = x;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    if (warp == 0) {
      uint32_t w = wsum[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t t = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += t;
      }
      wsum[lane] = w;                            // inclusive over the warps
    }
    __syncthreads();
    const uint32_t before = carry_s + (warp ? wsum[warp - 1] : 0u);
    if (i < n) a[i] = before + incl;             // inclusive: sizes were stored shifted by one, so this IS the exclusive offset
    __syncthreads();
    if (threadIdx.x == 1023) carry_s = before + incl;
    __syncthreads();
  }
}

template <int WR>
struct K1PCfg {
  using SM = K1Cfg<WR, 1, 1, 1>;
  static constexpr int BR = SM::BR;
  static constexpr int SLOT = 4 * BR + BR * 128 + 64;            // header + a fully dense slab + slack for the decoders' look-ahead
  static constexpr int NST = SM::NSTAGE > 6 ? 6 : SM::NSTAGE;    // stages of the main ring (the staging ring needs room too)
  static constexpr int NDW = BR * PK_DT / 32;                    // decoder warps
  static constexpr int STAGING_OFFSET = (NST * SM::STAGE_BYTES + 1023) & ~1023;
  static constexpr int PTR_OFFSET = STAGING_OFFSET + PK_NSS * SLOT;      // slab_ptr entries of the CTA's block row (<= 2048)
  static constexpr int MAXPTR = 2048;
  static constexpr int BAR_OFFSET = PTR_OFFSET + MAXPTR * 4;
  static constexpr int TOTAL = BAR_OFFSET + (2 * NST + 2 * PK_NSS) * 8 + 1024;
  static constexpr int THREADS = 32 * (SM::NCW + 1 + NDW);
  static_assert(TOTAL <= 232448, "shared memory");
};

__device__ __forceinline__ void bulk_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
               "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// One CTA per block row I (one 16-column tile: ncols <= 16).  Warps: 2 WR consumers | producer | 4 WR decoders.
template <int WR>
__global__ void __launch_bounds__(K1PCfg<WR>::THREADS, 1)
bsr_dmma_packed_kernel(const __grid_constant__ CUtensorMap tmX, const K1Params prm, const uint32_t* __restrict__ slab_ptr,
                       const uint8_t* __restrict__ pdata) {
  using Cf = K1PCfg<WR>;
  using SM = typename Cf::SM;
  constexpr int NCW = SM::NCW;
  constexpr int NST = Cf::NST;
  constexpr int NDW = Cf::NDW;
  constexpr int BR = SM::BR;
  constexpr int NSLAB = BR / K1_KS;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* staging = smem + Cf::STAGING_OFFSET;
  uint32_t* ptr_s = reinterpret_cast<uint32_t*>(smem + Cf::PTR_OFFSET);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + Cf::BAR_OFFSET);
  uint64_t* empty = full + NST;
  uint64_t* sfull = empty + NST;
  uint64_t* sempty = sfull + PK_NSS;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int32_t I = blockIdx.x;
  const int32_t p_begin = prm.brow_ptr[I], p_end = prm.brow_ptr[I + 1];
  if (prm.skip_empty && p_begin == p_end) return;      // CTA-uniform, before any barrier
  const int32_t nsl = (p_end - p_begin) * NSLAB;       // slabs of this block row (<= MAXPTR - 1, checked on the host)
  for (int i = threadIdx.x; i <= nsl; i += blockDim.x) ptr_s[i] = slab_ptr[(int64_t)p_begin * NSLAB + i];
  if (threadIdx.x == 0) {
    for (int s = 0; s < NST; ++s) {
      mbar_init(&full[s], 1 + NDW);              // the X rows (TMA) + one arrival per decoder warp
      mbar_init(&empty[s], NCW);
    }
    for (int s = 0; s < PK_NSS; ++s) {
      mbar_init(&sfull[s], 1);
      mbar_init(&sempty[s], NDW);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  __syncthreads();

  if (warp == NCW) {
    // ============ producer (one lane): packed slab -> staging ring (bulk copy), X rows -> stage (TMA) ============
    if (lane == 0) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmX) : "memory");
      int stage = 0, ss = 0;
      uint32_t phase = 0, sphase = 0;
      int32_t it = 0;
      for (int32_t p = p_begin; p < p_end; ++p) {
        const int32_t J = prm.bcol[p];
#pragma unroll 1
        for (int k0 = 0; k0 < BR; k0 += K1_KS, ++it) {
          mbar_wait(&sempty[ss], sphase ^ 1);
          const uint32_t bytes = (ptr_s[it + 1] - ptr_s[it]) * 16u;
          mbar_expect_tx(&sfull[ss], bytes);
          bulk_load_1d(staging + ss * Cf::SLOT, pdata + (size_t)ptr_s[it] * 16, bytes, &sfull[ss]);
          if (++ss == PK_NSS) { ss = 0; sphase ^= 1; }
          mbar_wait(&empty[stage], phase ^ 1);
          uint8_t* Bs = smem + stage * SM::STAGE_BYTES + SM::A_BYTES;
          mbar_expect_tx(&full[stage], (uint32_t)K1_BGRP_BYTES);
          tma_load_2d(Bs, &tmX, 0, J * BR + k0, &full[stage]);
          if (++stage == NST) { stage = 0; phase ^= 1; }
        }
      }
    }
    return;
  }
  if (warp > NCW) {
    // ============ decoders: PK_DT threads per tile row, thread (r, h) expands k-columns 4h..4h+3 of the slab into the stage's A
    // buffer (TMA's SWIZZLE_128B layout).  The four value loads are independent (offsets from popcounts), so a slab costs a
    // thread one round of shared-memory latency, and 4 WR warps keep several slabs in flight.
    const int d = (warp - NCW - 1) * 32 + lane;
    const int r = d >> 2, h = d & 3;             // 0 .. BR-1, 0 .. 3
    int stage = 0, ss = 0;
    uint32_t phase = 0, sphase = 0;
#pragma unroll 1
    for (int32_t it = 0; it < nsl; ++it) {
      mbar_wait(&sfull[ss], sphase);
      const uint8_t* slot = staging + ss * Cf::SLOT;
      const uint32_t m = reinterpret_cast<const uint16_t*>(slot)[BR + r];
      const uint32_t o0 = reinterpret_cast<const uint16_t*>(slot)[r] + __popc(m & ((1u << (4 * h)) - 1u));
      const uint32_t mb = (m >> (4 * h)) & 15u;
      const uint32_t o1 = o0 + (mb & 1u), o2 = o1 + ((mb >> 1) & 1u), o3 = o2 + ((mb >> 2) & 1u);
      const double* vals = reinterpret_cast<const double*>(slot + 4 * BR);
      const double x0 = vals[o0], x1 = vals[o1], x2 = vals[o2], x3 = vals[o3];   // past-the-end reads stay inside the slot
      double2 lo, hi;
      lo.x = (mb & 1u) ? x0 : 0.0;
      lo.y = (mb & 2u) ? x1 : 0.0;
      hi.x = (mb & 4u) ? x2 : 0.0;
      hi.y = (mb & 8u) ? x3 : 0.0;
      mbar_wait(&empty[stage], phase ^ 1);       // the consumers have released this stage
      uint8_t* arow = smem + stage * SM::STAGE_BYTES + r * 128;
      *reinterpret_cast<double2*>(arow + (((2 * h) ^ (r & 7)) << 4)) = lo;
      *reinterpret_cast<double2*>(arow + (((2 * h + 1) ^ (r & 7)) << 4)) = hi;
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&full[stage]);
        mbar_arrive(&sempty[ss]);
      }
      if (++stage == NST) { stage = 0; phase ^= 1; }
      if (++ss == PK_NSS) { ss = 0; sphase ^= 1; }
    }
    return;
  }
  k1_consume<WR, 1, 1, 1, Cf::NST>(prm, smem, full, empty, I, 0, 0, p_begin, p_end);
}

}  // namespace ttdft
