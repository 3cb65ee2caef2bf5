// bsr_i8.cuh -- kernel K3: the filter step  O = alpha*(H*Y_k) + gamma*Y_k + beta*Y_{k-1}
// (the product is "the main kernel", L236) with the block-dense contraction
// carried by the 5th-generation tensor cores as exact int8 digit-plane products (i8_digits.cuh).
//
// sm_100a design:
//   * persistent CTAs (one per SM) in clusters of C along the columns: the C CTAs of a cluster work on the
//     same block row I and C adjacent 64-column tiles, static round-robin over (I, tile group) work items
//   * warp 0 (one lane): TMA producer.  Per tile (I,J) of the block row it brings the S digit planes of
//     Y_k rows J*b.., 64 columns, with ONE 3-D bulk-tensor load (S x 64 x 128 B, SWIZZLE_128B; the planes of
//     a tile are contiguous in HBM) into one of two Y buffers, and the S digit planes of H_IJ (b x 128 B
//     each) through a ring of 16 KB slots.  Every CTA of the cluster fetches b/C rows of each H plane and
//     MULTICASTS them into the same slot of all C CTAs, so a plane leaves L2 once per cluster: the kernel
//     was bound by L2->SM throughput before (profiles/r01a_*), H being 2/3 of those bytes.  H planes carry an
//     L2 evict-first hint (streamed), Y tiles evict-last (re-used by up to 27 block rows)
//   * warp 1 (one lane): tcgen05.mma.kind::i8 issuer.  For H plane p it multiplies against the
//     CONCATENATION of Y planes 0..S-1-p (N = 64*(S-p), issued as <=256-column instructions), which lands
//     in the contiguous TMEM column groups p..S-1 because digit-pair level g = p+q lives at columns
//     [64g, 64g+64): 10 wide MMAs per k-step instead of S(S+1)/2 = 28 narrow ones
//   * accumulators: S levels x 64 columns of int32 in TMEM (448 of 512 columns for S = 7), exact
//   * warps 2-9: epilogue, two warps per TMEM lane quarter (32 columns each).  Drain: three int32 levels are packed
//     exactly into one int64 before the conversion to fp64; TMEM released.  Output: the warp's 32 x 32 block is
//     transposed in registers so that every access is one contiguous 256-byte row segment, then
//     out = scale_pow2(alpha*2^(eH_i-30)*v, eY_j) + (alpha*hdiag_i+gamma)*y + beta*z, and the column maxima of `out`
//     for the next step's digit scaling (per lane, then shared/global atomicMax on the upper word)
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "bsr_dmma.cuh"   // smem_u32, mbarrier and TMA wrappers
#include "i8_digits.cuh"

namespace ttdft {

constexpr int K3_NT = 64;        // columns per work item
constexpr int K3_THREADS = 320;  // producer warp, MMA warp, 8 epilogue warps (two per TMEM lane quarter, 32 columns each)
constexpr int K4_THREADS = 192;  // gram_i8.cuh: producer warp, MMA warp, 4 epilogue warps

struct K3Params {
  const int32_t* brow_ptr;
  const int32_t* bcol;
  int32_t nb, b, vec;
  int32_t nct;                     // 64-column tiles of the whole panel (index space of the Y digit tiles)
  int32_t ct_begin, nctg, cgc;     // this launch: first column tile, tile groups (of C tiles), groups per scheduling group
  int32_t hplanes;                 // digit planes STORED per tile of H (>= S; the kernel uses the leading S)
  int64_t ncols;
  double alpha, gamma, beta;
  const double* S;  int64_t lds;   // Y_k at the output position (diagonal + shift term); NULL: no such term
  const double* Z;  int64_t ldz;   // Y_{k-1}; unused if beta == 0
  double* O;        int64_t ldo;
  const int32_t* eH;               // row exponents of H          [M]
  const double* hdiag;             // diagonal of H (fp64)         [M]; NULL: zero
  const int32_t* eS;               // exponents the digits of Y_k were taken with   [ncols]
  uint32_t* cmaxO;                 // out: column maxima of O (upper words), or NULL
  // digits of O for the next step, written by the epilogue (NULL: not wanted).  dO: digit tiles in the layout of i8_digits.cuh,
  // taken with the PREDICTED exponents ePredO[j]; a column whose maximum outgrows its prediction sets flagsO[its 64-column tile]
  // (the tile is then redone by y_digits_fix_kernel).  Requires cmaxO and mrows == nb * b.
  int8_t* dO = nullptr;
  const int32_t* ePredO = nullptr;
  uint32_t* flagsO = nullptr;
  uint32_t* counter = nullptr;     // work counter of this launch (one word, ZERO at launch): clusters draw their work items from it
  int32_t skip_empty = 0;          // 1: block rows without tiles are not this handle's: their output rows are left untouched
  int64_t mrows;                   // valid rows (= nb*b for a Hamiltonian; < nb*b for the ragged last block of ttdft_rotate)
  int32_t l2hints;                 // 1: evict-first H planes, evict-last Y digit tiles; 2: only the latter; 0: none (< 0 on the host: chosen per launch)
  int32_t jlimit = 0;              // > 0: only the first jlimit tiles of every block row are multiplied; < 0: the right factor is
                                   // upper triangular (the R^-1 of ttdft_orthonormalize's rotation; tiles = 128 rows of it in order):
                                   // a cluster whose last column tile is ct multiplies the first ceil((ct + 1) / 2) tiles only
#ifdef TTDFT_EXPERIMENT
  int32_t exp = 0;                 // experiment builds only (-DTTDFT_EXPERIMENT, env TTDFT_K3_EXP): 2 no TMA after priming,
                                   // 4 epilogue without global traffic, 8 epilogue without drain
#endif
#ifdef TTDFT_DEBUG_TRACE
  unsigned long long* trace = nullptr;   // debug builds only (-DTTDFT_DEBUG_TRACE): 8 clock64 stamps per work item of CTA 0, or NULL
#endif
};

#ifdef TTDFT_EXPERIMENT
#define K3_EXP(bit) ((prm.exp & (bit)) != 0)
#else
#define K3_EXP(bit) false
#endif
// clock trace of CTA 0 (debug builds only: the shipped kernel carries no trace stores)
#ifdef TTDFT_DEBUG_TRACE
#define K3_TRACE_DECL(cond) const bool tr_ = prm.trace && blockIdx.x == 0 && (cond)
#define K3_TRACE(slot, val) do { if (tr_) prm.trace[it * 8 + (slot)] = (val); } while (0)
#else
#define K3_TRACE_DECL(cond) (void)it
#define K3_TRACE(slot, val) do { } while (0)
#endif

template <int S>
struct K3Cfg {
  static constexpr int YBUF = S * K3_NT * 128;            // one Y buffer: S planes x 64 columns x 128 k-bytes
  static constexpr int HSLOT = 128 * 128;                 // one H plane of one tile
  static constexpr int NH = (232448 - 2048 - 2 * YBUF) / HSLOT;   // ring slots that fit beside two Y buffers
  static constexpr int BAR_OFFSET = 2 * YBUF + NH * HSLOT;
  static constexpr int NBAR = 4 + 2 * NH + 2;
  static constexpr int CS_OFFSET = BAR_OFFSET + 8 * ((NBAR + 1) & ~1);   // 64 doubles: column scales
  static constexpr int CM_OFFSET = CS_OFFSET + 64 * 8;                   // 64 words: column maxima
  static constexpr int CP_OFFSET = CM_OFFSET + 64 * 4 + 16;              // 64 words: predicted exponents of the output columns (behind the tmem slot)
  static constexpr int Q_OFFSET = CP_OFFSET + 64 * 4;                    // work-item queue (K3Queue, 8-byte aligned)
  static constexpr int TOTAL = Q_OFFSET + 192 + 1024;                    // + alignment slack
  static_assert(S * K3_NT <= 512, "digit levels must fit TMEM");
  static_assert(NH >= 3, "H ring too short");
};

__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int32_t x, int32_t y, int32_t z, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar))
      : "memory");
}
// L2 eviction-priority hints for TMA loads (the fixed policy encodings CUTLASS passes as cache hints)
constexpr uint64_t L2_EVICT_FIRST = 0x12F0000000000000ull;   // streamed once: the H digit planes
constexpr uint64_t L2_EVICT_LAST = 0x14F0000000000000ull;    // reused by up to 27 block rows: the Y digit tiles
__device__ __forceinline__ void tma_load_3d_hint(void* dst, const CUtensorMap* map, int32_t x, int32_t y, int32_t z, uint64_t* bar,
                                                 uint64_t hint) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(z), "r"(smem_u32(bar)), "l"(hint)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d_hint(void* dst, const CUtensorMap* map, int32_t x, int32_t y, uint64_t* bar, uint64_t hint) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)), "l"(hint)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d_mc_hint(void* dst, const CUtensorMap* map, int32_t x, int32_t y, uint64_t* bar, uint16_t mask,
                                                    uint64_t hint) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5, %6;" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)), "h"(mask), "l"(hint)
      : "memory");
}

// shared-memory matrix descriptor: K-major rows of 128 bytes, SWIZZLE_128B, 8-row groups 1024 B apart
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3ffffu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)2 << 61);
}
// instruction descriptor, kind::i8: D = s32, A = B = signed int8, both K-major, M = 128
__device__ __forceinline__ uint32_t umma_idesc_i8(uint32_t n) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((128u >> 4) << 24);
}
// COLL: what the tensor pipe's A collector does with this instruction's A operand -- 0: read from shared memory and dropped (the
// default), 1 (collector::a::fill): read and KEPT, 2 (collector::a::lastuse): TAKEN from the collector (same descriptor as the
// fill just before it) and dropped.  A product wider than one instruction (N > 256) goes as a fill + lastuse pair, so its 4 KB of A
// are read once: the MMA loop is bound by operand reads (~101 B per clock and SM sustained, measured on both K3 and K3T), and A
// re-reads were 12 % of them.
template <int COLL = 0>
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  if constexpr (COLL == 1)
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::i8.collector::a::fill [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
  else if constexpr (COLL == 2)
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::i8.collector::a::lastuse [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
  else
    asm volatile(
        "{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\n"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr));
}

__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t (&r)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7])
               : "r"(taddr));
}

// Accumulators of one TMEM lane (row) -> v[j] = 2^16 * sum_g L_g[j] * 256^-g  for NC consecutive columns of the item.
// fp64 instructions are scarce while the tensor pipe runs int8 MMAs (ncu: "math pipe throttle" on every DFMA of
// the epilogue), so three int32 levels are packed EXACTLY into one int64 (|L| < 2^31: L_a*2^16 + L_b*2^8 + L_c
// < 2^48) before the conversion: ceil(S/3) conversions and ceil(S/3)-1 FMAs per element instead of S and S-1.
// LS: TMEM columns between two levels (the width of a work item's accumulator block).
template <int S, int NC, int LS = K3_NT>
__device__ __forceinline__ void k3_drain(uint32_t trow, double (&v)[NC]) {   // trow: TMEM address of the first column
  constexpr int NG = (S + 2) / 3;
#pragma unroll
  for (int c = 0; c < NC / 8; ++c) {
    uint32_t a[S][8];
#pragma unroll
    for (int g = 0; g < S; ++g) tmem_ld8(trow + (uint32_t)(g * LS + c * 8), a[g]);
    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      double acc = 0.0;
#pragma unroll
      for (int k = NG - 1; k >= 0; --k) {       // least significant group first
        long long t = 0;
#pragma unroll
        for (int l = 0; l < 3; ++l) {
          const int g = 3 * k + l;
          if (g < S) {
            asm volatile("" : "+r"(a[g][i]));   // consumers must stay behind the wait
            t += (long long)(int32_t)a[g][i] << (8 * (2 - l));
          }
        }
        const double d = __ll2double_rn(t);
        acc = (k == NG - 1) ? d : fma(acc, 5.9604644775390625e-8 /* 2^-24 */, d);
      }
      v[c * 8 + i] = acc;
    }
  }
}

// x * 2^e by an integer add on the exponent field (no fp64 instruction); zero, subnormal and out-of-range
// cases take the slow, exact route
__device__ __forceinline__ double scale_pow2(double x, int32_t e) {
  const int32_t hi = __double2hiint(x);
  const int32_t ex = (hi >> 20) & 0x7ff;
  const int32_t en = ex + e;
  if (ex != 0 && en > 0 && en < 2047) return __hiloint2double(hi + (e << 20), __double2loint(x));
  if (x == 0.0) return x;
  const int32_t e1 = max(-1000, min(1000, e / 2)), e2 = max(-1000, min(1000, e - e / 2));
  return x * pow2i(e1) * pow2i(e2);
}

// Order in which the S planes of a tile travel through the ring and are multiplied: i-th plane = k3_plane<S>(i).
// Natural order.  (Alternating wide and narrow products -- 0, S-1, 1, S-2, ... -- was measured and changes nothing:
// the MMA phase is bound by shared-memory operand bandwidth, ~96 B/clk for A + B, not by the issuing thread.
// Plane 0 must stay first: its first MMA of a work item overwrites every accumulator level.)
template <int S>
__host__ __device__ constexpr int k3_plane(int i) { return i; }

// one lane of the (converged) calling warp; lets ptxas feed the uniform-register operands of
// UTMALDG / UTCIMMA from that lane directly instead of through a broadcast loop
__device__ __forceinline__ bool elect_one() {
  uint32_t pred;
  asm volatile("{\n.reg .pred P;\nelect.sync _|P, 0xffffffff;\nselp.u32 %0, 1, 0, P;\n}\n" : "=r"(pred));
  return pred != 0;
}

__device__ __forceinline__ void tma_load_2d_mc(void* dst, const CUtensorMap* map, int32_t x, int32_t y, uint64_t* bar, uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3}], [%4], %5;" ::"r"(
          smem_u32(dst)),
      "l"(map), "r"(x), "r"(y), "r"(smem_u32(bar)), "h"(mask)
      : "memory");
}
// arrive on the barrier at this offset in every CTA of the mask once the MMAs issued so far have completed
__device__ __forceinline__ void umma_commit_mc(uint64_t* bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(smem_u32(bar)),
               "h"(mask)
               : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// ------------------------------------------------------------------------------------------------
// Dynamic work distribution.  Work items are drawn from ONE global counter, so the clusters that run at the same time always work
// on a contiguous window of items -- with a static round-robin the clusters drift apart by the differences in item length (8..27
// tiles per block row) until the active block rows are spread over hundreds of rows, and the Y digit tiles that neighbouring block
// rows share leave L2 between their uses (ncu, config 4: 204 GB of DRAM traffic per launch, 76 % of the HBM peak).
// The producer lane of the cluster's CTA 0 draws the items (a few ahead) and hands each one to every role of every CTA of the
// cluster through a small queue in shared memory: item word + `qfull` mbarrier in each CTA (written remotely for the peers),
// `qempty` in CTA 0 (every consumer arrives there as soon as it has read the item).
// ------------------------------------------------------------------------------------------------
constexpr int K3_NQ = 8;                         // queue slots
constexpr int K3_QAHEAD = 4;                     // items drawn ahead of the producer's own position
constexpr int K3_QCONS = 10;                     // consumers per CTA: producer lane, MMA lane, 8 epilogue warps
constexpr uint32_t K3_NOITEM = 0xffffffffu;
struct K3Queue {
  uint64_t qfull[K3_NQ];
  uint64_t qempty[K3_NQ];
  uint32_t item[K3_NQ];
};
__device__ __forceinline__ uint32_t mapa_u32(uint32_t laddr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(laddr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_wait_cluster(uint64_t* bar, uint32_t parity) {      // acquires writes of the whole cluster
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAITC_%=:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONEC_%=;\n"
      "bra WAITC_%=;\n"
      "DONEC_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// the fetcher (CTA 0 of the cluster): item -> slot of every CTA
template <int C>
__device__ __forceinline__ void k3_q_push(K3Queue* q, int slot, uint32_t u) {
#pragma unroll
  for (int r = 0; r < C; ++r) {
    const uint32_t ia = mapa_u32(smem_u32(&q->item[slot]), (uint32_t)r), ba = mapa_u32(smem_u32(&q->qfull[slot]), (uint32_t)r);
    asm volatile("st.shared::cluster.u32 [%0], %1;" ::"r"(ia), "r"(u) : "memory");
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(ba) : "memory");
  }
}
// a consumer: next item of this CTA's queue; `arrive`: this thread reports the slot as read (one thread per consumer)
__device__ __forceinline__ uint32_t k3_q_pop(K3Queue* q, int& slot, uint32_t& phase, bool arrive) {
  mbar_wait_cluster(&q->qfull[slot], phase);
  const uint32_t u = q->item[slot];
  if (arrive) {
    const uint32_t ea = mapa_u32(smem_u32(&q->qempty[slot]), 0u);
    asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(ea) : "memory");
  }
  if (++slot == K3_NQ) { slot = 0; phase ^= 1; }
  return u;
}
// the same for a whole (converged) warp: lane 0 waits, reads and reports, the others take the item from it
__device__ __forceinline__ uint32_t k3_q_pop_warp(K3Queue* q, int& slot, uint32_t& phase) {
  uint32_t u = 0;
  if ((threadIdx.x & 31) == 0) {
    int s = slot;
    uint32_t ph = phase;
    u = k3_q_pop(q, s, ph, true);
  }
  u = __shfl_sync(0xffffffffu, u, 0);
  if (++slot == K3_NQ) { slot = 0; phase ^= 1; }
  return u;
}
// state of the fetcher
struct K3Fetch {
  int slot = 0;
  uint32_t phase = 0;
  bool done = false;
};
template <int C>
__device__ __forceinline__ void k3_q_fetch(K3Queue* q, K3Fetch& f, uint32_t* counter, uint32_t nitems) {
  if (f.done) return;
  mbar_wait_cluster(&q->qempty[f.slot], f.phase ^ 1);       // every consumer of every CTA has read the slot's previous item
  uint32_t u = atomicAdd(counter, 1u);
  if (u >= nitems) { u = K3_NOITEM; f.done = true; }        // one end marker, then nothing more is drawn
  k3_q_push<C>(q, f.slot, u);
  if (++f.slot == K3_NQ) { f.slot = 0; f.phase ^= 1; }
}

// cluster work item u -> (block row I, tile group ctg): scheduling groups of cgc tile groups outermost, then
// block rows, tile group fastest (clusters that run at the same time share H planes and Y rows in L2)
__device__ __forceinline__ void k3_decode(const K3Params& prm, int64_t u, int32_t& I, int32_t& ctg) {
  const int64_t per_group = (int64_t)prm.nb * prm.cgc;
  const int32_t ngroups = (prm.nctg + prm.cgc - 1) / prm.cgc;
  int32_t g = (int32_t)(u / per_group);
  if (g > ngroups - 1) g = ngroups - 1;
  const int64_t rem = u - (int64_t)g * per_group;
  const int32_t width = min(prm.cgc, prm.nctg - g * prm.cgc);
  I = (int32_t)(rem / width);
  ctg = g * prm.cgc + (int32_t)(rem % width);
}

// tiles of a block row that the cluster of tile group ctg multiplies (K3Params::jlimit)
template <int C>
__device__ __forceinline__ int32_t k3_jlimit(const K3Params& prm, int32_t ctg) {
  if (prm.jlimit == 0) return 0x7fffffff;
  if (prm.jlimit > 0) return prm.jlimit;
  return (prm.ct_begin + ctg * C + C + 1) / 2;      // ceil((ct_last + 1) / 2), ct_last = ct_begin + ctg * C + C - 1
}

// tmHd: box (b/C rows) x 128 B of the H digit planes; tmYd: box S x 64 x 128 B of the Y digit tiles.
// Launched with cluster dimension C (C == 1: a plain launch).  gridDim.x is a multiple of C.
template <int S, int C>
__global__ void __launch_bounds__(K3_THREADS, 1)
bsr_i8_kernel(const __grid_constant__ CUtensorMap tmHd, const __grid_constant__ CUtensorMap tmYd, const K3Params prm) {
  using Cf = K3Cfg<S>;
  constexpr int NH = Cf::NH;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
  uint8_t* ybuf = smem;                          // 2 x YBUF
  uint8_t* hring = smem + 2 * Cf::YBUF;           // NH x HSLOT
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cf::BAR_OFFSET);
  uint64_t* yfull = bars;                        // [2]
  uint64_t* yempty = bars + 2;                   // [2]
  uint64_t* hfull = bars + 4;                    // [NH]
  uint64_t* hempty = bars + 4 + NH;              // [NH]
  uint64_t* accfull = bars + 4 + 2 * NH;
  uint64_t* accempty = accfull + 1;
  int32_t* ce_s = reinterpret_cast<int32_t*>(smem + Cf::CS_OFFSET);      // eY_j of the current tile
  uint32_t* cm_s = reinterpret_cast<uint32_t*>(smem + Cf::CM_OFFSET);    // column maxima of the current tile
  uint32_t* tmem_slot = cm_s + 64;
  int32_t* cp_s = reinterpret_cast<int32_t*>(smem + Cf::CP_OFFSET);      // predicted exponents of the output columns
  K3Queue* wq = reinterpret_cast<K3Queue*>(smem + Cf::Q_OFFSET);         // work items of this cluster

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t nitems = (uint32_t)((int64_t)prm.nb * prm.nctg);   // cluster work items (< 2^32, checked on the host)
  const int32_t crank = (C > 1) ? (int32_t)cluster_ctarank() : 0;
  constexpr uint16_t cmask = (uint16_t)((1u << C) - 1u);
  const int32_t b = prm.b;
  const int32_t ksteps = b >> 5;                 // 32-deep int8 MMAs per tile of H

  if (threadIdx.x == 0) {
    for (int i = 0; i < 2; ++i) { mbar_init(&yfull[i], 1); mbar_init(&yempty[i], 1); }
    for (int i = 0; i < NH; ++i) { mbar_init(&hfull[i], 1); mbar_init(&hempty[i], C); }   // a slot is free once all C CTAs have read it
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
  if (C > 1) cluster_sync_all();                 // peers' barriers are initialised before anything is sent to them
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ===================================== TMA producer =====================================
    if (elect_one()) {
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmHd) : "memory");
      asm volatile("prefetch.tensormap [%0];" ::"l"(&tmYd) : "memory");
      int yb = 0, hs = 0;
      uint32_t yph = 0, hph = 0;
      const int32_t hrows = b / C;               // rows of every H plane this CTA fetches for the cluster
      int qs = 0;
      uint32_t qph = 0;
      bool primed = false;                       // (experiment builds) the rings hold real data
      K3Fetch fetch;
      if (crank == 0)
        for (int i = 0; i < K3_QAHEAD; ++i) k3_q_fetch<C>(wq, fetch, prm.counter, nitems);
      for (;;) {
        const uint32_t u = k3_q_pop(wq, qs, qph, true);
        if (u == K3_NOITEM) break;
        if (crank == 0) k3_q_fetch<C>(wq, fetch, prm.counter, nitems);
        int32_t I, ctg;
        k3_decode(prm, u, I, ctg);
        const int32_t ct = prm.ct_begin + ctg * C + crank;
        const int32_t p0 = prm.brow_ptr[I];
        const int32_t p1 = p0 + min(prm.brow_ptr[I + 1] - p0, k3_jlimit<C>(prm, ctg));
        for (int32_t p = p0; p < p1; ++p) {
          const int32_t J = K3_EXP(16) ? 0 : prm.bcol[p];       // experiment builds: every Y load hits the same tiles (no DRAM traffic for Y)
          mbar_wait(&yempty[yb], yph ^ 1);
          const bool skip_tma = K3_EXP(2) && (primed || p >= p0 + 2);
          mbar_expect_tx(&yfull[yb], skip_tma ? 0u : (uint32_t)Cf::YBUF);
          if (skip_tma) {}
          else if (prm.l2hints) tma_load_3d_hint(ybuf + yb * Cf::YBUF, &tmYd, 0, 0, (J * prm.nct + ct) * S, &yfull[yb], L2_EVICT_LAST);
          else tma_load_3d(ybuf + yb * Cf::YBUF, &tmYd, 0, 0, (J * prm.nct + ct) * S, &yfull[yb]);
#pragma unroll 1
          for (int q = 0; q < S; ++q) {
            mbar_wait(&hempty[hs], hph ^ 1);       // all C CTAs have finished with this slot
            mbar_expect_tx(&hfull[hs], skip_tma ? 0u : (uint32_t)b * 128u);
            if (skip_tma) { if (++hs == NH) { hs = 0; hph ^= 1; } continue; }
            uint8_t* hdst = hring + hs * Cf::HSLOT + (C > 1 ? crank * hrows * 128 : 0);
            const int32_t hrow = ((K3_EXP(32) ? 0 : p) * prm.hplanes + k3_plane<S>(q)) * b + (C > 1 ? crank * hrows : 0);   // (32: none for H)
            if (C > 1) {
              if (prm.l2hints == 1) tma_load_2d_mc_hint(hdst, &tmHd, 0, hrow, &hfull[hs], cmask, L2_EVICT_FIRST);
              else tma_load_2d_mc(hdst, &tmHd, 0, hrow, &hfull[hs], cmask);
            } else {
              if (prm.l2hints == 1) tma_load_2d_hint(hdst, &tmHd, 0, hrow, &hfull[hs], L2_EVICT_FIRST);
              else tma_load_2d(hdst, &tmHd, 0, hrow, &hfull[hs]);
            }
            if (++hs == NH) { hs = 0; hph ^= 1; }
          }
          yb ^= 1;
          if (yb == 0) yph ^= 1;
        }
        primed = true;
      }
    }
  } else if (warp == 1) {
    // ====================================== MMA issuer ======================================
    if (elect_one()) {
      int yb = 0, hs = 0;
      uint32_t yph = 0, hph = 0, aph = 0;
      // descriptors differ only in the 14-bit start-address field of the low word
      const uint64_t dbase = umma_desc_sw128(0);
      const uint32_t ylo0 = (smem_u32(ybuf) & 0x3ffffu) >> 4, hlo0 = (smem_u32(hring) & 0x3ffffu) >> 4;
      int qs = 0;
      uint32_t qph = 0;
      int64_t it = -1;
      for (;;) {
        const uint32_t u = k3_q_pop(wq, qs, qph, true);
        if (u == K3_NOITEM) break;
        ++it;
        int32_t I, ctg;
        k3_decode(prm, u, I, ctg);
        const int32_t nJ = min(prm.brow_ptr[I + 1] - prm.brow_ptr[I], k3_jlimit<C>(prm, ctg));
        if (nJ == 0) continue;
        K3_TRACE_DECL(it < 512);
        K3_TRACE(0, clock64());
        mbar_wait(accempty, aph ^ 1);            // the epilogue has drained the previous item's accumulators
        asm volatile("tcgen05.fence::after_thread_sync;");
        K3_TRACE(1, clock64());
        K3_TRACE(7, (unsigned long long)nJ);
        for (int32_t j = 0; j < nJ; ++j) {
          mbar_wait(&yfull[yb], yph);
          const uint32_t ylo = ylo0 + (uint32_t)yb * (Cf::YBUF >> 4);
#pragma unroll
          for (int ip = 0; ip < S; ++ip) {
            const int p = k3_plane<S>(ip);
            mbar_wait(&hfull[hs], hph);
            asm volatile("tcgen05.fence::after_thread_sync;");
            const uint32_t hlo = hlo0 + (uint32_t)hs * (Cf::HSLOT >> 4);
            const int ntot = (S - p) * K3_NT;       // Y planes 0..S-1-p side by side -> levels p..S-1
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {
              if (kk < ksteps) {
                const uint64_t da = dbase | (uint64_t)(hlo + kk * 2);
                // plane 0 comes first and spans every level: its first MMA of a work item overwrites the accumulators
                const uint32_t acc = (ip > 0 || kk > 0) ? 1u : (j > 0 ? 1u : 0u);
                // products wider than one instruction (256 columns) go as two EQUAL halves (448 = 224 + 224, 384 = 192 + 192,
                // 320 = 160 + 160): a 256 + 64 split leaves a narrow MMA that is bound by its shared-memory operand reads
                // ((4 KB of A + 32 N B) / 128 B per clock > N / 2 clocks for N < 128); -1.5 % cycles per tile measured
                if (ntot > 256) {
                  const int nh = ntot / 2;            // a multiple of 32 for every S - p
                  umma_i8<1>(tmem_base + (uint32_t)(p * K3_NT), da, dbase | (uint64_t)(ylo + kk * 2), umma_idesc_i8(nh), acc);
                  umma_i8<2>(tmem_base + (uint32_t)(p * K3_NT + nh), da, dbase | (uint64_t)(ylo + nh * 8 + kk * 2), umma_idesc_i8(nh), acc);
                } else {
                  umma_i8(tmem_base + (uint32_t)(p * K3_NT), da, dbase | (uint64_t)(ylo + kk * 2), umma_idesc_i8(ntot), acc);
                }
              }
            }
            if (C > 1) umma_commit_mc(&hempty[hs], cmask);   // slot free (in every CTA) once these MMAs have read it
            else umma_commit(&hempty[hs]);
            if (++hs == NH) { hs = 0; hph ^= 1; }
          }
          umma_commit(&yempty[yb]);
          yb ^= 1;
          if (yb == 0) yph ^= 1;
        }
        umma_commit(accfull);
        K3_TRACE(2, clock64());
        aph ^= 1;
      }
    }
  } else {
    // ======================================= epilogue =======================================
    // 8 warps: warp w reads TMEM lane quarter w & 3 (rows 32q..32q+31 of the block row) and column half
    // (w - 2) >> 2 (32 of the item's 64 columns): twice the warps of a one-warp-per-quarter epilogue and half the
    // registers per thread, i.e. four times the loads in flight -- the output phase is a chain of dependent
    // load -> fma -> store batches whose latency is ~8 K cycles behind the TMA traffic of the same SM, and with
    // 4 warps it took 70 K cycles per item, longer than the MMAs of every block row with <= 18 tiles.
    constexpr int NCW = K3_NT / 2;               // columns per warp
    const int quarter = warp & 3;
    const int half = (warp - 2) >> 2;
    const int et = (warp - 2) * 32 + lane;       // 0..255 among the epilogue threads
    const int r = quarter * 32 + lane;           // row inside the block row
    const bool row_ok = r < b;
    const bool warp_ok = (quarter * 32) < b;     // b is a multiple of 32: a warp's rows are all valid or all padding
    const double alpha = prm.alpha, beta = prm.beta;
    const bool use_z = (beta != 0.0);
    const bool use_s = (prm.S != nullptr);
    uint32_t aph = 0;
    int qs = 0;
    uint32_t qph = 0;
    int64_t it = -1;
    for (;;) {
      const uint32_t u = k3_q_pop_warp(wq, qs, qph);
      if (u == K3_NOITEM) break;
      ++it;
      int32_t I, ctg;
      k3_decode(prm, u, I, ctg);
      const int32_t ct = prm.ct_begin + ctg * C + crank;
      const int32_t nJ = prm.brow_ptr[I + 1] - prm.brow_ptr[I];
      if (prm.skip_empty && nJ == 0) continue;           // uniform over the epilogue warps
      const int64_t col0 = (int64_t)ct * K3_NT;          // first column of the item
      const int64_t colw = col0 + half * NCW;            // first column of this warp
      const int64_t row = (int64_t)I * b + r;
      const bool row_in = row_ok && row < prm.mrows;
      if (et < 64) {
        const int64_t cj = col0 + et;
        ce_s[et] = cj < prm.ncols ? prm.eS[cj] : I8_EMIN;
        cm_s[et] = 0;
        if (prm.dO) cp_s[et] = cj < prm.ncols ? prm.ePredO[cj] : I8_EMIN;
      }
      double rsp = 0.0, gi = prm.gamma;
      const bool full = (col0 + K3_NT <= prm.ncols);
      if (row_in) {
        rsp = alpha * pow2i(prm.eH[row] - 30);    // alpha * 2^(eH_i - 14) / 2^16 (k3_drain returns 2^16 * v)
        gi = prm.hdiag ? fma(alpha, prm.hdiag[row], prm.gamma) : prm.gamma;
        if (full) {   // pull this thread's two lines of Y_k and Y_{k-1} towards L2 while the warp waits for the accumulators
          const double* sp0 = prm.S + row * prm.lds + colw;
          const double* zp0 = prm.Z + row * prm.ldz + colw;
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            if (use_s) asm volatile("prefetch.global.L2 [%0];" ::"l"(sp0 + 16 * k));
            if (use_z) asm volatile("prefetch.global.L2 [%0];" ::"l"(zp0 + 16 * k));
          }
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");

      double v[NCW];
      K3_TRACE_DECL(it < 512 && et == 0);
      K3_TRACE(3, clock64());
      if (nJ > 0) {
        mbar_wait(accfull, aph);
        aph ^= 1;
        K3_TRACE(4, clock64());
        asm volatile("tcgen05.fence::after_thread_sync;");
        if (K3_EXP(8)) {
#pragma unroll
          for (int i = 0; i < NCW; ++i) v[i] = 1.0;
        } else
        k3_drain<S, NCW>(tmem_base + ((uint32_t)(quarter * 32) << 16) + (uint32_t)(half * NCW), v);
        asm volatile("tcgen05.fence::before_thread_sync;");
        mbar_arrive(accempty);                   // TMEM is free for the next work item
        K3_TRACE(5, clock64());
      } else {
#pragma unroll
        for (int i = 0; i < NCW; ++i) v[i] = 0.0;
      }

      // ---- out = alpha * 2^(eH+eY-30) * v + (alpha*hdiag + gamma) * y + beta * z   (v = 2^16 * Horner) ----
      // three fp64 instructions per element: v * (alpha 2^(eH-30)), then the column's 2^eY by an exponent add, two FMAs
      uint32_t cmx = 0;                           // column maximum (upper word) this lane has seen
      bool cmax_done = false;
      if (K3_EXP(4)) {
        double sacc = 0.0;
#pragma unroll
        for (int c = 0; c < NCW; ++c) sacc += v[c] * rsp;
        if (sacc == 1.2345e-300) prm.O[0] = sacc;      // keeps the drain alive, never true
        cmax_done = true;
      } else
      if (full) {
        // Coalesced output: after the drain a thread owns one ROW (32 columns); written that way every access of
        // a warp would touch 32 different lines.  The 32 x 32 block of the warp is transposed in registers (5 shuffle
        // stages): afterwards lane l owns column l of all 32 rows and every access is one contiguous 256-byte segment.
#pragma unroll
        for (int c = 0; c < NCW; ++c) v[c] *= rsp;               // x alpha 2^(eH_i-30), own row
#pragma unroll
        for (int k = 16; k >= 1; k >>= 1) {
          const bool up = (lane & k) != 0;
#pragma unroll
          for (int j = 0; j < 32; ++j) {
            if (j & k) continue;
            const double snd = up ? v[j] : v[j | k];
            const double rcv = __shfl_xor_sync(0xffffffffu, snd, k);
            if (up) v[j] = rcv; else v[j | k] = rcv;
          }
        }
        // v[r] = (row r of this warp, column colw + lane)
        const int32_t ce = ce_s[half * NCW + lane];
        // digits of the output for the next step (prm.dO): lane l owns column l, four consecutive rows give one k-major word per plane
        const bool digits_out = (prm.dO != nullptr);
        const int32_t cpred = digits_out ? cp_s[half * NCW + lane] : 0;
        const double dscale = pow2i(8 * S - 1 - cpred);
        uint8_t* dtile = digits_out ? reinterpret_cast<uint8_t*>(prm.dO) + ((int64_t)I * prm.nct + ct) * (int64_t)(S * K3_NT * 128) +
                                          (half * NCW + lane) * 128 + quarter * 32
                                    : nullptr;
        if (digits_out && !warp_ok) {
          // rows beyond b of a narrow tile: the k bytes of this quarter stay zero in every plane
#pragma unroll
          for (int q = 0; q < S; ++q) {
            *reinterpret_cast<uint4*>(dtile + q * (K3_NT * 128)) = make_uint4(0, 0, 0, 0);
            *reinterpret_cast<uint4*>(dtile + q * (K3_NT * 128) + 16) = make_uint4(0, 0, 0, 0);
          }
        }
        if (warp_ok) {
          const int64_t wrow0 = (int64_t)I * b + quarter * 32;
          const double* sw = prm.S + wrow0 * prm.lds + colw + lane;
          const double* zw = prm.Z + wrow0 * prm.ldz + colw + lane;
          double* ow = prm.O + wrow0 * prm.ldo + colw + lane;
          const int nrow = (int)min((int64_t)32, prm.mrows - wrow0);       // < 32 only in a ragged last block (warp-uniform)
          uint32_t dw[S][4];                       // digit words of 16 rows: one 16-byte store per plane
#pragma unroll
          for (int r0 = 0; r0 < 32; r0 += 8) {
            if (r0 < nrow) {
              double y[8], z[8], ov[8];
              if (use_s) {
#pragma unroll
                for (int i = 0; i < 8; ++i) y[i] = (r0 + i < nrow) ? __ldcs(sw + (int64_t)(r0 + i) * prm.lds) : 0.0;   // read once: evict first
              }
              if (use_z) {
#pragma unroll
                for (int i = 0; i < 8; ++i) z[i] = (r0 + i < nrow) ? __ldcs(zw + (int64_t)(r0 + i) * prm.ldz) : 0.0;
              }
#pragma unroll
              for (int i = 0; i < 8; ++i) {
                const double gr = __shfl_sync(0xffffffffu, gi, r0 + i);     // alpha * hdiag + gamma of row r0+i
                double o = scale_pow2(v[r0 + i], ce);
                if (use_s) o = fma(gr, y[i], o);
                if (use_z) o = fma(beta, z[i], o);
                ov[i] = o;
                if (r0 + i < nrow) {
                  __stcs(ow + (int64_t)(r0 + i) * prm.ldo, o);
                  cmx = max(cmx, abs_hi(o));
                }
              }
              if (digits_out) {
#pragma unroll
                for (int g = 0; g < 2; ++g) {
                  const double x4[4] = {ov[4 * g], ov[4 * g + 1], ov[4 * g + 2], ov[4 * g + 3]};
                  uint32_t w[S];
                  digits4<S>(x4, dscale, w);
#pragma unroll
                  for (int q = 0; q < S; ++q) dw[q][((r0 >> 2) & 3) + g] = w[q];
                }
                if (r0 & 8) {
#pragma unroll
                  for (int q = 0; q < S; ++q)
                    *reinterpret_cast<uint4*>(dtile + q * (K3_NT * 128) + (r0 & 16)) = make_uint4(dw[q][0], dw[q][1], dw[q][2], dw[q][3]);
                }
              }
            }
          }
          // a column that outgrew its predicted exponent: its digits are invalid, the tile is redone before the next step
          if (digits_out && exp_from_hi(cmx) > cpred) atomicOr(&prm.flagsO[ct], 1u);
        }
        if (prm.cmaxO && cmx) atomicMax(&cm_s[half * NCW + lane], cmx);   // this lane has seen all 32 rows of its column
        cmax_done = true;
      } else {
        // ragged last column tile: every thread writes its own row; its digit tile is left to y_digits_fix_kernel
        if (prm.dO && et == 0) atomicOr(&prm.flagsO[ct], 1u);
        const double* sp = prm.S + row * prm.lds + colw;
        const double* zp = prm.Z + row * prm.ldz + colw;
        double* op = prm.O + row * prm.ldo + colw;
#pragma unroll
        for (int j = 0; j < NCW; ++j) {
          double o = 0.0;
          if (row_in && colw + j < prm.ncols) {
            o = scale_pow2(v[j] * rsp, ce_s[half * NCW + j]);
            if (use_s) o = fma(gi, sp[j], o);
            if (use_z) o = fma(beta, zp[j], o);
            op[j] = o;
          }
          v[j] = o;
        }
      }
      // ---- column maxima of the new iterate (upper words), for the next step's digit scaling ----
      if (prm.cmaxO) {
        if (!cmax_done) {
#pragma unroll
          for (int j = 0; j < NCW; ++j) {
            const uint32_t m = __reduce_max_sync(0xffffffffu, abs_hi(v[j]));
            if (lane == j && m) atomicMax(&cm_s[half * NCW + j], m);
          }
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (et < 64 && col0 + et < prm.ncols && cm_s[et]) atomicMax(&prm.cmaxO[col0 + et], cm_s[et]);
      }
      K3_TRACE(6, clock64());
      asm volatile("bar.sync 1, 256;" ::: "memory");   // ce_s / cm_s are rewritten by the next item
    }
  }

  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  if (C > 1) cluster_sync_all();                 // no CTA leaves while a peer may still signal its barriers
  if (warp == 1) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "n"(512));
}

}  // namespace ttdft
