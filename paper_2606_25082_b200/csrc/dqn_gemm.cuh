// dqn_gemm.cuh -- the dense contraction of the DQN training step on the 5th-generation
// tensor cores: C[M][N] = sum_k A[m][k] * B[n][k], fp32 in, fp32 out, both operands K-major (k contiguous), computed as a
// 3 x TF32 split so that the result is fp32-accurate:
//     a = a_hi + a_lo, a_hi = a with the low 13 mantissa bits cleared (exactly a TF32 number), a_lo = a - a_hi (exact);
//     a b ~ a_hi b_hi + a_hi b_lo + a_lo b_hi   (the dropped a_lo b_lo term is 2^-22 relative, a_lo / b_lo lose 2^-11 of
//     themselves when the tensor core reads them as TF32: about 2^-21 of each product in all, fp32 accumulation in TMEM).
// One CTA computes one 128 x BN tile of C (or one split-K partial of it):
//   warp 0      TMA producer: cp.async.bulk.tensor loads of a 128 x 32 tile of A and a BN x 32 tile of B per stage (one
//               128-byte swizzled row = 32 floats of k), completion on an mbarrier; it also owns the TMEM allocation;
//   warps 2..5  split the landed tiles in place (hi over the TMA'd data, lo into a second buffer at the SAME offsets, so
//               the 128-byte swizzle never has to be decoded), fence.proxy.async, arrive;
//   warps 6..9  epilogue: tcgen05.ld of the accumulator (each warp its own 32 TMEM lanes = 32 rows), bias / ReLU / ReLU-mask,
//               row-major store and / or TRANSPOSED store (32 lanes = 32 consecutive m: coalesced), or a split-K partial;
//               TMEM holds TWO accumulators, so this overlaps the products of the CTA's next tile (persistent kernel);
//   warp 1      one elected lane issues 3 x 4 tcgen05.mma.kind::tf32 per stage (UMMA K = 8 floats = 32 bytes; the shared-
//               memory descriptor advances by 32 bytes inside the swizzled row), accumulator in TMEM (BN columns x 128
//               lanes), tcgen05.commit frees the stage / publishes the accumulator.
// Every matrix product of the training step goes through this one kernel.  The weight-gradient products contract over the
// BATCH rows of two row-major activations: they run the MN = true instantiation, which reads both operands MN-major straight
// from the row-major tensors (no transposed copy of an activation exists).  The epilogue can still write a transposed result
// (out_t): the K-major weight-gradient path over such copies is kept behind MIG_DQN_MN=0 (dqn.cu) for A/B timing.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace migsim {

constexpr int kGemmBM = 128;           // rows of C per CTA = TMEM lanes
constexpr int kGemmBK = 32;            // floats of k per stage: one 128-byte swizzled row
constexpr int kGemmThreads = 320;      // 10 warps: TMA, MMA, 4 x hi/lo split, 4 x epilogue

enum { EPI_BIAS = 1, EPI_RELU = 2, EPI_MASK = 4 /* multiply by (mask[m][n] > 0) */ };

struct GemmArgs {
  uint32_t M, N, K;                    // C is M x N; K = the contraction length of ONE split
  uint32_t k_blocks;                   // K / 32 per split (the last block may run past K: TMA fills zeros)
  uint32_t splits;                     // split-K factor (1 = none)
  float *out; uint32_t ldo;            // row-major result (or NULL); split z writes at out + z * out_split_stride
  float *out_t; uint32_t ldt;          // transposed result out_t[n][m] (or NULL)
  size_t out_split_stride;             // elements between the partials of consecutive splits (0 without split-K)
  const float *bias;                   // [N] (EPI_BIAS)
  const float *mask; uint32_t ldm;     // [M][ldm] (EPI_MASK): the forward activation whose ReLU is differentiated
  uint32_t epi;
  uint32_t b_lo_row;                   // 0: B is fp32 and split here.  > 0: B was written split (TF32 high parts in rows [0, N), the
                                       // remainders in rows [b_lo_row, b_lo_row + N) of the same map): both tiles are loaded, none is split
};

// ---------------------------------------------------------------------------------------------- PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred P1;\n\tWAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n\t"
      "@P1 bra DONE_%=;\n\tbra WAIT_%=;\n\tDONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *map, uint64_t *bar, int c0, int c1) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];"
               ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1) : "memory");
}
// shared-memory matrix descriptor of a K-major tile with 128-byte swizzle: rows of 128 bytes, 8-row groups 1024 bytes apart
__device__ __forceinline__ uint64_t umma_desc_k_sw128(uint32_t saddr) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)1 << 16) | ((uint64_t)(1024 >> 4) << 32) | ((uint64_t)1 << 46) | ((uint64_t)2 << 61);
}
// the same for an MN-major tile (the m / n index contiguous in memory: a row-major [k][m] block, as TMA brings it from a
// row-major activation [batch][features] when the contraction runs over the batch).  32-bit MN-major operands have ONE
// shared-memory layout: 128-byte rows of 32 m, swizzled in 32-byte chunks (layout type 1; TMA's SWIZZLE_128B_ATOM_32B), in
// atoms of 4 k-rows (512 bytes); LBO = bytes between atoms along m / n (the next 32 columns), SBO = bytes between atoms
// along k.  One UMMA (K = 8) reads two k-atoms = 8 rows = 1024 bytes of every 32-column block.
__device__ __forceinline__ uint64_t umma_desc_mn_sw128_32b(uint32_t saddr, uint32_t lbo_bytes) {
  return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) | ((uint64_t)(512 >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)1 << 61);
}
// instruction descriptor: D = fp32, A = B = TF32, M x N; both operands K-major, or both MN-major (bits 15, 16)
__device__ __forceinline__ uint32_t umma_idesc_tf32(uint32_t m, uint32_t n, bool mn_major = false) {
  return (1u << 4) | (2u << 7) | (2u << 10) | ((n >> 3) << 17) | ((m >> 4) << 24) | (mn_major ? (3u << 15) : 0u);
}
__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\ttcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
               ::"r"(tmem_d), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t *bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, float v[8]) {
  uint32_t r[8];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 8; ++i) v[i] = __uint_as_float(r[i]);
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float v[16]) {
  uint32_t r[16];
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]),
                 "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]) : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int i = 0; i < 16; ++i) v[i] = __uint_as_float(r[i]);
}

template <int BN> struct GemmSmem {
  static constexpr int kStageA = kGemmBM * kGemmBK * 4;        // 16 KB
  static constexpr int kStageB = BN * kGemmBK * 4;
  static constexpr int kStage = 2 * (kStageA + kStageB);      // hi + lo of both operands
  static constexpr int kStages = (200 * 1024) / kStage >= 4 ? 4 : (200 * 1024) / kStage;
  static constexpr int kBytes = kStages * kStage + 1024 /* alignment slack */ + 256 /* barriers, tmem address */;
  static constexpr int kAccCols = BN < 32 ? 32 : BN;         // TMEM columns of one accumulator
  static constexpr int kTmemCols = 2 * kAccCols;             // two accumulators: the epilogue of tile i overlaps the products of tile i + 1
};

// ---------------------------------------------------------------------------------------------- the kernel
// PERSISTENT: gridDim.x CTAs (one per SM) walk the tiles t = blockIdx.x, + gridDim.x, ... of the tiles_m x tiles_n x splits
// grid (n fastest: consecutive tiles share their rows of A in L2).  The shared-memory ring and its mbarrier phases run
// straight through the tile boundaries, so the producer is already loading tile i + 1 while tile i's last stages are
// multiplied and its accumulator is drained.
// MN = true: C[M][N] = sum_k A[k][m] * B[k][n] -- both operands MN-major (row-major [K][M] and [K][N] in global memory: the
// weight-gradient products, whose contraction runs over the batch rows of two row-major activations).  A stage then holds
// 4 blocks [32 k][32 m] of A (4 KB each) and BN / 32 such blocks of B (BN a multiple of 32); everything else (split,
// accumulators, epilogues) is the same.
template <int BN, bool MN = false>
__global__ void __launch_bounds__(kGemmThreads, 1)
gemm_tf32x3_kernel(const __grid_constant__ CUtensorMap map_a, const __grid_constant__ CUtensorMap map_b, const GemmArgs g) {
  using S = GemmSmem<BN>;
  extern __shared__ unsigned char gemm_smem_raw[];
  unsigned char *base = reinterpret_cast<unsigned char *>((reinterpret_cast<uintptr_t>(gemm_smem_raw) + 1023) & ~(uintptr_t)1023);
  unsigned char *tiles = base;
  uint64_t *bars = reinterpret_cast<uint64_t *>(base + S::kStages * S::kStage);
  uint64_t *full = bars, *split = bars + S::kStages, *empty = bars + 2 * S::kStages, *acc_full = bars + 3 * S::kStages, *acc_empty = acc_full + 2;
  uint32_t *tmem_slot = reinterpret_cast<uint32_t *>(acc_empty + 2);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t tiles_n = g.N / BN, tiles_mn = ((g.M + kGemmBM - 1) / kGemmBM) * tiles_n, n_tiles = tiles_mn * g.splits;

  if (warp == 0) {
    if (lane == 0) {
      for (int s = 0; s < S::kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&split[s], 128); mbar_init(&empty[s], 1); }
      for (int s = 0; s < 2; ++s) { mbar_init(&acc_full[s], 1); mbar_init(&acc_empty[s], 128); }
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncwarp();
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "n"(S::kTmemCols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  const uint32_t tmem = *tmem_slot;

  if (warp == 0) {
    // ===== TMA producer
    if (lane == 0) {
      uint32_t it = 0;                                         // k-blocks issued so far, over all tiles of this CTA
      for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint32_t z = tile / tiles_mn, mn = tile - z * tiles_mn, m0 = (mn / tiles_n) * kGemmBM, n0 = (mn % tiles_n) * BN;
        const int k_first = (int)(z * g.k_blocks * kGemmBK);
        for (uint32_t kb = 0; kb < g.k_blocks; ++kb, ++it) {
          const int s = it % S::kStages; const uint32_t round = it / S::kStages;
          if (round) mbar_wait(&empty[s], (round - 1) & 1u);
          unsigned char *st = tiles + s * S::kStage;
          mbar_expect_tx(&full[s], S::kStageA + (g.b_lo_row ? 2 : 1) * S::kStageB);
          if constexpr (MN) {                                  // boxes of {32 (or 16) columns, 32 batch rows}: coordinates {column, row}
            const int k0 = k_first + (int)kb * kGemmBK;
#pragma unroll
            for (int j = 0; j < kGemmBM / 32; ++j) tma_load_2d(st + j * 4096, &map_a, &full[s], (int)m0 + 32 * j, k0);
            static_assert(!MN || BN % 32 == 0, "MN-major tiles are blocks of 32 columns");
#pragma unroll
            for (int j = 0; j < BN / 32; ++j) tma_load_2d(st + 2 * S::kStageA + j * 4096, &map_b, &full[s], (int)n0 + 32 * j, k0);
            continue;
          }
          tma_load_2d(st, &map_a, &full[s], k_first + (int)kb * kGemmBK, (int)m0);
          tma_load_2d(st + 2 * S::kStageA, &map_b, &full[s], k_first + (int)kb * kGemmBK, (int)n0);
          if (g.b_lo_row)                                      // B was split when it was written (weights): its low parts are rows of the same map
            tma_load_2d(st + 2 * S::kStageA + S::kStageB, &map_b, &full[s], k_first + (int)kb * kGemmBK, (int)(g.b_lo_row + n0));
        }
      }
    }
  } else if (warp == 1) {
    // ===== MMA issuer
    const uint32_t idesc = umma_idesc_tf32(kGemmBM, BN, MN);
    uint32_t it = 0, ti = 0;
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++ti) {
      const uint32_t as = ti & 1u, around = ti >> 1;          // accumulator stage and how often it has been used
      if (around) mbar_wait(&acc_empty[as], (around - 1) & 1u);      // the epilogue has drained this accumulator
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t acc = tmem + as * (uint32_t)S::kAccCols;
      for (uint32_t kb = 0; kb < g.k_blocks; ++kb, ++it) {
        const int s = it % S::kStages; const uint32_t round = it / S::kStages;
        mbar_wait(&split[s], round & 1u);
        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
        if (lane == 0) {                                       // ONE thread issues every MMA: they execute in its issue order
          const uint32_t a_hi = smem_u32(tiles + s * S::kStage), a_lo = a_hi + S::kStageA, b_hi = a_hi + 2 * S::kStageA, b_lo = b_hi + S::kStageB;
          if constexpr (MN) {
#pragma unroll
            for (int k = 0; k < kGemmBK / 8; ++k) {            // UMMA K = 8 batch rows = 1024 bytes down every 32-column block
              const uint32_t o = (uint32_t)k * 1024u;
              umma_tf32(acc, umma_desc_mn_sw128_32b(a_lo + o, 4096), umma_desc_mn_sw128_32b(b_hi + o, 4096), idesc, (kb | (uint32_t)k) != 0u);
              umma_tf32(acc, umma_desc_mn_sw128_32b(a_hi + o, 4096), umma_desc_mn_sw128_32b(b_lo + o, 4096), idesc, 1u);
              umma_tf32(acc, umma_desc_mn_sw128_32b(a_hi + o, 4096), umma_desc_mn_sw128_32b(b_hi + o, 4096), idesc, 1u);
            }
          } else
#pragma unroll
          for (int k = 0; k < kGemmBK / 8; ++k) {              // UMMA K = 8 floats = 32 bytes inside the swizzled row
            const uint32_t o = (uint32_t)k * 32u;
            umma_tf32(acc, umma_desc_k_sw128(a_lo + o), umma_desc_k_sw128(b_hi + o), idesc, (kb | (uint32_t)k) != 0u);
            umma_tf32(acc, umma_desc_k_sw128(a_hi + o), umma_desc_k_sw128(b_lo + o), idesc, 1u);
            umma_tf32(acc, umma_desc_k_sw128(a_hi + o), umma_desc_k_sw128(b_hi + o), idesc, 1u);
          }
          umma_commit(&empty[s]);                              // (implies tcgen05.fence::before_thread_sync)
          if (kb + 1 == g.k_blocks) umma_commit(&acc_full[as]);
        }
        __syncwarp();
      }
    }
  } else if (warp < 6) {
    // ===== hi / lo split of every landed stage, in place
    const int t = threadIdx.x - 64;                            // 0..127
    uint32_t it = 0;
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
      for (uint32_t kb = 0; kb < g.k_blocks; ++kb, ++it) {
        const int s = it % S::kStages; const uint32_t round = it / S::kStages;
        mbar_wait(&full[s], round & 1u);
        unsigned char *st = tiles + s * S::kStage;
        float4 *a_hi = reinterpret_cast<float4 *>(st), *a_lo = reinterpret_cast<float4 *>(st + S::kStageA);
        float4 *b_hi = reinterpret_cast<float4 *>(st + 2 * S::kStageA), *b_lo = reinterpret_cast<float4 *>(st + 2 * S::kStageA + S::kStageB);
#pragma unroll 4
        for (int i = t; i < S::kStageA / 16; i += 128) {
          const float4 x = a_hi[i];
          float4 h, l;
          h.x = __uint_as_float(__float_as_uint(x.x) & 0xFFFFE000u); l.x = x.x - h.x;
          h.y = __uint_as_float(__float_as_uint(x.y) & 0xFFFFE000u); l.y = x.y - h.y;
          h.z = __uint_as_float(__float_as_uint(x.z) & 0xFFFFE000u); l.z = x.z - h.z;
          h.w = __uint_as_float(__float_as_uint(x.w) & 0xFFFFE000u); l.w = x.w - h.w;
          a_hi[i] = h; a_lo[i] = l;
        }
        if (!g.b_lo_row)
#pragma unroll 4
        for (int i = t; i < S::kStageB / 16; i += 128) {
          const float4 x = b_hi[i];
          float4 h, l;
          h.x = __uint_as_float(__float_as_uint(x.x) & 0xFFFFE000u); l.x = x.x - h.x;
          h.y = __uint_as_float(__float_as_uint(x.y) & 0xFFFFE000u); l.y = x.y - h.y;
          h.z = __uint_as_float(__float_as_uint(x.z) & 0xFFFFE000u); l.z = x.z - h.z;
          h.w = __uint_as_float(__float_as_uint(x.w) & 0xFFFFE000u); l.w = x.w - h.w;
          b_hi[i] = h; b_lo[i] = l;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core
        mbar_arrive(&split[s]);
      }
    }
  } else {
    // ===== epilogue (warps 6..9: warp % 4 = 2, 3, 0, 1 -> each its own 32 TMEM lanes)
    const uint32_t q = (uint32_t)warp & 3u;
    uint32_t ti = 0;
    for (uint32_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x, ++ti) {
      const uint32_t z = tile / tiles_mn, mn = tile - z * tiles_mn, m0 = (mn / tiles_n) * kGemmBM, n0 = (mn % tiles_n) * BN;
      const uint32_t as = ti & 1u, around = ti >> 1;
      mbar_wait(&acc_full[as], around & 1u);
      asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
      const uint32_t m = m0 + q * 32u + (uint32_t)lane;
      const uint32_t trow = tmem + as * (uint32_t)S::kAccCols + ((q * 32u) << 16);
      float *orow = g.out ? g.out + (size_t)z * g.out_split_stride + (size_t)m * g.ldo + n0 : nullptr;
      const float *mrow = (g.epi & EPI_MASK) ? g.mask + (size_t)m * g.ldm + n0 : nullptr;
#pragma unroll 1
      for (int c = 0; c < BN; c += 16) {
        float v[16];
        tmem_ld16(trow + (uint32_t)c, v);
        if (g.epi & EPI_BIAS) {                                // (warp-uniform addresses: four 16-byte loads, not sixteen scalar ones)
          const float4 *b4 = reinterpret_cast<const float4 *>(g.bias + n0 + c);
#pragma unroll
          for (int j4 = 0; j4 < 4; ++j4) {
            const float4 bb = __ldg(b4 + j4);
            v[4 * j4] += bb.x; v[4 * j4 + 1] += bb.y; v[4 * j4 + 2] += bb.z; v[4 * j4 + 3] += bb.w;
          }
        }
        if (g.epi & EPI_RELU) {
#pragma unroll
          for (int j = 0; j < 16; ++j) v[j] = fmaxf(v[j], 0.0f);
        }
        if (mrow && m < g.M) {
#pragma unroll
          for (int j4 = 0; j4 < 4; ++j4) {
            const float4 k4 = *reinterpret_cast<const float4 *>(mrow + c + 4 * j4);
            v[4 * j4] = k4.x > 0.0f ? v[4 * j4] : 0.0f; v[4 * j4 + 1] = k4.y > 0.0f ? v[4 * j4 + 1] : 0.0f;
            v[4 * j4 + 2] = k4.z > 0.0f ? v[4 * j4 + 2] : 0.0f; v[4 * j4 + 3] = k4.w > 0.0f ? v[4 * j4 + 3] : 0.0f;
          }
        }
        if (m < g.M) {
          if (orow) {
#pragma unroll
            for (int j4 = 0; j4 < 4; ++j4) *reinterpret_cast<float4 *>(orow + c + 4 * j4) = make_float4(v[4 * j4], v[4 * j4 + 1], v[4 * j4 + 2], v[4 * j4 + 3]);
          }
          if (g.out_t) {
#pragma unroll
            for (int j = 0; j < 16; ++j) g.out_t[(size_t)(n0 + c + j) * g.ldt + m] = v[j];
          }
        }
      }
      asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
      mbar_arrive(&acc_empty[as]);                             // this accumulator may be overwritten
    }
  }
  __syncthreads();
  if (warp == 0) {
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(S::kTmemCols) : "memory");
  }
}

}  // namespace migsim
