// qnet_device.cuh -- batched Q-network forward, MLP 64 -> H -> H -> A, ReLU, fp32.
//
// Every output is accumulated as acc = b[n]; for k ascending: acc = fmaf(in[k], W[k][n], acc): one rounding per
// term, fixed order, so the result is bit-identical to a sequential CPU fmaf loop.  That is why this is a CUDA-core
// register-tiled kernel and not a tensor-core GEMM (split accumulation would change the argmax on near-ties and
// fork the DQN-driven event trace).  One CTA = 32 batch rows, H threads; activations live in shared memory
// k-major ([k][row]); weights stream from L2 (334 KB, resident) through a cp.async double buffer.
#pragma once
#include <cuda_runtime.h>

#include "philox.cuh"
#include "sim_common.h"

namespace migsim {

constexpr int kQRows = 32;

struct QArgs {
  const float *W1, *b1, *W2, *b2, *W3, *b3;
  uint32_t H, A;
  const float *state;   // [B][64]
  uint32_t B;
  float *q_out;         // [B][A] or NULL
  uint8_t *argmax_out;  // [B] or NULL
  // epsilon-greedy from Philox stream 2 (R2): action_out[B]
  uint8_t *action_out;  // NULL = no policy
  uint32_t eps_thr;     // explore iff w_explore < eps_thr = min(round(eps 2^32), 2^32 - 1)
  uint32_t epoch, k0, k1, episode, env_base;
};

// one dense layer for the CTA's 32 rows.  A thread computes a register tile of kQCols adjacent columns x kQRpt rows
// (32 accumulators); W is streamed through shared memory in chunks of kQChunk rows with cp.async (one copy per CTA, no
// register waits for a weight), activations are read as broadcast LDS.128: per k three LDS.128 feed 32 FFMAs.
// Measured on B200: 34.2 TFLOP/s at B = 262 144 (46 % of the FP32 peak), 25.7 at C4's B = 8192; the first version (one
// column x 32 rows per thread, weights by LDG from L2) reached 24.6 / 18.5.  Each output is still ONE chain
// acc = fmaf(in[k], W[k][n], acc) in ascending k: the tiling changes which thread owns an output, not its arithmetic.
// in: [K][32] k-major, out: [H][32].
constexpr int kQCols = 4, kQRpt = 8;

constexpr int kQChunk = 16, kQStages = 2;    // rows of W per cp.async stage; stages in flight

// W is streamed through shared memory in chunks of kQChunk rows (cp.async, kQStages deep): one copy per CTA instead of
// one L2 fetch per row group, and no register waits for a weight.
template <bool RELU>
__device__ __forceinline__ void q_layer(const float *__restrict__ W, const float *__restrict__ b, int K, int H,
                                        const float *in, float *out, float4 *stage, int tid) {
  const int n0 = (tid / (kQRows / kQRpt)) * kQCols, r0 = (tid % (kQRows / kQRpt)) * kQRpt;
  float acc[kQCols][kQRpt];
  const float4 bias = *reinterpret_cast<const float4 *>(b + n0);
#pragma unroll
  for (int r = 0; r < kQRpt; ++r) { acc[0][r] = bias.x; acc[1][r] = bias.y; acc[2][r] = bias.z; acc[3][r] = bias.w; }
  const int nch = K / kQChunk, per = kQChunk * H / 4;          // float4 per chunk = 2 per thread (blockDim.x == H)
  auto issue = [&](int c) {
    if (c < nch) {
      const float4 *src = reinterpret_cast<const float4 *>(W + (size_t)c * kQChunk * H);
      float4 *dst = stage + (c % kQStages) * per;
      for (int e = tid; e < per; e += H) {
        const uint32_t d = (uint32_t)__cvta_generic_to_shared(dst + e);
        asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(src + e) : "memory");
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");        // (an empty group keeps the count uniform)
  };
  for (int c = 0; c < kQStages - 1; ++c) issue(c);
  for (int c = 0; c < nch; ++c) {
    asm volatile("cp.async.wait_group %0;" ::"n"(kQStages - 2) : "memory");   // chunk c has landed
    __syncthreads();                                            // ... for every thread; and chunk c - 1 is consumed
    issue(c + kQStages - 1);
    const float *ws = reinterpret_cast<const float *>(stage + (c % kQStages) * per) + n0;
    const float *xs = in + c * kQChunk * kQRows + r0;
#pragma unroll
    for (int kk = 0; kk < kQChunk; ++kk) {
      const float4 w = *reinterpret_cast<const float4 *>(ws + kk * H);
      const float4 *row = reinterpret_cast<const float4 *>(xs + kk * kQRows);
#pragma unroll
      for (int r4 = 0; r4 < kQRpt / 4; ++r4) {
        const float4 x = row[r4];
        const float xv[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          acc[0][4 * r4 + j] = __fmaf_rn(xv[j], w.x, acc[0][4 * r4 + j]);
          acc[1][4 * r4 + j] = __fmaf_rn(xv[j], w.y, acc[1][4 * r4 + j]);
          acc[2][4 * r4 + j] = __fmaf_rn(xv[j], w.z, acc[2][4 * r4 + j]);
          acc[3][4 * r4 + j] = __fmaf_rn(xv[j], w.w, acc[3][4 * r4 + j]);
        }
      }
    }
  }
  asm volatile("cp.async.wait_group 0;" ::: "memory");
#pragma unroll
  for (int c = 0; c < kQCols; ++c)
#pragma unroll
    for (int r = 0; r < kQRpt; ++r) {
      float v = acc[c][r];
      if (RELU) v = v > 0.0f ? v : 0.0f;
      out[(n0 + c) * kQRows + r0 + r] = v;
    }
}

__global__ void __launch_bounds__(256) qnet_kernel(const QArgs a) {      // H / kQCols * (32 / kQRpt) = H threads
  extern __shared__ __align__(16) float qsm[];
  const int H = (int)a.H, A = (int)a.A;
  float *x = qsm;                               // [64][32]
  float *h1 = x + MIG_STATE_DIM * kQRows;       // [H][32]
  float *h2 = h1 + H * kQRows;                  // [H][32]
  float *qo = h2 + H * kQRows;                  // [A][32]
  float4 *stage = reinterpret_cast<float4 *>(qo + ((A * kQRows + 3) & ~3));   // [kQStages][kQChunk * H / 4]
  const int tid = threadIdx.x;
  const uint32_t row0 = blockIdx.x * kQRows;
  for (int i = tid; i < MIG_STATE_DIM * kQRows; i += blockDim.x) {   // coalesced read of [row][k], transposed store
    int r = i / MIG_STATE_DIM, k = i % MIG_STATE_DIM;
    uint32_t row = row0 + r;
    x[k * kQRows + r] = row < a.B ? a.state[(size_t)row * MIG_STATE_DIM + k] : 0.0f;
  }
  __syncthreads();
  q_layer<true>(a.W1, a.b1, MIG_STATE_DIM, H, x, h1, stage, tid);
  __syncthreads();
  q_layer<true>(a.W2, a.b2, H, H, h1, h2, stage, tid);
  __syncthreads();
  for (int o = tid; o < A * kQRows; o += blockDim.x) {                // output layer: (n, row) pairs
    int n = o / kQRows, r = o % kQRows;
    float acc = a.b3[n];
    for (int k = 0; k < H; ++k) acc = __fmaf_rn(h2[k * kQRows + r], __ldg(&a.W3[(size_t)k * A + n]), acc);
    qo[n * kQRows + r] = acc;
  }
  __syncthreads();
  if (a.q_out)
    for (int o = tid; o < A * kQRows; o += blockDim.x) {
      int r = o / A, n = o % A;
      if (row0 + r < a.B) a.q_out[(size_t)(row0 + r) * A + n] = qo[n * kQRows + r];
    }
  if (tid < kQRows && row0 + tid < a.B) {
    const uint32_t row = row0 + tid;
    int best = 0; float bv = qo[tid];
    for (int n = 1; n < A; ++n) { float v = qo[n * kQRows + tid]; if (v > bv) { bv = v; best = n; } }   // lowest index on ties
    if (a.argmax_out) a.argmax_out[row] = (uint8_t)best;
    if (a.action_out) {
      uint4 w = philox4x32_10(a.epoch, 2u, a.env_base + row, a.episode, a.k0, a.k1);
      bool explore = w.x < a.eps_thr;
      a.action_out[row] = explore ? (uint8_t)(((unsigned long long)w.y * (unsigned long long)A) >> 32) : (uint8_t)best;
    }
  }
}

}  // namespace migsim
