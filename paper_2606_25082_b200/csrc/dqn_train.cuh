// dqn_train.cuh -- the small kernels around the tensor-core products of the DQN training step (dqn_gemm.cuh): replay
// sampling + gather (+ the transposed copy of the batch), the TD error, bias gradients, the SGD update that also keeps the
// transposed copies of the weights.  PAPER.md:L208, L214; readings #33-#36.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/migsim.h"
#include "philox.cuh"

namespace migsim {

constexpr int kDqnApad = 16;            // the action dimension is padded to 16 columns (UMMA N = 16)

// ---------------------------------------------------------------------------------------------- sampling + gather
// Block = 32 batch rows.  idx_b = (w * size) >> 32 with w = word 0 of Philox(counter (b, 3, step, 0), key seed): stream 3
// (reading #36); with `identity` the batch is rows 0..B-1 of the given arrays.  Writes X[B][64], X2[B][64], a, r, done and,
// if Xt is not NULL, the transposed copy Xt[64][B] (through shared memory: both the reads and the writes are coalesced).
struct GatherArgs {
  const float *S, *S2; const uint8_t *A; const float *R; const uint8_t *D;     // the replay buffer (or an explicit batch)
  float *X, *X2, *Xt; uint8_t *a; float *r; uint8_t *done;
  uint32_t B, size, step, k0, k1; int identity;
};
__global__ void __launch_bounds__(256) dqn_gather_kernel(const GatherArgs g) {
  __shared__ float tile[32][MIG_STATE_DIM + 1];
  __shared__ uint32_t idx[32];
  const uint32_t b0 = blockIdx.x * 32u;
  if (threadIdx.x < 32) {
    const uint32_t b = b0 + threadIdx.x;
    uint32_t i = b;
    if (!g.identity) i = __umulhi(philox4x32_10(b, 3u, g.step, 0u, g.k0, g.k1).x, g.size);
    idx[threadIdx.x] = i;
    if (b < g.B) { g.a[b] = g.A[i]; g.r[b] = g.R[i]; g.done[b] = g.D ? g.D[i] : (uint8_t)0; }
  }
  __syncthreads();
  for (int e = threadIdx.x; e < 32 * MIG_STATE_DIM; e += 256) {
    const int row = e / MIG_STATE_DIM, k = e % MIG_STATE_DIM;
    const uint32_t b = b0 + row;
    if (b >= g.B) continue;
    const float v = g.S[(size_t)idx[row] * MIG_STATE_DIM + k];
    tile[row][k] = v;
    g.X[(size_t)b * MIG_STATE_DIM + k] = v;
    g.X2[(size_t)b * MIG_STATE_DIM + k] = g.S2[(size_t)idx[row] * MIG_STATE_DIM + k];
  }
  __syncthreads();
  if (!g.Xt) return;                                        // (the transposed copy is only read by the K-major weight-gradient path)
  for (int e = threadIdx.x; e < 32 * MIG_STATE_DIM; e += 256) {
    const int k = e / 32, row = e % 32;
    if (b0 + row < g.B) g.Xt[(size_t)k * g.B + b0 + row] = tile[row][k];
  }
}

// ---------------------------------------------------------------------------------------------- TD error
// y_b = r_b + gamma (1 - done_b) max_a' Q_target(s'_b, a');  delta_b = Q(s_b, a_b) - y_b;  dL/dQ[b][j] = (j == a_b) delta_b / B;
// lossrow[b] = delta_b^2 / (2B).  dQ is written row-major [B][ldq] (16 live columns; the caller keeps the others zero) and
// transposed [16][B].
__global__ void __launch_bounds__(256) dqn_td_kernel(const float *Q, const float *Qt, const uint8_t *a, const float *r, const uint8_t *done,
                                                     uint32_t B, uint32_t n_actions, float gamma, float *dQ, uint32_t ldq, float *dQt, float *lossrow) {
  const uint32_t b = blockIdx.x * 256u + threadIdx.x;
  if (b >= B) return;
  const float4 *q4 = reinterpret_cast<const float4 *>(Q + (size_t)b * kDqnApad), *t4 = reinterpret_cast<const float4 *>(Qt + (size_t)b * kDqnApad);
  float q[kDqnApad], t[kDqnApad];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const float4 x = q4[i], y = t4[i];
    q[4 * i] = x.x; q[4 * i + 1] = x.y; q[4 * i + 2] = x.z; q[4 * i + 3] = x.w;
    t[4 * i] = y.x; t[4 * i + 1] = y.y; t[4 * i + 2] = y.z; t[4 * i + 3] = y.w;
  }
  float mx = t[0];
  for (uint32_t j = 1; j < n_actions; ++j) mx = fmaxf(mx, t[j]);
  const uint32_t ab = a[b];
  float qa = 0.0f;
#pragma unroll
  for (int j = 0; j < kDqnApad; ++j) qa = (uint32_t)j == ab ? q[j] : qa;
  const float y = done[b] ? r[b] : fmaf(gamma, mx, r[b]);
  const float delta = qa - y, gq = delta / (float)B;
  lossrow[b] = delta * delta / (2.0f * (float)B);
  float4 *o4 = reinterpret_cast<float4 *>(dQ + (size_t)b * ldq);
#pragma unroll
  for (int i = 0; i < 4; ++i)
    o4[i] = make_float4(4 * i == (int)ab ? gq : 0.0f, 4 * i + 1 == (int)ab ? gq : 0.0f, 4 * i + 2 == (int)ab ? gq : 0.0f, 4 * i + 3 == (int)ab ? gq : 0.0f);
#pragma unroll
  for (int j = 0; j < kDqnApad; ++j) dQt[(size_t)j * B + b] = (uint32_t)j == ab ? gq : 0.0f;
}

// ---------------------------------------------------------------------------------------------- SGD update
// One block per row `i` of a weight matrix W [rows][cols] (cols <= 256): W[i][:] -= lr * sum_z partial[z][i][:], in the fixed
// order z = 0, 1, ...; the transposed copy Wt[cols][ldt] is kept in step.  Blocks beyond `rows` update the bias: bias[o] -= lr *
// sum_b dZt[o][b] (one block per output o, a fixed-order tree over the batch), block `rows + n_bias` sums the loss.
// The products read the weights as TF32 pairs (dqn_gemm.cuh): the copies are kept SPLIT, high parts first -- Wt [2 cols][ldt]
// (transposed: rows [0, cols) high, [cols, 2 cols) low) and, where the backward pass reads the matrix untransposed, Ws [2 rows][ldw].
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xFFFFE000u); }
struct UpdateArgs {
  float *W, *Wt, *Ws; uint32_t rows, cols, ldw, ldt;       // W [rows][ldw] (first `cols` columns live), Wt [2 cols][ldt], Ws [2 rows][ldw] or NULL
  const float *partial; uint32_t n_splits; size_t split_stride; uint32_t ldp;   // partial [z][rows][ldp]
  float *bias; const float *dZt; uint32_t n_bias, B;       // bias [n_bias], dZt [n_bias][B]
  const float *bias_part; uint32_t n_chunks;               // or (dZt == NULL) column sums of the row-major dZ: bias_part [n_chunks][n_bias]
  float lr;
  const float *lossrow; float *loss_out;                   // (only the launch that passes them sums the loss)
};
__device__ __forceinline__ float block_sum_256(float v, float *red) {
#pragma unroll
  for (int d = 16; d; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
  __syncthreads();
  float s = 0.0f;
  if (threadIdx.x == 0) for (int w = 0; w < 8; ++w) s += red[w];
  __syncthreads();
  return s;                                                 // valid in thread 0
}
// (one launch updates the three layers: blocks [first[l], first[l + 1]) run layer l's update)
struct UpdateArgs3 { UpdateArgs l[3]; uint32_t first[4]; };
__device__ __forceinline__ void dqn_update_block(const UpdateArgs &u, const uint32_t blk, float *red) {
  if (blk < u.rows) {
    for (uint32_t c = threadIdx.x; c < u.cols; c += 256) {
      float g = 0.0f;
      for (uint32_t z = 0; z < u.n_splits; ++z) g += u.partial[z * u.split_stride + (size_t)blk * u.ldp + c];
      const float w = u.W[(size_t)blk * u.ldw + c] - u.lr * g;
      u.W[(size_t)blk * u.ldw + c] = w;
      const float h = tf32_hi(w), l = w - h;
      u.Wt[(size_t)c * u.ldt + blk] = h; u.Wt[(size_t)(u.cols + c) * u.ldt + blk] = l;
      if (u.Ws) { u.Ws[(size_t)blk * u.ldw + c] = h; u.Ws[(size_t)(u.rows + blk) * u.ldw + c] = l; }
    }
    return;
  }
  if (blk < u.rows + u.n_bias) {
    const uint32_t o = blk - u.rows;
    if (u.bias_part) {                                        // partial column sums (dqn_colsum_kernel), added in the fixed order z = 0, 1, ...
      if (threadIdx.x == 0) {
        float s = 0.0f;
        for (uint32_t z = 0; z < u.n_chunks; ++z) s += u.bias_part[(size_t)z * u.n_bias + o];
        u.bias[o] -= u.lr * s;
      }
      return;
    }
    float acc = 0.0f;
    for (uint32_t b = threadIdx.x; b < u.B; b += 256) acc += u.dZt[(size_t)o * u.B + b];
    const float s = block_sum_256(acc, red);
    if (threadIdx.x == 0) u.bias[o] -= u.lr * s;
    return;
  }
  if (u.loss_out) {
    float acc = 0.0f;
    for (uint32_t b = threadIdx.x; b < u.B; b += 256) acc += u.lossrow[b];
    const float s = block_sum_256(acc, red);
    if (threadIdx.x == 0) *u.loss_out = s;
  }
}
__global__ void __launch_bounds__(256) dqn_update_kernel(const UpdateArgs3 a) {
  __shared__ float red[8];
  const uint32_t b = blockIdx.x;
  const int l = b >= a.first[2] ? 2 : (b >= a.first[1] ? 1 : 0);   // (block-uniform)
  dqn_update_block(a.l[l], b - a.first[l], red);
}

// Partial column sums of a row-major Z [B][H] (the bias gradients when no transposed copy of dZ exists): block (x, z) sums
// rows [z B / n_chunks, (z + 1) B / n_chunks) of columns [32 x, 32 x + 32) -- a warp reads 128 contiguous bytes of a row, the
// eight warps of the block take every eighth row, their sums are added in warp order: part[z][col].  Fixed order throughout.
// blockIdx.z selects the tensor: one launch sums dZ2 (z = 0, into part0) and dZ1 (z = 1, into part1).
__global__ void __launch_bounds__(256) dqn_colsum_kernel(const float *Z0, const float *Z1, uint32_t B, uint32_t H, uint32_t n_chunks, float *part0, float *part1) {
  __shared__ float red[8][32];
  const float *Z = blockIdx.z ? Z1 : Z0; float *part = blockIdx.z ? part1 : part0;
  const uint32_t lane = threadIdx.x & 31u, w = threadIdx.x >> 5, col = blockIdx.x * 32u + lane, z = blockIdx.y;
  const uint32_t r0 = (uint32_t)(((uint64_t)z * B) / n_chunks), r1 = (uint32_t)(((uint64_t)(z + 1) * B) / n_chunks);
  float acc = 0.0f;
  for (uint32_t r = r0 + w; r < r1; r += 8u) acc += Z[(size_t)r * H + col];
  red[w][lane] = acc;
  __syncthreads();
  if (w == 0) {
    float s = 0.0f;
#pragma unroll
    for (int i = 0; i < 8; ++i) s += red[i][lane];
    part[(size_t)z * H + col] = s;
  }
}

// the split copies of a small matrix W [rows][ldw] (initialisation): Wt [2 cols][ldt] transposed, Ws [2 rows][ldw] (or NULL)
__global__ void dqn_split_kernel(const float *W, float *Wt, float *Ws, uint32_t rows, uint32_t cols, uint32_t ldw, uint32_t ldt) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows * cols) return;
  const uint32_t r = i / cols, c = i % cols;
  const float w = W[(size_t)r * ldw + c], h = tf32_hi(w), l = w - h;
  Wt[(size_t)c * ldt + r] = h; Wt[(size_t)(cols + c) * ldt + r] = l;
  if (Ws) { Ws[(size_t)r * ldw + c] = h; Ws[(size_t)(rows + r) * ldw + c] = l; }
}

}  // namespace migsim
