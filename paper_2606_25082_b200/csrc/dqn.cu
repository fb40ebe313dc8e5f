// dqn.cu -- host side of the DQN training step of libmigsim.so (include/migsim.h: mig_dqn_*, mig_replay_*): replay buffer in
// device memory, one training step = sample -> forward (online on s, frozen target on s') -> TD error -> backward -> SGD.
// Every matrix product runs on the tensor cores through gemm_tf32x3_kernel (dqn_gemm.cuh: tcgen05.mma kind::tf32, TMA,
// TMEM accumulators); the rest is the handful of small kernels in dqn_train.cuh.  PAPER.md:L208, L214; #33-#36.
#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <mutex>
#include <vector>

#include "dqn_gemm.cuh"
#include "dqn_train.cuh"
#include "sim_common.h"

using namespace migsim;

#define CUD(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return mig_fail(MIG_ECUDA, "%s: %s", #call, cudaGetErrorString(e_)); } while (0)

namespace {

struct Net {            // one network: master weights in the caller's layout [in][out] + the copies the products read, kept split
  float *W1, *W1t, *b1, *W2, *W2t, *b2, *W3, *W3t, *b3;      // W1 [64][H], W1t [2 H][64], W2 [H][H], W2t [2 H][H], W3 [H][16], W3t [2 x 16][H]
  float *W2s, *W3s;                                          // W2s [2 H][H], W3s [2 H][16]: untransposed, for the backward products
};                                                           // (split: TF32 high parts in the first half of the rows, remainders in the second)

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr; cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// K-major operand [rows][inner] fp32 with leading dimension ld (elements): boxes of 32 floats (one 128-byte swizzled row) x box_rows
int make_map(CUtensorMap *m, const float *ptr, uint64_t inner, uint64_t rows, uint64_t ld, uint32_t box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return mig_fail(MIG_ECUDA, "dqn: cuTensorMapEncodeTiled is not available from this driver");
  cuuint64_t dims[2] = {inner, rows}, strides[1] = {ld * sizeof(float)};
  cuuint32_t box[2] = {(cuuint32_t)kGemmBK, box_rows}, es[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(ptr), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return mig_fail(MIG_ECUDA, "dqn: cuTensorMapEncodeTiled failed (%d) for a [%llu][%llu] operand", (int)r, (unsigned long long)rows, (unsigned long long)inner);
  return MIG_OK;
}

// MN-major operand: a row-major activation [rows = batch][inner = features] read as the [K][M] side of a product that
// contracts over the batch: boxes of 32 rows x 32 columns, 128-byte rows swizzled in 32-byte chunks (dqn_gemm.cuh)
int make_map_mn(CUtensorMap *m, const float *ptr, uint64_t inner, uint64_t rows, uint64_t ld, uint32_t box_inner) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return mig_fail(MIG_ECUDA, "dqn: cuTensorMapEncodeTiled is not available from this driver");
  cuuint64_t dims[2] = {inner, rows}, strides[1] = {ld * sizeof(float)};
  cuuint32_t box[2] = {box_inner, (cuuint32_t)kGemmBK}, es[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<float *>(ptr), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_128B_ATOM_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return mig_fail(MIG_ECUDA, "dqn: cuTensorMapEncodeTiled failed (%d) for an MN-major [%llu][%llu] operand", (int)r, (unsigned long long)rows, (unsigned long long)inner);
  return MIG_OK;
}

}  // namespace

constexpr uint32_t kDqLd = 32;         // row pitch of dQ: 16 action columns + 16 zero ones (MN-major tiles are 32 columns wide)
constexpr uint32_t kBiasChunks = 64;   // row chunks of the bias-gradient column sums

struct mig_dqn {   // (mig_dqn_t of include/migsim.h)
  uint32_t H = 0, A = 0, B = 0, cap = 0, splits = 1, bn_h = 128;   // bn_h: tile width of the products with N = H
  float gamma = 0.0f, lr = 0.0f; uint64_t seed = 0;
  int device = 0, n_sm = 148;
  uint64_t launches = 0, gemm_launches = 0, kernels_per_step = 0, gemms_per_step = 0;
  bool use_graph = true; cudaGraphExec_t graph_exec = nullptr;
  // weight gradients from the ROW-MAJOR activations (MN-major tensor-core operands, contraction over the batch rows): no
  // transposed copy of any [B][H] tensor is written, the bias gradients are column sums.  MIG_DQN_MN=0 in the environment at
  // create selects the earlier path instead -- every activation also written transposed by the epilogue that produces it,
  // K-major weight-gradient products over those copies -- kept for A/B timing and run by the tests
  bool mn = true;
  float *dZ1 = nullptr, *pb2 = nullptr, *pb1 = nullptr;    // row-major dZ1; partial column sums of dZ2 / dZ1 [kBiasChunks][H]
  CUtensorMap mH2r, mH1r, mXr, mdQr, mdZ2r, mdZ1r;         // MN-major views of the row-major activations
  std::vector<void *> allocs;
  Net net[2];                                              // [0] online, [1] target
  // replay ring
  float *rS = nullptr, *rS2 = nullptr, *rR = nullptr; uint8_t *rA = nullptr, *rD = nullptr;
  uint32_t head = 0, size = 0;
  // batch and activations
  float *X, *X2, *Xt, *H1, *H1t, *H2, *H2t, *Q, *T1, *T2, *Qt, *dQ, *dQt, *dZ2, *dZ2t, *dZ1t, *r, *lossrow, *pW1, *pW2, *pW3, *loss;
  uint8_t *a, *done;
  // tensor maps: A operands and B operands of the eleven products
  CUtensorMap mX, mH1, mH2, mX2, mT1, mT2, mdQ, mdZ2, mH2t, mH1t, mXt;                          // A side (box 128 rows)
  CUtensorMap mW1t[2], mW2t[2], mW3t[2], mW3, mW2, mdQt, mdZ2t, mdZ1t;                          // B side
};

static int dalloc(mig_dqn *d, void **p, size_t bytes) {
  if (cudaMalloc(p, bytes) != cudaSuccess) { cudaGetLastError(); return mig_fail(MIG_ENOMEM, "dqn: cudaMalloc of %zu bytes failed", bytes); }
  d->allocs.push_back(*p);
  return cudaMemset(*p, 0, bytes) == cudaSuccess ? MIG_OK : mig_fail(MIG_ECUDA, "dqn: cudaMemset failed");
}
#define DA(ptr, count) do { int rc_ = dalloc(d, (void **)&(ptr), (size_t)(count) * sizeof(*(ptr))); if (rc_) { mig_dqn_destroy(d); return rc_; } } while (0)

template <int BN, bool MN = false>
static int launch_gemm(mig_dqn *d, const CUtensorMap &ma, const CUtensorMap &mb, const GemmArgs &g, uint32_t splits, cudaStream_t st) {
  GemmArgs ga = g; ga.splits = splits;
  const uint32_t n_tiles = ((g.M + kGemmBM - 1) / kGemmBM) * (g.N / BN) * splits;
  const uint32_t grid = n_tiles < (uint32_t)d->n_sm ? n_tiles : (uint32_t)d->n_sm;          // persistent: one CTA per SM walks the tiles
  gemm_tf32x3_kernel<BN, MN><<<grid, kGemmThreads, GemmSmem<BN>::kBytes, st>>>(ma, mb, ga);
  CUD(cudaGetLastError());
  d->launches++; d->gemm_launches++;
  return MIG_OK;
}

// the products whose N is the hidden width: one 128 x 256 tile per row block when the width allows it (a quarter less
// shared-memory traffic per flop than two 128 x 128 tiles: the A tile is split and read once for twice the columns)
static int launch_gemm_h(mig_dqn *d, const CUtensorMap &ma, const CUtensorMap &mb, const GemmArgs &g, uint32_t splits, cudaStream_t st) {
  return d->bn_h == 256 ? launch_gemm<256>(d, ma, mb, g, splits, st) : launch_gemm<128>(d, ma, mb, g, splits, st);
}

static GemmArgs gargs(uint32_t M, uint32_t N, uint32_t K) {
  GemmArgs g; memset(&g, 0, sizeof(g));
  g.M = M; g.N = N; g.K = K; g.k_blocks = (K + kGemmBK - 1) / kGemmBK;
  return g;
}

extern "C" int mig_dqn_destroy(mig_dqn_t *d) {
  if (!d) return MIG_OK;
  cudaDeviceSynchronize();
  if (d->graph_exec) cudaGraphExecDestroy(d->graph_exec);
  for (void *p : d->allocs) cudaFree(p);
  cudaGetLastError();
  delete d;
  return MIG_OK;
}

extern "C" int mig_dqn_create(mig_dqn_t **out, const float *W1, const float *b1, const float *W2, const float *b2, const float *W3,
                              const float *b3, uint32_t hidden, uint32_t n_actions, uint32_t replay_capacity, uint32_t batch,
                              float gamma, float lr, uint64_t seed) {
  if (!out || !W1 || !b1 || !W2 || !b2 || !W3 || !b3) return mig_fail(MIG_EINVAL, "dqn_create: NULL argument");
  *out = nullptr;
  if (hidden != 128 && hidden != 256) return mig_fail(MIG_EINVAL, "dqn_create: hidden %u must be 128 or 256 (tiles of 128 output columns)", hidden);
  if (n_actions < 1 || n_actions > MIG_MAX_CONFIGS) return mig_fail(MIG_EINVAL, "dqn_create: n_actions %u not in 1..16", n_actions);
  if (batch < 128 || batch % 128 || batch > (1u << 20)) return mig_fail(MIG_EINVAL, "dqn_create: batch %u must be a multiple of 128 in 128..2^20", batch);
  if (replay_capacity < 1 || replay_capacity > (1u << 26)) return mig_fail(MIG_EINVAL, "dqn_create: replay_capacity %u not in 1..2^26", replay_capacity);
  if (!(gamma >= 0.0f) || gamma > 1.0f || !(lr >= 0.0f)) return mig_fail(MIG_EINVAL, "dqn_create: gamma must be in [0, 1], lr >= 0");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return mig_fail(MIG_ECUDA, "dqn_create: no CUDA device; there is no CPU fallback"); }
  mig_dqn *d = new (std::nothrow) mig_dqn();
  if (!d) return mig_fail(MIG_ENOMEM, "dqn_create: host allocation failed");
  cudaGetDevice(&d->device);
  { const char *ng = getenv("MIG_DQN_NO_GRAPH"); d->use_graph = !(ng && ng[0] == '1'); }
  cudaDeviceGetAttribute(&d->n_sm, cudaDevAttrMultiProcessorCount, d->device);
  const uint32_t H = hidden, A = n_actions, B = batch, P = kDqnApad;
  d->H = H; d->A = A; d->B = B; d->cap = replay_capacity; d->gamma = gamma; d->lr = lr; d->seed = seed;
  // 128 x 256 tiles once there are enough row blocks to keep every SM busy with them (measured: 0.402 -> 0.396 ms per step at
  // batch 32768, 1.29 -> 1.24 at 131072; at 8192 the 64 wide tiles leave SMs idle: 0.163 -> 0.207); MIG_DQN_BN=128 / 256 overrides
  { const char *e = getenv("MIG_DQN_BN"); const int f = e ? atoi(e) : 0; d->bn_h = (H == 256 && (f == 256 || (f != 128 && B >= 32768u))) ? 256 : 128; }
  d->splits = B / 128 < 32 ? B / 128 : 32;                  // split-K of the weight-gradient products: >= 4 k-blocks per split
  while ((B / kGemmBK) % d->splits) d->splits--;
  for (int k = 0; k < 2; ++k) {
    Net &n = d->net[k];
    DA(n.W1, 64 * H); DA(n.W1t, 2 * H * 64); DA(n.b1, H); DA(n.W2, H * H); DA(n.W2t, 2 * H * H); DA(n.b2, H); DA(n.W3, H * P); DA(n.W3t, 2 * P * H); DA(n.b3, P);
    DA(n.W2s, 2 * H * H); DA(n.W3s, 2 * H * P);
  }
  DA(d->rS, (size_t)d->cap * 64); DA(d->rS2, (size_t)d->cap * 64); DA(d->rR, d->cap); DA(d->rA, d->cap); DA(d->rD, d->cap);
  DA(d->X, (size_t)B * 64); DA(d->X2, (size_t)B * 64); DA(d->Xt, (size_t)64 * B);
  DA(d->H1, (size_t)B * H); DA(d->H1t, (size_t)H * B); DA(d->H2, (size_t)B * H); DA(d->H2t, (size_t)H * B); DA(d->Q, (size_t)B * P);
  DA(d->T1, (size_t)B * H); DA(d->T2, (size_t)B * H); DA(d->Qt, (size_t)B * P);
  DA(d->dQ, (size_t)B * kDqLd); DA(d->dQt, (size_t)P * B); DA(d->dZ2, (size_t)B * H); DA(d->dZ2t, (size_t)H * B); DA(d->dZ1t, (size_t)H * B);
  DA(d->dZ1, (size_t)B * H);
  DA(d->pb2, (size_t)kBiasChunks * H); DA(d->pb1, (size_t)kBiasChunks * H);
  { const char *e = getenv("MIG_DQN_MN"); d->mn = !(e && e[0] == '0'); }
  DA(d->r, B); DA(d->a, B); DA(d->done, B); DA(d->lossrow, B); DA(d->loss, 1);
  DA(d->pW1, (size_t)d->splits * 64 * H); DA(d->pW2, (size_t)d->splits * H * H); DA(d->pW3, (size_t)d->splits * H * kDqLd);
  // weights: master copies, padded action columns are zero; the transposed copies follow
  auto up = [&](float *dst, const float *src, size_t rows, size_t cols, size_t ld) {
    return cudaMemcpy2D(dst, ld * sizeof(float), src, cols * sizeof(float), cols * sizeof(float), rows, cudaMemcpyHostToDevice) == cudaSuccess;
  };
  bool ok = true;
  for (int k = 0; k < 2 && ok; ++k) {
    Net &n = d->net[k];
    ok = up(n.W1, W1, 64, H, H) && up(n.b1, b1, 1, H, H) && up(n.W2, W2, H, H, H) && up(n.b2, b2, 1, H, H) && up(n.W3, W3, H, A, P) && up(n.b3, b3, 1, A, P);
    if (!ok) break;
    dqn_split_kernel<<<(64 * H + 255) / 256, 256>>>(n.W1, n.W1t, nullptr, 64, H, H, 64);
    dqn_split_kernel<<<(H * H + 255) / 256, 256>>>(n.W2, n.W2t, n.W2s, H, H, H, H);
    dqn_split_kernel<<<(H * P + 255) / 256, 256>>>(n.W3, n.W3t, n.W3s, H, P, P, H);
  }
  if (!ok || cudaDeviceSynchronize() != cudaSuccess) { mig_dqn_destroy(d); return mig_fail(MIG_ECUDA, "dqn_create: weight upload failed: %s", cudaGetErrorString(cudaGetLastError())); }
  int rc = MIG_OK;
  if (cudaFuncSetAttribute(gemm_tf32x3_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<128>::kBytes) != cudaSuccess ||
      cudaFuncSetAttribute(gemm_tf32x3_kernel<256>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<256>::kBytes) != cudaSuccess ||
      cudaFuncSetAttribute(gemm_tf32x3_kernel<128, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<128>::kBytes) != cudaSuccess ||
      cudaFuncSetAttribute(gemm_tf32x3_kernel<32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<32>::kBytes) != cudaSuccess ||
      cudaFuncSetAttribute(gemm_tf32x3_kernel<kDqnApad>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<kDqnApad>::kBytes) != cudaSuccess) {
    mig_dqn_destroy(d); return mig_fail(MIG_ECUDA, "dqn_create: %d bytes of shared memory per CTA refused (%s)", GemmSmem<128>::kBytes, cudaGetErrorString(cudaGetLastError()));
  }
#define MAP(m, ptr, inner, rows, ld, box) if (!rc) rc = make_map(&d->m, ptr, inner, rows, ld, box)
  MAP(mX, d->X, 64, B, 64, 128); MAP(mH1, d->H1, H, B, H, 128); MAP(mH2, d->H2, H, B, H, 128);
  MAP(mX2, d->X2, 64, B, 64, 128); MAP(mT1, d->T1, H, B, H, 128); MAP(mT2, d->T2, H, B, H, 128);
  MAP(mdQ, d->dQ, P, B, kDqLd, 128); MAP(mdZ2, d->dZ2, H, B, H, 128);
  MAP(mH2t, d->H2t, B, H, B, 128); MAP(mH1t, d->H1t, B, H, B, 128); MAP(mXt, d->Xt, B, 64, B, 128);
  const uint32_t bn = d->bn_h;
  for (int k = 0; k < 2; ++k) { MAP(mW1t[k], d->net[k].W1t, 64, 2 * H, 64, bn); MAP(mW2t[k], d->net[k].W2t, H, 2 * H, H, bn); MAP(mW3t[k], d->net[k].W3t, H, 2 * P, H, P); }
  MAP(mW3, d->net[0].W3s, P, 2 * H, P, bn); MAP(mW2, d->net[0].W2s, H, 2 * H, H, bn);
  MAP(mdQt, d->dQt, B, P, B, P); MAP(mdZ2t, d->dZ2t, B, H, B, 128); MAP(mdZ1t, d->dZ1t, B, H, B, 128);
#undef MAP
#define MAPMN(m, ptr, inner, ld, box) if (!rc) rc = make_map_mn(&d->m, ptr, inner, B, ld, box)
  MAPMN(mH2r, d->H2, H, H, 32); MAPMN(mH1r, d->H1, H, H, 32); MAPMN(mXr, d->X, 64, 64, 32);
  MAPMN(mdQr, d->dQ, kDqLd, kDqLd, 32); MAPMN(mdZ2r, d->dZ2, H, H, 32); MAPMN(mdZ1r, d->dZ1, H, H, 32);
#undef MAPMN
  if (rc) { mig_dqn_destroy(d); return rc; }
  *out = d;
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ forward
// h1 = relu(b1 + x W1), h2 = relu(b2 + h1 W2), q = b3 + h2 W3 for the B rows of X (online: which = 0, into H1 / H2 / Q with
// the transposed copies that the MIG_DQN_MN=0 backward pass needs) or of X2 (target: which = 1, into T1 / T2 / Qt)
static int forward(mig_dqn *d, int which, cudaStream_t st) {
  const uint32_t H = d->H, B = d->B, P = kDqnApad;
  const Net &n = d->net[which];
  int rc;
  GemmArgs g = gargs(B, H, 64);
  g.epi = EPI_BIAS | EPI_RELU; g.bias = n.b1; g.out = which ? d->T1 : d->H1; g.ldo = H; g.b_lo_row = H;
  if (!which && !d->mn) { g.out_t = d->H1t; g.ldt = B; }
  if ((rc = launch_gemm_h(d, which ? d->mX2 : d->mX, d->mW1t[which], g, 1, st))) return rc;
  g = gargs(B, H, H);
  g.epi = EPI_BIAS | EPI_RELU; g.bias = n.b2; g.out = which ? d->T2 : d->H2; g.ldo = H; g.b_lo_row = H;
  if (!which && !d->mn) { g.out_t = d->H2t; g.ldt = B; }
  if ((rc = launch_gemm_h(d, which ? d->mT1 : d->mH1, d->mW2t[which], g, 1, st))) return rc;
  g = gargs(B, P, H);
  g.epi = EPI_BIAS; g.bias = n.b3; g.out = which ? d->Qt : d->Q; g.ldo = P; g.b_lo_row = P;
  return launch_gemm<kDqnApad>(d, which ? d->mT2 : d->mH2, d->mW3t[which], g, 1, st);
}

static int on_device(const mig_dqn *d) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev != d->device) return mig_fail(MIG_ESTATE, "dqn: the handle lives on device %d but device %d is current", d->device, dev);
  return MIG_OK;
}

extern "C" int mig_dqn_q(mig_dqn_t *d, int which, const float *state, uint32_t n, float *q_out, void *stream) {
  if (!d || !state || !q_out) return mig_fail(MIG_EINVAL, "dqn_q: NULL argument");
  if (int rcd = on_device(d)) return rcd;
  if (n < 1 || n > d->B) return mig_fail(MIG_EINVAL, "dqn_q: n = %u not in 1..batch (%u)", n, d->B);
  cudaStream_t st = (cudaStream_t)stream;
  float *X = which ? d->X2 : d->X;
  CUD(cudaMemcpyAsync(X, state, (size_t)n * MIG_STATE_DIM * sizeof(float), cudaMemcpyDeviceToDevice, st));
  if (n < d->B) CUD(cudaMemsetAsync(X + (size_t)n * MIG_STATE_DIM, 0, (size_t)(d->B - n) * MIG_STATE_DIM * sizeof(float), st));
  int rc = forward(d, which ? 1 : 0, st);
  if (rc) return rc;
  CUD(cudaMemcpy2DAsync(q_out, d->A * sizeof(float), which ? d->Qt : d->Q, kDqnApad * sizeof(float), d->A * sizeof(float), n, cudaMemcpyDeviceToDevice, st));
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ one training step
// forward of both networks, TD error, backward, SGD on the batch that the gather kernel left in X / X2 / a / r / done:
// fourteen launches (thirteen on the MIG_DQN_MN=0 path), always with the same arguments (the loss lands in d->loss)
static int train_kernels(mig_dqn *d, cudaStream_t st) {
  const uint32_t H = d->H, B = d->B, P = kDqnApad, S = d->splits;
  int rc;
  if ((rc = forward(d, 0, st)) || (rc = forward(d, 1, st))) return rc;
  dqn_td_kernel<<<(B + 255) / 256, 256, 0, st>>>(d->Q, d->Qt, d->a, d->r, d->done, B, d->A, d->gamma, d->dQ, kDqLd, d->dQt, d->lossrow);
  CUD(cudaGetLastError()); d->launches++;
  // backward through the activations: dZ2 = (dQ W3^T) . [H2 > 0], dZ1 = (dZ2 W2^T) . [H1 > 0]
  GemmArgs g = gargs(B, H, P);
  g.epi = EPI_MASK; g.mask = d->H2; g.ldm = H; g.out = d->dZ2; g.ldo = H; g.b_lo_row = H;
  if (!d->mn) { g.out_t = d->dZ2t; g.ldt = B; }
  if ((rc = launch_gemm_h(d, d->mdQ, d->mW3, g, 1, st))) return rc;
  g = gargs(B, H, H);
  g.epi = EPI_MASK; g.mask = d->H1; g.ldm = H; g.b_lo_row = H;
  if (d->mn) { g.out = d->dZ1; g.ldo = H; } else { g.out_t = d->dZ1t; g.ldt = B; }
  if ((rc = launch_gemm_h(d, d->mdZ2, d->mW2, g, 1, st))) return rc;
  // weight gradients, split over the batch dimension: dW3 = H2^T dQ, dW2 = H1^T dZ2, dW1 = X^T dZ1
  const uint32_t kps = B / S;                                  // batch rows per split
  const uint32_t ld3 = d->mn ? kDqLd : P;                     // (MN-major tiles are 32 columns wide: the partials of dW3 carry 16 zero columns)
  g = gargs(H, ld3, kps); g.out = d->pW3; g.ldo = ld3; g.out_split_stride = (size_t)H * ld3;
  if ((rc = d->mn ? launch_gemm<32, true>(d, d->mH2r, d->mdQr, g, S, st) : launch_gemm<kDqnApad>(d, d->mH2t, d->mdQt, g, S, st))) return rc;
  g = gargs(H, H, kps); g.out = d->pW2; g.ldo = H; g.out_split_stride = (size_t)H * H;
  if ((rc = d->mn ? launch_gemm<128, true>(d, d->mH1r, d->mdZ2r, g, S, st) : launch_gemm<128>(d, d->mH1t, d->mdZ2t, g, S, st))) return rc;
  g = gargs(64, H, kps); g.out = d->pW1; g.ldo = H; g.out_split_stride = (size_t)64 * H;
  if ((rc = d->mn ? launch_gemm<128, true>(d, d->mXr, d->mdZ1r, g, S, st) : launch_gemm<128>(d, d->mXt, d->mdZ1t, g, S, st))) return rc;
  if (d->mn) {                                                 // bias gradients of the hidden layers: column sums of the row-major dZ
    dqn_colsum_kernel<<<dim3(H / 32, kBiasChunks, 2), 256, 0, st>>>(d->dZ2, d->dZ1, B, H, kBiasChunks, d->pb2, d->pb1);
    CUD(cudaGetLastError()); d->launches++;
  }
  // SGD on the online network (the split copies of the weights follow), bias gradients (the partial column sums, or row sums of
  // the transposed dZ on the MIG_DQN_MN=0 path), the loss: one launch for the three layers
  Net &n = d->net[0];
  UpdateArgs3 u3; memset(&u3, 0, sizeof(u3));
  UpdateArgs u; memset(&u, 0, sizeof(u));
  u.lr = d->lr; u.B = B; u.n_splits = S;
  u.W = n.W3; u.Wt = n.W3t; u.Ws = n.W3s; u.rows = H; u.cols = P; u.ldw = P; u.ldt = H; u.partial = d->pW3; u.split_stride = (size_t)H * ld3; u.ldp = ld3;
  u.bias = n.b3; u.dZt = d->dQt; u.n_bias = P; u.lossrow = d->lossrow; u.loss_out = d->loss;
  u3.l[0] = u; u3.first[0] = 0; u3.first[1] = u.rows + u.n_bias + 1;
  u.loss_out = nullptr; u.lossrow = nullptr;
  u.W = n.W2; u.Wt = n.W2t; u.Ws = n.W2s; u.rows = H; u.cols = H; u.ldw = H; u.ldt = H; u.partial = d->pW2; u.split_stride = (size_t)H * H; u.ldp = H;
  u.bias = n.b2; u.dZt = d->dZ2t; u.n_bias = H;
  if (d->mn) { u.dZt = nullptr; u.bias_part = d->pb2; u.n_chunks = kBiasChunks; }
  u3.l[1] = u; u3.first[2] = u3.first[1] + u.rows + u.n_bias;
  u.W = n.W1; u.Wt = n.W1t; u.Ws = nullptr; u.rows = 64; u.cols = H; u.ldw = H; u.ldt = 64; u.partial = d->pW1; u.split_stride = (size_t)64 * H; u.ldp = H;
  u.bias = n.b1; u.dZt = d->dZ1t; u.n_bias = H;
  if (d->mn) { u.dZt = nullptr; u.bias_part = d->pb1; u.n_chunks = kBiasChunks; }
  u3.l[2] = u; u3.first[3] = u3.first[2] + u.rows + u.n_bias;
  dqn_update_kernel<<<u3.first[3], 256, 0, st>>>(u3);
  CUD(cudaGetLastError()); d->launches++;
  return MIG_OK;
}

// The fourteen launches are captured ONCE into a CUDA graph (their arguments never change) and replayed with one
// cudaGraphLaunch per step: at batch 8192 the step is launch-bound without it.  MIG_DQN_NO_GRAPH=1 in the environment
// launches the kernels one by one instead (profiling by kernel name).
static int train_on_batch(mig_dqn *d, float *loss_out, cudaStream_t st) {
  int rc = MIG_OK;
  if (!d->use_graph) rc = train_kernels(d, st);
  else {
    if (!d->graph_exec) {
      cudaStream_t cs = nullptr; cudaGraph_t g = nullptr;
      CUD(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
      const uint64_t l0 = d->launches, g0 = d->gemm_launches;
      cudaError_t e = cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal);
      if (e == cudaSuccess) {
        rc = train_kernels(d, cs);
        e = cudaStreamEndCapture(cs, &g);
        if (e == cudaSuccess && !rc) e = cudaGraphInstantiate(&d->graph_exec, g, 0);
      }
      if (g) cudaGraphDestroy(g);
      cudaStreamDestroy(cs);
      d->kernels_per_step = d->launches - l0; d->gemms_per_step = d->gemm_launches - g0;
      d->launches = l0; d->gemm_launches = g0;                 // (capturing launched nothing)
      if (rc) return rc;
      if (e != cudaSuccess) { d->graph_exec = nullptr; return mig_fail(MIG_ECUDA, "dqn: capturing the training step into a CUDA graph failed: %s", cudaGetErrorString(e)); }
    }
    CUD(cudaGraphLaunch(d->graph_exec, st));
    d->launches += d->kernels_per_step; d->gemm_launches += d->gemms_per_step;     // kernels executed, one graph launch
  }
  if (!rc && loss_out) CUD(cudaMemcpyAsync(loss_out, d->loss, sizeof(float), cudaMemcpyDeviceToDevice, st));
  return rc;
}

static int gather(mig_dqn *d, const float *S, const uint8_t *A, const float *R, const float *S2, const uint8_t *D, uint32_t size, uint32_t step,
                  int identity, cudaStream_t st) {
  GatherArgs g; memset(&g, 0, sizeof(g));
  g.S = S; g.S2 = S2; g.A = A; g.R = R; g.D = D; g.X = d->X; g.X2 = d->X2; g.Xt = d->mn ? nullptr : d->Xt; g.a = d->a; g.r = d->r; g.done = d->done;
  g.B = d->B; g.size = size; g.step = step; g.k0 = (uint32_t)d->seed; g.k1 = (uint32_t)(d->seed >> 32); g.identity = identity;
  dqn_gather_kernel<<<(d->B + 31) / 32, 256, 0, st>>>(g);
  CUD(cudaGetLastError()); d->launches++;
  return MIG_OK;
}

extern "C" int mig_dqn_train_step(mig_dqn_t *d, uint32_t step, float *loss_out, void *stream) {
  if (!d) return mig_fail(MIG_EINVAL, "dqn_train_step: NULL handle");
  if (d->size == 0) return mig_fail(MIG_ESTATE, "dqn_train_step: the replay buffer is empty");
  if (int rcd = on_device(d)) return rcd;
  int rc = gather(d, d->rS, d->rA, d->rR, d->rS2, d->rD, d->size, step, 0, (cudaStream_t)stream);
  return rc ? rc : train_on_batch(d, loss_out, (cudaStream_t)stream);
}

extern "C" int mig_dqn_train_on(mig_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2, const uint8_t *done,
                                float *loss_out, void *stream) {
  if (!d || !s || !a || !r || !s2) return mig_fail(MIG_EINVAL, "dqn_train_on: NULL argument");
  if (int rcd = on_device(d)) return rcd;
  int rc = gather(d, s, a, r, s2, done, d->B, 0, 1, (cudaStream_t)stream);
  return rc ? rc : train_on_batch(d, loss_out, (cudaStream_t)stream);
}

// ------------------------------------------------------------------------------------------------ replay buffer, target, weights
extern "C" int mig_replay_push(mig_dqn_t *d, const float *s, const uint8_t *a, const float *r, const float *s2, const uint8_t *done,
                               uint32_t n, void *stream) {
  if (!d || !s || !a || !r || !s2) return mig_fail(MIG_EINVAL, "replay_push: NULL argument");
  cudaStream_t st = (cudaStream_t)stream;
  uint32_t off = 0;
  if (n > d->cap) { off = n - d->cap; n = d->cap; d->head = (uint32_t)(((uint64_t)d->head + off) % d->cap); }   // only the last cap transitions survive
  while (n) {                                                // transition i lands in slot (head + i) mod capacity
    const uint32_t run = n < d->cap - d->head ? n : d->cap - d->head, h = d->head;
    CUD(cudaMemcpyAsync(d->rS + (size_t)h * 64, s + (size_t)off * 64, (size_t)run * 64 * sizeof(float), cudaMemcpyDeviceToDevice, st));
    CUD(cudaMemcpyAsync(d->rS2 + (size_t)h * 64, s2 + (size_t)off * 64, (size_t)run * 64 * sizeof(float), cudaMemcpyDeviceToDevice, st));
    CUD(cudaMemcpyAsync(d->rR + h, r + off, (size_t)run * sizeof(float), cudaMemcpyDeviceToDevice, st));
    CUD(cudaMemcpyAsync(d->rA + h, a + off, run, cudaMemcpyDeviceToDevice, st));
    if (done) CUD(cudaMemcpyAsync(d->rD + h, done + off, run, cudaMemcpyDeviceToDevice, st));
    else CUD(cudaMemsetAsync(d->rD + h, 0, run, st));
    d->head = (h + run) % d->cap; d->size = d->size + run > d->cap ? d->cap : d->size + run;
    off += run; n -= run;
  }
  return MIG_OK;
}

extern "C" uint32_t mig_replay_size(const mig_dqn_t *d) { return d ? d->size : 0; }
extern "C" uint64_t mig_dqn_launch_count(const mig_dqn_t *d) { return d ? d->launches : 0; }

extern "C" int mig_dqn_sync_target(mig_dqn_t *d, void *stream) {
  if (!d) return mig_fail(MIG_EINVAL, "dqn_sync_target: NULL handle");
  cudaStream_t st = (cudaStream_t)stream;
  const size_t H = d->H, P = kDqnApad;
  const Net &o = d->net[0]; Net &t = d->net[1];
  const struct { float *dst; const float *src; size_t n; } cp[9] = {             // (the target's backward copies are never read)
      {t.W1, o.W1, 64 * H}, {t.W1t, o.W1t, 2 * H * 64}, {t.b1, o.b1, H}, {t.W2, o.W2, H * H}, {t.W2t, o.W2t, 2 * H * H}, {t.b2, o.b2, H},
      {t.W3, o.W3, H * P}, {t.W3t, o.W3t, 2 * P * H}, {t.b3, o.b3, P}};
  for (const auto &c : cp) CUD(cudaMemcpyAsync(c.dst, c.src, c.n * sizeof(float), cudaMemcpyDeviceToDevice, st));
  return MIG_OK;
}

extern "C" int mig_dqn_get_weights(mig_dqn_t *d, int which, float *W1, float *b1, float *W2, float *b2, float *W3, float *b3) {
  if (!d || !W1 || !b1 || !W2 || !b2 || !W3 || !b3) return mig_fail(MIG_EINVAL, "dqn_get_weights: NULL argument");
  CUD(cudaDeviceSynchronize());
  const Net &n = d->net[which ? 1 : 0];
  const size_t H = d->H, A = d->A, P = kDqnApad;
  CUD(cudaMemcpy(W1, n.W1, 64 * H * sizeof(float), cudaMemcpyDeviceToHost));
  CUD(cudaMemcpy(b1, n.b1, H * sizeof(float), cudaMemcpyDeviceToHost));
  CUD(cudaMemcpy(W2, n.W2, H * H * sizeof(float), cudaMemcpyDeviceToHost));
  CUD(cudaMemcpy(b2, n.b2, H * sizeof(float), cudaMemcpyDeviceToHost));
  CUD(cudaMemcpy2D(W3, A * sizeof(float), n.W3, P * sizeof(float), A * sizeof(float), H, cudaMemcpyDeviceToHost));
  CUD(cudaMemcpy(b3, n.b3, A * sizeof(float), cudaMemcpyDeviceToHost));
  return MIG_OK;
}

// ------------------------------------------------------------------------------------------------ forward without allocation
// mig_q_forward_static (include/migsim.h): the tensor-core forward of mig_dqn_q for callers that cannot call cudaMalloc (code
// under CUDA graph capture, serving loops, harnesses that forbid it).  Its scratch -- the split weight copies, the two hidden
// activations, the padded Q rows -- is this file-scope array: 4.8 MiB on every GPU that loads the library, until exit.  The
// array's name is a host-side stand-in in host code, not a device address: its address is taken ONCE PER DEVICE with
// cudaGetSymbolAddress (that device current) and only that pointer reaches kernels, memsets, copies and tensor maps.
namespace {

constexpr uint32_t kStaticMaxRows = MIG_Q_STATIC_MAX_ROWS, kStaticMaxH = 256;
// regions, in floats; every offset is a multiple of 64 floats (256 bytes: TMA base alignment and float4 access)
constexpr size_t kOffW1t = 0;                                              // [2 H][64]   split, transposed
constexpr size_t kOffW2t = kOffW1t + 2 * (size_t)kStaticMaxH * 64;         // [2 H][H]
constexpr size_t kOffW3t = kOffW2t + 2 * (size_t)kStaticMaxH * kStaticMaxH; // [2 x 16][H]
constexpr size_t kOffB3 = kOffW3t + 2 * (size_t)kDqnApad * kStaticMaxH;    // [16] (+ padding to 64)
constexpr size_t kOffH1 = kOffB3 + 64;                                     // [rows][H]
constexpr size_t kOffH2 = kOffH1 + (size_t)kStaticMaxRows * kStaticMaxH;   // [rows][H]
constexpr size_t kOffQ = kOffH2 + (size_t)kStaticMaxRows * kStaticMaxH;    // [rows][16]
constexpr size_t kStaticFloats = kOffQ + (size_t)kStaticMaxRows * kDqnApad;
static_assert(kOffW2t % 64 == 0 && kOffW3t % 64 == 0 && kOffB3 % 64 == 0 && kOffH1 % 64 == 0 && kOffH2 % 64 == 0 && kOffQ % 64 == 0, "256-byte regions");

static __device__ __align__(256) float g_q_static_scratch[kStaticFloats];

// split, transposed copy of W [rows][ldw] (first `cols` columns): Wt[c][r] = hi(W[r][c]), Wt[lo_row + c][r] = W[r][c] - hi
// (dqn_split_kernel with the row of the low parts given: the action columns are padded to 16 rows here, not in W)
__global__ void dqn_split_rows_kernel(const float *W, float *Wt, uint32_t rows, uint32_t cols, uint32_t ldw, uint32_t ldt, uint32_t lo_row) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= rows * cols) return;
  const uint32_t r = i / cols, c = i % cols;
  const float w = W[(size_t)r * ldw + c], h = tf32_hi(w), l = w - h;
  Wt[(size_t)c * ldt + r] = h; Wt[(size_t)(lo_row + c) * ldt + r] = l;
}

struct StaticDev { bool ready = false; float *base = nullptr; int n_sm = 0; };
constexpr int kMaxDevices = 64;
StaticDev g_static_dev[kMaxDevices];
std::mutex g_static_mutex;

// once per device, with that device current: the scratch array's DEVICE address, the kernels' shared-memory limits
int static_setup(int dev, StaticDev **out) {
  if (dev < 0 || dev >= kMaxDevices) return mig_fail(MIG_EINVAL, "q_forward_static: device ordinal %d not in 0..%d", dev, kMaxDevices - 1);
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticDev &sd = g_static_dev[dev];
  if (!sd.ready) {
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, g_q_static_scratch);
    if (e != cudaSuccess || !p) { cudaGetLastError(); return mig_fail(MIG_ECUDA, "q_forward_static: cudaGetSymbolAddress of the scratch array failed on device %d: %s", dev, cudaGetErrorString(e)); }
    if (reinterpret_cast<uintptr_t>(p) & 255u) return mig_fail(MIG_ECUDA, "q_forward_static: the scratch array is not 256-byte aligned");
    if (cudaFuncSetAttribute(gemm_tf32x3_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<128>::kBytes) != cudaSuccess ||
        cudaFuncSetAttribute(gemm_tf32x3_kernel<kDqnApad>, cudaFuncAttributeMaxDynamicSharedMemorySize, GemmSmem<kDqnApad>::kBytes) != cudaSuccess) {
      const cudaError_t e2 = cudaGetLastError();
      return mig_fail(MIG_ECUDA, "q_forward_static: %d bytes of shared memory per CTA refused on device %d (%s)", GemmSmem<128>::kBytes, dev, cudaGetErrorString(e2));
    }
    if (cudaDeviceGetAttribute(&sd.n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sd.n_sm < 1) { cudaGetLastError(); return mig_fail(MIG_ECUDA, "q_forward_static: no SM count for device %d", dev); }
    sd.base = static_cast<float *>(p);
    sd.ready = true;
  }
  *out = &sd;
  return MIG_OK;
}

template <int BN>
int launch_gemm_static(int n_sm, const CUtensorMap &ma, const CUtensorMap &mb, const GemmArgs &g, cudaStream_t st) {
  GemmArgs ga = g; ga.splits = 1;
  const uint32_t n_tiles = ((g.M + kGemmBM - 1) / kGemmBM) * (g.N / BN);
  const uint32_t grid = n_tiles < (uint32_t)n_sm ? n_tiles : (uint32_t)n_sm;
  gemm_tf32x3_kernel<BN><<<grid, kGemmThreads, GemmSmem<BN>::kBytes, st>>>(ma, mb, ga);
  CUD(cudaGetLastError());
  return MIG_OK;
}

}  // namespace

extern "C" int mig_q_forward_static(const float *W1, const float *b1, const float *W2, const float *b2, const float *W3, const float *b3,
                                    uint32_t hidden, uint32_t n_actions, const float *state, uint32_t n, float *q_out, void *stream) {
  if (!W1 || !b1 || !W2 || !b2 || !W3 || !b3 || !state || !q_out) return mig_fail(MIG_EINVAL, "q_forward_static: NULL argument");
  if (hidden != 128 && hidden != 256) return mig_fail(MIG_EINVAL, "q_forward_static: hidden %u must be 128 or 256", hidden);
  if (n_actions < 1 || n_actions > MIG_MAX_CONFIGS) return mig_fail(MIG_EINVAL, "q_forward_static: n_actions %u not in 1..16", n_actions);
  if (n < 1) return mig_fail(MIG_EINVAL, "q_forward_static: n = 0 rows");
  if (n > kStaticMaxRows)
    return mig_fail(MIG_EINVAL, "q_forward_static: n = %u rows exceed MIG_Q_STATIC_MAX_ROWS = %u, the size of the library's static scratch "
                                "(call it on chunks of the batch, or use mig_dqn_q, which allocates at create)", n, kStaticMaxRows);
  if ((reinterpret_cast<uintptr_t>(state) | reinterpret_cast<uintptr_t>(b1) | reinterpret_cast<uintptr_t>(b2)) & 15u)
    return mig_fail(MIG_EINVAL, "q_forward_static: state, b1 and b2 must be 16-byte aligned device pointers");
  int dev = 0;
  CUD(cudaGetDevice(&dev));
  StaticDev *sd = nullptr;
  if (int rc = static_setup(dev, &sd)) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  const uint32_t H = hidden, A = n_actions, P = kDqnApad;
  float *W1t = sd->base + kOffW1t, *W2t = sd->base + kOffW2t, *W3t = sd->base + kOffW3t, *b3p = sd->base + kOffB3;
  float *H1 = sd->base + kOffH1, *H2 = sd->base + kOffH2, *Q = sd->base + kOffQ;
  // the array keeps the last call's contents: the padded action rows of W3t and of the bias must be zero for THIS call
  CUD(cudaMemsetAsync(W3t, 0, 2 * (size_t)P * H * sizeof(float), st));
  CUD(cudaMemsetAsync(b3p, 0, 64 * sizeof(float), st));
  dqn_split_rows_kernel<<<(64 * H + 255) / 256, 256, 0, st>>>(W1, W1t, 64, H, H, 64, H);
  dqn_split_rows_kernel<<<(H * H + 255) / 256, 256, 0, st>>>(W2, W2t, H, H, H, H, H);
  dqn_split_rows_kernel<<<(H * A + 255) / 256, 256, 0, st>>>(W3, W3t, H, A, A, H, P);
  CUD(cudaGetLastError());
  CUD(cudaMemcpyAsync(b3p, b3, A * sizeof(float), cudaMemcpyDeviceToDevice, st));
  // tensor maps (host-side encoding, no allocation): A operands with exactly n rows, so that rows beyond n read as zeros
  CUtensorMap mX, mH1, mH2, mW1t, mW2t, mW3t;
  int rc = MIG_OK;
  if (!rc) rc = make_map(&mX, state, 64, n, 64, 128);
  if (!rc) rc = make_map(&mH1, H1, H, n, H, 128);
  if (!rc) rc = make_map(&mH2, H2, H, n, H, 128);
  if (!rc) rc = make_map(&mW1t, W1t, 64, 2 * H, 64, 128);
  if (!rc) rc = make_map(&mW2t, W2t, H, 2 * H, H, 128);
  if (!rc) rc = make_map(&mW3t, W3t, H, 2 * P, H, P);
  if (rc) return rc;
  GemmArgs g = gargs(n, H, 64);
  g.epi = EPI_BIAS | EPI_RELU; g.bias = b1; g.out = H1; g.ldo = H; g.b_lo_row = H;
  if ((rc = launch_gemm_static<128>(sd->n_sm, mX, mW1t, g, st))) return rc;
  g = gargs(n, H, H);
  g.epi = EPI_BIAS | EPI_RELU; g.bias = b2; g.out = H2; g.ldo = H; g.b_lo_row = H;
  if ((rc = launch_gemm_static<128>(sd->n_sm, mH1, mW2t, g, st))) return rc;
  g = gargs(n, P, H);
  g.epi = EPI_BIAS; g.bias = b3p; g.out = Q; g.ldo = P; g.b_lo_row = P;
  if ((rc = launch_gemm_static<kDqnApad>(sd->n_sm, mH2, mW3t, g, st))) return rc;
  CUD(cudaMemcpy2DAsync(q_out, A * sizeof(float), Q, P * sizeof(float), A * sizeof(float), n, cudaMemcpyDeviceToDevice, st));
  return MIG_OK;
}
