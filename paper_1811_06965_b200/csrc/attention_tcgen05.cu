// attention_tcgen05.cu - attention forward / backward on the 5th-generation tensor cores (sm_100a)
// for sequences of at most 256 tokens and d_head = 64 (every bf16 workload of BASELINE.json;
// SURVEY 8(a) a7, a16; K5/K6 of DESIGN.md).
//
// With S <= 256 a whole row of scores fits one TMEM accumulator (128 lanes x 256 fp32 columns), so
// the forward softmax is a plain two-pass row softmax over TMEM: no online rescaling.  All five
// backward products of a head run on tcgen05.mma from 128-byte-swizzled shared-memory tiles that TMA
// fetched where the tensors lie (head h = 64 columns of the [tokens, 3*d_a] qkv matrix; 3-D tensor
// maps [seq][row][col] zero-fill past the end of a sequence).
//
// forward  (one CTA = 128 query rows of one (sequence, head), 8 warps, 2 CTAs / SM):
//   TMA Q, K, V -> S = Q K^T (M 128, N <= 256, K 64) in TMEM -> row max, P = exp2(..) written back into
//   TENSOR MEMORY as packed bf16 pairs (tcgen05.st) over score columns the writing thread has already
//   consumed -> O = P V with the A operand read from TMEM (M 128, N 64, K <= 256; V is the MN-major B
//   operand as it lies) -> O / l and the LSE stored directly.  No shared-memory P panels, no proxy fence.
// backward (one CTA = one (sequence, head), 8 compute warps + 1 control warp, 1 CTA / SM):
//   for key block j, query block i (128 x 128 each):  S = Q_i K_j^T, dP = dO_i V_j^T  (TMEM)
//   -> P = exp2(S - lse), dS = P (dP - D) as bf16 panels in shared memory
//   -> dV_j += P^T dO_i, dK_j += dS^T Q_i (the panels read as MN-major A), dQ_i += dS K_j (K-major A);
//   dV_j, dK_j, dQ_0, dQ_1 stay in TMEM (4 x 64 columns) next to S and dP (2 x 128): 512 columns.
//   The control thread issues S/dP of the next block pair as soon as the compute warps have pulled
//   the current pair into registers, so the tensor pipe works under the exponentials; dV_j / dK_j are
//   read out inside the first pair of the next key block.  Gradients leave through a per-warp
//   shared-memory transposer (coalesced 64-byte row segments).
//   Deterministic: no atomics, fixed accumulation order.
// What bounds them (profiles/attn_r01.md): forward - MUFU.EX2 and the serial load / S / softmax / P V
// chain of a CTA; backward - the panel hand-over between the compute warps and the N = 64 products.
#include <cuda.h>
#include <math.h>

#include <mutex>
#include <unordered_map>

#include "common.cuh"
#include "tcgen05.cuh"

namespace gp {
namespace fat {

using namespace tc;

constexpr int DH = 64;
constexpr uint32_t TILE = 128 * 128;          // bytes of a [128 rows x 64 bf16] swizzled tile
constexpr float LOG2E = 1.4426950408889634f;
#if GP_PROBES
static unsigned long long *g_attn_tl = nullptr;     // host: timeline buffer handed to the next launches
#else
constexpr unsigned long long *g_attn_tl = nullptr;
#endif

__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *map, uint32_t bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(dst), "l"((uint64_t)map), "r"(bar), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}
__device__ __forceinline__ float ex2(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ uint32_t pack2(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&v);
}
// instruction descriptor: D fp32, A / B bf16, majorness (1 = MN-major), N, M = 128
__device__ __forceinline__ uint32_t idesc(int a_mn, int b_mn, int N) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)a_mn << 15) | ((uint32_t)b_mn << 16) |
         ((uint32_t)(N >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
}
// K-major operand tile [rows x 64 k] (8-row atoms 1024 B apart): descriptor of k-step ks (16 k = 32 B)
__device__ __forceinline__ uint64_t desc_k(uint32_t tile, int ks) { return make_smem_desc(tile + ks * 32, 16, 1024); }
// MN-major operand: [k rows x 64 mn] panels (128 B rows), panels TILE bytes apart; k-step = 16 rows
__device__ __forceinline__ uint64_t desc_mn(uint32_t tile, int ks) { return make_smem_desc(tile + ks * 2048, TILE, 1024); }

// one row of a swizzled [128 x 128 B] panel: 16-byte chunk c of row r
__device__ __forceinline__ uint32_t panel_addr(uint32_t panel, int r, int c) {
  return panel + (uint32_t)r * 128u + (uint32_t)((c ^ (r & 7)) << 4);
}

// ---------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------
// One CTA = one (sequence, head): its query blocks of 128 rows one after the other (qpb = 2; qpb = 1: one block per CTA),
// K and V loaded once; the score product of block b + 1 is issued as soon as every thread holds block b's output in
// registers, so the output stores run under it.
// shared memory (from a 1024-byte aligned base): Q_0 [0,16K) | K [16K,48K) | Q_1 [48K,64K) | V [64K,96K).
// TMEM (256 columns): S in [0, N).  The thread pair of a row splits the 32-key chunks [0, split) / [split, nch); P chunk
// c (16 columns of bf16 pairs) goes to column 16 c for the first half and to 32 split + 16 (c - split) for the second:
// always inside score columns its own thread has already read in this pass (chunk c's P lies in chunk <= c of the same
// thread; the next chunk's load, in flight, is never touched).  O accumulates once every thread is done, in 64 columns
// clear of both P regions: [64, 128) when split = 4, else [192, 256).
// 8 warps: warps w and w + 4 own TMEM lane quadrant w & 3 (32 query rows) and split the row's key
// chunks (32 columns each) in two halves; the halves exchange row max and row sum through shared
// memory.  TMEM read bandwidth (S is read twice: max, then exp) bounds the softmax, so each thread
// keeps the next chunk's tcgen05.ld in flight while it works on the current one.
constexpr size_t FWD_SMEM = 96 * 1024 + 1024;
constexpr int FWD_THREADS = 256;

__global__ void __launch_bounds__(FWD_THREADS, 2)
attn_fwd_tc_kernel(const __grid_constant__ CUtensorMap map_qkv, bf16 *__restrict__ o, float *__restrict__ lse, int S,
                   int A, int causal, float scale, int qpb, unsigned long long *tl) {
  extern __shared__ uint8_t smem_raw[];
  // optional timeline probe (attn_tc_set_timeline): 8 %globaltimer stamps per CTA, written by thread 0
  auto stamp = [&](int slot) {
#if GP_PROBES
    if (tl && threadIdx.x == 0) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
      tl[((size_t)blockIdx.y * gridDim.x + blockIdx.x) * 8 + slot] = t;
    }
#else
    (void)slot; (void)tl;
#endif
  };
  stamp(0);
  __shared__ __align__(8) uint64_t bars[5];
  __shared__ uint32_t tmem_base_smem;
  __shared__ float xm[2][128], xl[2][128];
  const uint32_t sb = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = sb, sK = sb + TILE, sV = sb + 4 * TILE;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int quad = warp & 3, chalf = warp >> 2;
  const int da = A * DH, seq = blockIdx.y / A, h = blockIdx.y - seq * A;
  // this CTA's query blocks [qb0, qb1) of 128 rows (qpb per CTA: 1, or 2 = the whole (sequence, head) for S <= 256 with
  // K and V loaded once) and the key tiles the last of them sees
  const int qb0 = blockIdx.x * qpb, qb1 = min((S + 127) >> 7, qb0 + qpb);
  const int nk_all = causal ? min(S, qb1 * 128) : S;
  const int nkb_all = (nk_all + 127) >> 7;
  const uint32_t bar_qk = smem_u32(&bars[0]), bar_v = smem_u32(&bars[1]), bar_s = smem_u32(&bars[2]),
                 bar_o = smem_u32(&bars[3]), bar_q1 = smem_u32(&bars[4]);
  if (threadIdx.x == 0) {
    tma_prefetch_desc(&map_qkv);
    for (int i = 0; i < 5; ++i) mbar_init(bar_qk + 8 * i, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_smem)), "n"(256));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem = tmem_base_smem;

  if (threadIdx.x == 0) {
    mbar_expect_tx(bar_qk, (1 + nkb_all) * TILE);
    tma_load_3d(sQ, &map_qkv, bar_qk, h * DH, qb0 * 128, seq);
    for (int b = 0; b < nkb_all; ++b) tma_load_3d(sK + b * TILE, &map_qkv, bar_qk, da + h * DH, b * 128, seq);
    mbar_expect_tx(bar_v, nkb_all * TILE);
    for (int b = 0; b < nkb_all; ++b) tma_load_3d(sV + b * TILE, &map_qkv, bar_v, 2 * da + h * DH, b * 128, seq);
    if (qb1 - qb0 > 1) {                                 // the second query block: into the 16 KB between K and V
      mbar_expect_tx(bar_q1, TILE);
      tma_load_3d(sb + 3 * TILE, &map_qkv, bar_q1, h * DH, (qb0 + 1) * 128, seq);
    }
  }
  // S = Q_b K^T of query block b into TMEM columns [0, N_b) (thread 0): block qb0 before the loop, block b + 1 as soon as
  // every thread holds block b's output in registers - its global stores then run under the next score product
  auto issue_scores = [&](int b) {
    const int it_ = b - qb0;
    const int nk_ = causal ? min(S, b * 128 + 128) : S;
    mbar_wait(it_ ? bar_q1 : bar_qk, 0, 0x21);
    tcgen05_fence_after();
    const uint32_t id = idesc(0, 0, (nk_ + 15) & ~15);
    const uint32_t sQb = it_ ? sb + 3 * TILE : sQ;
#pragma unroll
    for (int ks = 0; ks < DH / 16; ++ks) umma_bf16(tmem, desc_k(sQb, ks), desc_k(sK, ks), id, ks ? 1u : 0u);
    tcgen05_commit(bar_s);
  };
  if (threadIdx.x == 0) {
    issue_scores(qb0);
    stamp(1);
  }
  __syncwarp();
  for (int qb = qb0; qb < qb1; ++qb) {
  const int it = qb - qb0;
  const uint32_t par = (uint32_t)(it & 1);               // bar_s / bar_o complete once per query block
  const int q0 = qb * 128;
  const int nk = causal ? min(S, q0 + 128) : S;          // keys this block can see
  const int N = (nk + 15) & ~15;                         // MMA N of the score product / K of P V

  // ---- softmax: this thread's row, this half's chunks ----
  const int r_loc = quad * 32 + lane, row = q0 + r_loc;
  const uint32_t t_row = tmem + ((uint32_t)(quad * 32) << 16);
  const float sl2 = scale * LOG2E;
  const int kmax = min(nk - 1, causal ? row : nk - 1);              // last key this row sees
  const int kvis_w = causal ? min(nk, q0 + quad * 32 + 32) : nk;    // keys any row of this warp sees
  const int nch_all = (N + 31) >> 5, split = (nch_all + 1) >> 1;
  const int c0 = chalf ? split : 0, c1 = chalf ? nch_all : split;
  const int cv = min(c1, (kvis_w + 31) >> 5);                        // chunks [c0, cv) hold visible keys
  // chunk c needs per-element masking when it reaches past the first row's diagonal or past nk
  auto edge = [&](int c) { return c * 32 + 32 > nk || (causal && c * 32 + 31 > q0 + quad * 32); };
  mbar_wait(bar_s, par, 0x22);
  tcgen05_fence_after();
  stamp(2);
  uint32_t ra[32], rb[32];
  float mx = -INFINITY;
  auto max_chunk = [&](const uint32_t *r, int c) {
    if (edge(c)) {
#pragma unroll
      for (int j = 0; j < 32; ++j) mx = fmaxf(mx, c * 32 + j <= kmax ? __uint_as_float(r[j]) : -INFINITY);
    } else {
#pragma unroll
      for (int j = 0; j < 32; ++j) mx = fmaxf(mx, __uint_as_float(r[j]));
    }
  };
  if (c0 < cv) tmem_ld32(t_row + c0 * 32, ra);
  for (int c = c0; c < cv; c += 2) {
    tmem_ld_wait();
    if (c + 1 < cv) tmem_ld32(t_row + (c + 1) * 32, rb);
    max_chunk(ra, c);
    if (c + 1 < cv) {
      tmem_ld_wait();
      if (c + 2 < cv) tmem_ld32(t_row + (c + 2) * 32, ra);
      max_chunk(rb, c + 1);
    }
  }
  xm[chalf][r_loc] = mx;
  if (c0 < cv) tmem_ld32(t_row + c0 * 32, ra);           // first chunk of the second pass: in flight over the barrier
  __syncthreads();
  stamp(3);
  mx = fmaxf(xm[0][r_loc], xm[1][r_loc]);                // finite: key 0 is visible to every row
  const float ms = mx * sl2;
  float l = 0.f;
  // where P chunk c lives in tensor memory (see the layout note above)
  auto pcol = [&](int c) { return (uint32_t)(c < split ? c * 16 : 32 * split + (c - split) * 16); };
  const uint32_t ocol = split == 4 ? 64u : 192u;          // 64 output columns clear of both P regions
  auto exp_chunk = [&](const uint32_t *r, int c) {
    float p[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) p[j] = ex2(fmaf(__uint_as_float(r[j]), sl2, -ms));
    if (edge(c)) {
#pragma unroll
      for (int j = 0; j < 32; ++j) p[j] = c * 32 + j <= kmax ? p[j] : 0.f;
    }
#pragma unroll
    for (int j = 0; j < 32; ++j) l += p[j];
    uint32_t pk[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) pk[q] = pack2(p[2 * q], p[2 * q + 1]);
    tmem_st16(t_row + pcol(c), pk);
  };
  for (int c = c0; c < cv; c += 2) {
    tmem_ld_wait();
    if (c + 1 < cv) tmem_ld32(t_row + (c + 1) * 32, rb);
    exp_chunk(ra, c);
    if (c + 1 < cv) {
      tmem_ld_wait();
      if (c + 2 < cv) tmem_ld32(t_row + (c + 2) * 32, ra);
      exp_chunk(rb, c + 1);
    }
  }
  for (int c = max(cv, c0); c < c1; ++c) {                // chunks no row of this warp sees: P = 0
    uint32_t pk[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) pk[q] = 0u;
    tmem_st16(t_row + pcol(c), pk);
  }
  tmem_st_wait();
  xl[chalf][r_loc] = l;
  tcgen05_fence_before();
  __syncthreads();

  stamp(4);
  if (threadIdx.x == 0) {
    tcgen05_fence_after();
    mbar_wait(bar_v, 0, 0x23);
    const uint32_t id = idesc(0, 1, DH);
    // descriptors differ only in their (address >> 4) field: one base each, a constant added per k-step - the
    // N = 64 products retire in ~40 cycles, so the issuing thread must not spend longer than that per MMA
    const uint64_t bV = desc_mn(sV, 0);
    const int nkk = N / 16;
#pragma unroll
    for (int kk = 0; kk < 16; ++kk)                       // 16 keys = 8 columns of P per k-step
      if (kk < nkk) umma_bf16_ts(tmem + ocol, tmem + pcol(kk >> 1) + (kk & 1) * 8, bV + (uint64_t)(kk * 128), id, kk ? 1u : 0u);
    tcgen05_commit(bar_o);
  }
  __syncwarp();
  l = xl[0][r_loc] + xl[1][r_loc];
  mbar_wait(bar_o, par, 0x24);
  tcgen05_fence_after();
  stamp(5);
  tmem_ld32(t_row + ocol + chalf * 32, ra);               // this thread's 32 of the row's 64 output columns
  tmem_ld_wait();
  if (qb + 1 < qb1) {                                    // every thread has read its part of O: the columns are free
    tcgen05_fence_before();
    __syncthreads();
    tcgen05_fence_after();
    if (threadIdx.x == 0) issue_scores(qb + 1);
    __syncwarp();
  }
  if (row < S) {
    const float inv = 1.f / l;
    uint4 *dst = reinterpret_cast<uint4 *>(o + ((int64_t)seq * S + row) * da + h * DH + chalf * 32);
#pragma unroll
    for (int q = 0; q < 4; ++q)
      dst[q] = make_uint4(pack2(__uint_as_float(ra[8 * q]) * inv, __uint_as_float(ra[8 * q + 1]) * inv),
                          pack2(__uint_as_float(ra[8 * q + 2]) * inv, __uint_as_float(ra[8 * q + 3]) * inv),
                          pack2(__uint_as_float(ra[8 * q + 4]) * inv, __uint_as_float(ra[8 * q + 5]) * inv),
                          pack2(__uint_as_float(ra[8 * q + 6]) * inv, __uint_as_float(ra[8 * q + 7]) * inv));
    if (chalf == 0) lse[((int64_t)seq * A + h) * S + row] = mx * scale + logf(l);
  }
  stamp(6);
  }                                                      // qb
  tcgen05_fence_before();
  __syncthreads();
  if (warp == 1) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(256));
  }
}

// ---------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------
// shared memory: Q | K | V | dO (2 tiles each: 128 KB) | P (2 panels) | dS (2 panels)
constexpr size_t BWD_SMEM = 12 * TILE + 1024;
constexpr int BWD_THREADS = 288;
// TMEM columns
constexpr uint32_t C_S = 0, C_DP = 128, C_DV = 256, C_DK = 320, C_DQ = 384;

__global__ void __launch_bounds__(BWD_THREADS, 1)
attn_bwd_tc_kernel(const __grid_constant__ CUtensorMap map_qkv, const __grid_constant__ CUtensorMap map_do,
                   const bf16 *__restrict__ o, const bf16 *__restrict__ d_o, const float *__restrict__ lse,
                   bf16 *__restrict__ dqkv, float *__restrict__ colpart, int S, int A, int causal, float scale,
                   unsigned long long *tl) {
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t bars[5];
  __shared__ float cs_part[8][4][32];    // per-warp column sums of what it stored: [dV|dK cols 0-31, 32-63, dQ cols 0-31, 32-63]
  // optional timeline probe (attn_tc_set_timeline): 32 %globaltimer stamps per CTA
  auto stamp = [&](int slot) {
#if GP_PROBES
    if (tl) {
      unsigned long long t;
      asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
      tl[(size_t)blockIdx.x * 32 + slot] = t;
    }
#else
    (void)slot; (void)tl;
#endif
  };
  __shared__ uint32_t tmem_base_smem;
  __shared__ float Lsm[256], Dsm[256];
  __shared__ __align__(16) uint8_t xpose[8 * 32 * 80];   // per-warp output transposer (store_acc)
  const uint32_t sb = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sQ = sb, sK = sb + 2 * TILE, sV = sb + 4 * TILE, sdO = sb + 6 * TILE, sP = sb + 8 * TILE,
                 sdS = sb + 10 * TILE;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int da = A * DH, seq = blockIdx.x / A, h = blockIdx.x - seq * A;
  const int nblk = (S + 127) >> 7;                       // 1 or 2 blocks of 128 rows
  const uint32_t bar_ld = smem_u32(&bars[0]), bar_sp = smem_u32(&bars[1]), bar_tfree = smem_u32(&bars[2]),
                 bar_pds = smem_u32(&bars[3]), bar_acc = smem_u32(&bars[4]);
  if (threadIdx.x == 0) {
    tma_prefetch_desc(&map_qkv);
    tma_prefetch_desc(&map_do);
    mbar_init(bar_ld, 1);
    mbar_init(bar_sp, 1);
    mbar_init(bar_tfree, 256);
    mbar_init(bar_pds, 256);
    mbar_init(bar_acc, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 8) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_smem)), "n"(512));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  tcgen05_fence_before();
  __syncthreads();
  tcgen05_fence_after();
  const uint32_t tmem = tmem_base_smem;

  if (warp == 8) {
    // ===================== control: TMA loads, every tcgen05.mma =====================
    if (lane == 0) {
      stamp(0);
      mbar_expect_tx(bar_ld, 4 * nblk * TILE);
      for (int b = 0; b < nblk; ++b) {
        tma_load_3d(sQ + b * TILE, &map_qkv, bar_ld, h * DH, b * 128, seq);
        tma_load_3d(sK + b * TILE, &map_qkv, bar_ld, da + h * DH, b * 128, seq);
        tma_load_3d(sV + b * TILE, &map_qkv, bar_ld, 2 * da + h * DH, b * 128, seq);
        tma_load_3d(sdO + b * TILE, &map_do, bar_ld, h * DH, b * 128, seq);
      }
      mbar_wait(bar_ld, 0, 0x31);
      tcgen05_fence_after();
      stamp(1);
      const uint32_t id_sp = idesc(0, 0, 128), id_g_mn = idesc(1, 1, DH), id_g_k = idesc(0, 1, DH);
      // Descriptors differ only in their (address >> 4) field: bases are built once and a constant is added
      // per tile / k-step, so that the issuing thread spends a few instructions per MMA (an N = 64 product
      // retires in ~40 cycles; rebuilding two descriptors per MMA took ~90 and made the issue the bottleneck).
      constexpr uint64_t T16 = TILE >> 4;                 // one tile further
      const uint64_t kQ = desc_k(sQ, 0), kK = desc_k(sK, 0), kV = desc_k(sV, 0), kdO = desc_k(sdO, 0), kdS = desc_k(sdS, 0);
      const uint64_t mP = desc_mn(sP, 0), mdS = desc_mn(sdS, 0), mQ = desc_mn(sQ, 0), mK = desc_mn(sK, 0), mdO = desc_mn(sdO, 0);
      auto issue_sp = [&](int i, int j) {
        const uint64_t a0 = kQ + i * T16, b0 = kK + j * T16, a1 = kdO + i * T16, b1 = kV + j * T16;
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) umma_bf16(tmem + C_S, a0 + ks * 2, b0 + ks * 2, id_sp, ks ? 1u : 0u);
#pragma unroll
        for (int ks = 0; ks < 4; ++ks) umma_bf16(tmem + C_DP, a1 + ks * 2, b1 + ks * 2, id_sp, ks ? 1u : 0u);
        tcgen05_commit(bar_sp);
      };
      // block pairs in order: j outer, i inner (i >= j when causal)
      int n = 0;
      uint32_t dq_started = 0;                            // bit i: dQ_i already holds a partial sum
      issue_sp(0, 0);
      for (int j = 0; j < nblk; ++j) {
        const int i_first = causal ? j : 0;
        for (int i = i_first; i < nblk; ++i, ++n) {
          mbar_wait(bar_tfree, n & 1, 0x32);              // S / dP of this pair are in registers
          tcgen05_fence_after();
          if (n < 4) stamp(2 + 3 * n);
          int ni = i + 1, nj = j;                         // next pair
          if (ni == nblk) { nj = j + 1; ni = causal ? nj : 0; }
          if (nj < nblk) issue_sp(ni, nj);
          mbar_wait(bar_pds, n & 1, 0x33);                // P / dS panels written (and dV_{j-1}, dK_{j-1} read out)
          tcgen05_fence_after();
          if (n < 4) stamp(3 + 3 * n);
          {
            const uint64_t bdO = mdO + i * T16, bQ = mQ + i * T16, bK = mK + j * T16;
            const uint32_t acc_kv = i > i_first ? 1u : 0u, acc_q = (dq_started >> i) & 1u;
            // the three products are independent accumulation chains of eight N = 64 k-steps each: issued round-robin,
            // consecutive tcgen05.mma never wait on the accumulator of the one before
#pragma unroll
            for (int kk = 0; kk < 8; ++kk) {
              umma_bf16(tmem + C_DV, mP + kk * 128, bdO + kk * 128, id_g_mn, kk ? 1u : acc_kv);      // dV_j += P^T dO_i   (K = 128 queries)
              umma_bf16(tmem + C_DK, mdS + kk * 128, bQ + kk * 128, id_g_mn, kk ? 1u : acc_kv);      // dK_j += dS^T Q_i
              umma_bf16(tmem + C_DQ + 64 * i, kdS + (kk >> 2) * T16 + (kk & 3) * 2, bK + kk * 128, id_g_k, kk ? 1u : acc_q);   // dQ_i += dS K_j (K = 128 keys)
            }
          }
          dq_started |= 1u << i;
          tcgen05_commit(bar_acc);
          if (n < 4) stamp(4 + 3 * n);
        }
      }
    }
    __syncwarp();
  } else {
    // ===================== compute warps =====================
    const int quad = warp & 3, chalf = warp >> 2;
    const int64_t sbase = ((int64_t)seq * A + h) * S;
    // D = rowsum(dO * O), L = lse * log2(e): 8 lanes per row, 4 rows per pass; all 16 loads of a thread
    // are issued before the first is used
    {
      const int sub = lane >> 3, l8 = lane & 7;
      uint4 ua[8], ub[8];
#pragma unroll
      for (int it = 0; it < 8; ++it) {
        const int rr = min(warp * 32 + it * 4 + sub, S - 1);
        const int64_t off = ((int64_t)seq * S + rr) * da + h * DH + l8 * 8;
        ua[it] = __ldg(reinterpret_cast<const uint4 *>(d_o + off));
        ub[it] = __ldg(reinterpret_cast<const uint4 *>(o + off));
      }
      const float lv = lane < 32 && warp * 32 + lane < S ? lse[sbase + warp * 32 + lane] * LOG2E : 0.f;
#pragma unroll
      for (int it = 0; it < 8; ++it) {
        const int rr = warp * 32 + it * 4 + sub;
        const __nv_bfloat162 *ha = reinterpret_cast<const __nv_bfloat162 *>(&ua[it]);
        const __nv_bfloat162 *hb = reinterpret_cast<const __nv_bfloat162 *>(&ub[it]);
        float acc = 0.f;
#pragma unroll
        for (int e = 0; e < 4; ++e) {
          const float2 a = __bfloat1622float2(ha[e]), b = __bfloat1622float2(hb[e]);
          acc += a.x * b.x + a.y * b.y;
        }
        acc += __shfl_xor_sync(0xffffffffu, acc, 1);
        acc += __shfl_xor_sync(0xffffffffu, acc, 2);
        acc += __shfl_xor_sync(0xffffffffu, acc, 4);
        if (l8 == 0) Dsm[rr] = rr < S ? acc : 0.f;
      }
      Lsm[warp * 32 + lane] = lv;
    }
    asm volatile("bar.sync 1, 256;" ::: "memory");
    if (threadIdx.x == 0) stamp(16);
    const float sl2 = scale * LOG2E;
    const int r_loc = quad * 32 + lane;                   // row within the 128-row block
    const uint32_t t_lane = tmem + ((uint32_t)(quad * 32) << 16);
    // 32 rows x 32 columns of a finished accumulator (this warp's lane quadrant) -> bf16 -> a padded
    // shared-memory transposer (80-byte rows) -> global with 4 lanes per 64-byte row segment: 8 lines per
    // store instruction instead of 32 (one lane per row costs 32 LSU cycles per instruction)
    const uint32_t xp = smem_u32(xpose) + (uint32_t)warp * (32 * 80);
    // column sums over this sequence's tokens of everything this warp stores (the bias gradient db_qkv = sum_t dqkv[t],
    // fused here instead of a separate pass over dqkv): lane j holds column j
    float cs_acc[4] = {0.f, 0.f, 0.f, 0.f};
    auto store_acc = [&](uint32_t col, float mul, bf16 *dst_row0, int rows_valid, float &cs) {
      uint32_t rr[32];
      tmem_ld32(t_lane + col, rr);
      tmem_ld_wait();
#pragma unroll
      for (int q = 0; q < 4; ++q)
        st_shared_v4(xp + (uint32_t)lane * 80u + (uint32_t)q * 16u,
                     pack2(__uint_as_float(rr[8 * q]) * mul, __uint_as_float(rr[8 * q + 1]) * mul),
                     pack2(__uint_as_float(rr[8 * q + 2]) * mul, __uint_as_float(rr[8 * q + 3]) * mul),
                     pack2(__uint_as_float(rr[8 * q + 4]) * mul, __uint_as_float(rr[8 * q + 5]) * mul),
                     pack2(__uint_as_float(rr[8 * q + 6]) * mul, __uint_as_float(rr[8 * q + 7]) * mul));
      __syncwarp();
#pragma unroll
      for (int it = 0; it < 4; ++it) {
        const int r = it * 8 + (lane >> 2), seg = lane & 3;
        uint4 v;
        asm volatile("ld.shared.v4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(xp + (uint32_t)r * 80u + (uint32_t)seg * 16u));
        if (r < rows_valid) *reinterpret_cast<uint4 *>(dst_row0 + (int64_t)r * (3 * da) + seg * 8) = v;
      }
      if (colpart) {                                       // column `lane` of the 32 x 32 bf16 tile just staged, rows in order
        float t = 0.f;
        const int nr = rows_valid < 32 ? rows_valid : 32;
        for (int r = 0; r < nr; ++r) {
          unsigned short hv;
          asm volatile("ld.shared.u16 %0, [%1];" : "=h"(hv) : "r"(xp + (uint32_t)r * 80u + (uint32_t)lane * 2u));
          t += __uint_as_float((uint32_t)hv << 16);
        }
        cs += t;
      }
      __syncwarp();
    };
    // dV_j (warps 0-3) / dK_j (warps 4-7): this warp's 32 key rows, 64 columns
    auto store_dvdk = [&](int j) {
      const int key0w = j * 128 + quad * 32;
      bf16 *dst = dqkv + ((int64_t)seq * S + key0w) * (3 * da) + (chalf ? da : 2 * da) + h * DH;
      store_acc((chalf ? C_DK : C_DV), chalf ? scale : 1.f, dst, S - key0w, cs_acc[0]);
      store_acc((chalf ? C_DK : C_DV) + 32, chalf ? scale : 1.f, dst + 32, S - key0w, cs_acc[1]);
    };
    int n = 0;
    for (int j = 0; j < nblk; ++j) {
      const int i_first = causal ? j : 0;
      for (int i = i_first; i < nblk; ++i, ++n) {
        const int row = i * 128 + r_loc;
        const int key0 = j * 128 + chalf * 64;             // first key of this thread's 64-column strip
        // last key this row sees (-1: none)
        const int kmax = row < S ? min(S - 1, causal ? row : S - 1) : -1;
        // keys any row of this warp sees end before ...
        const int kvis_w = causal ? min(S, i * 128 + quad * 32 + 32) : S;
        uint32_t ppk[32], dpk[32];
        mbar_wait(bar_sp, n & 1, 0x34);
        tcgen05_fence_after();
        if (threadIdx.x == 0 && n < 4) stamp(17 + 3 * n);
        const float Lr = Lsm[row], Dr = Dsm[row];
#pragma unroll
        for (int c = 0; c < 2; ++c) {
          const int kc = key0 + c * 32;
          if (kc < kvis_w) {                               // warp-uniform
            uint32_t rs[32], rd[32];
            tmem_ld32(t_lane + C_S + chalf * 64 + c * 32, rs);
            tmem_ld32(t_lane + C_DP + chalf * 64 + c * 32, rd);
            tmem_ld_wait();
            const bool edge = kc + 31 > min(S - 1, causal ? i * 128 + quad * 32 : S - 1) || i * 128 + quad * 32 + 31 >= S;
#pragma unroll
            for (int jj = 0; jj < 32; jj += 2) {
              float p0 = ex2(fmaf(__uint_as_float(rs[jj]), sl2, -Lr));
              float p1 = ex2(fmaf(__uint_as_float(rs[jj + 1]), sl2, -Lr));
              if (edge) {
                p0 = kc + jj <= kmax ? p0 : 0.f;
                p1 = kc + jj + 1 <= kmax ? p1 : 0.f;
              }
              ppk[c * 16 + (jj >> 1)] = pack2(p0, p1);
              dpk[c * 16 + (jj >> 1)] = pack2(p0 * (__uint_as_float(rd[jj]) - Dr), p1 * (__uint_as_float(rd[jj + 1]) - Dr));
            }
          } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) { ppk[c * 16 + q] = 0u; dpk[c * 16 + q] = 0u; }
          }
        }
        tcgen05_fence_before();
        mbar_arrive(bar_tfree);                            // TMEM S / dP may be overwritten
        if (threadIdx.x == 0 && n < 4) stamp(18 + 3 * n);
        if (n > 0) {
          mbar_wait(bar_acc, (n - 1) & 1, 0x35);           // the products that read the previous panels are done
          tcgen05_fence_after();
          // ... and with them, at the first pair of a new key block, dV / dK of the previous one
          if (i == i_first) store_dvdk(j - 1);
        }
        const uint32_t pp = sP + (uint32_t)chalf * TILE, dp = sdS + (uint32_t)chalf * TILE;
#pragma unroll
        for (int q = 0; q < 8; ++q) {
          st_shared_v4(panel_addr(pp, r_loc, q), ppk[4 * q], ppk[4 * q + 1], ppk[4 * q + 2], ppk[4 * q + 3]);
          st_shared_v4(panel_addr(dp, r_loc, q), dpk[4 * q], dpk[4 * q + 1], dpk[4 * q + 2], dpk[4 * q + 3]);
        }
        fence_proxy_async_smem();
        tcgen05_fence_before();                            // the dV / dK read-out precedes the next products
        mbar_arrive(bar_pds);
        if (threadIdx.x == 0 && n < 4) stamp(19 + 3 * n);
      }
    }
    // ---- tail: dV / dK of the last key block, then dQ (warps 0-3: block 0, warps 4-7: block 1) ----
    mbar_wait(bar_acc, (n - 1) & 1, 0x36);
    tcgen05_fence_after();
    store_dvdk(nblk - 1);
    if (chalf < nblk) {
      const int q0w = chalf * 128 + quad * 32;
      bf16 *dst = dqkv + ((int64_t)seq * S + q0w) * (3 * da) + h * DH;
      store_acc(C_DQ + 64 * chalf, scale, dst, S - q0w, cs_acc[2]);
      store_acc(C_DQ + 64 * chalf + 32, scale, dst + 32, S - q0w, cs_acc[3]);
    }
    if (colpart) {
      // this (sequence, head)'s 3 x 64 column sums, summed over the warps in a fixed order: dQ from all eight warps (query
      // block 0: warps 0-3, block 1: warps 4-7), dK from warps 4-7, dV from warps 0-3
#pragma unroll
      for (int i = 0; i < 4; ++i) cs_part[warp][i][lane] = cs_acc[i];
      asm volatile("bar.sync 1, 256;" ::: "memory");
      const int t = threadIdx.x;
      if (t < 192) {
        const int which = t >> 6, colh = (t >> 5) & 1, cl = t & 31;      // 0: q, 1: k, 2: v
        float v = 0.f;
        if (which == 0) {
          for (int wq = 0; wq < 8; ++wq) v += cs_part[wq][2 + colh][cl];
        } else {
          const int w0 = which == 1 ? 4 : 0;
          for (int wq = w0; wq < w0 + 4; ++wq) v += cs_part[wq][colh][cl];
        }
        colpart[(int64_t)seq * (3 * da) + which * da + h * DH + colh * 32 + cl] = v;
      }
    }
    if (threadIdx.x == 0) stamp(31);
  }
  tcgen05_fence_before();
  __syncthreads();
  if (warp == 8) {
    tcgen05_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
  }
}

// ------------------------------------------------------------------------------------------
// host side
// ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  });
  return fn;
}

struct Key {
  const void *ptr;
  int64_t width, S, n_seq;
  int box_rows;
  bool operator==(const Key &o) const {
    return ptr == o.ptr && width == o.width && S == o.S && n_seq == o.n_seq && box_rows == o.box_rows;
  }
};
struct KeyHash {
  size_t operator()(const Key &k) const {
    size_t h = (size_t)k.ptr;
    auto mix = [&](uint64_t v) { h ^= v + 0x9e3779b97f4a7c15ull + (h << 6) + (h >> 2); };
    mix((uint64_t)k.width); mix((uint64_t)k.S); mix((uint64_t)k.n_seq); mix((uint64_t)k.box_rows);
    return h;
  }
};

// bf16 [n_seq][S][width] (row pitch = width), box [1][box_rows][64], 128-byte swizzle, zero fill
static bool get_map3(const void *ptr, int64_t width, int64_t S, int64_t n_seq, int box_rows, CUtensorMap *out) {
  static std::unordered_map<Key, CUtensorMap, KeyHash> cache;
  static std::mutex mu;
  Key key{ptr, width, S, n_seq, box_rows};
  std::lock_guard<std::mutex> lock(mu);
  auto it = cache.find(key);
  if (it != cache.end()) {
    *out = it->second;
    return true;
  }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  cuuint64_t dims[3] = {(cuuint64_t)width, (cuuint64_t)S, (cuuint64_t)n_seq};
  cuuint64_t strides[2] = {(cuuint64_t)width * 2, (cuuint64_t)width * 2 * (cuuint64_t)S};
  cuuint32_t box[3] = {64, (cuuint32_t)box_rows, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUtensorMap m;
  CUresult r = fn(&m, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void *>(ptr), dims, strides, box, estr,
                  CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return false;
  if (cache.size() > 16384) cache.clear();
  cache.emplace(key, m);
  *out = m;
  return true;
}

}  // namespace fat

// Profiling hook: when set, every backward CTA writes 32 %globaltimer stamps to buf (control thread:
// 0 start, 1 operands landed, 2+3n / 3+3n / 4+3n: pair n registers pulled / panels written / products
// issued; compute thread 0: 16 D done, 17+3n / 18+3n / 19+3n: pair n S,dP ready / pulled / panels
// written, 30 last store issued, 31 stores complete).  buf: 32 * n_seq * A uint64.
#if GP_PROBES
void attn_tc_set_timeline(unsigned long long *buf) { fat::g_attn_tl = buf; }
#endif

cudaError_t attn_tc_set_watchdog(unsigned long long *mapped) {
  return cudaMemcpyToSymbol(tc::g_watchdog, &mapped, sizeof(mapped));
}

bool attn_tc_supported(int dt, int S, int A, int dh) {
  (void)A;
  return dt == GP_BF16 && dh == 64 && S >= 1 && S <= 256;
}

cudaError_t attn_fwd_tc(const Ctx &c, const void *qkv, void *o, float *lse, int n_seq, int S, int A, int causal) {
  if (n_seq == 0) return cudaSuccess;
  const int da = A * fat::DH;
  CUtensorMap mq;
  if (!fat::get_map3(qkv, 3 * da, S, n_seq, 128, &mq)) return cudaErrorInvalidValue;
  if ((int64_t)n_seq * A > 65535) return cudaErrorInvalidValue;       // grid.y
  {
    cudaError_t e = ensure_dyn_smem<fat::attn_fwd_tc_kernel>(fat::FWD_SMEM, c.device);
    if (e != cudaSuccess) return e;
  }
  // One CTA per (sequence, head) walks both 128-row query blocks (S <= 256) with K and V loaded once: 256 CTAs of the
  // config-5 micro-batch are ONE wave at two CTAs per SM (512 one-block CTAs were 1.73), and a third less operand
  // traffic.  Alone the launch takes the same 20.5 us (two serial chains per CTA); in the step, where SM-time counts,
  // config 5 measured 1406.3 / 1406.9 ms against 1415.3 / 1416.4 ms with one block per CTA (qpb = 1).
  const int qpb = 2;
  const int nqb = (S + 127) / 128;
  dim3 grid((nqb + qpb - 1) / qpb, n_seq * A);
  fat::attn_fwd_tc_kernel<<<grid, fat::FWD_THREADS, fat::FWD_SMEM, c.stream>>>(mq, (bf16 *)o, lse, S, A, causal,
                                                                              1.f / sqrtf((float)fat::DH), qpb, fat::g_attn_tl);
  GP_LAUNCH_CHECK(c);
}

cudaError_t attn_bwd_tc(const Ctx &c, const void *qkv, const void *o, const void *d_o, const float *lse, void *dqkv,
                        float *colpart, int n_seq, int S, int A, int causal) {
  if (n_seq == 0) return cudaSuccess;
  const int da = A * fat::DH;
  CUtensorMap mq, md;
  if (!fat::get_map3(qkv, 3 * da, S, n_seq, 128, &mq) || !fat::get_map3(d_o, da, S, n_seq, 128, &md)) return cudaErrorInvalidValue;
  {
    cudaError_t e = ensure_dyn_smem<fat::attn_bwd_tc_kernel>(fat::BWD_SMEM, c.device);
    if (e != cudaSuccess) return e;
  }
  fat::attn_bwd_tc_kernel<<<n_seq * A, fat::BWD_THREADS, fat::BWD_SMEM, c.stream>>>(
      mq, md, (const bf16 *)o, (const bf16 *)d_o, lse, (bf16 *)dqkv, colpart, S, A, causal, 1.f / sqrtf((float)fat::DH),
      fat::g_attn_tl);
  GP_LAUNCH_CHECK(c);
}

}  // namespace gp
