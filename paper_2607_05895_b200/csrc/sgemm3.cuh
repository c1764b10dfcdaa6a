// Grouped fp32-class GEMM on the bf16 tensor cores (tcgen05), used by the owner-local Shampoo step (shampoo.cu).
//
// Shampoo's preconditioner statistics and inverse fourth roots need fp32-class arithmetic (PAPER.md:182 runs them in
// "float32"); Blackwell has no fp32 tensor-core path and its FFMA pipes deliver ~1/30 of the bf16 tensor rate.  An
// fp32 value v is therefore carried as THREE bf16 terms  v = b1 + b2 + b3  (b1 = rn(v), b2 = rn(v - b1),
// b3 = rn(v - b1 - b2): 24 significand bits, fp32's exponent range, no scaling), stored as three row-major planes,
// and a product of two such matrices is the sum of the six term products with i + j <= 2 (the three dropped ones are
// below 2^-24 of the leading one), all accumulated into ONE fp32 TMEM accumulator:
//     C = sum_{i + j <= 2} A_i B_j^T          6 UMMAs per 16-element k step for 6 operand tiles in shared memory.
// bf16 inputs (a bf16 gradient) are exact single terms: 1 or 3 UMMAs per k step.
//
// Accumulation.  The tensor core adds into its fp32 accumulator with truncation, one truncating add per UMMA k step:
// a chain of K / 16 (x 6) adds shrinks every sum by ~ (adds / 2) 2^-24 -- measured 1.8e-6 at K = 904 with one term,
// 5e-5 at K = 4096 with six: not fp32-class.  So the TMEM accumulator only ever holds the partial sum of ONE chunk of
// k (kKC blocks of 64), the five small term products are issued first (their truncation is relative to sums 2^-8
// smaller) and the four leading-term k steps last; the epilogue warps fold each chunk into registers with
// round-to-nearest fp32 adds (128 accumulator registers per thread = the thread's row of the 128 x 128 tile) while the
// UMMAs of the next chunks run into the other three TMEM buffers.  Residual bias ~ 2 .. 8 x 2^-24 per chunk, unbiased
// rounding across chunks.
//
// One launch works through the tiles of MANY independent problems (every L and every R of the resident set at
// once): 128 x 128 output tiles, k blocks of 64, one CTA per SM, static round-robin over a host-built tile list
// whose order keeps the tiles in flight a compact block of one output (operand panels shared through L2).
// Warp 0 = TMA producer (3-D tensor maps: column, row, term plane; 128-byte swizzle; out-of-range elements read as
// zero, so ragged edges need no special cases), warp 1 = TMEM owner + UMMA issuer, warps 2-5 = epilogue.  Four
// chunk accumulators (4 x 128 TMEM columns) rotate, so the stores of one tile overlap the UMMAs of the next.
// Operands may be K-major (row-major with k contiguous) or MN-major (row-major with the output index
// contiguous: G^T G and P_L G read G in place, never transposed in memory).
//
// Epilogue (all optional, per problem): v = alpha acc + beta Cin;  fp32 store;  three-term split store;  the split of
// T = (5 I - v) / 4 (the next coupled-Newton step matrix);  max |v - I| into an error word;  the weight update
// W <- decay W - lr v.  Symmetric problems compute only the tiles on and above the block diagonal and store the
// mirror image as well; their three-plane outputs leave through asynchronous TMA stores of 32 x 32 blocks staged in
// shared memory (sg_store_block).  Two kernels share all of this: k_sgemm3 (single CTA, 128 x 128 tiles, below) and
// k_sgemm3p (CTA pair, 256 x 256 tiles, further down), chosen per launch by the host; instances <3, 3> (root
// iteration), <2, 2> / <2, 1> (preconditioning products on two-term operands), <1, 1> (statistics of a bf16 gradient).
#ifndef MFSDP_SGEMM3_CUH_
#define MFSDP_SGEMM3_CUH_

#include <cuda.h>
#include <cuda_bf16.h>
#include <stdint.h>

#include "ptx_sm100.cuh"

namespace mfsdp {

struct alignas(64) SgProb {
  CUtensorMap ta, tb;               // operand storage: dims (cols, rows, planes)
  CUtensorMap to, tt;               // store maps of out_split / t_split: box 32 cols x 32 rows x 1 plane, no swizzle
  uint32_t M, N, K;                 // output rows, columns; reduction length
  uint32_t a_mn, b_mn;              // 1: operand stored [k][m] (MN-major) instead of [m][k]
  uint32_t sym;                     // symmetric output: tiles with n0 >= m0 only, mirrored by the epilogue
  uint32_t f32_pitch;               // row pitch of cin / out_f32 (elements; multiple of 64 so that 32-column chunks fit)
  uint32_t sp_pitch;                // row pitch of the split planes (elements, multiple of 64)
  uint64_t sp_plane;                // elements between the planes of out_split / t_split
  const float* cin;                 // optional; may alias out_f32 (read before written by the same thread)
  float* out_f32;                   // optional
  __nv_bfloat16* out_split;         // optional: three planes
  __nv_bfloat16* t_split;           // optional: split of (5 I - v) / 4
  uint32_t* err;                    // optional: atomicMax of the bits of max |v - delta|
  const uint32_t* done;             // optional: non-zero -> the problem is finished, its tiles are skipped
  const float* alpha_dev;           // optional: per-problem factor on top of the launch's alpha (read at tile start)
  void* W;                          // optional: rank-flat weights of this matrix (pitch = N), updated in place
  uint32_t w_bf16;                  // dtype of W
  uint32_t pad;
};
struct SgTile { uint32_t prob, m0, n0; };
struct SgParams {
  const SgProb* probs;
  const SgTile* tiles;
  uint32_t n_tiles;
  float alpha, beta;                // v = alpha acc + beta Cin
  float decay, lr;                  // W <- decay W - lr v
  unsigned long long* trace;        // mfsdp_debug_trace target or null: [0] = record counter, then 6-word records
  uint32_t trace_cap;               // (k_sgemm3p: per tile and role {role << 32 | tile, begin, end, wait a, wait b, sm})
};

constexpr uint32_t kSgThreads = 192;
constexpr uint32_t kSgBox = 16384;  // one term of one operand of one stage: 128 rows x 64 k, or 2 x (64 k x 64 mn)
template <int AT, int BT> struct SgCfg {
  static constexpr uint32_t kStage = (AT + BT) * kSgBox;
  static constexpr uint32_t kStages = (AT + BT) == 2 ? 6 : (AT + BT) == 3 ? 4 : (AT + BT) == 4 ? 3 : 2;
  // term products kept: i + j <= kOrder.  Three terms: the six with i + j <= 2 (2^-24-class); two terms: the three with
  // i + j <= 1 (2^-16-class, for the products around a preconditioner that is itself accurate to 1e-3 at best)
  static constexpr int kOrder = (AT > BT ? AT : BT) - 1;
  static constexpr uint32_t kSmem = kStages * kStage + 256 + 1024 + 8 * 32 * 33 * 4;   // ring, barriers, alignment, 8 transposition tiles
  // k blocks per TMEM chunk.  One: at most four truncating adds of leading-term products per partial sum.  (With one
  // term per operand a block is 256 cycles of UMMA, less than the epilogue warps need to fold it -- 4 tcgen05.ld of 32
  // columns + 128 adds -- so the statistics GEMM of a bf16 gradient runs fold-bound; it is a few percent of a step.)
  static constexpr uint32_t kKC = 1;
};
constexpr uint32_t kSgAccs = 4;      // TMEM chunk accumulators of 128 columns
constexpr uint32_t kSgPrefetch = 3;  // k blocks between the L2 prefetch of a box and its load

namespace sg {
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const void* tmap, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(dst),
      "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}
// TMA prefetch of one box into L2 (no shared memory, no completion): issued a few k blocks ahead of the load, so that
// the load itself finds its lines in L2 -- the operand ring holds only two stages, i.e. a load has one k block of UMMA
// time to land, less than a DRAM round trip under load.
__device__ __forceinline__ void tma_prefetch_3d(const void* tmap, int c0, int c1, int c2) {
  asm volatile("cp.async.bulk.prefetch.tensor.3d.L2.global.tile [%0, {%1, %2, %3}];" ::"l"(tmap), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}
__device__ __forceinline__ void tma_store_3d(const void* tmap, int c0, int c1, int c2, uint32_t src_smem) {
  asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tmap), "r"(c0), "r"(c1),
               "r"(c2), "r"(src_smem)
               : "memory");
}
__device__ __forceinline__ void split3(float v, uint32_t& b1, uint32_t& b2, uint32_t& b3) {   // bf16 bit patterns
  const __nv_bfloat16 h1 = __float2bfloat16_rn(v);
  const float r1 = v - __bfloat162float(h1);                      // exact
  const __nv_bfloat16 h2 = __float2bfloat16_rn(r1);
  const float r2 = r1 - __bfloat162float(h2);                     // exact
  const __nv_bfloat16 h3 = __float2bfloat16_rn(r2);
  b1 = __bfloat16_as_ushort(h1); b2 = __bfloat16_as_ushort(h2); b3 = __bfloat16_as_ushort(h3);
}
// 8 consecutive values of one row -> the three planes (16 bytes each)
__device__ __forceinline__ void store_split8(__nv_bfloat16* p0, uint64_t plane, const float* v) {
  uint32_t w[3][4];
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    uint32_t a1, a2, a3, c1, c2, c3;
    split3(v[2 * j], a1, a2, a3);
    split3(v[2 * j + 1], c1, c2, c3);
    w[0][j] = a1 | (c1 << 16); w[1][j] = a2 | (c2 << 16); w[2][j] = a3 | (c3 << 16);
  }
#pragma unroll
  for (int t = 0; t < 3; ++t)
    *reinterpret_cast<uint4*>(p0 + t * plane) = make_uint4(w[t][0], w[t][1], w[t][2], w[t][3]);
}
// 16 consecutive values of one row -> the three planes, one 32-byte store each: a full L2 sector per lane and plane
// (the 16-byte form fills half a sector per store; with one row per lane that doubles the write transactions, and the
// stores of a short-k tile cost as much as its UMMAs)
__device__ __forceinline__ void st_global_v8(void* p, const uint32_t (&w)[8]) {
  asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(w[0]), "r"(w[1]), "r"(w[2]),
               "r"(w[3]), "r"(w[4]), "r"(w[5]), "r"(w[6]), "r"(w[7])
               : "memory");
}
__device__ __forceinline__ void store_split16(__nv_bfloat16* p0, uint64_t plane, const float* v) {
  uint32_t w[3][8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    uint32_t a1, a2, a3, c1, c2, c3;
    split3(v[2 * j], a1, a2, a3);
    split3(v[2 * j + 1], c1, c2, c3);
    w[0][j] = a1 | (c1 << 16); w[1][j] = a2 | (c2 << 16); w[2][j] = a3 | (c3 << 16);
  }
#pragma unroll
  for (int t = 0; t < 3; ++t) st_global_v8(p0 + t * plane, w[t]);
}
__device__ __forceinline__ void store_f32x8(float* p, const float* v) {
  const uint32_t w[8] = {__float_as_uint(v[0]), __float_as_uint(v[1]), __float_as_uint(v[2]), __float_as_uint(v[3]),
                         __float_as_uint(v[4]), __float_as_uint(v[5]), __float_as_uint(v[6]), __float_as_uint(v[7])};
  st_global_v8(p, w);
}
__device__ __forceinline__ void store_split1(__nv_bfloat16* d, uint64_t plane, float v) {
  uint32_t b1, b2, b3;
  split3(v, b1, b2, b3);
  d[0] = __ushort_as_bfloat16((unsigned short)b1);
  d[plane] = __ushort_as_bfloat16((unsigned short)b2);
  d[2 * plane] = __ushort_as_bfloat16((unsigned short)b3);
}
}  // namespace sg


// One warp's 32 x 32 block of a three-plane output (lane = row, v = its 32 columns) -> global memory through TMA
// stores: per plane the block is staged in shared memory (32 rows x 64 bytes, dense) and stored asynchronously, so the
// warp is not held up by the write burst (all CTAs finish their tiles together: with plain stores the epilogue of a
// tile took ~55 K cycles, during which the UMMAs of the next tile wait for the fold).  TMA clips at the matrix edges.
//   mode 0: the block as it is, at (row0, cb)
//   mode 1: as it is at (row0, cb) AND transposed at (cb, row0)          (strictly above the diagonal of a symmetric output)
//   mode 2: a block ON the diagonal: upper triangle from the rows themselves, lower triangle = its mirror image
//           (bit-symmetric although the two triangles were summed in different orders)
// `stg`: two 2 KB staging tiles of this warp; `n_st`: TMA stores issued so far by this warp (staging tile parity).
__device__ __forceinline__ void sg_store_block(const CUtensorMap* tm, const float* v, uint32_t row0, uint32_t cb, int mode,
                                               uint32_t lane, uint32_t stg, uint32_t& n_st, bool as_t) {
  // as_t: store T = (5 I - v) / 4 instead of v (formed on the fly; r = row0 + lane is this lane's row)
  const uint32_t dcol = row0 + lane - cb;                      // column offset of the diagonal element in this block, if any
#pragma unroll 1
  for (int t = 0; t < 3; ++t) {                                // not unrolled: one plane's 16 packed words live at a time
    uint32_t w[16];                                            // plane t of the lane's 32 values, packed pairs
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      float x0 = v[2 * j], x1 = v[2 * j + 1];
      if (as_t) {
        x0 = 0.25f * (((uint32_t)(2 * j) == dcol ? 5.f : 0.f) - x0);
        x1 = 0.25f * (((uint32_t)(2 * j + 1) == dcol ? 5.f : 0.f) - x1);
      }
      uint32_t a[3], c[3];
      sg::split3(x0, a[0], a[1], a[2]);
      sg::split3(x1, c[0], c[1], c[2]);
      w[j] = (t == 0 ? a[0] : t == 1 ? a[1] : a[2]) | ((t == 0 ? c[0] : t == 1 ? c[1] : c[2]) << 16);
    }
    {   // the block itself
      const uint32_t buf = stg + (n_st & 1u) * 2048u;
      if (lane == 0) ptx::bulk_wait_read<1>();                 // the store issued two stores ago has read this tile
      __syncwarp();
#pragma unroll
      for (int qd = 0; qd < 4; ++qd)
        ptx::st_shared_v4(buf + lane * 64u + 16u * qd, w[4 * qd], w[4 * qd + 1], w[4 * qd + 2], w[4 * qd + 3]);
      if (mode == 2) {
        __syncwarp();
#pragma unroll
        for (int j = 0; j < 32; ++j)                           // element (lane, j), j > lane, also is element (j, lane)
          if (j > (int)lane) ptx::st_shared_b16(buf + (uint32_t)j * 64u + lane * 2u, (uint16_t)(j & 1 ? w[j >> 1] >> 16 : w[j >> 1] & 0xffffu));
      }
      ptx::fence_async_smem();
      __syncwarp();
      if (lane == 0) { sg::tma_store_3d(tm, (int)cb, (int)row0, t, buf); ptx::bulk_commit(); }
      ++n_st;
    }
    if (mode == 1) {   // the transposed block
      const uint32_t buf = stg + (n_st & 1u) * 2048u;
      if (lane == 0) ptx::bulk_wait_read<1>();
      __syncwarp();
#pragma unroll
      for (int j = 0; j < 32; ++j)
        ptx::st_shared_b16(buf + (uint32_t)j * 64u + lane * 2u, (uint16_t)(j & 1 ? w[j >> 1] >> 16 : w[j >> 1] & 0xffffu));
      ptx::fence_async_smem();
      __syncwarp();
      if (lane == 0) { sg::tma_store_3d(tm, (int)row0, (int)cb, t, buf); ptx::bulk_commit(); }
      ++n_st;
    }
  }
}

// The stores of one thread's row of a tile: `acc` = 128 consecutive columns starting at n0 of output row r (this warp's
// rows start at row0, a multiple of 32), already summed over k.  Worked through in chunks of 32 columns, groups of 8
// inside, to keep few values live beside the 128 accumulators.  The mirror image of a symmetric output goes through
// `tbuf` (32 x 33 floats of shared memory per warp): the warp's 32 x 32 block is transposed there, so that a lane owns
// 32 consecutive elements of one mirrored row and stores them as 16-byte vectors like the direct image (element-wise
// scattered 2-byte stores of the three planes cost more than the UMMAs of a short-k tile).
__device__ __forceinline__ void sg_finish_row(const SgProb* pr, const SgParams& p, float (&acc)[128], uint32_t row0,
                                              uint32_t r, uint32_t n0, bool mirror, bool diag, uint32_t lane,
                                              uint32_t tbuf, uint32_t& n_st) {
  const uint32_t M = pr->M, N = pr->N;
  const bool row_ok = r < M;
  uint32_t emax = 0u;                                         // bits of max |v - delta| (NaN sorts above everything)
  if (row0 >= M) return;                                      // warp-uniform
  const float alpha = pr->alpha_dev != nullptr ? p.alpha * *pr->alpha_dev : p.alpha;
  const float* cin = pr->cin;
  float* of32 = pr->out_f32;
  __nv_bfloat16* osp = pr->out_split;
  __nv_bfloat16* tsp = pr->t_split;
  const uint32_t* errp = pr->err;
  const uint32_t fp = pr->f32_pitch;
#pragma unroll
  for (int ch = 0; ch < 4; ++ch) {
    const uint32_t cb = n0 + 32u * ch;
    if (cb >= N) continue;                                    // warp-uniform
#pragma unroll
    for (int gg = 0; gg < 2; ++gg) {
      const int g = 2 * ch + gg;
      const uint32_t c0 = n0 + 16u * g;
      float* v = acc + 16 * g;                                  // compile-time offsets: stays in registers
#pragma unroll
      for (int j = 0; j < 16; ++j) v[j] *= alpha;
      if (!row_ok) continue;
      if (cin != nullptr) {
        const float4* src = reinterpret_cast<const float4*>(cin + (size_t)r * fp + c0);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float4 a = src[j];
          v[4 * j] = fmaf(p.beta, a.x, v[4 * j]); v[4 * j + 1] = fmaf(p.beta, a.y, v[4 * j + 1]);
          v[4 * j + 2] = fmaf(p.beta, a.z, v[4 * j + 2]); v[4 * j + 3] = fmaf(p.beta, a.w, v[4 * j + 3]);
        }
      }
      if (errp != nullptr) {
#pragma unroll
        for (int j = 0; j < 16; ++j)
          if (c0 + j < N) emax = max(emax, __float_as_uint(fabsf(v[j] - (c0 + j == r ? 1.f : 0.f))));
      }
      if (of32 != nullptr) {
        if (!diag) {
          sg::store_f32x8(of32 + (size_t)r * fp + c0, v);
          sg::store_f32x8(of32 + (size_t)r * fp + c0 + 8, v + 8);
        } else {
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            if (c0 + j < N && c0 + j >= r) of32[(size_t)r * fp + c0 + j] = v[j];
            if (c0 + j < N && c0 + j > r) of32[(size_t)(c0 + j) * fp + r] = v[j];
          }
        }
      }
      if (pr->W != nullptr) {
        // W <- decay W - lr v (rank-flat, pitch = N: no padding, element-wise predicates at the right edge)
        if (pr->w_bf16) {
          __nv_bfloat16* w = reinterpret_cast<__nv_bfloat16*>(pr->W) + (size_t)r * N + c0;
          if ((N & 7u) == 0u) {                                   // 16-byte vectors never straddle the row end
#pragma unroll
            for (int h = 0; h < 2; ++h) {
              if (c0 + 8u * h < N) {
                const uint4 x = reinterpret_cast<const uint4*>(w)[h];
                uint32_t xs[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  const float w0 = __uint_as_float(xs[i] << 16), w1 = __uint_as_float(xs[i] & 0xffff0000u);
                  const __nv_bfloat162 hh = __floats2bfloat162_rn(fmaf(-p.lr, v[8 * h + 2 * i], p.decay * w0),
                                                                  fmaf(-p.lr, v[8 * h + 2 * i + 1], p.decay * w1));
                  xs[i] = *reinterpret_cast<const uint32_t*>(&hh);
                }
                reinterpret_cast<uint4*>(w)[h] = make_uint4(xs[0], xs[1], xs[2], xs[3]);
              }
            }
          } else {
#pragma unroll
            for (int j = 0; j < 16; ++j)
              if (c0 + j < N) w[j] = __float2bfloat16_rn(fmaf(-p.lr, v[j], p.decay * __bfloat162float(w[j])));
          }
        } else {
          float* w = reinterpret_cast<float*>(pr->W) + (size_t)r * N + c0;
#pragma unroll
          for (int j = 0; j < 16; ++j)
            if (c0 + j < N) w[j] = fmaf(-p.lr, v[j], p.decay * w[j]);
        }
      }
    }
    if (of32 != nullptr && mirror && !diag) {
      // fp32 mirror image: transpose this warp's 32 x 32 block through the scratch tile, so that a lane owns 32
      // consecutive elements of one mirrored row.  (rows >= M hold alpha * 0 = 0 and land in the pitch padding)
      float* v = acc + 32 * ch;
      if (lane == 0) ptx::bulk_wait_read<0>();                  // no TMA store of this warp still reads the scratch
      __syncwarp();
#pragma unroll
      for (int j = 0; j < 32; ++j) ptx::st_shared_u32(tbuf + (lane * 33u + j) * 4u, __float_as_uint(row_ok ? v[j] : 0.f));
      __syncwarp();
      float w[32];
#pragma unroll
      for (int i = 0; i < 32; ++i) w[i] = __uint_as_float(ptx::ld_shared_u32(tbuf + (i * 33u + lane) * 4u));
      __syncwarp();
      const uint32_t mr = cb + lane;
      if (mr < N) {
#pragma unroll
        for (int g = 0; g < 4; ++g) sg::store_f32x8(of32 + (size_t)mr * fp + row0 + 8 * g, w + 8 * g);
      }
    }
    // three-plane outputs: asynchronous TMA stores of 32 x 32 blocks (see sg_store_block)
    const int mode = !mirror ? 0 : cb > row0 ? 1 : cb == row0 ? 2 : -1;   // below the diagonal: the mirror image covers it
    if (mode == 0 && osp != nullptr) {
      // a general (non-symmetric) output has no mirror image and no write burst worth hiding: plain 32-byte stores
      if (row_ok) {
        sg::store_split16(osp + (size_t)r * pr->sp_pitch + cb, pr->sp_plane, acc + 32 * ch);
        sg::store_split16(osp + (size_t)r * pr->sp_pitch + cb + 16, pr->sp_plane, acc + 32 * ch + 16);
      }
    } else
    if (mode >= 0 && osp != nullptr) sg_store_block(&pr->to, acc + 32 * ch, row0, cb, mode, lane, tbuf, n_st, false);
    if (mode >= 0 && tsp != nullptr) sg_store_block(&pr->tt, acc + 32 * ch, row0, cb, mode, lane, tbuf, n_st, true);   // T = (5 I - v) / 4
  }
  if (errp != nullptr) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) emax = max(emax, __shfl_xor_sync(0xffffffffu, emax, o));
    if (lane == 0 && emax != 0u) atomicMax(pr->err, emax);
  }
}

template <int AT, int BT>
__global__ void __launch_bounds__(kSgThreads, 1) k_sgemm3(const SgParams p) {
  using Cfg = SgCfg<AT, BT>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t ring0 = ptx::smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cfg::kStages * Cfg::kStage);
  const uint32_t full0 = ptx::smem_u32(bars), empty0 = ptx::smem_u32(bars + Cfg::kStages);
  const uint32_t tfull0 = ptx::smem_u32(bars + 2 * Cfg::kStages), tempty0 = ptx::smem_u32(bars + 2 * Cfg::kStages + kSgAccs);
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 2 * Cfg::kStages + 2 * kSgAccs);
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (uint32_t s = 0; s < Cfg::kStages; ++s) { ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 1); }
    for (uint32_t s = 0; s < kSgAccs; ++s) { ptx::mbar_init(tfull0 + 8 * s, 1); ptx::mbar_init(tempty0 + 8 * s, 4); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc<512, 1>(ptx::smem_u32(tmem_holder));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;

  uint32_t stage = 0, ring_phase = 0;   // producer, issuer
  uint32_t cc = 0;                      // k chunks this CTA has worked on: TMEM accumulator = cc % 4 (issuer, epilogue)
  uint32_t n_st = 0;                    // TMA stores issued by this (epilogue) warp

  for (uint32_t ti = blockIdx.x; ti < p.n_tiles; ti += gridDim.x) {
    const SgTile t = p.tiles[ti];
    const SgProb* pr = p.probs + t.prob;
    if (pr->done != nullptr && *pr->done != 0u) continue;       // stable during the launch: every role agrees
    const uint32_t K = pr->K, nkb = (K + 63u) >> 6;
    const uint32_t a_mn = pr->a_mn, b_mn = pr->b_mn;

    if (warp == 0) {
      // ===== TMA producer =====
      for (uint32_t kb = 0; kb < nkb; ++kb) {
        ptx::mbar_wait(empty0 + 8 * stage, ring_phase ^ 1u);
        if (ptx::elect_one()) {
          const uint32_t dst = ring0 + stage * Cfg::kStage, fb = full0 + 8 * stage;
          ptx::mbar_arrive_expect_tx(fb, Cfg::kStage);
#pragma unroll
          for (int i = 0; i < AT; ++i) {
            if (!a_mn) sg::tma_load_3d(dst + i * kSgBox, &pr->ta, (int)(64 * kb), (int)t.m0, i, fb);
            else {
              sg::tma_load_3d(dst + i * kSgBox, &pr->ta, (int)t.m0, (int)(64 * kb), i, fb);
              sg::tma_load_3d(dst + i * kSgBox + 8192, &pr->ta, (int)t.m0 + 64, (int)(64 * kb), i, fb);
            }
          }
#pragma unroll
          for (int j = 0; j < BT; ++j) {
            const uint32_t d = dst + (AT + j) * kSgBox;
            if (!b_mn) sg::tma_load_3d(d, &pr->tb, (int)(64 * kb), (int)t.n0, j, fb);
            else {
              sg::tma_load_3d(d, &pr->tb, (int)t.n0, (int)(64 * kb), j, fb);
              sg::tma_load_3d(d + 8192, &pr->tb, (int)t.n0 + 64, (int)(64 * kb), j, fb);
            }
          }
          if (kb + kSgPrefetch < nkb) {
            const int kp = (int)(64 * (kb + kSgPrefetch));
#pragma unroll
            for (int i = 0; i < AT; ++i) {
              if (!a_mn) sg::tma_prefetch_3d(&pr->ta, kp, (int)t.m0, i);
              else { sg::tma_prefetch_3d(&pr->ta, (int)t.m0, kp, i); sg::tma_prefetch_3d(&pr->ta, (int)t.m0 + 64, kp, i); }
            }
#pragma unroll
            for (int j = 0; j < BT; ++j) {
              if (!b_mn) sg::tma_prefetch_3d(&pr->tb, kp, (int)t.n0, j);
              else { sg::tma_prefetch_3d(&pr->tb, (int)t.n0, kp, j); sg::tma_prefetch_3d(&pr->tb, (int)t.n0 + 64, kp, j); }
            }
          }
        }
        __syncwarp();
        if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1u; }
      }
    } else if (warp == 1) {
      // ===== UMMA issuer: loops run converged (warp-uniform descriptors), one elected lane issues =====
      const uint32_t idesc = ptx::idesc_bf16_f32(128, 128, a_mn, b_mn);
      const uint32_t a_step = a_mn ? (2048u >> 4) : (32u >> 4), b_step = b_mn ? (2048u >> 4) : (32u >> 4);
      const uint32_t a_lbo = a_mn ? 8192u : 16u, b_lbo = b_mn ? 8192u : 16u;
      for (uint32_t kb0 = 0; kb0 < nkb; kb0 += Cfg::kKC) {
        const uint32_t buf = cc % kSgAccs, use = cc / kSgAccs;
        ptx::mbar_wait(tempty0 + 8 * buf, (use & 1u) ^ 1u);       // the epilogue has folded this accumulator's last chunk
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + buf * 128u;
        const uint32_t kb1 = min(nkb, kb0 + Cfg::kKC);
        for (uint32_t kb = kb0; kb < kb1; ++kb) {
          ptx::mbar_wait(full0 + 8 * stage, ring_phase);
          ptx::tc_fence_after();
          // Descriptors are formed in warp-uniform code and every UMMA of the block is unrolled with constant offsets
          // (always four k steps: a ragged last block reads TMA's zero fill), so that the elected lane issues from
          // uniform registers without per-instruction register moves (~200 cycles per UMMA otherwise: issue-bound).
          const uint32_t base = ring0 + stage * Cfg::kStage;
          uint64_t ad[AT], bd[BT];
#pragma unroll
          for (int i = 0; i < AT; ++i) ad[i] = ptx::smem_desc_sw128(base + i * kSgBox, a_lbo, 1024);
#pragma unroll
          for (int j = 0; j < BT; ++j) bd[j] = ptx::smem_desc_sw128(base + (AT + j) * kSgBox, b_lbo, 1024);
          if (ptx::elect_one()) {
            // the small term products first, the leading one last (see "Accumulation" above)
            bool first = true;
#pragma unroll
            for (int i = 0; i < AT; ++i)
#pragma unroll
              for (int j = 0; j < BT; ++j)
                if (i + j <= Cfg::kOrder && i + j > 0) {
#pragma unroll
                  for (uint32_t ks = 0; ks < 4; ++ks) {
                    ptx::umma_bf16(d_tmem, ad[i] + (uint64_t)(ks * a_step), bd[j] + (uint64_t)(ks * b_step), idesc, first ? 0u : 1u);
                    first = false;
                  }
                }
#pragma unroll
            for (uint32_t ks = 0; ks < 4; ++ks) {
              ptx::umma_bf16(d_tmem, ad[0] + (uint64_t)(ks * a_step), bd[0] + (uint64_t)(ks * b_step), idesc, first ? 0u : 1u);
              first = false;
            }
            ptx::umma_commit(empty0 + 8 * stage);
            if (kb + 1 == kb1) ptx::umma_commit(tfull0 + 8 * buf);
          }
          __syncwarp();
          if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1u; }
        }
        ++cc;
      }
    } else {
      // ===== epilogue: warp owns TMEM lanes 32 q .. + 31 = rows m0 + 32 q .. of the tile =====
      const uint32_t q = warp & 3u;
      const uint32_t r = t.m0 + q * 32u + lane;
      // symmetric outputs: a tile above the block diagonal also stores its mirror image; a tile ON the diagonal stores
      // its upper triangle (c >= r) and the mirror of the strict upper triangle, so that the result is bit-symmetric
      // (with several terms the two triangles of a diagonal tile are summed in different orders)
      const bool mirror = pr->sym != 0u && t.n0 >= t.m0;
      const bool diag = pr->sym != 0u && t.n0 == t.m0;
      // fold the k chunks into registers: this thread's row of the tile, round-to-nearest adds
      float acc[128];
      for (uint32_t kb0 = 0; kb0 < nkb; kb0 += Cfg::kKC) {
        const uint32_t buf = cc % kSgAccs, use = cc / kSgAccs;
        ptx::mbar_wait(tfull0 + 8 * buf, use & 1u);
        ptx::tc_fence_after();
#pragma unroll
        for (int h = 0; h < 4; ++h) {
          uint32_t raw[32];
          ptx::tmem_ld32(tmem_base + ((q * 32u) << 16) + buf * 128u + 32u * h, raw);
          ptx::tmem_ld_wait();
          if (kb0 == 0) {
#pragma unroll
            for (int j = 0; j < 32; ++j) acc[32 * h + j] = __uint_as_float(raw[j]);
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) acc[32 * h + j] += __uint_as_float(raw[j]);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(tempty0 + 8 * buf);
        ++cc;
      }
      sg_finish_row(pr, p, acc, t.m0 + q * 32u, r, t.n0, mirror, diag, lane,
                    ring0 + Cfg::kStages * Cfg::kStage + 256u + (warp - 2u) * (32u * 33u * 4u), n_st);
    }
  }

  if (warp >= 2 && lane == 0) ptx::bulk_wait<0>();          // this warp's TMA stores have been performed
  __syncwarp();
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<512, 1>(tmem_base);
  }
}


// ---- CTA-pair form ---------------------------------------------------------------------------------------------------
// The same product on 256 x 256 tiles owned by a cluster of two CTAs (tcgen05 cta_group::2: M = 256 over the two SMs,
// each CTA stages its 128 rows of A and its 128 rows of B per term and k block).  Per CTA and k block that is the same
// 96 KB of operands as the single-CTA tile for TWICE the UMMA time (6 x 4 UMMAs of 128 cycles): 31 B/clk/SM asked of
// the L2 -> SM path instead of 62, which is what keeps the single-CTA form at 52-59 % tensor-pipe activity.  Each CTA
// holds its 128 rows x 256 columns of the chunk accumulator (2 x 256 TMEM columns); eight epilogue warps per CTA fold
// and store it (warps w and w + 4 share a TMEM lane quarter and split the columns).  384 threads leave 168 registers
// per thread, too few beside 128 accumulators: the control warpgroup (producer, issuer, two idle warps) gives its
// registers back (setmaxnreg.dec 40) and the two epilogue warpgroups take them (setmaxnreg.inc 232).  Used when a
// launch has at least ~ one wave of 256-tiles; small problem sets stay on the single-CTA kernel.
constexpr uint32_t kSgPairThreads = 384;   // warps 0-7 epilogue (two warpgroups), 8 producer, 9 UMMA issuer, 10-11 idle
namespace sg {
__device__ __forceinline__ void tma_load_3d_cg2(uint32_t dst, const void* tmap, int c0, int c1, int c2, uint32_t bar_cluster) {
  asm volatile(
      "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], "
      "[%5];" ::"r"(dst),
      "l"(tmap), "r"(c0), "r"(c1), "r"(c2), "r"(bar_cluster)
      : "memory");
}
}  // namespace sg

__device__ __forceinline__ void sg_trace(const SgParams& p, uint32_t role, uint32_t tile, long long t0, long long t1,
                                         long long wa, long long wb) {
  const unsigned long long i = atomicAdd(p.trace, 1ull);
  if (i < p.trace_cap) {
    unsigned long long* r = p.trace + 1 + 6 * i;
    r[0] = ((unsigned long long)role << 32) | tile; r[1] = (unsigned long long)t0; r[2] = (unsigned long long)t1;
    r[3] = (unsigned long long)wa; r[4] = (unsigned long long)wb; r[5] = ptx::smid();
  }
}

template <int AT, int BT>
__global__ void __launch_bounds__(kSgPairThreads, 1) k_sgemm3p(const SgParams p) {
  using Cfg = SgCfg<AT, BT>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t ring0 = ptx::smem_u32(smem);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + Cfg::kStages * Cfg::kStage);
  const uint32_t full0 = ptx::smem_u32(bars), empty0 = ptx::smem_u32(bars + Cfg::kStages);
  const uint32_t tfull0 = ptx::smem_u32(bars + 2 * Cfg::kStages), tempty0 = ptx::smem_u32(bars + 2 * Cfg::kStages + 2);
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 2 * Cfg::kStages + 4);
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = ptx::cluster_ctarank();                  // 0 = leader: owns the full / tempty barriers, issues the UMMAs
  const uint32_t unit = blockIdx.x >> 1, n_units = gridDim.x >> 1;

  if (threadIdx.x == 0) {
    for (uint32_t s = 0; s < Cfg::kStages; ++s) { ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 1); }
    for (uint32_t s = 0; s < 2; ++s) { ptx::mbar_init(tfull0 + 8 * s, 1); ptx::mbar_init(tempty0 + 8 * s, 16); }
    ptx::fence_barrier_init();
  }
  if (warp == 9) ptx::tmem_alloc<512, 2>(ptx::smem_u32(tmem_holder));
  ptx::tc_fence_before();
  ptx::cluster_sync();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;
  const uint32_t full_lead0 = ptx::mapa(full0, 0), tempty_lead0 = ptx::mapa(tempty0, 0);

  // Every role walks the same static tile sequence in its own loop, so that the register budget of a role is set once,
  // before its loop (ptxas allocates per region dominated by the setmaxnreg).
  if (warp >= 8) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == 8) {
      // ===== TMA producer (both CTAs; the bytes of both are counted on the leader's full barrier) =====
      uint32_t stage = 0, ring_phase = 0;
      for (uint32_t ti = unit; ti < p.n_tiles; ti += n_units) {
        const SgTile t = p.tiles[ti];
        const SgProb* pr = p.probs + t.prob;
        if (pr->done != nullptr && *pr->done != 0u) continue;   // stable during the launch: every role agrees
        const uint32_t nkb = (pr->K + 63u) >> 6;
        const uint32_t a_mn = pr->a_mn, b_mn = pr->b_mn;
        const int am0 = (int)(t.m0 + rank * 128u), bn0 = (int)(t.n0 + rank * 128u);
        const long long tr0 = p.trace ? clock64() : 0;
        long long wa = 0;
        for (uint32_t kb = 0; kb < nkb; ++kb) {
          if (p.trace) { const long long c0 = clock64(); ptx::mbar_wait(empty0 + 8 * stage, ring_phase ^ 1u); wa += clock64() - c0; }
          else ptx::mbar_wait(empty0 + 8 * stage, ring_phase ^ 1u);
          if (ptx::elect_one()) {
            if (rank == 0) ptx::mbar_arrive_expect_tx(full0 + 8 * stage, 2u * Cfg::kStage);
            const uint32_t dst = ring0 + stage * Cfg::kStage, fb = full_lead0 + 8 * stage;
#pragma unroll
            for (int i = 0; i < AT; ++i) {
              if (!a_mn) sg::tma_load_3d_cg2(dst + i * kSgBox, &pr->ta, (int)(64 * kb), am0, i, fb);
              else {
                sg::tma_load_3d_cg2(dst + i * kSgBox, &pr->ta, am0, (int)(64 * kb), i, fb);
                sg::tma_load_3d_cg2(dst + i * kSgBox + 8192, &pr->ta, am0 + 64, (int)(64 * kb), i, fb);
              }
            }
#pragma unroll
            for (int j = 0; j < BT; ++j) {
              const uint32_t d = dst + (AT + j) * kSgBox;
              if (!b_mn) sg::tma_load_3d_cg2(d, &pr->tb, (int)(64 * kb), bn0, j, fb);
              else {
                sg::tma_load_3d_cg2(d, &pr->tb, bn0, (int)(64 * kb), j, fb);
                sg::tma_load_3d_cg2(d + 8192, &pr->tb, bn0 + 64, (int)(64 * kb), j, fb);
              }
            }
            if (kb + kSgPrefetch < nkb) {
              const int kp = (int)(64 * (kb + kSgPrefetch));
#pragma unroll
              for (int i = 0; i < AT; ++i) {
                if (!a_mn) sg::tma_prefetch_3d(&pr->ta, kp, am0, i);
                else { sg::tma_prefetch_3d(&pr->ta, am0, kp, i); sg::tma_prefetch_3d(&pr->ta, am0 + 64, kp, i); }
              }
#pragma unroll
              for (int j = 0; j < BT; ++j) {
                if (!b_mn) sg::tma_prefetch_3d(&pr->tb, kp, bn0, j);
                else { sg::tma_prefetch_3d(&pr->tb, bn0, kp, j); sg::tma_prefetch_3d(&pr->tb, bn0 + 64, kp, j); }
              }
            }
          }
          __syncwarp();
          if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1u; }
        }
        if (p.trace && rank == 0 && lane == 0) sg_trace(p, 0, ti, tr0, clock64(), wa, 0);
      }
    } else if (warp == 9 && rank == 0) {
      // ===== UMMA issuer: the leader CTA issues for the pair =====
      uint32_t stage = 0, ring_phase = 0, cc = 0;               // cc = k chunks so far: TMEM accumulator = cc & 1
      for (uint32_t ti = unit; ti < p.n_tiles; ti += n_units) {
        const SgTile t = p.tiles[ti];
        const SgProb* pr = p.probs + t.prob;
        if (pr->done != nullptr && *pr->done != 0u) continue;
        const uint32_t nkb = (pr->K + 63u) >> 6;
        const uint32_t a_mn = pr->a_mn, b_mn = pr->b_mn;
        const uint32_t idesc = ptx::idesc_bf16_f32(256, 256, a_mn, b_mn);
        const uint32_t a_step = a_mn ? (2048u >> 4) : (32u >> 4), b_step = b_mn ? (2048u >> 4) : (32u >> 4);
        const uint32_t a_lbo = a_mn ? 8192u : 16u, b_lbo = b_mn ? 8192u : 16u;
        const long long tr0 = p.trace ? clock64() : 0;
        long long wa = 0, wb = 0;
        for (uint32_t kb = 0; kb < nkb; ++kb) {
          const uint32_t buf = cc & 1u, use = cc >> 1;
          if (p.trace) {
            const long long c0 = clock64();
            ptx::mbar_wait(tempty0 + 8 * buf, (use & 1u) ^ 1u);
            const long long c1 = clock64();
            ptx::mbar_wait(full0 + 8 * stage, ring_phase);
            wa += c1 - c0; wb += clock64() - c1;
          } else {
          ptx::mbar_wait(tempty0 + 8 * buf, (use & 1u) ^ 1u);     // all 16 epilogue warps have folded this accumulator
          ptx::mbar_wait(full0 + 8 * stage, ring_phase);
          }
          ptx::tc_fence_after();
          const uint32_t d_tmem = tmem_base + buf * 256u;
          // Descriptors are formed in warp-uniform code and every UMMA of the block is unrolled with constant offsets
          // (always four k steps: a ragged last block reads TMA's zero fill), so that the elected lane issues from
          // uniform registers without per-instruction register moves (~200 cycles per UMMA otherwise: issue-bound).
          const uint32_t base = ring0 + stage * Cfg::kStage;
          uint64_t ad[AT], bd[BT];
#pragma unroll
          for (int i = 0; i < AT; ++i) ad[i] = ptx::smem_desc_sw128(base + i * kSgBox, a_lbo, 1024);
#pragma unroll
          for (int j = 0; j < BT; ++j) bd[j] = ptx::smem_desc_sw128(base + (AT + j) * kSgBox, b_lbo, 1024);
          if (ptx::elect_one()) {
            // the small term products first, the leading one last (see "Accumulation" above)
            bool first = true;
            {
#pragma unroll
            for (int i = 0; i < AT; ++i)
#pragma unroll
              for (int j = 0; j < BT; ++j)
                if (i + j <= Cfg::kOrder && i + j > 0) {
#pragma unroll
                  for (uint32_t ks = 0; ks < 4; ++ks) {
                    ptx::umma_bf16_cg2(d_tmem, ad[i] + (uint64_t)(ks * a_step), bd[j] + (uint64_t)(ks * b_step), idesc, first ? 0u : 1u);
                    first = false;
                  }
                }
#pragma unroll
            for (uint32_t ks = 0; ks < 4; ++ks) {
              ptx::umma_bf16_cg2(d_tmem, ad[0] + (uint64_t)(ks * a_step), bd[0] + (uint64_t)(ks * b_step), idesc, first ? 0u : 1u);
              first = false;
            }
            }
            ptx::umma_commit_cg2(empty0 + 8 * stage);
            ptx::umma_commit_cg2(tfull0 + 8 * buf);
          }
          __syncwarp();
          if (++stage == Cfg::kStages) { stage = 0; ring_phase ^= 1u; }
          ++cc;
        }
        if (p.trace && lane == 0) sg_trace(p, 1, ti, tr0, clock64(), wa, wb);
      }
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    // ===== epilogue: warps 0 .. 7; TMEM lane quarter q = warp % 4, column half = warp / 4 =====
    const uint32_t q = warp & 3u, half = warp >> 2;
    uint32_t cc = 0, n_st = 0;
    for (uint32_t ti = unit; ti < p.n_tiles; ti += n_units) {
      const SgTile t = p.tiles[ti];
      const SgProb* pr = p.probs + t.prob;
      if (pr->done != nullptr && *pr->done != 0u) continue;
      const uint32_t nkb = (pr->K + 63u) >> 6;
      const uint32_t row0 = t.m0 + rank * 128u + q * 32u, r = row0 + lane;
      const uint32_t n0 = t.n0 + half * 128u;
      const bool diag = pr->sym != 0u && t.n0 == t.m0;
      const bool mirror = pr->sym != 0u && t.n0 >= t.m0;
      float acc[128];
      const long long tr0 = p.trace ? clock64() : 0;
      long long wa = 0;
      for (uint32_t kb = 0; kb < nkb; ++kb) {
        const uint32_t buf = cc & 1u, use = cc >> 1;
        if (p.trace) { const long long c0 = clock64(); ptx::mbar_wait(tfull0 + 8 * buf, use & 1u); wa += clock64() - c0; }
        else ptx::mbar_wait(tfull0 + 8 * buf, use & 1u);
        ptx::tc_fence_after();
#pragma unroll
        for (int h = 0; h < 4; ++h) {
          uint32_t raw[32];
          ptx::tmem_ld32(tmem_base + ((q * 32u) << 16) + buf * 256u + half * 128u + 32u * h, raw);
          ptx::tmem_ld_wait();
          if (kb == 0) {
#pragma unroll
            for (int j = 0; j < 32; ++j) acc[32 * h + j] = __uint_as_float(raw[j]);
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) acc[32 * h + j] += __uint_as_float(raw[j]);
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive_cluster_relaxed(tempty_lead0 + 8 * buf);
        ++cc;
      }
      // (in a 256-wide diagonal tile a warp's 32 x 128 block may lie wholly below the diagonal: nothing is stored)
      const long long tr1 = p.trace ? clock64() : 0;
      sg_finish_row(pr, p, acc, row0, r, n0, mirror, diag, lane, ring0 + Cfg::kStages * Cfg::kStage + 256u + warp * (32u * 33u * 4u), n_st);
      if (p.trace && rank == 0 && warp == 0 && lane == 0) sg_trace(p, 2, ti, tr0, clock64(), wa, tr1 - tr0);
    }
    if (lane == 0) ptx::bulk_wait<0>();                        // this warp's TMA stores have been performed
  }

  __syncwarp();
  ptx::tc_fence_before();
  ptx::cluster_sync();
  if (warp == 9) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<512, 2>(tmem_base);
  }
}

}  // namespace mfsdp

#endif  // MFSDP_SGEMM3_CUH_
