// Newton-Schulz on the 5th-generation tensor cores (MFSDP_NS_BF16): grouped, persistent, warp-specialised GEMM
// tiles for ALL resident matrices of ragged shapes in one launch per phase and tile class.
//
// Per iteration and matrix (north_star), with Y the d x n "wide" view of X (Y = X when
// rows <= cols, Y = X^T otherwise -- the transposition is done by the UMMA operand descriptors (MN-major operands),
// never by moving data):
//   GRAM   A = alpha Y Y^T            symmetric: only blocks (I, J >= I) are computed, written and mirrored
//   POLY   P = a I + b A + c A A      symmetric, same tiling; the b A + a I terms are fused in the epilogue
//   APPLY  Y <- beta P Y              (the a X term of X <- a X + B X lives in P = aI + B)
// alpha = 1/||U||^2 and beta = 1/||U|| at iteration 0 (Frobenius normalisation folded in), 1 afterwards.
//
// Two tile classes share one kernel template (kCG = tcgen05 cta_group):
//   kCG = 2  matrices with d >= MFSDP_TUNE_PAIR_MIN_D: a CTA PAIR (cluster of two SMs of one TPC) owns a 256 x 256
//            output tile; each CTA stages its 128 rows of the A operand and its 128-column half of the B operand
//            (32 KB per 64-k stage instead of 48 KB per 128 x 256 tile -> 2/3 of the L2->smem traffic per flop),
//            the leader CTA issues tcgen05.mma.cta_group::2 (M = 256), 6-stage ring;
//   kCG = 1  small / ragged matrices: one CTA owns a 128 x (64..256) tile, 4-stage ring.
// Kernel anatomy (192 threads per CTA): warp 0 = TMA producer (one lane), warp 1 = TMEM owner + UMMA issuer (one
// lane, leader CTA only when paired), warps 2-5 = epilogue (TMEM -> registers -> global).  Two TMEM accumulator
// stages (2 x 256 columns) let the epilogue of tile t overlap the main loop of tile t + 1.
#include <cuda.h>
#include <cuda_bf16.h>

#include <algorithm>
#include <cstdlib>

#include "mfsdp_internal.h"
#include "ptx_sm100.cuh"

namespace mfsdp {

enum { PH_GRAM = 0, PH_POLY = 1, PH_APPLY = 2 };

struct TcMat {                 // device, one per matrix
  uint64_t x_off[2], a_off, p_off;
  uint32_t rows, cols, d, n_long, pitch_x, pitch_a, tall, pad;
};
// Output tile: origin (rows, cols of the OUTPUT buffer), k blocks, UMMA N (multiple of 64; of 128 when paired).
struct TcTile { uint32_t mat, m0, n0; uint16_t nkb, nw; };

struct NsTcPlan {
  CUtensorMap* d_tmaps = nullptr;   // 4 per matrix: X0, X1, A, P   (box 64 x 64 bf16, 128-byte swizzle)
  TcMat* d_mats = nullptr;
  TcTile* d_tiles[2][3] = {{nullptr, nullptr, nullptr}, {nullptr, nullptr, nullptr}};   // [kCG - 1][phase]
  uint32_t n_tiles[2][3] = {{0, 0, 0}, {0, 0, 0}};
  uint32_t* d_counters = nullptr;   // one tile counter per launch of a pass (zeroed at the start of every pass)
  int sms = 148;
  int max_pairs = 74;               // co-resident CTA pairs
};

namespace {

constexpr uint32_t kBM = 128;                  // UMMA M per CTA
constexpr uint32_t kBNMax = 256;               // max UMMA N per tile
constexpr uint32_t kBK = 64;                   // k elements per stage (one 128-byte swizzle row)
constexpr uint32_t kBoxBytes = 64 * 64 * 2;    // one TMA box: 64 rows x 128 B
constexpr uint32_t kABytes = 2 * kBoxBytes;    // 128 x 64
constexpr uint32_t kThreads = 192;
constexpr uint32_t kMaxLaunches = 64 * 3 * 2;   // ns_steps <= 64, three phases, two tile classes
constexpr uint32_t kTmemCols = 512;

template <int kCG>
struct Geo {
  static constexpr uint32_t kBBoxes = kCG == 1 ? 4 : 2;           // B-operand boxes per CTA and stage
  static constexpr uint32_t kBBytes = kBBoxes * kBoxBytes;
  static constexpr uint32_t kStageBytes = kABytes + kBBytes;      // 48 KB | 32 KB
  static constexpr uint32_t kStages = kCG == 1 ? 4 : 6;
  static constexpr uint32_t kTileM = kBM * kCG;                   // rows of the output tile
  static constexpr uint32_t kSmemBytes = kStages * kStageBytes + 1024 /*align slack*/ + 256 /*barriers*/;
};

struct TcParams {
  const TcTile* tiles;
  uint32_t n_tiles;
  const TcMat* mats;
  const CUtensorMap* tmaps;
  uint8_t* ws;
  const float* inv_norm;
  int phase, src, first;
  float a, b, c;
  uint32_t* counter;            // dynamic tile scheduler: next unclaimed tile of THIS launch (zero at launch)
  unsigned long long* trace;    // optional (mfsdp_debug_trace): [0] = record counter, then 4 words per tile
  uint32_t trace_cap, launch_idx;
};

struct TileCfg {
  const CUtensorMap *ta, *tb;
  uint32_t a_mn, b_mn;          // operand majorness (1 = MN-major)
  uint32_t a_ext;               // extent of the A operand's M dimension
  uint32_t out_rows, out_cols;  // bounds of the output buffer
};

__device__ __forceinline__ TileCfg decode(const TcParams& p, const TcTile& t, const TcMat& M) {
  TileCfg c;
  const CUtensorMap* tm = p.tmaps + 4 * (size_t)t.mat;
  if (p.phase == PH_GRAM) {
    c.ta = c.tb = tm + p.src; c.a_mn = c.b_mn = M.tall; c.a_ext = M.d; c.out_rows = c.out_cols = M.d;
  } else if (p.phase == PH_POLY) {
    c.ta = c.tb = tm + 2; c.a_mn = c.b_mn = 0; c.a_ext = M.d; c.out_rows = c.out_cols = M.d;
  } else if (!M.tall) {          // X_new (d x n) = P (K-major) * X (k x n, MN-major)
    c.ta = tm + 3; c.a_mn = 0; c.a_ext = M.d; c.tb = tm + p.src; c.b_mn = 1;
    c.out_rows = M.rows; c.out_cols = M.cols;
  } else {                       // X_new (n x d) = X (K-major) * P^T, P symmetric (K-major)
    c.ta = tm + p.src; c.a_mn = 0; c.a_ext = M.rows; c.tb = tm + 3; c.b_mn = 0;
    c.out_rows = M.rows; c.out_cols = M.cols;
  }
  return c;
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}

// ---- dynamic tile scheduler ------------------------------------------------------------------------------------
// The producer thread of a walking unit (CTA, or leader CTA of a pair) claims the next tile of the launch with one
// atomicAdd when it is ready to start loading it, and publishes the index through a small shared-memory ring
// (kFeed slots, full/empty mbarriers) to the other roles: UMMA issuer and epilogue warps of its own CTA and, when
// paired, the producer and epilogue warps of the peer CTA (remote store + remote arrive).  Tiles are therefore
// handed out in list order at the pace of the fastest units: the tiles in flight are always a contiguous window of
// the (rasterised) list, started at staggered times, and no unit idles while tiles remain.
constexpr uint32_t kFeed = 4;
constexpr uint32_t kNoTile = 0xffffffffu;

template <int kCG>
struct Feed {
  uint32_t full0, empty0, slots0;        // shared::cta addresses: full barriers, empty barriers (used by the leader), slots
  uint32_t empty_lead0;                  // the leader's empty barriers as a shared::cluster address (paired) / = empty0
  uint32_t s = 0, ph = 0;
  __device__ __forceinline__ void advance() { if (++s == kFeed) { s = 0; ph ^= 1; } }
  // leader producer: claim and publish.  Returns the tile index or kNoTile.
  __device__ __forceinline__ uint32_t claim(uint32_t* counter, uint32_t n_tiles) {
    ptx::mbar_wait(empty0 + 8 * s, ph ^ 1);                // every consumer has read the slot's previous content
    uint32_t ti = atomicAdd(counter, 1u);
    if (ti >= n_tiles) ti = kNoTile;
    ptx::st_shared_u32(slots0 + 4 * s, ti);
    if constexpr (kCG == 2) {
      ptx::st_shared_cluster_u32(ptx::mapa(slots0 + 4 * s, 1), ti);
      ptx::mbar_arrive_cluster(ptx::mapa(full0 + 8 * s, 1));
    }
    ptx::mbar_arrive(full0 + 8 * s);
    advance();
    return ti;
  }
  // any other role: wait for the next index ...
  __device__ __forceinline__ uint32_t peek() const {
    if constexpr (kCG == 2) ptx::mbar_wait_cluster(full0 + 8 * s, ph); else ptx::mbar_wait(full0 + 8 * s, ph);
    return ptx::ld_shared_u32(slots0 + 4 * s);
  }
  // ... and report the slot as consumed (`arrive`: one thread per role, after every thread of the role has read it).
  __device__ __forceinline__ void release(bool arrive) {
    if (arrive) {
      if constexpr (kCG == 2) ptx::mbar_arrive_cluster(empty_lead0 + 8 * s); else ptx::mbar_arrive(empty_lead0 + 8 * s);
    }
    advance();
  }
  __device__ __forceinline__ uint32_t next_single() {      // single-thread roles
    const uint32_t ti = peek();
    release(true);
    return ti;
  }
};

template <int kCG>
__global__ void __launch_bounds__(kThreads, 1) k_ns_tc(const TcParams p) {
  using G = Geo<kCG>;
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + G::kStages * G::kStageBytes);
  const uint32_t full0 = ptx::smem_u32(bars), empty0 = ptx::smem_u32(bars + G::kStages);
  const uint32_t tfull0 = ptx::smem_u32(bars + 2 * G::kStages), tempty0 = ptx::smem_u32(bars + 2 * G::kStages + 2);
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 2 * G::kStages + 4);
  Feed<kCG> feed;
  feed.full0 = ptx::smem_u32(bars + 2 * G::kStages + 5);
  feed.empty0 = ptx::smem_u32(bars + 2 * G::kStages + 5 + kFeed);
  feed.slots0 = ptx::smem_u32(bars + 2 * G::kStages + 5 + 2 * kFeed);
  const uint32_t stage0 = ptx::smem_u32(smem);
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = kCG == 2 ? ptx::cluster_ctarank() : 0u;          // 0 = leader of the pair
  const uint32_t unit = kCG == 2 ? blockIdx.x >> 1 : blockIdx.x;          // tile-walking unit: CTA or CTA pair
  feed.empty_lead0 = kCG == 2 ? ptx::mapa(feed.empty0, 0) : feed.empty0;

  if (threadIdx.x == 0) {
    for (uint32_t s = 0; s < G::kStages; ++s) { ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 1); }
    for (uint32_t s = 0; s < 2; ++s) { ptx::mbar_init(tfull0 + 8 * s, 1); ptx::mbar_init(tempty0 + 8 * s, 4 * kCG); }
    // feed consumers per slot: UMMA issuer + 4 epilogue warps of the leader, producer + 4 epilogue warps of the peer
    for (uint32_t s = 0; s < kFeed; ++s) { ptx::mbar_init(feed.full0 + 8 * s, 1); ptx::mbar_init(feed.empty0 + 8 * s, 5 * kCG); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc<kTmemCols, kCG>(ptx::smem_u32(tmem_holder));
  ptx::tc_fence_before();
  if constexpr (kCG == 2) ptx::cluster_sync(); else __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;

  if (warp == 0) {
    // ===== TMA producer (both CTAs of a pair; the bytes of both are counted on the leader's full barrier) =====
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      const uint32_t full_lead0 = kCG == 2 ? ptx::mapa(full0, 0) : full0;
      for (;;) {
        const uint32_t ti = rank == 0 ? feed.claim(p.counter, p.n_tiles) : feed.next_single();
        if (ti == kNoTile) break;
        const TcTile t = p.tiles[ti];
        const TcMat M = p.mats[t.mat];
        const TileCfg c = decode(p, t, M);
        const uint32_t am0 = t.m0 + rank * kBM;
        uint32_t a_boxes, b_boxes, bn0;
        if constexpr (kCG == 2) {      // fixed box counts (out-of-range boxes are zero-filled) keep the byte count static
          a_boxes = 2; b_boxes = t.nw >> 7; bn0 = t.n0 + rank * (t.nw >> 1);
        } else {
          a_boxes = (c.a_ext - t.m0 > 64u) ? 2u : 1u; b_boxes = t.nw >> 6; bn0 = t.n0;
        }
        const uint32_t tx = (a_boxes + b_boxes) * kBoxBytes * kCG;
        for (uint32_t kb = 0; kb < t.nkb; ++kb) {
          ptx::mbar_wait(empty0 + 8 * stage, phase ^ 1);
          if (rank == 0) ptx::mbar_arrive_expect_tx(full0 + 8 * stage, tx);
          const uint32_t fb = full_lead0 + 8 * stage;
          const uint32_t sa = stage0 + stage * G::kStageBytes, sb = sa + kABytes;
          const int k0 = (int)(kb * kBK);
          for (uint32_t h = 0; h < a_boxes; ++h) {
            const int mn = (int)(am0 + 64 * h);
            if constexpr (kCG == 2) ptx::tma_load_2d_cg2(sa + h * kBoxBytes, c.ta, c.a_mn ? mn : k0, c.a_mn ? k0 : mn, fb);
            else ptx::tma_load_2d(sa + h * kBoxBytes, c.ta, c.a_mn ? mn : k0, c.a_mn ? k0 : mn, fb);
          }
          for (uint32_t j = 0; j < b_boxes; ++j) {
            const int mn = (int)(bn0 + 64 * j);
            if constexpr (kCG == 2) ptx::tma_load_2d_cg2(sb + j * kBoxBytes, c.tb, c.b_mn ? mn : k0, c.b_mn ? k0 : mn, fb);
            else ptx::tma_load_2d(sb + j * kBoxBytes, c.tb, c.b_mn ? mn : k0, c.b_mn ? k0 : mn, fb);
          }
          if (++stage == G::kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== UMMA issuer (leader CTA only when paired) =====
    if (lane == 0 && rank == 0) {
      uint32_t stage = 0, phase = 0, acc = 0, acc_phase = 0;
      for (;;) {
        const uint32_t ti = feed.next_single();
        if (ti == kNoTile) break;
        const TcTile t = p.tiles[ti];
        const TcMat M = p.mats[t.mat];
        const TileCfg c = decode(p, t, M);
        const uint32_t idesc = ptx::idesc_bf16_f32(G::kTileM, t.nw, c.a_mn, c.b_mn);
        // K-major: +32 B per 16-k step; MN-major: +16 rows of 128 B.  (descriptor address field is in 16-byte units)
        const uint32_t a_step = c.a_mn ? (2048u >> 4) : (32u >> 4), b_step = c.b_mn ? (2048u >> 4) : (32u >> 4);
        const uint32_t a_lbo = c.a_mn ? kBoxBytes : 16u, b_lbo = c.b_mn ? kBoxBytes : 16u;
        ptx::mbar_wait(tempty0 + 8 * acc, acc_phase ^ 1);       // every epilogue warp has drained this accumulator
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * kBNMax;
        for (uint32_t kb = 0; kb < t.nkb; ++kb) {
          ptx::mbar_wait(full0 + 8 * stage, phase);
          ptx::tc_fence_after();
          const uint32_t sa = stage0 + stage * G::kStageBytes, sb = sa + kABytes;
          const uint64_t ad = ptx::smem_desc_sw128(sa, a_lbo, 1024), bd = ptx::smem_desc_sw128(sb, b_lbo, 1024);
#pragma unroll
          for (uint32_t ks = 0; ks < kBK / 16; ++ks) {
            if constexpr (kCG == 2)
              ptx::umma_bf16_cg2(d_tmem, ad + (uint64_t)(ks * a_step), bd + (uint64_t)(ks * b_step), idesc, (kb | ks) != 0);
            else
              ptx::umma_bf16(d_tmem, ad + (uint64_t)(ks * a_step), bd + (uint64_t)(ks * b_step), idesc, (kb | ks) != 0);
          }
          // frees the smem slot (in both CTAs when paired) once these MMAs have finished
          if constexpr (kCG == 2) ptx::umma_commit_cg2(empty0 + 8 * stage); else ptx::umma_commit(empty0 + 8 * stage);
          if (++stage == G::kStages) { stage = 0; phase ^= 1; }
        }
        // accumulator ready for the epilogue warps (of both CTAs)
        if constexpr (kCG == 2) ptx::umma_commit_cg2(tfull0 + 8 * acc); else ptx::umma_commit(tfull0 + 8 * acc);
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
    }
  } else {
    // ===== epilogue: warps 2..5, warp w owns TMEM lanes 32 (w % 4) .. + 31 =====
    const uint32_t q = warp & 3;
    uint32_t acc = 0, acc_phase = 0;
    const uint32_t tempty_lead0 = kCG == 2 ? ptx::mapa(tempty0, 0) : tempty0;
    for (;;) {
      const uint32_t ti = feed.peek();
      __syncwarp();
      feed.release(lane == 0);
      if (ti == kNoTile) break;
      const TcTile t = p.tiles[ti];
      const TcMat M = p.mats[t.mat];
      const TileCfg c = decode(p, t, M);
      const float inv = p.first ? p.inv_norm[t.mat] : 1.f;
      const float alpha = p.phase == PH_GRAM ? inv * inv : inv;
      const uint32_t rb0 = t.m0 + rank * kBM;                    // first output row of this CTA
      const uint32_t r = rb0 + q * 32 + lane;                    // output row of this thread
      const bool row_ok = r < c.out_rows;
      __nv_bfloat16* out;
      uint32_t pitch;
      if (p.phase == PH_GRAM) { out = reinterpret_cast<__nv_bfloat16*>(p.ws + M.a_off); pitch = M.pitch_a; }
      else if (p.phase == PH_POLY) { out = reinterpret_cast<__nv_bfloat16*>(p.ws + M.p_off); pitch = M.pitch_a; }
      else { out = reinterpret_cast<__nv_bfloat16*>(p.ws + M.x_off[p.src ^ 1]); pitch = M.pitch_x; }
      const __nv_bfloat16* Ain = reinterpret_cast<const __nv_bfloat16*>(p.ws + M.a_off);
      const bool sym = p.phase != PH_APPLY;

      ptx::mbar_wait(tfull0 + 8 * acc, acc_phase);
      ptx::tc_fence_after();
      const unsigned long long t_ready = p.trace ? ptx::globaltimer() : 0ull;
      const uint32_t taddr0 = tmem_base + ((q * 32u) << 16) + acc * kBNMax;
      for (uint32_t c0 = 0; c0 < t.nw; c0 += 32) {
        const uint32_t col0 = t.n0 + c0;
        if (col0 >= c.out_cols) break;                           // warp-uniform
        // symmetric outputs: a 128-block below the diagonal is the mirror image of one that is written from above
        if (sym && (col0 >> 7) < (rb0 >> 7)) continue;           // warp-uniform
        uint32_t v[32];
        ptx::tmem_ld32(taddr0 + c0, v);
        ptx::tmem_ld_wait();
        float f[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) f[j] = __uint_as_float(v[j]);
        const bool full_cols = col0 + 32 <= c.out_cols;
        if (p.phase == PH_POLY) {
          if (row_ok) {
            const __nv_bfloat16* arow = Ain + (size_t)r * pitch + col0;
            if (full_cols) {
#pragma unroll
              for (int g4 = 0; g4 < 4; ++g4) {
                const uint4 u = *reinterpret_cast<const uint4*>(arow + 8 * g4);
                const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                  const int j = 8 * g4 + 2 * i;
                  f[j] = fmaf(p.c, f[j], p.b * __uint_as_float(w[i] << 16));
                  f[j + 1] = fmaf(p.c, f[j + 1], p.b * __uint_as_float(w[i] & 0xffff0000u));
                }
              }
            } else {
              for (int j = 0; j < 32; ++j)
                if (col0 + j < c.out_cols) f[j] = fmaf(p.c, f[j], p.b * __bfloat162float(arow[j]));
            }
            if (r >= col0 && r < col0 + 32) {                    // the diagonal element: + a
#pragma unroll
              for (int j = 0; j < 32; ++j) if (col0 + j == r) f[j] += p.a;
            }
          }
        } else {
#pragma unroll
          for (int j = 0; j < 32; ++j) f[j] *= alpha;
        }
        // direct write: row r, columns col0 .. col0 + 31
        if (row_ok) {
          __nv_bfloat16* orow = out + (size_t)r * pitch + col0;
          if (full_cols) {
#pragma unroll
            for (int g4 = 0; g4 < 4; ++g4) {
              uint4 u;
              u.x = pack_bf16(f[8 * g4 + 0], f[8 * g4 + 1]); u.y = pack_bf16(f[8 * g4 + 2], f[8 * g4 + 3]);
              u.z = pack_bf16(f[8 * g4 + 4], f[8 * g4 + 5]); u.w = pack_bf16(f[8 * g4 + 6], f[8 * g4 + 7]);
              *reinterpret_cast<uint4*>(orow + 8 * g4) = u;
            }
          } else {
            for (int j = 0; j < 32; ++j)
              if (col0 + j < c.out_cols) orow[j] = __float2bfloat16_rn(f[j]);
          }
        }
        // mirrored write of strictly-upper 128-blocks (lanes = consecutive r -> 64-byte runs)
        if (sym && (col0 >> 7) > (rb0 >> 7) && row_ok) {
#pragma unroll
          for (int j = 0; j < 32; ++j)
            if (col0 + j < c.out_cols) out[(size_t)(col0 + j) * pitch + r] = __float2bfloat16_rn(f[j]);
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (p.trace && q == 0 && lane == 0 && rank == 0) {         // one record per tile: when its accumulator was ready
        const unsigned long long slot = atomicAdd(p.trace, 1ull);   // and when this warp had stored its share
        if (slot < p.trace_cap) {
          unsigned long long* rec = p.trace + 1 + 4 * slot;
          rec[0] = ((unsigned long long)p.launch_idx << 32) | ti;
          rec[1] = ((unsigned long long)unit << 32) | ptx::smid();
          rec[2] = t_ready;
          rec[3] = ptx::globaltimer();
        }
      }
      if (lane == 0) {
        if constexpr (kCG == 2) ptx::mbar_arrive_cluster(tempty_lead0 + 8 * acc); else ptx::mbar_arrive(tempty0 + 8 * acc);
      }
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
  }

  __syncwarp();
  ptx::tc_fence_before();
  if constexpr (kCG == 2) ptx::cluster_sync(); else __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<kTmemCols, kCG>(tmem_base);
  }
}

// ---- host: tensor maps, tile lists ------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(sym);
  }
  return fn;
}

// Row-major bf16 matrix rows x cols with row pitch `pitch` elements; box = 64 (inner) x 64 (outer), 128-byte swizzle,
// out-of-bounds elements read as zero (ragged edges, partial k blocks and whole out-of-range boxes rely on it).
int make_tmap(CUtensorMap* out, void* base, uint32_t rows, uint32_t cols, uint32_t pitch) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return cuda_fail(cudaErrorSymbolNotFound);
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {(cuuint64_t)pitch * 2};
  const cuuint32_t box[2] = {64, 64};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? MFSDP_OK : cuda_fail(cudaErrorInvalidValue);
}

// Tile rasterisation.  The units (CTAs or CTA pairs) claim tiles in list order, so at any moment the tiles in
// flight are a contiguous window of about n_units list entries, started at staggered times: entry j + s starts about
// s / n_units of a tile duration after entry j.  An operand box fetched from DRAM by one tile is re-read from L2 by
// the tiles that share it as long as the next sharer follows soon enough.  The list is therefore ordered so that a
// window covers a compact block of the output (`band` row blocks x the column tiles that go with them) and sharers
// are few entries apart: column-panel sharers adjacent, row-panel sharers `band` entries apart.
uint16_t tile_n(uint32_t remaining, uint32_t gran) {     // UMMA N of a tile that has `remaining` columns to cover
  return (uint16_t)std::min(kBNMax, (remaining + gran - 1) / gran * gran);
}
// rectangular output (APPLY): column panels of `group` tiles stay L2-resident while all row blocks sweep over them.
void tiles_rect(std::vector<TcTile>& v, uint32_t mat, uint32_t out_rows, uint32_t out_cols, uint32_t nkb, uint32_t cg) {
  const uint32_t bm = kBM * cg;
  const uint32_t tm = (out_rows + bm - 1) / bm, tn = (out_cols + kBNMax - 1) / kBNMax;
  const uint32_t group = (uint32_t)std::max(1, tune_value(MFSDP_TUNE_RECT_GROUP));
  for (uint32_t g0 = 0; g0 < tn; g0 += group)
    for (uint32_t i = 0; i < tm; ++i)
      for (uint32_t j = g0; j < std::min(tn, g0 + group); ++j)
        v.push_back(TcTile{mat, i * bm, j * kBNMax, (uint16_t)nkb, tile_n(out_cols - j * kBNMax, 64 * cg)});
}
// symmetric output (GRAM, POLY): upper row blocks only; bands of `band` row blocks, inside a band column-major
// (all row blocks of the band for one 256-column step, then the next step).
void tiles_sym(std::vector<TcTile>& v, uint32_t mat, uint32_t d, uint32_t nkb, uint32_t cg) {
  const uint32_t bm = kBM * cg;
  const uint32_t tm = (d + bm - 1) / bm;
  const uint32_t band = (uint32_t)std::max(1, tune_value(cg == 2 ? MFSDP_TUNE_SYM_BAND2 : MFSDP_TUNE_SYM_BAND));
  for (uint32_t b0 = 0; b0 < tm; b0 += band) {
    const uint32_t b1 = std::min(tm, b0 + band);
    for (uint32_t c0 = b0 * bm; c0 < d; c0 += kBNMax)            // 256-column steps from the band's first diagonal
      for (uint32_t i = b0; i < b1; ++i) {
        // row block i owns columns >= i * bm; clip the step to that range (128 x 256 tiles: N = 128 when only half
        // of the step is owned; 256 x 256 tiles are aligned with the steps)
        const uint32_t lo = std::max(c0, i * bm);
        const uint32_t hi = std::min(d, c0 + kBNMax);
        if (lo >= hi) continue;
        v.push_back(TcTile{mat, i * bm, lo, (uint16_t)nkb, tile_n(hi - lo, 64 * cg)});
      }
  }
}

template <typename T>
int dev_upload(T** dptr, const std::vector<T>& h) {
  *dptr = nullptr;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(dptr), std::max<size_t>(1, h.size()) * sizeof(T));
  if (e != cudaSuccess) return cuda_fail(e);
  if (!h.empty()) {
    e = cudaMemcpy(*dptr, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(e);
  }
  return MFSDP_OK;
}

template <int kCG>
cudaError_t launch_phase(const TcParams& p, uint32_t units, cudaStream_t st) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(units * kCG);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = Geo<kCG>::kSmemBytes;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = kCG; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_ns_tc<kCG>, p);
}

int build_tc_plan(Plan& pl) {
  NsTcPlan* tc = new NsTcPlan();
  pl.tc = tc;
  const WsLayout& lay = pl.lay;
  uint8_t* ws = static_cast<uint8_t*>(pl.workspace);
  std::vector<CUtensorMap> maps(4 * lay.mats.size());
  std::vector<TcMat> mats(lay.mats.size());
  std::vector<TcTile> tiles[2][3];
  // big matrices first so that the static round-robin over units ends with the cheap tiles
  std::vector<uint32_t> order(lay.mats.size());
  for (uint32_t i = 0; i < order.size(); ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](uint32_t x, uint32_t y) {
    const MatLayout &a = lay.mats[x], &b = lay.mats[y];
    return (uint64_t)a.d * a.d * a.n_long > (uint64_t)b.d * b.d * b.n_long;
  });
  for (uint32_t i = 0; i < lay.mats.size(); ++i) {
    const MatLayout& L = lay.mats[i];
    TcMat& m = mats[i];
    m.x_off[0] = L.x_off[0]; m.x_off[1] = L.x_off[1]; m.a_off = L.a_off; m.p_off = L.p_off;
    m.rows = L.rows; m.cols = L.cols; m.d = L.d; m.n_long = L.n_long; m.pitch_x = L.pitch_x; m.pitch_a = L.pitch_a;
    m.tall = L.tall; m.pad = 0;
    int rc;
    if ((rc = make_tmap(&maps[4 * i + 0], ws + L.x_off[0], L.rows, L.cols, L.pitch_x)) ||
        (rc = make_tmap(&maps[4 * i + 1], ws + L.x_off[1], L.rows, L.cols, L.pitch_x)) ||
        (rc = make_tmap(&maps[4 * i + 2], ws + L.a_off, L.d, L.d, L.pitch_a)) ||
        (rc = make_tmap(&maps[4 * i + 3], ws + L.p_off, L.d, L.d, L.pitch_a)))
      return rc;
  }
  const uint32_t pair_min_d = (uint32_t)std::max(1, tune_value(MFSDP_TUNE_PAIR_MIN_D));
  for (uint32_t i : order) {
    const MatLayout& L = lay.mats[i];
    const uint32_t cg = L.d >= pair_min_d ? 2u : 1u;
    tiles_sym(tiles[cg - 1][PH_GRAM], i, L.d, (L.n_long + kBK - 1) / kBK, cg);
    tiles_sym(tiles[cg - 1][PH_POLY], i, L.d, (L.d + kBK - 1) / kBK, cg);
    tiles_rect(tiles[cg - 1][PH_APPLY], i, L.rows, L.cols, (L.d + kBK - 1) / kBK, cg);
  }
  int rc;
  if ((rc = dev_upload(&tc->d_tmaps, maps)) || (rc = dev_upload(&tc->d_mats, mats))) return rc;
  for (int g = 0; g < 2; ++g)
    for (int ph = 0; ph < 3; ++ph) {
      tc->n_tiles[g][ph] = (uint32_t)tiles[g][ph].size();
      if ((rc = dev_upload(&tc->d_tiles[g][ph], tiles[g][ph]))) return rc;
    }
  cudaDeviceGetAttribute(&tc->sms, cudaDevAttrMultiProcessorCount, pl.device);
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&tc->d_counters), kMaxLaunches * sizeof(uint32_t));
  if (e != cudaSuccess) return cuda_fail(e);
  e = cudaFuncSetAttribute(k_ns_tc<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Geo<1>::kSmemBytes);
  if (e != cudaSuccess) return cuda_fail(e);
  e = cudaFuncSetAttribute(k_ns_tc<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)Geo<2>::kSmemBytes);
  if (e != cudaSuccess) return cuda_fail(e);
  // how many CTA pairs can be co-resident (one CTA per SM; the two CTAs of a pair share a TPC)
  {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)tc->sms / 2 * 2);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = Geo<2>::kSmemBytes;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, k_ns_tc<2>, &cfg) == cudaSuccess && n > 0) tc->max_pairs = std::min(n, tc->sms / 2);
    else { cudaGetLastError(); tc->max_pairs = std::max(1, tc->sms / 2); }
  }
  return MFSDP_OK;
}

}  // namespace

void destroy_ns_tc(NsTcPlan* p) {
  if (!p) return;
  cudaFree(p->d_tmaps); cudaFree(p->d_mats); cudaFree(p->d_counters);
  for (int g = 0; g < 2; ++g)
    for (int ph = 0; ph < 3; ++ph) cudaFree(p->d_tiles[g][ph]);
  delete p;
}

int launch_ns_tc(Plan& pl, const mfsdp_muon_hparams_t& hp, cudaStream_t st) {
  if (pl.lay.mats.empty()) return MFSDP_OK;
  if (!pl.tc) {
    const int rc = build_tc_plan(pl);
    if (rc) { destroy_ns_tc(pl.tc); pl.tc = nullptr; return rc; }
  }
  NsTcPlan& tc = *pl.tc;
  TcParams p;
  p.mats = tc.d_mats; p.tmaps = tc.d_tmaps;
  p.ws = static_cast<uint8_t*>(pl.workspace);
  p.inv_norm = reinterpret_cast<const float*>(p.ws + pl.lay.invn_off);
  p.a = (float)hp.a; p.b = (float)hp.b; p.c = (float)hp.c;
  get_trace(&p.trace, &p.trace_cap);
  p.launch_idx = 0;
  {
    const cudaError_t e = cudaMemsetAsync(tc.d_counters, 0, kMaxLaunches * sizeof(uint32_t), st);
    if (e != cudaSuccess) return cuda_fail(e);
  }
  for (int it = 0; it < hp.ns_steps; ++it) {
    p.src = it & 1;
    p.first = (it == 0);
    for (int ph = 0; ph < 3; ++ph) {
      p.phase = ph;
      // the two tile classes touch disjoint matrices: their launches of one phase are independent
      for (int g = 1; g >= 0; --g) {
        p.tiles = tc.d_tiles[g][ph];
        p.n_tiles = tc.n_tiles[g][ph];
        if (p.n_tiles == 0) continue;
        p.counter = tc.d_counters + p.launch_idx;
        cudaError_t e;
        if (g == 1) e = launch_phase<2>(p, std::min<uint32_t>(p.n_tiles, (uint32_t)tc.max_pairs), st);
        else e = launch_phase<1>(p, std::min<uint32_t>(p.n_tiles, (uint32_t)tc.sms), st);
        if (e != cudaSuccess) return cuda_fail(e);
        ++p.launch_idx;
        count_launch();
        const int rc = check_last_launch();
        if (rc) return rc;
      }
    }
  }
  return MFSDP_OK;
}

}  // namespace mfsdp
