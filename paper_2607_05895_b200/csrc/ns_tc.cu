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
//   kCG = 2  matrices with d >= MFSDP_TUNE_PAIR_MIN_D: a CTA PAIR (cluster of two SMs of one TPC) owns a 256 x 512
//            output tile held as two 256-column TMEM accumulators.  Per 64-k stage a CTA stages its 128 rows of the
//            A operand and its half of both 256-column B panels (48 KB): 171 flop per byte fetched from L2, which
//            is what the measured L2->SM ceiling (~7 KB/clk chip-wide) needs to keep the tensor pipes busy (a
//            256 x 256 tile has 128 flop/B and measured 75 % pipe utilisation, L2-bound).  The leader CTA issues
//            tcgen05.mma.cta_group::2 (M = 256, N = 256) for the two halves in turn; the halves finish 4 MMAs
//            apart, so the epilogue of half 0 starts while half 1 still runs, and the next tile's MMAs into a half
//            start as soon as that half has been drained.
//   kCG = 1  small / ragged matrices: one CTA owns a 128 x (64..256) tile, two accumulator stages alternate
//            between tiles (the epilogue of tile t overlaps the main loop of tile t + 1).
// Kernel anatomy (224 threads per CTA): warp 0 = TMA producer, warp 1 = TMEM owner + UMMA issuer (leader CTA only when
// paired) -- both run their loops converged with one elected lane issuing --, warps 2-5 = epilogue: TMEM -> registers
// -> fused scale / polynomial -> bf16 -> swizzled shared-memory staging -> TMA tensor stores (direct tile and, for the
// symmetric phases, the transposed mirror tile), warp 6 = tile scheduler (leader CTA, one lane).  4-stage operand ring.
//
// One launch per tile class walks the tiles of ALL iterations and phases: the scheduler claims tiles from a global
// counter in list order, waits until the tile's inputs (every tile of the same matrix in the preceding phases) have
// been reported complete through a per-matrix counter, and publishes the index to the other roles through a
// shared-memory ring.
//
// On the last iteration the APPLY epilogue can also apply the weight update W <- W (1 - lr wd) - lr s O from the O tile
// it holds (UpdArgs; bf16 weights, every cols % 8 == 0) and copy the new W to a fan-out destination; O is then stored
// only on request.  Small matrices do not come here at all: d <= 128 runs in ns_fused.cu, 128 < d <= 256 (n <= 512) in
// ns_fused2.cu (one CTA per matrix for all iterations); the classes of one pass run concurrently on forked streams.
#include <cuda.h>
#include <cuda_bf16.h>

#include <algorithm>
#include <cstdlib>

#include "mfsdp_internal.h"
#include "ns_plan.h"
#include "ptx_sm100.cuh"

namespace mfsdp {

namespace {

constexpr uint32_t kBM = 128;                  // UMMA M per CTA
constexpr uint32_t kBN = 256;                  // UMMA N = columns of one TMEM accumulator
constexpr uint32_t kBK = 64;                   // k elements per stage (one 128-byte swizzle row)
constexpr uint32_t kBoxBytes = 64 * 64 * 2;    // one TMA box: 64 rows x 128 B
constexpr uint32_t kABytes = 2 * kBoxBytes;    // 128 x 64
constexpr uint32_t kBBytes = 4 * kBoxBytes;    // single CTA: 256 x 64; paired: 2 halves x (128 x 64)
constexpr uint32_t kStageBytes = kABytes + kBBytes;   // 48 KB
constexpr uint32_t kStages = 4;
constexpr uint32_t kPairGroup = 2;             // CTA-pair class: ring stages consumed per accumulator visit
constexpr uint32_t kThreads = 224;   // producer, UMMA issuer, 4 epilogue warps, tile scheduler
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kEpiBufBytes = 4096;        // one staging tile: 32 rows x 64 cols (or 64 x 32 transposed) bf16
constexpr uint32_t kEpiBytes = 4 * 2 * kEpiBufBytes;   // 4 epilogue warps x 2 buffers
constexpr uint32_t kBarBytes = 512;            // mbarriers, TMEM address, scheduler feed slots
constexpr uint32_t kSmemBytes = kStages * kStageBytes + kEpiBytes + kBarBytes + 1024 /*align slack*/;

struct TcParams {
  const TcTile* tiles;
  uint32_t n_tiles;
  const TcMat* mats;
  const CUtensorMap* tmaps;
  uint8_t* ws;
  const float* inv_norm;
  uint32_t n_iter_tiles, ns_steps;   // the launch walks ns_steps x n_iter_tiles tiles (iteration-major)
  float a, b, c;
  uint32_t* counter;            // dynamic tile scheduler: next unclaimed tile of THIS launch (zero at launch)
  uint32_t* done;               // [n_mat] completion reports of the pass so far (zero at the start of the pass)
  unsigned long long* trace;    // optional (mfsdp_debug_trace): [0] = record counter, then 6 words per tile
  uint32_t trace_cap, launch_idx;
  UpdArgs ua;                   // weight update fused into the APPLY epilogue of the last iteration (ua.W != nullptr)
};

struct TileCfg {
  const CUtensorMap *ta, *tb;   // operand loads
  const CUtensorMap *tout, *tmir, *tain;   // epilogue: output tile, mirror tile (symmetric phases), A tile (POLY)
  uint32_t a_mn, b_mn;          // operand majorness (1 = MN-major)
  uint32_t a_ext;               // extent of the A operand's M dimension
  uint32_t out_rows, out_cols;  // bounds of the output buffer
};

// One claimed unit of work: tile j of iteration it.
struct Work { TcTile t; uint32_t it, src, first; };
__device__ __forceinline__ Work fetch(const TcParams& p, uint32_t ti) {
  Work w;
  w.it = ti / p.n_iter_tiles;
  w.t = p.tiles[ti - w.it * p.n_iter_tiles];
  w.src = w.it & 1u;
  w.first = w.it == 0u;
  return w;
}

__device__ __forceinline__ TileCfg decode(const TcParams& p, const TcTile& t, const TcMat& M, uint32_t src) {
  TileCfg c;
  const CUtensorMap* tm = p.tmaps + TM_COUNT * (size_t)t.mat;
  c.tmir = nullptr; c.tain = tm + TM_A_ST;
  if (t.phase == PH_GRAM) {
    c.ta = c.tb = tm + src; c.a_mn = c.b_mn = M.tall; c.a_ext = M.d; c.out_rows = c.out_cols = M.d;
    c.tout = tm + TM_A_ST; c.tmir = tm + TM_A_MIR;
  } else if (t.phase == PH_POLY) {
    c.ta = c.tb = tm + TM_A; c.a_mn = c.b_mn = 0; c.a_ext = M.d; c.out_rows = c.out_cols = M.d;
    c.tout = tm + TM_P_ST; c.tmir = tm + TM_P_MIR;
  } else if (!M.tall) {          // X_new (d x n) = P (K-major) * X (k x n, MN-major)
    c.ta = tm + TM_P; c.a_mn = 0; c.a_ext = M.d; c.tb = tm + src; c.b_mn = 1;
    c.out_rows = M.rows; c.out_cols = M.cols; c.tout = tm + TM_X0_ST + (src ^ 1);
  } else {                       // X_new (n x d) = X (K-major) * P^T, P symmetric (K-major)
    c.ta = tm + src; c.a_mn = 0; c.a_ext = M.rows; c.tb = tm + TM_P; c.b_mn = 0;
    c.out_rows = M.rows; c.out_cols = M.cols; c.tout = tm + TM_X0_ST + (src ^ 1);
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
  // leader producer: claim ...
  __device__ __forceinline__ uint32_t claim(uint32_t* counter, uint32_t n_tiles) {
    const uint32_t ti = atomicAdd(counter, 1u);
    return ti < n_tiles ? ti : kNoTile;
  }
  // ... and publish it with its descriptors (after the tile's inputs are known to be complete).  A slot is 16 words:
  // the TcTile (word 7 = the claimed index or kNoTile), the iteration, and the matrix fields the roles need -- so that
  // no consumer has to chase tile / matrix tables through global memory at the start of every tile.
  __device__ __forceinline__ void publish(uint32_t ti, const Work& w, const TcMat& M) {
    ptx::mbar_wait(empty0 + 8 * s, ph ^ 1);                // every consumer has read the slot's previous content
    uint32_t v[16];
    v[0] = w.t.mat; v[1] = w.t.m0; v[2] = w.t.n0; v[3] = (uint32_t)w.t.nkb | ((uint32_t)w.t.nw << 16);
    v[4] = w.t.need; v[5] = w.t.phase; v[6] = w.t.reports_per_iter; v[7] = ti;
    v[8] = w.it; v[9] = M.rows; v[10] = M.cols; v[11] = M.d; v[12] = M.tall; v[13] = M.pitch_a;
    v[14] = (uint32_t)M.a_off; v[15] = (uint32_t)(M.a_off >> 32);
    const uint32_t slot = slots0 + 64 * s;
#pragma unroll
    for (int i = 0; i < 4; ++i) ptx::st_shared_v4(slot + 16 * i, v[4 * i], v[4 * i + 1], v[4 * i + 2], v[4 * i + 3]);
    if constexpr (kCG == 2) {
      const uint32_t rslot = ptx::mapa(slot, 1);
#pragma unroll
      for (int i = 0; i < 16; ++i) ptx::st_shared_cluster_u32(rslot + 4 * i, v[i]);
      ptx::mbar_arrive_cluster(ptx::mapa(full0 + 8 * s, 1));
    }
    ptx::mbar_arrive(full0 + 8 * s);
    advance();
  }
  // has the next index been published? (non-blocking)
  __device__ __forceinline__ bool ready() const {
    if constexpr (kCG == 2) return ptx::mbar_try_wait_cluster(full0 + 8 * s, ph) != 0;
    else return ptx::mbar_try_wait(full0 + 8 * s, ph) != 0;
  }
  // any other role: wait for the next index ...
  __device__ __forceinline__ uint32_t peek() const {
    if constexpr (kCG == 2) ptx::mbar_wait_cluster(full0 + 8 * s, ph); else ptx::mbar_wait(full0 + 8 * s, ph);
    return ptx::ld_shared_u32(slots0 + 64 * s + 28);
  }
  // ... read its descriptors (before release) ...
  __device__ __forceinline__ void read(Work& w, TcMat& M) const {
    uint32_t a[4], b[4], c[4], d[4];
    const uint32_t slot = slots0 + 64 * s;
    ptx::ld_shared_v4(slot, a[0], a[1], a[2], a[3]);
    ptx::ld_shared_v4(slot + 16, b[0], b[1], b[2], b[3]);
    ptx::ld_shared_v4(slot + 32, c[0], c[1], c[2], c[3]);
    ptx::ld_shared_v4(slot + 48, d[0], d[1], d[2], d[3]);
    w.t.mat = a[0]; w.t.m0 = a[1]; w.t.n0 = a[2]; w.t.nkb = (uint16_t)(a[3] & 0xffffu); w.t.nw = (uint16_t)(a[3] >> 16);
    w.t.need = b[0]; w.t.phase = b[1]; w.t.reports_per_iter = b[2]; w.t.pad = 0;
    w.it = c[0]; w.src = c[0] & 1u; w.first = c[0] == 0u;
    M.rows = c[1]; M.cols = c[2]; M.d = c[3]; M.tall = d[0]; M.pitch_a = d[1];
    M.a_off = (uint64_t)d[2] | ((uint64_t)d[3] << 32);
  }
  // ... and report the slot as consumed (`arrive`: one thread per role, after every thread of the role has read it).
  __device__ __forceinline__ void release(bool arrive) {
    if (arrive) {
      if constexpr (kCG == 2) ptx::mbar_arrive_cluster(empty_lead0 + 8 * s); else ptx::mbar_arrive(empty_lead0 + 8 * s);
    }
    advance();
  }
};

template <int kCG>
__global__ void __launch_bounds__(kThreads, 1) k_ns_tc(const TcParams p) {
  constexpr uint32_t kGroup = kCG == 2 ? kPairGroup : 1;   // ring stages per accumulator visit
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  // [operand ring: kStages x 48 KB][epilogue staging: 4 warps x 2 x 4 KB][barriers]
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kStages * kStageBytes + kEpiBytes);
  const uint32_t full0 = ptx::smem_u32(bars), empty0 = ptx::smem_u32(bars + kStages);
  const uint32_t tfull0 = ptx::smem_u32(bars + 2 * kStages), tempty0 = ptx::smem_u32(bars + 2 * kStages + 2);
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 2 * kStages + 4);
  Feed<kCG> feed;
  feed.full0 = ptx::smem_u32(bars + 2 * kStages + 5);
  feed.empty0 = ptx::smem_u32(bars + 2 * kStages + 5 + kFeed);
  feed.slots0 = ptx::smem_u32(bars) + 256;          // kFeed slots of 64 bytes in the second half of the region
  const uint32_t prod_done = ptx::smem_u32(bars + 2 * kStages + 5 + 2 * kFeed);   // tiles whose loads the producer has issued
  const uint32_t stage0 = ptx::smem_u32(smem);
  const uint32_t epi0 = stage0 + kStages * kStageBytes;
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = kCG == 2 ? ptx::cluster_ctarank() : 0u;          // 0 = leader of the pair
  const uint32_t unit = kCG == 2 ? blockIdx.x >> 1 : blockIdx.x;          // tile-walking unit: CTA or CTA pair
  feed.empty_lead0 = kCG == 2 ? ptx::mapa(feed.empty0, 0) : feed.empty0;

  if (threadIdx.x == 0) {
    for (uint32_t s = 0; s < kStages; ++s) { ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 1); }
    for (uint32_t s = 0; s < 2; ++s) { ptx::mbar_init(tfull0 + 8 * s, 1); ptx::mbar_init(tempty0 + 8 * s, 4 * kCG); }
    // feed consumers per slot: producer + UMMA issuer + 4 epilogue warps of the leader, producer + 4 epilogue warps of
    // the peer
    for (uint32_t s = 0; s < kFeed; ++s) { ptx::mbar_init(feed.full0 + 8 * s, 1); ptx::mbar_init(feed.empty0 + 8 * s, kCG == 2 ? 11 : 6); }
    ptx::st_shared_volatile_u32(prod_done, 0u);
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc<kTmemCols, kCG>(ptx::smem_u32(tmem_holder));
  ptx::tc_fence_before();
  if constexpr (kCG == 2) ptx::cluster_sync(); else __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;

  if (warp == 0) {
    // ===== TMA producer (both CTAs of a pair; the bytes of both are counted on the leader's full barrier).  Like the
    // UMMA warp it runs converged with one elected lane issuing (uniform-register operands without election loops:
    // the single-lane version spent ~700 cycles per k block issuing 4-6 loads).  Tiles come from the scheduler warp. =====
    {
      uint32_t stage = 0, phase = 0, n_done = 0;
      const uint32_t full_lead0 = kCG == 2 ? ptx::mapa(full0, 0) : full0;
      for (;;) {
        const uint32_t ti = __shfl_sync(0xffffffffu, feed.peek(), 0);
        Work w;
        TcMat M;
        feed.read(w, M);
        __syncwarp();
        feed.release(lane == 0);
        if (ti == kNoTile) break;
        ptx::fence_proxy_async();          // reported (generic-proxy) completion -> this thread's TMA reads
        const TcTile t = w.t;
        const TileCfg c = decode(p, t, M, w.src);
        const uint32_t am0 = t.m0 + rank * kBM;
        // B boxes of this CTA: single CTA: nw / 64 consecutive boxes.  Paired: per 256-column half h its own half of
        // the panel, nh / 128 boxes (nh = width of the half), stored at box slot 2 h + j.
        uint32_t a_boxes, n_b = 0, b_mask = 0;
        uint32_t b_col[4];
        if constexpr (kCG == 2) {      // fixed box counts (out-of-range boxes are zero-filled) keep the byte count static
          a_boxes = 2;
#pragma unroll
          for (uint32_t h = 0; h < 2; ++h) {
            const uint32_t nh = h * kBN < t.nw ? min((uint32_t)t.nw - h * kBN, kBN) : 0u;
#pragma unroll
            for (uint32_t j = 0; j < 2; ++j) {
              b_col[2 * h + j] = t.n0 + h * kBN + rank * (nh >> 1) + 64 * j;
              if (j < (nh >> 7)) { b_mask |= 1u << (2 * h + j); ++n_b; }
            }
          }
        } else {
          a_boxes = (c.a_ext - t.m0 > 64u) ? 2u : 1u; n_b = t.nw >> 6;
#pragma unroll
          for (uint32_t j = 0; j < 4; ++j) { b_col[j] = t.n0 + 64 * j; if (j < n_b) b_mask |= 1u << j; }
        }
        const uint32_t tx = (a_boxes + n_b) * kBoxBytes * kCG;
        for (uint32_t kb = 0; kb < t.nkb; ++kb) {
          ptx::mbar_wait(empty0 + 8 * stage, phase ^ 1);
          if (ptx::elect_one()) {
          if (rank == 0) ptx::mbar_arrive_expect_tx(full0 + 8 * stage, tx);
          const uint32_t fb = full_lead0 + 8 * stage;
          const uint32_t sa = stage0 + stage * kStageBytes, sb = sa + kABytes;
          const int k0 = (int)(kb * kBK);
          for (uint32_t h = 0; h < a_boxes; ++h) {
            const int mn = (int)(am0 + 64 * h);
            if constexpr (kCG == 2) ptx::tma_load_2d_cg2(sa + h * kBoxBytes, c.ta, c.a_mn ? mn : k0, c.a_mn ? k0 : mn, fb);
            else ptx::tma_load_2d(sa + h * kBoxBytes, c.ta, c.a_mn ? mn : k0, c.a_mn ? k0 : mn, fb);
          }
#pragma unroll
          for (uint32_t j = 0; j < 4; ++j) {
            if (b_mask & (1u << j)) {
              const int mn = (int)b_col[j];
              const uint32_t dst = sb + j * kBoxBytes;
              if constexpr (kCG == 2) ptx::tma_load_2d_cg2(dst, c.tb, c.b_mn ? mn : k0, c.b_mn ? k0 : mn, fb);
              else ptx::tma_load_2d(dst, c.tb, c.b_mn ? mn : k0, c.b_mn ? k0 : mn, fb);
            }
          }
          }
          __syncwarp();
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        ++n_done;                                               // tells the scheduler that this tile's loads are issued
        if (rank == 0 && lane == 0) ptx::st_shared_volatile_u32(prod_done, n_done);
      }
    }
  } else if (warp == 6) {
    // ===== tile scheduler (leader CTA, one lane): claims tiles, waits for their dependencies, publishes them.  It runs
    // ahead of the producer, which takes the atomic, the descriptor fetch and the dependency check (~2 K cycles, three
    // dependent trips to L2) off the load-issue path: by up to the feed depth on tiny tiles (< 8 k blocks), by one tile
    // on medium ones (queueing more costs load balance at the end of a phase), not at all on long ones (>= 32 k
    // blocks: it waits until the producer has issued the tile's last load -- claiming long tiles early widens the
    // window of tiles in flight and measured 19 % more DRAM traffic on the Llama-70B set, because the L2 reuse between
    // list neighbours relies on their starting close in time). =====
    if (rank == 0 && lane == 0) {
      constexpr uint32_t kLongKb = 32, kTinyKb = 8;
      const uint32_t total = p.n_iter_tiles * p.ns_steps;
      for (uint32_t n_pub = 0;; ++n_pub) {
        const uint32_t ti = feed.claim(p.counter, total);
        uint32_t wait_for = 0;                                   // producer progress required before the next claim
        Work w0;
        TcMat M0;
        w0.it = 0; w0.t = TcTile{0u, 0u, 0u, 0, 0, 0u, 0u, 0u, 0u};
        M0.rows = M0.cols = M0.d = M0.tall = M0.pitch_a = 0; M0.a_off = 0;
        if (ti != kNoTile) {
          // inputs of the tile = outputs of every tile of the same matrix in the preceding phases: wait until all of
          // them have been reported complete (tiles are claimed in phase order and every unit works through its
          // claims in order, so those tiles are running or done, never waiting on a later one)
          w0 = fetch(p, ti);
          M0 = p.mats[w0.t.mat];
          const uint32_t need = w0.it * w0.t.reports_per_iter + w0.t.need;
          const uint32_t* flag = p.done + w0.t.mat;
          wait_for = w0.t.nkb >= kLongKb ? n_pub + 1 : (w0.t.nkb >= kTinyKb ? n_pub : 0u);
          if (ptx::ld_acquire_gpu(flag) < need) {
            const long long t0 = clock64();
            while (ptx::ld_acquire_gpu(flag) < need) {
              __nanosleep(64);
              if (clock64() - t0 > 20000000000ll) __trap();
            }
          }
        }
        feed.publish(ti, w0, M0);
        if (ti == kNoTile) break;
        if (ptx::ld_shared_volatile_u32(prod_done) < wait_for) {
          const long long t0 = clock64();
          while (ptx::ld_shared_volatile_u32(prod_done) < wait_for) {
            __nanosleep(256);
            if (clock64() - t0 > 20000000000ll) __trap();
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===== UMMA issuer (leader CTA only when paired).  The whole warp runs the loop converged, so that descriptors,
    // barrier addresses and the TMEM address are warp-uniform values (uniform registers, no per-instruction
    // vector->uniform election loops); one elected lane issues the UMMAs and their commits. =====
    if (rank == 0) {
      const uint32_t tmem_u = __shfl_sync(0xffffffffu, tmem_base, 0);
      uint32_t stage = 0, phase = 0, acc_next = 0;
      uint32_t acc_phase = 0;                                      // bit per accumulator
      for (;;) {
        const uint32_t ti = __shfl_sync(0xffffffffu, feed.peek(), 0);
        Work w;
        TcMat M;
        feed.read(w, M);
        __syncwarp();
        feed.release(lane == 0);
        if (ti == kNoTile) break;
        const TcTile t = w.t;
        const TileCfg c = decode(p, t, M, w.src);
        // K-major: +32 B per 16-k step; MN-major: +16 rows of 128 B.  (descriptor address field is in 16-byte units)
        const uint32_t a_step = c.a_mn ? (2048u >> 4) : (32u >> 4), b_step = c.b_mn ? (2048u >> 4) : (32u >> 4);
        const uint32_t a_lbo = c.a_mn ? kBoxBytes : 16u, b_lbo = c.b_mn ? kBoxBytes : 16u;
        // accumulators of this tile: wider than 256 columns -> both, halves h = 0, 1 in TMEM columns 256 h; else one,
        // alternating from tile to tile (the epilogue of one such tile overlaps the main loop of the next)
        const uint32_t n_acc = t.nw > kBN ? 2u : 1u;
        const uint32_t acc0 = n_acc == 2 ? 0u : acc_next;
        acc_next = n_acc == 2 ? 0u : acc_next ^ 1u;
        // The two accumulators of a paired tile are visited in turn; a visit covers kGroup ring stages (switching the
        // accumulator after every stage measured ~20 % slower UMMA issue than staying on one).
        for (uint32_t kb = 0; kb < t.nkb; kb += kGroup) {
          const uint32_t gcnt = min(kGroup, (uint32_t)t.nkb - kb);
          for (uint32_t s = 0; s < gcnt; ++s) {
            const uint32_t st = stage + s;
            ptx::mbar_wait(full0 + 8 * (st % kStages), phase ^ (st >= kStages ? 1u : 0u));
          }
          ptx::tc_fence_after();
          for (uint32_t h = 0; h < n_acc; ++h) {
            const uint32_t acc = acc0 + h;
            const uint32_t nh = kCG == 2 ? min((uint32_t)t.nw - h * kBN, kBN) : (uint32_t)t.nw;
            const uint32_t idesc = ptx::idesc_bf16_f32(kBM * kCG, nh, c.a_mn, c.b_mn);
            const uint32_t d_tmem = tmem_u + acc * kBN;
            if (kb == 0) {                                         // every epilogue warp has drained this accumulator
              ptx::mbar_wait(tempty0 + 8 * acc, ((acc_phase >> acc) & 1u) ^ 1u);
              ptx::tc_fence_after();
            }
            if (ptx::elect_one()) {
            for (uint32_t s = 0; s < gcnt; ++s) {
              const uint32_t sa = stage0 + ((stage + s) % kStages) * kStageBytes, sb = sa + kABytes;
              const uint64_t ad = ptx::smem_desc_sw128(sa, a_lbo, 1024);
              const uint64_t bd = ptx::smem_desc_sw128(sb + h * 2 * kBoxBytes, b_lbo, 1024);
#pragma unroll
              for (uint32_t ks = 0; ks < kBK / 16; ++ks) {
                if constexpr (kCG == 2)
                  ptx::umma_bf16_cg2(d_tmem, ad + (uint64_t)(ks * a_step), bd + (uint64_t)(ks * b_step), idesc, (kb | s | ks) != 0);
                else
                  ptx::umma_bf16(d_tmem, ad + (uint64_t)(ks * a_step), bd + (uint64_t)(ks * b_step), idesc, (kb | s | ks) != 0);
              }
            }
            if (kb + gcnt == t.nkb) {                              // accumulator complete: hand it to the epilogue warps
              if constexpr (kCG == 2) ptx::umma_commit_cg2(tfull0 + 8 * acc); else ptx::umma_commit(tfull0 + 8 * acc);
            }
            }
            __syncwarp();
            if (kb + gcnt == t.nkb) acc_phase ^= 1u << acc;
          }
          // free the smem slots (in both CTAs when paired) once these MMAs have finished
          for (uint32_t s = 0; s < gcnt; ++s) {
            if (ptx::elect_one()) {
              if constexpr (kCG == 2) ptx::umma_commit_cg2(empty0 + 8 * stage); else ptx::umma_commit(empty0 + 8 * stage);
            }
            __syncwarp();
            if (++stage == kStages) { stage = 0; phase ^= 1; }
          }
        }
      }
    }
  } else {
    // ===== epilogue: warps 2..5, warp w owns TMEM lanes 32 (w % 4) .. + 31 = 32 rows of the CTA's 128 =====
    const uint32_t q = warp & 3, ew = warp - 2;
    const uint32_t buf0 = epi0 + ew * 2 * kEpiBufBytes;          // two 4 KB staging tiles, used alternately
    uint32_t n_store = 0, epi_phase = 0, acc_next = 0;
    uint32_t pend_mat = kNoTile, pend_seq = 0;                   // tile whose completion has not been reported yet
    const uint32_t tempty_lead0 = kCG == 2 ? ptx::mapa(tempty0, 0) : tempty0;
    const uint32_t sw = (lane & 7) << 4;                         // 128-byte swizzle: 16-byte chunk j of row i sits at j ^ (i & 7)
    const uint32_t row_smem = lane * 128;
    // Completion report of this warp's share of a tile: its TMA stores have been performed, then a release at gpu
    // scope.  `newer` = stores issued after the tile's last one: waiting for "all but the newest k <= newer groups"
    // does not wait for those.  A report is deferred while the next accumulator is already waiting to be drained (then
    // it is made after that tile's stores, by which time it costs nothing) and made at once otherwise.
    auto report = [&](uint32_t newer) {
      if (lane == 0) {
        if (newer >= 8) ptx::bulk_wait<8>(); else if (newer >= 4) ptx::bulk_wait<4>();
        else if (newer >= 2) ptx::bulk_wait<2>(); else if (newer >= 1) ptx::bulk_wait<1>(); else ptx::bulk_wait<0>();
        ptx::fence_proxy_async();
        ptx::red_release_gpu_add(p.done + pend_mat, 1u);
      }
      pend_mat = kNoTile;
    };
    for (;;) {
      // the producer may be waiting for the pending report before it publishes the next tile: never block on the feed
      // with a report outstanding
      if (pend_mat != kNoTile && !__shfl_sync(0xffffffffu, (uint32_t)feed.ready(), 0)) report(n_store - pend_seq);
      const uint32_t ti = feed.peek();
      Work w;
      TcMat M;
      feed.read(w, M);
      __syncwarp();
      feed.release(lane == 0);
      if (ti == kNoTile) break;
      const TcTile t = w.t;
      const TileCfg c = decode(p, t, M, w.src);
      const float inv = w.first ? p.inv_norm[t.mat] : 1.f;
      const float alpha = t.phase == PH_GRAM ? inv * inv : inv;
      const uint32_t rb0 = t.m0 + rank * kBM;                    // first output row of this CTA
      const uint32_t rw0 = rb0 + q * 32;                         // ... of this warp
      const uint32_t r = rw0 + lane;                             // ... of this thread
      const bool rows_ok = rw0 < c.out_rows;                     // warp-uniform
      const bool sym = t.phase != PH_APPLY;
      const bool poly = t.phase == PH_POLY;
      // last iteration's APPLY: W <- W (1 - lr wd) - lr s O right here, from the O tile held in registers (a4)
      const bool upd = p.ua.W != nullptr && t.phase == PH_APPLY && w.it + 1 == p.ns_steps;   // warp-uniform
      float coef = 0.f;
      uint64_t w_elem = 0;
      __nv_bfloat16* fan_row = nullptr;                          // this thread's row of the fan-out copy of W, at t.n0
      if (upd) {
        const TcUpd* u = p.ua.upd + t.mat;
        coef = (float)(p.ua.lr * u->scale[p.ua.scale_mode]);           // lr s, rounded once (as k_update does)
        w_elem = u->elem_off;
        const uint64_t fb = p.ua.fan ? p.ua.fan[t.mat] : 0ull;
        if (fb) fan_row = reinterpret_cast<__nv_bfloat16*>(fb) + (size_t)r * c.out_cols + t.n0;
      }
      const uint32_t n_acc = t.nw > kBN ? 2u : 1u;
      const uint32_t acc0 = n_acc == 2 ? 0u : acc_next;
      acc_next = n_acc == 2 ? 0u : acc_next ^ 1u;
      unsigned long long t_ready = 0ull;
      long long c_ready = 0ll;
      // chunks of 64 columns; chunk cc lives in accumulator acc0 + cc / 4.  Which chunks this warp writes:
      const uint32_t n_chunks = min((uint32_t)t.nw, c.out_cols - t.n0 + 63u) >> 6;
      auto writes = [&](uint32_t cc) {       // warp-uniform
        // symmetric outputs: a 128-block below the diagonal is the mirror image of one that is written from above
        return cc < n_chunks && rows_ok && !(sym && ((t.n0 + 64 * cc) >> 7) < (rb0 >> 7));
      };
      // POLY: this thread's 64 A values of a chunk (row r, 128 contiguous bytes), fetched one chunk ahead through L2
      // (A was written by other SMs during this launch: no L1).  Fused update: the thread's 64 W values likewise
      // (bf16, row pitch = cols, cols % 8 == 0 so that a 16-byte vector never straddles the row end).
      const __nv_bfloat16* arow = nullptr;
      if (poly) arow = reinterpret_cast<const __nv_bfloat16*>(p.ws + M.a_off) + (size_t)r * M.pitch_a + t.n0;
      else if (upd) arow = reinterpret_cast<const __nv_bfloat16*>(p.ua.W) + w_elem + (size_t)r * c.out_cols + t.n0;
      const bool a_ok = (poly || upd) && r < c.out_rows;
      uint4 an[8];
      auto fetch_a = [&](uint32_t cc) {
        if (a_ok && writes(cc)) {
          if (poly) {
#pragma unroll
            for (int j = 0; j < 8; ++j) an[j] = ptx::ld_global_cg_v4(arow + 64 * cc + 8 * j);
          } else {
#pragma unroll
            for (int j = 0; j < 8; ++j)
              an[j] = t.n0 + 64 * cc + 8 * j < c.out_cols ? *reinterpret_cast<const uint4*>(arow + 64 * cc + 8 * j)
                                                         : make_uint4(0u, 0u, 0u, 0u);
          }
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j) an[j] = make_uint4(0u, 0u, 0u, 0u);
        }
      };
      uint32_t first_cc = 0;
      while (first_cc < n_chunks && !writes(first_cc)) ++first_cc;
      if (poly || upd) fetch_a(first_cc);

      for (uint32_t h = 0; h < n_acc; ++h) {
        const uint32_t acc = acc0 + h;
        if (pend_mat != kNoTile && h == 0 &&
            !__shfl_sync(0xffffffffu, ptx::mbar_try_wait(tfull0 + 8 * acc, (epi_phase >> acc) & 1u), 0))
          report(n_store - pend_seq);                            // the accumulator is not ready anyway: report now
        ptx::mbar_wait(tfull0 + 8 * acc, (epi_phase >> acc) & 1u);
        epi_phase ^= 1u << acc;
        ptx::tc_fence_after();
        if (p.trace && h == 0) { t_ready = ptx::globaltimer(); c_ready = clock64(); }
        const uint32_t taddr0 = tmem_base + ((q * 32u) << 16) + acc * kBN;
        for (uint32_t cc = 4 * h; cc < 4 * h + 4; ++cc) {
          if (!writes(cc)) continue;
          const uint32_t c0 = 64 * (cc & 3u), col0 = t.n0 + 64 * cc;
          uint4 a4[8];
          if (poly || upd) {
#pragma unroll
            for (int j = 0; j < 8; ++j) a4[j] = an[j];
            uint32_t nx = cc + 1;
            while (nx < n_chunks && !writes(nx)) ++nx;
            fetch_a(nx);                                         // next chunk's A values: in flight during this chunk
          }
          const uint32_t buf = buf0 + (n_store & 1u) * kEpiBufBytes;
          if (lane == 0) ptx::bulk_wait_read<1>();               // the store issued two stores ago has released `buf`
          __syncwarp();
          uint32_t v[64];
          {
            uint32_t lo[32], hi[32];
            ptx::tmem_ld32(taddr0 + c0, lo);
            ptx::tmem_ld32(taddr0 + c0 + 32, hi);
            ptx::tmem_ld_wait();
#pragma unroll
            for (int j = 0; j < 32; ++j) { v[j] = lo[j]; v[32 + j] = hi[j]; }
          }
          uint32_t pk[32];                                       // the thread's 64 outputs as bf16 pairs
          if (poly) {
            const bool on_diag = col0 < rw0 + 32u && rw0 < col0 + 64u;   // warp-uniform: the chunk crosses the diagonal
#pragma unroll
            for (int j = 0; j < 8; ++j) {
              const uint32_t aw[4] = {a4[j].x, a4[j].y, a4[j].z, a4[j].w};
#pragma unroll
              for (int i = 0; i < 4; ++i) {
                float f0 = fmaf(p.c, __uint_as_float(v[8 * j + 2 * i]), p.b * __uint_as_float(aw[i] << 16));
                float f1 = fmaf(p.c, __uint_as_float(v[8 * j + 2 * i + 1]), p.b * __uint_as_float(aw[i] & 0xffff0000u));
                if (on_diag) {                                   // the diagonal element: + a
                  if (col0 + 8 * j + 2 * i == r) f0 += p.a;
                  if (col0 + 8 * j + 2 * i + 1 == r) f1 += p.a;
                }
                pk[4 * j + i] = pack_bf16(f0, f1);
              }
            }
          } else if (w.first) {                                  // iteration 0: the folded Frobenius normalisation
#pragma unroll
            for (int j = 0; j < 32; ++j)
              pk[j] = pack_bf16(alpha * __uint_as_float(v[2 * j]), alpha * __uint_as_float(v[2 * j + 1]));
          } else {
#pragma unroll
            for (int j = 0; j < 32; ++j) pk[j] = pack_bf16(__uint_as_float(v[2 * j]), __uint_as_float(v[2 * j + 1]));
          }
          if (upd) {                                             // W <- fl(1 - lr wd) W - fl(lr s) O, O as stored (bf16)
            if (a_ok) {
              __nv_bfloat16* wrow = const_cast<__nv_bfloat16*>(arow) + 64 * cc;
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                if (col0 + 8 * j < c.out_cols) {
                  const uint32_t ww[4] = {a4[j].x, a4[j].y, a4[j].z, a4[j].w};
                  uint32_t nw[4];
#pragma unroll
                  for (int i = 0; i < 4; ++i) {
                    const float o0 = __uint_as_float(pk[4 * j + i] << 16), o1 = __uint_as_float(pk[4 * j + i] & 0xffff0000u);
                    const float w0 = __uint_as_float(ww[i] << 16), w1 = __uint_as_float(ww[i] & 0xffff0000u);
                    nw[i] = pack_bf16(fmaf(-coef, o0, p.ua.decay * w0), fmaf(-coef, o1, p.ua.decay * w1));
                  }
                  *reinterpret_cast<uint4*>(wrow + 8 * j) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
                  if (fan_row) *reinterpret_cast<uint4*>(fan_row + 64 * cc + 8 * j) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
                }
              }
            }
            if (!p.ua.keep_o) continue;                          // O itself is not needed: nothing to store
          }
          // direct tile: row `lane` of the staging tile, swizzled; then one TMA store (clipped at the matrix edges)
#pragma unroll
          for (int j = 0; j < 8; ++j)
            ptx::st_shared_v4(buf + row_smem + (((uint32_t)j << 4) ^ sw), pk[4 * j], pk[4 * j + 1], pk[4 * j + 2], pk[4 * j + 3]);
          ptx::fence_async_smem();
          __syncwarp();
          if (lane == 0) { ptx::tma_store_2d(c.tout, (int)col0, (int)rw0, buf); ptx::bulk_commit(); }
          ++n_store;
          // mirror tile of strictly-upper 128-blocks: staged transposed (64 x 32), stored at (row col0, column rw0)
          if (sym && (col0 >> 7) > (rb0 >> 7)) {
            const uint32_t mbuf = buf0 + (n_store & 1u) * kEpiBufBytes;
            if (lane == 0) ptx::bulk_wait_read<1>();
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              ptx::st_shared_b16(mbuf + (2 * j) * 64 + lane * 2, (uint16_t)(pk[j] & 0xffffu));
              ptx::st_shared_b16(mbuf + (2 * j + 1) * 64 + lane * 2, (uint16_t)(pk[j] >> 16));
            }
            ptx::fence_async_smem();
            __syncwarp();
            if (lane == 0) { ptx::tma_store_2d(c.tmir, (int)rw0, (int)col0, mbuf); ptx::bulk_commit(); }
            ++n_store;
          }
        }
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          if constexpr (kCG == 2) ptx::mbar_arrive_cluster(tempty_lead0 + 8 * acc); else ptx::mbar_arrive(tempty0 + 8 * acc);
        }
      }
      if (pend_mat != kNoTile) report(n_store - pend_seq);       // the previous tile: its stores are at least a tile old
      pend_mat = t.mat;
      pend_seq = n_store;
      if (p.trace && q == 0 && lane == 0 && rank == 0) {         // one record per tile: when its (first) accumulator was
        const unsigned long long slot = atomicAdd(p.trace, 1ull);   // ready and when this warp had issued its stores
        if (slot < p.trace_cap) {
          unsigned long long* rec = p.trace + 1 + 6 * slot;
          rec[0] = ((unsigned long long)(3u * w.it + t.phase) << 32) | ti;
          rec[1] = ((unsigned long long)unit << 32) | ptx::smid();
          rec[2] = t_ready;
          rec[3] = ptx::globaltimer();
          rec[4] = (unsigned long long)c_ready;
          rec[5] = ((unsigned long long)t.nkb << 32) | t.nw;
        }
      }
    }
    if (pend_mat != kNoTile) report(n_store - pend_seq);
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

// Row-major bf16 matrix rows x cols with row pitch `pitch` elements; box = box_cols (inner) x box_rows (outer);
// out-of-bounds elements read as zero (ragged edges, partial k blocks and whole out-of-range boxes rely on it) and
// are dropped by stores.
int make_tmap(CUtensorMap* out, void* base, uint32_t rows, uint32_t cols, uint32_t pitch, uint32_t box_cols,
              uint32_t box_rows, CUtensorMapSwizzle swz) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return cuda_fail(cudaErrorSymbolNotFound);
  const cuuint64_t dims[2] = {cols, rows};
  const cuuint64_t strides[1] = {(cuuint64_t)pitch * 2};
  const cuuint32_t box[2] = {box_cols, box_rows};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? MFSDP_OK : cuda_fail(cudaErrorInvalidValue);
}

// Tile rasterisation.  The units (CTAs or CTA pairs) claim tiles in list order, so at any moment the tiles in
// flight are a contiguous window of about n_units list entries, started at staggered times: entry j + s starts about
// s / n_units of a tile duration after entry j.  An operand box fetched from DRAM by one tile is re-read from L2 by
// the tiles that share it as long as the next sharer follows soon enough.  The list is therefore ordered so that a
// window covers a compact block of the output (`band` row blocks x the column tiles that go with them) and sharers
// are few entries apart: column-panel sharers adjacent, row-panel sharers `band` entries apart.
uint16_t tile_w(uint32_t remaining, uint32_t cg, uint32_t bn) {   // width of a tile that has `remaining` columns to cover
  const uint32_t gran = 64 * cg;
  return (uint16_t)std::min(bn, (remaining + gran - 1) / gran * gran);
}
// rectangular output (APPLY): column panels of `group` tiles stay L2-resident while all row blocks sweep over them.
void tiles_rect(std::vector<TcTile>& v, uint32_t mat, uint32_t out_rows, uint32_t out_cols, uint32_t nkb, uint32_t cg,
                uint32_t bn, uint32_t phase) {
  const uint32_t bm = kBM * cg;
  const uint32_t tm = (out_rows + bm - 1) / bm, tn = (out_cols + bn - 1) / bn;
  const uint32_t group = (uint32_t)std::max(1, tune_value(MFSDP_TUNE_RECT_GROUP));
  for (uint32_t g0 = 0; g0 < tn; g0 += group)
    for (uint32_t i = 0; i < tm; ++i)
      for (uint32_t j = g0; j < std::min(tn, g0 + group); ++j)
        v.push_back(TcTile{mat, i * bm, j * bn, (uint16_t)nkb, tile_w(out_cols - j * bn, cg, bn), 0u, phase, 0u, 0u});
}
// symmetric output (GRAM, POLY): upper row blocks only; bands of `band` row blocks, inside a band column-major
// (all row blocks of the band for one column step of a tile width, then the next step).
void tiles_sym(std::vector<TcTile>& v, uint32_t mat, uint32_t d, uint32_t nkb, uint32_t cg, uint32_t bn, uint32_t phase) {
  const uint32_t bm = kBM * cg;
  const uint32_t tm = (d + bm - 1) / bm;
  const uint32_t band = (uint32_t)std::max(1, tune_value(cg == 2 ? MFSDP_TUNE_SYM_BAND2 : MFSDP_TUNE_SYM_BAND));
  for (uint32_t b0 = 0; b0 < tm; b0 += band) {
    const uint32_t b1 = std::min(tm, b0 + band);
    for (uint32_t c0 = b0 * bm; c0 < d; c0 += bn)                // column steps from the band's first diagonal
      for (uint32_t i = b0; i < b1; ++i) {
        // row block i owns columns >= i * bm; clip the step to that range (the tile is half as wide when only half
        // of the step is owned)
        const uint32_t lo = std::max(c0, i * bm);
        const uint32_t hi = std::min(d, c0 + bn);
        if (lo >= hi) continue;
        v.push_back(TcTile{mat, i * bm, lo, (uint16_t)nkb, tile_w(hi - lo, cg, bn), 0u, phase, 0u, 0u});
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
cudaError_t launch_class(const TcParams& p, uint32_t units, cudaStream_t st) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(units * kCG);
  cfg.blockDim = dim3(kThreads);
  cfg.dynamicSmemBytes = kSmemBytes;
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
  std::vector<CUtensorMap> maps(TM_COUNT * lay.mats.size());
  std::vector<TcMat> mats(lay.mats.size());
  std::vector<TcTile> tiles[2];
  // big matrices first so that every phase of the tile list ends with the cheap tiles (dynamic claims, list order)
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
    m.tall = L.tall; m.reports_per_iter = 0;
    CUtensorMap* tm = &maps[TM_COUNT * i];
    void *x0 = ws + L.x_off[0], *x1 = ws + L.x_off[1], *pa = ws + L.a_off, *pp = ws + L.p_off;
    const CUtensorMapSwizzle s128 = CU_TENSOR_MAP_SWIZZLE_128B, s0 = CU_TENSOR_MAP_SWIZZLE_NONE;
    int rc;
    if ((rc = make_tmap(tm + TM_X0, x0, L.rows, L.cols, L.pitch_x, 64, 64, s128)) ||
        (rc = make_tmap(tm + TM_X1, x1, L.rows, L.cols, L.pitch_x, 64, 64, s128)) ||
        (rc = make_tmap(tm + TM_A, pa, L.d, L.d, L.pitch_a, 64, 64, s128)) ||
        (rc = make_tmap(tm + TM_P, pp, L.d, L.d, L.pitch_a, 64, 64, s128)) ||
        (rc = make_tmap(tm + TM_X0_ST, x0, L.rows, L.cols, L.pitch_x, 64, 32, s128)) ||
        (rc = make_tmap(tm + TM_X1_ST, x1, L.rows, L.cols, L.pitch_x, 64, 32, s128)) ||
        (rc = make_tmap(tm + TM_A_ST, pa, L.d, L.d, L.pitch_a, 64, 32, s128)) ||
        (rc = make_tmap(tm + TM_P_ST, pp, L.d, L.d, L.pitch_a, 64, 32, s128)) ||
        (rc = make_tmap(tm + TM_A_MIR, pa, L.d, L.d, L.pitch_a, 32, 64, s0)) ||
        (rc = make_tmap(tm + TM_P_MIR, pp, L.d, L.d, L.pitch_a, 32, 64, s0)))
      return rc;
  }
  // One iteration's tiles per class, phase-major (all GRAM tiles, then POLY, then APPLY): a launch walks this list
  // ns_steps times.  Paired tiles are 512 columns wide (one pass over the A operand feeds two accumulators) when the
  // k loop is long enough to hide the non-overlapped part of their epilogue, else 256 wide (double-buffered).
  const uint32_t wide_min_kb = (uint32_t)std::max(1, tune_value(MFSDP_TUNE_WIDE_MIN_KB));
  const uint32_t fused_below_d = (uint32_t)std::max(1, tune_value(MFSDP_TUNE_FUSED_BELOW_D));
  // class 0 = whole-matrix kernel (ns_fused.cu: small d, X resident in shared memory), 1 = single-CTA tiles, 2 = CTA pairs
  std::vector<uint32_t> cls(lay.mats.size());
  const uint32_t fused2_below_d = (uint32_t)std::max(1, tune_value(MFSDP_TUNE_FUSED2_BELOW_D));
  std::vector<FusedMat> fused[3];
  for (uint32_t i : order) {                      // cost-sorted: the fused CTAs claim the expensive matrices first
    const MatLayout& L = lay.mats[i];
    FusedMat f;
    int fc = 0;
    cls[i] = (uint32_t)ns_class(L.rows, L.cols);
    if (cls[i] == 0) {
      if (!fused_eligible(L.rows, L.cols, fused_below_d, &f, &fc)) { fused2_eligible(L.rows, L.cols, fused2_below_d, &f); fc = 2; }
      f.mat = i;
      fused[fc].push_back(f);
    }
  }
  for (uint32_t ph = 0; ph < 3; ++ph)
    for (uint32_t i : order) {
      const MatLayout& L = lay.mats[i];
      const uint32_t cg = cls[i];
      if (cg == 0) continue;
      const uint32_t nkb = ((ph == PH_GRAM ? L.n_long : L.d) + kBK - 1) / kBK;
      const uint32_t bn = cg == 2 && nkb >= wide_min_kb ? 2 * kBN : kBN;
      if (ph == PH_APPLY) tiles_rect(tiles[cg - 1], i, L.rows, L.cols, nkb, cg, bn, ph);
      else tiles_sym(tiles[cg - 1], i, L.d, nkb, cg, bn, ph);
    }
  // dependencies: a tile needs every completion report of its matrix' earlier phases (4 epilogue warps per CTA report)
  for (int g = 0; g < 2; ++g) {
    const uint32_t per_tile = 4u * (uint32_t)(g + 1);
    std::vector<uint32_t> cnt[3];
    for (int ph = 0; ph < 3; ++ph) cnt[ph].assign(lay.mats.size(), 0u);
    for (const TcTile& t : tiles[g]) cnt[t.phase][t.mat] += per_tile;
    for (TcTile& t : tiles[g]) {
      t.need = (t.phase >= 1 ? cnt[0][t.mat] : 0u) + (t.phase >= 2 ? cnt[1][t.mat] : 0u);
      t.reports_per_iter = cnt[0][t.mat] + cnt[1][t.mat] + cnt[2][t.mat];
    }
    for (size_t i = 0; i < lay.mats.size(); ++i)
      if (cls[i] == (uint32_t)g + 1) mats[i].reports_per_iter = cnt[0][i] + cnt[1][i] + cnt[2][i];
  }
  int rc;
  if ((rc = dev_upload(&tc->d_tmaps, maps)) || (rc = dev_upload(&tc->d_mats, mats))) return rc;
  for (int g = 0; g < 2; ++g) {
    tc->n_tiles[g] = (uint32_t)tiles[g].size();
    if ((rc = dev_upload(&tc->d_tiles[g], tiles[g]))) return rc;
  }
  {
    std::vector<TcUpd> upd(lay.mats.size());
    tc->upd_ok = lay.mat_dtype == MFSDP_BF16;
    for (size_t i = 0; i < lay.mats.size(); ++i) {
      upd[i].elem_off = lay.mats[i].elem_off;
      for (int k = 0; k < 3; ++k) upd[i].scale[k] = lay.mats[i].scale[k];
      if (lay.mats[i].cols % 8u) tc->upd_ok = false;     // a 16-byte vector of a W row must not straddle the row end
    }
    if ((rc = dev_upload(&tc->d_upd, upd))) return rc;
  }
  for (int g = 0; g < 3; ++g) {
    tc->n_fused[g] = (uint32_t)fused[g].size();
    if ((rc = dev_upload(&tc->d_fused[g], fused[g]))) return rc;
  }
  if ((rc = fused_setup()) || (rc = fused2_setup())) return rc;
  tc->n_mat = (uint32_t)lay.mats.size();
  cudaDeviceGetAttribute(&tc->sms, cudaDevAttrMultiProcessorCount, pl.device);
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(&tc->d_counters), (kCounterWords + (size_t)tc->n_mat) * sizeof(uint32_t));
  if (e != cudaSuccess) return cuda_fail(e);
  // the classes touch disjoint matrices: each runs on its own forked stream, joined before the pass returns
  if ((e = cudaEventCreateWithFlags(&tc->fork, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e);
  for (int k = 0; k < 4; ++k) {
    if ((e = cudaStreamCreateWithFlags(&tc->side[k], cudaStreamNonBlocking)) != cudaSuccess) return cuda_fail(e);
    if ((e = cudaEventCreateWithFlags(&tc->join[k], cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e);
  }
  e = cudaFuncSetAttribute(k_ns_tc<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return cuda_fail(e);
  e = cudaFuncSetAttribute(k_ns_tc<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return cuda_fail(e);
  // how many CTA pairs can be co-resident (one CTA per SM; the two CTAs of a pair share a TPC)
  {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)tc->sms / 2 * 2);
    cfg.blockDim = dim3(kThreads);
    cfg.dynamicSmemBytes = kSmemBytes;
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

int ns_class(uint32_t rows, uint32_t cols) {
  FusedMat f;
  int fc = 0;
  if (fused_eligible(rows, cols, (uint32_t)std::max(1, tune_value(MFSDP_TUNE_FUSED_BELOW_D)), &f, &fc)) return 0;
  if (fused2_eligible(rows, cols, (uint32_t)std::max(1, tune_value(MFSDP_TUNE_FUSED2_BELOW_D)), &f)) return 0;
  return std::min(rows, cols) >= (uint32_t)std::max(1, tune_value(MFSDP_TUNE_PAIR_MIN_D)) ? 2 : 1;
}

void destroy_ns_tc(NsTcPlan* p) {
  if (!p) return;
  cudaFree(p->d_tmaps); cudaFree(p->d_mats); cudaFree(p->d_counters); cudaFree(p->d_upd);
  for (int g = 0; g < 2; ++g) cudaFree(p->d_tiles[g]);
  for (int g = 0; g < 3; ++g) cudaFree(p->d_fused[g]);
  if (p->fork) cudaEventDestroy(p->fork);
  for (int k = 0; k < 4; ++k) {
    if (p->join[k]) cudaEventDestroy(p->join[k]);
    if (p->side[k]) cudaStreamDestroy(p->side[k]);
  }
  delete p;
}

bool ns_tc_can_fuse_update(Plan& pl) {
  std::lock_guard<std::mutex> lock(plan_mutex());
  if (!pl.tc && build_tc_plan(pl)) { destroy_ns_tc(pl.tc); pl.tc = nullptr; return false; }
  return pl.tc->upd_ok;
}

// W != nullptr (and ns_tc_can_fuse_update): the last APPLY epilogue also applies the weight update; O is then stored
// only when keep_o is set.
int launch_ns_tc(Plan& pl, const mfsdp_muon_hparams_t& hp, cudaStream_t st, void* W, bool keep_o, const uint64_t* fan) {
  if (pl.lay.mats.empty()) return MFSDP_OK;
  {
    std::lock_guard<std::mutex> lock(plan_mutex());     // two threads stepping the same table build it once
    if (!pl.tc) {
      const int rc = build_tc_plan(pl);
      if (rc) { destroy_ns_tc(pl.tc); pl.tc = nullptr; return rc; }
    }
  }
  NsTcPlan& tc = *pl.tc;
  TcParams p;
  p.mats = tc.d_mats; p.tmaps = tc.d_tmaps;
  p.ws = static_cast<uint8_t*>(pl.workspace);
  p.inv_norm = reinterpret_cast<const float*>(p.ws + pl.lay.invn_off);
  p.a = (float)hp.a; p.b = (float)hp.b; p.c = (float)hp.c;
  get_trace(&p.trace, &p.trace_cap);
  p.launch_idx = 0;
  p.ua.W = W && tc.upd_ok ? W : nullptr;
  p.ua.upd = tc.d_upd;
  p.ua.lr = hp.lr;
  p.ua.decay = (float)(1.0 - hp.lr * hp.weight_decay);
  p.ua.scale_mode = hp.scale_mode;
  p.ua.keep_o = keep_o ? 1u : 0u;
  p.ua.fan = p.ua.W ? fan : nullptr;
  p.ns_steps = (uint32_t)hp.ns_steps;
  p.done = tc.d_counters + kCounterWords;
  {
    const cudaError_t e = cudaMemsetAsync(tc.d_counters, 0, (kCounterWords + (size_t)tc.n_mat) * sizeof(uint32_t), st);
    if (e != cudaSuccess) return cuda_fail(e);
  }
  // One launch per class for the whole pass (all iterations, all phases).  The classes touch disjoint matrices, so
  // they run concurrently: the largest class stays on the caller's stream, the others are forked onto side streams
  // and joined back.  The whole-matrix kernels go first: their CTAs leave the SMs after a few tens of microseconds and
  // the persistent tile kernels pick the SMs up as they become free (tiles are claimed dynamically, so CTAs that
  // start late simply claim later tiles).
  struct Job { int kind; uint64_t work; };       // kind 0, 1, 2 = fused class; 3 = single-CTA tiles; 4 = CTA-pair tiles
  Job jobs[5];
  int n_jobs = 0;
  for (int c = 2; c >= 0; --c)
    if (tc.n_fused[c]) jobs[n_jobs++] = Job{c, (uint64_t)tc.n_fused[c] * (c == 2 ? 16u : 1u)};
  for (int g = 1; g >= 0; --g)
    if (tc.n_tiles[g]) jobs[n_jobs++] = Job{3 + g, (uint64_t)tc.n_tiles[g] * p.ns_steps * 64};
  if (n_jobs == 0) return MFSDP_OK;
  int main_job = 0;
  for (int j = 1; j < n_jobs; ++j)
    if (jobs[j].work > jobs[main_job].work) main_job = j;
  cudaError_t e;
  if (n_jobs > 1 && (e = cudaEventRecord(tc.fork, st)) != cudaSuccess) return cuda_fail(e);
  int side_used = 0;
  for (int j = 0; j < n_jobs; ++j) {
    cudaStream_t js = st;
    if (j != main_job) {
      js = tc.side[side_used];
      if ((e = cudaStreamWaitEvent(js, tc.fork, 0)) != cudaSuccess) return cuda_fail(e);
    }
    int rc = MFSDP_OK;
    if (jobs[j].kind < 2) {
      rc = launch_ns_fused(tc, jobs[j].kind, p.ws, p.inv_norm, hp, p.ua, js);
    } else if (jobs[j].kind == 2) {
      rc = launch_ns_fused2(tc, p.inv_norm, hp, p.ua, js);
    } else {
      const int g = jobs[j].kind - 3;
      p.tiles = tc.d_tiles[g];
      p.n_iter_tiles = tc.n_tiles[g];
      p.counter = tc.d_counters + g;
      const uint64_t total = (uint64_t)p.n_iter_tiles * p.ns_steps;
      if (total >= 0xffffffffull) return MFSDP_EINVAL;
      if (g == 1) e = launch_class<2>(p, (uint32_t)std::min<uint64_t>(total, (uint64_t)tc.max_pairs), js);
      else e = launch_class<1>(p, (uint32_t)std::min<uint64_t>(total, (uint64_t)tc.sms), js);
      if (e != cudaSuccess) return cuda_fail(e);
      ++p.launch_idx;
      count_launch();
      rc = check_last_launch();
    }
    if (rc) return rc;
    if (j != main_job) {
      if ((e = cudaEventRecord(tc.join[side_used], js)) != cudaSuccess) return cuda_fail(e);
      if ((e = cudaStreamWaitEvent(st, tc.join[side_used], 0)) != cudaSuccess) return cuda_fail(e);
      ++side_used;
    }
  }
  return MFSDP_OK;
}

}  // namespace mfsdp
