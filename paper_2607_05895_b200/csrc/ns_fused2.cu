// Newton-Schulz, whole-matrix kernel for MEDIUM matrices (MFSDP_NS_BF16): 128 < d = min(rows, cols) <= 256,
// max(rows, cols) <= 512.  One CTA owns one matrix for ALL K iterations; A and P = aI + bA + cA^2 (d x d) never leave
// the SM (128 KB of shared memory, written by the epilogue warps straight from TMEM, read back as UMMA operands); X is
// too large to stay (256 x 512 bf16 = 256 KB) and streams through a 2 x 32 KB TMA ring from the L2-resident ping-pong
// buffers: once for GRAM, once for APPLY per iteration, while X_new goes out through TMA stores.  Compared with the
// tile kernel (ns_tc.cu) on such matrices: no gpu-scope dependency counters, no tile feed, A and P never round-trip
// through global memory, and X is read twice per iteration instead of once per output tile.  (The single-CTA tiles
// there are bound by the instruction issue of their producer and UMMA threads -- ~650 and ~520 cycles per 64-k block
// for 6 TMA loads and 4 UMMAs of 128 cycles -- and by one exposed load latency per tile: DESIGN.md section 9.)
//
// Per iteration (same arithmetic and rounding points as ns_tc.cu; Y = X for wide, X^T for tall matrices):
//   GRAM   A = alpha Y Y^T     two row blocks of 128, accumulators 2 x 256 TMEM columns; k streams in 64-blocks
//   POLY   P = a I + b A + c A A   operands from shared memory; P overwrites A in place
//   APPLY  wide: X_new[:, c0:c0+128] = beta P X[:, c0:c0+128]   (B operand MN-major, streamed in 128-row k stages)
//          tall: X_new[m0:m0+128, :] = beta X[m0:m0+128, :] P    (A operand K-major, streamed; P symmetric)
//          accumulators double-buffered (2 x 256 columns): the epilogue of one chunk overlaps the UMMAs of the next
// 192 threads: warp 0 TMA producer, warp 1 TMEM owner + UMMA issuer, warps 2-5 epilogue (TMEM lane quarter = warp % 4).
#include <cuda.h>
#include <cuda_bf16.h>

#include <algorithm>

#include "mfsdp_internal.h"
#include "ns_plan.h"
#include "ptx_sm100.cuh"

namespace mfsdp {
namespace {

constexpr uint32_t kThreads2 = 192;
constexpr uint32_t kAPanel = 256 * 128;            // one 64-column panel of A / P: 256 rows x 128 B
constexpr uint32_t kABytes2 = 4 * kAPanel;         // 128 KB
constexpr uint32_t kStage2 = 32 * 1024;
constexpr uint32_t kStages2 = 2;
constexpr uint32_t kEpiBuf2 = 4096;                // one staging tile: 32 rows x 64 cols bf16
constexpr uint32_t kEpiBytes2 = 4 * 2 * kEpiBuf2;  // 4 epilogue warps x 2 buffers
constexpr uint32_t kBarBytes2 = 256;
constexpr uint32_t kSmem2 = kABytes2 + kStages2 * kStage2 + kEpiBytes2 + kBarBytes2 + 1024;
constexpr uint32_t kBox = 8192;                    // one 64 x 64 TMA box

struct Fused2Params {
  const FusedMat* list;
  uint32_t n_list;
  const CUtensorMap* tmaps;
  const float* inv_norm;
  uint32_t* counter;
  uint32_t ns_steps;
  float a, b, c;
  UpdArgs ua;
};

__device__ __forceinline__ uint32_t pack2(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ void ld64_2(uint32_t taddr, uint32_t (&v)[64]) {
  uint32_t lo[32], hi[32];
  ptx::tmem_ld32(taddr, lo);
  ptx::tmem_ld32(taddr + 32, hi);
  ptx::tmem_ld_wait();
#pragma unroll
  for (int j = 0; j < 32; ++j) { v[j] = lo[j]; v[32 + j] = hi[j]; }
}

// Shape of the streamed phases of one matrix (warp-uniform, recomputed by every role).
struct Shape2 {
  uint32_t d16, kd;            // d rounded up to 16, and its 16-element k steps
  uint32_t gram_stages;        // 64-element k blocks along n
  uint32_t apply_chunks;       // wide: 128-column chunks of n; tall: 128-row blocks of n
  __device__ __forceinline__ Shape2(const FusedMat& f) {
    const uint32_t n = f.tall ? f.rows : f.cols;
    d16 = f.d16; kd = d16 >> 4;
    gram_stages = (n + 63u) >> 6;
    apply_chunks = (n + 127u) >> 7;
  }
};

__global__ void __launch_bounds__(kThreads2, 1) k_ns_fused2(const Fused2Params p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t a0 = ptx::smem_u32(smem);                              // A / P: 4 panels x 256 rows x 128 B
  const uint32_t ring0 = a0 + kABytes2;
  const uint32_t epi0 = ring0 + kStages2 * kStage2;
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kABytes2 + kStages2 * kStage2 + kEpiBytes2);
  const uint32_t full0 = ptx::smem_u32(bars), empty0 = ptx::smem_u32(bars + 2);
  const uint32_t tfull0 = ptx::smem_u32(bars + 4), tempty0 = ptx::smem_u32(bars + 6);
  const uint32_t gfull = ptx::smem_u32(bars + 8);                       // GRAM / POLY accumulator complete
  const uint32_t pdone = ptx::smem_u32(bars + 9);                       // an epilogue phase complete (4 warp arrivals): issuer
  const uint32_t xdone = ptx::smem_u32(bars + 10);                      // X_new of an iteration stored (4 arrivals): producer
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 11);
  uint32_t* next_holder = tmem_holder + 1;
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (uint32_t s = 0; s < 2; ++s) {
      ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 1);
      ptx::mbar_init(tfull0 + 8 * s, 1); ptx::mbar_init(tempty0 + 8 * s, 4);
    }
    ptx::mbar_init(gfull, 1);
    ptx::mbar_init(pdone, 4);
    ptx::mbar_init(xdone, 4);
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc<512, 1>(ptx::smem_u32(tmem_holder));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;

  // pipeline state that persists across matrices (every role advances its own copy in the same way)
  uint32_t stage = 0, ring_phase = 0;        // operand ring (producer, issuer)
  uint32_t chunk_cnt = 0;                    // APPLY chunks so far: accumulator buffer = chunk_cnt & 1 (issuer, epilogue)
  uint32_t g_phase = 0;                      // gfull parity (issuer commits, epilogue waits)
  uint32_t pd_phase = 0;                     // pdone parity (epilogue arrives three times per iteration; the issuer waits
                                             // for every completion in order -- a parity wait must never fall two behind)
  uint32_t xd_phase = 0;                     // xdone parity (once per iteration; the producer waits in order)
  uint32_t n_store = 0;                      // epilogue: TMA stores issued by this warp (staging buffer parity)

  for (;;) {
    if (threadIdx.x == 0) *next_holder = atomicAdd(p.counter, 1u);
    __syncthreads();
    const uint32_t idx = *next_holder;
    __syncthreads();
    if (idx >= p.n_list) break;
    const FusedMat fm = p.list[idx];
    const Shape2 sh(fm);
    const CUtensorMap* tm = p.tmaps + TM_COUNT * (size_t)fm.mat;

    if (warp == 0) {
      // ===== TMA producer: per iteration the GRAM stream, then the APPLY stream (it runs ahead into APPLY while POLY
      // executes: both read the same X buffer) =====
      for (uint32_t it = 0; it < p.ns_steps; ++it) {
        const CUtensorMap* tx = tm + TM_X0 + (it & 1u);
        if (it > 0) {                        // X_new of the previous iteration: every store performed (APPLY epilogue)
          ptx::mbar_wait(xdone, xd_phase);
          xd_phase ^= 1u;
          ptx::fence_proxy_async();
        }
        for (uint32_t s = 0; s < sh.gram_stages; ++s) {
          ptx::mbar_wait(empty0 + 8 * stage, ring_phase ^ 1);
          if (ptx::elect_one()) {
            const uint32_t dst = ring0 + stage * kStage2, fb = full0 + 8 * stage;
            ptx::mbar_arrive_expect_tx(fb, kStage2);
            for (uint32_t j = 0; j < 4; ++j) {
              if (!fm.tall) ptx::tma_load_2d(dst + j * kBox, tx, (int)(64 * s), (int)(64 * j), fb);   // rows 64 j of Y, k block s
              else ptx::tma_load_2d(dst + j * kBox, tx, (int)(64 * j), (int)(64 * s), fb);             // columns 64 j of X, rows = k
            }
          }
          __syncwarp();
          if (++stage == kStages2) { stage = 0; ring_phase ^= 1; }
        }
        for (uint32_t ch = 0; ch < sh.apply_chunks; ++ch)
          for (uint32_t s = 0; s < 2; ++s) {           // two k stages of 128
            ptx::mbar_wait(empty0 + 8 * stage, ring_phase ^ 1);
            if (ptx::elect_one()) {
              const uint32_t dst = ring0 + stage * kStage2, fb = full0 + 8 * stage;
              ptx::mbar_arrive_expect_tx(fb, kStage2);
              for (uint32_t j = 0; j < 2; ++j)
                for (uint32_t h = 0; h < 2; ++h) {
                  if (!fm.tall)      // B operand: k rows 128 s + 64 h, columns 128 ch + 64 j   (MN chunk j, k contiguous)
                    ptx::tma_load_2d(dst + j * 2 * kBox + h * kBox, tx, (int)(128 * ch + 64 * j), (int)(128 * s + 64 * h), fb);
                  else               // A operand: rows 128 ch + 64 h, k columns 128 s + 64 j     (k panel j, rows contiguous)
                    ptx::tma_load_2d(dst + j * 2 * kBox + h * kBox, tx, (int)(128 * s + 64 * j), (int)(128 * ch + 64 * h), fb);
                }
            }
            __syncwarp();
            if (++stage == kStages2) { stage = 0; ring_phase ^= 1; }
          }
      }
      // the completion of the last iteration is not awaited (the __syncthreads at the top of the next matrix orders it)
      xd_phase ^= 1u;
    } else if (warp == 1) {
      // ===== UMMA issuer =====
      for (uint32_t it = 0; it < p.ns_steps; ++it) {
        // --- GRAM: both row blocks, N = d16, accumulators at TMEM columns 0 and 256 ---
        if (it > 0) {                        // both APPLY buffers drained (the APPLY epilogue has finished)
          ptx::mbar_wait(pdone, pd_phase);
          pd_phase ^= 1u;
        }
        ptx::tc_fence_after();
        {
          const uint32_t idesc = ptx::idesc_bf16_f32(128, sh.d16, fm.tall, fm.tall);
          for (uint32_t s = 0; s < sh.gram_stages; ++s) {
            ptx::mbar_wait(full0 + 8 * stage, ring_phase);
            ptx::tc_fence_after();
            if (ptx::elect_one()) {
              const uint32_t base = ring0 + stage * kStage2;
#pragma unroll
              for (uint32_t ks = 0; ks < 4; ++ks)
                for (uint32_t rb = 0; rb < 2; ++rb) {
                  uint64_t ad, bd;
                  if (!fm.tall) {            // K-major: 256 rows x 128 B; row block rb starts 16 KB further
                    ad = ptx::smem_desc_sw128(base + rb * 2 * kBox + ks * 32u, 16, 1024);
                    bd = ptx::smem_desc_sw128(base + ks * 32u, 16, 1024);
                  } else {                   // MN-major: 4 boxes of 64 columns; 16 k rows = 2 KB
                    ad = ptx::smem_desc_sw128(base + rb * 2 * kBox + ks * 2048u, kBox, 1024);
                    bd = ptx::smem_desc_sw128(base + ks * 2048u, kBox, 1024);
                  }
                  ptx::umma_bf16(tmem_base + rb * 256u, ad, bd, idesc, (s | ks) != 0);
                }
              ptx::umma_commit(empty0 + 8 * stage);
              if (s + 1 == sh.gram_stages) ptx::umma_commit(gfull);
            }
            __syncwarp();
            if (++stage == kStages2) { stage = 0; ring_phase ^= 1; }
          }
        }
        // --- POLY: A A from shared memory, once the GRAM epilogue has written A ---
        ptx::mbar_wait(pdone, pd_phase);
        pd_phase ^= 1u;
        ptx::tc_fence_after();
        if (ptx::elect_one()) {
          const uint32_t idesc = ptx::idesc_bf16_f32(128, sh.d16, 0, 0);
          for (uint32_t ks = 0; ks < sh.kd; ++ks)
            for (uint32_t rb = 0; rb < 2; ++rb) {
              const uint32_t koff = (ks >> 2) * kAPanel + (ks & 3u) * 32u;
              const uint64_t ad = ptx::smem_desc_sw128(a0 + koff + rb * 2 * kBox, 16, 1024);
              const uint64_t bd = ptx::smem_desc_sw128(a0 + koff, 16, 1024);
              ptx::umma_bf16(tmem_base + rb * 256u, ad, bd, idesc, ks != 0);
            }
          ptx::umma_commit(gfull);
        }
        __syncwarp();
        // --- APPLY, once the POLY epilogue has written P ---
        ptx::mbar_wait(pdone, pd_phase);
        pd_phase ^= 1u;
        ptx::tc_fence_after();
        for (uint32_t ch = 0; ch < sh.apply_chunks; ++ch) {
          const uint32_t buf = chunk_cnt & 1u, use = chunk_cnt >> 1;
          ptx::mbar_wait(tempty0 + 8 * buf, (use & 1u) ^ 1u);           // the epilogue has drained this buffer
          ptx::tc_fence_after();
          const uint32_t n = fm.tall ? fm.rows : fm.cols;
          const uint32_t nc = fm.tall ? sh.d16 : min(128u, (n - 128u * ch + 15u) & ~15u);
          const uint32_t idesc = ptx::idesc_bf16_f32(128, nc, 0, fm.tall ? 0u : 1u);
          bool first = true;
          for (uint32_t s = 0; s < 2; ++s) {
            ptx::mbar_wait(full0 + 8 * stage, ring_phase);
            ptx::tc_fence_after();
            const uint32_t ksteps = sh.kd > 8u * s ? min(8u, sh.kd - 8u * s) : 0u;
            if (ptx::elect_one()) {
              const uint32_t base = ring0 + stage * kStage2;
              for (uint32_t ks = 0; ks < ksteps; ++ks) {
                const uint32_t kg = 8u * s + ks;                        // global 16-element k step over d
                const uint32_t poff = (kg >> 2) * kAPanel + (kg & 3u) * 32u;
                if (!fm.tall) {
                  const uint64_t bd = ptx::smem_desc_sw128(base + ks * 2048u, 2 * kBox, 1024);   // X: MN-major, 2 chunks
                  for (uint32_t rb = 0; rb < 2; ++rb) {
                    const uint64_t ad = ptx::smem_desc_sw128(a0 + poff + rb * 2 * kBox, 16, 1024);   // P rows rb
                    ptx::umma_bf16(tmem_base + buf * 256u + rb * 128u, ad, bd, idesc, !first);
                  }
                } else {
                  const uint64_t ad = ptx::smem_desc_sw128(base + (ks >> 2) * 2 * kBox + (ks & 3u) * 32u, 16, 1024);  // X rows
                  const uint64_t bd = ptx::smem_desc_sw128(a0 + poff, 16, 1024);                   // P (symmetric), N = d16
                  ptx::umma_bf16(tmem_base + buf * 256u, ad, bd, idesc, !first);
                }
                first = false;
              }
              ptx::umma_commit(empty0 + 8 * stage);
              if (s == 1) ptx::umma_commit(tfull0 + 8 * buf);
            }
            __syncwarp();
            if (++stage == kStages2) { stage = 0; ring_phase ^= 1; }
          }
          ++chunk_cnt;
        }
      }
      // the APPLY completion of the last iteration is not awaited by this role
      pd_phase ^= 1u;
    } else {
      // ===== epilogue: warp owns TMEM lanes 32 q .. + 31 (q = warp % 4) = rows 32 q .. of each 128-row block =====
      const uint32_t q = warp & 3u, ew = warp - 2u;
      const uint32_t rq = q * 32u + lane;                               // row within a 128-row block
      const uint32_t sw = (lane & 7u) << 4;
      const uint32_t taddr = tmem_base + ((q * 32u) << 16);
      const uint32_t buf0 = epi0 + ew * 2 * kEpiBuf2;
      const float inv = p.inv_norm[fm.mat];
      const uint32_t n_dchunks = (sh.d16 + 63u) >> 6;
      float coef = 0.f;
      __nv_bfloat16 *wmat = nullptr, *fmat = nullptr;
      if (p.ua.W != nullptr) {
        const TcUpd* u = p.ua.upd + fm.mat;
        coef = (float)(p.ua.lr * u->scale[p.ua.scale_mode]);
        wmat = reinterpret_cast<__nv_bfloat16*>(p.ua.W) + u->elem_off;
        if (p.ua.fan) fmat = reinterpret_cast<__nv_bfloat16*>(p.ua.fan[fm.mat]);
      }
      uint32_t v[64], pk[32];
      for (uint32_t it = 0; it < p.ns_steps; ++it) {
        const float alpha = it == 0 ? inv * inv : 1.f, beta = it == 0 ? inv : 1.f;
        const bool last = it + 1 == p.ns_steps;
        const bool upd = wmat != nullptr && last;
        const bool store_x = !upd || p.ua.keep_o || !last;
        // --- GRAM: A = alpha acc -> shared memory ---
        ptx::mbar_wait(gfull, g_phase);
        g_phase ^= 1u;
        ptx::tc_fence_after();
        for (uint32_t rb = 0; rb < 2; ++rb)
          for (uint32_t cc = 0; cc < n_dchunks; ++cc) {
            ld64_2(taddr + rb * 256u + 64u * cc, v);
#pragma unroll
            for (int j = 0; j < 32; ++j)
              pk[j] = pack2(alpha * __uint_as_float(v[2 * j]), alpha * __uint_as_float(v[2 * j + 1]));
            const uint32_t row_addr = a0 + cc * kAPanel + (rb * 128u + rq) * 128u;
#pragma unroll
            for (int j = 0; j < 8; ++j)
              ptx::st_shared_v4(row_addr + (((uint32_t)j << 4) ^ sw), pk[4 * j], pk[4 * j + 1], pk[4 * j + 2], pk[4 * j + 3]);
          }
        ptx::fence_async_smem();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(pdone);
        // --- POLY: P = a I + b A + c acc, in place ---
        ptx::mbar_wait(gfull, g_phase);
        g_phase ^= 1u;
        ptx::tc_fence_after();
        for (uint32_t rb = 0; rb < 2; ++rb)
          for (uint32_t cc = 0; cc < n_dchunks; ++cc) {
            const uint32_t r = rb * 128u + rq;
            const uint32_t row_addr = a0 + cc * kAPanel + r * 128u;
            uint32_t aw[32];
#pragma unroll
            for (int j = 0; j < 8; ++j)
              ptx::ld_shared_v4(row_addr + (((uint32_t)j << 4) ^ sw), aw[4 * j], aw[4 * j + 1], aw[4 * j + 2], aw[4 * j + 3]);
            ld64_2(taddr + rb * 256u + 64u * cc, v);
            const bool on_diag = (r >> 6) == cc;
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              float f0 = fmaf(p.c, __uint_as_float(v[2 * j]), p.b * __uint_as_float(aw[j] << 16));
              float f1 = fmaf(p.c, __uint_as_float(v[2 * j + 1]), p.b * __uint_as_float(aw[j] & 0xffff0000u));
              if (on_diag) {
                if (64u * cc + 2 * j == r) f0 += p.a;
                if (64u * cc + 2 * j + 1 == r) f1 += p.a;
              }
              pk[j] = pack2(f0, f1);
            }
#pragma unroll
            for (int j = 0; j < 8; ++j)
              ptx::st_shared_v4(row_addr + (((uint32_t)j << 4) ^ sw), pk[4 * j], pk[4 * j + 1], pk[4 * j + 2], pk[4 * j + 3]);
          }
        ptx::fence_async_smem();
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) ptx::mbar_arrive(pdone);
        // --- APPLY: X_new chunk by chunk -> staging -> TMA store (and the weight update on the last iteration) ---
        const CUtensorMap* tout = tm + TM_X0_ST + ((it & 1u) ^ 1u);
        for (uint32_t ch = 0; ch < sh.apply_chunks; ++ch) {
          const uint32_t buf = chunk_cnt & 1u, use = chunk_cnt >> 1;
          ptx::mbar_wait(tfull0 + 8 * buf, use & 1u);
          ptx::tc_fence_after();
          // sub-chunks of 64 columns: wide: row block rb, columns 128 ch + 64 cc (TMEM column 128 rb + 64 cc);
          //                           tall: rows 128 ch .., columns 64 cc (TMEM column 64 cc)
          const uint32_t n_sub = fm.tall ? n_dchunks : 4u;
          for (uint32_t sc = 0; sc < n_sub; ++sc) {
            uint32_t row0, col0, tcol;
            if (!fm.tall) { const uint32_t rb = sc >> 1, cc = sc & 1u; row0 = rb * 128u + q * 32u; col0 = 128u * ch + 64u * cc; tcol = rb * 128u + 64u * cc; }
            else { row0 = 128u * ch + q * 32u; col0 = 64u * sc; tcol = 64u * sc; }
            if (row0 >= fm.rows || col0 >= fm.cols) continue;           // warp-uniform: nothing of this sub-chunk exists
            ld64_2(taddr + buf * 256u + tcol, v);
#pragma unroll
            for (int j = 0; j < 32; ++j)
              pk[j] = pack2(beta * __uint_as_float(v[2 * j]), beta * __uint_as_float(v[2 * j + 1]));
            const uint32_t r = row0 + lane;
            if (upd && r < fm.rows) {                                    // W <- fl(1 - lr wd) W - fl(lr s) O, as k_update
              __nv_bfloat16* wrow = wmat + (size_t)r * fm.cols + col0;
              __nv_bfloat16* frow = fmat ? fmat + (size_t)r * fm.cols + col0 : nullptr;
              const uint32_t n_valid = fm.cols - col0;
#pragma unroll
              for (int j = 0; j < 8; ++j) {
                if (8u * j < n_valid) {
                  const uint4 wv = *reinterpret_cast<const uint4*>(wrow + 8 * j);
                  const uint32_t ww[4] = {wv.x, wv.y, wv.z, wv.w};
                  uint32_t nw[4];
#pragma unroll
                  for (int i = 0; i < 4; ++i) {
                    const float o0 = __uint_as_float(pk[4 * j + i] << 16), o1 = __uint_as_float(pk[4 * j + i] & 0xffff0000u);
                    const float w0 = __uint_as_float(ww[i] << 16), w1 = __uint_as_float(ww[i] & 0xffff0000u);
                    nw[i] = pack2(fmaf(-coef, o0, p.ua.decay * w0), fmaf(-coef, o1, p.ua.decay * w1));
                  }
                  *reinterpret_cast<uint4*>(wrow + 8 * j) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
                  if (frow) *reinterpret_cast<uint4*>(frow + 8 * j) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
                }
              }
            }
            if (store_x) {
              const uint32_t sbuf = buf0 + (n_store & 1u) * kEpiBuf2;
              if (lane == 0) ptx::bulk_wait_read<1>();                  // the store issued two stores ago has released it
              __syncwarp();
#pragma unroll
              for (int j = 0; j < 8; ++j)
                ptx::st_shared_v4(sbuf + lane * 128u + (((uint32_t)j << 4) ^ sw), pk[4 * j], pk[4 * j + 1], pk[4 * j + 2], pk[4 * j + 3]);
              ptx::fence_async_smem();
              __syncwarp();
              if (lane == 0) { ptx::tma_store_2d(tout, (int)col0, (int)row0, sbuf); ptx::bulk_commit(); }
              ++n_store;
            }
          }
          ptx::tc_fence_before();
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(tempty0 + 8 * buf);
          ++chunk_cnt;
        }
        // X_new complete: every store of this warp performed, visible to the TMA loads of the next iteration
        if (lane == 0) {
          ptx::bulk_wait<0>();
          ptx::fence_proxy_async();
          ptx::mbar_arrive(xdone);
          ptx::mbar_arrive(pdone);
        }
        __syncwarp();
      }
    }
  }

  __syncwarp();
  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<512, 1>(tmem_base);
  }
}

}  // namespace

bool fused2_eligible(uint32_t rows, uint32_t cols, uint32_t below_d, FusedMat* out) {
  const uint32_t d = std::min(rows, cols), n = std::max(rows, cols);
  if (d <= 128u || d > 256u || d >= below_d || n > 512u) return false;   // one SM per matrix: longer ones run faster tiled
  FusedMat f;
  f.mat = 0; f.rows = rows; f.cols = cols; f.tall = rows > cols ? 1u : 0u;
  f.d16 = (d + 15u) / 16u * 16u;
  f.rpad = 0; f.panels = 0;
  f.k16 = (n + 15u) / 16u;
  *out = f;
  return true;
}

int fused2_setup() {
  const cudaError_t e = cudaFuncSetAttribute(k_ns_fused2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmem2);
  return e == cudaSuccess ? MFSDP_OK : cuda_fail(e);
}

int launch_ns_fused2(const NsTcPlan& tc, const float* inv_norm, const mfsdp_muon_hparams_t& hp, const UpdArgs& ua,
                     cudaStream_t st) {
  if (tc.n_fused[2] == 0) return MFSDP_OK;
  Fused2Params p;
  p.list = tc.d_fused[2];
  p.n_list = tc.n_fused[2];
  p.tmaps = tc.d_tmaps;
  p.inv_norm = inv_norm;
  p.counter = tc.d_counters + 4;
  p.ns_steps = (uint32_t)hp.ns_steps;
  p.a = (float)hp.a; p.b = (float)hp.b; p.c = (float)hp.c;
  p.ua = ua;
  const uint32_t grid = std::min<uint32_t>(p.n_list, (uint32_t)tc.sms);
  k_ns_fused2<<<grid, kThreads2, kSmem2, st>>>(p);
  count_launch();
  return check_last_launch();
}

}  // namespace mfsdp
