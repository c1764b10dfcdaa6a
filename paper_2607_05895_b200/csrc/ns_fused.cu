// Newton-Schulz, whole-matrix kernel for SMALL matrices (MFSDP_NS_BF16): d = min(rows, cols) <= 128 and a padded X of
// at most 128 KB.  One CTA owns one matrix for ALL K iterations: X streams in once by TMA, X, A and P never leave the
// SM (shared memory operands, TMEM accumulators), only X_K = O is written back.  No tile feed, no gpu-scope counters,
// no global round trips between the 3 K phases -- the per-tile fixed costs that bound the tile kernel (ns_tc.cu) on
// hundreds of tiny matrices (BASELINE.json config 3: 512 matrices of 64..512 rows / columns) do not exist here.
//
// Per iteration (north_star; same arithmetic and rounding points as ns_tc.cu):
//   GRAM   A = alpha Y Y^T              Y = X (wide) or X^T (tall), read through the UMMA operand majorness bits
//   POLY   P = a I + b A + c A A        the b A + a I terms fused in the epilogue; P overwrites A in place
//   APPLY  X <- beta P X  (wide)   or   X <- beta X P  (tall; P symmetric), written over X in place
// alpha = 1/||U||^2, beta = 1/||U|| at iteration 0 (Frobenius normalisation folded in), 1 afterwards.
//
// Shared memory: X row-major as `panels` column panels of 64 elements (128 B) x rpad rows, 128-byte swizzled -- the
// layout TMA writes (box 64 x 64) and UMMA reads both K-major (k along a row) and MN-major (k along the rows); A / P
// as 2 panels x 128 rows (32 KB).  Rows / columns beyond the matrix are zero (TMA out-of-bounds fill) and stay zero
// through the iteration, so every UMMA runs with M = 128 and N, K rounded up to 16.
// CTA = 160 threads: warps 0-3 epilogue (warp w owns TMEM lanes 32 w .. + 31 = rows of the accumulator), warp 4 = TMEM
// owner, TMA issue and UMMA issue (converged, one elected lane).  Two size classes, one launch each: padded X <= 64 KB
// (97 KB shared memory, 256 TMEM columns: two CTAs per SM, so one CTA's epilogue overlaps the other's UMMAs) and
// <= 128 KB (161 KB, 512 columns).  Matrices are claimed from a cost-sorted list with one atomicAdd each.
#include <cuda.h>
#include <cuda_bf16.h>

#include <algorithm>

#include "mfsdp_internal.h"
#include "ns_plan.h"
#include "ptx_sm100.cuh"

namespace mfsdp {
namespace {

constexpr uint32_t kThreadsF = 160;
constexpr uint32_t kABytesF = 2 * 128 * 128;        // A / P: 2 column panels x 128 rows x 128 B
constexpr uint32_t kBarBytesF = 64;
constexpr uint32_t kXBytesCls[2] = {64 * 1024, 128 * 1024};
constexpr uint32_t kTmemColsCls[2] = {256, 512};

struct FusedParams {
  const FusedMat* list;
  uint32_t n_list;
  const CUtensorMap* tmaps;
  const float* inv_norm;
  uint32_t* counter;
  uint32_t x_bytes;        // shared-memory bytes reserved for X (class maximum)
  uint32_t tmem_cols;
  uint32_t ns_steps;
  float a, b, c;
  UpdArgs ua;              // weight update fused into the last APPLY epilogue (ua.W != nullptr)
};

__device__ __forceinline__ uint32_t pack_bf16f(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}

// W <- fl(1 - lr wd) W - fl(lr s) O for this thread's 64 consecutive elements of one W row (bf16, 16-byte aligned),
// O as stored (bf16 pairs in pk); columns at or beyond `n_valid` are left alone.  Same arithmetic as k_update.
__device__ __forceinline__ void update_row64(__nv_bfloat16* wrow, __nv_bfloat16* fan_row, uint32_t n_valid,
                                             const uint32_t (&pk)[32], float coef, float decay) {
  uint4 wv[8];
#pragma unroll
  for (int j = 0; j < 8; ++j)
    wv[j] = 8u * j < n_valid ? *reinterpret_cast<const uint4*>(wrow + 8 * j) : make_uint4(0u, 0u, 0u, 0u);
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    if (8u * j < n_valid) {
      const uint32_t ww[4] = {wv[j].x, wv[j].y, wv[j].z, wv[j].w};
      uint32_t nw[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float o0 = __uint_as_float(pk[4 * j + i] << 16), o1 = __uint_as_float(pk[4 * j + i] & 0xffff0000u);
        const float w0 = __uint_as_float(ww[i] << 16), w1 = __uint_as_float(ww[i] & 0xffff0000u);
        nw[i] = pack_bf16f(fmaf(-coef, o0, decay * w0), fmaf(-coef, o1, decay * w1));
      }
      *reinterpret_cast<uint4*>(wrow + 8 * j) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
      if (fan_row) *reinterpret_cast<uint4*>(fan_row + 8 * j) = make_uint4(nw[0], nw[1], nw[2], nw[3]);
    }
  }
}

__device__ __forceinline__ void tmem_alloc_dyn(uint32_t holder_smem, uint32_t cols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(holder_smem), "r"(cols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc_dyn(uint32_t taddr, uint32_t cols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void named_bar_sync(uint32_t id, uint32_t n) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory");
}

// 64 accumulator columns of this thread's row -> registers
__device__ __forceinline__ void ld64(uint32_t taddr, uint32_t (&v)[64]) {
  uint32_t lo[32], hi[32];
  ptx::tmem_ld32(taddr, lo);
  ptx::tmem_ld32(taddr + 32, hi);
  ptx::tmem_ld_wait();
#pragma unroll
  for (int j = 0; j < 32; ++j) { v[j] = lo[j]; v[32 + j] = hi[j]; }
}

// this thread's 64 bf16 (128 B) of one panel row, 128-byte swizzled: 16-byte chunk j sits at j ^ (row & 7)
__device__ __forceinline__ void st_row(uint32_t row_addr, uint32_t sw, const uint32_t (&pk)[32]) {
#pragma unroll
  for (int j = 0; j < 8; ++j)
    ptx::st_shared_v4(row_addr + (((uint32_t)j << 4) ^ sw), pk[4 * j], pk[4 * j + 1], pk[4 * j + 2], pk[4 * j + 3]);
}

__global__ void __launch_bounds__(kThreadsF, 2) k_ns_fused(const FusedParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  const uint32_t x0 = ptx::smem_u32(smem);                 // X panels
  const uint32_t a0 = x0 + p.x_bytes;                      // A / P panels
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + p.x_bytes + kABytesF);
  const uint32_t bar_load = ptx::smem_u32(bars), bar_mma = ptx::smem_u32(bars + 1);
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 2);
  uint32_t* next_holder = tmem_holder + 1;
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    ptx::mbar_init(bar_load, 1);
    ptx::mbar_init(bar_mma, 1);
    ptx::fence_barrier_init();
  }
  if (warp == 4) tmem_alloc_dyn(ptx::smem_u32(tmem_holder), p.tmem_cols);
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;
  uint32_t load_phase = 0, mma_phase = 0;

  for (;;) {
    if (threadIdx.x == 0) *next_holder = atomicAdd(p.counter, 1u);
    __syncthreads();
    const uint32_t idx = *next_holder;
    if (idx >= p.n_list) break;
    const FusedMat fm = p.list[idx];
    const CUtensorMap* tm = p.tmaps + TM_COUNT * (size_t)fm.mat;
    const uint32_t panel_bytes = fm.rpad * 128u;
    const uint32_t d16 = fm.d16;
    const uint32_t kd = d16 >> 4;                            // 16-element k steps over d

    // ---- X~ -> shared memory: 64 x 64 boxes, rows and columns beyond the matrix zero-filled ----
    if (warp == 4) {
      if (ptx::elect_one()) {
        const uint32_t row_boxes = fm.rpad >> 6;
        ptx::mbar_arrive_expect_tx(bar_load, fm.panels * row_boxes * 8192u);
        for (uint32_t pn = 0; pn < fm.panels; ++pn)
          for (uint32_t rb = 0; rb < row_boxes; ++rb)
            ptx::tma_load_2d(x0 + pn * panel_bytes + rb * 8192u, tm + TM_X0, (int)(pn * 64), (int)(rb * 64), bar_load);
      }
      __syncwarp();
    }
    ptx::mbar_wait(bar_load, load_phase);
    load_phase ^= 1;

    const float inv = p.inv_norm[fm.mat];
    const uint32_t n_dchunks = (d16 + 63) >> 6;              // 64-column chunks of a d-wide accumulator
    const uint32_t n_rb = fm.rpad >> 7;                      // 128-row blocks of X (tall: several; wide: 1)

    // last iteration: the APPLY epilogue also updates W (this thread's rows of it) from the O values it holds
    float coef = 0.f;
    __nv_bfloat16 *wmat = nullptr, *fmat = nullptr;          // the matrix in W, and its optional fan-out copy
    if (p.ua.W != nullptr) {
      const TcUpd* u = p.ua.upd + fm.mat;
      coef = (float)(p.ua.lr * u->scale[p.ua.scale_mode]);
      wmat = reinterpret_cast<__nv_bfloat16*>(p.ua.W) + u->elem_off;
      if (p.ua.fan) fmat = reinterpret_cast<__nv_bfloat16*>(p.ua.fan[fm.mat]);
    }

    for (uint32_t it = 0; it < p.ns_steps; ++it) {
      const float alpha = it == 0 ? inv * inv : 1.f, beta = it == 0 ? inv : 1.f;
      const bool upd = wmat != nullptr && it + 1 == p.ns_steps;
#pragma unroll 1
      for (uint32_t ph = 0; ph < 3; ++ph) {
        if (warp == 4) {
          // ===== UMMA issue: the whole phase, then one commit =====
          ptx::tc_fence_after();
          if (ptx::elect_one()) {
            if (ph == PH_GRAM) {
              if (!fm.tall) {                                // A = X X^T: both operands K-major, one panel per 64 k
                const uint32_t idesc = ptx::idesc_bf16_f32(128, d16, 0, 0);
                for (uint32_t s = 0; s < fm.k16; ++s) {
                  const uint32_t addr = x0 + (s >> 2) * panel_bytes + (s & 3u) * 32u;
                  const uint64_t desc = ptx::smem_desc_sw128(addr, 16, 1024);
                  ptx::umma_bf16(tmem_base, desc, desc, idesc, s != 0);
                }
              } else {                                       // A = X^T X: both operands MN-major, 16 rows of X per step
                const uint32_t idesc = ptx::idesc_bf16_f32(128, d16, 1, 1);
                for (uint32_t s = 0; s < fm.k16; ++s) {
                  const uint64_t desc = ptx::smem_desc_sw128(x0 + s * 2048u, panel_bytes, 1024);
                  ptx::umma_bf16(tmem_base, desc, desc, idesc, s != 0);
                }
              }
            } else if (ph == PH_POLY) {                      // A A: both operands K-major from the A panels
              const uint32_t idesc = ptx::idesc_bf16_f32(128, d16, 0, 0);
              for (uint32_t s = 0; s < kd; ++s) {
                const uint64_t desc = ptx::smem_desc_sw128(a0 + (s >> 2) * 16384u + (s & 3u) * 32u, 16, 1024);
                ptx::umma_bf16(tmem_base, desc, desc, idesc, s != 0);
              }
            } else if (!fm.tall) {                           // X_new (d x n) = P (K-major) X (MN-major), 256 columns at a time
              const uint32_t cpad = fm.panels * 64u;
              for (uint32_t c0 = 0; c0 < cpad; c0 += 256u) {
                const uint32_t nc = min(256u, cpad - c0);
                const uint32_t idesc = ptx::idesc_bf16_f32(128, nc, 0, 1);
                for (uint32_t s = 0; s < kd; ++s) {
                  const uint64_t ad = ptx::smem_desc_sw128(a0 + (s >> 2) * 16384u + (s & 3u) * 32u, 16, 1024);
                  const uint64_t bd = ptx::smem_desc_sw128(x0 + (c0 >> 6) * panel_bytes + s * 2048u, panel_bytes, 1024);
                  ptx::umma_bf16(tmem_base + c0, ad, bd, idesc, s != 0);
                }
              }
            } else {                                         // X_new (n x d) = X (K-major) P^T, P symmetric (K-major)
              const uint32_t idesc = ptx::idesc_bf16_f32(128, d16, 0, 0);
              for (uint32_t rb = 0; rb < n_rb; ++rb)
                for (uint32_t s = 0; s < kd; ++s) {
                  const uint64_t ad = ptx::smem_desc_sw128(x0 + (s >> 2) * panel_bytes + rb * 16384u + (s & 3u) * 32u, 16, 1024);
                  const uint64_t bd = ptx::smem_desc_sw128(a0 + (s >> 2) * 16384u + (s & 3u) * 32u, 16, 1024);
                  ptx::umma_bf16(tmem_base + rb * 128u, ad, bd, idesc, s != 0);
                }
            }
            ptx::umma_commit(bar_mma);
          }
          __syncwarp();
        } else {
          // ===== epilogue: this thread owns accumulator row r = 32 warp + lane =====
          ptx::mbar_wait(bar_mma, mma_phase);
          ptx::tc_fence_after();
          const uint32_t r = warp * 32u + lane;
          const uint32_t sw = (r & 7u) << 4;
          const uint32_t taddr = tmem_base + ((warp * 32u) << 16);
          uint32_t v[64], pk[32];
          if (ph == PH_GRAM) {
            for (uint32_t cc = 0; cc < n_dchunks; ++cc) {
              ld64(taddr + 64u * cc, v);
#pragma unroll
              for (int j = 0; j < 32; ++j)
                pk[j] = pack_bf16f(alpha * __uint_as_float(v[2 * j]), alpha * __uint_as_float(v[2 * j + 1]));
              st_row(a0 + cc * 16384u + r * 128u, sw, pk);
            }
          } else if (ph == PH_POLY) {
            for (uint32_t cc = 0; cc < n_dchunks; ++cc) {
              const uint32_t row_addr = a0 + cc * 16384u + r * 128u;
              uint32_t aw[32];
#pragma unroll
              for (int j = 0; j < 8; ++j)
                ptx::ld_shared_v4(row_addr + (((uint32_t)j << 4) ^ sw), aw[4 * j], aw[4 * j + 1], aw[4 * j + 2], aw[4 * j + 3]);
              ld64(taddr + 64u * cc, v);
              const bool on_diag = (r >> 6) == cc;
#pragma unroll
              for (int j = 0; j < 32; ++j) {
                float f0 = fmaf(p.c, __uint_as_float(v[2 * j]), p.b * __uint_as_float(aw[j] << 16));
                float f1 = fmaf(p.c, __uint_as_float(v[2 * j + 1]), p.b * __uint_as_float(aw[j] & 0xffff0000u));
                if (on_diag) {
                  if (64u * cc + 2 * j == r) f0 += p.a;
                  if (64u * cc + 2 * j + 1 == r) f1 += p.a;
                }
                pk[j] = pack_bf16f(f0, f1);
              }
              st_row(row_addr, sw, pk);                      // P over A, in place (every UMMA that read A has completed)
            }
          } else if (!fm.tall) {
            for (uint32_t cc = 0; cc < fm.panels; ++cc) {
              ld64(taddr + 64u * cc, v);
#pragma unroll
              for (int j = 0; j < 32; ++j)
                pk[j] = pack_bf16f(beta * __uint_as_float(v[2 * j]), beta * __uint_as_float(v[2 * j + 1]));
              st_row(x0 + cc * panel_bytes + r * 128u, sw, pk);
              if (upd && r < fm.rows && 64u * cc < fm.cols)
                update_row64(wmat + (size_t)r * fm.cols + 64u * cc, fmat ? fmat + (size_t)r * fm.cols + 64u * cc : nullptr,
                             fm.cols - 64u * cc, pk, coef, p.ua.decay);
            }
          } else {
            for (uint32_t rb = 0; rb < n_rb; ++rb)
              for (uint32_t cc = 0; cc < n_dchunks; ++cc) {
                ld64(taddr + rb * 128u + 64u * cc, v);
#pragma unroll
                for (int j = 0; j < 32; ++j)
                  pk[j] = pack_bf16f(beta * __uint_as_float(v[2 * j]), beta * __uint_as_float(v[2 * j + 1]));
                st_row(x0 + cc * panel_bytes + (rb * 128u + r) * 128u, sw, pk);
                if (upd && rb * 128u + r < fm.rows && 64u * cc < fm.cols)
                  update_row64(wmat + (size_t)(rb * 128u + r) * fm.cols + 64u * cc,
                               fmat ? fmat + (size_t)(rb * 128u + r) * fm.cols + 64u * cc : nullptr, fm.cols - 64u * cc, pk,
                               coef, p.ua.decay);
              }
          }
          ptx::fence_async_smem();                           // generic-proxy writes -> the next UMMAs / the TMA store
          ptx::tc_fence_before();
        }
        mma_phase ^= 1;
        named_bar_sync(1, kThreadsF);
      }
    }

    // ---- O = X_K -> global (the buffer mfsdp_workspace_view reports), 32-row x 64-column boxes clipped at the edges ----
    if (warp == 4 && (wmat == nullptr || p.ua.keep_o)) {
      if (ptx::elect_one()) {
        const CUtensorMap* tout = tm + TM_X0_ST + (p.ns_steps & 1u);
        const uint32_t col_panels = (fm.cols + 63u) >> 6;
        for (uint32_t pn = 0; pn < col_panels; ++pn)
          for (uint32_t r0 = 0; r0 < fm.rows; r0 += 32u)
            ptx::tma_store_2d(tout, (int)(pn * 64), (int)r0, x0 + pn * panel_bytes + r0 * 128u);
        ptx::bulk_commit();
        ptx::bulk_wait_read<0>();                            // shared memory may be overwritten by the next matrix
      }
      __syncwarp();
    }
    __syncthreads();
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 4) {
    ptx::tc_fence_after();
    tmem_dealloc_dyn(tmem_base, p.tmem_cols);
  }
}

uint32_t smem_bytes_cls(int cls) { return kXBytesCls[cls] + kABytesF + kBarBytesF + 1024; }

}  // namespace

// Which matrices run here: d < below_d (<= 129), padded X within 128 KB.  Fills the launch record and the size class.
bool fused_eligible(uint32_t rows, uint32_t cols, uint32_t below_d, FusedMat* out, int* cls) {
  const uint32_t d = std::min(rows, cols), n = std::max(rows, cols);
  if (d >= below_d || d > 128u) return false;
  const bool tall = rows > cols;
  FusedMat f;
  f.mat = 0; f.rows = rows; f.cols = cols; f.tall = tall ? 1u : 0u;
  f.d16 = (d + 15u) / 16u * 16u;
  f.rpad = tall ? (n + 127u) / 128u * 128u : 128u;
  f.panels = tall ? 2u : (n + 63u) / 64u;
  f.k16 = (n + 15u) / 16u;
  const uint64_t xb = (uint64_t)f.rpad * 128u * f.panels;
  if (xb > kXBytesCls[1]) return false;
  *cls = xb <= kXBytesCls[0] ? 0 : 1;
  *out = f;
  return true;
}

int fused_setup() {
  const cudaError_t e = cudaFuncSetAttribute(k_ns_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_bytes_cls(1));
  return e == cudaSuccess ? MFSDP_OK : cuda_fail(e);
}

int launch_ns_fused(const NsTcPlan& tc, int cls, uint8_t* ws, const float* inv_norm, const mfsdp_muon_hparams_t& hp,
                    const UpdArgs& ua, cudaStream_t st) {
  (void)ws;
  if (tc.n_fused[cls] == 0) return MFSDP_OK;
  FusedParams p;
  p.list = tc.d_fused[cls];
  p.n_list = tc.n_fused[cls];
  p.tmaps = tc.d_tmaps;
  p.inv_norm = inv_norm;
  p.counter = tc.d_counters + 2 + cls;
  p.x_bytes = kXBytesCls[cls];
  p.tmem_cols = kTmemColsCls[cls];
  p.ns_steps = (uint32_t)hp.ns_steps;
  p.a = (float)hp.a; p.b = (float)hp.b; p.c = (float)hp.c;
  p.ua = ua;
  const uint32_t per_sm = cls == 0 ? 2u : 1u;
  const uint32_t grid = std::min<uint32_t>(p.n_list, (uint32_t)tc.sms * per_sm);
  k_ns_fused<<<grid, kThreadsF, smem_bytes_cls(cls), st>>>(p);
  count_launch();
  return check_last_launch();
}

}  // namespace mfsdp
