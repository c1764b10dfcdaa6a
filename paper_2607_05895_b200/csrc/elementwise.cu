// HBM-bound passes of the owner-local step, one grid over all resident segments.
//   k_momentum  M <- mu M + (1-mu) G ; U = (1-mu) G + mu M | M ; X~ = cast(U) ; partial sums of U^2
//               (k_momentum_gated: the same per chunk, matrices taken in the order their gradients land)
//   k_ssq       fixed-order reduction of the partials -> ||U||_F^2 (double), 1 / max(||U||_F, eps) (float)
//   k_update    W <- W (1 - lr wd) - lr s(rows, cols) O
//   k_adamw     decoupled-decay Adam on the packed tails
// Work unit = a chunk of kChunk consecutive elements of ONE segment (never straddles segments), so every access
// is a 128-bit vector on a 128-byte aligned run; chunk -> segment through a host-built table.  A thread owns
// kVecPerThread 8-element vectors of the chunk and moves them in batches of kBatch: all loads of a batch are issued
// before the first use, so each thread keeps 4-12 independent 128-bit loads in flight (HBM latency x bandwidth needs
// ~40 KB in flight per SM).
#include <cuda_bf16.h>

#include <algorithm>

#include "mfsdp_internal.h"

namespace mfsdp {
namespace {

constexpr int kVecPerThread = (int)(kChunk / (kEwThreads * 8));   // 8
constexpr int kBatch = 4;                                          // vectors per batch
static_assert(kVecPerThread % kBatch == 0, "chunk = whole batches");

// ---- 8-element vector access ------------------------------------------------------------------------------------
struct F8 { float v[8]; };

__device__ __forceinline__ F8 load8(const float* p) {
  F8 r;
  const float4 a = *reinterpret_cast<const float4*>(p);
  const float4 b = *reinterpret_cast<const float4*>(p + 4);
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w; r.v[4] = b.x; r.v[5] = b.y; r.v[6] = b.z; r.v[7] = b.w;
  return r;
}
__device__ __forceinline__ F8 load8(const __nv_bfloat16* p) {
  F8 r;
  const uint4 u = *reinterpret_cast<const uint4*>(p);
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {               // bf16 -> fp32 is a 16-bit shift
    r.v[2 * i] = __uint_as_float(w[i] << 16);
    r.v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
  return r;
}
__device__ __forceinline__ F8 load8_ro(const float* p) {
  F8 r;
  const float4 a = __ldg(reinterpret_cast<const float4*>(p));
  const float4 b = __ldg(reinterpret_cast<const float4*>(p + 4));
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w; r.v[4] = b.x; r.v[5] = b.y; r.v[6] = b.z; r.v[7] = b.w;
  return r;
}
__device__ __forceinline__ F8 load8_ro(const __nv_bfloat16* p) {
  F8 r;
  const uint4 u = __ldg(reinterpret_cast<const uint4*>(p));
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    r.v[2 * i] = __uint_as_float(w[i] << 16);
    r.v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
  return r;
}
__device__ __forceinline__ void store8_cs(__nv_bfloat16* p, const F8& x) {
  uint32_t w[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(x.v[2 * i], x.v[2 * i + 1]);   // RNE
    w[i] = *reinterpret_cast<const uint32_t*>(&h);
  }
  __stcs(reinterpret_cast<uint4*>(p), make_uint4(w[0], w[1], w[2], w[3]));
}
// L2-only loads (gated pass: the gradient is written by another agent -- copy engine, peer GPU -- while this kernel runs)
__device__ __forceinline__ F8 load8_cg(const float* p) {
  F8 r;
  const float4 a = __ldcg(reinterpret_cast<const float4*>(p));
  const float4 b = __ldcg(reinterpret_cast<const float4*>(p + 4));
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w; r.v[4] = b.x; r.v[5] = b.y; r.v[6] = b.z; r.v[7] = b.w;
  return r;
}
__device__ __forceinline__ F8 load8_cg(const __nv_bfloat16* p) {
  F8 r;
  const uint4 u = __ldcg(reinterpret_cast<const uint4*>(p));
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    r.v[2 * i] = __uint_as_float(w[i] << 16);
    r.v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
  return r;
}
__device__ __forceinline__ float load1_cg(const float* p) { return __ldcg(p); }
__device__ __forceinline__ float load1_cg(const __nv_bfloat16* p) {
  return __uint_as_float((uint32_t)__ldcg(reinterpret_cast<const unsigned short*>(p)) << 16);
}
__device__ __forceinline__ void store8(float* p, const F8& x) {
  *reinterpret_cast<float4*>(p) = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]);
  *reinterpret_cast<float4*>(p + 4) = make_float4(x.v[4], x.v[5], x.v[6], x.v[7]);
}
// streaming (evict-first) forms for data that is touched exactly once per pass
__device__ __forceinline__ F8 load8_cs(const float* p) {
  F8 r;
  const float4 a = __ldcs(reinterpret_cast<const float4*>(p));
  const float4 b = __ldcs(reinterpret_cast<const float4*>(p + 4));
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w; r.v[4] = b.x; r.v[5] = b.y; r.v[6] = b.z; r.v[7] = b.w;
  return r;
}
__device__ __forceinline__ void store8_cs(float* p, const F8& x) {
  __stcs(reinterpret_cast<float4*>(p), make_float4(x.v[0], x.v[1], x.v[2], x.v[3]));
  __stcs(reinterpret_cast<float4*>(p + 4), make_float4(x.v[4], x.v[5], x.v[6], x.v[7]));
}
__device__ __forceinline__ void store8(__nv_bfloat16* p, const F8& x) {
  uint32_t w[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(x.v[2 * i], x.v[2 * i + 1]);   // RNE
    w[i] = *reinterpret_cast<const uint32_t*>(&h);
  }
  *reinterpret_cast<uint4*>(p) = make_uint4(w[0], w[1], w[2], w[3]);
}
__device__ __forceinline__ float load1(const float* p) { return *p; }
__device__ __forceinline__ float load1(const __nv_bfloat16* p) { return __bfloat162float(*p); }
__device__ __forceinline__ void store1(float* p, float x) { *p = x; }
__device__ __forceinline__ void store1(__nv_bfloat16* p, float x) { *p = __float2bfloat16_rn(x); }

// Deterministic block sum (fixed shuffle tree, then warp 0 in order).  Result valid in thread 0.
__device__ __forceinline__ double block_sum(double x, double* smem) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (lane == 0) smem[warp] = x;
  __syncthreads();
  double s = 0.0;
  if (threadIdx.x == 0)
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += smem[w];
  __syncthreads();
  return s;
}

// ---- a1: momentum + Nesterov + cast + partial squared norm ---------------------------------------------------------
// One chunk.  kL2: G is read through L2 only (gated pass: the gradient is written by another agent while the kernel runs).
template <typename GT, typename XT, bool kL2>
__device__ __forceinline__ void momentum_chunk(const MatLayout* __restrict__ mats, uint32_t mi, uint32_t c,
                                               const GT* __restrict__ G, float* __restrict__ M,
                                               uint8_t* __restrict__ ws, double* __restrict__ partial, float mu,
                                               float omm, int nesterov, double* red) {
  const MatLayout L = mats[mi];
  const uint64_t base = (uint64_t)(c - L.chunk_begin) * kChunk;
  const GT* g = G + L.elem_off;
  float* m = M + L.elem_off;
  XT* x = reinterpret_cast<XT*>(ws + L.x_off[0]);
  const bool vec = (L.cols % 8u) == 0u;      // then pitch_x == cols and a vector never straddles a row
  double acc = 0.0;
  if (vec && base + kChunk <= L.numel) {     // full chunk: batched 128-bit accesses
#pragma unroll
    for (int b = 0; b < kVecPerThread / kBatch; ++b) {
      F8 gv[kBatch], mv[kBatch];
#pragma unroll
      for (int v = 0; v < kBatch; ++v) {
        const uint64_t e0 = base + ((uint64_t)(b * kBatch + v) * kEwThreads + threadIdx.x) * 8;
        gv[v] = kL2 ? load8_cg(g + e0) : load8_ro(g + e0);
        mv[v] = load8_cs(m + e0);
      }
#pragma unroll
      for (int v = 0; v < kBatch; ++v) {
        const uint64_t e0 = base + ((uint64_t)(b * kBatch + v) * kEwThreads + threadIdx.x) * 8;
        F8 uv;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float gs = omm * gv[v].v[i];
          mv[v].v[i] = fmaf(mu, mv[v].v[i], gs);                       // M <- mu M + (1-mu) G
          uv.v[i] = nesterov ? fmaf(mu, mv[v].v[i], gs) : mv[v].v[i];  // U = (1-mu) G + mu M   |   U = M
          acc = fma((double)uv.v[i], (double)uv.v[i], acc);
        }
        store8_cs(m + e0, mv[v]);        // M is touched once per step: evict-first
        store8(x + e0, uv);              // X~ is the next kernel's input: keep it in L2 (small sets fit)
      }
    }
  } else {                                   // ragged chunk or odd pitch: same element -> thread mapping, guarded
    for (int it = 0; it < kVecPerThread; ++it) {
      const uint64_t e0 = base + ((uint64_t)it * kEwThreads + threadIdx.x) * 8;
      if (e0 >= L.numel) break;
      if (vec && e0 + 8 <= L.numel) {
        const F8 gv = kL2 ? load8_cg(g + e0) : load8_ro(g + e0);
        F8 mv = load8(m + e0);
        F8 uv;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float gs = omm * gv.v[i];
          mv.v[i] = fmaf(mu, mv.v[i], gs);
          uv.v[i] = nesterov ? fmaf(mu, mv.v[i], gs) : mv.v[i];
          acc = fma((double)uv.v[i], (double)uv.v[i], acc);
        }
        store8(m + e0, mv);
        store8(x + e0, uv);
      } else {
        const uint64_t e1 = (e0 + 8 < L.numel) ? e0 + 8 : L.numel;
        for (uint64_t e = e0; e < e1; ++e) {
          const float gs = omm * (kL2 ? load1_cg(g + e) : load1(g + e));
          const float mn = fmaf(mu, m[e], gs);
          const float u = nesterov ? fmaf(mu, mn, gs) : mn;
          acc = fma((double)u, (double)u, acc);
          m[e] = mn;
          const uint64_t r = e / L.cols, col = e - r * L.cols;
          store1(x + r * L.pitch_x + col, u);
        }
      }
    }
  }
  const double s = block_sum(acc, red);
  if (threadIdx.x == 0) partial[c] = s;
}

template <typename GT, typename XT>
__global__ void __launch_bounds__(kEwThreads) k_momentum(const MatLayout* __restrict__ mats,
                                                         const uint32_t* __restrict__ chunk_mat, uint32_t n_chunks,
                                                         const GT* __restrict__ G, float* __restrict__ M,
                                                         uint8_t* __restrict__ ws, double* __restrict__ partial,
                                                         float mu, float omm, int nesterov) {
  __shared__ double red[kEwThreads / 32];
  for (uint32_t c = blockIdx.x; c < n_chunks; c += gridDim.x)
    momentum_chunk<GT, XT, false>(mats, chunk_mat[c], c, G, M, ws, partial, mu, omm, nesterov, red);
}

// Gated form (mfsdp_muon_step_gated): the chunks of matrix i may be touched once ready[i] >= epoch.  A CTA owns the
// chunks c = blockIdx.x + k gridDim.x; consecutive ones of one matrix form a RUN.  The CTA lists its runs once, then
// sweeps the list: a run whose flag is up is processed and dropped, the others stay for the next sweep.  So the order
// in which the gradients land does not matter -- with the reduction's reverse block order (mfsdp_reduce_schedule) the
// LAST matrices of the table arrive first, and a CTA that waited for its first chunk's matrix would idle until the very
// last gradient.  Which run is processed when changes no value: every chunk's partial sum is written by the one CTA
// that owns it, in a fixed order.  More than kGateRuns runs per CTA (a table of thousands of tiny matrices): that CTA
// falls back to waiting in table order.
constexpr uint32_t kGateRuns = 2048;

__device__ __forceinline__ bool flag_up(const uint32_t* flag, uint32_t epoch) {
  uint32_t v;
  asm volatile("ld.acquire.sys.global.u32 %0, [%1];" : "=r"(v) : "l"(flag) : "memory");
  return (int32_t)(v - epoch) >= 0;
}

template <typename GT, typename XT>
__global__ void __launch_bounds__(kEwThreads) k_momentum_gated(const MatLayout* __restrict__ mats,
                                                               const uint32_t* __restrict__ chunk_mat,
                                                               const uint32_t* __restrict__ chunk_begin,
                                                               uint32_t n_chunks, const GT* __restrict__ G,
                                                               float* __restrict__ M, uint8_t* __restrict__ ws,
                                                               double* __restrict__ partial, float mu, float omm,
                                                               int nesterov, const uint32_t* __restrict__ ready,
                                                               uint32_t epoch) {
  __shared__ double red[kEwThreads / 32];
  __shared__ uint32_t run_first[kGateRuns];      // first chunk of each pending run
  __shared__ uint32_t n_runs_s;
  if (threadIdx.x == 0) n_runs_s = 0;
  __syncthreads();
  const uint32_t mine = blockIdx.x < n_chunks ? (n_chunks - blockIdx.x + gridDim.x - 1) / gridDim.x : 0u;
  for (uint32_t k = threadIdx.x; k < mine; k += kEwThreads) {
    const uint32_t c = blockIdx.x + k * gridDim.x;
    if (k == 0 || chunk_mat[c] != chunk_mat[c - gridDim.x]) {
      const uint32_t slot = atomicAdd(&n_runs_s, 1u);
      if (slot < kGateRuns) run_first[slot] = c;
    }
  }
  __syncthreads();
  uint32_t n_runs = n_runs_s;
  if (n_runs > kGateRuns) {                      // too many runs to list: wait in table order
    for (uint32_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
      const uint32_t mi = chunk_mat[c];
      if (threadIdx.x == 0 && !flag_up(ready + mi, epoch)) {
        const long long t0 = clock64();
        do {
          __nanosleep(200);
          if (clock64() - t0 > 20000000000ll) __trap();       // ~10 s: the producer never signalled
        } while (!flag_up(ready + mi, epoch));
      }
      __syncthreads();
      momentum_chunk<GT, XT, true>(mats, mi, c, G, M, ws, partial, mu, omm, nesterov, red);
    }
    return;
  }
  long long idle_since = 0;
  bool idle = false;
  while (n_runs) {
    uint32_t kept = 0;
    for (uint32_t j = 0; j < n_runs; ++j) {
      const uint32_t c0 = run_first[j];
      const uint32_t mi = chunk_mat[c0];
      const int up = __syncthreads_or(threadIdx.x == 0 ? (int)flag_up(ready + mi, epoch) : 0);
      if (!up) {                                 // every thread has read run_first[j] (barrier above); kept <= j
        if (threadIdx.x == 0) run_first[kept] = c0;
        ++kept;
        continue;
      }
      const uint32_t ce = chunk_begin[mi + 1];
      for (uint32_t c = c0; c < ce; c += gridDim.x)
        momentum_chunk<GT, XT, true>(mats, mi, c, G, M, ws, partial, mu, omm, nesterov, red);
    }
    __syncthreads();                             // run_first[0 .. kept) complete before the next sweep reads it
    if (kept == n_runs) {                        // a sweep without progress
      if (!idle) { idle = true; idle_since = clock64(); }
      else if (clock64() - idle_since > 20000000000ll) __trap();   // ~10 s: the producer never signalled
      __nanosleep(500);
    } else {
      idle = false;
    }
    n_runs = kept;
  }
}

// ---- a2 (scalar part): ||U||^2 and 1 / max(||U||, eps), one block per matrix, fixed order --------------------------
__global__ void __launch_bounds__(kEwThreads) k_ssq(const uint32_t* __restrict__ chunk_begin,
                                                    const double* __restrict__ partial, double* __restrict__ ssq,
                                                    float* __restrict__ inv_norm, double eps) {
  __shared__ double red[kEwThreads / 32];
  const uint32_t mi = blockIdx.x;
  const uint32_t b = chunk_begin[mi], e = chunk_begin[mi + 1];
  double acc = 0.0;
  for (uint32_t c = b + threadIdx.x; c < e; c += kEwThreads) acc += partial[c];
  const double s = block_sum(acc, red);
  if (threadIdx.x == 0) {
    ssq[mi] = s;
    const double nrm = sqrt(s);
    inv_norm[mi] = (float)(1.0 / (nrm > eps ? nrm : eps));
  }
}

// ---- a4: scaled, weight-decayed update ------------------------------------------------------------------------------
// s(rows, cols) is tabulated per matrix on the host (MatLayout::scale, one entry per MFSDP_SCALE_* mode).
template <typename WT, typename OT>
__global__ void __launch_bounds__(kEwThreads) k_update(const MatLayout* __restrict__ mats,
                                                       const uint32_t* __restrict__ chunk_mat, uint32_t n_chunks,
                                                       WT* __restrict__ W, const uint8_t* __restrict__ ws, int o_buf,
                                                       double lr, float decay, int scale_mode,
                                                       const uint64_t* __restrict__ fan) {
  for (uint32_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
    const uint32_t mi = chunk_mat[c];
    const MatLayout L = mats[mi];
    const uint64_t base = (uint64_t)(c - L.chunk_begin) * kChunk;
    WT* w = W + L.elem_off;
    WT* f = fan ? reinterpret_cast<WT*>(fan[mi]) : nullptr;    // fan-out copy of the updated matrix (rows x cols), or none
    const OT* o = reinterpret_cast<const OT*>(ws + (o_buf ? L.x_off[1] : L.x_off[0]));
    const float coef = (float)(lr * mats[mi].scale[scale_mode]);   // lr s, rounded once
    const bool vec = (L.cols % 8u) == 0u;
    if (vec && base + kChunk <= L.numel) {
#pragma unroll
      for (int b = 0; b < kVecPerThread / kBatch; ++b) {
        F8 wv[kBatch], ov[kBatch];
#pragma unroll
        for (int v = 0; v < kBatch; ++v) {
          const uint64_t e0 = base + ((uint64_t)(b * kBatch + v) * kEwThreads + threadIdx.x) * 8;
          wv[v] = load8(w + e0);
          ov[v] = load8_ro(o + e0);
        }
#pragma unroll
        for (int v = 0; v < kBatch; ++v) {
          const uint64_t e0 = base + ((uint64_t)(b * kBatch + v) * kEwThreads + threadIdx.x) * 8;
#pragma unroll
          for (int i = 0; i < 8; ++i) wv[v].v[i] = fmaf(-coef, ov[v].v[i], decay * wv[v].v[i]);
          store8(w + e0, wv[v]);
          if (f) store8(f + e0, wv[v]);
        }
      }
    } else {
      for (int it = 0; it < kVecPerThread; ++it) {
        const uint64_t e0 = base + ((uint64_t)it * kEwThreads + threadIdx.x) * 8;
        if (e0 >= L.numel) break;
        if (vec && e0 + 8 <= L.numel) {
          F8 wv = load8(w + e0);
          const F8 ov = load8(o + e0);
#pragma unroll
          for (int i = 0; i < 8; ++i) wv.v[i] = fmaf(-coef, ov.v[i], decay * wv.v[i]);
          store8(w + e0, wv);
          if (f) store8(f + e0, wv);
        } else {
          const uint64_t e1 = (e0 + 8 < L.numel) ? e0 + 8 : L.numel;
          for (uint64_t e = e0; e < e1; ++e) {
            const uint64_t r = e / L.cols, col = e - r * L.cols;
            const float ov = load1(o + r * L.pitch_x + col);
            const float wn = fmaf(-coef, ov, decay * load1(w + e));
            store1(w + e, wn);
            if (f) store1(f + e, wn);
          }
        }
      }
    }
  }
}

// ---- a5: AdamW on packed tails -----------------------------------------------------------------------------------------
struct AdamConst { float decay, b1, omb1, b2, omb2, inv_bc1, inv_bc2, lr, eps; };

__device__ __forceinline__ void adam1(float& p, float g, float& m, float& v, const AdamConst& k) {
  p *= k.decay;                                     // p <- p (1 - lr wd)
  m = fmaf(k.b1, m, k.omb1 * g);                    // m <- b1 m + (1-b1) g
  v = fmaf(k.b2, v, k.omb2 * (g * g));              // v <- b2 v + (1-b2) g^2
  const float mh = m * k.inv_bc1, vh = v * k.inv_bc2;
  p -= k.lr * (mh / (sqrtf(vh) + k.eps));           // p <- p - lr m^ / (sqrt(v^) + eps)
}

template <typename PT>
__global__ void __launch_bounds__(kEwThreads) k_adamw(const TailLayout* __restrict__ tails,
                                                      const uint32_t* __restrict__ chunk_tail, uint32_t n_chunks,
                                                      PT* __restrict__ P, const PT* __restrict__ G,
                                                      float* __restrict__ Mo, float* __restrict__ Vo, AdamConst k) {
  for (uint32_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
    const TailLayout L = tails[chunk_tail[c]];
    const uint64_t base = (uint64_t)(c - L.chunk_begin) * kTailChunk;
    PT* p = P + L.elem_off;
    const PT* g = G + L.elem_off;
    float* m = Mo + L.elem_off;
    float* v = Vo + L.elem_off;
    for (int it = 0; it < (int)(kTailChunk / (kEwThreads * 8)); ++it) {
      const uint64_t e0 = base + ((uint64_t)it * kEwThreads + threadIdx.x) * 8;
      if (e0 >= L.numel) break;
      if (e0 + 8 <= L.numel) {
        F8 pv = load8(p + e0);
        const F8 gv = load8_ro(g + e0);
        F8 mv = load8(m + e0), vv = load8(v + e0);
#pragma unroll
        for (int i = 0; i < 8; ++i) adam1(pv.v[i], gv.v[i], mv.v[i], vv.v[i], k);
        store8(p + e0, pv); store8(m + e0, mv); store8(v + e0, vv);
      } else {
        for (uint64_t e = e0; e < L.numel; ++e) {
          float pe = load1(p + e), me = m[e], ve = v[e];
          adam1(pe, load1(g + e), me, ve, k);
          store1(p + e, pe); m[e] = me; v[e] = ve;
        }
      }
    }
  }
}

int ew_grid(uint32_t n_chunks) {
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const uint32_t cap = (uint32_t)sms * 8u;        // 8 resident CTAs of 256 threads per SM
  return (int)(n_chunks < cap ? n_chunks : cap);
}

}  // namespace

int launch_momentum(const Plan& pl, const void* G, void* M, const mfsdp_muon_hparams_t& hp, cudaStream_t st,
                    const uint32_t* ready, uint32_t epoch) {
  const WsLayout& lay = pl.lay;
  const uint32_t n_mat = (uint32_t)lay.mats.size();
  if (n_mat == 0) return MFSDP_OK;
  uint8_t* ws = static_cast<uint8_t*>(pl.workspace);
  double* partial = reinterpret_cast<double*>(ws + lay.partial_off);
  const float mu = (float)hp.momentum, omm = (float)(1.0 - hp.momentum);
  // Gated: CTAs spin while they wait for their matrix; at most 2 per SM, so that whatever produces the gradients
  // (a copy kernel, a collective launched late) still finds room on every SM.
  int grid = ew_grid(lay.n_chunks);
  if (ready) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    grid = std::min(grid, 2 * sms);
  }
  const bool gbf = lay.mat_dtype == MFSDP_BF16, xbf = pl.precision == MFSDP_NS_BF16;
#define MOM(GT, XT)                                                                                                    \
  do {                                                                                                                 \
    if (ready)                                                                                                         \
      k_momentum_gated<GT, XT><<<grid, kEwThreads, 0, st>>>(pl.d_mats, pl.d_chunk_mat, pl.d_chunk_begin, lay.n_chunks, \
                                                            static_cast<const GT*>(G), static_cast<float*>(M), ws,     \
                                                            partial, mu, omm, hp.nesterov, ready, epoch);              \
    else                                                                                                               \
      k_momentum<GT, XT><<<grid, kEwThreads, 0, st>>>(pl.d_mats, pl.d_chunk_mat, lay.n_chunks,                         \
                                                      static_cast<const GT*>(G), static_cast<float*>(M), ws,           \
                                                      partial, mu, omm, hp.nesterov);                                  \
  } while (0)
  if (gbf && xbf) MOM(__nv_bfloat16, __nv_bfloat16);
  else if (gbf) MOM(__nv_bfloat16, float);
  else if (xbf) MOM(float, __nv_bfloat16);
  else MOM(float, float);
#undef MOM
  count_launch();
  int rc = check_last_launch();
  if (rc) return rc;
  k_ssq<<<n_mat, kEwThreads, 0, st>>>(pl.d_chunk_begin, partial, reinterpret_cast<double*>(ws + lay.ssq_off),
                                      reinterpret_cast<float*>(ws + lay.invn_off), hp.eps);
  count_launch();
  return check_last_launch();
}

int launch_update(const Plan& pl, void* W, const mfsdp_muon_hparams_t& hp, cudaStream_t st, const uint64_t* fan) {
  const WsLayout& lay = pl.lay;
  const uint32_t n_mat = (uint32_t)lay.mats.size();
  if (n_mat == 0) return MFSDP_OK;
  const uint8_t* ws = static_cast<const uint8_t*>(pl.workspace);
  const float decay = (float)(1.0 - hp.lr * hp.weight_decay);
  const int o_buf = hp.ns_steps & 1;
  const int grid = ew_grid(lay.n_chunks);
  const bool wbf = lay.mat_dtype == MFSDP_BF16, obf = pl.precision == MFSDP_NS_BF16;
#define UPD(WT, OT)                                                                                      \
  k_update<WT, OT><<<grid, kEwThreads, 0, st>>>(pl.d_mats, pl.d_chunk_mat, lay.n_chunks,                 \
                                                static_cast<WT*>(W), ws, o_buf, hp.lr, decay, hp.scale_mode, fan)
  if (wbf && obf) UPD(__nv_bfloat16, __nv_bfloat16);
  else if (wbf) UPD(__nv_bfloat16, float);
  else if (obf) UPD(float, __nv_bfloat16);
  else UPD(float, float);
#undef UPD
  count_launch();
  return check_last_launch();
}

int launch_adamw(const Plan& pl, void* P, const void* G, void* m, void* v, const mfsdp_adamw_hparams_t& hp,
                 cudaStream_t st) {
  const WsLayout& lay = pl.lay;
  const uint32_t n_tail = (uint32_t)lay.tails.size();
  if (n_tail == 0) return MFSDP_OK;
  AdamConst k;
  k.decay = (float)(1.0 - hp.lr * hp.weight_decay);
  k.b1 = (float)hp.beta1; k.omb1 = (float)(1.0 - hp.beta1);
  k.b2 = (float)hp.beta2; k.omb2 = (float)(1.0 - hp.beta2);
  double p1 = 1.0, p2 = 1.0;                          // beta^t by repeated squaring, in double
  { double b = hp.beta1, c = hp.beta2; for (int64_t t = hp.step; t > 0; t >>= 1) { if (t & 1) { p1 *= b; p2 *= c; } b *= b; c *= c; } }
  k.inv_bc1 = (float)(1.0 / (1.0 - p1));
  k.inv_bc2 = (float)(1.0 / (1.0 - p2));
  k.lr = (float)hp.lr; k.eps = (float)hp.eps;
  const int grid = ew_grid(lay.n_tail_chunks);
  if (lay.tail_dtype == MFSDP_BF16)
    k_adamw<__nv_bfloat16><<<grid, kEwThreads, 0, st>>>(pl.d_tails, pl.d_chunk_tail, lay.n_tail_chunks,
                                                        static_cast<__nv_bfloat16*>(P),
                                                        static_cast<const __nv_bfloat16*>(G), static_cast<float*>(m),
                                                        static_cast<float*>(v), k);
  else
    k_adamw<float><<<grid, kEwThreads, 0, st>>>(pl.d_tails, pl.d_chunk_tail, lay.n_tail_chunks,
                                                static_cast<float*>(P), static_cast<const float*>(G),
                                                static_cast<float*>(m), static_cast<float*>(v), k);
  count_launch();
  return check_last_launch();
}

}  // namespace mfsdp
