// Newton-Schulz on the 5th-generation tensor cores (MFSDP_NS_BF16): grouped, persistent, warp-specialised GEMM
// tiles for ALL resident matrices of ragged shapes in one launch per phase.
//
// Per iteration and matrix (north_star), with Y the d x n "wide" view of X (Y = X when
// rows <= cols, Y = X^T otherwise -- the transposition is done by the UMMA operand descriptors (MN-major operands),
// never by moving data):
//   GRAM   A = alpha Y Y^T            symmetric: only 128-blocks (I, J >= I) are computed, written and mirrored
//   POLY   P = a I + b A + c A A      symmetric, same tiling; the b A + a I terms are fused in the epilogue
//   APPLY  Y <- beta P Y              (the a X term of X <- a X + B X lives in P = aI + B)
// alpha = 1/||U||^2 and beta = 1/||U|| at iteration 0 (Frobenius normalisation folded in), 1 afterwards.
//
// Kernel anatomy (one CTA per SM, 192 threads): warp 0 = TMA producer (one lane), warp 1 = TMEM owner + UMMA issuer
// (one lane), warps 2-5 = epilogue (TMEM -> registers -> global).  A 4-stage smem ring (128 x 64 A-operand +
// up to 256 x 64 B-operand, bf16, 128-byte swizzle) feeds tcgen05.mma M = 128, N = 64..256, K = 16; two TMEM
// accumulator stages (2 x 256 columns) let the epilogue of tile t overlap the main loop of tile t + 1.
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
struct TcTile { uint32_t mat, m0, n0; uint16_t nkb, nw; };   // output tile origin (rows, cols of the OUTPUT buffer), k blocks, UMMA N (multiple of 64)

struct NsTcPlan {
  CUtensorMap* d_tmaps = nullptr;   // 4 per matrix: X0, X1, A, P   (box 64 x 64 bf16, 128-byte swizzle)
  TcMat* d_mats = nullptr;
  TcTile* d_tiles[3] = {nullptr, nullptr, nullptr};
  uint32_t n_tiles[3] = {0, 0, 0};
  int sms = 148;
};

namespace {

constexpr uint32_t kBM = 128;                  // UMMA M
constexpr uint32_t kBNMax = 256;               // max UMMA N per tile
constexpr uint32_t kBK = 64;                   // k elements per stage (one 128-byte swizzle row)
constexpr uint32_t kBoxBytes = 64 * 64 * 2;    // one TMA box: 64 rows x 128 B
constexpr uint32_t kABytes = 2 * kBoxBytes;    // 128 x 64
constexpr uint32_t kBBytes = 4 * kBoxBytes;    // 256 x 64
constexpr uint32_t kStageBytes = kABytes + kBBytes;
constexpr uint32_t kStages = 4;
constexpr uint32_t kThreads = 192;
constexpr uint32_t kTmemCols = 512;
constexpr uint32_t kSmemBytes = kStages * kStageBytes + 1024 /*align slack*/ + 256 /*barriers*/;

struct TcParams {
  const TcTile* tiles;
  uint32_t n_tiles;
  const TcMat* mats;
  const CUtensorMap* tmaps;
  uint8_t* ws;
  const float* inv_norm;
  int phase, src, first;
  float a, b, c;
};

struct TileCfg {
  const CUtensorMap *ta, *tb;
  uint32_t a_mn, b_mn;          // operand majorness (1 = MN-major)
  uint32_t a_boxes, b_boxes;    // 64-row (K-major) / 64-column (MN-major) boxes to load
  uint32_t n_valid;             // UMMA N
  uint32_t out_rows, out_cols;  // bounds of the output buffer
};

__device__ __forceinline__ TileCfg decode(const TcParams& p, const TcTile& t, const TcMat& M) {
  TileCfg c;
  const CUtensorMap* tm = p.tmaps + 4 * (size_t)t.mat;
  uint32_t a_ext, b_ext;
  if (p.phase == PH_GRAM) {
    c.ta = c.tb = tm + p.src; c.a_mn = c.b_mn = M.tall; a_ext = b_ext = M.d; c.out_rows = c.out_cols = M.d;
  } else if (p.phase == PH_POLY) {
    c.ta = c.tb = tm + 2; c.a_mn = c.b_mn = 0; a_ext = b_ext = M.d; c.out_rows = c.out_cols = M.d;
  } else if (!M.tall) {          // X_new (d x n) = P (K-major) * X (k x n, MN-major)
    c.ta = tm + 3; c.a_mn = 0; a_ext = M.d; c.tb = tm + p.src; c.b_mn = 1; b_ext = M.cols;
    c.out_rows = M.rows; c.out_cols = M.cols;
  } else {                       // X_new (n x d) = X (K-major) * P^T, P symmetric (K-major)
    c.ta = tm + p.src; c.a_mn = 0; a_ext = M.rows; c.tb = tm + 3; c.b_mn = 0; b_ext = M.d;
    c.out_rows = M.rows; c.out_cols = M.cols;
  }
  c.a_boxes = (a_ext - t.m0 > 64u) ? 2u : 1u;
  (void)b_ext;
  c.n_valid = t.nw;
  c.b_boxes = c.n_valid >> 6;
  return c;
}

__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}

__global__ void __launch_bounds__(kThreads, 1) k_ns_tc(const TcParams p) {
  extern __shared__ uint8_t smem_raw[];
  uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
  uint64_t* bars = reinterpret_cast<uint64_t*>(smem + kStages * kStageBytes);
  const uint32_t full0 = ptx::smem_u32(bars), empty0 = ptx::smem_u32(bars + kStages);
  const uint32_t tfull0 = ptx::smem_u32(bars + 2 * kStages), tempty0 = ptx::smem_u32(bars + 2 * kStages + 2);
  uint32_t* tmem_holder = reinterpret_cast<uint32_t*>(bars + 2 * kStages + 4);
  const uint32_t stage0 = ptx::smem_u32(smem);
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (uint32_t s = 0; s < kStages; ++s) { ptx::mbar_init(full0 + 8 * s, 1); ptx::mbar_init(empty0 + 8 * s, 1); }
    for (uint32_t s = 0; s < 2; ++s) { ptx::mbar_init(tfull0 + 8 * s, 1); ptx::mbar_init(tempty0 + 8 * s, 4); }
    ptx::fence_barrier_init();
  }
  if (warp == 1) ptx::tmem_alloc<kTmemCols>(ptx::smem_u32(tmem_holder));
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_holder;

  if (warp == 0) {
    // ===== TMA producer =====
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      for (uint32_t ti = blockIdx.x; ti < p.n_tiles; ti += gridDim.x) {
        const TcTile t = p.tiles[ti];
        const TcMat M = p.mats[t.mat];
        const TileCfg c = decode(p, t, M);
        const uint32_t tx = (c.a_boxes + c.b_boxes) * kBoxBytes;
        for (uint32_t kb = 0; kb < t.nkb; ++kb) {
          ptx::mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t fb = full0 + 8 * stage;
          ptx::mbar_arrive_expect_tx(fb, tx);
          const uint32_t sa = stage0 + stage * kStageBytes, sb = sa + kABytes;
          const int k0 = (int)(kb * kBK);
          for (uint32_t h = 0; h < c.a_boxes; ++h) {
            const int mn = (int)(t.m0 + 64 * h);
            ptx::tma_load_2d(sa + h * kBoxBytes, c.ta, c.a_mn ? mn : k0, c.a_mn ? k0 : mn, fb);
          }
          for (uint32_t j = 0; j < c.b_boxes; ++j) {
            const int mn = (int)(t.n0 + 64 * j);
            ptx::tma_load_2d(sb + j * kBoxBytes, c.tb, c.b_mn ? mn : k0, c.b_mn ? k0 : mn, fb);
          }
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ===== UMMA issuer =====
    if (lane == 0) {
      uint32_t stage = 0, phase = 0, acc = 0, acc_phase = 0;
      for (uint32_t ti = blockIdx.x; ti < p.n_tiles; ti += gridDim.x) {
        const TcTile t = p.tiles[ti];
        const TcMat M = p.mats[t.mat];
        const TileCfg c = decode(p, t, M);
        const uint32_t idesc = ptx::idesc_bf16_f32(kBM, c.n_valid, c.a_mn, c.b_mn);
        // K-major: +32 B per 16-k step; MN-major: +16 rows of 128 B.  (descriptor address field is in 16-byte units)
        const uint32_t a_step = c.a_mn ? (2048u >> 4) : (32u >> 4), b_step = c.b_mn ? (2048u >> 4) : (32u >> 4);
        const uint32_t a_lbo = c.a_mn ? kBoxBytes : 16u, b_lbo = c.b_mn ? kBoxBytes : 16u;
        ptx::mbar_wait(tempty0 + 8 * acc, acc_phase ^ 1);       // epilogue has drained this accumulator
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + acc * kBNMax;
        for (uint32_t kb = 0; kb < t.nkb; ++kb) {
          ptx::mbar_wait(full0 + 8 * stage, phase);
          ptx::tc_fence_after();
          const uint32_t sa = stage0 + stage * kStageBytes, sb = sa + kABytes;
          const uint64_t ad = ptx::smem_desc_sw128(sa, a_lbo, 1024), bd = ptx::smem_desc_sw128(sb, b_lbo, 1024);
#pragma unroll
          for (uint32_t ks = 0; ks < kBK / 16; ++ks)
            ptx::umma_bf16(d_tmem, ad + (uint64_t)(ks * a_step), bd + (uint64_t)(ks * b_step), idesc, (kb | ks) != 0);
          ptx::umma_commit(empty0 + 8 * stage);                  // frees the smem slot when these MMAs finish
          if (++stage == kStages) { stage = 0; phase ^= 1; }
        }
        ptx::umma_commit(tfull0 + 8 * acc);                      // accumulator ready for the epilogue
        if (++acc == 2) { acc = 0; acc_phase ^= 1; }
      }
    }
  } else {
    // ===== epilogue: warps 2..5, warp w owns TMEM lanes 32 (w % 4) .. + 31 =====
    const uint32_t q = warp & 3;
    uint32_t acc = 0, acc_phase = 0;
    for (uint32_t ti = blockIdx.x; ti < p.n_tiles; ti += gridDim.x) {
      const TcTile t = p.tiles[ti];
      const TcMat M = p.mats[t.mat];
      const TileCfg c = decode(p, t, M);
      const float inv = p.first ? p.inv_norm[t.mat] : 1.f;
      const float alpha = p.phase == PH_GRAM ? inv * inv : inv;
      const uint32_t r = t.m0 + q * 32 + lane;                   // output row of this thread
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
      const uint32_t taddr0 = tmem_base + ((q * 32u) << 16) + acc * kBNMax;
      for (uint32_t c0 = 0; c0 < c.n_valid; c0 += 32) {
        const uint32_t col0 = t.n0 + c0;
        if (col0 >= c.out_cols) break;                           // warp-uniform
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
        if (sym && (col0 >> 7) > (t.m0 >> 7) && row_ok) {
#pragma unroll
          for (int j = 0; j < 32; ++j)
            if (col0 + j < c.out_cols) out[(size_t)(col0 + j) * pitch + r] = __float2bfloat16_rn(f[j]);
        }
      }
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(tempty0 + 8 * acc);
      if (++acc == 2) { acc = 0; acc_phase ^= 1; }
    }
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc<kTmemCols>(tmem_base);
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
// out-of-bounds elements read as zero (ragged edges and partial k blocks rely on it).
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

// Tile rasterisation.  The 148 CTAs walk the tile list round-robin, so at any moment ~148 consecutive list entries
// are in flight and advance along k roughly in lock step; an operand box is fetched from DRAM once and served from
// L2 to every in-flight tile that shares it.  The list is therefore ordered so that 148 consecutive tiles cover a
// compact block of the output: `band` row blocks x the column tiles that go with them.
int tune(const char* name, int dflt) {
  const char* e = getenv(name);
  return e && *e ? atoi(e) : dflt;
}
// rectangular output (APPLY): column panels of `group` tiles stay L2-resident while all row blocks sweep over them.
void tiles_rect(std::vector<TcTile>& v, uint32_t mat, uint32_t out_rows, uint32_t out_cols, uint32_t nkb) {
  const uint32_t tm = (out_rows + kBM - 1) / kBM, tn = (out_cols + kBNMax - 1) / kBNMax;
  const uint32_t group = (uint32_t)std::max(1, tune("MFSDP_TUNE_RECT_GROUP", 8));
  for (uint32_t g0 = 0; g0 < tn; g0 += group)
    for (uint32_t i = 0; i < tm; ++i)
      for (uint32_t j = g0; j < std::min(tn, g0 + group); ++j) v.push_back(TcTile{mat, i * kBM, j * kBNMax, (uint16_t)nkb, (uint16_t)std::min(kBNMax, (out_cols - j * kBNMax + 63u) & ~63u)});
}
// symmetric output (GRAM, POLY): upper 128-row blocks only; bands of `band` row blocks, inside a band column-major
// (all row blocks of the band for one 256-column step, then the next step).
void tiles_sym(std::vector<TcTile>& v, uint32_t mat, uint32_t d, uint32_t nkb) {
  const uint32_t tm = (d + kBM - 1) / kBM;
  const uint32_t band = (uint32_t)std::max(1, tune("MFSDP_TUNE_SYM_BAND", 16));
  for (uint32_t b0 = 0; b0 < tm; b0 += band) {
    const uint32_t b1 = std::min(tm, b0 + band);
    for (uint32_t c0 = b0 * kBM; c0 < d; c0 += kBNMax)          // 256-column steps from the band's first diagonal
      for (uint32_t i = b0; i < b1; ++i) {
        // row block i owns columns >= i * 128; clip the step to that range (N = 128 when only half of it is owned)
        const uint32_t lo = std::max(c0, i * kBM);
        const uint32_t hi = std::min(d, c0 + kBNMax);
        if (lo >= hi) continue;
        v.push_back(TcTile{mat, i * kBM, lo, (uint16_t)nkb, (uint16_t)((hi - lo + 63u) & ~63u)});
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

int build_tc_plan(Plan& pl) {
  NsTcPlan* tc = new NsTcPlan();
  pl.tc = tc;
  const WsLayout& lay = pl.lay;
  uint8_t* ws = static_cast<uint8_t*>(pl.workspace);
  std::vector<CUtensorMap> maps(4 * lay.mats.size());
  std::vector<TcMat> mats(lay.mats.size());
  std::vector<TcTile> tiles[3];
  // big matrices first so that the static round-robin over CTAs ends with the cheap tiles
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
  for (uint32_t i : order) {
    const MatLayout& L = lay.mats[i];
    tiles_sym(tiles[PH_GRAM], i, L.d, (L.n_long + kBK - 1) / kBK);
    tiles_sym(tiles[PH_POLY], i, L.d, (L.d + kBK - 1) / kBK);
    tiles_rect(tiles[PH_APPLY], i, L.rows, L.cols, (L.d + kBK - 1) / kBK);
  }
  int rc;
  if ((rc = dev_upload(&tc->d_tmaps, maps)) || (rc = dev_upload(&tc->d_mats, mats))) return rc;
  for (int ph = 0; ph < 3; ++ph) {
    tc->n_tiles[ph] = (uint32_t)tiles[ph].size();
    if ((rc = dev_upload(&tc->d_tiles[ph], tiles[ph]))) return rc;
  }
  cudaDeviceGetAttribute(&tc->sms, cudaDevAttrMultiProcessorCount, pl.device);
  cudaError_t e = cudaFuncSetAttribute(k_ns_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemBytes);
  if (e != cudaSuccess) return cuda_fail(e);
  return MFSDP_OK;
}

}  // namespace

void destroy_ns_tc(NsTcPlan* p) {
  if (!p) return;
  cudaFree(p->d_tmaps); cudaFree(p->d_mats);
  for (int ph = 0; ph < 3; ++ph) cudaFree(p->d_tiles[ph]);
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
  for (int it = 0; it < hp.ns_steps; ++it) {
    p.src = it & 1;
    p.first = (it == 0);
    for (int ph = 0; ph < 3; ++ph) {
      p.phase = ph;
      p.tiles = tc.d_tiles[ph];
      p.n_tiles = tc.n_tiles[ph];
      const uint32_t grid = std::min<uint32_t>(p.n_tiles, (uint32_t)tc.sms);
      k_ns_tc<<<grid, kThreads, kSmemBytes, st>>>(p);
      count_launch();
      const int rc = check_last_launch();
      if (rc) return rc;
    }
  }
  return MFSDP_OK;
}

}  // namespace mfsdp
