// Owner-local Shampoo on the descriptor table of the Muon step ("swapping owner-Muon for Shampoo (full
// L/R preconditioners with inverse fourth root)"; readings S1-S7 of DESIGN.md section 4).
//
// Per resident matrix G (rows x cols), statistics L (rows x rows), R (cols x cols) in fp32:
//   S1  L <- beta2 L + w G G^T ; R <- beta2 R + w G^T G                       one grouped GEMM launch (k_sgemm3)
//   S2  A = S + rho I, rho = max(eps tr S / d, eps_floor ||S||_F) (S7)         k_sh_reduce, k_sh_power, k_sh_root_init
//   S3  P = A^{-1/4}  by the coupled Newton iteration (reading S6):           3 grouped GEMM launches + k_sh_root_ctl
//         M_0 = z A, X_0 = z^{1/4} I, z = 5 / (2 bound), bound from ||S||_F and   per iteration, for every L and R of the
//         eight power-iteration steps;
//         T = (5 I - M) / 4 ; X <- X T ; M <- T^4 M ; stop at max |M - I| < tol  group at once; the first iterations
//         also scale M by 2.5 and X by 2.5^(1/4) (k_sh_root_init: 6.1 x instead of 2.44 x growth of small eigenvalues)
//   S4  D = P_L G P_R ; W <- W (1 - lr wd) - lr D                             two grouped GEMM launches, update fused
//   S5  roots only at steps with (t - 1) % root_every == 0; P_L, P_R are kept (as three bf16 planes) in the state.
// All matrix products run on the tensor cores with three-term bf16 operands (sgemm3.cuh).  Every problem of a launch is
// independent; a problem that has converged raises its `done` word and its tiles are skipped by later launches, so
// the host enqueues a fixed number of launches and never synchronises.
#include <cuda.h>
#include <cuda_bf16.h>

#include <algorithm>
#include <cmath>
#include <cstring>
#include <memory>
#include <vector>

#include "mfsdp_internal.h"
#include "sgemm3.cuh"

namespace mfsdp {
namespace {

constexpr uint32_t kRedBlocks = 64;      // row groups of the trace / Frobenius reduction (fixed: deterministic sums)
constexpr uint32_t kRootBufs = 7;        // X ping-pong, M ping-pong, T, T^2, T^4
constexpr uint32_t kPartWords = 4;       // per row group: sum of squares, trace, |S x|^2 of the even / odd power iterations
constexpr uint32_t kPowerIters = 8;      // power iterations for the bound on lambda_max (reading S6)

struct ShCtl {                           // per root problem, device (layout documented in mfsdp.h: tests read it)
  double tr, fro2;
  float rho, z, x0, prev_err;
  uint32_t err, iters, done, identity;
  float alpha_m, alpha_x;                // factors on the NEXT iteration's M' and X' (scaled phase: 2.5 and 2.5^(1/4))
  uint32_t n_scaled, pad;                // iterations whose outputs are scaled
};
static_assert(sizeof(ShCtl) == 64, "ShCtl layout is part of the debug ABI");

struct RootInfo {                        // per root problem, device
  const float* S;                        // statistic, d x pitch fp32
  uint32_t d, pitch;
  uint64_t plane;                        // elements per split plane
  __nv_bfloat16* X[2];
  __nv_bfloat16* M0;
  __nv_bfloat16* T;
  __nv_bfloat16* P;                      // state: the root, three planes
  float* vec;                            // two vectors of `pitch` floats for the power iteration (inside the T^2 buffer)
  uint32_t ctl;                          // index into the ShCtl array
  uint32_t pad;
};

struct GprepItem {                       // stage a gradient as bf16 term planes with a TMA-friendly pitch
  const void* src;                       // rows x cols, pitch = cols
  __nv_bfloat16* dst;
  uint32_t rows, cols, pitch, terms, src_bf16, pad;
  uint64_t plane;
};

// ---- elementwise kernels -----------------------------------------------------------------------------------------
__global__ void k_sh_gprep(const GprepItem* items) {
  const GprepItem it = items[blockIdx.y];
  for (uint32_t r = blockIdx.x; r < it.rows; r += gridDim.x)
    for (uint32_t c = threadIdx.x; c < it.pitch; c += blockDim.x) {
      float v = 0.f;
      if (c < it.cols)
        v = it.src_bf16 ? __bfloat162float(reinterpret_cast<const __nv_bfloat16*>(it.src)[(size_t)r * it.cols + c])
                        : reinterpret_cast<const float*>(it.src)[(size_t)r * it.cols + c];
      uint32_t b1, b2, b3;
      sg::split3(v, b1, b2, b3);
      __nv_bfloat16* d = it.dst + (size_t)r * it.pitch + c;
      d[0] = __ushort_as_bfloat16((unsigned short)b1);
      if (it.terms == 3) {
        d[it.plane] = __ushort_as_bfloat16((unsigned short)b2);
        d[2 * it.plane] = __ushort_as_bfloat16((unsigned short)b3);
      }
    }
}

// trace and squared Frobenius norm of every statistic: fp64 partials per row group, fixed-order tree inside the block
__global__ void __launch_bounds__(256) k_sh_reduce(const RootInfo* roots, double* partials) {
  const RootInfo ri = roots[blockIdx.y];
  double s2 = 0.0, tr = 0.0;
  for (uint32_t r = blockIdx.x; r < ri.d; r += gridDim.x) {
    const float* row = ri.S + (size_t)r * ri.pitch;
    for (uint32_t c = threadIdx.x; c < ri.d; c += blockDim.x) {
      const double v = (double)row[c];
      s2 += v * v;
      if (c == r) tr += v;
    }
  }
  __shared__ double sh[2][256];
  sh[0][threadIdx.x] = s2; sh[1][threadIdx.x] = tr;
  __syncthreads();
  for (uint32_t o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) { sh[0][threadIdx.x] += sh[0][threadIdx.x + o]; sh[1][threadIdx.x] += sh[1][threadIdx.x + o]; }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    double* out = partials + ((size_t)ri.ctl * kRedBlocks + blockIdx.x) * kPartWords;
    out[0] = sh[0][0]; out[1] = sh[1][0];
  }
}

// One step of the power iteration y = S x / |x| for every statistic of the group (a lower bound on lambda_max: the
// Frobenius norm alone costs 4-5 extra Newton iterations).  x of step 0 is a fixed pseudo-random vector; the squared
// norm of y is left as per-block partials (fixed order: deterministic) and divides the next step's x on the fly.
__global__ void __launch_bounds__(256) k_sh_power(const RootInfo* roots, double* partials, uint32_t it) {
  const RootInfo ri = roots[blockIdx.y];
  const float* xin = ri.vec + (it & 1u) * ri.pitch;
  float* yout = ri.vec + ((it + 1u) & 1u) * ri.pitch;
  __shared__ float scale_sh;
  if (threadIdx.x == 0) {
    double n2 = 0.0;
    if (it > 0)
      for (uint32_t b = 0; b < kRedBlocks; ++b) n2 += partials[((size_t)ri.ctl * kRedBlocks + b) * kPartWords + 2 + ((it - 1u) & 1u)];
    scale_sh = it > 0 ? (n2 > 0.0 ? (float)(1.0 / sqrt(n2)) : 0.f) : 1.f;
  }
  __syncthreads();
  const float sc = scale_sh;
  // one warp per row (8 rows in flight per block), float4 loads, shuffle reduction; fixed orders throughout
  const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
  double acc2 = 0.0;
  for (uint32_t r = blockIdx.x * 8u + warp; r < ri.d; r += gridDim.x * 8u) {
    const float* row = ri.S + (size_t)r * ri.pitch;
    float sum = 0.f;
    for (uint32_t c = 4u * lane; c < ri.d; c += 128u) {          // pitch is a multiple of 64: a float4 never leaves the row
      const float4 a = *reinterpret_cast<const float4*>(row + c);
      const float av[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
      for (uint32_t k = 0; k < 4; ++k) {
        const uint32_t cc = c + k;
        if (cc < ri.d) {
          const float x = it > 0 ? xin[cc] * sc : (float)((cc * 2654435761u + 0x9e3779b9u) >> 16 & 0xffffu) * (1.f / 32768.f) - 1.f;
          sum = fmaf(av[k], x, sum);
        }
      }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if (lane == 0) { yout[r] = sum; acc2 += (double)sum * (double)sum; }
  }
  __shared__ double red2[8];
  if (lane == 0) red2[warp] = acc2;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red2[w];
    partials[((size_t)ri.ctl * kRedBlocks + blockIdx.x) * kPartWords + 2 + (it & 1u)] = t;
  }
}

__global__ void k_sh_root_init(const RootInfo* roots, uint32_t n, ShCtl* ctl, const double* partials, double eps,
                               double eps_floor) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const RootInfo ri = roots[i];
  double s2 = 0.0, tr = 0.0, lam2 = 0.0;
  for (uint32_t b = 0; b < kRedBlocks; ++b) {
    s2 += partials[((size_t)ri.ctl * kRedBlocks + b) * kPartWords];
    tr += partials[((size_t)ri.ctl * kRedBlocks + b) * kPartWords + 1];
    lam2 += partials[((size_t)ri.ctl * kRedBlocks + b) * kPartWords + 2 + ((kPowerIters - 1u) & 1u)];
  }
  ShCtl c;
  c.tr = tr; c.fro2 = s2;
  c.err = 0u; c.iters = 0u; c.prev_err = 3.0e38f;
  if (!(tr > 0.0)) {                      // reading S2: no gradient seen yet -> the preconditioner is I
    c.identity = 1u; c.done = 1u; c.rho = 0.f; c.z = 1.f; c.x0 = 1.f;
    c.alpha_m = c.alpha_x = 1.f; c.n_scaled = 0u; c.pad = 0u;
  } else {
    const double rho = fmax(eps * tr / (double)ri.d, eps_floor * sqrt(s2));   // readings S2, S7
    // lambda_max(S) <= ||S||_F always; the power iteration gives |S x| <= lambda_max from below, within a factor of
    // d^(1 / 2k) = 1.8 of it at worst after k = 8 steps from a start vector with a 1 / sqrt(d) component along the top
    // eigenvector (d = 14336) and within a few percent on spectra with a cluster at the top; M_0's eigenvalues have to
    // stay below 5 for the iteration to converge: bound / lambda_max >= 1.6 / 1.8 * ... is ample (2.5 lambda_max /
    // bound < 5 needs bound > lambda_max / 2).  A tighter bound saves iterations: ||S||_F overestimates a flat
    // rank-r spectrum by sqrt(r), i.e. log(sqrt(r)) / log(2.44) = 4-5 of ~18 iterations.
    const double lam = sqrt(lam2);
    const double top = lam > 0.0 && lam == lam ? fmin(sqrt(s2), 1.6 * lam) : sqrt(s2);
    const double bound = top + rho;       // taken as lambda_max(S + rho I)
    const double z = 2.5 / bound;         // (1 + p) / (2 ||A||), p = 4
    c.identity = 0u; c.done = 0u;
    c.rho = (float)rho; c.z = (float)z; c.x0 = (float)sqrt(sqrt(z));
    // Scaled phase.  After any iteration every eigenvalue of M is <= 1 (mu ((5 - mu) / 4)^4 <= 1 on (0, 5)), so M may
    // be multiplied by 2.5 (and X by 2.5^(1/4): X^4 S~ z = M is kept) without leaving the convergence region: small
    // eigenvalues then grow by 2.5 x 2.44 = 6.1 per iteration instead of 2.44.  The smallest eigenvalue of M_0 is at
    // least mu0 = 2.5 rho / bound; scaling stops when that lower bound has reached 0.2, the plain iteration finishes.
    const double mu0 = 2.5 * rho / bound;
    c.n_scaled = mu0 > 0.0 && mu0 < 0.2 ? (uint32_t)floor(log(0.2 / mu0) / log(6.103515625)) : 0u;
    c.alpha_m = c.n_scaled >= 1u ? 2.5f : 1.f;
    c.alpha_x = c.n_scaled >= 1u ? 1.2574334f : 1.f;        // 2.5^(1/4)
    c.pad = 0u;
  }
  ctl[ri.ctl] = c;
}

// M_0 = z (S + rho I), T_0 = (5 I - M_0) / 4, X_0 = x0 I as three-term planes
__global__ void __launch_bounds__(256) k_sh_root_prep(const RootInfo* roots, const ShCtl* ctl) {
  const RootInfo ri = roots[blockIdx.y];
  const ShCtl c = ctl[ri.ctl];
  for (uint32_t r = blockIdx.x; r < ri.d; r += gridDim.x) {
    const float* row = ri.S + (size_t)r * ri.pitch;
    for (uint32_t col = 8u * threadIdx.x; col < ri.pitch; col += 8u * blockDim.x) {   // 8 columns per thread; the pitch
      float m[8], t[8], x[8];                                                          // padding is written too (zeros)
      const float4 a = *reinterpret_cast<const float4*>(row + col), b = *reinterpret_cast<const float4*>(row + col + 4);
      const float sv[8] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w};
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const float diag = col + k == r ? 1.f : 0.f;
        m[k] = col + k >= ri.d ? 0.f : c.identity ? diag : c.z * (sv[k] + c.rho * diag);
        t[k] = 0.25f * (5.f * diag - m[k]);
        x[k] = c.x0 * diag;
      }
      const size_t o = (size_t)r * ri.pitch + col;
      sg::store_split8(ri.M0 + o, ri.plane, m);
      sg::store_split8(ri.T + o, ri.plane, t);
      sg::store_split8(ri.X[0] + o, ri.plane, x);
    }
  }
}

// after the M launch of an iteration: count it, decide, clear the error word
__global__ void k_sh_root_ctl(const RootInfo* roots, uint32_t n, ShCtl* ctl, float tol, uint32_t max_iters) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  ShCtl* c = ctl + roots[i].ctl;
  if (c->done) return;
  const float e = __uint_as_float(c->err);
  c->iters += 1u;
  // converged; or at the fp32-class noise floor (the error no longer falls); or not a number; or out of budget
  // (the stagnation rule only inside the quadratic regime: far from convergence the error sits just below 1 and
  // consecutive values may round to the same float)
  if (!(e >= tol) || (e < 1e-2f && !(e < c->prev_err))) c->done = 1u;
  else if (c->iters >= max_iters) c->done = 3u;     // out of budget: X is the best iterate so far, NOT a converged root
  if (!(e == e)) c->done = 2u;
  c->prev_err = e;
  c->err = 0u;
  const bool scale_next = c->iters + 1u <= c->n_scaled;      // the outputs of iteration iters + 1
  c->alpha_m = scale_next ? 2.5f : 1.f;
  c->alpha_x = scale_next ? 1.2574334f : 1.f;
}

// Status record of the last root refresh, behind the control block (mfsdp_shampoo_view out[11]): how many of the n
// root problems ended converged (done == 1, identity problems included), not positive definite (2), out of budget (3).
__global__ void __launch_bounds__(256) k_sh_status(const ShCtl* ctl, uint32_t n, uint32_t* status) {
  __shared__ uint32_t cnt[4];
  if (threadIdx.x < 4) cnt[threadIdx.x] = 0u;
  __syncthreads();
  for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
    const uint32_t d = ctl[i].done;
    atomicAdd(&cnt[d == 1u ? 0 : d == 2u ? 1 : d == 3u ? 2 : 3], 1u);      // [3]: still running (never after a refresh)
  }
  __syncthreads();
  if (threadIdx.x < 3) status[threadIdx.x] = cnt[threadIdx.x];
  if (threadIdx.x == 3) status[3] = n;
}

// P <- X[iters & 1].  A root whose iteration produced a NaN (done == 2: S + rho I was not positive definite in this
// arithmetic, i.e. the ridge sits below the rounding noise of the statistic) falls back to the scalar preconditioner
// (tr S / d + rho)^{-1/4} I and stays flagged in its control record.
__global__ void __launch_bounds__(256) k_sh_root_finish(const RootInfo* roots, const ShCtl* ctl) {
  const RootInfo ri = roots[blockIdx.y];
  const ShCtl c = ctl[ri.ctl];
  if (c.done == 2u) {
    const float s = (float)(1.0 / sqrt(sqrt(c.tr / (double)ri.d + (double)c.rho)));
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < ri.plane; i += (size_t)gridDim.x * blockDim.x) {
      const uint32_t r = (uint32_t)(i / ri.pitch), col = (uint32_t)(i % ri.pitch);
      sg::store_split1(ri.P + i, ri.plane, r == col ? s : 0.f);
    }
    return;
  }
  const uint4* src = reinterpret_cast<const uint4*>(ri.X[c.iters & 1u]);
  uint4* dst = reinterpret_cast<uint4*>(ri.P);
  const size_t n8 = 3 * ri.plane / 8;                             // planes are rows x pitch, pitch a multiple of 64
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n8; i += (size_t)gridDim.x * blockDim.x) {
    const uint32_t col = (uint32_t)((i * 8) % ri.pitch);
    uint4 v = src[i];
    if (col + 8u > ri.d) {                                        // the pitch padding of the state is zero
      uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (uint32_t k = 0; k < 4; ++k) {
        if (col + 2 * k >= ri.d) w[k] = 0u;
        else if (col + 2 * k + 1 >= ri.d) w[k] &= 0xffffu;
      }
      v = make_uint4(w[0], w[1], w[2], w[3]);
    }
    dst[i] = v;
  }
}

// ---- host: tensor maps ------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn sh_encode() {
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
// bf16 planes [planes][rows][pitch], logical width cols; mn = operand read MN-major (box 64 x 64) else K-major (64 x 128)
int make_tmap3(CUtensorMap* out, const void* base, uint32_t rows, uint32_t cols, uint32_t pitch, uint64_t plane_elems,
               uint32_t planes, bool mn) {
  EncodeTiledFn enc = sh_encode();
  if (!enc) return cuda_fail(cudaErrorSymbolNotFound);
  const cuuint64_t dims[3] = {cols, rows, planes};
  const cuuint64_t strides[2] = {(cuuint64_t)pitch * 2, (cuuint64_t)plane_elems * 2};
  const cuuint32_t box[3] = {64, mn ? 64u : 128u, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? MFSDP_OK : cuda_fail(cudaErrorInvalidValue);
}

// store map of a three-plane output: box 32 cols x 32 rows x 1 plane, dense (no swizzle); stores are clipped at the edges
int make_store_tmap3(CUtensorMap* out, const void* base, uint32_t rows, uint32_t cols, uint32_t pitch, uint64_t plane_elems) {
  EncodeTiledFn enc = sh_encode();
  if (!enc) return cuda_fail(cudaErrorSymbolNotFound);
  const cuuint64_t dims[3] = {cols, rows, 3};
  const cuuint64_t strides[2] = {(cuuint64_t)pitch * 2, (cuuint64_t)plane_elems * 2};
  const cuuint32_t box[3] = {32, 32, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                         CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? MFSDP_OK : cuda_fail(cudaErrorInvalidValue);
}

// ---- host: layout ---------------------------------------------------------------------------------------------------
inline uint32_t pitch64(uint32_t n) { return (n + 63u) / 64u * 64u; }

struct ShMat {
  uint64_t elem_off;
  uint32_t rows, cols, pr, pc, dtype;
  bool g_direct;                           // bf16 gradient with cols % 8 == 0: TMA reads it in place
  uint32_t g_terms;
  uint64_t L_off, R_off, PL_off, PR_off;   // state, bytes
  uint64_t Gs_off, Tm_off, D_off;          // workspace, bytes
};
struct ShLayout {
  std::vector<ShMat> mats;
  uint64_t state_bytes = 0;
  uint64_t ctl_off = 0, partial_off = 0, base_bytes = 0;   // workspace: control block, reduction partials, end of the fixed part
  uint64_t max_root_bytes = 0, all_root_bytes = 0;
  int dtype = -1;
};
inline uint64_t root_bytes(uint32_t d) { return align_up_u64((uint64_t)kRootBufs * 3 * d * pitch64(d) * 2, kBufAlign); }

int build_sh_layout(const mfsdp_desc_t* desc, size_t n_desc, bool keep_d, ShLayout& out) {
  if (n_desc && !desc) return MFSDP_EINVAL;
  int rc = mfsdp_validate_desc(desc, n_desc);
  if (rc) return rc;
  uint64_t st = 0;
  for (size_t i = 0; i < n_desc; ++i) {
    if (desc[i].role != MFSDP_ROLE_MATRIX) continue;
    if (out.dtype < 0) out.dtype = (int)desc[i].dtype;
    else if (out.dtype != (int)desc[i].dtype) return MFSDP_EINVAL;
    ShMat m;
    m.elem_off = desc[i].elem_off; m.rows = desc[i].rows; m.cols = desc[i].cols; m.dtype = desc[i].dtype;
    m.pr = pitch64(m.rows); m.pc = pitch64(m.cols);
    m.g_direct = m.dtype == MFSDP_BF16 && (m.cols % 8u) == 0u;
    m.g_terms = m.dtype == MFSDP_BF16 ? 1u : 3u;
    m.L_off = st; st = align_up_u64(st + (uint64_t)m.rows * m.pr * 4, kBufAlign);
    m.R_off = st; st = align_up_u64(st + (uint64_t)m.cols * m.pc * 4, kBufAlign);
    m.PL_off = st; st = align_up_u64(st + (uint64_t)3 * m.rows * m.pr * 2, kBufAlign);
    m.PR_off = st; st = align_up_u64(st + (uint64_t)3 * m.cols * m.pc * 2, kBufAlign);
    m.Gs_off = m.Tm_off = m.D_off = 0;
    out.mats.push_back(m);
  }
  out.state_bytes = st;
  const uint64_t n_prob = 2 * out.mats.size();
  uint64_t ws = 0;
  out.ctl_off = ws; ws = align_up_u64(ws + n_prob * sizeof(ShCtl) + 4 * sizeof(uint32_t), kBufAlign);   // + status record
  out.partial_off = ws; ws = align_up_u64(ws + n_prob * kRedBlocks * kPartWords * sizeof(double), kBufAlign);
  for (ShMat& m : out.mats) {
    if (!m.g_direct) { m.Gs_off = ws; ws = align_up_u64(ws + (uint64_t)m.g_terms * m.rows * m.pc * 2, kBufAlign); }
    m.Tm_off = ws; ws = align_up_u64(ws + (uint64_t)3 * m.rows * m.pc * 2, kBufAlign);
    if (keep_d) { m.D_off = ws; ws = align_up_u64(ws + (uint64_t)m.rows * m.pc * 4, kBufAlign); }
    out.max_root_bytes = std::max({out.max_root_bytes, root_bytes(m.rows), root_bytes(m.cols)});
    out.all_root_bytes += root_bytes(m.rows) + root_bytes(m.cols);
  }
  out.base_bytes = ws;
  return MFSDP_OK;
}

// ---- host: launch tables ----------------------------------------------------------------------------------------------
struct SgLaunch { uint32_t prob_off = 0, tile_off = 0, n_tiles = 0; int at = 3, bt = 3; bool pair = false; };   // offsets into the plan's arrays
struct RootGroup {
  uint32_t root_off = 0, n_roots = 0;      // into the RootInfo array
  SgLaunch a[2], b, c[2];                  // X T and T T (by iteration parity); T^2 T^2; T^4 M (by parity)
  uint32_t max_d = 0;
};
struct ShPlan {
  std::vector<uint8_t> key;
  int device = -1, sms = 148;
  ShLayout lay;
  std::vector<RootGroup> groups;
  SgLaunch stat, pre1, pre2;
  uint32_t n_gprep = 0, max_rows = 0;
  // device blob
  void* blob = nullptr;
  SgProb* d_probs = nullptr;
  SgTile* d_tiles = nullptr;
  RootInfo* d_roots = nullptr;
  GprepItem* d_gprep = nullptr;
  // W and G are not part of the cache key (training code often hands over a fresh gradient tensor every step): the
  // records that hold their addresses are kept on the host as well and re-pointed + re-uploaded when they change
  uint8_t* W = nullptr;
  const uint8_t* G = nullptr;
  std::vector<SgProb> h_probs;
  std::vector<GprepItem> h_gprep;
  struct GwRef { uint32_t prob, mat, kind; };   // kind 0: statistics (both maps, side in bit 8), 1: P_L G (map b), 2: W
  std::vector<GwRef> gw;
};
std::vector<std::unique_ptr<ShPlan>> g_sh_plans;
constexpr size_t kMaxShPlans = 64;

// Tiles of one problem, edge `ts` (128: single CTA, 256: CTA pair).  Bands of row blocks, column-major inside a band:
// the tiles in flight form a compact block of the output and share operand panels through L2.
void sh_tiles(std::vector<SgTile>& v, uint32_t prob, uint32_t M, uint32_t N, bool sym, uint32_t ts) {
  const uint32_t tm = (M + ts - 1) / ts, tn = (N + ts - 1) / ts, band = ts == 128u ? 12u : 8u;
  for (uint32_t i0 = 0; i0 < tm; i0 += band)
    for (uint32_t j = sym ? i0 : 0u; j < tn; ++j)
      for (uint32_t i = i0; i < std::min(tm, i0 + band); ++i)
        if (!sym || j >= i) v.push_back(SgTile{prob, i * ts, j * ts});
}
uint32_t sh_tile_count(uint32_t M, uint32_t N, bool sym, uint32_t ts) {
  const uint32_t tm = (M + ts - 1) / ts, tn = (N + ts - 1) / ts;
  return sym ? tm * (tm + 1) / 2 : tm * tn;
}
constexpr uint32_t kPairMinTiles = 64;   // a launch runs on CTA pairs when it has about a wave of 256-tiles (74 pairs)

template <int AT, int BT>
int sg_setup() {
  cudaError_t e = cudaFuncSetAttribute(k_sgemm3<AT, BT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (int)SgCfg<AT, BT>::kSmem);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(k_sgemm3p<AT, BT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SgCfg<AT, BT>::kSmem);
  return e == cudaSuccess ? MFSDP_OK : cuda_fail(e);
}

template <int AT, int BT>
cudaError_t sg_launch_pair(const SgParams& p, uint32_t pairs, cudaStream_t st) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(2 * pairs); cfg.blockDim = dim3(kSgPairThreads);
  cfg.dynamicSmemBytes = SgCfg<AT, BT>::kSmem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_sgemm3p<AT, BT>, p);
}

int sg_launch(const ShPlan& pl, const SgLaunch& L, float alpha, float beta, float decay, float lr, cudaStream_t st) {
  if (L.n_tiles == 0) return MFSDP_OK;
  SgParams p;
  p.probs = pl.d_probs + L.prob_off; p.tiles = pl.d_tiles + L.tile_off; p.n_tiles = L.n_tiles;
  p.alpha = alpha; p.beta = beta; p.decay = decay; p.lr = lr;
  get_trace(&p.trace, &p.trace_cap);
  if (L.pair) {
    const uint32_t pairs = std::min<uint32_t>(L.n_tiles, (uint32_t)pl.sms / 2);
    const cudaError_t e = L.at == 1 && L.bt == 1 ? sg_launch_pair<1, 1>(p, pairs, st)
                          : L.at == 2 && L.bt == 1 ? sg_launch_pair<2, 1>(p, pairs, st)
                          : L.at == 2 && L.bt == 2 ? sg_launch_pair<2, 2>(p, pairs, st) : sg_launch_pair<3, 3>(p, pairs, st);
    count_launch();
    return e == cudaSuccess ? check_last_launch() : cuda_fail(e);
  }
  const uint32_t grid = std::min<uint32_t>(L.n_tiles, (uint32_t)pl.sms);
  if (L.at == 1 && L.bt == 1) k_sgemm3<1, 1><<<grid, kSgThreads, SgCfg<1, 1>::kSmem, st>>>(p);
  else if (L.at == 2 && L.bt == 1) k_sgemm3<2, 1><<<grid, kSgThreads, SgCfg<2, 1>::kSmem, st>>>(p);
  else if (L.at == 2 && L.bt == 2) k_sgemm3<2, 2><<<grid, kSgThreads, SgCfg<2, 2>::kSmem, st>>>(p);
  else k_sgemm3<3, 3><<<grid, kSgThreads, SgCfg<3, 3>::kSmem, st>>>(p);
  count_launch();
  return check_last_launch();
}

int build_sh_plan(ShPlan& pl, uint8_t* W, const uint8_t* G, uint8_t* state, uint8_t* ws, size_t ws_bytes, bool keep_d) {
  const ShLayout& lay = pl.lay;
  const size_t n_mat = lay.mats.size();
  const size_t esz = lay.dtype == MFSDP_BF16 ? 2 : 4;
  std::vector<SgProb> probs;
  std::vector<SgTile> tiles;
  std::vector<RootInfo> roots;
  std::vector<GprepItem> gprep;
  int rc;
  ShCtl* d_ctl = reinterpret_cast<ShCtl*>(ws + lay.ctl_off);

  auto zero_prob = [] {
    SgProb q;
    std::memset(&q, 0, sizeof(q));
    return q;
  };
  struct Pending { uint32_t prob, M, N; bool sym; };
  std::vector<Pending> pending;
  auto begin = [&](SgLaunch& L, int at, int bt) {
    L.prob_off = (uint32_t)probs.size(); L.tile_off = (uint32_t)tiles.size(); L.at = at; L.bt = bt;
    pending.clear();
  };
  auto add_tiles = [&](uint32_t prob, uint32_t M, uint32_t N, bool sym) { pending.push_back(Pending{prob, M, N, sym}); };
  auto end = [&](SgLaunch& L) {     // the tile edge is chosen per launch, once its problems are known
    uint32_t t256 = 0;
    for (const Pending& q : pending) t256 += sh_tile_count(q.M, q.N, q.sym, 256);
    L.pair = t256 >= kPairMinTiles;
    for (const Pending& q : pending) sh_tiles(tiles, q.prob, q.M, q.N, q.sym, L.pair ? 256u : 128u);
    L.n_tiles = (uint32_t)tiles.size() - L.tile_off;
  };
  // matrices by size, largest first (static round-robin: the long tiles lead, the short ones fill the tail)
  std::vector<size_t> order(n_mat);
  for (size_t i = 0; i < n_mat; ++i) order[i] = i;
  std::stable_sort(order.begin(), order.end(), [&](size_t a, size_t b) {
    return (uint64_t)lay.mats[a].rows * lay.mats[a].cols > (uint64_t)lay.mats[b].rows * lay.mats[b].cols;
  });

  // gradient operands
  struct GOp { const void* base; uint32_t pitch; uint64_t plane; uint32_t terms; };
  std::vector<GOp> gop(n_mat);
  for (size_t i = 0; i < n_mat; ++i) {
    const ShMat& m = lay.mats[i];
    pl.max_rows = std::max(pl.max_rows, std::max(m.rows, m.cols));
    if (m.g_direct) gop[i] = GOp{G + m.elem_off * esz, m.cols, (uint64_t)m.rows * m.cols, 1u};
    else {
      gop[i] = GOp{ws + m.Gs_off, m.pc, (uint64_t)m.rows * m.pc, m.g_terms};
      GprepItem it;
      it.src = G + m.elem_off * esz; it.dst = reinterpret_cast<__nv_bfloat16*>(ws + m.Gs_off);
      it.rows = m.rows; it.cols = m.cols; it.pitch = m.pc; it.terms = m.g_terms; it.src_bf16 = m.dtype == MFSDP_BF16;
      it.pad = 0; it.plane = (uint64_t)m.rows * m.pc;
      gprep.push_back(it);
    }
  }
  pl.n_gprep = (uint32_t)gprep.size();
  const int gt = lay.dtype == MFSDP_BF16 ? 1 : 3;

  // S1: statistics, every L and R in one launch
  begin(pl.stat, gt, gt);
  for (size_t oi = 0; oi < n_mat; ++oi) {
    const size_t i = order[oi];
    const ShMat& m = lay.mats[i];
    for (int side = 0; side < 2; ++side) {
      SgProb q = zero_prob();
      const bool mn = side == 1;             // R = G^T G reads G with the output index contiguous
      if ((rc = make_tmap3(&q.ta, gop[i].base, m.rows, m.cols, gop[i].pitch, gop[i].plane, gop[i].terms, mn))) return rc;
      q.tb = q.ta;
      q.M = q.N = side ? m.cols : m.rows; q.K = side ? m.rows : m.cols;
      q.a_mn = q.b_mn = mn; q.sym = 1;
      q.f32_pitch = side ? m.pc : m.pr;
      q.cin = q.out_f32 = reinterpret_cast<float*>(state + (side ? m.R_off : m.L_off));
      pl.gw.push_back(ShPlan::GwRef{(uint32_t)probs.size(), (uint32_t)i, (uint32_t)(side << 8)});
      add_tiles((uint32_t)probs.size() - pl.stat.prob_off, q.M, q.N, true);
      probs.push_back(q);
    }
  }
  end(pl.stat);

  // S3: root problems in groups that fit the workspace behind the fixed part
  const uint64_t root_cap = ws_bytes > lay.base_bytes ? ws_bytes - lay.base_bytes : 0;
  struct RootRef { size_t mat; int side; uint32_t d, pitch; };
  std::vector<RootRef> refs;
  for (size_t oi = 0; oi < n_mat; ++oi)
    for (int side = 0; side < 2; ++side) {
      const ShMat& m = lay.mats[order[oi]];
      refs.push_back(RootRef{order[oi], side, side ? m.cols : m.rows, side ? m.pc : m.pr});
    }
  std::stable_sort(refs.begin(), refs.end(), [](const RootRef& a, const RootRef& b) { return a.d > b.d; });
  size_t at = 0;
  while (at < refs.size()) {
    RootGroup g;
    g.root_off = (uint32_t)roots.size();
    uint64_t used = 0;
    size_t first = at;
    while (at < refs.size() && used + root_bytes(refs[at].d) <= root_cap) { used += root_bytes(refs[at].d); ++at; }
    if (at == first) return MFSDP_ECAP;
    // buffers
    uint64_t off = lay.base_bytes;
    struct Bufs { __nv_bfloat16* b[kRootBufs]; };
    std::vector<Bufs> bufs;
    for (size_t k = first; k < at; ++k) {
      const RootRef& r = refs[k];
      const ShMat& m = lay.mats[r.mat];
      const uint64_t one = (uint64_t)3 * r.d * r.pitch * 2;
      Bufs b;
      for (uint32_t j = 0; j < kRootBufs; ++j) b.b[j] = reinterpret_cast<__nv_bfloat16*>(ws + off + j * one);
      off += root_bytes(r.d);
      bufs.push_back(b);
      RootInfo ri;
      ri.S = reinterpret_cast<const float*>(state + (r.side ? m.R_off : m.L_off));
      ri.d = r.d; ri.pitch = r.pitch; ri.plane = (uint64_t)r.d * r.pitch;
      ri.X[0] = b.b[0]; ri.X[1] = b.b[1]; ri.M0 = b.b[2]; ri.T = b.b[4];
      ri.P = reinterpret_cast<__nv_bfloat16*>(state + (r.side ? m.PR_off : m.PL_off));
      ri.vec = reinterpret_cast<float*>(b.b[5]);
      ri.ctl = (uint32_t)(2 * r.mat + r.side); ri.pad = 0;
      roots.push_back(ri);
      g.max_d = std::max(g.max_d, r.d);
    }
    g.n_roots = (uint32_t)(at - first);
    // buffer roles: 0, 1 = X ping-pong; 2, 3 = M ping-pong; 4 = T; 5 = T^2; 6 = T^4
    auto sym_prob = [&](const RootRef& r, const __nv_bfloat16* a, const __nv_bfloat16* b, __nv_bfloat16* out,
                        __nv_bfloat16* tsplit, bool err, SgProb& q, int scaled = 0) -> int {
      q = zero_prob();
      const uint64_t plane = (uint64_t)r.d * r.pitch;
      int e;
      if ((e = make_tmap3(&q.ta, a, r.d, r.d, r.pitch, plane, 3, false))) return e;
      if ((e = make_tmap3(&q.tb, b, r.d, r.d, r.pitch, plane, 3, false))) return e;
      q.M = q.N = q.K = r.d; q.sym = 1;
      q.sp_pitch = r.pitch; q.sp_plane = plane;
      q.out_split = out; q.t_split = tsplit;
      if ((e = make_store_tmap3(&q.to, out, r.d, r.d, r.pitch, plane))) return e;
      if (tsplit && (e = make_store_tmap3(&q.tt, tsplit, r.d, r.d, r.pitch, plane))) return e;
      ShCtl* c = d_ctl + (2 * r.mat + r.side);
      q.done = &c->done;
      q.err = err ? &c->err : nullptr;
      q.alpha_dev = scaled == 1 ? &c->alpha_x : scaled == 2 ? &c->alpha_m : nullptr;
      return MFSDP_OK;
    };
    for (int par = 0; par < 2; ++par) {
      begin(g.a[par], 3, 3);
      for (size_t k = first; k < at; ++k) {
        const Bufs& b = bufs[k - first];
        SgProb q;
        if ((rc = sym_prob(refs[k], b.b[par], b.b[4], b.b[par ^ 1], nullptr, false, q, 1))) return rc;   // X' = X T
        add_tiles((uint32_t)probs.size() - g.a[par].prob_off, q.M, q.N, true);
        probs.push_back(q);
        if ((rc = sym_prob(refs[k], b.b[4], b.b[4], b.b[5], nullptr, false, q))) return rc;           // T^2 = T T
        add_tiles((uint32_t)probs.size() - g.a[par].prob_off, q.M, q.N, true);
        probs.push_back(q);
      }
      end(g.a[par]);
    }
    begin(g.b, 3, 3);
    for (size_t k = first; k < at; ++k) {
      const Bufs& b = bufs[k - first];
      SgProb q;
      if ((rc = sym_prob(refs[k], b.b[5], b.b[5], b.b[6], nullptr, false, q))) return rc;             // T^4 = T^2 T^2
      add_tiles((uint32_t)probs.size() - g.b.prob_off, q.M, q.N, true);
      probs.push_back(q);
    }
    end(g.b);
    for (int par = 0; par < 2; ++par) {
      begin(g.c[par], 3, 3);
      for (size_t k = first; k < at; ++k) {
        const Bufs& b = bufs[k - first];
        SgProb q;
        if ((rc = sym_prob(refs[k], b.b[6], b.b[2 + par], b.b[2 + (par ^ 1)], b.b[4], true, q, 2))) return rc;   // M' = T^4 M
        add_tiles((uint32_t)probs.size() - g.c[par].prob_off, q.M, q.N, true);
        probs.push_back(q);
      }
      end(g.c[par]);
    }
    pl.groups.push_back(g);
  }

  // S4: Tm = P_L G, then D = Tm P_R with the weight update in the epilogue
  // S4 runs with TWO terms per operand (products with i + j <= 1: 2^-16-class).  The roots themselves carry a relative
  // error of 1e-3 .. 1e-2 in their ridge directions (Shampoo tolerances); a third term in the products
  // around them buys nothing and costs twice the UMMAs.
  begin(pl.pre1, 2, gt == 1 ? 1 : 2);
  for (size_t oi = 0; oi < n_mat; ++oi) {
    const size_t i = order[oi];
    const ShMat& m = lay.mats[i];
    SgProb q = zero_prob();
    if ((rc = make_tmap3(&q.ta, state + m.PL_off, m.rows, m.rows, m.pr, (uint64_t)m.rows * m.pr, 3, false))) return rc;
    if ((rc = make_tmap3(&q.tb, gop[i].base, m.rows, m.cols, gop[i].pitch, gop[i].plane, gop[i].terms, true))) return rc;
    q.M = m.rows; q.N = m.cols; q.K = m.rows; q.b_mn = 1;
    q.sp_pitch = m.pc; q.sp_plane = (uint64_t)m.rows * m.pc;
    q.out_split = reinterpret_cast<__nv_bfloat16*>(ws + m.Tm_off);
    if ((rc = make_store_tmap3(&q.to, q.out_split, m.rows, m.cols, m.pc, (uint64_t)m.rows * m.pc))) return rc;
    pl.gw.push_back(ShPlan::GwRef{(uint32_t)probs.size(), (uint32_t)i, 1u});
    add_tiles((uint32_t)probs.size() - pl.pre1.prob_off, q.M, q.N, false);
    probs.push_back(q);
  }
  end(pl.pre1);
  begin(pl.pre2, 2, 2);
  for (size_t oi = 0; oi < n_mat; ++oi) {
    const size_t i = order[oi];
    const ShMat& m = lay.mats[i];
    SgProb q = zero_prob();
    if ((rc = make_tmap3(&q.ta, ws + m.Tm_off, m.rows, m.cols, m.pc, (uint64_t)m.rows * m.pc, 3, false))) return rc;
    if ((rc = make_tmap3(&q.tb, state + m.PR_off, m.cols, m.cols, m.pc, (uint64_t)m.cols * m.pc, 3, false))) return rc;
    q.M = m.rows; q.N = m.cols; q.K = m.cols;
    q.f32_pitch = m.pc;
    q.out_f32 = keep_d ? reinterpret_cast<float*>(ws + m.D_off) : nullptr;
    q.W = W + m.elem_off * esz; q.w_bf16 = m.dtype == MFSDP_BF16;
    pl.gw.push_back(ShPlan::GwRef{(uint32_t)probs.size(), (uint32_t)i, 2u});
    add_tiles((uint32_t)probs.size() - pl.pre2.prob_off, q.M, q.N, false);
    probs.push_back(q);
  }
  end(pl.pre2);

  // upload
  const size_t b_probs = align_up_u64(probs.size() * sizeof(SgProb), 256), b_tiles = align_up_u64(tiles.size() * sizeof(SgTile), 256);
  const size_t b_roots = align_up_u64(roots.size() * sizeof(RootInfo), 256), b_gprep = align_up_u64(gprep.size() * sizeof(GprepItem), 256);
  cudaError_t e = cudaMalloc(&pl.blob, b_probs + b_tiles + b_roots + b_gprep + 256);
  if (e != cudaSuccess) return cuda_fail(e);
  uint8_t* base = reinterpret_cast<uint8_t*>(pl.blob);
  pl.d_probs = reinterpret_cast<SgProb*>(base);
  pl.d_tiles = reinterpret_cast<SgTile*>(base + b_probs);
  pl.d_roots = reinterpret_cast<RootInfo*>(base + b_probs + b_tiles);
  pl.d_gprep = reinterpret_cast<GprepItem*>(base + b_probs + b_tiles + b_roots);
  if (!probs.empty() && (e = cudaMemcpy(pl.d_probs, probs.data(), probs.size() * sizeof(SgProb), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e);
  if (!tiles.empty() && (e = cudaMemcpy(pl.d_tiles, tiles.data(), tiles.size() * sizeof(SgTile), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e);
  if (!roots.empty() && (e = cudaMemcpy(pl.d_roots, roots.data(), roots.size() * sizeof(RootInfo), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e);
  if (!gprep.empty() && (e = cudaMemcpy(pl.d_gprep, gprep.data(), gprep.size() * sizeof(GprepItem), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e);
  if ((rc = sg_setup<1, 1>()) || (rc = sg_setup<2, 1>()) || (rc = sg_setup<2, 2>()) || (rc = sg_setup<3, 3>())) return rc;
  pl.W = W; pl.G = G;
  pl.h_probs = std::move(probs);
  pl.h_gprep = std::move(gprep);
  return MFSDP_OK;
}

// The caller came with other W / G buffers than the tables were built for: re-point the records that hold their
// addresses (tensor maps of an in-place bf16 gradient, staging sources, weight pointers) and upload them in stream order.
int repoint_sh_plan(ShPlan& pl, uint8_t* W, const uint8_t* G, cudaStream_t st) {
  const size_t esz = pl.lay.dtype == MFSDP_BF16 ? 2 : 4;
  int rc;
  for (const ShPlan::GwRef& ref : pl.gw) {
    const ShMat& m = pl.lay.mats[ref.mat];
    SgProb& q = pl.h_probs[ref.prob];
    const uint8_t* g = G + m.elem_off * esz;
    if ((ref.kind & 0xffu) == 0u) {
      if (!m.g_direct) continue;
      if ((rc = make_tmap3(&q.ta, g, m.rows, m.cols, m.cols, (uint64_t)m.rows * m.cols, 1, (ref.kind >> 8) != 0u))) return rc;
      q.tb = q.ta;
    } else if (ref.kind == 1u) {
      if (!m.g_direct) continue;
      if ((rc = make_tmap3(&q.tb, g, m.rows, m.cols, m.cols, (uint64_t)m.rows * m.cols, 1, true))) return rc;
    } else {
      q.W = W + m.elem_off * esz;
    }
  }
  size_t k = 0;
  for (const ShMat& m : pl.lay.mats)
    if (!m.g_direct) pl.h_gprep[k++].src = G + m.elem_off * esz;
  cudaError_t e = cudaMemcpyAsync(pl.d_probs, pl.h_probs.data(), pl.h_probs.size() * sizeof(SgProb), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess && !pl.h_gprep.empty())
    e = cudaMemcpyAsync(pl.d_gprep, pl.h_gprep.data(), pl.h_gprep.size() * sizeof(GprepItem), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return cuda_fail(e);
  pl.W = W; pl.G = G;
  return MFSDP_OK;
}

int get_sh_plan(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* state, void* ws, size_t ws_bytes,
                bool keep_d, ShPlan** out) {
  int dev = 0, major = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? MFSDP_EARCH : cuda_fail(e);
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? MFSDP_EARCH : cuda_fail(e);
  if (major != 10) return MFSDP_EARCH;
  std::vector<uint8_t> key(n_desc * sizeof(mfsdp_desc_t) + 64);
  if (n_desc) std::memcpy(key.data(), desc, n_desc * sizeof(mfsdp_desc_t));
  const uint64_t tail[8] = {(uint64_t)dev, 0u, 0u, (uint64_t)(uintptr_t)state,
                            (uint64_t)(uintptr_t)ws, (uint64_t)ws_bytes, keep_d ? 1u : 0u, 0u};
  std::memcpy(key.data() + n_desc * sizeof(mfsdp_desc_t), tail, 64);
  std::lock_guard<std::mutex> lock(plan_mutex());
  for (auto& p : g_sh_plans)
    if (p->key == key) { *out = p.get(); return MFSDP_OK; }
  if (g_sh_plans.size() >= kMaxShPlans) return MFSDP_ECACHE;
  std::unique_ptr<ShPlan> pl(new ShPlan);
  pl->key = key; pl->device = dev;
  int rc = build_sh_layout(desc, n_desc, keep_d, pl->lay);
  if (rc) return rc;
  cudaDeviceGetAttribute(&pl->sms, cudaDevAttrMultiProcessorCount, dev);
  if (ws_bytes < pl->lay.base_bytes + pl->lay.max_root_bytes) return MFSDP_ECAP;
  rc = build_sh_plan(*pl, reinterpret_cast<uint8_t*>(W), reinterpret_cast<const uint8_t*>(G),
                     reinterpret_cast<uint8_t*>(state), reinterpret_cast<uint8_t*>(ws), ws_bytes, keep_d);
  if (rc) { cudaFree(pl->blob); return rc; }
  *out = pl.get();
  g_sh_plans.push_back(std::move(pl));
  return MFSDP_OK;
}

}  // namespace

void release_shampoo_plans() {           // under plan_mutex (mfsdp_release_plans)
  for (auto& p : g_sh_plans) {
    if (cudaSetDevice(p->device) == cudaSuccess) cudaDeviceSynchronize();
    cudaFree(p->blob);
  }
  g_sh_plans.clear();
}

}  // namespace mfsdp

using namespace mfsdp;

extern "C" int mfsdp_shampoo_state_bytes(const mfsdp_desc_t* desc, size_t n_desc, size_t* bytes) {
  if (!bytes) return MFSDP_EINVAL;
  ShLayout lay;
  const int rc = build_sh_layout(desc, n_desc, false, lay);
  if (rc) return rc;
  *bytes = (size_t)lay.state_bytes;
  return MFSDP_OK;
}

extern "C" int mfsdp_shampoo_workspace_bytes(const mfsdp_desc_t* desc, size_t n_desc, uint32_t flags, size_t* min_bytes,
                                             size_t* full_bytes) {
  if (flags & ~(uint32_t)MFSDP_SHAMPOO_KEEP_D) return MFSDP_EINVAL;
  ShLayout lay;
  const int rc = build_sh_layout(desc, n_desc, (flags & MFSDP_SHAMPOO_KEEP_D) != 0, lay);
  if (rc) return rc;
  if (min_bytes) *min_bytes = (size_t)(lay.base_bytes + lay.max_root_bytes);
  if (full_bytes) *full_bytes = (size_t)(lay.base_bytes + lay.all_root_bytes);
  return MFSDP_OK;
}

extern "C" int mfsdp_shampoo_view(const mfsdp_desc_t* desc, size_t n_desc, uint32_t flags, size_t index, size_t out[12]) {
  if (!out || (flags & ~(uint32_t)MFSDP_SHAMPOO_KEEP_D)) return MFSDP_EINVAL;
  ShLayout lay;
  const int rc = build_sh_layout(desc, n_desc, (flags & MFSDP_SHAMPOO_KEEP_D) != 0, lay);
  if (rc) return rc;
  if (index >= lay.mats.size()) return MFSDP_EINVAL;
  const ShMat& m = lay.mats[index];
  out[0] = m.L_off; out[1] = m.R_off; out[2] = m.PL_off; out[3] = m.PR_off;
  out[4] = m.pr; out[5] = m.pc;
  out[6] = (size_t)m.rows * m.pr; out[7] = (size_t)m.cols * m.pc;
  out[8] = (flags & MFSDP_SHAMPOO_KEEP_D) ? m.D_off : 0;
  out[9] = lay.ctl_off + 2 * index * sizeof(ShCtl);
  out[10] = sizeof(ShCtl);
  out[11] = lay.ctl_off + 2 * lay.mats.size() * sizeof(ShCtl);
  return MFSDP_OK;
}

extern "C" int mfsdp_shampoo_step(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* state,
                                  size_t state_bytes, void* workspace, size_t ws_bytes,
                                  const mfsdp_shampoo_hparams_t* hp, void* cuda_stream) {
  if (!hp || (n_desc && !desc)) return MFSDP_EINVAL;
  if (hp->step < 1 || hp->root_every < 1 || hp->max_root_iters < 0 || hp->max_root_iters > 1000) return MFSDP_EINVAL;
  if (!(hp->beta2 > 0.0 && hp->beta2 <= 1.0) || !(hp->eps >= 0.0) || !(hp->eps_floor >= 0.0) || !(hp->root_tol >= 0.0)) return MFSDP_EINVAL;
  if (!(hp->lr == hp->lr) || !(hp->weight_decay == hp->weight_decay)) return MFSDP_EINVAL;
  if ((hp->flags & ~(uint32_t)MFSDP_SHAMPOO_KEEP_D) || hp->reserved) return MFSDP_EINVAL;
  bool any = false;
  for (size_t i = 0; i < n_desc; ++i) any |= desc[i].role == MFSDP_ROLE_MATRIX;
  if (!any) return mfsdp_validate_desc(desc, n_desc);
  if (!W || !G || !state || !workspace) return MFSDP_EINVAL;
  if ((reinterpret_cast<uintptr_t>(state) % kBufAlign) || (reinterpret_cast<uintptr_t>(workspace) % kBufAlign) ||
      (reinterpret_cast<uintptr_t>(W) % 16) || (reinterpret_cast<uintptr_t>(G) % 16))
    return MFSDP_EINVAL;
  const bool keep_d = (hp->flags & MFSDP_SHAMPOO_KEEP_D) != 0;
  ShPlan* pl = nullptr;
  int rc = get_sh_plan(desc, n_desc, W, G, state, workspace, ws_bytes, keep_d, &pl);
  if (rc) return rc;
  if (state_bytes < pl->lay.state_bytes) return MFSDP_ECAP;
  cudaStream_t st = reinterpret_cast<cudaStream_t>(cuda_stream);
  {                                       // the addresses the records point to are plan state: compare under the lock
    std::lock_guard<std::mutex> lock(plan_mutex());
    if (pl->W != W || pl->G != G)
      if ((rc = repoint_sh_plan(*pl, reinterpret_cast<uint8_t*>(W), reinterpret_cast<const uint8_t*>(G), st))) return rc;
  }
  uint8_t* ws = reinterpret_cast<uint8_t*>(workspace);
  ShCtl* d_ctl = reinterpret_cast<ShCtl*>(ws + pl->lay.ctl_off);
  double* d_part = reinterpret_cast<double*>(ws + pl->lay.partial_off);

  if (pl->n_gprep) {
    k_sh_gprep<<<dim3(std::min<uint32_t>(pl->max_rows, 2048u), pl->n_gprep), 256, 0, st>>>(pl->d_gprep);
    count_launch();
    if ((rc = check_last_launch())) return rc;
  }
  const double w = hp->beta2 == 1.0 ? 1.0 : 1.0 - hp->beta2;                    // reading S1
  if ((rc = sg_launch(*pl, pl->stat, (float)w, (float)hp->beta2, 0.f, 0.f, st))) return rc;

  if ((hp->step - 1) % hp->root_every == 0) {                                   // reading S5
    // Launch budget.  The smallest eigenvalue of M_0 is at least mu0 = 2.5 rho / bound >= 2.5 eps_floor / (1 + eps_floor);
    // the scaled phase takes it to 0.2 in log(0.2 / mu0) / log(6.1) iterations (7 with the default floor 2^-20), the
    // plain iteration needs at most 9 more down to the noise floor: 16 (13 observed at most); without a floor 40.
    // Converged problems skip their tiles anyway; the budget only bounds the number of (then empty) launches enqueued.
    uint32_t max_iters = 40u;
    if (hp->max_root_iters) max_iters = (uint32_t)hp->max_root_iters;
    else if (hp->eps_floor > 0.0)
      max_iters = std::min<uint32_t>(40u, (uint32_t)std::ceil(std::log(0.08 * (1.0 + hp->eps_floor) / hp->eps_floor) / std::log(6.103515625)) + 9u);
    const float tol = hp->root_tol > 0.0 ? (float)hp->root_tol : 1e-6f;
    for (const RootGroup& g : pl->groups) {
      const RootInfo* roots = pl->d_roots + g.root_off;
      k_sh_reduce<<<dim3(kRedBlocks, g.n_roots), 256, 0, st>>>(roots, d_part);
      for (uint32_t it = 0; it < kPowerIters; ++it) k_sh_power<<<dim3(kRedBlocks, g.n_roots), 256, 0, st>>>(roots, d_part, it);
      count_launch(kPowerIters);
      k_sh_root_init<<<(g.n_roots + 127) / 128, 128, 0, st>>>(roots, g.n_roots, d_ctl, d_part, hp->eps, hp->eps_floor);
      k_sh_root_prep<<<dim3(std::min<uint32_t>(g.max_d, 1024u), g.n_roots), 256, 0, st>>>(roots, d_ctl);
      count_launch(3);
      if ((rc = check_last_launch())) return rc;
      for (uint32_t it = 0; it < max_iters; ++it) {
        if ((rc = sg_launch(*pl, g.a[it & 1u], 1.f, 0.f, 0.f, 0.f, st))) return rc;
        if ((rc = sg_launch(*pl, g.b, 1.f, 0.f, 0.f, 0.f, st))) return rc;
        if ((rc = sg_launch(*pl, g.c[it & 1u], 1.f, 0.f, 0.f, 0.f, st))) return rc;
        k_sh_root_ctl<<<(g.n_roots + 127) / 128, 128, 0, st>>>(roots, g.n_roots, d_ctl, tol, max_iters);
        count_launch();
      }
      k_sh_root_finish<<<dim3(std::min<uint32_t>(g.max_d, 1024u), g.n_roots), 256, 0, st>>>(roots, d_ctl);
      count_launch();
      if ((rc = check_last_launch())) return rc;
    }
    const uint32_t n_prob = 2u * (uint32_t)pl->lay.mats.size();
    k_sh_status<<<1, 256, 0, st>>>(d_ctl, n_prob, reinterpret_cast<uint32_t*>(d_ctl + n_prob));
    count_launch();
    if ((rc = check_last_launch())) return rc;
  }
  if ((rc = sg_launch(*pl, pl->pre1, 1.f, 0.f, 0.f, 0.f, st))) return rc;
  const float decay = (float)(1.0 - hp->lr * hp->weight_decay);
  return sg_launch(*pl, pl->pre2, 1.f, 0.f, decay, (float)hp->lr, st);
}
