// mfsdp_momentum_pass_static: the momentum pass of ONE matrix (SURVEY.md 8(a) a1 + the scalar part of a2) for callers
// that may not allocate device memory.
//
// Who that is.  Every other step call of this library builds, on its first use of a (table, workspace) pair, a set of
// launch tables in device memory of its own (cudaMalloc + cudaMemcpy in get_plan / the tensor-map builders), and wants a
// workspace the caller allocates.  Some callers can do neither:
//   * a trainer whose framework allocator has claimed the device up to a planned budget (180 GB filled on purpose with
//     shards, state and activations): a raw cudaMalloc behind that allocator's back may fail, or may push the job over
//     a memory limit the cluster manager enforces;
//   * code that runs inside the step loop while other streams are busy (the gradient reduction of PAPER.md:83 is still
//     in flight when the owner starts its optimizer work): cudaMalloc and cudaFree synchronise the whole device, which
//     stalls exactly the overlap MatrixFSDP's owner layout is there to give;
//   * a plug-in called from a host callback or from a library that forbids CUDA memory management in its hooks.
// For them this entry point keeps the one piece of scratch the pass needs -- the per-chunk partial sums of ||U||^2 that
// sit between the streaming kernel and the fixed-order reduction -- in a file-scope array in device memory that ships
// with the library image.  The caller passes inputs and outputs only; nothing is allocated, copied from the host or freed.
//
// The price, stated once:
//   * the array has a fixed size (kStaticMaxChunks doubles = 512 KiB), and every GPU that loads the library holds it
//     until the process exits, whether or not this entry point is ever called;
//   * matrices above kStaticMaxChunks * 16384 = 2^30 elements are refused (MFSDP_ETOOBIG), not split;
//   * all calls on one device share the array.  It keeps whatever the last call left in it; that is harmless here
//     because a call writes every partial it later reads and nothing has to start at zero.  Two calls that overlap on
//     the GPU (different streams, no ordering between them) write the same partials and race: order them.
//
// Set-up.  In host code the name of a __device__ array is only a handle, not an address the GPU can use, so the first
// call on each device looks the address up with cudaGetSymbolAddress (with that device current), checks the result and
// keeps it.  That first call also makes the runtime load the library's device code, so it should be made before any
// stream capture begins; later calls on the same device only launch two kernels.
//
// The arithmetic, the element -> thread mapping and both reduction orders repeat k_momentum / k_ssq of elementwise.cu
// exactly (this file shares no code with it, so that the existing path is untouched): M, X~ and ||U||^2 come out
// bit-identical to mfsdp_muon_momentum_pass on a table that holds the same matrix (tests/test_zz_no_alloc.py).
#include <cuda_bf16.h>

#include <mutex>

#include "mfsdp_internal.h"

namespace mfsdp {
namespace {

constexpr uint32_t kStaticMaxChunks = 65536;                         // 512 KiB of doubles
constexpr uint64_t kStaticMaxElems = (uint64_t)kStaticMaxChunks * kChunk;   // 2^30
constexpr int kMaxDevices = 64;
constexpr int kVecs = (int)(kChunk / (kEwThreads * 8));              // 8 vectors of 8 elements per thread and chunk

// The scratch itself.  Host code below never passes this name to a kernel: it passes the address looked up at set-up.
static __device__ __align__(256) double g_static_partial[kStaticMaxChunks];

std::mutex g_setup_mu;
double* g_partial_addr[kMaxDevices] = {};      // per device ordinal, filled on that device's first call
int g_sm_count[kMaxDevices] = {};

struct V8 { float v[8]; };

__device__ __forceinline__ V8 ld8(const float* p) {
  V8 r;
  const float4 a = *reinterpret_cast<const float4*>(p);
  const float4 b = *reinterpret_cast<const float4*>(p + 4);
  r.v[0] = a.x; r.v[1] = a.y; r.v[2] = a.z; r.v[3] = a.w; r.v[4] = b.x; r.v[5] = b.y; r.v[6] = b.z; r.v[7] = b.w;
  return r;
}
__device__ __forceinline__ V8 ld8(const __nv_bfloat16* p) {
  V8 r;
  const uint4 u = *reinterpret_cast<const uint4*>(p);
  const uint32_t w[4] = {u.x, u.y, u.z, u.w};
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    r.v[2 * i] = __uint_as_float(w[i] << 16);
    r.v[2 * i + 1] = __uint_as_float(w[i] & 0xffff0000u);
  }
  return r;
}
__device__ __forceinline__ void st8(float* p, const V8& x) {
  *reinterpret_cast<float4*>(p) = make_float4(x.v[0], x.v[1], x.v[2], x.v[3]);
  *reinterpret_cast<float4*>(p + 4) = make_float4(x.v[4], x.v[5], x.v[6], x.v[7]);
}
__device__ __forceinline__ void st8(__nv_bfloat16* p, const V8& x) {
  uint32_t w[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const __nv_bfloat162 h = __floats2bfloat162_rn(x.v[2 * i], x.v[2 * i + 1]);
    w[i] = *reinterpret_cast<const uint32_t*>(&h);
  }
  *reinterpret_cast<uint4*>(p) = make_uint4(w[0], w[1], w[2], w[3]);
}
__device__ __forceinline__ float ld1(const float* p) { return *p; }
__device__ __forceinline__ float ld1(const __nv_bfloat16* p) { return __bfloat162float(*p); }
__device__ __forceinline__ void st1(float* p, float x) { *p = x; }
__device__ __forceinline__ void st1(__nv_bfloat16* p, float x) { *p = __float2bfloat16_rn(x); }

// Fixed shuffle tree, then warp 0 adds the warp sums in order: the same order as block_sum of elementwise.cu.
__device__ __forceinline__ double block_sum_fixed(double x, double* smem) {
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

// M <- mu M + (1-mu) G ; U = (1-mu) G + mu M | M ; X = cast(U) ; partial[c] = sum of U^2 over chunk c.
// One matrix, everything contiguous (X has row pitch = cols), so every whole 8-element vector moves as 128 bits.
template <typename GT, typename XT>
__global__ void __launch_bounds__(kEwThreads) k_momentum_one(const GT* __restrict__ g, float* __restrict__ m,
                                                             XT* __restrict__ x, uint64_t numel, uint32_t n_chunks,
                                                             double* __restrict__ partial, float mu, float omm,
                                                             int nesterov) {
  __shared__ double red[kEwThreads / 32];
  for (uint32_t c = blockIdx.x; c < n_chunks; c += gridDim.x) {
    const uint64_t base = (uint64_t)c * kChunk;
    double acc = 0.0;
    for (int it = 0; it < kVecs; ++it) {
      const uint64_t e0 = base + ((uint64_t)it * kEwThreads + threadIdx.x) * 8;
      if (e0 >= numel) break;
      if (e0 + 8 <= numel) {
        const V8 gv = ld8(g + e0);
        V8 mv = ld8(m + e0);
        V8 uv;
#pragma unroll
        for (int i = 0; i < 8; ++i) {
          const float gs = omm * gv.v[i];
          mv.v[i] = fmaf(mu, mv.v[i], gs);
          uv.v[i] = nesterov ? fmaf(mu, mv.v[i], gs) : mv.v[i];
          acc = fma((double)uv.v[i], (double)uv.v[i], acc);
        }
        st8(m + e0, mv);
        st8(x + e0, uv);
      } else {
        for (uint64_t e = e0; e < numel; ++e) {
          const float gs = omm * ld1(g + e);
          const float mn = fmaf(mu, m[e], gs);
          const float u = nesterov ? fmaf(mu, mn, gs) : mn;
          acc = fma((double)u, (double)u, acc);
          m[e] = mn;
          st1(x + e, u);
        }
      }
    }
    const double s = block_sum_fixed(acc, red);
    if (threadIdx.x == 0) partial[c] = s;
  }
}

// ||U||^2 = the partials added in a fixed order by one block; 1 / max(||U||, eps).
__global__ void __launch_bounds__(kEwThreads) k_ssq_one(const double* __restrict__ partial, uint32_t n_chunks,
                                                        double* __restrict__ ssq, float* __restrict__ inv_norm,
                                                        double eps) {
  __shared__ double red[kEwThreads / 32];
  double acc = 0.0;
  for (uint32_t c = threadIdx.x; c < n_chunks; c += kEwThreads) acc += partial[c];
  const double s = block_sum_fixed(acc, red);
  if (threadIdx.x == 0) {
    *ssq = s;
    const double nrm = sqrt(s);
    *inv_norm = (float)(1.0 / (nrm > eps ? nrm : eps));
  }
}

// Once per device, with that device current: the device address of the scratch array and the SM count.
int static_setup(int dev, double** partial, int* sms) {
  std::lock_guard<std::mutex> lock(g_setup_mu);
  if (!g_partial_addr[dev]) {
    int major = 0, n_sm = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e != cudaSuccess) return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? MFSDP_EARCH : cuda_fail(e);
    if (major != 10) return MFSDP_EARCH;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return cuda_fail(e);
    double* addr = nullptr;
    if ((e = cudaGetSymbolAddress(reinterpret_cast<void**>(&addr), g_static_partial)) != cudaSuccess) return cuda_fail(e);
    if (!addr) return cuda_fail(cudaErrorInvalidSymbol);
    g_sm_count[dev] = n_sm;
    g_partial_addr[dev] = addr;
  }
  *partial = g_partial_addr[dev];
  *sms = g_sm_count[dev];
  return MFSDP_OK;
}

bool aligned_to(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

}  // namespace
}  // namespace mfsdp

using namespace mfsdp;

extern "C" uint64_t mfsdp_static_max_elems(void) { return kStaticMaxElems; }

extern "C" int mfsdp_momentum_pass_static(uint32_t rows, uint32_t cols, int dtype, int precision, const void* G, void* M,
                                          void* X, double* ssq, float* inv_norm, const mfsdp_muon_hparams_t* hp,
                                          void* cuda_stream) {
  if (!hp || !(hp->momentum >= 0.0 && hp->momentum < 1.0) || !(hp->eps > 0.0)) return MFSDP_EINVAL;
  if (dtype != MFSDP_BF16 && dtype != MFSDP_F32) return MFSDP_EINVAL;
  if (precision != MFSDP_NS_BF16 && precision != MFSDP_NS_FP32) return MFSDP_EINVAL;
  if (rows == 0 || cols == 0) return MFSDP_EINVAL;
  if (!G || !M || !X || !ssq || !inv_norm) return MFSDP_EINVAL;
  if (!aligned_to(G, 16) || !aligned_to(M, 16) || !aligned_to(X, 16) || !aligned_to(ssq, 8) || !aligned_to(inv_norm, 4))
    return MFSDP_EINVAL;
  const uint64_t numel = (uint64_t)rows * cols;
  if (numel > kStaticMaxElems) return MFSDP_ETOOBIG;     // the fixed array has no partial for the chunks beyond it

  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? MFSDP_EARCH : cuda_fail(e);
  if (dev < 0 || dev >= kMaxDevices) return MFSDP_EINVAL;
  double* partial = nullptr;
  int sms = 0;
  const int rc = static_setup(dev, &partial, &sms);
  if (rc) return rc;

  const uint32_t n_chunks = (uint32_t)((numel + kChunk - 1) / kChunk);
  const uint32_t cap = (uint32_t)sms * 8u;               // 8 resident CTAs of 256 threads per SM
  const int grid = (int)(n_chunks < cap ? n_chunks : cap);
  const float mu = (float)hp->momentum, omm = (float)(1.0 - hp->momentum);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const bool gbf = dtype == MFSDP_BF16, xbf = precision == MFSDP_NS_BF16;
#define MOM1(GT, XT)                                                                                                   \
  k_momentum_one<GT, XT><<<grid, kEwThreads, 0, st>>>(static_cast<const GT*>(G), static_cast<float*>(M),               \
                                                      static_cast<XT*>(X), numel, n_chunks, partial, mu, omm,          \
                                                      hp->nesterov)
  if (gbf && xbf) MOM1(__nv_bfloat16, __nv_bfloat16);
  else if (gbf) MOM1(__nv_bfloat16, float);
  else if (xbf) MOM1(float, __nv_bfloat16);
  else MOM1(float, float);
#undef MOM1
  count_launch();
  int lrc = check_last_launch();
  if (lrc) return lrc;
  k_ssq_one<<<1, kEwThreads, 0, st>>>(partial, n_chunks, ssq, inv_norm, hp->eps);
  count_launch();
  return check_last_launch();
}
