// Newton-Schulz in fp32 (MFSDP_NS_FP32): plain FFMA tiles, no tensor cores, no TF32 -- the "fp32 mode" of the
// north_star (<= 1e-4 against the fp64 oracle; the paper's own equivalence harness also disables TF32).
// Per iteration and matrix, with Y the d x n view of X (Y = X for wide, Y = X^T for tall, read through strides):
//   A = alpha Y Y^T ;  P = a I + b A + c A A ;  Y <- beta P Y          (alpha = 1/||U||^2, beta = 1/||U|| at iteration 0)
// One launch per phase for all matrices: blockIdx.y = matrix, blockIdx.x = 64x64 output tile.
#include "mfsdp_internal.h"

namespace mfsdp {
namespace {

constexpr int kK = 32;    // k slab
// Output tile kT x kT per CTA of 256 threads (thread = kT/16 x kT/16 outputs): 64 for throughput, 32 when the whole
// set has so few 64-tiles that most SMs would idle (BASELINE config 1: 2 matrices, 16-64 tiles per phase).

enum { PH_GRAM = 0, PH_POLY = 1, PH_APPLY = 2 };

struct NsArgs {
  const MatLayout* mats;
  uint8_t* ws;
  const float* inv_norm;
  int phase, src, first;     // src: X buffer read this iteration; first: iteration 0 (fold the normalisation)
  float a, b, c;
};

template <int kT>
__global__ void __launch_bounds__(256) k_ns_fp32(NsArgs g) {
  constexpr int kPer = kT * kK / 256;   // slab elements per thread and operand
  constexpr int kR = kT / 16;           // outputs per thread and dimension
  const MatLayout L = g.mats[blockIdx.y];
  const uint32_t d = L.d, n = L.n_long;
  const uint32_t Mo = d, No = (g.phase == PH_APPLY) ? n : d, Kd = (g.phase == PH_GRAM) ? n : d;
  const uint32_t tiles_n = (No + kT - 1) / kT, tiles_m = (Mo + kT - 1) / kT;
  if (blockIdx.x >= tiles_m * tiles_n) return;
  const uint32_t i0 = (blockIdx.x / tiles_n) * kT, j0 = (blockIdx.x % tiles_n) * kT;

  const float* X = reinterpret_cast<const float*>(g.ws + L.x_off[g.src]);
  float* Xn = reinterpret_cast<float*>(g.ws + L.x_off[g.src ^ 1]);
  float* A = reinterpret_cast<float*>(g.ws + L.a_off);
  float* P = reinterpret_cast<float*>(g.ws + L.p_off);
  // Y[i, k] = X[i * sy_i + k * sy_k]
  const uint64_t sy_i = L.tall ? 1 : L.pitch_x, sy_k = L.tall ? L.pitch_x : 1;
  const float *Ap, *Bp; float* Cp;
  uint64_t sa_i, sa_k, sb_k, sb_j, sc_i, sc_j;
  if (g.phase == PH_GRAM)      { Ap = X; sa_i = sy_i; sa_k = sy_k; Bp = X; sb_k = sy_k; sb_j = sy_i; Cp = A; sc_i = L.pitch_a; sc_j = 1; }
  else if (g.phase == PH_POLY) { Ap = A; sa_i = L.pitch_a; sa_k = 1; Bp = A; sb_k = L.pitch_a; sb_j = 1; Cp = P; sc_i = L.pitch_a; sc_j = 1; }
  else                         { Ap = P; sa_i = L.pitch_a; sa_k = 1; Bp = X; sb_k = sy_i; sb_j = sy_k; Cp = Xn; sc_i = sy_i; sc_j = sy_k; }

  __shared__ float sA[kK][kT + 1];
  __shared__ float sB[kK][kT + 1];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  // Slab element e = threadIdx.x + 256 r of an operand -> (mn, k): the index that is contiguous in memory runs fastest
  // across the threads (coalesced loads for both the plain and the transposed views).
  const bool a_kfast = sa_k == 1, b_kfast = sb_k == 1;
  float ra[kPer], rb[kPer];
  auto fetch = [&](uint32_t k0) {
#pragma unroll
    for (int r = 0; r < kPer; ++r) {
      const int e = threadIdx.x + 256 * r;
      const int am = a_kfast ? e / kK : e % kT, ak = a_kfast ? e % kK : e / kT;
      const uint32_t i = i0 + am, k = k0 + ak;
      ra[r] = (i < Mo && k < Kd) ? Ap[i * sa_i + k * sa_k] : 0.f;
      const int bm = b_kfast ? e / kK : e % kT, bk = b_kfast ? e % kK : e / kT;
      const uint32_t j = j0 + bm, k2 = k0 + bk;
      rb[r] = (j < No && k2 < Kd) ? Bp[k2 * sb_k + j * sb_j] : 0.f;
    }
  };
  auto stash = [&]() {
#pragma unroll
    for (int r = 0; r < kPer; ++r) {
      const int e = threadIdx.x + 256 * r;
      const int am = a_kfast ? e / kK : e % kT, ak = a_kfast ? e % kK : e / kT;
      sA[ak][am] = ra[r];
      const int bm = b_kfast ? e / kK : e % kT, bk = b_kfast ? e % kK : e / kT;
      sB[bk][bm] = rb[r];
    }
  };
  float acc[kR][kR] = {};
  fetch(0);
  for (uint32_t k0 = 0; k0 < Kd; k0 += kK) {
    stash();
    __syncthreads();
    if (k0 + kK < Kd) fetch(k0 + kK);        // next slab in flight (registers) while this one is multiplied
#pragma unroll
    for (int kk = 0; kk < kK; ++kk) {
      float av[kR], bv[kR];
#pragma unroll
      for (int r = 0; r < kR; ++r) { av[r] = sA[kk][ty * kR + r]; bv[r] = sB[kk][tx * kR + r]; }
#pragma unroll
      for (int r = 0; r < kR; ++r)
#pragma unroll
        for (int s = 0; s < kR; ++s) acc[r][s] = fmaf(av[r], bv[s], acc[r][s]);
    }
    __syncthreads();
  }
  const float inv = g.first ? g.inv_norm[blockIdx.y] : 1.f;
  const float alpha = (g.phase == PH_GRAM) ? inv * inv : (g.phase == PH_APPLY ? inv : 1.f);
#pragma unroll
  for (int r = 0; r < kR; ++r)
#pragma unroll
    for (int s = 0; s < kR; ++s) {
      const uint32_t i = i0 + ty * kR + r, j = j0 + tx * kR + s;
      if (i >= Mo || j >= No) continue;
      float out;
      if (g.phase == PH_POLY) out = fmaf(g.c, acc[r][s], fmaf(g.b, A[i * sc_i + j], (i == j) ? g.a : 0.f));
      else out = alpha * acc[r][s];
      Cp[i * sc_i + j * sc_j] = out;
    }
}

}  // namespace

int launch_ns_fp32(const Plan& pl, const mfsdp_muon_hparams_t& hp, cudaStream_t st) {
  const WsLayout& lay = pl.lay;
  const uint32_t n_mat = (uint32_t)lay.mats.size();
  if (n_mat == 0) return MFSDP_OK;
  int dev = 0, sms = 148;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  uint32_t max_gram = 1, max_apply = 1;
  uint64_t total_apply = 0;
  int kT = 64;
  for (int pass = 0; pass < 2; ++pass) {
    max_gram = max_apply = 1; total_apply = 0;
    for (const MatLayout& L : lay.mats) {
      const uint32_t td = (L.d + kT - 1) / kT, tn = (L.n_long + kT - 1) / kT;
      max_gram = td * td > max_gram ? td * td : max_gram;
      max_apply = td * tn > max_apply ? td * tn : max_apply;
      total_apply += (uint64_t)td * tn;
    }
    if (kT == 32 || total_apply >= 2ull * (uint64_t)sms) break;    // enough 64-tiles to fill the SMs
    kT = 32;
  }
  NsArgs g;
  g.mats = pl.d_mats;
  g.ws = static_cast<uint8_t*>(pl.workspace);
  g.inv_norm = reinterpret_cast<const float*>(g.ws + lay.invn_off);
  g.a = (float)hp.a; g.b = (float)hp.b; g.c = (float)hp.c;
  for (int it = 0; it < hp.ns_steps; ++it) {
    g.src = it & 1;
    g.first = (it == 0);
    for (int ph = 0; ph < 3; ++ph) {
      g.phase = ph;
      const dim3 grid(ph == PH_APPLY ? max_apply : max_gram, n_mat);
      if (kT == 64) k_ns_fp32<64><<<grid, 256, 0, st>>>(g); else k_ns_fp32<32><<<grid, 256, 0, st>>>(g);
      count_launch();
      const int rc = check_last_launch();
      if (rc) return rc;
    }
  }
  return MFSDP_OK;
}

}  // namespace mfsdp
