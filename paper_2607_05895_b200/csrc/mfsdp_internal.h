// Internal declarations shared by the translation units of libmfsdp (not part of the C ABI).
#ifndef MFSDP_INTERNAL_H_
#define MFSDP_INTERNAL_H_

#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>
#include <vector>

#include "mfsdp.h"

namespace mfsdp {

// ---- workspace layout ---------------------------------------------------------------------------------------
// [ssq: double x n_mat][inv_norm: float x n_mat][partials: double x n_chunks] then per matrix X0, X1 (rows x
// pitch_x), A, P (d x pitch_a), every buffer 1024-byte aligned (TMA / 128B-swizzle friendly).
constexpr uint32_t kChunk = 16384;       // elements per elementwise work unit (256 threads x 8 vectors of 8)
constexpr uint32_t kTailChunk = 2048;    // tails are short (<= ~1e5 elements per rank): one vector per thread spreads them over the SMs
constexpr uint32_t kEwThreads = 256;
constexpr size_t kBufAlign = 1024;

struct MatLayout {          // host + device; one per MATRIX descriptor, in table order
  uint64_t elem_off;        // element offset into W / G / M
  uint64_t numel;           // rows * cols
  uint64_t x_off[2];        // byte offsets of the X ping-pong buffers in the workspace
  uint64_t a_off, p_off;    // byte offsets of A and P = aI + bA + cA^2
  uint32_t rows, cols;      // as stored
  uint32_t d, n_long;       // d = min(rows, cols), n_long = max(rows, cols)
  uint32_t pitch_x, pitch_a;  // row pitches in elements
  uint32_t chunk_begin;     // index of this matrix' first chunk (partials / grid mapping)
  uint32_t tall;            // rows > cols
  double scale[3];          // update scale s(rows, cols) per MFSDP_SCALE_* mode (reading M7)
};

struct TailLayout {         // one per TAIL descriptor
  uint64_t elem_off;
  uint64_t numel;
  uint32_t chunk_begin;
  uint32_t pad;
};

struct WsLayout {
  std::vector<MatLayout> mats;
  std::vector<TailLayout> tails;
  uint32_t n_chunks = 0;        // matrix chunks
  uint32_t n_tail_chunks = 0;
  size_t ssq_off = 0, invn_off = 0, partial_off = 0;
  size_t total_bytes = 0;
  int mat_dtype = -1, tail_dtype = -1;   // MFSDP_BF16 / MFSDP_F32, -1 = none
};

// Builds the layout; returns an MFSDP_* code (EINVAL on mixed dtypes / bad table, ELAYOUT from validation).
int build_ws_layout(const mfsdp_desc_t* desc, size_t n_desc, int precision, WsLayout& out);

// ---- per-table device state (cached) --------------------------------------------------------------------------
struct NsTcPlan;   // tcgen05 path tables (ns_tc.cu)

struct Plan {
  WsLayout lay;
  int precision = 0;
  void* workspace = nullptr;
  int device = -1;
  MatLayout* d_mats = nullptr;      // device copies
  TailLayout* d_tails = nullptr;
  uint32_t* d_chunk_begin = nullptr;       // [n_mat + 1]
  uint32_t* d_tail_chunk_begin = nullptr;  // [n_tail + 1]
  uint32_t* d_chunk_mat = nullptr;         // [n_chunks] chunk -> matrix index
  uint32_t* d_chunk_tail = nullptr;        // [n_tail_chunks] chunk -> tail index
  uint64_t* d_fan = nullptr;               // [n_mat] fan-out destination address per matrix (mfsdp_muon_step_fanout)
  NsTcPlan* tc = nullptr;
};

// Finds or builds the plan for this (table, workspace, precision) on the current device.
int get_plan(const mfsdp_desc_t* desc, size_t n_desc, int precision, void* workspace, bool need_ws, Plan** out);

// ---- kernels (host launchers); all return an MFSDP_* code ------------------------------------------------------
int launch_momentum(const Plan& pl, const void* G, void* M, const mfsdp_muon_hparams_t& hp, cudaStream_t st,
                    const uint32_t* ready = nullptr, uint32_t epoch = 0);   // ready != nullptr: gated per matrix
int launch_update(const Plan& pl, void* W, const mfsdp_muon_hparams_t& hp, cudaStream_t st,
                  const uint64_t* fan = nullptr);   // fan != nullptr: device table of fan-out destinations (0 = none)
int launch_adamw(const Plan& pl, void* P, const void* G, void* m, void* v, const mfsdp_adamw_hparams_t& hp,
                 cudaStream_t st);
int launch_ns_fp32(const Plan& pl, const mfsdp_muon_hparams_t& hp, cudaStream_t st);
int launch_ns_tc(Plan& pl, const mfsdp_muon_hparams_t& hp, cudaStream_t st, void* W = nullptr, bool keep_o = true,
                 const uint64_t* fan = nullptr);
bool ns_tc_can_fuse_update(Plan& pl);   // bf16 weights, every cols % 8 == 0: the update runs in the last APPLY epilogue
void destroy_ns_tc(NsTcPlan* p);
void release_shampoo_plans();          // shampoo.cu; caller holds plan_mutex()
int ns_class(uint32_t rows, uint32_t cols);   // 0 whole-matrix kernel, 1 single-CTA tiles, 2 CTA-pair tiles

// ---- bookkeeping ---------------------------------------------------------------------------------------------
void count_launch(uint64_t n = 1);
int cuda_fail(cudaError_t e);          // records the error text, returns MFSDP_ECUDA
int check_last_launch();               // cudaGetLastError -> code

int tune_value(int knob);                                  // current value of an MFSDP_TUNE_* knob
void get_trace(unsigned long long** buf, uint32_t* cap);   // mfsdp_debug_trace target (null when off)
std::mutex& plan_mutex();                                  // guards the plan cache and lazily built launch tables

inline uint64_t align_up_u64(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

}  // namespace mfsdp

#endif  // MFSDP_INTERNAL_H_
