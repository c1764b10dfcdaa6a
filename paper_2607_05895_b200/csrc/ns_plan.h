// Launch tables of the bf16 Newton-Schulz path, shared by the tile kernel (ns_tc.cu) and the whole-matrix kernel
// (ns_fused.cu).  Internal to libmfsdp.
#ifndef MFSDP_NS_PLAN_H_
#define MFSDP_NS_PLAN_H_

#include <cuda.h>
#include <stdint.h>

#include "mfsdp_internal.h"

namespace mfsdp {

enum { PH_GRAM = 0, PH_POLY = 1, PH_APPLY = 2 };
// tensor maps per matrix
enum { TM_X0 = 0, TM_X1 = 1, TM_A = 2, TM_P = 3,            // operand loads: box 64 x 64, 128-byte swizzle
       TM_X0_ST = 4, TM_X1_ST = 5, TM_A_ST = 6, TM_P_ST = 7,  // epilogue tiles: box 64 cols x 32 rows, 128-byte swizzle
       TM_A_MIR = 8, TM_P_MIR = 9,                            // mirror tiles: box 32 cols x 64 rows, no swizzle
       TM_COUNT = 10 };

struct TcMat {                 // device, one per matrix
  uint64_t x_off[2], a_off, p_off;
  uint32_t rows, cols, d, n_long, pitch_x, pitch_a, tall;
  uint32_t reports_per_iter;   // completion reports (one per epilogue warp and tile) of one NS iteration of this matrix
};
// Output tile: origin (rows, cols of the OUTPUT buffer), k blocks, width in columns (multiple of 64; of 128 when
// paired; <= 256 single CTA, <= 512 paired).
// `need`: completion reports of the SAME matrix and iteration that must have been made before this tile's operands
// may be read (= every tile of the matrix' earlier phases); `phase`: PH_*.
struct TcTile { uint32_t mat, m0, n0; uint16_t nkb, nw; uint32_t need, phase, reports_per_iter, pad; };

// One matrix of the whole-matrix ("fused") class: d = min(rows, cols) <= 128 and the padded X fits shared memory.
// X is kept row-major as `panels` column panels of 64 elements (128 bytes) x rpad rows, 128-byte swizzled.
struct FusedMat {
  uint32_t mat;                 // index into the matrix tables (tensor maps, inv_norm)
  uint32_t rows, cols, tall;    // as stored
  uint32_t d16;                 // min(rows, cols) rounded up to 16: UMMA N of GRAM / POLY, K of POLY / APPLY
  uint32_t rpad, panels;        // padded rows (multiple of 128), column panels
  uint32_t k16;                 // 16-element k steps of GRAM = ceil(max(rows, cols) / 16)
};

// Weight-update inputs per matrix (the update fused into the last APPLY epilogue): W <- W (1 - lr wd) - lr s O.
struct TcUpd { uint64_t elem_off; double scale[3]; };   // element offset into the rank-flat W; s per MFSDP_SCALE_* mode
struct UpdArgs {                 // W == nullptr: no fused update (the pass only leaves O in the workspace)
  void* W;
  const TcUpd* upd;
  double lr;
  float decay;
  int scale_mode;
  uint32_t keep_o;               // also store O (tests, callers that consume the orthogonalised update)
  const uint64_t* fan;           // optional: per matrix the address of a fan-out copy of the updated W (0 = none)
};

enum { kCounterWords = 5 };         // [0], [1] tile counters of the single-CTA / CTA-pair class, [2], [3], [4] fused classes

struct NsTcPlan {
  CUtensorMap* d_tmaps = nullptr;   // TM_COUNT per matrix
  TcMat* d_mats = nullptr;
  TcTile* d_tiles[2] = {nullptr, nullptr};   // [kCG - 1]: the tiles of ONE iteration, GRAM then POLY then APPLY
  uint32_t n_tiles[2] = {0, 0};
  // whole-matrix classes: [0] d <= 128, padded X <= 64 KB (2 CTAs / SM), [1] d <= 128, X <= 128 KB (ns_fused.cu);
  // [2] 128 < d <= 256, A / P on chip, X streamed (ns_fused2.cu)
  FusedMat* d_fused[3] = {nullptr, nullptr, nullptr};
  uint32_t n_fused[3] = {0, 0, 0};
  TcUpd* d_upd = nullptr;
  bool upd_ok = false;              // bf16 weights and every cols % 8 == 0: the update can be fused into the epilogues
  uint32_t* d_counters = nullptr;   // kCounterWords work counters then [n_mat] completion reports; zeroed per pass
  uint32_t n_mat = 0;
  int sms = 148;
  int max_pairs = 74;               // co-resident CTA pairs
  cudaStream_t side[4] = {nullptr, nullptr, nullptr, nullptr};   // forked streams: the classes touch disjoint matrices
  cudaEvent_t fork = nullptr, join[4] = {nullptr, nullptr, nullptr, nullptr};
};

// ns_fused.cu
int fused_setup();                                        // kernel attributes (once per plan build)
int launch_ns_fused(const NsTcPlan& tc, int cls, uint8_t* ws, const float* inv_norm, const mfsdp_muon_hparams_t& hp,
                    const UpdArgs& ua, cudaStream_t st);
bool fused_eligible(uint32_t rows, uint32_t cols, uint32_t below_d, FusedMat* out, int* cls);
// ns_fused2.cu
int fused2_setup();
int launch_ns_fused2(const NsTcPlan& tc, const float* inv_norm, const mfsdp_muon_hparams_t& hp, const UpdArgs& ua,
                     cudaStream_t st);
bool fused2_eligible(uint32_t rows, uint32_t cols, uint32_t below_d, FusedMat* out);


}  // namespace mfsdp

#endif  // MFSDP_NS_PLAN_H_
