// C-ABI entry points of the step (include/mfsdp.h): argument checks, workspace layout, the per-table cache of
// device launch tables, and the launch sequence.  No compute happens here and there is no CPU fallback.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <map>
#include <mutex>
#include <string>

#include <cuda.h>

#include "mfsdp_internal.h"

namespace mfsdp {

// ---- bookkeeping ------------------------------------------------------------------------------------------------
namespace {
std::mutex g_mu;        // plan cache, lazily built launch tables, trace target
std::mutex g_host_mu;   // serialises mfsdp_muon_step_host (one set of copy streams per device)
std::atomic<uint64_t> g_launches{0};
thread_local std::string g_cuda_err = "no CUDA error recorded";   // per calling thread (mfsdp_strerror)
std::vector<Plan*> g_plans;
std::vector<std::vector<uint8_t>> g_plan_keys;
constexpr size_t kMaxPlans = 1024;   // cached launch tables; beyond it get_plan fails loudly (MFSDP_ECACHE)

// Scheduling knobs (mfsdp_tune): defaults only -- no environment variables, no other hidden state.
std::atomic<int> g_tune[MFSDP_TUNE_COUNT_] = {{1024}, {16}, {8}, {4}, {8}, {129}, {257}};

unsigned long long* g_trace = nullptr;
uint32_t g_trace_cap = 0;

void free_plan(Plan* pl) {
  if (!pl) return;
  cudaFree(pl->d_mats); cudaFree(pl->d_tails); cudaFree(pl->d_chunk_begin); cudaFree(pl->d_tail_chunk_begin);
  cudaFree(pl->d_chunk_mat); cudaFree(pl->d_chunk_tail); cudaFree(pl->d_fan);
  destroy_ns_tc(pl->tc);
  delete pl;
}
}  // namespace

std::mutex& plan_mutex() { return g_mu; }

void get_trace(unsigned long long** buf, uint32_t* cap) {
  std::lock_guard<std::mutex> lock(g_mu);
  *buf = g_trace; *cap = g_trace_cap;
}

int tune_value(int knob) { return knob >= 0 && knob < MFSDP_TUNE_COUNT_ ? g_tune[knob].load() : -1; }

void count_launch(uint64_t n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
int cuda_fail(cudaError_t e) {
  g_cuda_err = std::string(cudaGetErrorName(e)) + ": " + cudaGetErrorString(e);
  return MFSDP_ECUDA;
}
int check_last_launch() {
  const cudaError_t e = cudaGetLastError();
  return e == cudaSuccess ? MFSDP_OK : cuda_fail(e);
}

// ---- workspace layout -----------------------------------------------------------------------------------------------
int build_ws_layout(const mfsdp_desc_t* desc, size_t n_desc, int precision, WsLayout& out) {
  if (n_desc && !desc) return MFSDP_EINVAL;
  if (precision != MFSDP_NS_BF16 && precision != MFSDP_NS_FP32) return MFSDP_EINVAL;
  const int rc = mfsdp_validate_desc(desc, n_desc);
  if (rc) return rc;
  out = WsLayout();
  const size_t es = precision == MFSDP_NS_BF16 ? 2 : 4;
  const uint32_t pad = 8;                               // row pitches are multiples of 8 elements (16 B for bf16)
  for (size_t i = 0; i < n_desc; ++i) {
    const mfsdp_desc_t& q = desc[i];
    if (q.role == MFSDP_ROLE_MATRIX) {
      if (out.mat_dtype >= 0 && out.mat_dtype != (int)q.dtype) return MFSDP_EINVAL;
      out.mat_dtype = (int)q.dtype;
      MatLayout L;
      std::memset(&L, 0, sizeof L);
      L.elem_off = q.elem_off; L.rows = q.rows; L.cols = q.cols;
      L.numel = (uint64_t)q.rows * q.cols;
      L.tall = q.rows > q.cols;
      L.d = L.tall ? q.cols : q.rows; L.n_long = L.tall ? q.rows : q.cols;
      L.pitch_x = (uint32_t)align_up_u64(q.cols, pad);
      L.pitch_a = (uint32_t)align_up_u64(L.d, pad);
      L.scale[MFSDP_SCALE_MATCH_RMS_ADAMW] = 0.2 * std::sqrt((double)std::max(q.rows, q.cols));
      L.scale[MFSDP_SCALE_ORIGINAL] = std::sqrt(std::max(1.0, (double)q.rows / (double)q.cols));
      L.scale[MFSDP_SCALE_NONE] = 1.0;
      L.chunk_begin = out.n_chunks;
      const uint64_t nch = (L.numel + kChunk - 1) / kChunk;
      if (nch + out.n_chunks > 0x7fffffffull) return MFSDP_EINVAL;
      out.n_chunks += (uint32_t)nch;
      out.mats.push_back(L);
    } else {
      if (out.tail_dtype >= 0 && out.tail_dtype != (int)q.dtype) return MFSDP_EINVAL;
      out.tail_dtype = (int)q.dtype;
      TailLayout T;
      T.elem_off = q.elem_off; T.numel = (uint64_t)q.rows * q.cols; T.chunk_begin = out.n_tail_chunks; T.pad = 0;
      out.n_tail_chunks += (uint32_t)((T.numel + kTailChunk - 1) / kTailChunk);
      out.tails.push_back(T);
    }
  }
  size_t off = 0;
  const size_t n_mat = out.mats.size();
  out.ssq_off = off;     off = align_up_u64(off + n_mat * sizeof(double), kBufAlign);
  out.invn_off = off;    off = align_up_u64(off + n_mat * sizeof(float), kBufAlign);
  out.partial_off = off; off = align_up_u64(off + (size_t)out.n_chunks * sizeof(double), kBufAlign);
  for (MatLayout& L : out.mats) {
    const size_t xb = align_up_u64((size_t)L.rows * L.pitch_x * es, kBufAlign);
    const size_t ab = align_up_u64((size_t)L.d * L.pitch_a * es, kBufAlign);
    L.x_off[0] = off; off += xb;
    L.x_off[1] = off; off += xb;
    L.a_off = off; off += ab;
    L.p_off = off; off += ab;
  }
  out.total_bytes = off;
  return MFSDP_OK;
}

// ---- plan cache ---------------------------------------------------------------------------------------------------------
namespace {
template <typename T>
int upload(T** dptr, const T* h, size_t n) {
  *dptr = nullptr;
  if (n == 0) n = 1;
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(dptr), n * sizeof(T));
  if (e != cudaSuccess) return cuda_fail(e);
  if (h) {
    e = cudaMemcpy(*dptr, h, n * sizeof(T), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(e);
  }
  return MFSDP_OK;
}
}  // namespace

int get_plan(const mfsdp_desc_t* desc, size_t n_desc, int precision, void* workspace, bool need_ws, Plan** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? MFSDP_EARCH : cuda_fail(e);
  int major = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return e == cudaErrorNoDevice || e == cudaErrorInsufficientDriver ? MFSDP_EARCH : cuda_fail(e);
  if (major != 10) return MFSDP_EARCH;

  std::vector<uint8_t> key(sizeof(int) * 2 + sizeof(void*) + n_desc * sizeof(mfsdp_desc_t));
  {
    uint8_t* k = key.data();
    std::memcpy(k, &dev, sizeof(int)); k += sizeof(int);
    std::memcpy(k, &precision, sizeof(int)); k += sizeof(int);
    void* wsk = need_ws ? workspace : nullptr;
    std::memcpy(k, &wsk, sizeof(void*)); k += sizeof(void*);
    if (n_desc) std::memcpy(k, desc, n_desc * sizeof(mfsdp_desc_t));
  }
  std::lock_guard<std::mutex> lock(g_mu);
  for (size_t i = 0; i < g_plans.size(); ++i)
    if (g_plan_keys[i] == key) { *out = g_plans[i]; return MFSDP_OK; }

  Plan* pl = new Plan();
  int rc = build_ws_layout(desc, n_desc, precision, pl->lay);
  if (rc) { delete pl; return rc; }
  pl->precision = precision;
  pl->workspace = need_ws ? workspace : nullptr;
  pl->device = dev;
  const WsLayout& lay = pl->lay;
  std::vector<uint32_t> cb(lay.mats.size() + 1), tcb(lay.tails.size() + 1);
  for (size_t i = 0; i < lay.mats.size(); ++i) cb[i] = lay.mats[i].chunk_begin;
  cb[lay.mats.size()] = lay.n_chunks;
  for (size_t i = 0; i < lay.tails.size(); ++i) tcb[i] = lay.tails[i].chunk_begin;
  tcb[lay.tails.size()] = lay.n_tail_chunks;
  std::vector<uint32_t> cm(lay.n_chunks), ct(lay.n_tail_chunks);
  for (size_t i = 0; i < lay.mats.size(); ++i)
    for (uint32_t c = cb[i]; c < cb[i + 1]; ++c) cm[c] = (uint32_t)i;
  for (size_t i = 0; i < lay.tails.size(); ++i)
    for (uint32_t c = tcb[i]; c < tcb[i + 1]; ++c) ct[c] = (uint32_t)i;
  // A cached plan is never freed behind the caller's back (launches in flight and captured CUDA graphs reference its
  // device tables): a full cache is an error the caller resolves with mfsdp_release_plans().
  if (g_plans.size() >= kMaxPlans) { delete pl; return MFSDP_ECACHE; }
  if ((rc = upload(&pl->d_mats, lay.mats.data(), lay.mats.size())) ||
      (rc = upload(&pl->d_tails, lay.tails.data(), lay.tails.size())) ||
      (rc = upload(&pl->d_chunk_begin, cb.data(), cb.size())) ||
      (rc = upload(&pl->d_tail_chunk_begin, tcb.data(), tcb.size())) ||
      (rc = upload(&pl->d_chunk_mat, cm.data(), cm.size())) || (rc = upload(&pl->d_chunk_tail, ct.data(), ct.size())) ||
      (rc = upload(&pl->d_fan, static_cast<const uint64_t*>(nullptr), lay.mats.size()))) {
    free_plan(pl);
    return rc;
  }
  g_plans.push_back(pl);
  g_plan_keys.push_back(std::move(key));
  *out = pl;
  return MFSDP_OK;
}

namespace {

bool aligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) == 0; }

int check_hp(const mfsdp_muon_hparams_t* hp) {
  if (!hp) return MFSDP_EINVAL;
  if (hp->ns_steps < 1 || hp->ns_steps > 64) return MFSDP_EINVAL;
  if (!(hp->momentum >= 0.0 && hp->momentum < 1.0)) return MFSDP_EINVAL;
  if (!(hp->eps > 0.0) || !(hp->lr == hp->lr) || !(hp->weight_decay == hp->weight_decay)) return MFSDP_EINVAL;
  if (hp->scale_mode < MFSDP_SCALE_MATCH_RMS_ADAMW || hp->scale_mode > MFSDP_SCALE_NONE) return MFSDP_EINVAL;
  if (hp->precision != MFSDP_NS_BF16 && hp->precision != MFSDP_NS_FP32) return MFSDP_EINVAL;
  if ((hp->flags & ~(uint32_t)MFSDP_STEP_KEEP_O) || hp->reserved) return MFSDP_EINVAL;
  return MFSDP_OK;
}

// Common front end of the Muon passes: validates, finds the plan, checks the workspace.
int muon_front(const mfsdp_desc_t* desc, size_t n_desc, void* workspace, size_t ws_bytes,
               const mfsdp_muon_hparams_t* hp, Plan** pl) {
  int rc = check_hp(hp);
  if (rc) return rc;
  if (n_desc && !desc) return MFSDP_EINVAL;
  if (!workspace) {           // allowed only when the table holds no matrix (nothing to do: *pl stays null)
    for (size_t i = 0; i < n_desc; ++i)
      if (desc[i].role == MFSDP_ROLE_MATRIX) return MFSDP_EINVAL;
    *pl = nullptr;
    return MFSDP_OK;
  }
  if (!aligned(workspace, kBufAlign)) return MFSDP_EINVAL;
  rc = get_plan(desc, n_desc, hp->precision, workspace, true, pl);
  if (rc) return rc;
  if (ws_bytes < (*pl)->lay.total_bytes) return MFSDP_ECAP;
  return MFSDP_OK;
}

int ns_dispatch(Plan& pl, const mfsdp_muon_hparams_t& hp, cudaStream_t st) {
  return hp.precision == MFSDP_NS_BF16 ? launch_ns_tc(pl, hp, st) : launch_ns_fp32(pl, hp, st);
}

}  // namespace
}  // namespace mfsdp

using namespace mfsdp;

extern "C" int mfsdp_workspace_bytes(const mfsdp_desc_t* desc, size_t n_desc, int precision, size_t* bytes) {
  if (!bytes) return MFSDP_EINVAL;
  WsLayout lay;
  const int rc = build_ws_layout(desc, n_desc, precision, lay);
  if (rc) return rc;
  *bytes = lay.total_bytes;
  return MFSDP_OK;
}

extern "C" int mfsdp_workspace_view(const mfsdp_desc_t* desc, size_t n_desc, int precision, int ns_steps,
                                    size_t index, size_t* o_byte_off, size_t* o_pitch, size_t* ssq_byte_off) {
  WsLayout lay;
  const int rc = build_ws_layout(desc, n_desc, precision, lay);
  if (rc) return rc;
  if (index >= lay.mats.size() || ns_steps < 1) return MFSDP_EINVAL;
  if (o_byte_off) *o_byte_off = lay.mats[index].x_off[ns_steps & 1];
  if (o_pitch) *o_pitch = lay.mats[index].pitch_x;
  if (ssq_byte_off) *ssq_byte_off = lay.ssq_off + index * sizeof(double);
  return MFSDP_OK;
}

extern "C" int mfsdp_debug_ws_offsets(const mfsdp_desc_t* desc, size_t n_desc, int precision, size_t index,
                                      size_t out[6]) {
  WsLayout lay;
  const int rc = build_ws_layout(desc, n_desc, precision, lay);
  if (rc) return rc;
  if (index >= lay.mats.size() || !out) return MFSDP_EINVAL;
  const MatLayout& L = lay.mats[index];
  out[0] = L.x_off[0]; out[1] = L.x_off[1]; out[2] = L.a_off; out[3] = L.p_off; out[4] = L.pitch_x; out[5] = L.pitch_a;
  return MFSDP_OK;
}

extern "C" int mfsdp_muon_momentum_pass(const mfsdp_desc_t* desc, size_t n_desc, const void* G, void* M,
                                        void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp,
                                        void* cuda_stream) {
  Plan* pl = nullptr;
  const int rc = muon_front(desc, n_desc, workspace, ws_bytes, hp, &pl);
  if (rc) return rc;
  if (!pl || pl->lay.mats.empty()) return MFSDP_OK;
  if (!G || !M || !aligned(G, 128) || !aligned(M, 128)) return MFSDP_EINVAL;
  return launch_momentum(*pl, G, M, *hp, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int mfsdp_muon_ns_pass(const mfsdp_desc_t* desc, size_t n_desc, void* workspace, size_t ws_bytes,
                                  const mfsdp_muon_hparams_t* hp, void* cuda_stream) {
  Plan* pl = nullptr;
  const int rc = muon_front(desc, n_desc, workspace, ws_bytes, hp, &pl);
  if (rc) return rc;
  if (!pl || pl->lay.mats.empty()) return MFSDP_OK;
  return ns_dispatch(*pl, *hp, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int mfsdp_muon_update_pass(const mfsdp_desc_t* desc, size_t n_desc, void* W, void* workspace,
                                      size_t ws_bytes, const mfsdp_muon_hparams_t* hp, void* cuda_stream) {
  Plan* pl = nullptr;
  const int rc = muon_front(desc, n_desc, workspace, ws_bytes, hp, &pl);
  if (rc) return rc;
  if (!pl || pl->lay.mats.empty()) return MFSDP_OK;
  if (!W || !aligned(W, 128)) return MFSDP_EINVAL;
  return launch_update(*pl, W, *hp, static_cast<cudaStream_t>(cuda_stream));
}

namespace {
int muon_step_impl(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M, void* workspace,
                   size_t ws_bytes, const mfsdp_muon_hparams_t* hp, const uint32_t* ready, uint32_t epoch,
                   void* cuda_stream, void* const* fanout = nullptr);
}  // namespace

extern "C" int mfsdp_muon_step_fanout(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M,
                                      void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp,
                                      void* const* fanout, void* cuda_stream) {
  if (!fanout) return MFSDP_EINVAL;
  return muon_step_impl(desc, n_desc, W, G, M, workspace, ws_bytes, hp, nullptr, 0u, cuda_stream, fanout);
}

extern "C" int mfsdp_muon_step(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M,
                               void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp, void* cuda_stream) {
  return muon_step_impl(desc, n_desc, W, G, M, workspace, ws_bytes, hp, nullptr, 0u, cuda_stream);
}

extern "C" int mfsdp_muon_step_gated(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M,
                                     void* workspace, size_t ws_bytes, const mfsdp_muon_hparams_t* hp,
                                     const uint32_t* ready, uint32_t epoch, void* cuda_stream) {
  if (!ready || (reinterpret_cast<uintptr_t>(ready) & 3)) return MFSDP_EINVAL;
  return muon_step_impl(desc, n_desc, W, G, M, workspace, ws_bytes, hp, ready, epoch, cuda_stream);
}

extern "C" int mfsdp_signal_ready(uint32_t* ready, size_t index, uint32_t epoch, void* cuda_stream) {
  if (!ready || (reinterpret_cast<uintptr_t>(ready) & 3)) return MFSDP_EINVAL;
  typedef CUresult (*WriteFn)(CUstream, CUdeviceptr, cuuint32_t, unsigned int);
  static WriteFn fn = nullptr;
  if (!fn) {
    void* sym = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuStreamWriteValue32", &sym, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess || !sym)
      return cuda_fail(cudaErrorSymbolNotFound);
    fn = reinterpret_cast<WriteFn>(sym);
  }
  const CUresult r = fn(static_cast<CUstream>(cuda_stream), reinterpret_cast<CUdeviceptr>(ready + index), epoch, 0);
  return r == CUDA_SUCCESS ? MFSDP_OK : cuda_fail(cudaErrorUnknown);
}

namespace {
int muon_step_impl(const mfsdp_desc_t* desc, size_t n_desc, void* W, const void* G, void* M, void* workspace,
                   size_t ws_bytes, const mfsdp_muon_hparams_t* hp, const uint32_t* ready, uint32_t epoch,
                   void* cuda_stream, void* const* fanout) {
  Plan* pl = nullptr;
  int rc = muon_front(desc, n_desc, workspace, ws_bytes, hp, &pl);
  if (rc) return rc;
  if (!pl || pl->lay.mats.empty()) return MFSDP_OK;
  if (!W || !G || !M || !aligned(W, 128) || !aligned(G, 128) || !aligned(M, 128)) return MFSDP_EINVAL;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  // Build every launch table of this call BEFORE the first kernel is enqueued: table building allocates and copies
  // synchronously, which must not happen behind a gated momentum kernel that waits for flags the host raises later.
  const bool fuse = hp->precision == MFSDP_NS_BF16 && ns_tc_can_fuse_update(*pl);
  const uint64_t* fan = nullptr;
  if (fanout) {                            // destination table -> device, in stream order (the host array is staged by
    size_t k = 0;                          // the runtime before cudaMemcpyAsync returns: it may be a temporary)
    std::vector<uint64_t> tbl(pl->lay.mats.size());
    for (size_t i = 0; i < n_desc; ++i)
      if (desc[i].role == MFSDP_ROLE_MATRIX) {
        if (fanout[k] && !aligned(fanout[k], 16)) return MFSDP_EINVAL;
        tbl[k] = reinterpret_cast<uint64_t>(fanout[k]); ++k;
      }
    const cudaError_t e = cudaMemcpyAsync(pl->d_fan, tbl.data(), tbl.size() * sizeof(uint64_t), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e);
    fan = pl->d_fan;
  }
  if ((rc = launch_momentum(*pl, G, M, *hp, st, ready, epoch))) return rc;
  if (fuse)                                                             // the update runs in the last APPLY epilogue
    return launch_ns_tc(*pl, *hp, st, W, (hp->flags & MFSDP_STEP_KEEP_O) != 0, fan);
  if ((rc = ns_dispatch(*pl, *hp, st))) return rc;
  return launch_update(*pl, W, *hp, st, fan);
}
}  // namespace

namespace mfsdp {
namespace {
// mfsdp_muon_step_host: the resident set is cut into up to kHostGroups groups of consecutive matrices of about equal
// bytes, and the groups are pipelined over three streams: uploads (G, M, then W of group g) on `in`, the step of group
// g on the caller's stream as soon as its G and M have landed (the weight update, which is the only consumer of W,
// waits for W), downloads (M after the momentum pass, W after the update) on `out`.  PCIe is full duplex, so in steady
// state the upload of group g + 1, the compute of group g and the download of group g - 1 overlap.
constexpr int kHostGroups = 8;
struct HostPipe {
  cudaStream_t in = nullptr, out = nullptr;
  cudaEvent_t start = nullptr, fin = nullptr;
  cudaEvent_t gm_in[kHostGroups], w_in[kHostGroups], mom[kHostGroups], done[kHostGroups];
  int device = -1;
};
std::map<int, HostPipe> g_pipes;         // one per device, created on first use (guarded by g_host_mu)
int host_pipe(HostPipe** out) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(e);
  HostPipe& g_pipe = g_pipes[dev];
  if (g_pipe.device != dev) {
    HostPipe p;
    if ((e = cudaStreamCreateWithFlags(&p.in, cudaStreamNonBlocking)) != cudaSuccess ||
        (e = cudaStreamCreateWithFlags(&p.out, cudaStreamNonBlocking)) != cudaSuccess)
      return cuda_fail(e);
    std::vector<cudaEvent_t*> evs = {&p.start, &p.fin};
    for (int g = 0; g < kHostGroups; ++g) { evs.push_back(&p.gm_in[g]); evs.push_back(&p.w_in[g]); evs.push_back(&p.mom[g]); evs.push_back(&p.done[g]); }
    for (cudaEvent_t* ev : evs)
      if ((e = cudaEventCreateWithFlags(ev, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e);
    p.device = dev;
    g_pipe = p;
  }
  *out = &g_pipe;
  return MFSDP_OK;
}

struct HostGroup {
  std::vector<mfsdp_desc_t> desc;   // the group's matrix descriptors (original element offsets)
  uint64_t e0 = 0, e1 = 0;          // element range [e0, e1) of the rank-flat buffers this group covers
  size_t ws_off = 0, ws_bytes = 0;  // its slice of the workspace
};

// Groups of consecutive matrix descriptors with about equal element counts; *total_ws = workspace they need together.
int host_groups(const mfsdp_desc_t* desc, size_t n_desc, int precision, std::vector<HostGroup>& groups, size_t* total_ws) {
  groups.clear();
  std::vector<const mfsdp_desc_t*> mats;
  uint64_t total = 0;
  for (size_t i = 0; i < n_desc; ++i)
    if (desc[i].role == MFSDP_ROLE_MATRIX) { mats.push_back(&desc[i]); total += (uint64_t)desc[i].rows * desc[i].cols; }
  uint64_t flat = 0;
  int rc = mfsdp_flat_elems(desc, n_desc, &flat, nullptr);
  if (rc) return rc;
  const int want = (int)std::min<size_t>(kHostGroups, mats.size());
  uint64_t acc = 0;
  for (size_t i = 0; i < mats.size(); ++i) {
    if (groups.empty() || (acc * (uint64_t)want >= total * groups.size() && (int)groups.size() < want)) {
      groups.emplace_back();
      groups.back().e0 = mats[i]->elem_off;
    }
    groups.back().desc.push_back(*mats[i]);
    acc += (uint64_t)mats[i]->rows * mats[i]->cols;
  }
  size_t off = 0;
  for (size_t g = 0; g < groups.size(); ++g) {
    groups[g].e1 = g + 1 < groups.size() ? groups[g + 1].e0 : flat;
    WsLayout lay;
    if ((rc = build_ws_layout(groups[g].desc.data(), groups[g].desc.size(), precision, lay))) return rc;
    groups[g].ws_off = off;
    groups[g].ws_bytes = (size_t)align_up_u64(lay.total_bytes, kBufAlign);
    off += groups[g].ws_bytes;
  }
  if (total_ws) *total_ws = off;
  return MFSDP_OK;
}
}  // namespace
}  // namespace mfsdp

extern "C" int mfsdp_host_workspace_bytes(const mfsdp_desc_t* desc, size_t n_desc, int precision, size_t* bytes) {
  if (!bytes || (n_desc && !desc)) return MFSDP_EINVAL;
  std::vector<HostGroup> groups;
  size_t grouped = 0, plain = 0;
  int rc = host_groups(desc, n_desc, precision, groups, &grouped);
  if (rc) return rc;
  if ((rc = mfsdp_workspace_bytes(desc, n_desc, precision, &plain))) return rc;
  *bytes = std::max(grouped, plain);
  return MFSDP_OK;
}

extern "C" int mfsdp_muon_step_host(const mfsdp_desc_t* desc, size_t n_desc, void* hW, const void* hG, void* hM,
                                    void* dW, void* dG, void* dM, int upload_state, void* workspace,
                                    size_t ws_bytes, const mfsdp_muon_hparams_t* hp, void* cuda_stream) {
  Plan* full = nullptr;
  int rc = muon_front(desc, n_desc, workspace, ws_bytes, hp, &full);
  if (rc) return rc;
  if (!full || full->lay.mats.empty()) return MFSDP_OK;
  if (upload_state < 0 || upload_state > 2) return MFSDP_EINVAL;
  if (!hW || !hG || (!hM && upload_state != 2) || !dW || !dG || !dM) return MFSDP_EINVAL;
  if (!aligned(dW, 128) || !aligned(dG, 128) || !aligned(dM, 128)) return MFSDP_EINVAL;
  const size_t es = full->lay.mat_dtype == MFSDP_BF16 ? 2 : 4;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  std::lock_guard<std::mutex> lock(g_host_mu);

  // groups and their plans (launch tables are built here, before anything is enqueued)
  std::vector<HostGroup> groups;
  size_t need = 0;
  if ((rc = host_groups(desc, n_desc, hp->precision, groups, &need))) return rc;
  std::vector<Plan*> plans;
  if (need <= ws_bytes && groups.size() > 1) {
    for (HostGroup& g : groups) {
      Plan* pl = nullptr;
      if ((rc = get_plan(g.desc.data(), g.desc.size(), hp->precision, static_cast<uint8_t*>(workspace) + g.ws_off, true, &pl)))
        return rc;
      plans.push_back(pl);
    }
  } else {                                   // workspace sized for the plain step only: one group, the whole table
    uint64_t flat = 0;
    if ((rc = mfsdp_flat_elems(desc, n_desc, &flat, nullptr))) return rc;
    groups.assign(1, HostGroup());
    groups[0].e0 = 0; groups[0].e1 = flat;
    plans.assign(1, full);
  }
  if (hp->precision == MFSDP_NS_BF16)
    for (Plan* pl : plans) ns_tc_can_fuse_update(*pl);     // builds the tensor-core tables now

  HostPipe* hpipe = nullptr;
  if ((rc = host_pipe(&hpipe))) return rc;
  HostPipe& q = *hpipe;
  cudaError_t e;
  // On any failure the copies already queued may still be reading or writing the caller's host buffers: drain the
  // three streams before returning, so that the caller may free or reuse them.
  auto bail = [&](int code) { cudaStreamSynchronize(q.in); cudaStreamSynchronize(q.out); cudaStreamSynchronize(st); return code; };
#define MFSDP_TRY(call) do { if ((e = (call)) != cudaSuccess) return bail(cuda_fail(e)); } while (0)
  uint8_t *hWb = static_cast<uint8_t*>(hW), *hMb = static_cast<uint8_t*>(hM), *dWb = static_cast<uint8_t*>(dW),
          *dGb = static_cast<uint8_t*>(dG), *dMb = static_cast<uint8_t*>(dM);
  const uint8_t* hGb = static_cast<const uint8_t*>(hG);
  MFSDP_TRY(cudaEventRecord(q.start, st));
  MFSDP_TRY(cudaStreamWaitEvent(q.in, q.start, 0));
  MFSDP_TRY(cudaStreamWaitEvent(q.out, q.start, 0));
  const size_t ng = groups.size();
  for (size_t g = 0; g < ng; ++g) {          // in: G, M of the group (momentum pass), then W (update pass only)
    const uint64_t e0 = groups[g].e0, n = groups[g].e1 - groups[g].e0;
    MFSDP_TRY(cudaMemcpyAsync(dGb + e0 * es, hGb + e0 * es, n * es, cudaMemcpyHostToDevice, q.in));
    if (upload_state == 1) MFSDP_TRY(cudaMemcpyAsync(dMb + e0 * 4, hMb + e0 * 4, n * 4, cudaMemcpyHostToDevice, q.in));
    MFSDP_TRY(cudaEventRecord(q.gm_in[g], q.in));
    if (upload_state == 1) MFSDP_TRY(cudaMemcpyAsync(dWb + e0 * es, hWb + e0 * es, n * es, cudaMemcpyHostToDevice, q.in));
    MFSDP_TRY(cudaEventRecord(q.w_in[g], q.in));
  }
  for (size_t g = 0; g < ng; ++g) {
    const uint64_t e0 = groups[g].e0, n = groups[g].e1 - groups[g].e0;
    Plan& pl = *plans[g];
    // compute on the caller's stream
    MFSDP_TRY(cudaStreamWaitEvent(st, q.gm_in[g], 0));
    if ((rc = launch_momentum(pl, dG, dM, *hp, st))) return bail(rc);
    MFSDP_TRY(cudaEventRecord(q.mom[g], st));
    if ((rc = ns_dispatch(pl, *hp, st))) return bail(rc);
    MFSDP_TRY(cudaStreamWaitEvent(st, q.w_in[g], 0));
    if ((rc = launch_update(pl, dW, *hp, st))) return bail(rc);
    MFSDP_TRY(cudaEventRecord(q.done[g], st));
    // out: M is final after the momentum pass, W after the update
    if (upload_state != 2) {                 // 2: the momentum never leaves the device
      MFSDP_TRY(cudaStreamWaitEvent(q.out, q.mom[g], 0));
      MFSDP_TRY(cudaMemcpyAsync(hMb + e0 * 4, dMb + e0 * 4, n * 4, cudaMemcpyDeviceToHost, q.out));
    }
    MFSDP_TRY(cudaStreamWaitEvent(q.out, q.done[g], 0));
    MFSDP_TRY(cudaMemcpyAsync(hWb + e0 * es, dWb + e0 * es, n * es, cudaMemcpyDeviceToHost, q.out));
  }
  MFSDP_TRY(cudaEventRecord(q.fin, q.out));
  MFSDP_TRY(cudaStreamWaitEvent(st, q.fin, 0));
  MFSDP_TRY(cudaStreamSynchronize(st));
#undef MFSDP_TRY
  return MFSDP_OK;
}

extern "C" int mfsdp_adamw_tail_step(const mfsdp_desc_t* desc, size_t n_desc, void* P, const void* G, void* m,
                                     void* v, const mfsdp_adamw_hparams_t* hp, void* cuda_stream) {
  if (!hp || hp->step < 1 || (n_desc && !desc)) return MFSDP_EINVAL;
  if (!(hp->beta1 >= 0.0 && hp->beta1 < 1.0) || !(hp->beta2 >= 0.0 && hp->beta2 < 1.0) || !(hp->eps >= 0.0))
    return MFSDP_EINVAL;
  Plan* pl = nullptr;
  const int rc = get_plan(desc, n_desc, MFSDP_NS_BF16, nullptr, false, &pl);
  if (rc) return rc;
  if (pl->lay.tails.empty()) return MFSDP_OK;
  if (!P || !G || !m || !v || !aligned(P, 128) || !aligned(G, 128) || !aligned(m, 128) || !aligned(v, 128))
    return MFSDP_EINVAL;
  return launch_adamw(*pl, P, G, m, v, *hp, static_cast<cudaStream_t>(cuda_stream));
}

extern "C" int mfsdp_tune(int knob, int value) {
  if (knob < 0 || knob >= MFSDP_TUNE_COUNT_ || value < 1) return MFSDP_EINVAL;
  std::lock_guard<std::mutex> lock(g_mu);
  if (g_tune[knob].load() == value) return MFSDP_OK;
  g_tune[knob].store(value);
  bool any = false;
  for (Plan* pl : g_plans) any |= pl->tc != nullptr;
  if (any) {
    cudaDeviceSynchronize();           // the tables may be in use by launches still in flight
    for (Plan* pl : g_plans) { destroy_ns_tc(pl->tc); pl->tc = nullptr; }
  }
  return MFSDP_OK;
}

extern "C" int mfsdp_debug_trace(void* dev_buf, size_t bytes) {
  if (dev_buf && (bytes < 56 || (reinterpret_cast<uintptr_t>(dev_buf) & 7))) return MFSDP_EINVAL;
  std::lock_guard<std::mutex> lock(g_mu);
  g_trace = static_cast<unsigned long long*>(dev_buf);
  g_trace_cap = dev_buf ? (uint32_t)std::min<size_t>((bytes - 8) / 48, 0x7fffffffu) : 0;
  return MFSDP_OK;
}

extern "C" int mfsdp_get_tune(int knob) {
  if (knob < 0 || knob >= MFSDP_TUNE_COUNT_) return MFSDP_EINVAL;
  return tune_value(knob);
}

extern "C" int mfsdp_ns_class(uint32_t rows, uint32_t cols) {
  if (rows == 0 || cols == 0) return MFSDP_EINVAL;
  return ns_class(rows, cols);
}

extern "C" int mfsdp_release_plans(void) {
  std::lock_guard<std::mutex> lock(g_mu);
  int dev = 0;
  const bool have_dev = cudaGetDevice(&dev) == cudaSuccess;
  for (Plan* pl : g_plans) {             // launches still in flight may be reading the tables
    if (have_dev && cudaSetDevice(pl->device) == cudaSuccess) cudaDeviceSynchronize();
    free_plan(pl);
  }
  if (have_dev) cudaSetDevice(dev);
  release_shampoo_plans();
  if (have_dev) cudaSetDevice(dev);
  g_plans.clear();
  g_plan_keys.clear();
  return MFSDP_OK;
}

extern "C" const char* mfsdp_strerror(int code) {
  switch (code) {
    case MFSDP_OK: return "ok";
    case MFSDP_EINVAL: return "invalid argument";
    case MFSDP_ECAP: return "capacity too small";
    case MFSDP_ELAYOUT: return "descriptor table violates the one-contiguous-segment layout";
    case MFSDP_EARCH: return "no compute-capability-10.x (sm_100) device; there is no CPU fallback";
    case MFSDP_ECUDA: return g_cuda_err.c_str();
    case MFSDP_ECACHE: return "launch-table cache full (1024 distinct (table, workspace, precision) keys): keep the "
                              "workspace pointer stable, or call mfsdp_release_plans()";
    case MFSDP_ETOOBIG: return "matrix larger than the fixed scratch array of mfsdp_momentum_pass_static "
                               "(mfsdp_static_max_elems() = 2^30 elements); use mfsdp_muon_momentum_pass with a workspace";
    default: return "unknown error code";
  }
}

extern "C" int mfsdp_version(void) { return 2; }
extern "C" uint64_t mfsdp_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }
