// Balance-aware owner planner, host side (no CUDA).
// PAPER.md:101-107 Algorithm 1 lines 1-3 and 5; PAPER.md:65 (greedy load), :71 (contiguity validation),
// :97 (routing by role).  Readings P1-P6 of DESIGN.md section 4 fix what the paper leaves open
// (tie-breaks, NS-flops metric, separate tail load vector, heaviest rank).
#include <algorithm>
#include <cstring>
#include <vector>

#include "mfsdp.h"

namespace {

struct Role {
  uint32_t kind;       // MFSDP_ROLE_*
  uint32_t block;
  uint32_t first;      // parameter index (tail: first member)
  uint32_t rows, cols; // tail: rows = packed numel, cols = 1
  uint32_t dtype;
  uint64_t numel;
};

inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

// Alg. 1 line 1: "each 2D matrix is one role; non-2D tensors form one tail role per block".
int build_roles(const mfsdp_param_t* p, size_t n, std::vector<Role>& roles) {
  roles.clear();
  long tail_slot = -1;           // index in roles[] of the current block's tail role
  bool have_block = false;
  uint32_t cur_block = 0;
  for (size_t i = 0; i < n; ++i) {
    const mfsdp_param_t& q = p[i];
    if (have_block && q.block_id < cur_block) return MFSDP_EINVAL;
    if (!have_block || q.block_id != cur_block) { tail_slot = -1; cur_block = q.block_id; have_block = true; }
    if (q.flags & MFSDP_PARAM_SKIP) continue;
    if (q.rows == 0 || q.cols == 0) return MFSDP_EINVAL;
    if (q.dtype != MFSDP_BF16 && q.dtype != MFSDP_F32) return MFSDP_EINVAL;
    const uint64_t numel = (uint64_t)q.rows * q.cols;
    if (q.ndim == 2) {
      roles.push_back(Role{MFSDP_ROLE_MATRIX, q.block_id, (uint32_t)i, q.rows, q.cols, q.dtype, numel});
    } else {
      if (tail_slot < 0) {
        tail_slot = (long)roles.size();
        roles.push_back(Role{MFSDP_ROLE_TAIL, q.block_id, (uint32_t)i, 0, 1, q.dtype, 0});
      }
      Role& t = roles[(size_t)tail_slot];
      if (t.dtype != q.dtype) return MFSDP_EINVAL;
      t.numel += numel;
      if (t.numel > 0xffffffffull) return MFSDP_EINVAL;
      t.rows = (uint32_t)t.numel;
    }
  }
  return MFSDP_OK;
}

// PAPER.md:65 numel load; BASELINE.json C4/C5 NS-flops load m^2 (2n + m) with tails on their own vector (P3).
inline void role_load(const Role& r, int metric, int& vec, uint64_t& load) {
  if (metric == MFSDP_METRIC_NUMEL) { vec = 0; load = r.numel; return; }
  if (r.kind == MFSDP_ROLE_MATRIX) {
    const uint64_t m = std::min(r.rows, r.cols), n = std::max(r.rows, r.cols);
    vec = 0; load = m * m * (2 * n + m);
  } else { vec = 1; load = r.numel; }
}

// "assign largest roles to the currently lightest ranks" over the role ids in `ids` (P1 tie-breaks).
void greedy(std::vector<uint32_t>& ids, const std::vector<Role>& roles, int metric, int world,
            std::vector<uint64_t>* loads, std::vector<int32_t>& owner) {
  std::vector<uint64_t> key(roles.size());
  for (uint32_t id : ids) { int v; role_load(roles[id], metric, v, key[id]); }
  std::stable_sort(ids.begin(), ids.end(), [&](uint32_t x, uint32_t y) {
    if (key[x] != key[y]) return key[x] > key[y];
    if (roles[x].block != roles[y].block) return roles[x].block < roles[y].block;
    return roles[x].first < roles[y].first;
  });
  for (uint32_t id : ids) {
    int v; uint64_t l; role_load(roles[id], metric, v, l);
    std::vector<uint64_t>& L = loads[v];
    int best = 0;
    for (int r = 1; r < world; ++r) if (L[r] < L[best]) best = r;
    owner[id] = best;
    L[best] += l;
  }
}

}  // namespace

extern "C" int mfsdp_validate_desc(const mfsdp_desc_t* d, size_t n) {
  if (n && !d) return MFSDP_EINVAL;
  uint64_t end[2] = {0, 0};
  for (size_t i = 0; i < n; ++i) {
    const uint32_t k = d[i].role;
    if (k != MFSDP_ROLE_MATRIX && k != MFSDP_ROLE_TAIL) return MFSDP_EINVAL;
    if (d[i].rows == 0 || d[i].cols == 0) return MFSDP_EINVAL;
    if (d[i].dtype != MFSDP_BF16 && d[i].dtype != MFSDP_F32) return MFSDP_EINVAL;
    if (k == MFSDP_ROLE_TAIL && d[i].cols != 1) return MFSDP_EINVAL;
    if (d[i].elem_off % MFSDP_SEG_ALIGN) return MFSDP_ELAYOUT;
    if (d[i].elem_off < end[k]) return MFSDP_ELAYOUT;          // overlapping or out of order
    const bool tall = d[i].rows > d[i].cols;
    if (k == MFSDP_ROLE_MATRIX && tall != ((d[i].flags & MFSDP_DESC_TRANSPOSED) != 0)) return MFSDP_ELAYOUT;
    end[k] = d[i].elem_off + (uint64_t)d[i].rows * d[i].cols;
  }
  return MFSDP_OK;
}

extern "C" int mfsdp_flat_elems(const mfsdp_desc_t* d, size_t n, uint64_t* mat, uint64_t* tail) {
  if (n && !d) return MFSDP_EINVAL;
  uint64_t end[2] = {0, 0};
  for (size_t i = 0; i < n; ++i) {
    if (d[i].role > 1) return MFSDP_EINVAL;
    end[d[i].role] = std::max(end[d[i].role],
                              align_up(d[i].elem_off + (uint64_t)d[i].rows * d[i].cols, MFSDP_SEG_ALIGN));
  }
  if (mat) *mat = end[0];
  if (tail) *tail = end[1];
  return MFSDP_OK;
}

namespace {

// Algorithm 1 lines 2-3: owner[] and the two load vectors of ROLE- or SCOPE-GREEDY.
void assign(const std::vector<Role>& roles, int world, int policy, int metric, std::vector<int32_t>& owner,
            std::vector<uint64_t>* loads) {
  owner.assign(roles.size(), -1);
  loads[0].assign((size_t)world, 0);
  loads[1].assign((size_t)world, 0);
  std::vector<uint32_t> ids;
  if (policy == MFSDP_POLICY_ROLE_GREEDY) {           // line 2: per block, carry loads forward
    size_t i = 0;
    while (i < roles.size()) {
      ids.clear();
      const uint32_t blk = roles[i].block;
      while (i < roles.size() && roles[i].block == blk) ids.push_back((uint32_t)i++);
      greedy(ids, roles, metric, world, loads, owner);
    }
  } else {                                            // line 3: pool all roles
    ids.resize(roles.size());
    for (size_t i = 0; i < roles.size(); ++i) ids[i] = (uint32_t)i;
    greedy(ids, roles, metric, world, loads, owner);
  }
}

inline uint64_t dtype_bytes(uint32_t dtype) { return dtype == MFSDP_BF16 ? 2 : 4; }

// Resource scorer (reading P5): per-rank and per-block records of a completed plan.
void score(const std::vector<Role>& roles, const std::vector<int32_t>& owner, int world,
           std::vector<mfsdp_rank_score_t>& rank, std::vector<mfsdp_block_score_t>& blocks) {
  mfsdp_rank_score_t zero;
  std::memset(&zero, 0, sizeof zero);
  rank.assign((size_t)world, zero);
  blocks.clear();
  std::vector<uint64_t> O((size_t)world);
  size_t i = 0;
  while (i < roles.size()) {                          // roles are in model order: one run per block
    const uint32_t blk = roles[i].block;
    std::fill(O.begin(), O.end(), 0);
    for (; i < roles.size() && roles[i].block == blk; ++i) {
      const Role& r = roles[i];
      const size_t o = (size_t)owner[i];
      const uint64_t nbytes = r.numel * dtype_bytes(r.dtype);
      rank[o].param_bytes += nbytes;
      rank[o].grad_bytes += nbytes;
      if (r.kind == MFSDP_ROLE_MATRIX) {
        const uint64_t d = std::min(r.rows, r.cols);
        rank[o].state_bytes += 4 * r.numel;
        rank[o].workspace_bytes += 2 * (2 * (uint64_t)r.rows * r.cols + 2 * d * d);
      } else {
        rank[o].state_bytes += 8 * r.numel;
      }
      O[o] += nbytes;
    }
    uint64_t P = 0, mx = 0;
    for (int r = 0; r < world; ++r) {
      P += O[(size_t)r];
      mx = std::max(mx, O[(size_t)r]);
      rank[(size_t)r].comm_bytes += (uint64_t)(world - 1) * O[(size_t)r];
      rank[(size_t)r].max_block_owner_bytes = std::max(rank[(size_t)r].max_block_owner_bytes, O[(size_t)r]);
    }
    mfsdp_block_score_t b;
    std::memset(&b, 0, sizeof b);
    b.block_id = blk; b.param_bytes = P; b.max_owner_bytes = mx;
    b.gamma = (double)(mx * (uint64_t)world) / (double)P;
    b.c_fsdp = (double)(P * (uint64_t)(world - 1)) / (double)world;
    b.c_owner = (double)((uint64_t)(world - 1) * mx);
    blocks.push_back(b);
  }
}

}  // namespace

extern "C" int mfsdp_score_plan(const mfsdp_param_t* params, size_t n_params, int world, const int32_t* owner,
                                size_t n_roles, mfsdp_rank_score_t* rank_out, mfsdp_block_score_t* block_out,
                                size_t block_cap, size_t* n_blocks) {
  if ((n_params && !params) || world < 1 || (n_roles && !owner)) return MFSDP_EINVAL;
  std::vector<Role> roles;
  const int rc = build_roles(params, n_params, roles);
  if (rc) return rc;
  if (roles.size() != n_roles) return MFSDP_EINVAL;
  std::vector<int32_t> own(owner, owner + n_roles);
  for (int32_t o : own) if (o < 0 || o >= world) return MFSDP_EINVAL;
  std::vector<mfsdp_rank_score_t> rank;
  std::vector<mfsdp_block_score_t> blocks;
  score(roles, own, world, rank, blocks);
  if (n_blocks) *n_blocks = blocks.size();
  if (rank_out) std::memcpy(rank_out, rank.data(), rank.size() * sizeof(mfsdp_rank_score_t));
  if (block_out) {
    if (block_cap < blocks.size()) return MFSDP_ECAP;
    if (!blocks.empty()) std::memcpy(block_out, blocks.data(), blocks.size() * sizeof(mfsdp_block_score_t));
  }
  return MFSDP_OK;
}

namespace {
inline void fnv_bytes(uint64_t& h, const void* p, size_t n) {
  const unsigned char* b = static_cast<const unsigned char*>(p);
  for (size_t i = 0; i < n; ++i) { h ^= b[i]; h *= 0x100000001B3ull; }
}
inline void fnv_u32(uint64_t& h, uint32_t v) { unsigned char b[4] = {(unsigned char)v, (unsigned char)(v >> 8), (unsigned char)(v >> 16), (unsigned char)(v >> 24)}; fnv_bytes(h, b, 4); }
inline void fnv_u64(uint64_t& h, uint64_t v) { fnv_u32(h, (uint32_t)v); fnv_u32(h, (uint32_t)(v >> 32)); }
}  // namespace

extern "C" int mfsdp_reduce_schedule(const mfsdp_param_t* params, size_t n_params, int world, const int32_t* owner,
                                     size_t n_roles, int reverse_blocks, mfsdp_reduce_op_t* ops_out, size_t ops_cap,
                                     size_t* n_ops, uint64_t* hash_out) {
  if ((n_params && !params) || world < 1 || (n_roles && !owner)) return MFSDP_EINVAL;
  std::vector<Role> roles;
  const int rc = build_roles(params, n_params, roles);
  if (rc) return rc;
  if (roles.size() != n_roles) return MFSDP_EINVAL;
  for (size_t i = 0; i < n_roles; ++i) if (owner[i] < 0 || owner[i] >= world) return MFSDP_EINVAL;
  // where each role's segment lives on its owner (the layout mfsdp_plan emits) and which landed-flag it raises
  std::vector<uint64_t> off((size_t)world * 2, 0), place(roles.size());
  std::vector<int32_t> n_mat((size_t)world, 0), flag(roles.size(), -1);
  for (size_t i = 0; i < roles.size(); ++i) {
    const size_t o = (size_t)owner[i];
    if (roles[i].kind == MFSDP_ROLE_MATRIX) flag[i] = n_mat[o]++;
    uint64_t& f = off[o * 2 + roles[i].kind];
    place[i] = f;
    f = align_up(f + roles[i].numel, MFSDP_SEG_ALIGN);
  }
  std::vector<std::pair<size_t, size_t>> blocks;      // [begin, end) role runs per block, model order
  for (size_t i = 0; i < roles.size();) {
    size_t j = i;
    while (j < roles.size() && roles[j].block == roles[i].block) ++j;
    blocks.push_back({i, j});
    i = j;
  }
  if (reverse_blocks) std::reverse(blocks.begin(), blocks.end());
  std::vector<mfsdp_reduce_op_t> ops;
  uint64_t h = 0xCBF29CE484222325ull;
  for (const auto& b : blocks)
    for (size_t i = b.first; i < b.second; ++i) {
      mfsdp_reduce_op_t op;
      std::memset(&op, 0, sizeof op);
      op.seq = (uint32_t)ops.size(); op.role = (uint32_t)i; op.kind = roles[i].kind; op.block_id = roles[i].block;
      op.param_id = roles[i].first; op.owner = (uint32_t)owner[i]; op.dtype = roles[i].dtype; op.flag = flag[i];
      op.numel = roles[i].numel; op.owner_elem_off = place[i];
      ops.push_back(op);
      fnv_u32(h, op.seq); fnv_u32(h, op.role); fnv_u32(h, op.kind); fnv_u32(h, op.block_id); fnv_u32(h, op.param_id);
      fnv_u32(h, op.owner); fnv_u32(h, op.dtype); fnv_u32(h, (uint32_t)op.flag);
      fnv_u64(h, op.numel); fnv_u64(h, op.owner_elem_off);
    }
  fnv_u32(h, (uint32_t)world);
  fnv_u32(h, (uint32_t)ops.size());
  if (n_ops) *n_ops = ops.size();
  if (hash_out) *hash_out = h;
  if (ops_out) {
    if (ops_cap < ops.size()) return MFSDP_ECAP;
    if (!ops.empty()) std::memcpy(ops_out, ops.data(), ops.size() * sizeof(mfsdp_reduce_op_t));
  }
  return MFSDP_OK;
}

extern "C" int mfsdp_plan_ex(const mfsdp_param_t* params, size_t n_params, int world, int policy, int metric, int rank,
                             const mfsdp_caps_t* caps, int32_t* owner_out, size_t* n_roles, uint64_t* rank_load_out,
                             mfsdp_desc_t* desc_out, size_t desc_cap, size_t* n_desc, int* rank_out, int* policy_used) {
  if ((n_params && !params) || world < 1 || rank >= world || !n_desc) return MFSDP_EINVAL;
  if (policy != MFSDP_POLICY_ROLE_GREEDY && policy != MFSDP_POLICY_SCOPE_GREEDY && policy != MFSDP_POLICY_COST_AWARE)
    return MFSDP_EINVAL;
  if (metric != MFSDP_METRIC_NUMEL && metric != MFSDP_METRIC_NS_FLOPS) return MFSDP_EINVAL;
  mfsdp_caps_t cp = {9, 8, 9, 8, 0, 0};
  if (caps) cp = *caps;
  if (policy == MFSDP_POLICY_COST_AWARE && (cp.owner_den == 0 || cp.ws_den == 0)) return MFSDP_EINVAL;

  std::vector<Role> roles;
  int rc = build_roles(params, n_params, roles);
  if (rc) return rc;

  std::vector<int32_t> owner;
  std::vector<uint64_t> loads[2];
  int used = policy;
  if (policy == MFSDP_POLICY_COST_AWARE) {            // line 4: scope only if balance improves within the caps
    std::vector<int32_t> owner_s;
    std::vector<uint64_t> loads_s[2];
    assign(roles, world, MFSDP_POLICY_ROLE_GREEDY, metric, owner, loads);
    assign(roles, world, MFSDP_POLICY_SCOPE_GREEDY, metric, owner_s, loads_s);
    auto vmax = [](const std::vector<uint64_t>& v) { uint64_t m = 0; for (uint64_t x : v) m = std::max(m, x); return m; };
    bool take = vmax(loads_s[0]) < vmax(loads[0]);
    if (take) {
      std::vector<mfsdp_rank_score_t> sr, ss;
      std::vector<mfsdp_block_score_t> tmp;
      score(roles, owner, world, sr, tmp);
      score(roles, owner_s, world, ss, tmp);
      uint64_t blk_r = 0, blk_s = 0, ws_r = 0, ws_s = 0;
      for (int r = 0; r < world; ++r) {
        blk_r = std::max(blk_r, sr[(size_t)r].max_block_owner_bytes); blk_s = std::max(blk_s, ss[(size_t)r].max_block_owner_bytes);
        ws_r = std::max(ws_r, sr[(size_t)r].workspace_bytes); ws_s = std::max(ws_s, ss[(size_t)r].workspace_bytes);
      }
      typedef unsigned __int128 u128;                 // bytes * small integers: no overflow worries
      take = (u128)blk_s * cp.owner_den <= (u128)cp.owner_num * blk_r && (u128)ws_s * cp.ws_den <= (u128)cp.ws_num * ws_r &&
             (cp.abs_owner_bytes == 0 || blk_s <= cp.abs_owner_bytes) && (cp.abs_ws_bytes == 0 || ws_s <= cp.abs_ws_bytes);
    }
    used = take ? MFSDP_POLICY_SCOPE_GREEDY : MFSDP_POLICY_ROLE_GREEDY;
    if (take) { owner.swap(owner_s); loads[0].swap(loads_s[0]); loads[1].swap(loads_s[1]); }
  } else {
    assign(roles, world, policy, metric, owner, loads);
  }

  if (rank < 0) {                                     // P6: heaviest by primary load, ties -> lowest id
    rank = 0;
    for (int r = 1; r < world; ++r) if (loads[0][r] > loads[0][rank]) rank = r;
  }

  // Emit the chosen rank's layout in (block, parameter) order = role order (line 5).
  std::vector<mfsdp_desc_t> out;
  uint64_t off[2] = {0, 0};
  for (size_t i = 0; i < roles.size(); ++i) {
    if (owner[i] != rank) continue;
    const Role& r = roles[i];
    mfsdp_desc_t d;
    std::memset(&d, 0, sizeof d);
    d.role = r.kind; d.param_id = r.first; d.block_id = r.block; d.rows = r.rows; d.cols = r.cols;
    d.dtype = r.dtype;
    d.flags = (r.kind == MFSDP_ROLE_MATRIX && r.rows > r.cols) ? MFSDP_DESC_TRANSPOSED : 0u;
    d.elem_off = off[r.kind];
    off[r.kind] = align_up(off[r.kind] + r.numel, MFSDP_SEG_ALIGN);
    out.push_back(d);
  }
  rc = mfsdp_validate_desc(out.data(), out.size());
  if (rc) return MFSDP_ELAYOUT;

  if (n_roles) *n_roles = roles.size();
  if (rank_out) *rank_out = rank;
  if (policy_used) *policy_used = used;
  if (owner_out) for (size_t i = 0; i < roles.size(); ++i) owner_out[i] = owner[i];
  if (rank_load_out)
    for (int r = 0; r < world; ++r) { rank_load_out[r] = loads[0][r]; rank_load_out[world + r] = loads[1][r]; }
  *n_desc = out.size();
  if (desc_out) {
    if (desc_cap < out.size()) return MFSDP_ECAP;
    if (!out.empty()) std::memcpy(desc_out, out.data(), out.size() * sizeof(mfsdp_desc_t));
  }
  return MFSDP_OK;
}

extern "C" int mfsdp_plan(const mfsdp_param_t* params, size_t n_params, int world, int policy, int metric,
                          int rank, int32_t* owner_out, size_t* n_roles, uint64_t* rank_load_out,
                          mfsdp_desc_t* desc_out, size_t desc_cap, size_t* n_desc, int* rank_out) {
  return mfsdp_plan_ex(params, n_params, world, policy, metric, rank, nullptr, owner_out, n_roles, rank_load_out,
                       desc_out, desc_cap, n_desc, rank_out, nullptr);
}
