"""Oracle of the balance-aware owner planner (TEST INFRASTRUCTURE -- see oracle/__init__.py).

Follows PAPER.md Algorithm 1 line by line, plain Python ints only:

  1: "Build roles: each 2D matrix is one role; non-2D tensors form one tail role per block."
  2: "ROLEGREEDY: per block, assign largest roles to the currently lightest ranks; carry
      loads forward."
  3: "SCOPEGREEDY: pool all roles, assign largest roles to lightest ranks, then split
      layouts by block."
  5: "Validate one contiguous local segment per parameter; return one MatrixShard layout
      per block."
  4: "COSTAWARE: use SCOPEGREEDY only if balance improves within workspace caps; else use
      ROLEGREEDY."  ("COSTAWARE accepts the scope plan only when the balance gain
      does not exceed workspace caps.")  The paper defines neither the caps nor the scorer's
      formulas; reading P5 of DESIGN.md section 4 fixes them (cost_aware / score_plan below).

PAPER.md:65 "The greedy load is owner-resident numel, a proxy for resident parameter/
gradient bytes and Muon work" -> metric NUMEL.  BASELINE.json configs 4/5 "balances
Newton-Schulz flops" -> metric NS_FLOPS with matrix load m^2 (2n + m), m = min, n = max
(dense NS flops / 2K), tails balanced on a separate tail-numel vector (reading P3).
Ties (reading P1): roles sorted by (load desc, block asc, parameter index asc); lightest
rank = min load, ties -> lowest rank id.  "Heaviest" rank (reading P6): max primary load,
ties -> lowest rank id.

A parameter record is a tuple (block_id, ndim, rows, cols, dtype, flags); flags bit0 = skip
(TP-fragmented matrices "are skipped by the matrix-owner planner").
"""

ROLE_MATRIX = 0
ROLE_TAIL = 1
POLICY_ROLE_GREEDY = 0
POLICY_SCOPE_GREEDY = 1
POLICY_COST_AWARE = 2
METRIC_NUMEL = 0
METRIC_NS_FLOPS = 1
PARAM_SKIP = 1
DESC_TRANSPOSED = 1
SEG_ALIGN = 64   # elements; 128 bytes for bf16 storage


def build_roles(params):
    """Algorithm 1 line 1.  Returns roles in model order: dicts with kind, block, index
    (parameter index; a tail's index is that of its first member), rows, cols, numel, dtype, members."""
    roles = []
    tail_of_block = {}
    prev_block = None
    for idx, (block, ndim, rows, cols, dtype, flags) in enumerate(params):
        if prev_block is not None and block < prev_block:
            raise ValueError("block ids must be non-decreasing in model order")
        prev_block = block
        if flags & PARAM_SKIP:
            continue
        if rows <= 0 or cols <= 0:
            raise ValueError("zero-sized parameter")
        if ndim == 2:
            roles.append(dict(kind=ROLE_MATRIX, block=block, index=idx, rows=rows, cols=cols,
                              numel=rows * cols, dtype=dtype, members=[idx]))
        else:
            if block not in tail_of_block:
                tail = dict(kind=ROLE_TAIL, block=block, index=idx, rows=0, cols=1,
                            numel=0, dtype=dtype, members=[])
                tail_of_block[block] = tail
                roles.append(tail)
            tail = tail_of_block[block]
            if dtype != tail["dtype"]:
                raise ValueError("tail members of one block must share a dtype")
            tail["members"].append(idx)
            tail["numel"] += rows * cols
            tail["rows"] = tail["numel"]
    return roles


def role_load(role, metric):
    """(which load vector, load).  Vector 0 is the primary one, vector 1 the tail one (NS_FLOPS only)."""
    if metric == METRIC_NUMEL:
        return 0, role["numel"]
    if role["kind"] == ROLE_MATRIX:
        m = min(role["rows"], role["cols"])
        n = max(role["rows"], role["cols"])
        return 0, m * m * (2 * n + m)
    return 1, role["numel"]


def _greedy(role_ids, roles, metric, loads, owner):
    # "assign largest roles to the currently lightest ranks"
    order = sorted(role_ids, key=lambda r: (-role_load(roles[r], metric)[1], roles[r]["block"], roles[r]["index"]))
    for r in order:
        vec, load = role_load(roles[r], metric)
        lightest = min(range(len(loads[vec])), key=lambda k: (loads[vec][k], k))
        owner[r] = lightest
        loads[vec][lightest] += load


DTYPE_BYTES = {0: 2, 1: 4}     # BF16, F32 storage
DEFAULT_CAPS = dict(owner_num=9, owner_den=8, ws_num=9, ws_den=8, abs_owner_bytes=0, abs_ws_bytes=0)


def score_plan(params, world_size, owner):
    """Resource scorer ("the resource scorer expands a completed plan into per-rank parameter, gradient,
    optimizer-state, communication, and workspace estimates") and the per-block bandwidth model of PAPER.md:77-81.
    Reading P5 (the paper prints no formulas for the scorer), all integers, bytes:
      param[r]  = sum over roles owned by r of numel * sizeof(storage dtype)           (resident parameter shard)
      grad[r]   = param[r]                                                              (gradient of the same roles, same dtype)
      state[r]  = 4 * numel per owned matrix (fp32 Muon momentum, reading M9) + 8 * numel per owned tail (AdamW m, v)
      comm[r]   = sum over blocks B of (W - 1) * O_{B,r}     (bytes r sends per materialisation of all blocks = bytes it
                  receives per gradient reduction; the per-block maximum over r is the paper's C_B^owner)
      ws[r]     = sum over owned matrices of 2 * (2 * rows * cols + 2 * d * d), d = min(rows, cols)
                  (the owner-local step's Newton-Schulz workspace: X ping-pong + A + P in bf16, unpadded)
      blk[r]    = max over blocks of O_{B,r}                 (largest owner segment r must hold unsharded)
    and per block B, P_B = bytes of all its roles, O_{B,r} = bytes of it owned by r:
      gamma_B = max_r O_{B,r} / (P_B / W);  C_B^FSDP = P_B (W-1)/W;  C_B^owner = (W-1) max_r O_{B,r}.
    Returns dict(rank=[dict per rank], block=[dict per block in model order])."""
    roles = build_roles(params)
    if len(owner) != len(roles):
        raise ValueError("owner[] does not match the roles")
    W = world_size
    rank = [dict(param=0, grad=0, state=0, comm=0, ws=0, blk=0) for _ in range(W)]
    blocks = []
    per_block = {}
    for r, role in enumerate(roles):
        o = owner[r]
        if not 0 <= o < W:
            raise ValueError("owner out of range")
        nbytes = role["numel"] * DTYPE_BYTES[role["dtype"]]
        rank[o]["param"] += nbytes
        rank[o]["grad"] += nbytes
        if role["kind"] == ROLE_MATRIX:
            d = min(role["rows"], role["cols"])
            rank[o]["state"] += 4 * role["numel"]
            rank[o]["ws"] += 2 * (2 * role["rows"] * role["cols"] + 2 * d * d)
        else:
            rank[o]["state"] += 8 * role["numel"]
        if role["block"] not in per_block:
            per_block[role["block"]] = [0] * W
            blocks.append(role["block"])
        per_block[role["block"]][o] += nbytes
    out_blocks = []
    for b in blocks:
        O = per_block[b]
        P_B = sum(O)
        mx = max(O)
        for r in range(W):
            rank[r]["comm"] += (W - 1) * O[r]
            rank[r]["blk"] = max(rank[r]["blk"], O[r])
        out_blocks.append(dict(block=b, param=P_B, max_owner=mx, gamma=float(mx * W) / float(P_B),
                               c_fsdp=float(P_B * (W - 1)) / float(W), c_owner=float((W - 1) * mx)))
    return dict(rank=rank, block=out_blocks)


def cost_aware(params, world_size, metric=METRIC_NUMEL, caps=None):
    """Algorithm 1 line 4 under reading P5.  Run ROLE-GREEDY and SCOPE-GREEDY; take the scope plan iff
      (a) balance improves: max primary load (scope) < max primary load (role)  [same total, so max/avg improves], and
      (b) it stays within the workspace caps, both relative to the memory-conservative role plan and absolute:
            max_{B,r} O_{B,r}(scope) * owner_den <= owner_num * max_{B,r} O_{B,r}(role)
            max_r ws[r](scope)       * ws_den    <= ws_num    * max_r ws[r](role)
            max_{B,r} O_{B,r}(scope) <= abs_owner_bytes   (if non-zero),   max_r ws[r](scope) <= abs_ws_bytes (if non-zero);
    else the role plan.  Default caps: 9/8 on both ratios, no absolute cap.
    Returns (policy_used, owner, loads)."""
    caps = dict(DEFAULT_CAPS, **(caps or {}))
    role = _assign(params, world_size, POLICY_ROLE_GREEDY, metric)
    scope = _assign(params, world_size, POLICY_SCOPE_GREEDY, metric)
    take_scope = max(scope[1][0]) < max(role[1][0])
    if take_scope:
        sr = score_plan(params, world_size, role[0])["rank"]
        ss = score_plan(params, world_size, scope[0])["rank"]
        blk_r, blk_s = max(x["blk"] for x in sr), max(x["blk"] for x in ss)
        ws_r, ws_s = max(x["ws"] for x in sr), max(x["ws"] for x in ss)
        take_scope = (blk_s * caps["owner_den"] <= caps["owner_num"] * blk_r and
                      ws_s * caps["ws_den"] <= caps["ws_num"] * ws_r and
                      (caps["abs_owner_bytes"] == 0 or blk_s <= caps["abs_owner_bytes"]) and
                      (caps["abs_ws_bytes"] == 0 or ws_s <= caps["abs_ws_bytes"]))
    if take_scope:
        return POLICY_SCOPE_GREEDY, scope[0], scope[1]
    return POLICY_ROLE_GREEDY, role[0], role[1]


def _assign(params, world_size, policy, metric):
    """Algorithm 1 lines 1-3: (owner[], loads[2][W]) of ROLE- or SCOPE-GREEDY."""
    roles = build_roles(params)
    owner = [-1] * len(roles)
    loads = [[0] * world_size, [0] * world_size]
    if policy == POLICY_ROLE_GREEDY:
        blocks = []
        for r, role in enumerate(roles):
            if not blocks or blocks[-1][0] != role["block"]:
                blocks.append((role["block"], []))
            blocks[-1][1].append(r)
        for _, ids in blocks:                      # "per block ... carry loads forward"
            _greedy(ids, roles, metric, loads, owner)
    elif policy == POLICY_SCOPE_GREEDY:
        _greedy(list(range(len(roles))), roles, metric, loads, owner)   # "pool all roles"
    else:
        raise ValueError("unknown policy")
    return owner, loads


def plan(params, world_size, policy=POLICY_ROLE_GREEDY, metric=METRIC_NUMEL, rank=0, caps=None):
    """Algorithm 1 lines 1-5.  Returns dict(roles, owner, loads, rank, desc, policy_used)."""
    if world_size < 1:
        raise ValueError("world_size < 1")
    roles = build_roles(params)
    owner = [-1] * len(roles)
    loads = [[0] * world_size, [0] * world_size]
    policy_used = policy
    if policy == POLICY_COST_AWARE:
        policy_used, owner, loads = cost_aware(params, world_size, metric, caps)
    elif policy == POLICY_ROLE_GREEDY:
        blocks = []
        for r, role in enumerate(roles):
            if not blocks or blocks[-1][0] != role["block"]:
                blocks.append((role["block"], []))
            blocks[-1][1].append(r)
        for _, ids in blocks:                      # "per block ... carry loads forward"
            _greedy(ids, roles, metric, loads, owner)
    elif policy == POLICY_SCOPE_GREEDY:
        _greedy(list(range(len(roles))), roles, metric, loads, owner)   # "pool all roles"
    else:
        raise ValueError("unknown policy")
    if rank < 0:
        rank = min(range(world_size), key=lambda k: (-loads[0][k], k))
    if rank >= world_size:
        raise ValueError("rank out of range")
    desc = emit_desc(roles, owner, rank)
    validate_desc(desc)
    return dict(roles=roles, owner=owner, loads=loads, rank=rank, desc=desc, policy_used=policy_used)


def _align_up(x, a):
    return (x + a - 1) // a * a


def emit_desc(roles, owner, rank):
    """Descriptor table of one rank, in (block, parameter) order -- the per-block layouts
    concatenated.  Matrices live in one rank-flat element space (W, G, M), tails in another
    (P, G, m, v); every segment starts on a SEG_ALIGN-element boundary; a tail role's
    members are packed back to back in parameter order."""
    desc = []
    off = [0, 0]
    for r, role in enumerate(roles):
        if owner[r] != rank:
            continue
        kind = role["kind"]
        flags = DESC_TRANSPOSED if (kind == ROLE_MATRIX and role["rows"] > role["cols"]) else 0
        desc.append(dict(role=kind, param_id=role["index"], block_id=role["block"],
                         rows=role["rows"], cols=role["cols"], dtype=role["dtype"], flags=flags,
                         elem_off=off[kind]))
        off[kind] = _align_up(off[kind] + role["numel"], SEG_ALIGN)
    return desc


def validate_desc(desc):
    """Algorithm 1 line 5 / PAPER.md:71 as descriptor-table invariants: per element space,
    segments are aligned, in increasing order and non-overlapping (one contiguous local
    segment per resident parameter)."""
    end = [0, 0]
    for d in desc:
        kind = d["role"]
        if kind not in (ROLE_MATRIX, ROLE_TAIL):
            raise ValueError("bad role")
        if d["rows"] <= 0 or d["cols"] <= 0:
            raise ValueError("zero-sized segment")
        if d["elem_off"] % SEG_ALIGN:
            raise ValueError("misaligned segment")
        if d["elem_off"] < end[kind]:
            raise ValueError("overlapping segments")
        end[kind] = d["elem_off"] + d["rows"] * d["cols"]
    return True


def balance(load_vector):
    """max / avg of a per-rank load vector, the ratio PAPER.md:174 and Table 5 report."""
    total = sum(load_vector)
    if total == 0:
        return 1.0
    return max(load_vector) * len(load_vector) / total


# ---- owner-segment gradient reduction schedule ----------------------------------------------------------
# "For gradient reduction, each rank contributes its local full-gradient buffer, but the reduced result is written
# only to the nonempty owner segment.  The fast path uses deterministic native send/recv schedules ...  Cross-rank
# validation checks that every rank derives the same deterministic schedule and segment sizes before communication
# begins, turning mismatches into explicit errors rather than silent NCCL timeouts."
# Reading F1 (the paper prints no schedule): one reduce-to-owner per role, blocks in REVERSE model
# order (backward produces the last block's gradients first), roles of a block in parameter order; every record carries
# the root (owner), the segment size, where the segment lives in the owner's rank-flat gradient buffer (the layout of
# emit_desc) and which of the owner's per-matrix "gradient landed" flags it raises (tails: none).  The validation value
# is the 64-bit FNV-1a hash of the records serialised as little-endian 32/64-bit integers.

FNV_OFFSET = 0xCBF29CE484222325
FNV_PRIME = 0x100000001B3


def fnv1a64(data, h=FNV_OFFSET):
    for byte in data:
        h ^= byte
        h = (h * FNV_PRIME) & 0xFFFFFFFFFFFFFFFF
    return h


def reduce_schedule(params, world_size, owner, reverse_blocks=True):
    """Returns (ops, hash).  op = dict(seq, role, kind, block, param_id, owner, dtype, numel, owner_elem_off, flag)
    where role indexes build_roles(params), owner_elem_off is the element offset of the segment in the owner's
    rank-flat buffer of its kind (matrix space or tail space) and flag is the position of the matrix among the owner's
    matrix descriptors (-1 for tails)."""
    roles = build_roles(params)
    if len(owner) != len(roles):
        raise ValueError("owner[] does not match the roles")
    off = [[0, 0] for _ in range(world_size)]        # running offsets per rank and kind, as emit_desc lays them out
    n_mat = [0] * world_size
    place = []
    for r, role in enumerate(roles):
        o = owner[r]
        if not 0 <= o < world_size:
            raise ValueError("owner out of range")
        kind = role["kind"]
        flag = -1
        if kind == ROLE_MATRIX:
            flag = n_mat[o]
            n_mat[o] += 1
        place.append((off[o][kind], flag))
        off[o][kind] = _align_up(off[o][kind] + role["numel"], SEG_ALIGN)
    blocks = []
    for r, role in enumerate(roles):
        if not blocks or blocks[-1][0] != role["block"]:
            blocks.append((role["block"], []))
        blocks[-1][1].append(r)
    if reverse_blocks:
        blocks = blocks[::-1]
    ops = []
    h = FNV_OFFSET
    for _, ids in blocks:
        for r in ids:
            role = roles[r]
            op = dict(seq=len(ops), role=r, kind=role["kind"], block=role["block"], param_id=role["index"],
                      owner=owner[r], dtype=role["dtype"], numel=role["numel"], owner_elem_off=place[r][0],
                      flag=place[r][1])
            ops.append(op)
            rec = b"".join(int(v & 0xFFFFFFFF).to_bytes(4, "little") for v in
                           (op["seq"], op["role"], op["kind"], op["block"], op["param_id"], op["owner"], op["dtype"],
                            op["flag"]))
            rec += int(op["numel"]).to_bytes(8, "little") + int(op["owner_elem_off"]).to_bytes(8, "little")
            h = fnv1a64(rec, h)
    h = fnv1a64(int(world_size).to_bytes(4, "little") + len(ops).to_bytes(4, "little"), h)
    return ops, h
