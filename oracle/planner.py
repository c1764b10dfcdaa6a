"""Oracle of the balance-aware owner planner (TEST INFRASTRUCTURE -- see oracle/__init__.py).

Follows PAPER.md Algorithm 1 line by line, plain Python ints only:

  1: "Build roles: each 2D matrix is one role; non-2D tensors form one tail role per block."
  2: "ROLEGREEDY: per block, assign largest roles to the currently lightest ranks; carry
      loads forward."
  3: "SCOPEGREEDY: pool all roles, assign largest roles to lightest ranks, then split
      layouts by block."
  5: "Validate one contiguous local segment per parameter; return one MatrixShard layout
      per block."
  (4: COSTAWARE needs workspace caps and a scorer the paper never defines -- out of scope.)

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


def plan(params, world_size, policy=POLICY_ROLE_GREEDY, metric=METRIC_NUMEL, rank=0):
    """Algorithm 1 lines 1-3, 5.  Returns dict(roles, owner, loads, rank, desc)."""
    if world_size < 1:
        raise ValueError("world_size < 1")
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
    if rank < 0:
        rank = min(range(world_size), key=lambda k: (-loads[0][k], k))
    if rank >= world_size:
        raise ValueError("rank out of range")
    desc = emit_desc(roles, owner, rank)
    validate_desc(desc)
    return dict(roles=roles, owner=owner, loads=loads, rank=rank, desc=desc)


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
