"""Cross-rank host glue over torch.distributed (no method arithmetic): the validation step of PAPER.md:85 --
"Cross-rank validation checks that every rank derives the same deterministic schedule and segment sizes before
communication begins, turning mismatches into explicit errors rather than silent NCCL timeouts."

The schedule itself comes from the C library (mfsdp_reduce_schedule); this module only exchanges its 64-bit hash.
Works on any backend (gloo on CPU for the tests, nccl on GPUs)."""
import torch
import torch.distributed as dist

from . import binding as _b


class ScheduleMismatch(RuntimeError):
    """Raised on EVERY rank when the ranks did not derive the same reduction schedule."""

    def __init__(self, hashes):
        self.hashes = hashes
        groups = {}
        for r, h in enumerate(hashes):
            groups.setdefault(h, []).append(r)
        super().__init__("owner-segment reduction schedule differs between ranks: " +
                         "; ".join("ranks %s -> %016x" % (v, k) for k, v in groups.items()))


def validated_reduce_schedule(params, plan_world, owner, reverse_blocks=True, group=None, device="cpu"):
    """Derive the owner-segment gradient-reduction schedule locally, compare its hash across the process group and
    return (ops, hash).  Raises ScheduleMismatch on all ranks if any rank disagrees.  `device`: where the 8-byte
    exchange tensor lives ("cuda" under nccl)."""
    ops, h = _b.mfsdp_reduce_schedule(params, plan_world, owner, reverse_blocks)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        mine = torch.tensor([h - (1 << 64) if h >= (1 << 63) else h], dtype=torch.int64, device=device)
        every = [torch.zeros_like(mine) for _ in range(dist.get_world_size(group))]
        dist.all_gather(every, mine, group=group)
        hashes = [int(t.item()) & 0xFFFFFFFFFFFFFFFF for t in every]
        if any(x != hashes[0] for x in hashes):
            raise ScheduleMismatch(hashes)
    return ops, h


# ---- the exchange steps around the owner-local step, driven by the validated schedule --------------------
# These run the library's schedule records over torch.distributed collectives: on GPUs (backend nccl, one NVSwitch
# domain) dist.reduce / dist.broadcast per role on a communication stream; on CPU (gloo) the same calls, which is how
# the logic is tested.  Nothing here computes anything of the method; the reduction operator is the collective's SUM.

def _flat_of(op, matrix_flat, tail_flat):
    return matrix_flat if op.kind == _b.ROLE_MATRIX else tail_flat


def reduce_gradients_to_owners(ops, rank, full_grads, matrix_G, tail_G, group=None, ready=None, epoch=None,
                               average=False):
    """Owner-segment gradient reduction ("each rank contributes its local full-gradient buffer, but the
    reduced result is written only to the nonempty owner segment").

    ops          the (validated) schedule of mfsdp_reduce_schedule, reverse block order.
    full_grads   callable role -> this rank's full local gradient of that role (a contiguous 1-D tensor of op.numel
                 elements); it is used as the send buffer and, on the owner, also receives the sum.
    matrix_G, tail_G   this rank's rank-flat gradient buffers (the G arguments of mfsdp_muon_step_gated /
                 mfsdp_adamw_tail_step); segments of roles this rank owns are filled at op.owner_elem_off.
    ready, epoch if given (CUDA): after the reduction of an owned MATRIX role has been enqueued, its "gradient landed"
                 flag is raised in stream order (mfsdp_signal_ready on the current stream) -- the gated step may
                 already be waiting for it.
    average      divide the owner's result by the group size (data-parallel mean) before it is stored."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    for op in ops:
        buf = full_grads(op.role)
        if buf.numel() != op.numel:
            raise ValueError("role %d: gradient has %d elements, the schedule says %d" % (op.role, buf.numel(), op.numel))
        if world > 1:
            dist.reduce(buf, dst=op.owner if group is None else dist.get_global_rank(group, op.owner), op=dist.ReduceOp.SUM,
                        group=group)
        if op.owner == rank:
            seg = _flat_of(op, matrix_G, tail_G)[op.owner_elem_off:op.owner_elem_off + op.numel]
            if average and world > 1:
                seg.copy_(buf / world)
            else:
                seg.copy_(buf)
            if ready is not None and op.flag >= 0:
                _b.mfsdp_signal_ready(ready, op.flag, epoch)


def fanout_parameters(ops, rank, matrix_W, tail_P, full_params, group=None):
    """Owner-segment materialisation ("ranks with nonempty segments send only those segments to the ranks
    that need the full parameter ... in the common matrix case this is an owner fanout"), forward block order
    (mfsdp_reduce_schedule(reverse_blocks=False)): the fallback path over dist.broadcast.  The fused path is
    mfsdp_muon_step_fanout, whose update epilogue stores straight into peer-mapped / multicast destinations.

    full_params  callable role -> this rank's full-parameter buffer of that role (1-D, op.numel elements): filled on
                 every rank with the owner's segment."""
    world = dist.get_world_size(group) if dist.is_initialized() else 1
    for op in ops:
        buf = full_params(op.role)
        if op.owner == rank:
            buf.copy_(_flat_of(op, matrix_W, tail_P)[op.owner_elem_off:op.owner_elem_off + op.numel])
        if world > 1:
            dist.broadcast(buf, src=op.owner if group is None else dist.get_global_rank(group, op.owner), group=group)
