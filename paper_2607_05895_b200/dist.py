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
