"""Template sharding across GPUs (one process per GPU) — host logic only.

The path shards with no exchange step: templates are independent in the filter bank
 and a trigger's sky search reads the SNR series of its own template in
every detector, so each rank keeps whole "template banks" of
``bank_size`` templates (the per-second selection runs per bank of ~10^3
templates), receives the same strain chunk and the same sky tables, and returns its
own trigger / result lists.  The paper's deployment is the same: 412 000 templates on
103 independent nodes of 4000.  No collective is on the data path;
``torch.distributed`` is used for the barrier, the max-over-ranks timing and the
optional merge of the (small) result lists on rank 0.
"""
import numpy as np


def template_shard(rank, world, n_templates, bank_size=1):
    """[t0, t1) of rank ``rank``: contiguous, whole banks of ``bank_size`` templates,
    bank counts differing by at most one between ranks (lower ranks take the extra)."""
    if not (0 <= rank < world) or n_templates < 0 or bank_size < 1:
        raise ValueError("bad shard arguments")
    n_banks = (n_templates + bank_size - 1) // bank_size
    base, extra = divmod(n_banks, world)
    b0 = rank * base + min(rank, extra)
    b1 = b0 + base + (1 if rank < extra else 0)
    return min(b0 * bank_size, n_templates), min(b1 * bank_size, n_templates)


def slice_bank(bank, t0, t1):
    """The sub-bank of templates [t0, t1) of a workloads bank dict (CSR re-based)."""
    off = np.asarray(bank["tmpl_offset"], dtype=np.int64)
    f0, f1 = int(off[t0]), int(off[t1])
    out = dict(bank)
    out["n_templates"] = t1 - t0
    out["tmpl_offset"] = off[t0:t1 + 1] - f0
    for key in ("a", "b", "delay", "band"):
        out[key] = np.asarray(bank[key])[f0:f1]
    return out


def merge_triggers(local, t0, group=None):
    """Gathers every rank's valid trigger records on all ranks (small: <= 40 B per
    (detector, template) per second), with template indices made global by the rank's
    shard offset ``t0``.  ``local`` is a numpy structured array with fields
    ``valid`` and ``tmpl`` (binding.TRIGGER_DTYPE).  Order: rank, then slot."""
    import torch.distributed as dist
    mine = local[local["valid"] == 1].copy()
    mine["tmpl"] += t0
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return mine
    parts = [None] * dist.get_world_size(group)
    dist.all_gather_object(parts, mine, group=group)
    return np.concatenate(parts)


def max_over_ranks(value, device=None, group=None):
    """max of a python float over the ranks (device-timed durations: the slowest rank
    sets the job's time)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sum_over_ranks(value, device=None, group=None):
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device or "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return float(t.item())
