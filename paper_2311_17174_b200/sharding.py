"""Host-side plumbing for more than one GPU.

The path shards by walker -- every walker's orbit, waveform, transform and logL are independent given the shared
read-only data spectrum and PSD -- so there is no data-path collective.  bench.py gives every
rank its own ensemble (weak scaling) and calls every function of this module; torch.distributed is used only for the
barrier and the max-over-ranks of the timing.
"""
import dataclasses


def rank_config(cfg, rank):
    """the ensemble of `rank` in a weak-scaling run: the same recipe, a seed of its own (rank 0 keeps the config's)"""
    return cfg if rank == 0 else dataclasses.replace(cfg, seed=cfg.seed + 7919 * rank)


def max_over_ranks(x, world, device=None):
    if world == 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_step, steps, ms, world):
    """whole-job throughput: units all ranks processed / the slowest rank's time"""
    return world * units_per_rank_step * steps / (ms * 1e-3)
