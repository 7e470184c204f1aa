"""Host-side logic of the multi-GPU mode: "replicas only".  One Algorithm-2 step is a
sequential chain whose 3D FFTs would need an all-to-all per transform, so several GPUs run INDEPENDENT simulations
(one context per rank, no collective on the data path).  The only exchange is the timing reduction.
Holds none of the method's arithmetic."""


def replica_cfg(cfg, rank):
    """the workload of replica `rank`: same shape, its own seed (so the ranks do not time identical data)"""
    c = dict(cfg)
    c["seed"] = cfg["seed"] + int(rank)
    return c


def max_over_ranks(values, device, world):
    """element-wise MAX of a list of floats over all ranks (time-like metrics: the slowest replica counts)"""
    import torch
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def aggregate_ms_per_step(ms_per_rank_max):
    """weak scaling of a time-like metric: every replica advances one step in the time of the slowest one"""
    return float(ms_per_rank_max)
