"""Host-side logic of the multi-GPU path: REPLICAS ONLY.

north_star fixes one B200 per fibre with no sharding and no inter-GPU collective, so N GPUs run N independent
propagations (here: a launch-power sweep of the same fibre, one power per rank).  The only communication is the
bookkeeping of the timing contract: a barrier on both sides of the timed region and the max-over-ranks of the device
time.  No method arithmetic lives here; the functions work with any torch.distributed backend (nccl on GPUs, gloo in
the CPU tests).
"""
import os


def env_rank_world():
    """(rank, local_rank, world) from the torchrun environment; (0, 0, 1) when launched plainly."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def launch_power_db(rank, world, span_db=2.0):
    """Launch-power offset of replica `rank`: `world` powers spread evenly over [-span/2, +span/2] dB (0 dB alone)."""
    if world <= 1:
        return 0.0
    return -0.5 * span_db + span_db * rank / (world - 1)


def amplitude_scale(rank, world, span_db=2.0):
    """Field-amplitude factor of replica `rank` (power offset in dB -> amplitude)."""
    return 10.0 ** (launch_power_db(rank, world, span_db) / 20.0)


def whole_job(units_local, ms_local, dist=None, device=None):
    """Aggregate of the timing contract: (sum over ranks of the units processed, max over ranks of the device time
    [ms], units per second of the whole job).  dist = torch.distributed (initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(units_local), float(ms_local), float(units_local) / (float(ms_local) * 1e-3)
    import torch
    t_ms = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    t_un = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t_ms, op=dist.ReduceOp.MAX)
    dist.all_reduce(t_un, op=dist.ReduceOp.SUM)
    ms, units = float(t_ms.item()), float(t_un.item())
    return units, ms, units / (ms * 1e-3)
