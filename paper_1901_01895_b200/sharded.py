"""Row-sharded RK4IP over several GPUs (sections 4.1-4.3): every rank holds whole rows
of the signal matrix (M / world spatial modes, both polarisations), the linear operator is local, and every evaluation
of the nonlinear operator all-gathers the real mode powers |A_b|^2 — M x N doubles, four times per step (PAPER.md:111,
164).  This module is the multi-GPU PLUMBING only: it sequences the C-ABI stage calls of include/mmf.h
(mmf_shard_begin / powers / apply / linear / end) around torch.distributed's all-gather; every arithmetic step runs in
the library's kernels.  north_star's single-B200 path (binding.Plan.propagate) needs none of this; the sharded path is
for fibres that outgrow one GPU.

The step sequence is written against a small `stages` interface so that the SAME driver runs on the CUDA stage calls
(CudaShardStages, the product) and, in the world_size-2 gloo test on CPU, on a plain stand-in written from the
oracle's definitions (tests/, test infrastructure).
"""
import numpy as np

SH_PLAIN, SH_STAGE2, SH_STAGE3, SH_FINAL = 0, 1, 2, 3


def mode_range(M_total, rank, world):
    """Modes [mode0, mode0 + M_local) of `rank`: equal contiguous shares (the all-gather needs equal shares)."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank / world")
    if M_total % world != 0:
        raise ValueError("M_total = %d is not a multiple of the world size %d" % (M_total, world))
    m = M_total // world
    return rank * m, m


def shard_arguments(beta, kappa, rank, world):
    """The rank's slice of the fibre description: (mode0, M_local, beta[mode0:mode0+M_local], kappa[mode0:..., :])."""
    beta = np.asarray(beta, dtype=np.float64)
    kappa = np.asarray(kappa, dtype=np.float64)
    M_total = kappa.shape[0]
    assert kappa.shape == (M_total, M_total) and beta.shape[0] == M_total
    mode0, m = mode_range(M_total, rank, world)
    return mode0, m, np.ascontiguousarray(beta[mode0:mode0 + m]), np.ascontiguousarray(kappa[mode0:mode0 + m, :])


def all_gather_rows(P_all, mode0, M_local, dist=None):
    """Fill the rows of P_all [M_total][N] the other ranks own: rank r's rows are P_all[r * M_local : (r + 1) * M_local].
    dist = torch.distributed (initialised) or None for a single process.  Works with nccl (CUDA tensors; in place: the
    rank's own rows are already where the collective would put them) and gloo (CPU tensors)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return
    own = P_all[mode0:mode0 + M_local]
    if P_all.is_cuda:
        dist.all_gather_into_tensor(P_all, own)
    else:
        world = dist.get_world_size()
        parts = [P_all[r * M_local:(r + 1) * M_local] for r in range(world)]
        dist.all_gather(parts, own.clone())


class CudaShardStages:
    """The product backend: one shard plan of the CUDA library + the gathered power matrix."""

    def __init__(self, M_total, mode0, N, dt, h, alpha, beta_local, gamma, kappa_rows, device="cuda:0"):
        import torch
        from . import binding
        self.plan = binding.Plan(len(beta_local), N, dt, h, alpha, beta_local, gamma, kappa_rows, device=device,
                                 shard=(M_total, mode0))
        self.M_total, self.mode0, self.M_local, self.N = int(M_total), int(mode0), len(beta_local), int(N)
        self.P_all = torch.empty((self.M_total, self.N), dtype=torch.float64, device=device)

    def begin(self, A):
        self.plan.shard_begin(A)

    def powers(self, stage):
        self.plan.shard_powers(stage, self.P_all)

    def apply(self, stage, gain=1.0):
        self.plan.shard_apply(stage, self.P_all, gain)

    def linear(self, which):
        self.plan.shard_linear(which)

    def end(self):
        self.plan.shard_end()


def propagate(stages, A, nsteps, gather, span=0, gain=1.0):
    """nsteps RK4IP steps (Eq. 6a-6f) of the rank's rows A, in place.
    stages: begin / powers / apply / linear / end (see CudaShardStages); gather(): the all-gather of stages.P_all.
    span > 0: after every span-th step the new field is multiplied by `gain` (lumped amplifier)."""
    if nsteps <= 0:
        return A
    stages.begin(A)
    stages.powers(SH_PLAIN); gather(); stages.apply(SH_PLAIN)          # bracket of (6b): h N(A) A
    for s in range(nsteps):
        stages.linear(0)                                               # (6a) A_I, (6b) k1
        stages.powers(SH_STAGE2); gather(); stages.apply(SH_STAGE2)    # (6c) k2
        stages.powers(SH_STAGE3); gather(); stages.apply(SH_STAGE3)    # (6d) k3 and the brackets of (6e), (6f)
        stages.linear(1)                                               # (6e) argument u4, (6f) first term
        g = gain if (span > 0 and (s + 1) % span == 0) else 1.0
        stages.powers(SH_FINAL); gather(); stages.apply(SH_FINAL, g)   # (6e) + (6f): the new field
        if s + 1 < nsteps:
            stages.powers(SH_PLAIN); gather(); stages.apply(SH_PLAIN)  # the next step's (6b) bracket
    stages.end()
    return A
