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


def all_gather_rows(P, mode0, M_local, dist=None, async_op=False):
    """Fill the rows of the power block P [M_total][n] that the other ranks own: rank r's rows are
    P[r * M_local : (r + 1) * M_local].  dist = torch.distributed (initialised) or None for a single process.  Works with
    nccl (CUDA tensors; in place: the rank's own rows are already where the collective would put them) and gloo (CPU
    tensors).  async_op: return the work handle (its .wait() orders the current stream after the collective)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return None
    own = P[mode0:mode0 + M_local]
    if P.is_cuda:
        w = dist.all_gather_into_tensor(P, own, async_op=async_op)
    else:
        world = dist.get_world_size()
        parts = [P[r * M_local:(r + 1) * M_local] for r in range(world)]
        w = dist.all_gather(parts, own.clone(), async_op=async_op)
    return w if async_op else None


def chunk_ranges(N, chunks):
    """[(t_first, t_count)] of `chunks` equal time chunks (each a multiple of 32 samples)."""
    if chunks < 1 or N % chunks != 0 or (N // chunks) % 32 != 0:
        raise ValueError("N = %d does not split into %d chunks of a multiple of 32 samples" % (N, chunks))
    n = N // chunks
    return [(c * n, n) for c in range(chunks)]


class CudaShardStages:
    """The product backend: one shard plan of the CUDA library + the gathered power blocks, one per time chunk."""

    def __init__(self, M_total, mode0, N, dt, h, alpha, beta_local, gamma, kappa_rows, device="cuda:0", chunks=1):
        import torch
        from . import binding
        self.plan = binding.Plan(len(beta_local), N, dt, h, alpha, beta_local, gamma, kappa_rows, device=device,
                                 shard=(M_total, mode0))
        self.M_total, self.mode0, self.M_local, self.N = int(M_total), int(mode0), len(beta_local), int(N)
        self.ranges = chunk_ranges(self.N, chunks)
        self.P_all = torch.empty((chunks, self.M_total, self.N // chunks), dtype=torch.float64, device=device)

    def begin(self, A):
        self.plan.shard_begin(A)

    def powers(self, stage, c=0):
        t0, n = self.ranges[c]
        self.plan.shard_powers(stage, self.P_all[c], t0, n)

    def apply(self, stage, c=0, gain=1.0):
        t0, n = self.ranges[c]
        self.plan.shard_apply(stage, self.P_all[c], t0, n, gain)

    def linear(self, which):
        self.plan.shard_linear(which)

    def end(self):
        self.plan.shard_end()


def evaluate(stages, stage, gather, gain=1.0):
    """One evaluation of N across the ranks: per time chunk, powers -> all-gather -> apply, software-pipelined: the
    gathers are started as soon as their chunk's powers are enqueued and waited for one by one, so that the collective
    of chunk c + 1 runs while chunk c is being applied.  gather(c) starts the all-gather of
    stages.P_all[c] and returns None (done) or a handle with .wait()."""
    nchunk = len(stages.ranges)
    pending = []
    for c in range(nchunk):
        stages.powers(stage, c)
        pending.append(gather(c))
    for c in range(nchunk):
        if pending[c] is not None:
            pending[c].wait()
        stages.apply(stage, c, gain)


def propagate(stages, A, nsteps, gather, span=0, gain=1.0):
    """nsteps RK4IP steps (Eq. 6a-6f) of the rank's rows A, in place.
    stages: begin / powers / apply / linear / end + ranges, P_all (see CudaShardStages); gather(c): the all-gather of
    chunk c's power block.  span > 0: after every span-th step the new field is multiplied by `gain` (lumped amplifier,
    PAPER.md:255)."""
    if nsteps <= 0:
        return A
    stages.begin(A)
    try:
        evaluate(stages, SH_PLAIN, gather)                 # bracket of (6b): h N(A) A
        for s in range(nsteps):
            stages.linear(0)                               # (6a) A_I, (6b) k1
            evaluate(stages, SH_STAGE2, gather)            # (6c) k2
            evaluate(stages, SH_STAGE3, gather)            # (6d) k3 and the brackets of (6e), (6f)
            stages.linear(1)                               # (6e) argument u4, (6f) first term
            g = gain if (span > 0 and (s + 1) % span == 0) else 1.0
            evaluate(stages, SH_FINAL, gather, g)          # (6e) + (6f): the new field
            if s + 1 < nsteps:
                evaluate(stages, SH_PLAIN, gather)         # the next step's (6b) bracket
    finally:
        stages.end()                                   # also after a failed stage: the plan must not keep A attached
    return A
