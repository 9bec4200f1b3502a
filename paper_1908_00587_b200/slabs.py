"""Slab decomposition of one time step over several GPUs ("a one-dimensional
MPI-only slab decomposition into Fourier modes, which can be treated independently of each other in the computation of
the linear terms ... For computing the non-linear terms, global data transpositions (MPI_Alltoall) ... are employed to
gather all modes locally on each MPI task"; the number of tasks divides N_r).

Host-side plumbing only: which rank owns which Fourier modes in the linear stage (L1-L5) and
which radial levels in the nonlinear stage (N1-N6), and the two exchanges between those layouts, written on
``torch.distributed`` point-to-point batches so that they run over NCCL / NVLink on GPUs and over gloo in the CPU tests.
No arithmetic of the method happens here.

Layouts of one spectral field with n_modes = (M + 1)(2 K + 1) coefficients per radial level:

  mode slab    [N_r, e1 - e0]              all radial levels of the modes e0 .. e1 - 1 of this rank   (linear stage)
  radial slab  [h1 - h0, n_modes]          all modes of the levels h0 .. h1 - 1 = the rank's own levels j0 .. j1 - 1
                                           plus the levels their nine-point radial stencils of N1 reach: four on
                                           either side, all nine next to a wall                        (nonlinear stage)
"""
from __future__ import annotations

import dataclasses


@dataclasses.dataclass(frozen=True)
class SlabPlan:
    N_r: int
    n_modes: int
    world: int
    halo: int = 4

    def __post_init__(self):
        if self.world < 1 or self.N_r % self.world != 0:
            raise ValueError("the number of ranks must divide N_r (PAPER.md:72)")
        if self.n_modes < self.world:
            raise ValueError("fewer Fourier modes than ranks")
        if self.N_r < 2 * self.halo + 1:
            raise ValueError("fewer radial levels than one stencil")

    # ---- ownership
    def levels(self, rank: int) -> tuple[int, int]:
        """Radial levels [j0, j1) whose nonlinear term ``rank`` computes."""
        n = self.N_r // self.world
        return rank * n, (rank + 1) * n

    def levels_with_halo(self, rank: int) -> tuple[int, int]:
        """The levels ``rank`` needs as input of the nonlinear stage: the union of the radial stencils of its own
        levels.  The stencil of level j is the 2 halo + 1 levels starting at clamp(j - halo, 0, N_r - 2 halo - 1): halo
        levels on either side in the interior, one-sided next to a wall -- so a slab of fewer than halo + 1 levels at a
        wall still needs the first (last) 2 halo + 1 levels."""
        j0, j1 = self.levels(rank)
        width = 2 * self.halo + 1
        start = lambda j: min(max(j - self.halo, 0), self.N_r - width)
        return start(j0), start(j1 - 1) + width

    def modes(self, rank: int) -> tuple[int, int]:
        """Fourier modes [e0, e1) (flat index m (2K+1) + k + K) whose sub-step ``rank`` computes; the first
        n_modes % world ranks hold one mode more."""
        q, r = divmod(self.n_modes, self.world)
        e0 = rank * q + min(rank, r)
        return e0, e0 + q + (1 if rank < r else 0)

    def bytes_per_exchange(self, rank: int, n_fields: int, to_radial: bool) -> int:
        """Bytes ``rank`` sends in one exchange of ``n_fields`` complex128 fields (self-copies excluded)."""
        e0, e1 = self.modes(rank)
        j0, j1 = self.levels(rank)
        total = 0
        for peer in range(self.world):
            if peer == rank:
                continue
            if to_radial:
                h0, h1 = self.levels_with_halo(peer)
                total += (h1 - h0) * (e1 - e0)
            else:
                p0, p1 = self.modes(peer)
                total += (j1 - j0) * (p1 - p0)
        return 16 * n_fields * total


def _exchange(sends, recvs, rank, dist, group):
    """sends[p] / recvs[p]: contiguous tensors for peer p (None: nothing); the own block is copied locally."""
    if sends[rank] is not None:
        recvs[rank].copy_(sends[rank])
    if dist is None:
        return
    ops = []
    for p in range(len(sends)):
        if p == rank:
            continue
        if recvs[p] is not None:
            ops.append(dist.P2POp(dist.irecv, recvs[p], p, group))
        if sends[p] is not None:
            ops.append(dist.P2POp(dist.isend, sends[p], p, group))
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


def to_radial_slab(plan: SlabPlan, x_modes, rank: int, dist=None, group=None):
    """Mode slab [N_r, e1 - e0] of every rank  ->  radial slab with halo [h1 - h0, n_modes] on every rank.
    Rank r sends rows h0(p) .. h1(p) of its columns to every peer p (the halo rows go to two ranks)."""
    import torch
    h0, h1 = plan.levels_with_halo(rank)
    out = torch.empty((h1 - h0, plan.n_modes), dtype=x_modes.dtype, device=x_modes.device)
    sends, recvs = [], []
    for p in range(plan.world):
        p0, p1 = plan.levels_with_halo(p)
        sends.append(x_modes[p0:p1].contiguous())
        e0, e1 = plan.modes(p)
        recvs.append(torch.empty((h1 - h0, e1 - e0), dtype=x_modes.dtype, device=x_modes.device))
    _exchange(sends, recvs, rank, dist if plan.world > 1 else None, group)
    for p in range(plan.world):
        e0, e1 = plan.modes(p)
        out[:, e0:e1] = recvs[p]
    return out


def to_mode_slab(plan: SlabPlan, x_radial, rank: int, dist=None, group=None):
    """Own levels [j1 - j0, n_modes] of every rank (no halo)  ->  mode slab [N_r, e1 - e0] on every rank."""
    import torch
    e0, e1 = plan.modes(rank)
    out = torch.empty((plan.N_r, e1 - e0), dtype=x_radial.dtype, device=x_radial.device)
    sends, recvs = [], []
    for p in range(plan.world):
        p0, p1 = plan.modes(p)
        sends.append(x_radial[:, p0:p1].contiguous())
        j0, j1 = plan.levels(p)
        recvs.append(torch.empty((j1 - j0, e1 - e0), dtype=x_radial.dtype, device=x_radial.device))
    _exchange(sends, recvs, rank, dist if plan.world > 1 else None, group)
    for p in range(plan.world):
        j0, j1 = plan.levels(p)
        out[j0:j1] = recvs[p]
    return out


class SlabStepper:
    """One rank of a slab-decomposed time step.  The rank's context has the full size; its window
    (``nsc_set_window``) restricts the nonlinear term to the rank's radial levels and the sub-steps to its Fourier modes,
    and after every quarter of the step (``nsc_step_phase``) the freshly written slabs are exchanged in place inside the
    library's arrays:

        phase 0  N0 = N(u^n)   at the own levels   ->  rows to columns   (N0 of the own modes at every level)
        phase 1  u^1 = substep at the own modes    ->  columns to rows   (u^1 at the own levels + halo, every mode)
        phase 2  N1 = N(u^1)                       ->  rows to columns
        phase 3  u^{n+1} = substep, in place       ->  columns to rows

    The pressure and its radial derivative never leave the mode-slab layout.  The context must enqueue on the stream
    the exchanges run on (``ctx.set_stream(torch.cuda.current_stream())``)."""

    BUFFER_OF_PHASE = (2, 1, 3, 0)          # nsc_field_pointers' `which` written by phase 0..3

    def __init__(self, ctx, plan: SlabPlan, rank: int, dist=None, group=None):
        self.ctx, self.plan, self.rank, self.dist, self.group = ctx, plan, rank, dist, group
        j0, j1 = plan.levels(rank)
        e0, e1 = plan.modes(rank)
        ctx.set_window(j0, j1 - j0, e0, e1 - e0)

    def run_phase(self, phase: int, dt: float):
        self.ctx.step_phase(phase, dt)

    def written(self, phase: int):
        """Views of the arrays phase ``phase`` wrote (state arrays are re-read: their pointers may have been swapped)."""
        return self.ctx.field_tensors(self.BUFFER_OF_PHASE[phase])

    def exchange_after(self, phase: int):
        plan, rank = self.plan, self.rank
        j0, j1 = plan.levels(rank)
        h0, h1 = plan.levels_with_halo(rank)
        e0, e1 = plan.modes(rank)
        for f in self.written(phase):
            if phase in (0, 2):
                f[:, e0:e1] = to_mode_slab(plan, f[j0:j1], rank, self.dist, self.group)
            else:
                f[h0:h1] = to_radial_slab(plan, f[:, e0:e1], rank, self.dist, self.group)

    def step(self, dt: float):
        for phase in range(4):
            self.run_phase(phase, dt)
            self.exchange_after(phase)
