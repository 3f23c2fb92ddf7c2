"""Multi-GPU host logic: the 2D response R2[k][j] shards over its t1 rows.

The t2 propagations started from different t1 states are independent ("double loop of t1 and
t2"), so rank r takes the rows r, r+W, r+2W, ... of the t1 list, advances its own copy of the t1 trajectory (cheap:
recomputed, not sent) and fills its rows; one all_gather of n1*n2 doubles at the end is the only collective.  A single
propagation does not shard ("replicas only").  Works with any torch.distributed backend
(nccl on GPUs, gloo in the CPU tests); `engine` is anything with response_2d(A, B, C, t1_steps, t2_steps, dt).
"""
import numpy as np


def rows_for_rank(n1, rank, world):
    """Round-robin row indices of rank `rank` out of `world`; ascending, so the t1 sub-list stays sorted."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank/world")
    return list(range(rank, n1, world))


def gather_rows(local_rows, rows, n1, n2, group=None, device="cpu"):
    """All ranks contribute their rows (array [len(rows), n2]); every rank gets the full [n1, n2] matrix."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    per = (n1 + world - 1) // world
    buf = torch.zeros(per * n2, dtype=torch.float64, device=device)
    flat = np.ascontiguousarray(local_rows, dtype=np.float64).reshape(-1)
    buf[: flat.size] = torch.from_numpy(flat).to(device)
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf, group=group)
    R = np.empty((n1, n2))
    for r in range(world):
        idx = rows_for_rank(n1, r, world)
        R[idx, :] = parts[r][: len(idx) * n2].cpu().numpy().reshape(len(idx), n2)
    return R


def response_2d_sharded(engine, A, B, C, t1_steps, t2_steps, dt, group=None, device="cpu"):
    """R2 over the full (t1, t2) grid with the t1 rows split across the ranks of `group`."""
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    t1 = list(t1_steps)
    rows = rows_for_rank(len(t1), rank, world)
    if rows:
        local = engine.response_2d(A, B, C, [t1[i] for i in rows], list(t2_steps), dt)
    else:
        local = np.empty((0, len(t2_steps)))
    return gather_rows(local, rows, len(t1), len(t2_steps), group=group, device=device)


def response_3d_sharded(engine, A, B, C, D, t1_steps, t2_steps, t3_steps, dt, group=None, device="cpu"):
    """R3 (Eq. 17) over the full (t1, t2, t3) grid: the (t2, t3) blocks started from different t1 states are
    independent, so the t1 samples are split across the ranks exactly like the rows of R2 (one all_gather)."""
    import torch.distributed as dist
    rank, world = dist.get_rank(group), dist.get_world_size(group)
    t1 = list(t1_steps)
    n2, n3 = len(t2_steps), len(t3_steps)
    rows = rows_for_rank(len(t1), rank, world)
    if rows:
        local = engine.response_3d(A, B, C, D, [t1[i] for i in rows], list(t2_steps), list(t3_steps), dt)
    else:
        local = np.empty((0, n2, n3))
    return gather_rows(local.reshape(len(rows), n2 * n3), rows, len(t1), n2 * n3, group=group,
                       device=device).reshape(len(t1), n2, n3)


# ---------------------------------------------------------------------------------------------------------------------
# Slab decomposition of ONE propagation along q_1 (row f4).  Rank r owns a contiguous block of q_1 planes
# and keeps HALO = 2 copies of its neighbours' boundary planes on either side (the CENTRAL4 stencil reaches two planes);
# before every RK stage the halo planes of the STAGE INPUT are refreshed from the neighbours (K elements x 2 planes per
# face: 336 MB per face at config 4), everything else is local.  A rank's handle is an ordinary CHFPE handle on the
# local grid [owned planes + halos]: the kernels treat the halo planes as grid points, whatever they compute ON them is
# overwritten by the next exchange, and the physical ends of the q_1 axis keep their zero ghosts (reading R9).
# The exchange here is plain point-to-point (NCCL over NVLink on GPUs, gloo in the CPU test), one batch per stage.
# ---------------------------------------------------------------------------------------------------------------------
HALO = 2


def slab_range(n, rank, world):
    """Owned q_1 planes [lo, hi) of `rank`: contiguous blocks, sizes differing by at most one."""
    if world < 1 or not 0 <= rank < world:
        raise ValueError("bad rank/world")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def slab_config(cfg, rank, world):
    """Parameter dict of rank `rank`'s local grid and its geometry (lo, hi, halo_lo, halo_hi).  Every rank must own at
    least HALO planes (a halo is filled by ONE neighbour) and the local grid needs the library's minimum of 5 points."""
    n = cfg["nq"][0]
    lo, hi = slab_range(n, rank, world)
    if hi - lo < HALO:
        raise ValueError("every rank must own at least %d q_1 planes" % HALO)
    hl = HALO if rank > 0 else 0
    hh = HALO if rank < world - 1 else 0
    h = (cfg["qmax"][0] - cfg["qmin"][0]) / (n - 1)
    loc = dict(cfg)
    loc["nq"] = [hi - lo + hl + hh] + list(cfg["nq"][1:])
    loc["qmin"] = [cfg["qmin"][0] + (lo - hl) * h] + list(cfg["qmin"][1:])
    loc["qmax"] = [cfg["qmin"][0] + (hi + hh - 1) * h] + list(cfg["qmax"][1:])
    if loc["nq"][0] < 5:
        raise ValueError("local grid of rank %d has fewer than 5 q_1 planes" % rank)
    return loc, (lo, hi, hl, hh)


class DistExchange:
    """Halo exchange over torch.distributed point-to-point operations (backend nccl or gloo)."""

    def __init__(self, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)

    def run(self, X, hl, hh):
        """X: [K, n_local, plane] view of the stage input; fills X[:, :hl] and X[:, n-hh:] from the neighbours."""
        dist, n = self.dist, X.shape[1]
        ops, recv = [], []
        if hl:                                           # lower neighbour: gets my first owned planes, fills my lower halo
            sb = X[:, hl:hl + HALO].contiguous()
            rb = X.new_empty((X.shape[0], hl, X.shape[2]))
            ops += [dist.P2POp(dist.isend, sb, self.rank - 1, self.group), dist.P2POp(dist.irecv, rb, self.rank - 1, self.group)]
            recv.append((slice(0, hl), rb))
        if hh:                                           # upper neighbour
            sb = X[:, n - hh - HALO:n - hh].contiguous()
            rb = X.new_empty((X.shape[0], hh, X.shape[2]))
            ops += [dist.P2POp(dist.isend, sb, self.rank + 1, self.group), dist.P2POp(dist.irecv, rb, self.rank + 1, self.group)]
            recv.append((slice(n - hh, n), rb))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for sl, rb in recv:
            X[:, sl] = rb


class SlabPropagator:
    """RK4 propagation of one slab.  `engine` needs stage_input(stage) -> [K, n_local, plane] tensor view of the array
    the stage reads, and rk4_stage(stage, dt) (paper_2509_25840_b200.CHFPE has both); `exchange.run(X, hl, hh)` fills
    the halo planes.  expect() integrates over the owned planes only (halo copies are zeroed first; the next exchange
    restores them) -- the caller sums the partial values over the ranks (expect_sum does it with an all_reduce)."""

    def __init__(self, engine, geometry, exchange):
        self.engine, self.exchange = engine, exchange
        self.lo, self.hi, self.hl, self.hh = geometry

    def step(self, n_steps, dt):
        for _ in range(int(n_steps)):
            for stage in range(4):
                self.exchange.run(self.engine.stage_input(stage), self.hl, self.hh)
                self.engine.rk4_stage(stage, dt)

    def local_slice(self, X_global):
        """The part of a global canonical state [K, nq_1, ...] this rank holds (owned planes + halos)."""
        return X_global[:, self.lo - self.hl:self.hi + self.hh]

    def owned(self, X_local):
        n = X_local.shape[1]
        return X_local[:, self.hl:n - self.hh]

    def expect_partial(self, obs):
        y = self.engine.stage_input(0)
        n = y.shape[1]
        if self.hl:
            y[:, :self.hl] = 0.0
        if self.hh:
            y[:, n - self.hh:] = 0.0
        return float(self.engine.expect(obs)[0])

    def expect_sum(self, obs, group=None, device="cpu"):
        import torch
        import torch.distributed as dist
        t = torch.tensor([self.expect_partial(obs)], dtype=torch.float64, device=device)
        dist.all_reduce(t, group=group)
        return float(t[0])
