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
