"""Multi-GPU decomposition of the site-wise path: every site is
independent (the site loop has no cross-iteration dependence; points
in different SIMD lanes are independent), so the path shards with NO exchange step.  As in Grid,
the process grid splits the lattice first and the vector layout's virtual-node split
happens inside each rank's local lattice: rank r of N owns the slab x3 in [r*L3/N, (r+1)*L3/N)
of the global lattice, which in the site order of S2 (x0 fastest) is one contiguous range of
global sites.  Host logic only (no arithmetic of the method, no torch)."""


def local_extents(global_L, rank, world):
    """(local L[4], first global site, local volume) of rank's x3 slab."""
    L = tuple(int(v) for v in global_L)
    if not (0 <= rank < world):
        raise ValueError("rank %d outside 0..%d" % (rank, world - 1))
    if L[3] % world:
        raise ValueError("L[3] = %d is not divisible by %d ranks" % (L[3], world))
    l3 = L[3] // world
    vol = L[0] * L[1] * L[2] * l3
    return (L[0], L[1], L[2], l3), rank * vol, vol


def weak_global_extents(local_L, world):
    """Global lattice whose x3 slabs are `world` copies of local_L (weak scaling)."""
    L = tuple(int(v) for v in local_L)
    return (L[0], L[1], L[2], L[3] * world)


def matrix_range(global_L, n_lorentz, rank, world):
    """[m0, m1) of the global logical matrix index m = site*n_lorentz + mu owned by rank."""
    _, s0, vol = local_extents(global_L, rank, world)
    return s0 * n_lorentz, (s0 + vol) * n_lorentz


def job_throughput(local_units, local_ms, dist=None, device=None):
    """Whole-job throughput of independent shards: (sum over ranks of units) / (max over ranks of time).
    `dist` is an initialised torch.distributed module (or None for one process).  Returns
    (units_per_second, max_ms, total_units)."""
    total, worst = float(local_units), float(local_ms)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        import torch
        t = torch.tensor([worst], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        u = torch.tensor([total], dtype=torch.float64, device=device)
        dist.all_reduce(u, op=dist.ReduceOp.SUM)
        worst, total = float(t.item()), float(u.item())
    return total / (worst * 1e-3), worst, total
