"""Multi-GPU decomposition of the site-wise path: every site is
independent (the site loop has no cross-iteration dependence; points
in different SIMD lanes are independent), so the path shards with NO exchange step.  As in Grid,
the process grid splits the lattice first and the vector layout's virtual-node split
happens inside each rank's local lattice: rank r of N owns the slab x3 in [r*L3/N, (r+1)*L3/N)
of the global lattice, which in the site order of S2 (x0 fastest) is one contiguous range of
global sites.  The ONE operation with an exchange step is a shift along x3 (Cshift):
su3_cshift / su3_mul_shift are periodic on the local slab, so `cshift_plan` says which planes
each rank must get from which neighbour (executed by halo.py; shifts along x0..x2 stay local).
Host logic only (no arithmetic of the method, no torch)."""

SLAB_DIM = 3   # the dimension the process grid splits


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


def cshift_plan(l3, rank, world, disp):
    """Exchange plan of z[s] = x[s + disp*e3] on `world` x3 slabs of l3 planes each (global extent G3 = l3*world,
    periodic).  With D = disp reduced to (-G3/2, G3/2], q = trunc(D / l3) whole slabs and r = D - q*l3 planes
    (|r| < l3, sign of D), local plane p of the result is
        x of rank (rank+q) at plane p + r                     where 0 <= p + r < l3      (the bulk, a LOCAL shift by r)
        x of rank (rank+q+sign r) at plane p + r -+ l3        elsewhere                  (the face, |r| planes)
    Returns a dict:
      shift      r, the local (periodic) shift that puts the bulk in place
      bulk_from  rank whose whole slab is the bulk source (== rank: no bulk transfer), bulk_to: who needs mine
      nface      |r| planes in the face (0: none)
      face_from  rank that owns my face, face_to: rank whose face I own
      send_plane0  first of the nface planes of MY slab that face_to needs
      dst_plane0   first of the nface planes of my result the received face fills"""
    l3, rank, world, disp = int(l3), int(rank), int(world), int(disp)
    if l3 <= 0 or world <= 0 or not (0 <= rank < world):
        raise ValueError("bad slab geometry: l3 = %d, rank %d of %d" % (l3, rank, world))
    G3 = l3 * world
    D = disp % G3
    if 2 * D > G3:
        D -= G3
    q = abs(D) // l3 * (1 if D >= 0 else -1)
    r = D - q * l3
    sgn = (r > 0) - (r < 0)
    n = abs(r)
    return {"shift": r, "bulk_from": (rank + q) % world, "bulk_to": (rank - q) % world, "nface": n,
            "face_from": (rank + q + sgn) % world, "face_to": (rank - q - sgn) % world,
            "send_plane0": 0 if r > 0 else l3 - n, "dst_plane0": l3 - n if r > 0 else 0}


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
