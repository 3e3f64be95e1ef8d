"""Host-side logic of the multi-GPU run (bench.py --gpus N under torchrun).

What is measured shards over INDEPENDENT problems only: the six load cases of one image (S: 8(e)); rank r takes load case
(base + r) mod 6 on its own GPU.  There is no data-path collective; the only communication is the barrier and the
max-over-ranks reduction of the device time.

The second half of this file is the index logic of the z-slab decomposition of ONE solve (S: 8(e), 8(f) f5; the paper's
future item "several GPUs ... MPI"): which cell layers a rank owns, which ghost layer it keeps, and which planes it
must receive after every PT iteration.  No GPU path uses it yet (this run has one GPU); tests/test_shard_gloo.py drives it
with two gloo ranks over slabs of the CPU oracle's arrays and reproduces the single-domain iterate bit for bit.
No method arithmetic lives here.
"""
from __future__ import annotations


def load_case_of_rank(rank: int, world: int, base: int = 2) -> int:
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    return (base + rank) % 6 if world > 1 else base % 6


def max_over_ranks(ms: float, dist=None, device="cpu") -> float:
    """device time of the job = slowest rank (all_reduce MAX); dist = torch.distributed or None for one process"""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(voxels_per_rank: int, steps: int, world: int, ms: float) -> float:
    """whole-job voxel-updates/s: all ranks' units over the max-over-ranks time (weak scaling)"""
    return world * voxels_per_rank * steps / (ms * 1e-3)


# ------------------------------------------------------------------------------------------------ z-slab decomposition
# One PT iteration (stress update from the old velocities, then velocity update from the new stresses) on a slab that is
# cut off by an artificial wall one cell layer beyond its owned range leaves exactly these values of the ghost region
# wrong (everything the rank owns, both interface faces included, stays right):
#   v_x, v_y of the ghost cell layer, and v_z, tau_xz, tau_yz on the artificial wall face.
# These five planes per interface are what the neighbour sends after every iteration.

ZSLAB_HALO_FIELDS = (("vx", "layer"), ("vy", "layer"), ("vz", "face"), ("txz", "face"), ("tyz", "face"))


def zslab_bounds(nz: int, world: int, rank: int):
    """owned cell layers [k0, k1) of `rank`: as even as possible, the first nz % world ranks one layer thicker"""
    if not (0 <= rank < world) or nz < 2 * world:
        raise ValueError("need 0 <= rank < world and at least two layers per rank")
    q, r = divmod(nz, world)
    k0 = rank * q + min(rank, r)
    return k0, k0 + q + (1 if rank < r else 0)


def zslab_extent(nz: int, world: int, rank: int, depth: int = 1):
    """cell layers [e0, e1) the rank holds: its own plus `depth` ghost layers towards every neighbour"""
    k0, k1 = zslab_bounds(nz, world, rank)
    if depth < 1 or nz < (depth + 1) * world:
        raise ValueError("need depth >= 1 and more owned layers per rank than ghost layers")
    return (k0 - depth if rank > 0 else k0), (k1 + depth if rank < world - 1 else k1)


def zslab_halo_plan(nz: int, world: int, rank: int):
    """For every neighbour: (peer, send, recv); send / recv are lists of (field, local z index) in ZSLAB_HALO_FIELDS order.
    Local index = global index - e0 (cell layers and faces alike: face k is the lower face of layer k)."""
    k0, k1 = zslab_bounds(nz, world, rank)
    e0, _ = zslab_extent(nz, world, rank)
    plan = []
    if rank > 0:
        # the lower neighbour's ghost layer is my first owned layer k0, its artificial wall my face k0 + 1;
        # my ghost layer is k0 - 1, my artificial wall face k0 - 1
        send = [(f, (k0 if kind == "layer" else k0 + 1) - e0) for f, kind in ZSLAB_HALO_FIELDS]
        recv = [(f, (k0 - 1) - e0) for f, kind in ZSLAB_HALO_FIELDS]
        plan.append((rank - 1, send, recv))
    if rank < world - 1:
        # the upper neighbour's ghost layer is my last owned layer k1 - 1, its artificial wall my face k1 - 1;
        # my ghost layer is k1, my artificial wall face k1 + 1
        send = [(f, (k1 - 1) - e0) for f, kind in ZSLAB_HALO_FIELDS]
        recv = [(f, (k1 if kind == "layer" else k1 + 1) - e0) for f, kind in ZSLAB_HALO_FIELDS]
        plan.append((rank + 1, send, recv))
    return plan


def zslab_exchange(get_plane, set_plane, plan, dist):
    """One halo exchange: get_plane(field, z) -> 2-D tensor, set_plane(field, z, tensor).  Point-to-point, both
    directions posted before either is waited for (dist = torch.distributed)."""
    import torch
    ops, landing = [], []
    for peer, send, recv in plan:
        out = [get_plane(f, z).contiguous() for f, z in send]
        inn = [torch.empty_like(get_plane(f, z)) for f, z in recv]
        ops += [dist.P2POp(dist.isend, t, peer) for t in out] + [dist.P2POp(dist.irecv, t, peer) for t in inn]
        landing.append((recv, inn))
    for w in dist.batch_isend_irecv(ops) if ops else []:
        w.wait()
    for recv, inn in landing:
        for (f, z), t in zip(recv, inn):
            set_plane(f, z, t)


# Deeper ghost zones: one exchange per `depth` PT iterations (depth 2 is what the two-iterations-per-sweep kernel needs).
# After `depth` iterations without exchange the error of the artificial wall has travelled through the whole ghost zone but
# not into the owned range (one iteration moves it by at most one layer: the stress update reads velocities of the same and
# the next layer, the velocity update reads stresses of the same and the previous face).  The plan is therefore the plain
# refresh of the ghost zone: every field of the `depth` ghost cell layers and of the `depth` faces beyond the interface face.

def zslab_refresh_plan(nz: int, world: int, rank: int, depth: int, layer_fields, face_fields):
    """For every neighbour: (peer, send, recv) as in zslab_halo_plan, for an exchange every `depth` iterations.
    layer_fields / face_fields: names of the state arrays that live on cell layers / on z faces."""
    k0, k1 = zslab_bounds(nz, world, rank)
    e0, _ = zslab_extent(nz, world, rank, depth)
    plan = []
    if rank > 0:
        # I own layers k0 .. and faces k0 ..; the lower neighbour's ghost zone is my layers k0 .. k0+depth-1 and my faces
        # k0+1 .. k0+depth; mine is its layers k0-depth .. k0-1 and faces k0-depth .. k0-1
        send = [(f, k0 + d - e0) for d in range(depth) for f in layer_fields] + [(f, k0 + 1 + d - e0) for d in range(depth) for f in face_fields]
        recv = [(f, k0 - depth + d - e0) for d in range(depth) for f in layer_fields] + [(f, k0 - depth + d - e0) for d in range(depth) for f in face_fields]
        plan.append((rank - 1, send, recv))
    if rank < world - 1:
        # the upper neighbour's ghost zone is my layers k1-depth .. k1-1 and my faces k1-depth .. k1-1; mine is its layers
        # k1 .. k1+depth-1 and faces k1+1 .. k1+depth
        send = [(f, k1 - depth + d - e0) for d in range(depth) for f in layer_fields] + [(f, k1 - depth + d - e0) for d in range(depth) for f in face_fields]
        recv = [(f, k1 + d - e0) for d in range(depth) for f in layer_fields] + [(f, k1 + 1 + d - e0) for d in range(depth) for f in face_fields]
        plan.append((rank + 1, send, recv))
    return plan

