"""Host-side logic of INTRA-configuration sharding: one lattice split into t-slabs
over the ranks of a `torch.distributed` group, as the paper's CPU code splits its lattice over MPI ranks with PFFT
(PAPER.md:45).  No configuration of BASELINE.json needs it (64^4 fp64 is 9.7 GB of 180 GB) and `gpurun` offers one GPU,
so this module holds what can be built and tested without a second GPU: the partition, the halo and all-to-all PLANS
(who sends which index range to whom), the byte budget over NVLink, and backend-agnostic exchange routines over
`torch.distributed` (gloo on CPU in tests/test_slabs_gloo.py; the same calls run on NCCL with device tensors).
It contains none of the method's arithmetic: no Delta, no FFT, no g.

Layout of a field shard: a rank owns the t-slices [t0, t1) of every field, stored [t, z, y, x, ...] (x fastest within a
site index, as everywhere else).  Per iteration the path needs

  halo-   K1 reads U_t(x - t^): the rank's first slice needs the t-links of slice t0 - 1 (from the rank below);
  halo+   K5 reads g(x + t^): the rank's last slice needs Delta~ (8 reals per site) of slice t1 (from the rank above);
  a2a     the t lines of the FFT cross all ranks: after the x, y, z transforms every rank re-partitions its
          [t-slab, all z] block into [all t, z-slab] (one all-to-all), transforms and scales along t, and goes back
          (a second all-to-all) -- K3's tile is a whole (z,t) plane, so on the GPU this brackets K3's t stages.
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Sequence, Tuple


def split_extent(n: int, world: int) -> List[Tuple[int, int]]:
    """[start, stop) of each rank's contiguous share of an extent of n points (sizes differ by at most one; needs n >= world)."""
    if world < 1 or n < world:
        raise ValueError("split_extent: need 1 <= world <= n")
    base, rem = divmod(n, world)
    out, s = [], 0
    for r in range(world):
        e = s + base + (1 if r < rem else 0)
        out.append((s, e))
        s = e
    return out


@dataclass(frozen=True)
class SlabPlan:
    """Everything rank `rank` of `world` needs to know about its share of an Lx*Ly*Lz*Lt lattice."""
    L: Tuple[int, int, int, int]
    world: int
    rank: int
    t_ranges: Tuple[Tuple[int, int], ...]     # per rank: t-slab [t0, t1)
    z_ranges: Tuple[Tuple[int, int], ...]     # per rank: z-slab [z0, z1) held between the two all-to-alls

    @property
    def t0(self) -> int:
        return self.t_ranges[self.rank][0]

    @property
    def t1(self) -> int:
        return self.t_ranges[self.rank][1]

    @property
    def nt(self) -> int:
        return self.t1 - self.t0

    @property
    def z0(self) -> int:
        return self.z_ranges[self.rank][0]

    @property
    def z1(self) -> int:
        return self.z_ranges[self.rank][1]

    @property
    def below(self) -> int:
        """Rank that owns slice t0 - 1 (periodic)."""
        return (self.rank - 1) % self.world

    @property
    def above(self) -> int:
        """Rank that owns slice t1 (periodic)."""
        return (self.rank + 1) % self.world

    @property
    def slice_sites(self) -> int:
        return self.L[0] * self.L[1] * self.L[2]

    def a2a_send_counts(self) -> List[int]:
        """t -> z all-to-all: sites this rank sends to each peer (its t-slices x the peer's z-slab x the (x,y) plane)."""
        lxy = self.L[0] * self.L[1]
        return [self.nt * (z1 - z0) * lxy for (z0, z1) in self.z_ranges]

    def a2a_recv_counts(self) -> List[int]:
        """t -> z all-to-all: sites received from each peer (the peer's t-slices x this rank's z-slab)."""
        lxy = self.L[0] * self.L[1]
        return [(t1 - t0) * (self.z1 - self.z0) * lxy for (t0, t1) in self.t_ranges]


def make_plan(L: Sequence[int], world: int, rank: int) -> SlabPlan:
    L = tuple(int(v) for v in L)
    if len(L) != 4 or not (0 <= rank < world):
        raise ValueError("make_plan: need four extents and 0 <= rank < world")
    return SlabPlan(L, world, rank, tuple(split_extent(L[3], world)), tuple(split_extent(L[2], world)))


def bytes_per_iteration(L: Sequence[int], world: int, precision_bytes: int, storage: int) -> dict:
    """What one iteration moves over the interconnect PER RANK (bytes sent; as much is received), for the largest
    slab: two one-slice halos and two all-to-alls of the packed Delta field (8 reals per site).
    With P ranks a rank keeps 1/P of its block in each all-to-all."""
    plan = make_plan(L, world, 0)
    w = int(precision_bytes)
    halo_links = plan.slice_sites * storage * w                 # U_t of one slice (n_l reals per link)
    halo_delta = plan.slice_sites * 8 * w                       # packed Delta~ of one slice
    block = plan.nt * plan.slice_sites * 8 * w                  # the rank's whole packed Delta block
    a2a = block - block // world if world > 1 else 0            # the part that leaves the rank, per all-to-all
    total = (halo_links + halo_delta + 2 * a2a) if world > 1 else 0
    return {"halo_links": halo_links if world > 1 else 0, "halo_delta": halo_delta if world > 1 else 0,
            "all_to_all_each": a2a, "all_to_alls": 2 if world > 1 else 0, "total_sent": total}


def nvlink_budget(L: Sequence[int], world: int, precision_bytes: int, storage: int, link_GBps: float = 770.0,
                  hbm_GBps: float = 6533.0) -> dict:
    """Time of the exchanges against the rank's HBM time for its share of the iteration (algorithmic bytes
    (12 n_l + 64) w per site); link_GBps: measured peer copy per direction (B200_PROFILING.md)."""
    b = bytes_per_iteration(L, world, precision_bytes, storage)
    V = L[0] * L[1] * L[2] * L[3]
    sites = V // world + (1 if V % world else 0)
    hbm_s = sites * (12 * storage + 64) * precision_bytes / (hbm_GBps * 1e9)
    link_s = b["total_sent"] / (link_GBps * 1e9)
    return {"bytes_sent_per_rank": b["total_sent"], "link_seconds": link_s, "hbm_seconds": hbm_s,
            "link_over_hbm": link_s / hbm_s if hbm_s > 0 else 0.0}


# ---------------------------------------------------------------------------------------------------------------------
# exchanges over torch.distributed (tensors on CPU with gloo, on the device with NCCL)
# ---------------------------------------------------------------------------------------------------------------------
def _exchange(send, dst: int, src: int, group=None):
    """Send `send` to rank dst and receive a tensor of the same shape from rank src (deadlock-free pairing)."""
    import torch
    import torch.distributed as dist
    recv = torch.empty_like(send)
    if dist.get_world_size(group) == 1:
        recv.copy_(send)
        return recv
    reqs = [dist.isend(send.contiguous(), dst, group=group), dist.irecv(recv, src, group=group)]
    for r in reqs:
        r.wait()
    return recv


def halo_from_below(plan: SlabPlan, last_slice, group=None):
    """Every rank passes its LAST t-slice (any per-site payload, shape [z, y, x, ...]) to the rank above and gets the
    slice t0 - 1 from the rank below: the backward t-neighbours of its first slice (K1's halo)."""
    return _exchange(last_slice, plan.above, plan.below, group)


def halo_from_above(plan: SlabPlan, first_slice, group=None):
    """Every rank passes its FIRST t-slice to the rank below and gets slice t1 from the rank above: the forward
    t-neighbours of its last slice (K5's halo)."""
    return _exchange(first_slice, plan.below, plan.above, group)


def transpose_t_to_z(plan: SlabPlan, block, group=None):
    """[nt_local, Lz, Ly, Lx, ...] (this rank's t-slab, all z) -> [Lt, nz_local, Ly, Lx, ...] (all t, this rank's z-slab)."""
    import torch
    import torch.distributed as dist
    if plan.world == 1:
        return block.clone()
    sends = [block[:, z0:z1].contiguous() for (z0, z1) in plan.z_ranges]
    recvs = [torch.empty((t1 - t0, plan.z1 - plan.z0) + tuple(block.shape[2:]), dtype=block.dtype, device=block.device)
             for (t0, t1) in plan.t_ranges]
    _all_to_all(recvs, sends, plan, group)
    return torch.cat(recvs, dim=0)


def transpose_z_to_t(plan: SlabPlan, block, group=None):
    """Inverse of transpose_t_to_z: [Lt, nz_local, ...] -> [nt_local, Lz, ...]."""
    import torch
    if plan.world == 1:
        return block.clone()
    sends = [block[t0:t1].contiguous() for (t0, t1) in plan.t_ranges]
    recvs = [torch.empty((plan.nt, z1 - z0) + tuple(block.shape[2:]), dtype=block.dtype, device=block.device)
             for (z0, z1) in plan.z_ranges]
    _all_to_all(recvs, sends, plan, group)
    return torch.cat(recvs, dim=1)


def _all_to_all(recvs, sends, plan: SlabPlan, group=None):
    """dist.all_to_all where the backend has it (NCCL); pairwise isend/irecv otherwise (gloo)."""
    import torch.distributed as dist
    if dist.get_backend(group) == "nccl":
        dist.all_to_all(recvs, sends, group=group)
        return
    recvs[plan.rank].copy_(sends[plan.rank])
    reqs = []
    for peer in range(plan.world):
        if peer == plan.rank:
            continue
        reqs.append(dist.isend(sends[peer], peer, group=group))
        reqs.append(dist.irecv(recvs[peer], peer, group=group))
    for r in reqs:
        r.wait()
