"""Intra-configuration sharding on CPU: world_size 2 and 3, `gloo`.
Every rank holds one t-slab of the lattice and runs ONE full iteration with the plans and exchanges of
paper_1208_1186_b200/slabs.py -- halo slice from below for Delta, two all-to-alls around the t transform, halo slice
from above for the update -- using the oracle's per-site steps on its slab and torch.fft along the lines it owns.
The assembled result must be the single-lattice oracle's: Delta, theta, F and every link after the update."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1208_1186_b200 import slabs

ALPHA = 0.08


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _c(a):
    """numpy complex -> torch complex128 (contiguous)."""
    return torch.from_numpy(np.ascontiguousarray(a))


def _worker(rank: int, world: int, port: int, L, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import lgf_inputs as gi
        import oracle
        oracle.set_threads(1)
        Lx, Ly, Lz, Lt = L
        plan = slabs.make_plan(L, world, rank)
        U = gi.make_config(L, 71, 0.59).reshape(Lt, Lz, Ly, Lx, 4, 3, 3)        # every rank can make the field; it keeps its slab
        Us = U[plan.t0:plan.t1].contiguous()
        nt = plan.nt
        Lext = (Lx, Ly, Lz, nt + 1)

        # ---- step 1: Delta on the slab needs U_t of slice t0 - 1 (K1's halo) ----
        below = slabs.halo_from_below(plan, Us[-1])
        ext = torch.cat([below[None], Us], 0).reshape(-1, 4, 3, 3)
        D_ext, _, _ = oracle.measure(Lext, ext)
        D = _c(D_ext).reshape(nt + 1, Lz, Ly, Lx, 3, 3)[1:].contiguous()         # the halo slice's own Delta is not valid
        part = torch.tensor([float((D.abs() ** 2).sum()), float(torch.einsum("tzyxmii->", Us).real)], dtype=torch.float64)
        dist.all_reduce(part)
        V = Lx * Ly * Lz * Lt
        theta, F = float(part[0]) / (3 * V), float(part[1]) / (12 * V)

        # ---- steps 2-3: x, y, z lines are local; the t lines need the all-to-all pair ----
        S = torch.fft.fftn(D, dim=(1, 2, 3))
        Z = slabs.transpose_t_to_z(plan, S)                                     # [Lt, nz, Ly, Lx, 3, 3]
        Z = torch.fft.fft(Z, dim=0)
        kt = torch.arange(Lt, dtype=torch.float64)[:, None, None, None]
        kz = torch.arange(plan.z0, plan.z1, dtype=torch.float64)[None, :, None, None]
        ky = torch.arange(Ly, dtype=torch.float64)[None, None, :, None]
        kx = torch.arange(Lx, dtype=torch.float64)[None, None, None, :]
        p2 = (4 * torch.sin(torch.pi * kt / Lt) ** 2 + 4 * torch.sin(torch.pi * kz / Lz) ** 2 +
              4 * torch.sin(torch.pi * ky / Ly) ** 2 + 4 * torch.sin(torch.pi * kx / Lx) ** 2)
        pmax = sum(4 * np.sin(np.pi * (n // 2) / n) ** 2 for n in L)
        scale = torch.where(p2 > 0, pmax / torch.where(p2 > 0, p2, torch.ones_like(p2)), torch.zeros_like(p2))
        Z = torch.fft.ifft(Z * scale[..., None, None], dim=0)
        Dt = torch.fft.ifftn(slabs.transpose_z_to_t(plan, Z), dim=(1, 2, 3))

        # ---- steps 4-5: g on the slab; the update needs g of slice t1 (K5's halo) ----
        g = _c(oracle.build_g((Lx, Ly, Lz, nt), Dt.reshape(-1, 3, 3), ALPHA)).reshape(nt, Lz, Ly, Lx, 3, 3)
        above = slabs.halo_from_above(plan, g[0])
        g_ext = torch.cat([g, above[None]], 0).reshape(-1, 3, 3)
        U_ext = torch.cat([Us, Us[:1]], 0).reshape(-1, 4, 3, 3)                  # the extra slice's links are never used
        Unew = _c(oracle.update_links(Lext, U_ext, g_ext)).reshape(nt + 1, Lz, Ly, Lx, 4, 3, 3)[:nt].contiguous()

        pieces = [torch.empty((t1 - t0, Lz, Ly, Lx, 4, 3, 3), dtype=torch.complex128) for (t0, t1) in plan.t_ranges]
        dist.all_gather(pieces, Unew) if len({p.shape for p in pieces}) == 1 else _gather_uneven(pieces, Unew, plan)
        dpieces = [torch.empty((t1 - t0, Lz, Ly, Lx, 3, 3), dtype=torch.complex128) for (t0, t1) in plan.t_ranges]
        dist.all_gather(dpieces, D) if len({p.shape for p in dpieces}) == 1 else _gather_uneven(dpieces, D, plan)
        if rank == 0:
            out.put((theta, F, torch.cat(dpieces, 0).numpy(), torch.cat(pieces, 0).numpy(),
                     plan.a2a_send_counts(), plan.a2a_recv_counts()))
    finally:
        dist.destroy_process_group()


def _gather_uneven(pieces, mine, plan):
    """all_gather for slabs of different thickness: every rank broadcasts its piece in turn."""
    for r in range(plan.world):
        if r == plan.rank:
            pieces[r].copy_(mine)
        dist.broadcast(pieces[r], r)


@pytest.mark.parametrize("world,L", [(2, (4, 4, 6, 8)), (3, (4, 6, 6, 8)), (2, (6, 4, 3, 4))])
def test_one_iteration_on_t_slabs_equals_single_lattice_oracle(world, L):
    import lgf_inputs as gi
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, L, q)) for r in range(world)]
    for p in procs:
        p.start()
    theta, F, D, Unew, sc, rc = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    U = gi.make_config(L, 71, 0.59)
    D0, th0, F0 = oracle.measure(L, U)
    ref, thh, Fh = oracle.iterate(L, U, 1, ALPHA)
    V = gi.volume(L)
    assert np.max(np.abs(D.reshape(V, 3, 3) - D0)) == 0               # the same per-site arithmetic on the same links
    assert abs(theta - th0) <= 1e-13 * th0 and abs(F - F0) <= 1e-13
    assert np.max(np.abs(Unew.reshape(V, 4, 3, 3) - ref)) <= 1e-12
    # rank 0's all-to-all plan: what it sends is its t-slab split by the peers' z-slabs, and the counts add up
    nt0 = slabs.split_extent(L[3], world)[0]
    assert sum(sc) == (nt0[1] - nt0[0]) * L[0] * L[1] * L[2]
    nz0 = slabs.split_extent(L[2], world)[0]
    assert sum(rc) == L[3] * (nz0[1] - nz0[0]) * L[0] * L[1]


def test_partition_and_budget_host_logic():
    assert slabs.split_extent(8, 3) == [(0, 3), (3, 6), (6, 8)]
    assert slabs.split_extent(64, 8) == [(8 * r, 8 * r + 8) for r in range(8)]
    with pytest.raises(ValueError):
        slabs.split_extent(2, 3)
    p = slabs.make_plan((64, 64, 64, 64), 8, 3)
    assert (p.t0, p.t1, p.z0, p.z1, p.below, p.above) == (24, 32, 24, 32, 2, 4)
    assert slabs.make_plan((8, 8, 8, 8), 4, 0).below == 3 and slabs.make_plan((8, 8, 8, 8), 4, 3).above == 0
    # 64^4 fp64 on 8 GPUs -- each all-to-all sends 7/8 of a 134 MB block = 117 MB per rank
    b = slabs.bytes_per_iteration((64, 64, 64, 64), 8, 8, 12)
    assert b["all_to_all_each"] == 7 * (8 * 64 ** 3 * 8 * 8) // 8 == 117440512
    assert b["halo_delta"] == 64 ** 3 * 64 and b["halo_links"] == 64 ** 3 * 12 * 8
    assert slabs.bytes_per_iteration((64, 64, 64, 64), 1, 8, 12)["total_sent"] == 0
    n = slabs.nvlink_budget((64, 64, 64, 64), 8, 8, 12)
    assert 0.5 < n["link_over_hbm"] < 0.7                    # 0.36 ms of exchanges against 0.53 ms of HBM time: must overlap
