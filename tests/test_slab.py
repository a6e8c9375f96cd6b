"""Slab-distributed transform.

CPU: the partition every rank derives (sticks by k1 column ranges, z slabs) covers everything exactly once, and the
documented block layout of the exchange -- [peer][band][row][column] on both sides -- is checked against the oracle
with a real gloo all-to-all for world sizes 2, 4 and 8: rank s packs the oracle's z-only stage of ITS sticks, the
blocks travel, rank r unpacks and must hold the oracle's z-only stage of ALL sticks on ITS planes.
GPU (one device): the ranks of a world are simulated as R slab plans in one process; their pack / unpack kernels, z
passes and plane passes must reproduce the single-GPU plan bit for bit, through the staged blocks and through direct
peer pointers.  A 2-rank NCCL run is gated on two visible GPUs."""
import os
import sys

import numpy as np
import pytest

from paper_2406_05577_b200 import binding as fb
from paper_2406_05577_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_2406_05577_b200.build import build

    build()


def _slab(n, a, batch, world, rank, dtype="c128"):
    from paper_2406_05577_b200.slab import SlabPlan

    return SlabPlan(n, a, batch, world, rank, dtype=dtype)


@pytest.mark.parametrize("n,a", [((64, 64, 64), (16, 16, 16)), ((128, 128, 128), (32, 32, 32)), ((96, 96, 192), (24, 24, 48)), ((64, 64, 32), (3, 16, 8))])
@pytest.mark.parametrize("world", [1, 2, 3, 4, 8, 16])
def test_partition_covers_everything_once(oracle, n, a, world):
    m = oracle.stick_map(n, a)
    if 2 * a[0] + 1 < world:
        with pytest.raises(fb.FftbError) as e:
            _slab(n, a, 2, world, 0)
        assert e.value.code == fb.FFTB_EUNSUPPORTED
        return
    plans = [_slab(n, a, 2, world, r) for r in range(world)]
    p0 = plans[0]
    for p in plans:  # every rank derives the same partition
        assert np.array_equal(p.stick_lo, p0.stick_lo) and np.array_equal(p.packed_lo, p0.packed_lo) and np.array_equal(p.z_lo, p0.z_lo)
    assert p0.stick_lo[0] == 0 and p0.stick_lo[-1] == len(m["k1"]) and np.all(np.diff(p0.stick_lo) > 0)
    assert p0.z_lo[0] == 0 and p0.z_lo[-1] == n[2] and np.all(np.diff(p0.z_lo) > 0)
    assert np.array_equal(p0.packed_lo, m["off"][p0.stick_lo])
    # ranks own whole k1 columns, and the stick counts are balanced to within the largest column
    cuts = p0.stick_lo[1:-1]
    assert np.all(m["k1"][cuts] != m["k1"][cuts - 1])
    col_max = np.bincount(m["k1"] - m["k1"].min()).max()
    assert np.abs(np.diff(p0.stick_lo) - len(m["k1"]) / world).max() <= col_max
    for r, p in enumerate(plans):
        assert p.info["n_points_local"] == p0.packed_lo[r + 1] - p0.packed_lo[r]
        assert p.info["n_sticks_local"] == p0.stick_lo[r + 1] - p0.stick_lo[r]
        assert p.info["planes_local"] == p0.z_lo[r + 1] - p0.z_lo[r]
        s_cnt, r_cnt = p.counts("inverse", 3)
        fs_cnt, fr_cnt = p.counts("forward", 3)
        assert s_cnt == fr_cnt and r_cnt == fs_cnt  # the forward exchange is the inverse one run backwards
    for r in range(world):
        for d in range(world):
            assert plans[r].counts("inverse", 3)[0][d] == plans[d].counts("inverse", 3)[1][r]


def test_error_paths():
    with pytest.raises(fb.FftbError) as e:
        _slab((64, 64, 64), (16, 16, 16), 2, 4, 4)
    assert e.value.code == fb.FFTB_EINVAL
    with pytest.raises(fb.FftbError) as e:
        _slab((64, 64, 64), (16, 16, 16), 2, 17, 0)
    assert e.value.code == fb.FFTB_EUNSUPPORTED
    p = _slab((64, 64, 64), (16, 16, 16), 2, 2, 0)
    import ctypes

    ptr = ctypes.c_void_p()
    assert fb.lib().fftb_slab_plan_exchange_ptr(p._h, 0, ctypes.byref(ptr)) == fb.FFTB_ESTATE  # before bind
    assert fb.lib().fftb_slab_plan_destroy(None) == fb.FFTB_EINVAL


def _gloo_worker(rank, world, port, n, a, nb, out_dir):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    import oracle
    from paper_2406_05577_b200 import workloads as wl
    from paper_2406_05577_b200.slab import SlabPlan

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = SlabPlan(n, a, nb, world, rank)
    m = oracle.stick_map(n, a)
    k = oracle.enum_points(n, a)
    w = wl.Workload(0, "t", n, a, "c128", nb, "uniform", "inv_fwd")
    c = wl.coefficients(w, *k)
    # this rank's sticks only: zero the other ranks' coefficients, so the oracle's z-only stage holds nothing else
    mine = np.zeros(c.shape[1], bool)
    mine[p.packed_lo[rank]:p.packed_lo[rank + 1]] = True
    stage = oracle.inverse(n, k, np.where(mine[None, :], c, 0), n_axes=1)          # [b][z][y][x]
    s0, s1 = p.stick_lo[rank], p.stick_lo[rank + 1]
    A_local = stage[:, :, m["k2"][s0:s1] % n[1], m["k1"][s0:s1] % n[0]]             # [b][z][own sticks]
    # pack as fftb_slab_inverse_begin documents it: [peer][band][the peer's planes][own sticks]
    send = np.concatenate([A_local[:, p.z_lo[d]:p.z_lo[d + 1], :].ravel() for d in range(world)])
    s_cnt, r_cnt = p.counts("inverse", nb)
    assert send.size == sum(s_cnt)
    recv = torch.empty(sum(r_cnt), dtype=torch.complex128)
    dist.all_to_all_single(torch.view_as_real(recv), torch.view_as_real(torch.from_numpy(send)), r_cnt, s_cnt)
    # unpack as fftb_slab_inverse_end documents it: [peer][band][own planes][the peer's sticks]
    planes = p.z_lo[rank + 1] - p.z_lo[rank]
    A_full = np.zeros((nb, planes, len(m["k1"])), complex)
    off = 0
    for s in range(world):
        ns = p.stick_lo[s + 1] - p.stick_lo[s]
        A_full[:, :, p.stick_lo[s]:p.stick_lo[s + 1]] = recv.numpy()[off:off + nb * planes * ns].reshape(nb, planes, ns)
        off += nb * planes * ns
    np.save(os.path.join(out_dir, f"A_{rank}.npy"), A_full)
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4, 8])
def test_exchange_layout_vs_oracle_gloo(tmp_path, oracle, world):
    import torch.multiprocessing as mp

    n, a, nb = (64, 64, 64), (9, 16, 11), 2
    port = 29500 + (os.getpid() + 17 * world) % 2000
    mp.spawn(_gloo_worker, args=(world, port, n, a, nb, str(tmp_path)), nprocs=world, join=True)
    m = oracle.stick_map(n, a)
    k = oracle.enum_points(n, a)
    c = wl.coefficients(wl.Workload(0, "t", n, a, "c128", nb, "uniform", "inv_fwd"), *k)
    ref = oracle.inverse(n, k, c, n_axes=1)[:, :, m["k2"] % n[1], m["k1"] % n[0]]     # [b][z][stick], all sticks
    got = np.concatenate([np.load(tmp_path / f"A_{r}.npy") for r in range(world)], axis=1)
    assert got.shape == ref.shape and np.array_equal(got, ref)


# ---------------------------------------------------------------------------------------------------------------
# GPU
# ---------------------------------------------------------------------------------------------------------------
def _rel(x, y):
    x, y = np.asarray(x, np.complex128).ravel(), np.asarray(y, np.complex128).ravel()
    return float(np.linalg.norm(x - y) / np.linalg.norm(y))


@pytest.mark.gpu
@pytest.mark.parametrize("direct", [False, True], ids=["staged", "peer_pointers"])
@pytest.mark.parametrize("n,a,dtype,world", [((64, 64, 64), (16, 16, 16), "c128", 4), ((128, 128, 128), (32, 32, 32), "c128", 8),
                                             ((128, 128, 128), (32, 20, 32), "c64", 3), ((96, 96, 192), (24, 24, 48), "c64", 2),
                                             ((256, 256, 64), (64, 64, 16), "c128", 5)])
def test_simulated_ranks_reproduce_the_single_gpu_plan(oracle, n, a, dtype, world, direct):
    """R slab plans on one device stand for R ranks: z passes on the own sticks, pack, (simulated) all-to-all, unpack,
    plane passes on the own slab -- and back.  Concatenated over the ranks the cuboid and the packed result equal the
    single-GPU plan's bit for bit (every stick and every plane goes through the same kernel arithmetic), and the oracle
    within tolerance."""
    import torch

    nb = 3
    w = wl.Workload(0, "t", n, a, dtype, nb, "uniform", "inv_fwd")
    whole = fb.Plan(n, a, batch=nb, dtype=dtype).bind()
    k = whole.points()
    c = wl.coefficients(w, *k)
    d_c = torch.from_numpy(c).cuda()
    ranks = [_slab(n, a, nb, world, r, dtype=dtype).bind() for r in range(world)]
    p0 = ranks[0]
    ct = whole.torch_complex

    def transport(direction, sends):
        """the all-to-all: block d of rank s's send buffer becomes block s of rank d's receive buffer"""
        recvs = []
        for d in range(world):
            parts = []
            for s in range(world):
                cnt = ranks[s].counts(direction, nb)[0]
                o = sum(cnt[:d])
                parts.append(sends[s][o:o + cnt[d]])
            recvs.append(torch.cat(parts))
            assert recvs[-1].numel() == sum(ranks[d].counts(direction, nb)[1])
        return recvs

    # ---- inverse
    local = [d_c[:, p0.packed_lo[r]:p0.packed_lo[r + 1]].clone() for r in range(world)]
    slabs = [torch.empty(ranks[r].cuboid_slab_shape(nb), dtype=ct, device="cuda") for r in range(world)]
    if direct:
        peers = [ranks[r].exchange_ptr(0) for r in range(world)]
        for r in range(world):
            ranks[r].inverse_begin(local[r], peers=peers)
        for r in range(world):
            ranks[r].inverse_end(slabs[r])
    else:
        sends = [torch.empty(sum(ranks[r].counts("inverse", nb)[0]), dtype=ct, device="cuda") for r in range(world)]
        for r in range(world):
            ranks[r].inverse_begin(local[r], send=sends[r])
        recvs = transport("inverse", sends)
        for r in range(world):
            ranks[r].inverse_end(slabs[r], recv=recvs[r])
    psi = torch.cat(slabs, dim=1)
    ref = whole.inverse(d_c)
    torch.cuda.synchronize()
    assert torch.equal(psi, ref)
    if n[0] <= 128:
        assert _rel(psi[:1].cpu().numpy(), oracle.inverse(n, k, c[:1])) <= w.tol
    # ---- forward of a generic cuboid
    g = torch.from_numpy(wl.cuboid(w)).cuda()
    gs = [g[:, p0.z_lo[r]:p0.z_lo[r + 1]].contiguous() for r in range(world)]
    outs = [torch.empty((nb, ranks[r].info["n_points_local"]), dtype=ct, device="cuda") for r in range(world)]
    if direct:
        peers = [ranks[r].exchange_ptr(1) for r in range(world)]
        for r in range(world):
            ranks[r].forward_begin(gs[r], peers=peers)
        for r in range(world):
            ranks[r].forward_end(outs[r])
    else:
        sends = [torch.empty(sum(ranks[r].counts("forward", nb)[0]), dtype=ct, device="cuda") for r in range(world)]
        for r in range(world):
            ranks[r].forward_begin(gs[r], send=sends[r])
        recvs = transport("forward", sends)
        for r in range(world):
            ranks[r].forward_end(outs[r], recv=recvs[r])
    f = torch.cat(outs, dim=1)
    f_ref = whole.forward(g)
    torch.cuda.synchronize()
    assert torch.equal(f, f_ref)
    if n[0] <= 128:
        assert _rel(f[:1].cpu().numpy(), oracle.forward(n, k, wl.cuboid(w)[:1], 1.0 / float(np.prod(n)))) <= w.tol
    for p in ranks + [whole]:
        p.destroy()


def _nccl_worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    import torch
    import torch.distributed as dist

    from paper_2406_05577_b200 import binding as fb
    from paper_2406_05577_b200 import workloads as wl
    from paper_2406_05577_b200.slab import SlabPlan

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    n, a, nb = (128, 128, 128), (32, 32, 32), 4
    w = wl.Workload(0, "t", n, a, "c128", nb, "uniform", "inv_fwd")
    whole = fb.Plan(n, a, batch=nb).bind()
    c = wl.coefficients(w, *whole.points())
    p = SlabPlan(n, a, nb, world, rank).bind()
    d_c = torch.from_numpy(c).cuda()
    slab = p.inverse(d_c[:, p.packed_lo[rank]:p.packed_lo[rank + 1]].clone())
    back = p.forward(slab)
    ref = whole.inverse(d_c)
    torch.cuda.synchronize()
    ok = torch.equal(slab, ref[:, p.z_lo[rank]:p.z_lo[rank + 1]]) and torch.equal(back, whole.forward(ref)[:, p.packed_lo[rank]:p.packed_lo[rank + 1]])
    open(os.path.join(out_dir, f"ok_{rank}"), "w").write(str(bool(ok)))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.gpu
def test_two_ranks_nccl(tmp_path):
    """The real thing on two GPUs: SlabPlan.inverse / forward with an NCCL all-to-all between the begin and end halves."""
    import torch

    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs (this pool hands out one)")
    import torch.multiprocessing as mp

    mp.spawn(_nccl_worker, args=(2, 29500 + os.getpid() % 2000, str(tmp_path)), nprocs=2, join=True)
    assert all(open(tmp_path / f"ok_{r}").read() == "True" for r in range(2))
