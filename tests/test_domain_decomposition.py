"""Time-slab domain decomposition (row f2, first step; paper_2502_02490_b200/domain.py).

CPU: the decomposition and the ghost exchange are host logic; with the ORACLE as the rank-local operator the distributed
apply must reproduce the oracle's global D_w -- sequentially emulated ranks (world 1, 2, 4) and a real world_size-2 `gloo`
process group.  GPU: the same with the CUDA contexts as rank-local operators, ranks emulated one after the other on the one
GPU (their kernels never wait on one another)."""
import os
import socket

import numpy as np
import pytest

import synth
from oracle import qxd_ref as R
from paper_2502_02490_b200 import domain as D

KAPPA, CSW, CSWQ, Q = 0.12, 1.5, 1.0, 2.0 / 3.0


def global_reference(dims, cstar, ap, qed, psi):
    ref = R.Ref(*dims, cstar | (ap << 2))
    U = synth.su3_links(dims, 0.3, 1)
    A = synth.u1_field(dims, 0.3, 2) if qed else None
    ref.gauge_load(U, A, 1.0)
    ref.set_quark(KAPPA, Q if qed else 0.0)
    ref.clover_build(CSW, CSWQ if qed else 0.0)
    return U, A, ref.apply_Dw(psi)


def oracle_local_operator(ts, U, A, cstar, ap, qed):
    Ul, Al = ts.local_fields(U, A, antiperiodic=bool(ap))
    ref = R.Ref(*ts.local_dims, D.TimeSlabs.local_bc(cstar))
    ref.gauge_load(Ul, Al, 1.0)
    ref.set_quark(KAPPA, Q if qed else 0.0)
    ref.clover_build(CSW, CSWQ if qed else 0.0)
    return ref.apply_Dw


def emulate(dims, world, make_operator, psi):
    """All ranks in one process: scatter, copy ghosts by hand, apply, gather."""
    slabs = [D.TimeSlabs(dims, world, r) for r in range(world)]
    loc = [ts.scatter(psi) for ts in slabs]
    for r, ts in enumerate(slabs):       # what exchange_time_ghosts does with messages
        loc[r][0] = loc[ts.prev][ts.T_loc]
        loc[r][ts.T_loc + 1] = loc[ts.next][1]
    outs = [ts.interior(np.asarray(make_operator(ts)(loc[r])).reshape(loc[r].shape)) for r, ts in enumerate(slabs)]
    return np.concatenate(outs, axis=0)


def test_time_slabs_geometry():
    ts = D.TimeSlabs((8, 4, 4, 4), 2, 1)
    assert ts.T_loc == 4 and ts.local_dims == (6, 4, 4, 4) and ts.time_index() == [3, 4, 5, 6, 7, 0]
    assert (ts.prev, ts.next) == (0, 0)
    with pytest.raises(ValueError):
        D.TimeSlabs((6, 4, 4, 4), 2, 0)      # 3 slices per rank: odd
    U = synth.su3_links((8, 2, 2, 2), 0.3, 1)
    Ul, _ = ts.local_fields(U, None, antiperiodic=True)
    assert np.array_equal(Ul[4, ..., 0, :, :], -U[7, ..., 0, :, :]) and np.array_equal(Ul[4, ..., 1, :, :], U[7, ..., 1, :, :])
    assert np.array_equal(Ul[0], U[3]) and np.array_equal(Ul[5], U[0])


@pytest.mark.parametrize("dims,cstar,ap,qed,world", [((8, 4, 4, 4), 0, 1, False, 2), ((8, 2, 4, 4), 3, 1, True, 2),
                                                     ((8, 4, 2, 4), 2, 0, True, 4), ((4, 4, 4, 4), 0, 1, True, 1)])
def test_emulated_ranks_reproduce_the_global_operator(dims, cstar, ap, qed, world):
    X = (dims[0], 2 * dims[1] if cstar else dims[1], dims[2], dims[3])
    psi = synth.gaussian_spinor(X, 3)
    U, A, exp = global_reference(dims, cstar, ap, qed, psi)
    got = emulate(dims, world, lambda ts: oracle_local_operator(ts, U, A, cstar, ap, qed), psi)
    assert np.linalg.norm((got - exp).ravel()) / np.linalg.norm(exp.ravel()) < 1e-14


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, dims, cstar, ap, qed, out):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        X = (dims[0], 2 * dims[1] if cstar else dims[1], dims[2], dims[3])
        psi = synth.gaussian_spinor(X, 3)
        U = synth.su3_links(dims, 0.3, 1)
        A = synth.u1_field(dims, 0.3, 2) if qed else None
        ts = D.TimeSlabs(dims, world, rank)
        op = oracle_local_operator(ts, U, A, cstar, ap, qed)
        local = np.ascontiguousarray(ts.scatter(psi))
        res = D.apply_Dw_distributed(ts, local, op, dist)
        out.put((rank, np.array(res)))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_distributed_apply():
    import torch.multiprocessing as mp
    dims, cstar, ap, qed, world = (8, 2, 4, 4), 3, 1, True, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, dims, cstar, ap, qed, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=180) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    X = (dims[0], 2 * dims[1], dims[2], dims[3])
    psi = synth.gaussian_spinor(X, 3)
    _, _, exp = global_reference(dims, cstar, ap, qed, psi)
    got = np.concatenate([res[0], res[1]], axis=0)
    assert np.linalg.norm((got - exp).ravel()) / np.linalg.norm(exp.ravel()) < 1e-14


@pytest.mark.gpu
@pytest.mark.parametrize("dims,cstar,ap,qed,world", [((16, 4, 4, 4), 0, 1, False, 2), ((16, 2, 4, 4), 3, 1, True, 4)])
@pytest.mark.parametrize("prec", [0, 1])
def test_cuda_contexts_as_rank_local_operators(dims, cstar, ap, qed, world, prec):
    from paper_2502_02490_b200 import binding as B
    X = (dims[0], 2 * dims[1] if cstar else dims[1], dims[2], dims[3])
    psi = synth.gaussian_spinor(X, 3)
    U, A, exp = global_reference(dims, cstar, ap, qed, psi)
    ctxs = []

    def make(ts):
        Ul, Al = ts.local_fields(U, A, antiperiodic=bool(ap))
        g = B.Qxd(*ts.local_dims, D.TimeSlabs.local_bc(cstar), precisions=(B.QXD_F64, B.QXD_F32), pairing=cstar > 0)
        g.gauge_load(Ul, Al, 1.0)
        g.set_quark(KAPPA, Q if qed else 0.0)
        g.set_gauge_reconstruct(B.QXD_RECON_12)     # det W carries the boundary sign of the time links
        g.clover_build(CSW, CSWQ if qed else 0.0)
        ctxs.append(g)
        return lambda loc: g.apply_Dw(loc, prec).cpu().numpy()

    got = emulate(dims, world, make, psi)
    err = np.linalg.norm((got - exp).ravel()) / np.linalg.norm(exp.ravel())
    assert err < (1e-13 if prec == 0 else 1e-6), err
    for g in ctxs:
        g.close()
