"""The sharded single solve (include/poisson.h: poisson_shard_*) ACROSS A PROCESS BOUNDARY (PAPER.md:89,
"MPI subroutines between GPU memories").

tests/test_gpu_shard.py runs the R ranks as R plans inside one process.  Here every rank is its own process, as in a real
multi-GPU job: it creates its ShardPlan, allocates its two exchange slabs, hands them to the other ranks through CUDA IPC
(torch.multiprocessing moves a CUDA tensor between processes as a cudaIpcMemHandle; the receiver maps it and gets a device
pointer valid in ITS address space), passes every rank's pointers to poisson_shard_set_slabs, and runs

    forward | barrier A | middle | barrier B | inverse

with `torch.cuda.synchronize()` + a gloo `dist.barrier()` as the two barriers.  Passes F1 / I2 then really store into memory
owned by another process.  Only one GPU exists on the test box, so all ranks share cuda:0 (NCCL refuses two ranks on one
device; on a multi-GPU node the same code runs with one device per rank and NVLink peer mappings -- ShardedSolver).

Which barrier orders which write: A -- every rank's F1 stores into MY mid slab are complete before my
F2 reads it; B -- every rank's I2 stores into MY back slab are complete before my I1 reads it, and every rank's F2 has
consumed its mid slab before the next solve's F1 overwrites it.

Checked for all 8 boundary-condition combinations, R = 2 and R = 3 (ragged partition), two solves in a row: the concatenated
V equals poisson_solve's bit for bit and is within 1e-12 of the oracle."""
import itertools
import socket

import numpy as np
import pytest

import oracle
from workloads import generators as gen

pytestmark = pytest.mark.gpu

N = (32, 20, 24)
ALL_BC = list(itertools.product((0, 1), repeat=3))


def _inputs(bc_index, bc):
    """The same seeded rho and K^F in the parent and in every rank."""
    rng = np.random.default_rng(7000 + bc_index)
    sx, sy, sz = gen.padded_shape(N, bc)
    K = rng.standard_normal((sz, sy, sx))
    for ax in range(3):
        K = 0.5 * (K + np.roll(np.flip(K, axis=ax), 1, axis=ax))
    return rng.standard_normal((N[2], N[1], N[0])), oracle.kernel_spectrum(K)


def _rank_main(rank, R, port, inboxes, results):
    """One rank = one process.  Runs every BC combination; puts (bc_index, rep, rank, o0, o1, V slab) on `results`."""
    try:
        import torch
        import torch.distributed as dist
        import paper_1211_5244_b200 as pk
        torch.cuda.set_device(0)
        dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=R)
        for bi, bc in enumerate(ALL_BC):
            rho, Kf = _inputs(bi, bc)
            plan = pk.ShardPlan(N, bc, 0.25, pk.FP64, rank, R)
            info = plan.info
            mid = torch.full((info.mid_bytes // 8,), float("nan"), dtype=torch.float64, device="cuda")
            back = torch.full((info.back_bytes // 8,), float("nan"), dtype=torch.float64, device="cuda")
            for s in range(R):                                   # my slabs to every other rank: CUDA IPC handles
                if s != rank:
                    inboxes[s].put((rank, mid, back))
            mids, backs = [None] * R, [None] * R
            mids[rank], backs[rank] = mid, back
            for _ in range(R - 1):                               # their slabs, mapped into this process
                r, m, b = inboxes[rank].get(timeout=120)
                mids[r], backs[r] = m, b
            assert all(t.is_cuda for t in mids + backs)
            plan.set_slabs([t.data_ptr() for t in mids], [t.data_ptr() for t in backs], keep=(mids, backs))
            plan.set_kernel(torch.from_numpy(Kf).cuda())
            axis = 2 - info.split_axis
            sl = [slice(None)] * 3
            sl[axis] = slice(info.o0, info.o1)
            loc = torch.from_numpy(np.ascontiguousarray(rho[tuple(sl)])).cuda()
            for rep in range(2):
                mid.fill_(float("nan"))
                back.fill_(float("nan"))
                torch.cuda.synchronize()
                dist.barrier()                                   # no rank stores into a slab that is still being cleared
                plan.forward(loc)
                torch.cuda.synchronize()
                dist.barrier()                                   # barrier A
                assert bool(torch.isfinite(mid).all()), "a peer's F1 left part of my plane slab unwritten"
                plan.middle()
                torch.cuda.synchronize()
                dist.barrier()                                   # barrier B
                assert bool(torch.isfinite(back).all()), "a peer's I2 left part of my slab unwritten"
                V = torch.empty_like(loc)
                plan.inverse(V)
                torch.cuda.synchronize()
                results.put((bi, rep, rank, int(info.o0), int(info.o1), V.cpu().numpy()))
            dist.barrier()                                       # every rank is done with every slab of this BC
            plan.close()
            del mids, backs, mid, back
        results.put(("done", rank))
        dist.barrier()
        dist.destroy_process_group()
    except BaseException as e:  # noqa: BLE001 -- report, the parent fails the test
        import traceback
        results.put(("error", rank, f"{type(e).__name__}: {e}\n{traceback.format_exc()}"))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("R", [2, 3])
def test_sharded_solve_between_processes_through_cuda_ipc(R):
    import queue
    import torch
    import torch.multiprocessing as mp
    import paper_1211_5244_b200 as pk
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device; the solve has no fallback")
    pk.load_library()
    torch.cuda.set_device(0)
    ctx = mp.get_context("spawn")
    inboxes = [ctx.Queue() for _ in range(R)]
    results = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_rank_main, args=(r, R, port, inboxes, results), daemon=True) for r in range(R)]
    for p in procs:
        p.start()
    got, done = {}, 0
    try:
        while done < R:
            try:
                item = results.get(timeout=300)
            except queue.Empty:
                pytest.fail("a rank process stopped responding")
            if item[0] == "error":
                pytest.fail(f"rank {item[1]} failed: {item[2]}")
            if item[0] == "done":
                done += 1
                continue
            bi, rep, rank, o0, o1, V = item
            got[(bi, rep, rank)] = (o0, o1, V)
    finally:
        for p in procs:
            p.join(timeout=60)
            if p.is_alive():
                p.terminate()                                    # exactly the processes this test started
    for bi, bc in enumerate(ALL_BC):
        rho, Kf = _inputs(bi, bc)
        plan = pk.PoissonPlan(N, bc, 0.25, pk.FP64)
        try:
            plan.set_kernel(torch.from_numpy(Kf).cuda())
            V_ref = plan.solve(torch.from_numpy(rho).cuda()).cpu().numpy()
        finally:
            plan.close()
        info0 = pk.poisson_shard_describe(N[0], N[1], N[2], bc, pk.FP64, 0, R)
        axis = 2 - info0.split_axis
        for rep in range(2):
            parts = sorted((got[(bi, rep, r)] for r in range(R)), key=lambda t: t[0])
            assert parts[0][0] == 0 and parts[-1][1] == N[info0.split_axis]
            V = np.concatenate([p[2] for p in parts], axis=axis)
            assert np.array_equal(V, V_ref), (bc, R, rep)        # bitwise poisson_solve's
        err = float(np.linalg.norm(V - oracle.solve(rho, Kf, bc)) / np.linalg.norm(V_ref))
        assert err <= 1e-12, (bc, R, err)
