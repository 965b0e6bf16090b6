"""Host logic of the sharded single solve (include/poisson.h: poisson_shard_describe): the partition of the
split axis o and of the half-spectrum planes k_a, the slab shapes and the exchange volumes -- no GPU needed -- and a
world-size-2 gloo run in which two processes plan their shards independently and exchange an index-valued A1 the way
passes F1 / I2 do (every element to the rank that owns it), checking that what arrives is exactly each rank's slab."""
import itertools
import json
import os
import subprocess
import sys
from pathlib import Path

import pytest

import paper_1211_5244_b200 as pk

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module", autouse=True)
def lib():
    from paper_1211_5244_b200 import build
    build.build()
    return pk.load_library()


def _lo(total, s, R):
    return total * s // R


@pytest.mark.parametrize("R", [1, 2, 3, 5, 8])
def test_partition_tiles_split_axis_and_planes(R):
    n = (32, 20, 24)
    for bc in itertools.product((0, 1), repeat=3):
        plan = pk.poisson_plan_describe(*n, bc, pk.FP64)
        a = plan.order[0]
        o = 3 - a
        H = plan.half_len
        infos = [pk.poisson_shard_describe(*n, bc, pk.FP64, r, R) for r in range(R)]
        cplx = 16
        for r, i in enumerate(infos):
            assert (i.rank, i.nranks, i.split_axis, i.plane_axis) == (r, R, o, a)
            assert (i.o0, i.o1) == (_lo(n[o], r, R), _lo(n[o], r + 1, R)) and i.o1 > i.o0
            assert (i.k0, i.k1) == (_lo(H, r, R), _lo(H, r + 1, R)) and i.k1 > i.k0
            loc = [n[2], n[1], n[0]]; loc[2 - o] = i.o1 - i.o0
            assert list(i.local_dims) == loc
            a1 = [n[2], n[1], n[0]]; a1[2 - a] = H
            mid = list(a1); mid[2 - a] = i.k1 - i.k0
            back = list(a1); back[2 - o] = i.o1 - i.o0
            assert list(i.mid_dims) == mid and list(i.back_dims) == back
            assert i.mid_bytes == mid[0] * mid[1] * mid[2] * cplx and i.back_bytes == back[0] * back[1] * back[2] * cplx
            # every v has exactly one owner, and the closed form the kernels use finds it
            for v in range(H):
                s = ((v + 1) * R - 1) // H
                assert infos[s].k0 <= v < infos[s].k1
            for v in range(n[o]):
                s = ((v + 1) * R - 1) // n[o]
                assert infos[s].o0 <= v < infos[s].o1
        a1_bytes = H * n[o] * n[0] * cplx
        assert sum(i.mid_bytes for i in infos) == a1_bytes == sum(i.back_bytes for i in infos)
        kept = sum((i.k1 - i.k0) * (i.o1 - i.o0) * n[0] * cplx for i in infos)       # the part of A1 that never leaves its GPU
        assert sum(i.sent_bytes[0] for i in infos) == a1_bytes - kept == sum(i.sent_bytes[1] for i in infos)


def test_exchange_is_on_the_smallest_intermediate():
    """transposes act on the reduced data set.  Per direction the fabric carries A1 (H N_o N_x complex)
    minus what stays local -- half of SURVEY.md 8e's A2 figure for configs[1] -- and a quarter of rho's padded size."""
    infos = [pk.poisson_shard_describe(128, 128, 128, (0, 0, 0), pk.FP64, r, 8) for r in range(8)]
    a1 = 129 * 128 * 128 * 16
    sent = sum(i.sent_bytes[0] for i in infos)
    assert a1 * 7 // 8 - 129 * 128 * 16 <= sent <= a1 * 7 // 8 + 129 * 128 * 16 * 8      # ~ (R-1)/R of A1
    assert sent < 67.6e6 / 2 + 1e6                                                      # A2 would be 67.6 MB


def test_unsupported_and_invalid():
    for args, status in [(((30, 32, 32), (0, 0, 0), 0, 2), None),            # fine: S = 60 is compiled
                         (((31, 32, 32), (0, 0, 0), 0, 2), 2),               # odd N_x
                         (((32, 22, 32), (0, 0, 0), 0, 2), 2),               # S_y = 44: any-length kernel only
                         (((32, 4, 32), (0, 1, 0), 0, 5), 2),                # more ranks than points of the split axis
                         (((32, 32, 32), (0, 0, 0), 2, 2), 1),               # rank out of range
                         (((32, 32, 32), (0, 0, 0), 0, 0), 1)]:
        n, bc, r, R = args
        if status is None:
            pk.poisson_shard_describe(*n, bc, pk.FP64, r, R)
        else:
            with pytest.raises(pk.PoissonError) as ei:
                pk.poisson_shard_describe(*n, bc, pk.FP64, r, R)
            assert ei.value.status == status, args


WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
import paper_1211_5244_b200 as pk
dist.init_process_group(backend="gloo")
rank, R = dist.get_rank(), dist.get_world_size()
n, bc = (16, 12, 10), {bc!r}
me = pk.poisson_shard_describe(*n, bc, pk.FP64, rank, R)
plan = pk.poisson_plan_describe(*n, bc, pk.FP64)
a, o, H = plan.order[0], 3 - plan.order[0], plan.half_len
# every rank learns every rank's ranges (what a real run gets from planning all ranks locally: the partition is a closed form)
mine = torch.tensor([me.o0, me.o1, me.k0, me.k1], dtype=torch.int64)
allr = [torch.zeros(4, dtype=torch.int64) for _ in range(R)]
dist.all_gather(allr, mine)
for s in range(R):
    t = pk.poisson_shard_describe(*n, bc, pk.FP64, s, R)
    assert allr[s].tolist() == [t.o0, t.o1, t.k0, t.k1]
# A1 with value = global linear index, shape [z][y][x] with axis a -> H
shape = [n[2], n[1], n[0]]; shape[2 - a] = H
A1 = np.arange(int(np.prod(shape)), dtype=np.float64).reshape(shape)
def cut(arr, axis_id, lo, hi):
    sl = [slice(None)] * 3; sl[2 - axis_id] = slice(lo, hi); return arr[tuple(sl)]
# exchange 1: what F1 does -- my slab of o, every plane to the rank that owns it (send / recv over gloo)
my_f1_out = cut(A1, o, me.o0, me.o1)
mid = np.full(list(me.mid_dims), np.nan)
reqs, bufs = [], []
for s in range(R):
    o0, o1, k0, k1 = allr[s].tolist()
    part = np.ascontiguousarray(cut(my_f1_out, a, k0, k1))          # planes of rank s, my o range
    if s == rank:
        dst = cut(cut(mid, a, 0, me.k1 - me.k0), o, me.o0, me.o1); dst[...] = part
    else:
        reqs.append(dist.isend(torch.from_numpy(part), s))
        buf = torch.empty(list(cut(cut(A1, a, me.k0, me.k1), o, o0, o1).shape), dtype=torch.float64)
        bufs.append((s, o0, o1, buf)); reqs.append(dist.irecv(buf, s))
for q in reqs: q.wait()
for s, o0, o1, buf in bufs:
    cut(mid, o, o0, o1)[...] = buf.numpy()
ok1 = bool(np.array_equal(mid, cut(A1, a, me.k0, me.k1)))
# exchange 2: what I2 does -- my planes, every o to the rank that owns it
back = np.full(list(me.back_dims), np.nan)
reqs, bufs = [], []
for s in range(R):
    o0, o1, k0, k1 = allr[s].tolist()
    part = np.ascontiguousarray(cut(mid, o, o0, o1))
    if s == rank:
        cut(back, a, me.k0, me.k1)[...] = part
    else:
        reqs.append(dist.isend(torch.from_numpy(part), s))
        buf = torch.empty(list(cut(cut(A1, o, me.o0, me.o1), a, k0, k1).shape), dtype=torch.float64)
        bufs.append((k0, k1, buf)); reqs.append(dist.irecv(buf, s))
for q in reqs: q.wait()
for k0, k1, buf in bufs:
    cut(back, a, k0, k1)[...] = buf.numpy()
ok2 = bool(np.array_equal(back, cut(A1, o, me.o0, me.o1)))
sent = torch.tensor([me.sent_bytes[0], me.sent_bytes[1]], dtype=torch.int64)
dist.all_reduce(sent)
flags = torch.tensor([int(ok1), int(ok2)], dtype=torch.int64)
dist.all_reduce(flags, op=dist.ReduceOp.MIN)
if rank == 0:
    print(json.dumps({{"ok": flags.tolist(), "sent": sent.tolist(), "a1_bytes": int(A1.size) * 16, "world": R}}))
dist.destroy_process_group()
"""


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 1, 0)], ids=["split_y", "split_z"])
def test_two_ranks_exchange_with_planned_ranges_gloo(tmp_path, bc):
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=str(ROOT), bc=bc))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    out = subprocess.run(
        [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
         "--master-port", "29541", str(script)], capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    d = json.loads([l for l in out.stdout.splitlines() if l.startswith("{")][-1])
    assert d["world"] == 2 and d["ok"] == [1, 1]
    assert 0 < d["sent"][0] < d["a1_bytes"] and 0 < d["sent"][1] < d["a1_bytes"]
