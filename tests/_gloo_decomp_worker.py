"""Worker of tests/test_decomp_cpu.py: one rank of a world_size-2 gloo job running the host side of the
inter-block halo exchange (decomp.exchange_axis: who sends what to whom, in which order, axis by axis) on CPU
tensors.  The device kernels jf_pack_face / jf_unpack_face are replaced by numpy slicing with the same layer
convention (they are tested on the GPU); periodic passes of unsplit axes are numpy wraps."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2406_19494_b200 import cases, decomp  # noqa: E402

NH = 3
rank, world = int(os.environ["RANK"]), int(os.environ["WORLD_SIZE"])
dist.init_process_group("gloo")
blocks = tuple(int(v) for v in sys.argv[1].split(","))
c = cases.random_admissible(n=(16, 12, 8), seed=5)             # periodic on all axes
parts = decomp.split_case(c, blocks)
part = parts[rank]
n = part.case.n
U = part.case.U0.copy()                                        # [5, nz+6, ny+6, nx+6], x fastest (axis 3)
AX = {0: 3, 1: 2, 2: 1}                                        # grid axis -> numpy axis


def extents(axis):                                             # tangential extents of the pass of `axis` (reading O3)
    sl = [slice(None)] * 4
    if axis == 0:
        sl[AX[1]] = slice(NH, -NH)
    if axis <= 1:
        sl[AX[2]] = slice(NH, -NH)
    return sl


def layer(axis, idx):
    sl = extents(axis)
    sl[AX[axis]] = idx
    return tuple(sl)


def pack(f, buf):
    axis, side, N = f // 2, f % 2, n[f // 2]
    rows = [U[layer(axis, NH + (m - 1 if side == 0 else N - m))] for m in (1, 2, 3)]
    buf.copy_(torch.from_numpy(np.stack(rows, axis=1).ravel()))


def unpack(f, buf):
    axis, side, N = f // 2, f % 2, n[f // 2]
    shp = U[layer(axis, 0)].shape
    data = buf.numpy().reshape((5, 3) + shp[1:])
    for m in (1, 2, 3):
        U[layer(axis, NH + (-m if side == 0 else N - 1 + m))] = data[:, m - 1]


def new_buffer(f):
    return torch.empty(15 * int(np.prod(U[layer(f // 2, 0)].shape[1:])), dtype=torch.float64)


for axis in range(3):
    if part.neighbours[2 * axis] is None:                      # unsplit periodic axis: the physical pass
        N = n[axis]
        for m in (1, 2, 3):
            U[layer(axis, NH - m)] = U[layer(axis, NH + N - m)]
            U[layer(axis, NH + N - 1 + m)] = U[layer(axis, NH + m - 1)]
    decomp.exchange_axis(axis, part.neighbours, rank, pack, unpack, new_buffer, dist)

# expected: the periodic wrap of the undivided interior, cut out at this block's padded extents
G = c.U0[:, NH:-NH, NH:-NH, NH:-NH]
ix = [(part.lo[a] - NH + np.arange(n[a] + 2 * NH)) % c.n[a] for a in range(3)]
exp = G[:, ix[2]][:, :, ix[1]][:, :, :, ix[0]]
ok = bool(np.array_equal(U, exp))
res = torch.tensor([1.0 if ok else 0.0])
dist.all_reduce(res, op=dist.ReduceOp.MIN)
# the (status, dt) reduction of RankBlock.jf_cfl_dt: MIN of dt, and a failed rank fails every rank with dt = NaN
st_ok, dt_ok = decomp.reduce_dt(0, 0.5 + rank, torch, dist)
st_bad, dt_bad = decomp.reduce_dt(5 if rank == 1 else 0, float("nan") if rank == 1 else 0.25, torch, dist)
flags = torch.tensor([1.0 if (st_ok == 0 and dt_ok == 0.5 and st_bad == 5 and dt_bad != dt_bad) else 0.0])
dist.all_reduce(flags, op=dist.ReduceOp.MIN)                   # ... on EVERY rank
# the bench arm's own block: tgv_part materialises this rank's block only and must equal the cut of the global case
tp = decomp.tgv_part(8, blocks, rank)
g = cases.tgv(8, faces=tuple(cases.uniform_faces(0.0, 2.0 * np.pi * s, 8 * s) for s in blocks))
gp = decomp.split_case(g, blocks)[rank]
same = np.array_equal(tp.case.U0, gp.case.U0) and tp.neighbours == gp.neighbours and tp.lo == gp.lo and all(
    a.type == b.type and a.nb_width == b.nb_width and a.nb_face == b.nb_face for a, b in zip(tp.case.bc, gp.case.bc))
flags2 = torch.tensor([1.0 if same else 0.0])
dist.all_reduce(flags2, op=dist.ReduceOp.MIN)
if rank == 0:
    print(json.dumps({"all_ranks_match": bool(res.item() == 1.0), "dt_min": dt_ok, "status_reduction_ok": bool(flags.item() == 1.0),
                      "tgv_part_ok": bool(flags2.item() == 1.0), "blocks": blocks}), flush=True)
dist.destroy_process_group()
