"""CPU tests of the block decomposition's host logic (paper_2406_19494_b200/decomp.py):
the cut into sub-cases, and a world_size-2 gloo job exchanging halos point-to-point."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

from paper_2406_19494_b200 import cases, decomp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_split_geometry_neighbours_and_widths():
    c = cases.channel(24, 16, 8, n_steps=1)                  # periodic x, z; walls in y (tanh-stretched)
    parts = decomp.split_case(c, (2, 2, 1))
    assert len(parts) == 4 and [p.coords for p in parts] == [(0, 0, 0), (1, 0, 0), (0, 1, 0), (1, 1, 0)]
    dy = np.diff(c.yf)
    p00, p10, p01 = parts[0], parts[1], parts[2]
    assert p00.case.n == (12, 8, 8) and p01.lo == (0, 8, 0)
    # periodic x split in two: both x faces of a block exchange with the same neighbour (wrap)
    assert p00.neighbours[0] == 1 and p00.neighbours[1] == 1 and p10.neighbours[0] == 0
    assert p00.case.bc[0].type == cases.BC_EXCHANGE and p00.case.bc[1].type == cases.BC_EXCHANGE
    # walls stay on the outer y faces, the inner y faces exchange and carry the neighbour's true cell widths
    assert p00.case.bc[2].type == cases.BC_WALL_ISOTHERMAL and p00.neighbours[2] is None
    assert p00.case.bc[3].type == cases.BC_EXCHANGE and p00.neighbours[3] == 2
    assert np.allclose(p00.case.bc[3].nb_width, dy[8:11], rtol=0, atol=0)
    assert np.allclose(p01.case.bc[2].nb_width, dy[7:4:-1], rtol=0, atol=0)
    # the unsplit periodic z axis stays periodic
    assert p00.case.bc[4].type == cases.BC_PERIODIC and p00.neighbours[4] is None
    # the blocks tile the interior exactly
    G = decomp.gather_interior(c, parts, [p.case.U0 for p in parts])
    s = (slice(None),) + (slice(3, -3),) * 3
    assert np.array_equal(G[s], c.U0[s])
    assert np.array_equal(p10.case.xf, c.xf[12:])


def test_split_rejects_dirichlet_tangential_split_and_tiny_blocks():
    with pytest.raises(ValueError):
        decomp.split_case(cases.flat_plate(256, 32, 8), (1, 2, 1))
    with pytest.raises(ValueError):
        decomp.split_case(cases.random_admissible(n=(12, 10, 8)), (4, 1, 1))
    parts = decomp.split_case(cases.flat_plate(256, 32, 8), (4, 1, 1))      # splitting along the inflow normal is fine
    assert parts[0].case.bc[0].type == cases.BC_DIRICHLET and parts[1].case.bc[0].type == cases.BC_EXCHANGE
    assert parts[3].case.bc[1].type == cases.BC_ZEROGRAD


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("blocks", ["2,1,1", "1,2,1", "1,1,2"])
def test_two_rank_gloo_halo_exchange(blocks):
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "tests", "_gloo_decomp_worker.py"), blocks]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=300)
    assert out.returncode == 0, out.stderr[-3000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["all_ranks_match"] is True and d["dt_min"] == 0.5
    assert d["status_reduction_ok"] is True and d["tgv_part_ok"] is True


def test_interior_cuts_carry_the_neighbours_face_coordinates():
    # across an interior cut the halo cells take widths and centres from the neighbour's FACES (the undivided grid's
    # own expressions); across a periodic wrap from its cell widths (which is what the undivided grid does there)
    c = cases.channel(24, 16, 8, n_steps=1)
    parts = decomp.split_case(c, (2, 2, 1))
    p00, p01 = parts[0], parts[2]
    assert p00.case.bc[3].nb_face == tuple(c.yf[9:12]) and p01.case.bc[2].nb_face == tuple(c.yf[7:4:-1])
    assert p00.case.bc[0].nb_face is None and p00.case.bc[1].nb_face == tuple(c.xf[13:16])   # x-: wrap, x+: interior cut


def test_pid_is_equation_9():
    sys.path.insert(0, ROOT)
    import bench
    # PAPER.md:130 Eq. 9: wall time x ranks / DOF; the paper's own figures: < 0.1 s per step on 8 GPUs for 4.2 M cells
    assert bench.pid_seconds(100.0, 8, 256 * 128 * 128) == pytest.approx(0.1 * 8 / 4194304)
