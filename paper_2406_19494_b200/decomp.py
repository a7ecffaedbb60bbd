"""Block decomposition of a case (include/jf.h "Block decomposition").

The paper splits the domain into Sx x Sy x Sz blocks of shape [N/S + 2 Nh], one per device, and fills the
halos of interior block faces from exactly one neighbour per face (`jax.lax.ppermute`).  Here every block
is an ordinary jf solver whose inter-block faces have the type JF_BC_EXCHANGE:

  * `split_case`      cuts a `cases.Case` into sub-cases (host side, numpy only: no method arithmetic);
  * `MultiBlock`      drives all blocks from ONE process: the exchange is `jf_pull_face`, a kernel that reads
                      the neighbour's array directly (the same device here; a peer-mapped NVLink address on
                      a multi-GPU node) - on one GPU this is the emulation of the ranks as one launch
                      sequence over all ranks' data, used by the tests;
  * `RankBlock`       is the one-process-per-GPU form: `jf_pack_face` -> `torch.distributed` point-to-point
                      (NCCL over NVLink) -> `jf_unpack_face`, and an all-reduce(min) of dt.

The x -> y -> z order of the passes and their tangential extents are those of `jf_fill_halo`, so a
decomposed run reproduces the undivided one cell for cell (tests/test_gpu_decomp.py).
"""
import copy

import numpy as np

from . import cases

NH = cases.NH


def split_sizes(n, S):
    """Near-equal block sizes along one axis (the paper's blocks are equal: n divisible by S)."""
    q, r = divmod(n, S)
    sizes = [q + (1 if b < r else 0) for b in range(S)]
    if min(sizes) < 4:
        raise ValueError(f"blocks of {n} cells in {S} parts would have fewer than 4 cells")
    return sizes


def _tangential_axes(axis):
    return ((1, 2), (0, 2), (0, 1))[axis]          # (t1, t2) of the Dirichlet table prim[5][n_t2][n_t1]


class Part:
    """One block: its sub-case, block coordinates, interior offset in the global grid, and per face the
    rank of the neighbour (None on physical faces)."""

    def __init__(self, case, coords, lo, neighbours):
        self.case, self.coords, self.lo, self.neighbours = case, coords, lo, neighbours


def split_case(case, blocks):
    """Cut `case` into blocks[0] x blocks[1] x blocks[2] sub-cases; rank = (bz * Sy + by) * Sx + bx."""
    S = tuple(int(b) for b in blocks)
    faces = [np.asarray(f, dtype=np.float64) for f in (case.xf, case.yf, case.zf)]
    widths = [np.diff(f) for f in faces]
    sizes = [split_sizes(case.n[a], S[a]) for a in range(3)]
    offs = [np.concatenate(([0], np.cumsum(sz))) for sz in sizes]
    for f in range(6):
        if case.bc[f].type == cases.BC_DIRICHLET:
            for t in _tangential_axes(f // 2):
                if S[t] > 1:
                    raise ValueError("cannot split along an axis tangential to a Dirichlet face: its table is "
                                     "clamped at the block edge, which would change the edge halo cells")
    rank_of = lambda b: (b[2] * S[1] + b[1]) * S[0] + b[0]
    parts = []
    for bz in range(S[2]):
        for by in range(S[1]):
            for bx in range(S[0]):
                b = (bx, by, bz)
                lo = [int(offs[a][b[a]]) for a in range(3)]
                hi = [int(offs[a][b[a] + 1]) for a in range(3)]
                n = tuple(hi[a] - lo[a] for a in range(3))
                sub = copy.copy(case)
                sub.name = f"{case.name}@{bx}.{by}.{bz}"
                sub.n = n
                sub.xf, sub.yf, sub.zf = (faces[a][lo[a]:hi[a] + 1].copy() for a in range(3))
                U = cases.empty_state(n)
                U[:, NH:-NH, NH:-NH, NH:-NH] = case.U0[:, NH + lo[2]:NH + hi[2], NH + lo[1]:NH + hi[1], NH + lo[0]:NH + hi[0]]
                sub.U0 = U
                sub.bc, nbs = [], []
                for f in range(6):
                    a, side = f // 2, f % 2
                    N, g = case.n[a], case.bc[f]
                    at_edge = b[a] == (0 if side == 0 else S[a] - 1)
                    if at_edge and (g.type != cases.BC_PERIODIC or S[a] == 1):
                        fb = copy.copy(g)                    # physical face (or an unsplit periodic axis)
                        if g.type == cases.BC_DIRICHLET:
                            t1, t2 = _tangential_axes(a)
                            fb.dirichlet = np.ascontiguousarray(g.dirichlet[:, lo[t2]:hi[t2], lo[t1]:hi[t1]])
                        sub.bc.append(fb)
                        nbs.append(None)
                        continue
                    nb = list(b)
                    nb[a] = (b[a] + (-1 if side == 0 else 1)) % S[a]
                    # widths of the neighbour's three cells next to the face, nearest first (periodic wrap)
                    idx = [(lo[a] - m) % N for m in (1, 2, 3)] if side == 0 else [(hi[a] + m) % N for m in (0, 1, 2)]
                    # interior cut (no periodic wrap): hand over the neighbour's face coordinates, so that widths and
                    # centres of the halo cells are the undivided grid's own expressions, bit for bit
                    wrap = at_edge
                    nbf = None
                    if not wrap:
                        nbf = tuple(float(faces[a][lo[a] - m]) for m in (1, 2, 3)) if side == 0 else \
                            tuple(float(faces[a][hi[a] + m]) for m in (1, 2, 3))
                    sub.bc.append(cases.FaceBC(cases.BC_EXCHANGE, nb_width=tuple(float(widths[a][i]) for i in idx), nb_face=nbf))
                    nbs.append(rank_of(nb))
                parts.append(Part(sub, b, tuple(lo), nbs))
    return parts


def exchange_faces(case_bc, S, b, lo, hi, faces, widths, N):
    """Face BCs and neighbour ranks of block b = (bx, by, bz) of an S[0] x S[1] x S[2] cut: physical faces keep the
    case's BC (returned as None here: the caller copies it), faces between blocks become BC_EXCHANGE carrying the
    neighbour's geometry (face coordinates across an interior cut, cell widths across a periodic wrap)."""
    rank_of = lambda c: (c[2] * S[1] + c[1]) * S[0] + c[0]
    bcs, nbs = [], []
    for f in range(6):
        a, side = f // 2, f % 2
        at_edge = b[a] == (0 if side == 0 else S[a] - 1)
        if at_edge and (case_bc[f].type != cases.BC_PERIODIC or S[a] == 1):
            bcs.append(None)
            nbs.append(None)
            continue
        nb = list(b)
        nb[a] = (b[a] + (-1 if side == 0 else 1)) % S[a]
        idx = [(lo[a] - m) % N[a] for m in (1, 2, 3)] if side == 0 else [(hi[a] + m) % N[a] for m in (0, 1, 2)]
        nbf = None
        if not at_edge:
            nbf = tuple(float(faces[a][lo[a] - m]) for m in (1, 2, 3)) if side == 0 else \
                tuple(float(faces[a][hi[a] + m]) for m in (1, 2, 3))
        bcs.append(cases.FaceBC(cases.BC_EXCHANGE, nb_width=tuple(float(widths[a][i]) for i in idx), nb_face=nbf))
        nbs.append(rank_of(nb))
    return bcs, nbs


def tgv_part(n, S, rank):
    """Block `rank` of the weak-scaling decomposition bench: the Taylor-Green field (period 2 pi) on the box
    [0, 2 pi S[0]] x [0, 2 pi S[1]] x [0, 2 pi S[2]] cut into S[0] x S[1] x S[2] blocks of n^3 cells.  Only this
    rank's block is materialised (a 512^3 global state per rank would not be)."""
    S = tuple(int(v) for v in S)
    b = (rank % S[0], (rank // S[0]) % S[1], rank // (S[0] * S[1]))
    N = [n * S[a] for a in range(3)]
    faces = [cases.uniform_faces(0.0, 2.0 * np.pi * S[a], N[a]) for a in range(3)]
    widths = [np.diff(f) for f in faces]
    lo = [b[a] * n for a in range(3)]
    hi = [lo[a] + n for a in range(3)]
    sub = cases.tgv(n, faces=tuple(faces[a][lo[a]:hi[a] + 1].copy() for a in range(3)))
    bcs, nbs = exchange_faces(cases.periodic_bc(), S, b, lo, hi, faces, widths, N)
    sub.bc = [cases.FaceBC(cases.BC_PERIODIC) if x is None else x for x in bcs]
    sub.name = f"tgv{n}@{b[0]}.{b[1]}.{b[2]}of{S[0]}x{S[1]}x{S[2]}"
    return Part(sub, b, tuple(lo), nbs)


def gather_interior(case, parts, arrays):
    """Global padded array (halos zero) from the blocks' arrays [5, nz+6, ny+6, nx+6(, 2)]."""
    extra = arrays[0].shape[4:]
    nx, ny, nz = case.n
    out = np.zeros((5, nz + 2 * NH, ny + 2 * NH, nx + 2 * NH) + tuple(extra), dtype=arrays[0].dtype)
    for p, A in zip(parts, arrays):
        n, lo = p.case.n, p.lo
        out[:, NH + lo[2]:NH + lo[2] + n[2], NH + lo[1]:NH + lo[1] + n[1], NH + lo[0]:NH + lo[0] + n[0]] = \
            A[:, NH:-NH, NH:-NH, NH:-NH]
    return out


class MultiBlock:
    """All blocks of a decomposed case driven from one process, their arrays on ONE device (all launches on that
    device's current stream, which orders the blocks): inter-block halos by `jf_pull_face`, or pack -> unpack."""

    def __init__(self, case, blocks, dtype="f64", device="cuda:0", transport="pull"):
        from . import binding
        assert transport in ("pull", "pack")     # "pack": jf_pack_face on the neighbour -> jf_unpack_face here
        self.case, self.parts, self.transport = case, split_case(case, blocks), transport
        self.solvers = [binding.Solver(p.case, dtype, device) for p in self.parts]
        self.U = [s.state() for s in self.solvers]
        self._bufs = {}

    def fill_halos(self, ptrs):
        """Halo fill of the arrays at raw device pointers ptrs[rank], axis by axis (include/jf.h)."""
        for axis in range(3):
            for s, p in zip(self.solvers, ptrs):
                s.jf_fill_halo_axis(p, axis)
            for r, (s, part) in enumerate(zip(self.solvers, self.parts)):
                for side in (0, 1):
                    f = 2 * axis + side
                    nb = part.neighbours[f]
                    if nb is None:
                        continue
                    if self.transport == "pull":
                        s.jf_pull_face(ptrs[r], f, ptrs[nb], self.parts[nb].case.n)
                    else:                                # what the neighbour packs for its opposite face
                        sn = self.solvers[nb]
                        key = (nb, f ^ 1)
                        if key not in self._bufs:
                            self._bufs[key] = sn.torch.empty(sn.jf_face_elems(f ^ 1) * (2 if sn.dtype == "f64t" else 1),
                                                             dtype=sn.tdtype, device=sn.device)
                        buf = self._bufs[key]
                        sn.jf_pack_face(ptrs[nb], f ^ 1, buf)
                        s.jf_unpack_face(ptrs[r], f, buf)

    def jf_fill_halo(self):
        self.fill_halos([u.data_ptr() for u in self.U])

    def jf_rk3_step(self, dt):
        for stage in (1, 2, 3):
            self.fill_halos([s.jf_rk3_stage_input(u, stage) for s, u in zip(self.solvers, self.U)])
            for s, u in zip(self.solvers, self.U):
                s.jf_rk3_stage_advance(u, stage, dt)

    def jf_cfl_dt(self, cfl):
        """min over the blocks (the all-reduce(min) of the multi-rank form)."""
        dts = []
        for s, u in zip(self.solvers, self.U):
            st, dt = s.jf_cfl_dt(u, cfl)
            if st != 0:
                return st, float("nan")
            dts.append(dt)
        return 0, min(dts)

    def gather(self):
        return gather_interior(self.case, self.parts, [u.cpu().numpy() for u in self.U])


# ---------------------------------------------------------------- one block per rank (torch.distributed)
def exchange_axis(axis, neighbours, rank, pack, unpack, new_buffer, dist):
    """One axis of the inter-block halo exchange for this rank: pack the layers each neighbour needs,
    swap them point-to-point (the paper's `ppermute`: every rank sends to and receives from exactly one
    rank per face), unpack.  `pack(face, buf)`, `unpack(face, buf)`, `new_buffer(face)` are injected so that
    the host logic is testable on CPU tensors with the gloo backend (tests/test_decomp_cpu.py)."""
    # The neighbour across my face f fills ITS opposite face (f ^ 1) with what I pack for f.  Sends are posted
    # for side 0 then 1, receives for side 1 then 0: on a two-block periodic axis both messages go to the same
    # rank, and a transport that matches messages of a pair in order (NCCL) then pairs my first send (face
    # 2a) with the peer's first receive (its face 2a+1); tags say the same thing to transports that honour them.
    sends, recvs = [], []
    for side in (0, 1):
        f = 2 * axis + side
        if neighbours[f] is None:
            continue
        send = new_buffer(f)
        pack(f, send)
        sends.append((f, send))
    ops = [dist.P2POp(dist.isend, b, neighbours[f], tag=f) for f, b in sends]
    for side in (1, 0):
        f = 2 * axis + side
        if neighbours[f] is None:
            continue
        recv = new_buffer(f)
        ops.append(dist.P2POp(dist.irecv, recv, neighbours[f], tag=f ^ 1))
        recvs.append((f, recv))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    for f, recv in recvs:
        unpack(f, recv)


class RankBlock:
    """This rank's block of a decomposed case (one process per GPU; `torch.distributed` initialised by the
    caller, backend nccl): halos of inter-block faces by `jf_pack_face` -> point-to-point -> `jf_unpack_face`.
    The send / receive buffers of the six faces are allocated once.  Not measured on hardware: this environment
    has one GPU."""

    def __init__(self, case, blocks, dtype="f64", device=None, part=None):
        import torch
        import torch.distributed as dist
        from . import binding
        self.torch, self.dist = torch, dist
        self.rank, world = dist.get_rank(), dist.get_world_size()
        if part is None:
            parts = split_case(case, blocks)
            if len(parts) != world:
                raise ValueError(f"{len(parts)} blocks for {world} ranks")
            part = parts[self.rank]
        self.part = part
        device = device or f"cuda:{torch.cuda.current_device()}"
        self.solver = binding.Solver(self.part.case, dtype, device)
        self.U = self.solver.state()
        self._bufs = {}
        self._turn = {}

    def _new_buffer(self, face):
        # two persistent buffers per face, handed out alternately: exchange_axis asks for the send buffer of a
        # face first and for its receive buffer second
        if face not in self._bufs:
            n = self.solver.jf_face_elems(face) * (2 if self.solver.dtype == "f64t" else 1)
            self._bufs[face] = [self.torch.empty(n, dtype=self.solver.tdtype, device=self.solver.device) for _ in range(2)]
            self._turn[face] = 0
        b = self._bufs[face][self._turn[face]]
        self._turn[face] ^= 1
        return b

    def exchange_bytes_per_step(self):
        """Bytes this rank sends per RK3 step: 3 stages x its exchange faces x 3 layers x 5 variables."""
        esz = {"f64": 8, "f32": 4, "f64t": 16}[self.solver.dtype]
        return 3 * sum(self.solver.jf_face_elems(f) * esz for f in range(6) if self.part.neighbours[f] is not None)

    def fill_halos(self, ptr):
        s = self.solver
        for axis in range(3):
            s.jf_fill_halo_axis(ptr, axis)
            exchange_axis(axis, self.part.neighbours, self.rank, lambda f, b: s.jf_pack_face(ptr, f, b),
                          lambda f, b: s.jf_unpack_face(ptr, f, b), self._new_buffer, self.dist)

    def jf_rk3_step(self, dt):
        for stage in (1, 2, 3):
            self.fill_halos(self.solver.jf_rk3_stage_input(self.U, stage))
            self.solver.jf_rk3_stage_advance(self.U, stage, dt)

    def jf_cfl_dt(self, cfl):
        st, dt = self.solver.jf_cfl_dt(self.U, cfl)
        return reduce_dt(st, dt, self.torch, self.dist, self.solver.device)


def reduce_dt(st, dt, torch, dist, device=None):
    """All ranks get the same (status, dt): status = MAX over ranks, dt = MIN over ranks with +inf standing in for a
    rank whose reduction flagged an inadmissible state (a NaN fed to a MIN all-reduce is not reliably propagated);
    dt is NaN whenever the status is not 0, so that no rank steps on while another has failed."""
    t = torch.tensor([float("inf") if st != 0 else dt, -float(st)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    st_all = int(round(-float(t[1])))
    return st_all, (float("nan") if st_all != 0 else float(t[0]))
