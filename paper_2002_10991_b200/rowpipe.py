"""the row-pipelined multi-GPU variant of the back-transformation (PAPER.md:136-138:
the rows of an eigenvector are spread over a process column and a step exchanges at most ``nbw`` rows with
the neighbour).  Host-side logic only -- partition, schedule, message plumbing; every arithmetic step is
the library's row-block call ``elpa2_trans_ev_tridi_to_band_rows_{d,z}`` (include/elpa2_bt.h).

Rank ``r`` of ``R`` owns the rows ``[bounds[r], bounds[r+1])`` of its columns (rank 0 the top of the matrix)
and keeps them in a local buffer followed by the ``nbw`` halo rows of the rank below.  Chains run in
chain-major order (R5); within a chain the window travels from the bottom of the matrix to the
top, i.e. from rank R-1 to rank 0, so chain ``k`` on rank ``r`` overlaps with chain ``k+1`` on rank ``r+1``:
a pipeline with one hand-over of ``nbw`` rows per chain and boundary in each direction,

    halo(k):    rank r+1 -> r   the first nbw rows of r+1 after its part of chain k (r continues on them)
    return(k):  rank r -> r+1   the same rows once r's blocks of chain k have made them final for chain k

Per chain a rank runs its rows in two calls -- the lower part first, then its first ``nbw`` rows (the
upper part) -- so that it can start chain ``k+1`` before ``return(k)`` has come back.  The bounds follow
the work: row ``i`` is touched by about ``i / nbw`` chains, so equal work means equal ``bounds**2``
differences (``partition_rows``).

``schedule`` is pure Python and is what the tests pin (gloo, world size 2 and 3, against the oracle);
``run`` executes it with ``torch.distributed`` point-to-point calls (NCCL over NVLink on GPUs) or, with
``LocalExchange``, as R emulated ranks on ONE device in a dependency-respecting order -- the form the GPU
test compares bit for bit with the single call.
"""
from __future__ import annotations

import math
from dataclasses import dataclass


def partition_rows(N: int, world: int, nbw: int) -> list[int]:
    """Row bounds ``[0 = b_0 <= b_1 <= ... <= b_R = N]``: multiples of 8, every rank at least ``nbw`` rows,
    equal-work split ``b_r ~ N sqrt(r / R)``.  Raises if N is too small for ``world`` ranks."""
    if world < 1 or nbw < 8 or nbw % 8:
        raise ValueError("bad arguments")
    if world == 1:
        return [0, N]
    if N < world * nbw:
        raise ValueError(f"N = {N} rows cannot give {world} ranks {nbw} rows each")
    b = [0]
    for r in range(1, world):
        x = int(round(N * math.sqrt(r / world) / 8.0)) * 8
        x = max(x, b[-1] + nbw)                       # at least nbw rows for rank r-1 ...
        x = min(x, ((N - (world - r) * nbw) // 8) * 8)  # ... and for every rank below
        b.append(x)
    b.append(N)
    for r in range(world):
        if b[r + 1] - b[r] < nbw:
            raise ValueError(f"N = {N} rows cannot give {world} ranks {nbw} rows each")
    return b


def chains_of(N: int, nbw: int, bounds: list[int], r: int) -> int:
    """Number of chains (k = 0 .. Kp-1) that have a block whose first row lies in rank r's rows."""
    K0 = (N - 2 + nbw) // nbw if N >= 2 else 0
    if bounds[r + 1] >= N:
        return K0
    b_top = bounds[r + 1] // 8 - 1
    return min(K0, b_top // (nbw // 8) + 1)


@dataclass(frozen=True)
class Op:
    """One step of a rank's program.  kind: 'recv' / 'send' (peer, tag; local rows [lo, lo + n)) or 'apply'
    (chain k; the call's row0, nown and the local row offset ``lo`` of row0)."""
    kind: str
    k: int
    peer: int = -1
    tag: str = ""
    lo: int = 0
    n: int = 0
    row0: int = 0
    nown: int = 0


def schedule(N: int, nbw: int, bounds: list[int], r: int) -> list[Op]:
    """The program of rank ``r`` (see the module docstring).  Local row ``i`` is global row ``bounds[r] + i``."""
    R = len(bounds) - 1
    R0, R1 = bounds[r], bounds[r + 1]
    nown = R1 - R0
    Kp = chains_of(N, nbw, bounds, r)
    Kup = chains_of(N, nbw, bounds, r - 1) if r > 0 else 0        # chains of the rank above
    split = nbw if r > 0 else 0                                    # rank 0 has no upper neighbour: one call
    # the halo rows are final for chain k once every reflector that reaches them has been applied: after the
    # lower part if the upper part's reflectors (first rows < R0 + nbw) end above the halo, else after both
    early_return = nown >= 2 * nbw or split == 0
    ops: list[Op] = []
    for k in range(Kp):
        if r < R - 1:
            ops.append(Op("recv", k, peer=r + 1, tag="halo", lo=nown, n=nbw))
        if nown - split > 0:
            ops.append(Op("apply", k, lo=split, row0=R0 + split, nown=nown - split))
        if r < R - 1 and early_return:
            ops.append(Op("send", k, peer=r + 1, tag="return", lo=nown, n=nbw))
        if r > 0:
            if k >= 1 and k - 1 < Kup:
                ops.append(Op("recv", k - 1, peer=r - 1, tag="return", lo=0, n=nbw))
            ops.append(Op("apply", k, lo=0, row0=R0, nown=split))
            if r < R - 1 and not early_return:
                ops.append(Op("send", k, peer=r + 1, tag="return", lo=nown, n=nbw))
            if k < Kup:
                ops.append(Op("send", k, peer=r - 1, tag="halo", lo=0, n=nbw))
    if r > 0 and Kup == Kp and Kp >= 1:
        ops.append(Op("recv", Kp - 1, peer=r - 1, tag="return", lo=0, n=nbw))
    return ops


def local_rows(N: int, nbw: int, bounds: list[int], r: int) -> int:
    """Rows of rank r's buffer: its own rows plus the halo (the first nbw rows of the rank below)."""
    R = len(bounds) - 1
    return (bounds[r + 1] - bounds[r]) + (nbw if r < R - 1 else 0)


class LocalExchange:
    """R emulated ranks in one process: a 'send' parks a copy of the rows in a mailbox, the matching 'recv'
    takes it.  ``run_emulated`` steps the ranks in an order in which every recv finds its message."""

    def __init__(self):
        self.box = {}

    def send(self, src, dst, tag, k, rows):
        self.box[(src, dst, tag, k)] = rows.clone() if hasattr(rows, "clone") else rows.copy()

    def recv(self, src, dst, tag, k, rows):
        msg = self.box.pop((src, dst, tag, k))
        if hasattr(rows, "copy_"):
            rows.copy_(msg)
        else:
            rows[...] = msg


def run_emulated(N, nbw, bounds, bufs, apply_fn, exchange=None):
    """Execute all ranks' programs on local buffers ``bufs[r]`` ((local_rows, ncols), updated in place):
    round-robin over the ranks, each advancing until it reaches a recv whose message has not been sent.
    ``apply_fn(r, buf, op)`` applies one 'apply' op.  Raises on deadlock (a schedule bug)."""
    R = len(bounds) - 1
    ex = exchange or LocalExchange()
    progs = [schedule(N, nbw, bounds, r) for r in range(R)]
    pc = [0] * R
    while any(pc[r] < len(progs[r]) for r in range(R)):
        moved = False
        for r in range(R - 1, -1, -1):
            while pc[r] < len(progs[r]):
                op = progs[r][pc[r]]
                if op.kind == "recv":
                    if (op.peer, r, op.tag, op.k) not in ex.box:
                        break
                    ex.recv(op.peer, r, op.tag, op.k, bufs[r][op.lo:op.lo + op.n])
                elif op.kind == "send":
                    ex.send(r, op.peer, op.tag, op.k, bufs[r][op.lo:op.lo + op.n])
                else:
                    apply_fn(r, bufs[r], op)
                pc[r] += 1
                moved = True
        if not moved:
            raise RuntimeError("row pipeline deadlocked: " + repr([(r, progs[r][pc[r]]) for r in range(R) if pc[r] < len(progs[r])]))
    if ex.box:
        raise RuntimeError(f"row pipeline left {len(ex.box)} undelivered messages")


def device_apply(N, nbw, hh_v, hh_tau, stream=None):
    """``apply_fn`` for CUDA buffers: the library's row-block call on the rows ``op.lo ..`` of the buffer."""
    from . import binding

    def fn(r, buf, op):
        binding.trans_ev_tridi_to_band_rows(N, nbw, hh_v, hh_tau, buf[op.lo:], op.row0, op.nown, op.k, op.k + 1, stream=stream)

    return fn


def run(N, nbw, bounds, q_local, dist, apply_fn):
    """Rank ``dist.get_rank()`` of a ``len(bounds) - 1``-rank row pipeline: ``q_local`` is this rank's
    column-major buffer (``local_rows`` x ncols: own rows + halo rows, halo contents arbitrary on entry);
    on return the own rows hold the result.  ``apply_fn``: ``device_apply(...)`` on GPUs.  Messages are
    ``nbw x ncols`` blocks sent with ``dist.send`` / ``dist.recv`` (NCCL: stream-ordered device-to-device
    copies over NVLink; gloo in the CPU tests); between two neighbours both sides issue them in the same
    order, so no tags are needed and no cycle of waits exists."""
    import torch

    r = dist.get_rank()
    ncols = q_local.shape[1]
    stage = torch.empty((ncols, nbw), dtype=q_local.dtype, device=q_local.device)   # contiguous message buffer
    for op in schedule(N, nbw, bounds, r):
        rows = q_local[op.lo:op.lo + op.n]
        if op.kind == "recv":
            dist.recv(stage, src=op.peer)
            rows.copy_(stage.t())
        elif op.kind == "send":
            stage.copy_(rows.t())
            dist.send(stage, dst=op.peer)
        else:
            apply_fn(r, q_local, op)
