"""Multi-GPU slab decomposition of the explicit step: host logic.

The body is cut into `world` slabs along one coordinate axis.  Rank r OWNS the nodes of slab r and also holds a HALO:
every node within 2 delta of its slab along that axis.  One explicit step on the local body (owned + halo) with the
unmodified single-GPU library gives the exact u^{n+1} of the owned nodes:

    f_i (i owned) needs theta_j, m_j of every j within delta of i       (Eq. 2.1 / 2.2)
    theta_j, m_j need the complete family of j: every node within delta of j, i.e. within 2 delta of the slab,
    with its u^n (Eq. 1.6, Eq. 1.9); bond status is decided from u at both ends (Eq. 1.30), identically on every
    rank that holds the bond.

The halo nodes' own u^{n+1} is wrong (their families are cut by the artificial boundary) and is overwritten after
every step with the owners' values: ONE neighbour exchange of dim doubles per halo node and step -- the path's only
data-path communication (point-to-point send/recv between slab neighbours; NCCL over NVLink on GPUs, gloo in the CPU
test).  Nothing else crosses ranks: bond masks need no exchange, the damage of an owned node is local.

This module holds the partition (index lists) and the step loop; the per-rank stepper and the transport are passed
in, so the same code runs on pd.Sim + torch.distributed (GPUs), on several pd.Sim handles of one GPU with an
in-process exchange (tests/test_gpu_parity.py), and on the CPU oracle + gloo (tests/test_replicas_gloo.py).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class SlabPart:
    rank: int
    world: int
    local: np.ndarray                 # global ids of the local nodes (owned + halo), ascending
    owned_local: np.ndarray           # positions in `local` of the owned nodes
    send: dict = field(default_factory=dict)   # peer -> positions in `local` of the owned nodes the peer holds as halo
    recv: dict = field(default_factory=dict)   # peer -> positions in `local` of the halo nodes the peer owns
    precut_local: np.ndarray = None   # pre-cut pairs with both ends local, in local numbering


def partition(coords: np.ndarray, horizon: float, world: int, axis: int | None = None, precut=None):
    """SlabPart of every rank.  Cuts at equal node counts along `axis` (default: the longest extent); cut planes sit
    half-way between distinct coordinates so that no node lies on a plane."""
    x = np.asarray(coords, dtype=np.float64)
    n = len(x)
    if axis is None:
        axis = int(np.argmax(x.max(0) - x.min(0)))
    c = x[:, axis]
    order = np.argsort(c, kind="stable")
    cuts = [-np.inf]
    for r in range(1, world):
        k = (n * r) // world
        lo, hi = c[order[k - 1]], c[order[k]]
        while lo == hi and k < n - 1:      # do not split a layer of equal coordinates
            k += 1
            lo, hi = c[order[k - 1]], c[order[k]]
        cuts.append(0.5 * (lo + hi))
    cuts.append(np.inf)
    owner = np.searchsorted(np.asarray(cuts[1:-1]), c, side="right") if world > 1 else np.zeros(n, np.int64)
    halo = 2.0 * horizon * (1.0 + 1e-12)
    local_sets = []
    for r in range(world):
        lo, hi = cuts[r] - halo, cuts[r + 1] + halo
        local_sets.append(np.nonzero((c >= lo) & (c <= hi))[0])
    parts = []
    pre = None if precut is None or len(precut) == 0 else np.asarray(precut, np.int64).reshape(-1, 2)
    for r in range(world):
        loc = local_sets[r]
        g2l = -np.ones(n, np.int64)
        g2l[loc] = np.arange(len(loc))
        p = SlabPart(r, world, loc, np.nonzero(owner[loc] == r)[0])
        for s in range(world):
            if s == r:
                continue
            mine_there = loc[(owner[loc] == r) & np.isin(loc, local_sets[s])]     # my owned nodes that s holds
            theirs_here = loc[owner[loc] == s]                                    # s's owned nodes that I hold
            if len(mine_there):
                p.send[s] = g2l[mine_there]
            if len(theirs_here):
                p.recv[s] = g2l[theirs_here]
        if pre is not None:
            keep = (g2l[pre[:, 0]] >= 0) & (g2l[pre[:, 1]] >= 0)
            p.precut_local = np.stack([g2l[pre[keep, 0]], g2l[pre[keep, 1]]], 1).astype(np.int32)
        else:
            p.precut_local = np.zeros((0, 2), np.int32)
        parts.append(p)
    return parts, axis


def local_workload(wl, part: SlabPart):
    """the rank's share of a workloads.Workload (same scalars; arrays restricted to the local nodes)"""
    import dataclasses
    loc = part.local
    return dataclasses.replace(wl, coords=wl.coords[loc].copy(), volumes=wl.volumes[loc].copy(), flags=wl.flags[loc].copy(),
                               value=wl.value[loc].copy(), u0=wl.u0[loc].copy(), v0=wl.v0[loc].copy(),
                               precut=part.precut_local)


class SlabRunner:
    """The step loop of one rank.  `stepper` offers step(n), gather_u(local_idx) -> array/tensor (len, dim) and
    scatter_u(local_idx, values); `transport` offers exchange(rank, sends: {peer: payload}, recv_peers) -> {peer: payload}."""

    def __init__(self, part: SlabPart, stepper, transport):
        self.part, self.stepper, self.transport = part, stepper, transport

    def step(self, nsteps: int = 1):
        p = self.part
        for _ in range(nsteps):
            self.stepper.step(1)
            if p.world == 1:
                continue
            sends = {peer: self.stepper.gather_u(idx) for peer, idx in p.send.items()}
            got = self.transport.exchange(p.rank, sends, sorted(p.recv))
            for peer, idx in p.recv.items():
                self.stepper.scatter_u(idx, got[peer])


class TorchDistTransport:
    """point-to-point exchange between slab neighbours over torch.distributed (nccl on GPUs, gloo on CPU)"""

    def __init__(self, recv_shapes, dtype=None, device="cpu"):
        import torch
        self.torch, self.recv_shapes, self.device = torch, recv_shapes, device
        self.dtype = dtype or torch.float64

    def exchange(self, rank, sends, recv_peers):
        import torch.distributed as dist
        t = self.torch
        bufs = {p: t.empty(self.recv_shapes[p], dtype=self.dtype, device=self.device) for p in recv_peers}
        ops = []
        for p in sorted(set(sends) | set(recv_peers)):
            if p in sends:
                payload = sends[p] if t.is_tensor(sends[p]) else t.from_numpy(np.ascontiguousarray(sends[p]))
                ops.append(dist.P2POp(dist.isend, payload.to(self.device).contiguous(), p))
            if p in bufs:
                ops.append(dist.P2POp(dist.irecv, bufs[p], p))
        for w in dist.batch_isend_irecv(ops) if ops else []:
            w.wait()
        return bufs


class InProcessTransport:
    """all ranks live in one process (several handles on one GPU, or the CPU oracle): rank r posts its sends, the
    exchange completes when every rank has posted -- driven by run_lockstep below"""

    def __init__(self, world):
        self.world, self.box = world, {}

    def post(self, rank, sends):
        for peer, payload in sends.items():
            self.box[(rank, peer)] = payload

    def collect(self, rank, recv_peers):
        return {p: self.box.pop((p, rank)) for p in recv_peers}


def run_lockstep(parts, steppers, nsteps):
    """advance all slabs of one process in lockstep (no rank waits on another: step all, post all, deliver all)"""
    tr = InProcessTransport(len(parts))
    for _ in range(nsteps):
        for st in steppers:
            st.step(1)
        for p, st in zip(parts, steppers):
            tr.post(p.rank, {peer: st.gather_u(idx) for peer, idx in p.send.items()})
        for p, st in zip(parts, steppers):
            got = tr.collect(p.rank, sorted(p.recv))
            for peer, idx in p.recv.items():
                st.scatter_u(idx, got[peer])


def assemble_owned(parts, values_per_rank, n, width):
    """global array from the owned rows of every rank's local array"""
    out = np.zeros((n, width)) if width else np.zeros(n)
    for p, v in zip(parts, values_per_rank):
        out[p.local[p.owned_local]] = np.asarray(v)[p.owned_local]
    return out
