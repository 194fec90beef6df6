"""Multi-GPU plumbing of the bench: the path shards over independent problems -- one
inverse-design problem per rank, no data-path collective.  This module holds the only host logic the N > 1
run adds: which problem a rank works on and how the per-rank times combine into the whole-job figure.
It has none of the method's arithmetic."""
from __future__ import annotations

import torch
import torch.distributed as dist


def problem_seed(base_seed: int, rank: int) -> int:
    """Every rank draws its own design (rho) from its own seed; rank 0 is the single-GPU problem."""
    return base_seed + rank


def max_over_ranks(ms_local: float, device=None) -> float:
    """Device time of the slowest rank (the job is as slow as its slowest problem)."""
    t = torch.tensor([ms_local], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(cells_steps_per_rank: int, reps: int, ms_max: float, world: int) -> float:
    """Mcells/s summed over ranks: every rank processed cells_steps_per_rank * reps cell updates in ms_max."""
    return world * cells_steps_per_rank * reps / (ms_max * 1e-3) / 1e6


# --------------------------------------------------------------------------------------------------------------
# Domain decomposition of ONE grid into z slabs (include/fdtd.h "Domain decomposition";
# PAPER.md L116-118).  Host logic only: which planes a rank holds, how the inputs are cut, which planes travel.
# --------------------------------------------------------------------------------------------------------------
from dataclasses import dataclass, replace as _replace
from typing import List, Optional, Sequence, Tuple


@dataclass(frozen=True)
class ZSlab:
    """Planes of rank `rank` of `world`: owns [k_lo, k_hi), stores [z_offset, z_offset + nz) (one ghost plane per cut)."""
    rank: int
    world: int
    nz_global: int
    k_lo: int
    k_hi: int

    @property
    def ghost_lo(self) -> int:
        return 0 if self.k_lo == 0 else 1

    @property
    def ghost_hi(self) -> int:
        return 0 if self.k_hi == self.nz_global else 1

    @property
    def z_offset(self) -> int:
        return self.k_lo - self.ghost_lo

    @property
    def nz(self) -> int:
        return self.k_hi - self.k_lo + self.ghost_lo + self.ghost_hi

    def grid_kwargs(self) -> dict:
        return dict(nz=self.nz, z_global=self.nz_global, z_offset=self.z_offset, z_ghost_lo=self.ghost_lo, z_ghost_hi=self.ghost_hi)

    def local_planes(self) -> slice:
        return slice(self.z_offset, self.z_offset + self.nz)

    def owned_local(self) -> slice:
        """The owned planes in local indices."""
        return slice(self.ghost_lo, self.nz - self.ghost_hi)


def z_slabs(nz_global: int, world: int, pml_cells: int = 0, cuts: Optional[Sequence[int]] = None) -> List[ZSlab]:
    """Cuts [0, nz_global) into `world` slabs of (nearly) equal plane counts, or at the given cut planes.  Every slab
    must own at least one plane of the interior [pml_cells, nz_global - pml_cells)."""
    if cuts is None:
        cuts = [round(nz_global * r / world) for r in range(1, world)]
    edges = [0, *cuts, nz_global]
    if len(edges) != world + 1 or any(b <= a for a, b in zip(edges, edges[1:])):
        raise ValueError(f"bad cuts {cuts} for {world} slabs of {nz_global} planes")
    slabs = [ZSlab(r, world, nz_global, edges[r], edges[r + 1]) for r in range(world)]
    for s in slabs:
        if min(s.k_hi, nz_global - pml_cells) <= max(s.k_lo, pml_cells):
            raise ValueError(f"slab {s.rank} owns no interior plane")
    return slabs


def _clip_box(lo, hi, k0: int, k1: int, shift: int):
    """Box (lo, hi) clipped to global planes [k0, k1) and shifted to local plane indices; None if empty."""
    a, b = max(lo[2], k0), min(hi[2], k1)
    if b <= a:
        return None
    return (lo[0], lo[1], a - shift), (hi[0], hi[1], b - shift), (a - lo[2], b - lo[2])


def local_sources(sources, slab: ZSlab):
    """Sources clipped to the local planes (ghosts included: the E replica on the ghost plane above needs them)."""
    out = []
    for s in sources:
        c = _clip_box(s.lo, s.hi, slab.z_offset, slab.z_offset + slab.nz, slab.z_offset)
        if c is None:
            continue
        lo, hi, (a, b) = c
        prof = None if s.profile is None else s.profile[a:b]
        out.append(_replace(s, lo=lo, hi=hi, profile=prof))
    return out


def local_detectors(detectors, slab: ZSlab, with_ghosts: bool):
    """[(index of the global detector, local detector, slice of its box planes)]: clipped to the owned planes
    (forward) or to all local planes (backward: the cotangent injection must reach the ghost planes too)."""
    k0, k1 = (slab.z_offset, slab.z_offset + slab.nz) if with_ghosts else (slab.k_lo, slab.k_hi)
    out = []
    for idx, d in enumerate(detectors):
        c = _clip_box(d.lo, d.hi, k0, k1, slab.z_offset)
        if c is None:
            continue
        lo, hi, (a, b) = c
        out.append((idx, _replace(d, lo=lo, hi=hi), slice(a, b)))
    return out


def exchange_halos_dist(slab: ZSlab, send_down, send_up, recv_below, recv_above, group=None):
    """One halo exchange over torch.distributed point-to-point (NCCL on GPU tensors, gloo on CPU tensors):
    my lowest owned plane goes to rank-1 (its ghost above), my highest owned plane to rank+1 (its ghost below)."""
    ops = []
    if slab.ghost_lo:
        ops.append(dist.P2POp(dist.isend, send_down, slab.rank - 1, group))
        ops.append(dist.P2POp(dist.irecv, recv_below, slab.rank - 1, group))
    if slab.ghost_hi:
        ops.append(dist.P2POp(dist.isend, send_up, slab.rank + 1, group))
        ops.append(dist.P2POp(dist.irecv, recv_above, slab.rank + 1, group))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()


class SlabRunner:
    """One z slab of a workload on the current CUDA device: the local grid, the local slices of the inputs and the halo
    buffers.  Marshalling only -- every step runs in the library (fdtd_forward_range / fdtd_backward_range /
    fdtd_halo_export / fdtd_halo_import)."""

    def __init__(self, B, w, slab: ZSlab, n_total: int, record: int = 1, path=None, flags: int = 0):
        import numpy as np
        self.B, self.w, self.slab, self.n_total = B, w, slab, n_total
        t = self.torch = torch
        kw = w.grid_kwargs()
        kw.update(slab.grid_kwargs())
        kw.update(max_steps=n_total, record=record if w.pml_cells > 0 else 0, flags=flags)
        if path is not None:
            kw.update(path=path)
        self.grid = B.Grid(**kw)
        zs = slab.local_planes()
        self.ie = t.as_tensor(np.ascontiguousarray(w.inv_eps[zs])).cuda()
        im = w.meta.get("inv_mu")
        self.im = None if im is None else t.as_tensor(np.ascontiguousarray(im[zs])).cuda()
        self.fields = t.zeros((6, slab.nz, w.ny, w.nx), dtype=t.float32, device="cuda")
        self.sources = local_sources(w.sources, slab)
        self.det_fwd = local_detectors(w.detectors, slab, with_ghosts=False)
        self.det_bwd = local_detectors(w.detectors, slab, with_ghosts=True)
        self.phasors = [t.zeros(d.phasor_shape, dtype=t.float32, device="cuda") for _, d, _ in self.det_fwd]
        g = self.grid
        self.sarr, self.ns, self._k1 = g.marshal_sources(self.sources)
        self.darr, self.nd, self._k2 = g.marshal_detectors([d for _, d, _ in self.det_fwd], self.phasors)
        self.darr_b, self.nd_b, self._k3 = g.marshal_detectors([d for _, d, _ in self.det_bwd], None)
        plane = (3, w.ny, w.nx)
        self.send_down, self.send_up = t.empty(plane, device="cuda"), t.empty(plane, device="cuda")
        self.recv_below, self.recv_above = t.empty(plane, device="cuda"), t.empty(plane, device="cuda")
        self.grad = self.lam0 = self._cot = self._dLf = None
        self.want_grad = True          # False: the reverse steps are adjoint steps only (no gradient, nothing reconstructed)

    def close(self):
        self.grid.close()

    # ---- forward ------------------------------------------------------------------------------------------
    def forward_steps(self, n_begin: int, n_end: int):
        self.B.fdtd_forward_range(self.grid.h, self.fields, self.ie, self.im, self.sarr, self.ns, self.darr, self.nd,
                                  n_begin, n_end, self.n_total, self.grid.stream())

    def export_halos(self, which: int, n: int):
        B, g = self.B, self.grid
        if self.slab.ghost_lo:
            B.fdtd_halo_export(g.h, self.fields, which, n, 0, self.send_down, g.stream())
        if self.slab.ghost_hi:
            B.fdtd_halo_export(g.h, self.fields, which, n, 1, self.send_up, g.stream())

    def import_halos(self, which: int, n: int, from_below=None, from_above=None):
        B, g = self.B, self.grid
        if self.slab.ghost_lo:
            B.fdtd_halo_import(g.h, self.fields, which, n, 0, self.recv_below if from_below is None else from_below, g.stream())
        if self.slab.ghost_hi:
            B.fdtd_halo_import(g.h, self.fields, which, n, 1, self.recv_above if from_above is None else from_above, g.stream())

    # ---- peer stores: the step kernel writes the neighbour's ghost planes itself (include/fdtd.h "Peer stores") ----
    def volumes(self, which: int):
        """Device addresses of my two ping-pong volumes (which = 0 fields, 1 cotangents)."""
        return self.B.fdtd_halo_volumes(self.grid.h, self.fields, which)

    def attach(self, which: int, side: int, peer_vols, peer_nz: int):
        self.B.fdtd_halo_attach(self.grid.h, which, side, peer_vols[0], peer_vols[1], peer_nz)

    def flags(self, which: int) -> int:
        """Device address of my two ordering flags (include/fdtd.h "Device-side ordering")."""
        return self.B.fdtd_halo_flags(self.grid.h, which)

    def attach_flags(self, which: int, side: int, peer_flags):
        self.B.fdtd_halo_attach_flags(self.grid.h, which, side, peer_flags)

    def detach(self, which: int):
        for side in (0, 1):
            self.B.fdtd_halo_attach(self.grid.h, which, side, None, None, 0)

    # ---- backward -----------------------------------------------------------------------------------------
    def set_cotangents(self, dL_dphasor_global=None, dL_dfields_global=None):
        """Cotangents given on the GLOBAL boxes / volume (device tensors); this slab takes its planes, ghosts included."""
        import ctypes as C
        t = self.torch
        self._cot_keep = []
        cot = (C.c_void_p * max(self.nd_b, 1))()
        for q, (idx, d, sl) in enumerate(self.det_bwd):
            G = None if dL_dphasor_global is None else dL_dphasor_global[idx]
            if G is not None:
                G = G[:, :, sl].contiguous()
                self._cot_keep.append(G)
                cot[q] = G.data_ptr()
        self._cot = cot
        self._dLf = None if dL_dfields_global is None else dL_dfields_global[:, self.slab.local_planes()].contiguous()
        self.grad = t.empty((self.slab.nz, self.w.ny, self.w.nx), dtype=t.float32, device="cuda")
        self.lam0 = t.empty((6, self.slab.nz, self.w.ny, self.w.nx), dtype=t.float32, device="cuda")

    def backward_steps(self, n_hi: int, n_lo: int):
        self.B.fdtd_backward_range(self.grid.h, self.fields, self.ie, self.im, self.sarr, self.ns, self.darr_b, self.nd_b,
                                   self._cot, self._dLf, n_hi, n_lo, self.n_total, self.grad if self.want_grad else None,
                                   self.lam0, self.grid.stream())


def attach_neighbours_local(runners: List["SlabRunner"], which: int, flags: bool = False):
    """Slabs of one process: every runner gets its neighbours' volumes (plain device pointers) and, with flags = True,
    their ordering flags."""
    vols = [r.volumes(which) for r in runners]
    fl = [r.flags(which) for r in runners] if flags else None
    for q, r in enumerate(runners):
        for side, nb, has in ((0, q - 1, r.slab.ghost_lo), (1, q + 1, r.slab.ghost_hi)):
            if has:
                r.attach(which, side, vols[nb], runners[nb].slab.nz)
                if flags:
                    r.attach_flags(which, side, fl[nb])


def run_slabs_lockstep(runners: List["SlabRunner"], n_total: int, direction: str = "forward", peer: bool = False):
    """Advances the slabs of one process in lock step, one exchange per step (the single-device form of the protocol
    of include/fdtd.h; across processes every rank runs the same loop with exchange_halos_dist in the middle).
    peer = True: no exchange at all -- the step kernels store their boundary planes into the neighbours' volumes, and the
    one stream all slabs share orders step n of every slab before step n+1 of any.  peer = "flags": the same with the
    device-side ordering kernels in the stream as well (every wait finds its flag already set: on one device the slabs
    cannot run side by side, see include/fdtd.h)."""
    which = 0 if direction == "forward" else 1
    if peer:
        attach_neighbours_local(runners, which, flags=(peer == "flags"))
        try:
            for n in (range(n_total) if direction == "forward" else range(n_total - 1, -1, -1)):
                for r in runners:
                    r.forward_steps(n, n + 1) if direction == "forward" else r.backward_steps(n + 1, n)
        finally:
            for r in runners:
                r.detach(which)
        return

    def swap(which, n):
        for r in runners:
            r.export_halos(which, n)
        for q, r in enumerate(runners):
            r.import_halos(which, n, from_below=runners[q - 1].send_up if r.slab.ghost_lo else None,
                           from_above=runners[q + 1].send_down if r.slab.ghost_hi else None)
    if direction == "forward":
        for n in range(n_total):
            for r in runners:
                r.forward_steps(n, n + 1)
            if n + 1 < n_total:
                swap(0, n + 1)
    else:
        for n in range(n_total - 1, -1, -1):
            for r in runners:
                r.backward_steps(n + 1, n)
            if n > 0:
                swap(1, n)


class PeerLinks:
    """One rank's view of its neighbours' volumes in a torch.distributed job: every rank publishes the CUDA IPC handles of
    its two ping-pong volumes (fdtd_ipc_export), opens its neighbours' (fdtd_ipc_open: plain stores over NVLink when the
    neighbour is another GPU) and attaches them (fdtd_halo_attach).  Host logic only."""

    def __init__(self, runner: "SlabRunner", which: int, group=None, flags: bool = False):
        B, slab = runner.B, runner.slab
        self.runner, self.which, self.opened, self.flags = runner, which, [], flags
        if slab.world == 1:                                  # the whole grid on one rank: no neighbour, nothing to map
            return
        mine = [B.fdtd_ipc_export(v) for v in runner.volumes(which)]
        if flags:
            mine.append(B.fdtd_ipc_export(runner.flags(which)))
        table = [None] * slab.world
        dist.all_gather_object(table, (slab.nz, mine), group=group)
        for side, nb in ((0, slab.rank - 1), (1, slab.rank + 1)):
            if not (slab.ghost_lo if side == 0 else slab.ghost_hi):
                continue
            nz_nb, handles = table[nb]
            ptrs = [B.fdtd_ipc_open(h, off) for h, off in handles]
            self.opened += [(p, off) for p, (_, off) in zip(ptrs, handles)]
            runner.attach(which, side, ptrs[:2], nz_nb)
            if flags:
                runner.attach_flags(which, side, ptrs[2])

    def close(self):
        self.runner.detach(self.which)
        for p, off in self.opened:
            self.runner.B.fdtd_ipc_close(p, off)
        self.opened = []


def neighbour_tokens(slab: ZSlab, token, scratch, group=None):
    """The ordering that is left of the exchange with peer stores: a one-element message to and from every neighbour,
    enqueued behind this rank's step (stream-ordered over NCCL; blocking over gloo).  When it has completed, the
    neighbours have finished the step whose stores landed in my ghost planes, and they do not start the next one --
    which stores into the volume my step was reading -- before I have finished mine."""
    ops = []
    for has, nb, q in ((slab.ghost_lo, slab.rank - 1, 0), (slab.ghost_hi, slab.rank + 1, 1)):
        if has:
            ops.append(dist.P2POp(dist.isend, token, nb, group))
            ops.append(dist.P2POp(dist.irecv, scratch[q], nb, group))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()


def run_slab_distributed(runner: "SlabRunner", n_total: int, direction: str = "forward", group=None, peer: bool = False,
                         host_sync: bool = False, chunk: int = 64):
    """The same loop for one rank of a torch.distributed job (one slab per GPU, NCCL point-to-point).
    peer = True (or a PeerLinks built for this direction, to be reused over several runs): the step kernels store the halo
    planes into the neighbours' volumes; per step only a token travels.  host_sync = True (tokens on CPU tensors, e.g. a gloo group): the stream is synchronised before the token
    is sent -- for groups whose point-to-point calls are not stream-ordered."""
    which = 0 if direction == "forward" else 1
    steps = range(n_total) if direction == "forward" else range(n_total - 1, -1, -1)
    if peer:
        own_links = not isinstance(peer, PeerLinks)         # peer = a PeerLinks of this direction: reused, the caller closes it
        links = PeerLinks(runner, which, group) if own_links else peer
        assert links.which == which
        dev = "cpu" if host_sync else "cuda"
        token, scratch = torch.ones(1, device=dev), torch.zeros(2, 1, device=dev)
        try:
            multi = runner.slab.world > 1
            if multi:
                dist.barrier(group=group)              # every rank has attached before any kernel stores
            if links.flags:
                # device-side ordering: ranges of `chunk` steps per call, no token, nothing between the ranks but the
                # kernels' own stores and flags (one GPU per rank: the slabs must run side by side)
                for a in range(0, n_total, chunk):
                    b = min(a + chunk, n_total)
                    if direction == "forward":
                        runner.forward_steps(a, b)
                    else:
                        runner.backward_steps(n_total - a, n_total - b)
                steps = ()
            for n in steps:
                if direction == "forward":
                    runner.forward_steps(n, n + 1)
                else:
                    runner.backward_steps(n + 1, n)
                if host_sync:
                    torch.cuda.current_stream().synchronize()
                neighbour_tokens(runner.slab, token, scratch, group)
            torch.cuda.current_stream().synchronize()
            if links.flags and runner.B.fdtd_halo_sync_error(runner.grid.h):
                raise RuntimeError("a slab waited for a neighbour that never reached the state (fdtd_halo_sync_error)")
            if multi:
                dist.barrier(group=group)              # nobody closes a mapping a neighbour's kernel may still write
        finally:
            if own_links:
                links.close()
        return
    for n in steps:
        if direction == "forward":
            runner.forward_steps(n, n + 1)
            state, more = n + 1, n + 1 < n_total
        else:
            runner.backward_steps(n + 1, n)
            state, more = n, n > 0
        if more:
            runner.export_halos(which, state)
            exchange_halos_dist(runner.slab, runner.send_down, runner.send_up, runner.recv_below, runner.recv_above, group)
            runner.import_halos(which, state)
