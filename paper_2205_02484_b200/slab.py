"""Slab decomposition of the grid along X1 over several GPUs (paper: P:L271-273, one slab per GPU with neighbour
copies over NVLink): host-side sequencing only.  Every step of the update still runs in the
library's kernels on each rank's own slab; this module cuts the grid, moves the halo planes between neighbours after
each substep and takes the maximum of the face speeds over the slabs for eq. 26.

    per substep (predictor into the half-step array, corrector into the primitives):
        substep_update (fluxes, update, inversion, floors, ghost fill)  ->  halo exchange of the array and of the fail flags
        -> repair pass 0 on every slab; sum over the slabs of (failed zones, zones left waiting)
        -> only if any zone failed anywhere: [halo exchange of array + flags; next pass while zones are waiting] ...,
           second ghost fill, halo exchange of the array
    halo = the outermost ng interior (i) planes of a slab, whole (j, k) extent incl. ghosts  ->  the neighbour's ng
           ghost planes on that side (C4, ng = 3: 3 x 262 x 262 x 8 doubles = 13 MB per side and substep; flags 0.8 MB)
    With these exchanges every Jacobi pass of the eq. 34 repair sees across an INTERNAL boundary what the single-domain
    repair sees there: the decomposition does not change the answer when zones fail next to a cut (pinned bit for bit).
    One known exception, at a PERIODIC X1 wrap that falls on a cut: the single-domain repair (oracle and library alike)
    counts every ghost zone as a good donor (ghost flags stay 0; reading A13), so the periodic image of a failed zone
    donates its unrepaired value, whereas the slabs exchange the real flags and skip it -- the stricter reading of P:L248.
    With failed zones on BOTH sides of such a wrap the two answers differ (O(1) in the repaired zones); one failed zone
    alone is bit-equal.  The benchmark configurations have outflow in X1 and are not affected.

The objects below work on any `engine` with the split-step interface of `binding.Solver` (set_dt, substep_update, repair_pass,
substep_finish, work, flags, end_step, max_passes, cfl_cw, last_cw, dt_of_cw): the library on GPUs, or a CPU stand-in in the host-logic tests.

* `slab_params(p, nslabs, r)`      parameter block of slab r of nslabs
* `slab_slice(p, nslabs, r)`       the i-range of the full (ghost-padded) array that slab r starts from
* `SlabRank(engine, ...)`          one rank of a torch.distributed job (NCCL on GPUs, gloo on CPUs): isend / irecv with
                                   rank - 1 and rank + 1, all_reduce(MAX) of three doubles
* `SlabGroup(engines, p)`          all slabs in one process (one device), halos moved by plain copies: the reference for
                                   the sequencing, and what the single-GPU parity test runs

Not measured on more than one GPU in this build (the run's boxes have one); `bench.py --gpus N` keeps running N
replicas.
"""
from typing import List, Sequence, Tuple


def slab_ranges(n1: int, nslabs: int) -> List[Tuple[int, int]]:
    """(first zone, zone count) of every slab: as equal as possible, the first n1 % nslabs slabs one zone longer."""
    if nslabs < 1 or nslabs > n1:
        raise ValueError("need 1 <= nslabs <= n1")
    base, extra = divmod(n1, nslabs)
    out, i0 = [], 0
    for r in range(nslabs):
        n = base + (1 if r < extra else 0)
        out.append((i0, n))
        i0 += n
    return out


def slab_params(p: dict, nslabs: int, r: int) -> dict:
    """Parameter block of slab r: n1 local, coordinates of the full grid, internal sides marked."""
    if nslabs == 1:
        return dict(p)
    i0, n = slab_ranges(p["n1"], nslabs)[r]
    if n < p["ng"]:
        raise ValueError("a slab needs at least ng zones along X1")
    periodic = p["bc_x1"] == 1
    return dict(p, n1=n, n1_global=p["n1"], i_offset=i0, slab_lo=1 if (r > 0 or periodic) else 0,
                slab_hi=1 if (r < nslabs - 1 or periodic) else 0)


def slab_slice(p: dict, nslabs: int, r: int) -> slice:
    """i-range of the full array [8, n1 + 2 ng, ...] that holds slab r with its ghost / halo planes."""
    i0, n = slab_ranges(p["n1"], nslabs)[r]
    return slice(i0, i0 + n + 2 * p["ng"])


def neighbours(p: dict, nslabs: int, r: int) -> Tuple[int, int]:
    """Ranks of the lower and upper X1 neighbour (-1: a physical boundary)."""
    if nslabs == 1:
        return -1, -1
    if p["bc_x1"] == 1:
        return (r - 1) % nslabs, (r + 1) % nslabs
    return (r - 1 if r > 0 else -1), (r + 1 if r < nslabs - 1 else -1)


def _planes(arr, ng: int, n1: int):
    """(lowest ng interior planes, highest ng interior planes, lower ghost planes, upper ghost planes) as views."""
    return arr[:, ng:2 * ng], arr[:, n1:n1 + ng], arr[:, 0:ng], arr[:, n1 + ng:n1 + 2 * ng]


class SlabGroup:
    """All slabs of a grid in one process; halos move by copies between the engines' arrays."""

    def __init__(self, engines: Sequence, p: dict):
        self.engines, self.p, self.n = list(engines), p, len(engines)
        self.ranges = slab_ranges(p["n1"], self.n)

    def _exchange_arrays(self, arrs):
        ng = self.p["ng"]
        # snapshot of what every slab sends before anything is written: the copies must not depend on their order
        sends = []
        for r, a in enumerate(arrs):
            lo, hi, _, _ = _planes(a, ng, self.ranges[r][1])
            sends.append((lo.clone() if hasattr(lo, "clone") else lo.copy(), hi.clone() if hasattr(hi, "clone") else hi.copy()))
        for r, a in enumerate(arrs):
            rl, rh = neighbours(self.p, self.n, r)
            _, _, glo, ghi = _planes(a, ng, self.ranges[r][1])
            if rl >= 0:
                glo[...] = sends[rl][1]   # the lower neighbour's highest interior planes
            if rh >= 0:
                ghi[...] = sends[rh][0]   # the upper neighbour's lowest interior planes

    def _exchange(self, which: int, flags: bool):
        self._exchange_arrays([e.work(which) for e in self.engines])
        if flags:
            # the flag array has no leading component axis: give it one so that the same plane arithmetic applies
            self._exchange_arrays([e.flags[None] for e in self.engines])

    def _substep(self, which: int):
        for e in self.engines:
            e.substep_update(which)
        self._exchange(which, flags=True)
        res = [e.repair_pass(which, 0) for e in self.engines]
        if sum(r[0] for r in res) == 0:
            return
        npass, left = 0, sum(r[1] for r in res)
        self._exchange(which, flags=True)
        while left > 0 and npass < self.engines[0].max_passes:
            npass += 1
            left = sum(e.repair_pass(which, npass)[1] for e in self.engines)
            self._exchange(which, flags=True)
        for e in self.engines:
            e.substep_finish(which)
        self._exchange(which, flags=False)

    def step(self, dt: float):
        for e in self.engines:
            e.set_dt(dt)
        self._substep(0)
        self._substep(1)
        for e in self.engines:
            e.end_step()

    def _max_cw(self, cws):
        return [max(c[d] for c in cws) for d in range(3)]

    def cfl_dt(self, xi: float) -> float:
        return self.engines[0].dt_of_cw(xi, self._max_cw([e.cfl_cw() for e in self.engines]))

    def last_cfl_dt(self, xi: float) -> float:
        return self.engines[0].dt_of_cw(xi, self._max_cw([e.last_cw() for e in self.engines]))

    def gather(self, which: str = "prim"):
        """The full array (ghosts of the physical sides included) assembled from the slabs; numpy."""
        import numpy as np
        ng = self.p["ng"]
        parts = []
        for r, e in enumerate(self.engines):
            a = getattr(e, which)
            a = a.detach().cpu().numpy() if hasattr(a, "detach") else np.asarray(a)
            n = self.ranges[r][1]
            lo = 0 if r == 0 else ng
            hi = n + 2 * ng if r == self.n - 1 else n + ng
            parts.append(a[:, lo:hi])
        return np.concatenate(parts, axis=1)


class SlabRank:
    """One rank of a torch.distributed job: the same sequence with isend / irecv to the neighbouring ranks.

    `engine.prim` / `engine.half` must be torch tensors: CUDA with the NCCL backend; CPU or CUDA with gloo (CUDA arrays are
    then staged through pinned host buffers -- the way to run the library under this class where NCCL has one GPU only)."""

    def __init__(self, engine, p: dict, rank: int, world: int, group=None):
        import torch.distributed as dist
        self.dist, self.group = dist, group
        self.engine, self.p, self.rank, self.world = engine, p, rank, world
        self.n1 = slab_ranges(p["n1"], world)[rank][1]
        self.lo, self.hi = neighbours(p, world, rank)
        self._bufs = {}     # halo send / receive buffers by (device, layout)
        # gloo moves host memory only: with that backend and arrays on a GPU the packed halo buffers live in pinned host
        # memory and the planes are copied device -> host -> (gloo) -> host -> device.  With NCCL they stay on the device.
        self.stage_host = dist.get_backend(group) == "gloo"

    def _exchange(self, arr, flags=None):
        """Halo planes of `arr` (and, when given, of the flag array) to and from both neighbours: ONE message per neighbour
        and direction -- planes and flags packed into a byte buffer -- and buffers that are allocated once per layout and
        reused by every later exchange (no allocation, no .contiguous() copy in the steady state)."""
        import torch
        ng = self.p["ng"]
        parts = [arr] if flags is None else [arr, flags]
        planes = [_planes(a, ng, self.n1) for a in parts]
        sizes = [pl[0].numel() * pl[0].element_size() for pl in planes]      # bytes per side; the fp64 part comes first, so
        key = (str(arr.device), tuple(sizes))                                 # every part starts on a multiple of 8 bytes
        buf = self._bufs.get(key)
        if buf is None:
            if self.stage_host and arr.is_cuda:
                buf = [torch.empty(sum(sizes), dtype=torch.uint8, device="cpu").pin_memory() for _ in range(4)]
            else:
                buf = [torch.empty(sum(sizes), dtype=torch.uint8, device=arr.device) for _ in range(4)]
            self._bufs[key] = buf
        send_lo, send_hi, recv_lo, recv_hi = buf

        def pieces(b, which):
            off = 0
            for a, pl, sz in zip(parts, planes, sizes):
                yield b[off:off + sz].view(a.dtype).view(pl[which].shape), pl[which]
                off += sz

        # Order of the operations: [send lowest planes down, receive upper ghosts from above, send highest planes up,
        # receive lower ghosts from below].  NCCL pairs point-to-point operations between two ranks by ORDER, and with two
        # ranks and a periodic direction the lower and the upper neighbour are the same rank: in this order its first send
        # (its lowest planes) meets my first receive (my upper ghosts), as it must.
        ops = []
        if self.lo >= 0:
            for dst, src in pieces(send_lo, 0):
                dst.copy_(src)
            ops.append(self.dist.P2POp(self.dist.isend, send_lo, self.lo, self.group))
        if self.hi >= 0:
            ops.append(self.dist.P2POp(self.dist.irecv, recv_hi, self.hi, self.group))
            for dst, src in pieces(send_hi, 1):
                dst.copy_(src)
            ops.append(self.dist.P2POp(self.dist.isend, send_hi, self.hi, self.group))
        if self.lo >= 0:
            ops.append(self.dist.P2POp(self.dist.irecv, recv_lo, self.lo, self.group))
        if ops:
            for w in self.dist.batch_isend_irecv(ops):
                w.wait()
        if self.hi >= 0:
            for src, dst in pieces(recv_hi, 3):
                dst.copy_(src)
        if self.lo >= 0:
            for src, dst in pieces(recv_lo, 2):
                dst.copy_(src)

    def _scalar_device(self):
        return "cpu" if self.stage_host else self.engine.prim.device

    def _allsum(self, a, b):
        import torch
        t = torch.tensor([a, b], dtype=torch.int64, device=self._scalar_device())
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return int(t[0]), int(t[1])

    def _substep(self, which: int):
        e = self.engine
        e.substep_update(which)
        self._exchange(e.work(which), e.flags[None])
        nf, left = self._allsum(*e.repair_pass(which, 0))
        if nf == 0:
            return
        npass = 0
        self._exchange(e.work(which), e.flags[None])
        while left > 0 and npass < e.max_passes:
            npass += 1
            _, left = self._allsum(*e.repair_pass(which, npass))
            self._exchange(e.work(which), e.flags[None])
        e.substep_finish(which)
        self._exchange(e.work(which))

    def step(self, dt: float):
        self.engine.set_dt(dt)
        self._substep(0)
        self._substep(1)
        self.engine.end_step()

    def _allmax(self, cw):
        import torch
        t = torch.tensor(list(cw), dtype=torch.float64, device=self._scalar_device())
        if self.world > 1:
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
        return [float(x) for x in t.cpu()]

    def cfl_dt(self, xi: float) -> float:
        return self.engine.dt_of_cw(xi, self._allmax(self.engine.cfl_cw()))

    def last_cfl_dt(self, xi: float) -> float:
        return self.engine.dt_of_cw(xi, self._allmax(self.engine.last_cw()))
