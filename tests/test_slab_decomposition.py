"""Slab decomposition along X1: cutting the grid into slabs with an ng-deep halo
exchange after each substep and a maximum of the face speeds over the slabs must not change the answer.

* The oracle's own statement of a slab (coordinates of the full grid, internal sides never filled, the step in two
  calls) is pinned by exactly that: 2 and 3 slabs (uneven) reproduce the single-domain run BIT FOR BIT -- the per-zone
  arithmetic does not know about the cut.  Also with a periodic X1 direction (neighbours wrap around).
* The torch.distributed sequencing (`slab.SlabRank`: isend / irecv with rank +- 1, all_reduce(MAX) of the face speeds)
  runs on two gloo ranks on the CPU with the oracle as the engine, against the same single-domain run.
* GPU (one device): the library's slabs, moved by `slab.SlabGroup`, against the single-domain library run and the oracle.
"""
import os
import sys

import numpy as np
import pytest

import oracle
from paper_2205_02484_b200 import slab
from workloads import config
from workloads.states import minkowski_params, sound_wave
from workloads.torus import fm_torus

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


class OracleEngine:
    """The oracle behind the split-step interface of binding.Solver (host arrays)."""

    def __init__(self, p_local, prim_local, as_torch=False):
        self.g = oracle.Grid(p_local)
        self._prim = np.ascontiguousarray(prim_local)
        self.g.bind(self._prim)
        self._dt = None
        self._torch = as_torch
        self._maxp = p_local["fixup_max_passes"]

    def _wrap(self, a):
        if self._torch:
            import torch
            return torch.from_numpy(a)
        return a

    @property
    def prim(self):
        return self._wrap(self._prim)

    @property
    def half(self):
        return self._wrap(self.g.half())

    @property
    def flags(self):
        return self._wrap(self.g.flags())

    @property
    def max_passes(self):
        return self._maxp

    def work(self, which):
        return self.half if which == 0 else self._wrap(self.g.new())

    def set_dt(self, dt):
        self._dt = dt

    def substep_update(self, which):
        self.g.substep_update(which, self._dt)

    def repair_pass(self, which, npass):
        return self.g.repair_pass(which, npass)

    def substep_finish(self, which):
        self.g.substep_finish(which)

    def end_step(self):
        self.g.commit()

    def cfl_cw(self):
        return list(self.g.cfl_cw())

    def last_cw(self):
        return list(self.g.last_cw())

    def dt_of_cw(self, xi, cw):
        return self.g.dt_of_cw(xi, cw)


def single_domain(p, prim0, nsteps, xi=0.45):
    ref = prim0.copy()
    g = oracle.Grid(p)
    g.bind(ref)
    dt = g.cfl_dt(xi)
    for _ in range(nsteps):
        g.step(dt)
    return ref, dt, g.last_cfl_dt(xi)


def torus_case(name, **kw):
    p = config(name, **kw)
    prim0, _ = fm_torus(p)
    g = oracle.Grid(p)
    g.apply_bc(prim0)          # the slabs start from the full array with its physical ghosts filled
    return p, prim0


# ------------------------------------------------------------------ host logic
def test_slab_ranges_and_params():
    assert slab.slab_ranges(10, 3) == [(0, 4), (4, 3), (7, 3)]
    assert slab.slab_ranges(8, 1) == [(0, 8)]
    with pytest.raises(ValueError):
        slab.slab_ranges(2, 3)
    p = config("C3", n1=12, n2=8, n3=4)
    q = [slab.slab_params(p, 3, r) for r in range(3)]
    assert [(x["n1"], x["i_offset"], x["slab_lo"], x["slab_hi"]) for x in q] == [(4, 0, 0, 1), (4, 4, 1, 1), (4, 8, 1, 0)]
    assert all(x["n1_global"] == 12 for x in q)
    assert slab.slab_params(p, 1, 0) == p
    assert [slab.neighbours(p, 3, r) for r in range(3)] == [(-1, 1), (0, 2), (1, -1)]
    pp = dict(p, bc_x1=1)
    assert [slab.neighbours(pp, 3, r) for r in range(3)] == [(2, 1), (0, 2), (1, 0)]
    assert slab.slab_params(pp, 3, 0)["slab_lo"] == 1
    assert slab.slab_slice(p, 3, 1) == slice(4, 4 + 4 + 6)
    with pytest.raises(ValueError):
        slab.slab_params(config("C3", n1=4, n2=8, n3=4), 2, 0)      # 2 zones per slab < ng


# ------------------------------------------------------------------ the oracle's slabs == the single domain, bit for bit
@pytest.mark.parametrize("name,kw,nslabs", [("C3", dict(n1=22, n2=12, n3=6), 2), ("C4", dict(n1=23, n2=12, n3=6), 3),
                                            ("C3", dict(n1=40, n2=16, n3=1), 4), ("C1", dict(n1=32, n2=16), 2)])
def test_oracle_slabs_reproduce_the_single_domain_bit_for_bit(name, kw, nslabs):
    """Includes zones whose inversion fails right next to a cut (the C1 copy: flags ride with the halo and the repair's
    Jacobi passes alternate with exchanges, so the repair is the single-domain repair)."""
    p, prim0 = torus_case(name, **kw)
    ref, dt, dt_next = single_domain(p, prim0, 3)
    engines = [OracleEngine(slab.slab_params(p, nslabs, r), prim0[:, slab.slab_slice(p, nslabs, r)].copy()) for r in range(nslabs)]
    grp = slab.SlabGroup(engines, p)
    assert abs(grp.cfl_dt(0.45) / dt - 1.0) < 4e-16     # the maximum over slabs of the face speeds, then eq. 26 (the
    # oracle's cfl_dt sums 1 / (xi dx / c_w), dt_of_cw sums c_w / (xi dx): the same number to an ulp)
    for _ in range(3):
        grp.step(dt)
    assert grp.last_cfl_dt(0.45) == dt_next
    got = grp.gather()
    assert got.shape == ref.shape
    assert np.array_equal(got, ref)


def test_oracle_slabs_with_a_periodic_x1_direction():
    p = minkowski_params(24, 4, 4)
    prim0, _ = sound_wave(p, direction=0, amp=1e-3)
    oracle.Grid(p).apply_bc(prim0)
    ref, dt, _ = single_domain(p, prim0, 4)
    engines = [OracleEngine(slab.slab_params(p, 3, r), prim0[:, slab.slab_slice(p, 3, r)].copy()) for r in range(3)]
    grp = slab.SlabGroup(engines, p)
    for _ in range(4):
        grp.step(dt)
    ng = p["ng"]
    got = grp.gather()
    # interior: bit for bit; the periodic images in the outer ghost planes arrive through the wrap-around exchange
    assert np.array_equal(got[:, ng:-ng], ref[:, ng:-ng])
    assert np.array_equal(got, ref)


# ------------------------------------------------------------------ two gloo ranks, torch.distributed sequencing
def periodic_case():
    p = minkowski_params(24, 4, 4)
    prim0, _ = sound_wave(p, direction=0, amp=1e-3)
    oracle.Grid(p).apply_bc(prim0)
    return p, prim0


def _rank_main(rank, world, port, q, periodic=False):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p, prim0 = periodic_case() if periodic else torus_case("C4", n1=20, n2=12, n3=6)
    eng = OracleEngine(slab.slab_params(p, world, rank), prim0[:, slab.slab_slice(p, world, rank)].copy(), as_torch=True)
    me = slab.SlabRank(eng, p, rank, world)
    dt = me.cfl_dt(0.45)
    for _ in range(3):
        me.step(dt)
    q.put((rank, dt, me.last_cfl_dt(0.45), eng.prim.numpy().copy()))
    dist.barrier()
    dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_single_domain():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    p, prim0 = torus_case("C4", n1=20, n2=12, n3=6)
    ref, dt, dt_next = single_domain(p, prim0, 3)
    ng = p["ng"]
    assert res[0][1] == res[1][1] and abs(res[0][1] / dt - 1.0) < 4e-16 and res[0][2] == dt_next and res[1][2] == dt_next
    got = np.concatenate([res[0][3][:, :ng + 10], res[1][3][:, ng:]], axis=1)
    assert np.array_equal(got, ref)
    # and the halo planes each rank holds are its neighbour's interior planes
    assert np.array_equal(res[0][3][:, ng + 10:], ref[:, ng + 10:2 * ng + 10])
    assert np.array_equal(res[1][3][:, :ng], ref[:, 10:10 + ng])


def test_two_gloo_ranks_with_a_periodic_x1_direction():
    """Two ranks, periodic X1: each rank's lower AND upper neighbour is the other rank -- the pairing of the four
    point-to-point operations must still put the right planes into the right ghosts."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q, True)) for r in range(2)]
    for pr in procs:
        pr.start()
    res = sorted((q.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    p, prim0 = periodic_case()
    ref, dt, _ = single_domain(p, prim0, 3)
    ng = p["ng"]
    got = np.concatenate([res[0][3][:, :ng + 12], res[1][3][:, ng:]], axis=1)
    assert np.array_equal(got, ref)


# ------------------------------------------------------------------ GPU: the library's slabs on one device
@pytest.mark.gpu
@pytest.mark.parametrize("name,kw,nslabs", [("C4", dict(n1=30, n2=16, n3=40), 2), ("C3", dict(n1=33, n2=16, n3=20), 3)])
def test_gpu_slabs_match_the_single_domain_run_and_the_oracle(name, kw, nslabs):
    pytest.importorskip("torch")
    import paper_2205_02484_b200 as cu
    from test_gpu_parity import prim_errors
    p, prim0 = torus_case(name, **kw)
    ref, dt, dt_next = single_domain(p, prim0, 2)
    s = cu.Solver(p, prim0)
    for _ in range(2):
        s.step(dt)
    one = s.prim.cpu().numpy()
    engines = [cu.Solver(slab.slab_params(p, nslabs, r), np.ascontiguousarray(prim0[:, slab.slab_slice(p, nslabs, r)]))
               for r in range(nslabs)]
    grp = slab.SlabGroup(engines, p)
    assert abs(grp.cfl_dt(0.45) / dt - 1.0) < 1e-13
    for _ in range(2):
        grp.step(dt)
    assert abs(grp.last_cfl_dt(0.45) / dt_next - 1.0) < 1e-13
    got = grp.gather()
    # against the library's own single-domain run: the marching kernels restart their reconstruction at segment
    # boundaries that depend on the extent, so the two agree to round-off, not bit for bit
    assert (prim_errors(p, got, one, whole=True, tol=1e-12) < 1e-12).all(), prim_errors(p, got, one, whole=True, tol=1e-12)
    assert (prim_errors(p, got, ref, whole=True) < 2e-11).all(), prim_errors(p, got, ref, whole=True)
    assert sum(e.stats()[2] for e in engines) == s.stats()[2]      # floor hits add up over the slabs
    # split step == cuharm_step on a single domain, bit for bit
    s2 = cu.Solver(p, prim0)
    for _ in range(2):
        s2.set_dt(dt); s2.substep(0); s2.substep(1)
    assert np.array_equal(s2.prim.cpu().numpy(), one)


# ------------------------------------------------------------------ GPU: the library under SlabRank, two ranks on one device
def _gpu_rank_main(rank, world, port, q):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import torch
    import torch.distributed as dist
    import paper_2205_02484_b200 as cu
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    p, prim0 = torus_case("C4", n1=30, n2=16, n3=40)
    eng = cu.Solver(slab.slab_params(p, world, rank), np.ascontiguousarray(prim0[:, slab.slab_slice(p, world, rank)]))
    me = slab.SlabRank(eng, p, rank, world)
    dt = me.cfl_dt(0.45)
    for _ in range(2):
        me.step(dt)
    q.put((rank, dt, me.last_cfl_dt(0.45), eng.prim.cpu().numpy().copy(), eng.stats()[2]))
    dist.barrier()
    eng.close()
    dist.destroy_process_group()


@pytest.mark.gpu
def test_gpu_library_under_slabrank_two_ranks_on_one_device():
    """slab.SlabRank -- the torch.distributed sequencing a multi-GPU run would use -- with the LIBRARY as its
    engine: two processes, both on cuda:0, halo planes and flags moved over gloo through pinned host buffers (the box has
    one GPU, so NCCL cannot pair two ranks here; the kernels of the two ranks never wait on one another, the host
    sequences them).  Against the library's single-domain run (round-off: the marching kernels restart their
    reconstruction at extent-dependent segment boundaries) and against the oracle."""
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import torch.multiprocessing as mp
    import paper_2205_02484_b200 as cu
    from test_gpu_parity import prim_errors
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 35500 + os.getpid() % 2000
    procs = [ctx.Process(target=_gpu_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for pr in procs:
        pr.start()
    res = sorted((q.get(timeout=600) for _ in procs), key=lambda t: t[0])
    for pr in procs:
        pr.join(timeout=120)
        assert pr.exitcode == 0
    p, prim0 = torus_case("C4", n1=30, n2=16, n3=40)
    ref, dt, dt_next = single_domain(p, prim0, 2)
    s = cu.Solver(p, prim0)
    for _ in range(2):
        s.step(dt)
    one = s.prim.cpu().numpy()
    ng = p["ng"]
    assert res[0][1] == res[1][1] and abs(res[0][1] / dt - 1.0) < 1e-13
    assert res[0][2] == res[1][2] and abs(res[0][2] / dt_next - 1.0) < 1e-13
    got = np.concatenate([res[0][3][:, :ng + 15], res[1][3][:, ng:]], axis=1)
    assert (prim_errors(p, got, one, whole=True, tol=1e-12) < 1e-12).all(), prim_errors(p, got, one, whole=True, tol=1e-12)
    assert (prim_errors(p, got, ref, whole=True) < 2e-11).all(), prim_errors(p, got, ref, whole=True)
    assert res[0][4] + res[1][4] == s.stats()[2]
    # each rank's halo planes are its neighbour's interior planes
    assert np.array_equal(res[0][3][:, ng + 15:], res[1][3][:, ng:2 * ng])
    assert np.array_equal(res[1][3][:, :ng], res[0][3][:, 15:15 + ng])
    s.close()
