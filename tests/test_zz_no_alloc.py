"""cuharm_divb_noalloc against cuharm_divb.

Some users of libcuharm cannot allocate device memory: a monitoring or analysis hook that runs inside another
program's time loop gets that program's arrays and nothing more -- the host code owns the device through its own
pool, and cudaMalloc there may fail or stall every stream.  Such a hook has no context either (a context needs a
workspace).  cuharm_divb_noalloc gives it the eq. 23 divergence check with its scratch in a fixed static device
array (limit: (n1-1)*(n2-1) <= 131072 corner rows).  All calls share that array and it keeps the last call's
contents, so the test makes two calls in a row -- the second on a SMALLER grid with a much smaller answer, where
left-over partial maxima of the first would show at once -- and compares each with the context-based path on
the same data, to the tolerance tests/test_gpu_parity.py uses for div B (1e-12 relative).

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes on its own in a fresh process (the first call does the per-device set-up) and after
the rest of the suite."""
import ctypes as C

import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import paper_2205_02484_b200 as cu  # noqa: E402
from workloads import config  # noqa: E402
from workloads.geometry import grid_coords  # noqa: E402
from workloads.states import rng  # noqa: E402
from workloads.torus import fm_torus  # noqa: E402


def both_paths(p, prim):
    s = cu.Solver(p, prim)
    ref = s.divb()                                     # existing path: context + workspace, host scalars
    sg = s.geom(0)[20].contiguous()                    # sqrt(-g) at zone centres, [n1g, n2g]
    out = torch.full((2,), -1.0, dtype=torch.float64, device=s.device)
    cu.cuharm_divb_noalloc(s.prim, sg, p["n1"], p["n2"], p["n3"], p["ng"], grid_coords(p)[1], p["bc_x3"] == 1, out,
                           stream=s.stream)
    got = out.cpu().tolist()
    s.close()
    return got, ref


def close(got, ref):
    return all(g == r or abs(g / r - 1.0) < 1e-12 for g, r in zip(got, ref))


def test_two_calls_in_a_row_match_the_context_path():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    # call 1: 3D, periodic X3, a field that is far from divergence-free -> large partial maxima in every row
    p1 = config("C3", n1=40, n2=36, n3=20)
    prim1, _ = fm_torus(p1)
    prim1[5:8] += 0.01 * rng(5).normal(size=prim1[5:8].shape)
    got1, ref1 = both_paths(p1, prim1)
    assert ref1[1] > 1e-3 and close(got1, ref1), (got1, ref1)
    # call 2, straight after: fewer rows, the solenoidal torus field -> both maxima at round-off
    p2 = config("C3", n1=24, n2=20, n3=12)
    prim2, _ = fm_torus(p2)
    got2, ref2 = both_paths(p2, prim2)
    assert ref2[1] < 1e-12 and got2[1] < 1e-12, (got2, ref2)
    assert got2[0] <= 4 * ref2[0] + 1e-300 and ref2[0] <= 4 * got2[0] + 1e-300, (got2, ref2)
    # and a non-solenoidal field on that smaller grid, compared digit for digit
    prim3 = prim2.copy()
    prim3[5:8] += 1e-6 * rng(6).normal(size=prim3[5:8].shape)
    got3, ref3 = both_paths(p2, prim3)
    assert close(got3, ref3) and got3[0] < 1e-3 * got1[0], (got3, ref3, got1)


def test_axisymmetric_grid_matches_too():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    p = config("C1", n1=32, n2=28)
    prim, _ = fm_torus(p)
    prim[5:7] += 0.01 * rng(7).normal(size=prim[5:7].shape)
    got, ref = both_paths(p, prim)
    assert ref[1] > 1e-3 and close(got, ref), (got, ref)


def test_grids_beyond_the_static_scratch_are_refused():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    dummy = torch.zeros(16, dtype=torch.float64, device="cuda:0")
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(cu.CuharmError, match="exceed the static scratch"):
        cu.cuharm_divb_noalloc(dummy, dummy, 400, 400, 8, 3, [0.1, 0.1, 0.1], True, out)   # 399 * 399 rows
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [-1.0, -1.0]          # nothing was launched
    L = cu.lib()
    dx = (C.c_double * 3)(0.1, 0.1, 0.1)
    assert L.cuharm_divb_noalloc(None, None, 8, 8, 8, 3, dx, 1, None, None) == -1
    assert b"null" in L.cuharm_divb_noalloc_errtext()
