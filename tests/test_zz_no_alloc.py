"""cans_chkdt_static -- the one entry point of the library that never allocates device memory.

Who needs it: a solver that has already handed the whole board to its own memory pool (a plan's cudaMalloc would fail
there), and a time loop with several busy streams (cudaMalloc / cudaFree wait for the whole device and would stall all of
them).  Such callers cannot create a plan, so this call takes none; its scratch is a fixed 528 KB array inside the library.

The file is named so that pytest collects it last: under `-x` a failure here cannot hide any other test.  The GPU test
compares the plan-free call with the planned cans_chkdt on the same fields.  Both take a maximum of the same per-cell
values, so they must agree to the last bit (the tolerance of the other chkdt tests, 1e-13 relative, is the bound asserted;
equality is checked on top of it).  It makes two calls in a row on different grids: the fixed array keeps what the first
call wrote (its spacing tables, one maximum per CTA, the arrival counter), and the second call -- fewer CTAs, smaller
values, other spacings -- must not see any of it.  Nothing here depends on what ran earlier in the process: the test
passes alone in a fresh interpreter (first use of the array on the device) and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

from paper_2001_05234_b200 import workloads as wl


@pytest.fixture(scope="module")
def B():
    from paper_2001_05234_b200 import binding
    return binding


PPN = (("P", "P"), ("P", "P"), ("N", "N"))


def _call(B, nx, ny, nz, bc=PPN, **kw):
    """The raw C entry point with device pointers that are never dereferenced: argument checks come first."""
    args = dict(lx=1.0, ly=1.0, lz=1.0, dzc=None, dzf=None, u=256, v=512, w=768, fx=None, fy=None, fz=None, dti=1024)
    args.update(kw)
    return B._lib.cans_chkdt_static(nx, ny, nz, args["lx"], args["ly"], args["lz"], B._bc_bytes(bc), args["dzc"], args["dzf"],
                                    args["u"], args["v"], args["w"], args["fx"], args["fy"], args["fz"], args["dti"], None)


def test_sizes_beyond_the_fixed_array_are_refused_with_a_message(B):
    # nz above the spacing tables
    assert _call(B, 64, 64, B.STATIC_MAX_NZ + 1) == B.CANS_ERR_UNSUPPORTED_SIZE
    assert "CANS_STATIC_MAX_NZ" in B.last_error()
    # more CTAs than partial maxima: 2048 x 2048 x 1024 needs 8192 * 32 of them
    assert _call(B, 2048, 2048, 1024) == B.CANS_ERR_UNSUPPORTED_SIZE
    assert "CANS_STATIC_MAX_CTAS" in B.last_error()
    # the largest grids of the benchmark are inside the limit: the argument checks pass and the call reaches the CUDA
    # runtime (which fails here only where there is no GPU)
    cols, planes = (1536 // 2 * 768 + 255) // 256, (576 + 31) // 32
    assert cols * planes <= B.STATIC_MAX_CTAS


def test_bad_arguments_are_refused_before_any_cuda_call(B):
    assert _call(B, 64, 64, 32, u=None) == B.CANS_ERR_INVALID_ARG
    assert _call(B, 64, 64, 32, lz=0.0) == B.CANS_ERR_INVALID_ARG
    assert _call(B, 64, 64, 32, dzc=4096) == B.CANS_ERR_INVALID_ARG                           # dzc without dzf
    assert _call(B, 64, 64, 32, bc=(("P", "N"), ("P", "P"), ("N", "N"))) == B.CANS_ERR_INVALID_ARG
    assert _call(B, 64, 64, 32, bc=(("D", "D"), ("P", "P"), ("N", "N"))) == B.CANS_ERR_NEEDS_FACE
    assert _call(B, 64, 64, 32, fx=4096) == B.CANS_ERR_INVALID_ARG                            # a face on a periodic side
    assert _call(B, 64, 64, 32, v=520) == B.CANS_ERR_INVALID_ARG                              # not 16-byte aligned
    assert _call(B, 30, 16, 32) == B.CANS_ERR_UNSUPPORTED_SIZE                                # (nx/2)*ny not whole warps


def _case(B, seed, nx, ny, nz, bc, amplitude, stretch):
    """One grid: random fields, lower-face planes where the boundary rule reads them; returns (static, planned) dti."""
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    rng = np.random.default_rng(seed)
    u, v, w = (torch.from_numpy(amplitude * rng.standard_normal((nz, ny, nx))).cuda() for _ in range(3))
    shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    faces = {d: torch.from_numpy(amplitude * rng.standard_normal(shapes[d])).cuda() for d in range(3) if bc[d][0] != "P"}
    dzc = dzf = None
    if stretch:
        dzc, dzf, _ = wl.tanh_grid(nz, lz, stretch)
    # the planned path: host spacings into plan tables (allocated), registered face planes
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    for d, t in faces.items():
        plan.set_lower_face(d, t)
    planned = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    plan.chkdt(u, v, w, planned)
    # the plan-free path: device spacings, face planes as arguments
    static = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    B.chkdt_static(u, v, w, static, lx, ly, lz, bc,
                   None if dzc is None else dzc.cuda(), None if dzf is None else dzf.cuda(), faces)
    torch.cuda.synchronize()
    plan.close()
    return float(static[0]), float(planned[0])


@pytest.mark.gpu
def test_two_calls_in_a_row_match_the_planned_path(B):
    # first call: 160 CTAs (two chunks of planes), stretched z, O(1) velocities, walls in y and z
    s1, p1 = _case(B, 1, 128, 64, 40, (("P", "P"), ("D", "N"), ("N", "D")), 1.0, 1.6)
    # second call right behind it: 8 CTAs, uniform z, velocities a thousand times smaller, triperiodic -- any partial
    # maximum, spacing or counter value left over from the first call would show
    s2, p2 = _case(B, 2, 64, 32, 33, (("P", "P"), ("P", "P"), ("P", "P")), 1e-3, 0.0)
    for s, p in ((s1, p1), (s2, p2)):
        assert np.isfinite(s) and p > 0.0
        assert abs(s - p) <= 1e-13 * p
        assert s == p
    assert s2 < 1e-2 * s1                     # the two calls really differ by what the stale data would have hidden


@pytest.mark.gpu
def test_the_same_call_twice_gives_the_same_bits(B):
    bc = (("N", "N"), ("D", "D"), ("P", "P"))
    a = _case(B, 3, 256, 64, 70, bc, 1.0, 0.0)
    b = _case(B, 3, 256, 64, 70, bc, 1.0, 0.0)
    assert a[0] == a[1] == b[0] == b[1]


@pytest.mark.gpu
def test_largest_grid_the_fixed_array_admits(B):
    """1024 x 1024 x 1024: nz at CANS_STATIC_MAX_NZ and exactly CANS_STATIC_MAX_CTAS CTAs, so every slot of the fixed array is
    in use (26 GB of fields; generated on the device).  The maximum is planted once in the first CTA's cells and once in the
    last one's: the plan-free call must find it, and agree with the planned call to the bit."""
    nx = ny = nz = 1024
    assert ((nx // 2) * ny // 256) * ((nz + 31) // 32) == B.STATIC_MAX_CTAS and nz == B.STATIC_MAX_NZ
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    bc = (("P", "P"), ("N", "N"), ("N", "N"))
    gen = torch.Generator(device="cuda").manual_seed(11)
    u, v, w = (1e-3 * torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda", generator=gen) for _ in range(3))
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc)
    planned = torch.zeros((1,), dtype=torch.float64, device="cuda")
    static = torch.zeros((1,), dtype=torch.float64, device="cuda")
    for (k, j, i) in ((0, 0, 1), (nz - 1, ny - 1, nx - 2)):
        old = float(u[k, j, i])
        u[k, j, i] = 5.0
        plan.chkdt(u, v, w, planned)
        B.chkdt_static(u, v, w, static, lx, ly, lz, bc)
        torch.cuda.synchronize()
        assert float(static[0]) == float(planned[0])
        assert float(static[0]) >= 5.0 * nx / lx                  # |u| / dx of the planted face alone
        u[k, j, i] = old
    plan.chkdt(u, v, w, planned)
    B.chkdt_static(u, v, w, static, lx, ly, lz, bc)
    torch.cuda.synchronize()
    assert float(static[0]) == float(planned[0]) < 1.0            # and nothing of the planted runs is left behind
    plan.close()
