"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on identical seeded inputs.

Bar (BASELINE.json north_star): relative L2 <= 1e-11 on every output
field and max-abs <= 1e-10 on O(1)-scaled fields (Phi for Poisson; u, v, w and dt*Phi for projection).
"""
import itertools
import os

import numpy as np
import pytest
import torch

from oracle import cans_oracle as orc
from paper_2001_05234_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL_L2 = 1e-11
MAX_ABS = 1e-10


@pytest.fixture(scope="module")
def B():
    from paper_2001_05234_b200 import binding
    return binding


def np_of(t):
    return t.detach().cpu().numpy()


def dz_np(w):
    if w.dzc is None:
        return None, None
    return w.dzc.numpy(), w.dzf.numpy()


def check_field(got, ref, scale=1.0, what=""):
    got = np.asarray(got)
    diff = got - ref
    nrm = np.linalg.norm(ref.ravel())
    if nrm > 0:
        rel = np.linalg.norm(diff.ravel()) / nrm
        assert rel <= REL_L2, f"{what}: rel-L2 {rel:.3e}"
    mabs = np.max(np.abs(diff)) * scale
    assert mabs <= MAX_ABS, f"{what}: max-abs {mabs:.3e}"


def gpu_poisson(B, w, f_dev):
    plan = B.plan_for(w)
    p = f_dev.clone()
    plan.poisson_solve(p)
    torch.cuda.synchronize()
    plan.close()
    return p


def random_rhs(nx, ny, nz, bc, dzf, seed):
    rng = np.random.default_rng(seed)
    f = rng.uniform(-1, 1, (nz, ny, nx))
    if orc.is_singular(bc):
        wz = dzf if dzf is not None else np.ones(nz)
        f -= np.sum(f * wz[:, None, None]) / (np.sum(wz) * nx * ny)
    return f


# ----------------------------------------------------------------------------------------------
# BASELINE.json configs 1 and 2: full-size, element by element
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("name", ["C1", "C2"])
def test_config_full_parity(B, name):
    w = wl.make_workload(name, device="cuda")
    f = w.fields["f"]
    phi = gpu_poisson(B, w, f)
    dzc, dzf = dz_np(w)
    ref = orc.poisson_solve(np_of(f), *w.lengths, w.bc, dzc, dzf)
    check_field(np_of(phi), ref, what=name)
    wz = dzf if dzf is not None else np.ones(w.n[2])
    # zero dzf-weighted mean (reading S3)
    assert abs(np.sum(np_of(phi) * wz[:, None, None])) <= 1e-12 * np.sum(np.abs(ref) * wz[:, None, None]) + 1e-12


# ----------------------------------------------------------------------------------------------
# every supported boundary combination, sizes that span several tiles with ragged tails
# (nz = 33: three z segments, the last with one row; 48/96: radix-3 lengths; tiles of 16 columns)
# ----------------------------------------------------------------------------------------------
XY = ["PP", "NN", "DD", "ND", "DN"]        # "ND" / "DN": mixed pairs, DCT-IV / DST-IV
ZP = ["NN", "DD", "ND", "DN", "PP"]       # "PP": cyclic tridiagonal systems


@pytest.mark.parametrize("nx,ny,nz,stretch", [(48, 96, 33, 1.6), (128, 32, 40, None), (16, 16, 2, None),
                                               (192, 64, 17, 2.0)])
def test_all_boundary_combinations(B, nx, ny, nz, stretch):
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    if stretch is None:
        dzc = dzf = None
    else:
        dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, stretch)
        dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    seed = 100
    for px, py, pz in itertools.product(XY, XY, ZP):
        bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
        seed += 1
        f = random_rhs(nx, ny, nz, bc, dzf, seed)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        plan.close()
        ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        check_field(np_of(p), ref, what=f"{px}/{py}/{pz} {nx}x{ny}x{nz}")


@pytest.mark.parametrize("n", [16, 32, 48, 64, 96, 128, 192, 256, 384, 512, 768, 1024, 1536, 2048])
def test_every_transform_length_in_x_and_y(B, n):
    lx, ly, lz = 1.0, 2.0, 0.5
    nz = 18
    for (nx, ny, bc) in [(n, 32, (("N", "N"), ("P", "P"), ("D", "N"))), (32, n, (("P", "P"), ("D", "D"), ("N", "N"))),
                         (n, 32, (("N", "D"), ("D", "N"), ("N", "N"))), (32, n, (("D", "N"), ("N", "D"), ("P", "P")))]:
        f = random_rhs(nx, ny, nz, bc, None, n)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        plan.close()
        ref = orc.poisson_solve(f, lx, ly, lz, bc)
        check_field(np_of(p), ref, what=f"n={n} {nx}x{ny}")


# ----------------------------------------------------------------------------------------------
# projection (eqs. 2b-2c) against the oracle, plus its invariants evaluated with the oracle's operators
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("px,py,pz", [("PP", "PP", "NN"), ("PP", "NN", "NN"), ("NN", "NN", "NN"),
                                      ("PP", "PP", "ND"), ("NN", "PP", "NN"),
                                      ("PP", "PP", "PP"), ("NN", "PP", "PP"), ("PP", "NN", "PP")])
def test_projection_parity_and_invariants(B, px, py, pz):
    nx, ny, nz = 96, 64, 40
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
    rng = np.random.default_rng(7)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    if px[1] == "N":
        u[:, :, -1] = 0
    if py[1] == "N":
        v[:, -1, :] = 0
    if pz[1] == "N":
        w[-1] = 0
    dt = 1e-3
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
    pd = torch.full((nz, ny, nx), float("nan"), dtype=torch.float64, device="cuda")   # entry contents ignored
    plan.projection(ud, vd, wd, pd, dt)
    torch.cuda.synchronize()
    un, vn, wn, phi, _ = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf)
    check_field(np_of(ud), un, what="u")
    check_field(np_of(vd), vn, what="v")
    check_field(np_of(wd), wn, what="w")
    check_field(np_of(pd), phi, scale=dt, what="dt*Phi")
    # invariants of the GPU result, measured with the oracle's operators
    div = orc.divergence(np_of(ud), np_of(vd), np_of(wd), lx, ly, lz, bc, dzc, dzf)
    assert np.max(np.abs(div)) < 1e-11 * np.max(np.abs(u)) / min(lx / nx, ly / ny, dzf.min())
    if px[1] == "N":
        assert np.array_equal(np_of(ud)[:, :, -1], u[:, :, -1])
    if py[1] == "N":
        assert np.array_equal(np_of(vd)[:, -1, :], v[:, -1, :])
    if pz[1] == "N":
        assert np.array_equal(np_of(wd)[-1], w[-1])
    # idempotence: projecting the projected field changes nothing
    u1, v1, w1 = ud.clone(), vd.clone(), wd.clone()
    plan.projection(ud, vd, wd, pd, dt)
    torch.cuda.synchronize()
    assert float((ud - u1).abs().max()) < 1e-11 and float((pd * dt).abs().max()) < 1e-11
    plan.close()


def test_error_codes_on_device(B):
    bc = (("P", "P"), ("P", "P"), ("D", "N"))
    plan = B.PoissonPlan(32, 32, 16, 1.0, 1.0, 1.0, bc)
    z = torch.zeros((16, 32, 32), dtype=torch.float64, device="cuda")
    with pytest.raises(B.CansError) as ei:
        plan.projection(z, z.clone(), z.clone(), z.clone(), 1e-3)       # lower 'D' side in z
    assert ei.value.status == B.CANS_ERR_NEEDS_FACE
    with pytest.raises(B.CansError) as ei:
        B.PoissonPlan(32, 32, 16, 1.0, 1.0, 1.0, (("P", "P"), ("P", "P"), ("N", "N"))).projection(
            z, z.clone(), z.clone(), z.clone(), -1.0)
    assert ei.value.status == B.CANS_ERR_INVALID_ARG
    with pytest.raises(ValueError):
        plan.poisson_solve(torch.zeros((16, 32, 31), dtype=torch.float64, device="cuda"))
    plan.close()


def test_solve_runs_on_a_side_stream_without_syncing(B):
    w = wl.make_workload("C1", device="cuda")
    plan = B.plan_for(w)
    f = w.fields["f"]
    s = torch.cuda.Stream()
    p = f.clone()
    torch.cuda.synchronize()
    with torch.cuda.stream(s):
        plan.poisson_solve(p, stream=s)
    s.synchronize()
    ref = gpu_poisson(B, w, f)
    assert torch.equal(p, ref)          # deterministic: same bits on any stream
    plan.close()


def test_host_entry_point_matches_device_path(B):
    w = wl.make_workload("C5", device="cuda", n_override=(64, 48, 32))
    plan = B.plan_for(w)
    u, v, ww = (w.fields[c] for c in "uvw")
    ud, vd, wd = u.clone(), v.clone(), ww.clone()
    pd = torch.empty_like(u)
    plan.projection(ud, vd, wd, pd, w.dt)
    torch.cuda.synchronize()
    uh, vh, wh = (t.cpu().pin_memory() for t in (u, v, ww))
    ph = torch.empty(u.shape, dtype=torch.float64).pin_memory()
    plan.projection_host(uh, vh, wh, ph, w.dt)
    assert torch.equal(uh, ud.cpu()) and torch.equal(wh, wd.cpu()) and torch.equal(ph, pd.cpu())
    plan.close()


@pytest.mark.parametrize("nx,ny,nz", [(1024, 768, 32), (512, 512, 48), (256, 128, 33)])
def test_repeated_calls_are_bit_identical(B, nx, ny, nz):
    """The persistent z solve draws tiles from a ticket counter and the transform kernels run in several
    waves: whatever the scheduling, every call on the same input must return the same bits."""
    w = wl.make_workload("C5", device="cuda", n_override=(nx, ny, nz))
    plan = B.plan_for(w)
    ref = None
    for _ in range(6):
        u, v, ww = (w.fields[c].clone() for c in "uvw")
        p = torch.empty_like(u)
        plan.projection(u, v, ww, p, w.dt)
        torch.cuda.synchronize()
        if ref is None:
            ref = (u, v, ww, p)
        else:
            for a, b in zip(ref, (u, v, ww, p)):
                assert torch.equal(a, b)
    plan.close()


@pytest.mark.parametrize("nx,ny,nz", [(512, 512, 9), (768, 1024, 5), (1024, 768, 6)])
def test_warp_level_transform_kernels_every_kind_pair(B, nx, ny, nz):
    """Lengths 512 / 768 / 1024 run the warp-level 2-pass kernels (xw_pass.cuh, yt_pass.cuh): every (x, y)
    boundary-pair combination against the oracle, on a stretched grid, Poisson and (where allowed) projection."""
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    seed = 4000
    for px, py in itertools.product(XY, XY):
        pz = "ND" if (px == "PP" and py == "PP") else "NN"
        bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
        seed += 1
        f = random_rhs(nx, ny, nz, bc, dzf, seed)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        check_field(np_of(p), ref, what=f"poisson {px}/{py}/{pz} {nx}x{ny}x{nz}")
        if px[0] != "D" and py[0] != "D":
            rng = np.random.default_rng(seed)
            u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
            ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
            pd = torch.empty_like(ud)
            plan.projection(ud, vd, wd, pd, 1e-3)
            torch.cuda.synchronize()
            un, vn, wn, phi, _ = orc.projection(u, v, w, 1e-3, lx, ly, lz, bc, dzc, dzf)
            for got, refv, sc, nm in ((ud, un, 1.0, "u"), (vd, vn, 1.0, "v"), (wd, wn, 1.0, "w"), (pd, phi, 1e-3, "dt*Phi")):
                check_field(np_of(got), refv, scale=sc, what=f"projection {nm} {px}/{py}/{pz} {nx}x{ny}x{nz}")
        plan.close()


@pytest.mark.parametrize("ny", [512, 768, 1024])
def test_y_tile_pipeline_several_tiles_per_cta(B, ny):
    """The persistent TMA-fed y kernels with 600 tiles on 148 CTAs: every CTA walks 4-5 tiles, so the steady state of the
    tile pipeline runs -- two buffers for 512 / 768, ONE buffer refilled box by box behind its write-back for 1024."""
    nx, nz = 32, 300
    lx, ly, lz = 1.0, 2.0, 1.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.4)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    for n, bc in enumerate(((("P", "P"), ("P", "P"), ("N", "N")), (("N", "N"), ("D", "N"), ("D", "D")))):
        f = random_rhs(nx, ny, nz, bc, dzf, 7100 + ny + n)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        plan.close()
        ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        check_field(np_of(p), ref, what=f"ny={ny} {bc}")


@pytest.mark.parametrize("nx,ny,nz", [(1024, 768, 3), (768, 1024, 3), (512, 512, 17), (256, 128, 18), (48, 96, 33)])
def test_no_write_outside_the_fields(B, nx, ny, nz):
    """Every field lives inside a larger allocation whose guard zones (before and after, 1 MiB each) hold a
    sentinel: no kernel family (warp-level, TMA-fed, 3-pass, z tiles, gradient) may touch them."""
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    bc = (("P", "P"), ("N", "N"), ("N", "N"))
    n = nx * ny * nz
    guard = 131072                                     # doubles (1 MiB), keeps the fields 16-byte aligned
    sentinel = -7.25e300
    big = [torch.full((n + 2 * guard,), sentinel, dtype=torch.float64, device="cuda") for _ in range(4)]
    views = [b[guard:guard + n].view(nz, ny, nx) for b in big]
    g = torch.Generator(device="cuda").manual_seed(5)
    for v in views[:3]:
        v.copy_(torch.rand((nz, ny, nx), dtype=torch.float64, device="cuda", generator=g))
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc)
    plan.projection(views[0], views[1], views[2], views[3], 1e-3)
    plan.poisson_solve(views[3])
    torch.cuda.synchronize()
    plan.close()
    for b in big:
        assert bool((b[:guard] == sentinel).all()) and bool((b[guard + n:] == sentinel).all())
        assert bool(torch.isfinite(b[guard:guard + n]).all())


@pytest.mark.parametrize("nx,ny,nz", [(96, 64, 20), (512, 512, 5), (1024, 768, 3)])
@pytest.mark.parametrize("px,py,pz,inflow", [("DD", "PP", "NN", None), ("PP", "DD", "NN", None), ("NN", "NN", "DN", None),
                                              ("DD", "DD", "DD", None), ("NN", "PP", "ND", 0), ("PP", "NN", "ND", 1),
                                              ("DN", "ND", "PP", None), ("ND", "DN", "DN", 0)])
def test_projection_with_lower_face_planes(B, nx, ny, nz, px, py, pz, inflow):
    """Lower 'D' sides carry a registered face plane that the divergence reads and eq. 2c corrects; a plane on a lower
    'N' side is a prescribed inflow.  Fields and planes against the oracle; the result is divergence free."""
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
    rng = np.random.default_rng(nx + 7 * nz)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    faces = {d: rng.standard_normal(shapes[d]) for d, pr in enumerate((px, py, pz)) if pr[0] == "D"}
    if inflow is not None:
        faces[inflow] = rng.standard_normal(shapes[inflow])
    dt = 1e-3
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
    pd = torch.empty_like(ud)
    fd = {d: torch.from_numpy(f).cuda() for d, f in faces.items()}
    for d, t in fd.items():
        plan.set_lower_face(d, t)
    assert plan.launches_per_projection == 6 + sum(1 for d in fd if bc[d][0] == "D")
    plan.projection(ud, vd, wd, pd, dt)
    torch.cuda.synchronize()
    un, vn, wn, phi, fn = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf, faces)
    check_field(np_of(ud), un, what="u")
    check_field(np_of(vd), vn, what="v")
    check_field(np_of(wd), wn, what="w")
    check_field(np_of(pd), phi, scale=dt, what="dt*Phi")
    got_faces = {d: np_of(t) for d, t in fd.items()}
    for d in fd:
        check_field(got_faces[d], fn[d], what=f"face {d}")
        if bc[d][0] == "N":
            assert np.array_equal(got_faces[d], faces[d])        # prescribed inflow: untouched
    div = orc.divergence(np_of(ud), np_of(vd), np_of(wd), lx, ly, lz, bc, dzc, dzf, got_faces)
    assert np.max(np.abs(div)) < 1e-10 * max(np.max(np.abs(u)), 1.0) / min(lx / nx, ly / ny, dzf.min())
    # unregistering brings CANS_ERR_NEEDS_FACE back for 'D' sides
    d_sides = [d for d in fd if bc[d][0] == "D"]
    if d_sides:
        plan.set_lower_face(d_sides[0], None)
        with pytest.raises(B.CansError) as ei:
            plan.projection(ud, vd, wd, pd, dt)
        assert ei.value.status == B.CANS_ERR_NEEDS_FACE
    plan.close()


def test_lower_face_argument_checks(B):
    plan = B.PoissonPlan(32, 32, 16, 1.0, 1.0, 1.0, (("P", "P"), ("N", "N"), ("D", "N")))
    with pytest.raises(B.CansError) as ei:
        plan.set_lower_face(0, torch.zeros((16, 32, 1), dtype=torch.float64, device="cuda"))    # periodic direction
    assert ei.value.status == B.CANS_ERR_INVALID_ARG
    with pytest.raises(ValueError):
        plan.set_lower_face(2, torch.zeros((1, 32, 31), dtype=torch.float64, device="cuda"))    # wrong shape
    plan.set_lower_face(2, torch.zeros((1, 32, 32), dtype=torch.float64, device="cuda"))
    plan.set_lower_face(2, None)
    plan.close()


@pytest.mark.parametrize("nz", [1024, 1000, 590, 513])
def test_tallest_columns(B, nz):
    """nz up to the documented maximum (64 z segments, tiles of 8 columns, four TMA boxes per tile) and ragged heights;
    590: a prime number of segments (37), whose padded column is tiled by four boxes of 148 rows."""
    nx, ny = 48, 32
    lx, ly, lz = 1.0, 1.0, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.8)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    for bc in ((("P", "P"), ("P", "P"), ("N", "N")), (("N", "N"), ("D", "D"), ("D", "N"))):
        f = random_rhs(nx, ny, nz, bc, dzf, nz)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        plan.close()
        ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        check_field(np_of(p), ref, what=f"nz={nz} {bc}")
    with pytest.raises(B.CansError) as ei:
        B.PoissonPlan(nx, ny, 1025, lx, ly, lz, bc)
    assert ei.value.status == B.CANS_ERR_UNSUPPORTED_SIZE


@pytest.mark.parametrize("nz", [576, 1000])
def test_tall_columns_tile_pipeline(B, nz):
    """nz > 512 (tiles of 8 columns, up to 64 segments): 6144 columns = 768 tiles on 148 CTAs, so the ticket and the
    double-buffered tiles reach their steady state.  Singular and regular; a repeated call is bit-identical."""
    nx, ny = 96, 64
    lx, ly, lz = 1.0, 1.5, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.7)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    for n, bc in enumerate(((("P", "P"), ("N", "N"), ("N", "N")), (("D", "N"), ("P", "P"), ("N", "D")))):
        f = random_rhs(nx, ny, nz, bc, dzf, 8200 + nz + n)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        q = torch.from_numpy(f).cuda()
        plan.poisson_solve(q)                      # a second call: the ticket is reset, the result repeats bit for bit
        torch.cuda.synchronize()
        plan.close()
        assert torch.equal(p, q)
        ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        check_field(np_of(p), ref, what=f"nz={nz} {bc}")


# ----------------------------------------------------------------------------------------------
# the z-solve instantiation bench.py times on C4 / C5: 257 <= nz <= 512 runs z_solve_kernel<16,16> (tiles of 16 columns,
# up to 32 segments per column, two TMA boxes per tile).  48 x 32 columns = 96 tiles, so a persistent CTA sees several
# tiles (both buffers, the ticket hand-over); heights just above the switch (257), ragged (300, 497, 511) and full (512).
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("nz", [257, 300, 497, 511, 512])
def test_z_tiles_of_16_columns_every_z_pair(B, nz):
    nx, ny = 48, 32
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    seed = 9000 + nz
    for pz in ZP:
        for px, py in (("PP", "PP"), ("NN", "DD")):
            bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
            seed += 1
            f = random_rhs(nx, ny, nz, bc, dzf, seed)
            plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
            p = torch.from_numpy(f).cuda()
            plan.poisson_solve(p)
            torch.cuda.synchronize()
            ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
            check_field(np_of(p), ref, what=f"poisson {px}/{py}/{pz} nz={nz}")
            if px == "PP":
                rng = np.random.default_rng(seed)
                u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
                faces = {}
                if pz[0] == "D":
                    faces[2] = rng.standard_normal((1, ny, nx))
                ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
                fd = {d: torch.from_numpy(t).cuda() for d, t in faces.items()}
                for d, t in fd.items():
                    plan.set_lower_face(d, t)
                pd = torch.empty_like(ud)
                plan.projection(ud, vd, wd, pd, 1e-3)
                torch.cuda.synchronize()
                un, vn, wn, phi, fn = orc.projection(u, v, w, 1e-3, lx, ly, lz, bc, dzc, dzf, faces)
                for got, refv, sc, nm in ((ud, un, 1.0, "u"), (vd, vn, 1.0, "v"), (wd, wn, 1.0, "w"), (pd, phi, 1e-3, "dt*Phi")):
                    check_field(np_of(got), refv, scale=sc, what=f"projection {nm} {px}/{py}/{pz} nz={nz}")
                for d in fd:
                    check_field(np_of(fd[d]), fn[d], what=f"face {d} nz={nz}")
            plan.close()


@pytest.mark.parametrize("nz", [1024, 960, 513])
def test_tallest_periodic_columns(B, nz):
    """Periodic z (cyclic systems; the correction vector lives in the tile's own staging buffer): nz up to 1024 as for the
    open systems (tiles of 8 columns), beyond that the plan refuses."""
    nx, ny = 48, 32
    lx, ly, lz = 1.0, 1.0, 2.0
    for bc in ((("P", "P"), ("P", "P"), ("P", "P")), (("N", "N"), ("D", "D"), ("P", "P"))):
        f = random_rhs(nx, ny, nz, bc, None, nz + 1)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        plan.close()
        ref = orc.poisson_solve(f, lx, ly, lz, bc)
        check_field(np_of(p), ref, what=f"nz={nz} {bc}")
    with pytest.raises(B.CansError) as ei:
        B.PoissonPlan(nx, ny, 1025, lx, ly, lz, bc)
    assert ei.value.status == B.CANS_ERR_UNSUPPORTED_SIZE
