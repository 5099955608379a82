"""GPU parity of the two steps that follow the projection in a time loop: eq. 2d fused into the
correction kernel and the chkdt reduction of Listing 1, both through the C ABI against the CPU oracle."""
import itertools

import numpy as np
import pytest
import torch

from oracle import cans_oracle as orc
from paper_2001_05234_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2001_05234_b200 import binding
    return binding


def _faces(rng, bc, shape, inflow=()):
    nz, ny, nx = shape
    shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    return {d: rng.standard_normal(shapes[d]) for d in range(3) if bc[d][0] == "D" or d in inflow}


ALL_PAIRS = ["PP", "NN", "DD", "ND", "DN"]


@pytest.mark.parametrize("nx,ny,nz", [(48, 32, 37), (16, 16, 2), (512, 64, 5), (96, 1024, 3)])
def test_chkdt_matches_the_oracle_for_every_boundary_combination(B, nx, ny, nz):
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    rng = np.random.default_rng(nx * 7 + nz)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
    dti = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    combos = list(itertools.product(ALL_PAIRS, ALL_PAIRS, ALL_PAIRS))
    if nx * ny * nz > 200000:
        combos = combos[::9]
    for n, (px, py, pz) in enumerate(combos):
        bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
        inflow = tuple(d for d in range(3) if bc[d][0] == "N" and (n + d) % 3 == 0)     # some prescribed-inflow planes too
        faces = _faces(rng, bc, (nz, ny, nx), inflow)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        fd = {d: torch.from_numpy(f).cuda() for d, f in faces.items()}
        for d, t in fd.items():
            plan.set_lower_face(d, t)
        plan.chkdt(ud, vd, wd, dti)
        torch.cuda.synchronize()
        want = orc.chkdt(u, v, w, lx, ly, lz, bc, dzc, dzf, faces)
        assert abs(float(dti[0]) - want) <= 1e-13 * want, (px, py, pz)
        plan.close()


@pytest.mark.parametrize("bcs", ["PP/PP/PP", "NN/NN/NN", "DD/DD/DD", "ND/DN/NN", "PP/NN/DD", "DN/PP/ND"])
def test_chkdt_localised_maxima_at_every_kind_of_boundary(B, bcs):
    """The reduction returns one number: to see a wrong stencil at a boundary, the maximum is planted there.  Small noise
    everywhere plus O(1) values in the 3 x 3 x 3 neighbourhood of one cell -- the corners, edge and face centres of the box, a
    warp edge in x (i = 63 | 64) and an interior cell -- each compared with the oracle."""
    nx, ny, nz = 128, 32, 35            # nz > 32: the marching chunks meet inside the column
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    px, py, pz = bcs.split("/")
    bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
    rng = np.random.default_rng(5)
    faces = _faces(rng, bc, (nz, ny, nx), inflow=tuple(d for d in range(3) if bc[d][0] == "N"))
    for f in faces.values():
        f *= 1e-3
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    fd = {d: torch.from_numpy(f.copy()).cuda() for d, f in faces.items()}
    for d, t in fd.items():
        plan.set_lower_face(d, t)
    dti = torch.zeros((1,), dtype=torch.float64, device="cuda")
    spots = [(i, j, k) for i in (0, nx - 1) for j in (0, ny - 1) for k in (0, nz - 1)]
    spots += [(nx // 2, 0, 0), (0, ny // 2, nz - 1), (nx - 1, ny - 1, nz // 2), (63, 7, 31), (64, 8, 32), (nx // 2, ny // 2, nz // 2),
              (nx // 2, ny // 2, 0), (nx // 2, ny // 2, nz - 1), (0, ny // 2, nz // 2), (nx - 1, ny // 2, nz // 2),
              (nx // 2, 0, nz // 2), (nx // 2, ny - 1, nz // 2)]
    base = [1e-3 * rng.standard_normal((nz, ny, nx)) for _ in range(3)]
    for (i, j, k) in spots:
        fields = [b.copy() for b in base]
        for f in fields:
            for dk in (-1, 0, 1):
                for dj in (-1, 0, 1):
                    for di in (-1, 0, 1):
                        kk, jj, ii = k + dk, j + dj, i + di
                        if 0 <= kk < nz and 0 <= jj < ny and 0 <= ii < nx:
                            f[kk, jj, ii] = rng.uniform(0.5, 1.5) * rng.choice((-1.0, 1.0))
        # the boundary planes next to the spot carry O(1) values too
        fl = {d: f.copy() for d, f in faces.items()}
        for d, f in fl.items():
            near = (i, j, k)[d] <= 1
            if near:
                f += rng.uniform(0.5, 1.5, size=f.shape) * (np.abs(rng.standard_normal(f.shape)) < 0.3)
        for d, t in fd.items():
            t.copy_(torch.from_numpy(fl[d]))
        u, v, w = fields
        plan.chkdt(*(torch.from_numpy(a).cuda() for a in (u, v, w)), dti)
        torch.cuda.synchronize()
        want = orc.chkdt(u, v, w, lx, ly, lz, bc, dzc, dzf, fl)
        assert abs(float(dti[0]) - want) <= 1e-13 * want, (bcs, (i, j, k), float(dti[0]), want)
    plan.close()


@pytest.mark.parametrize("path", ["planned", "static"])
@pytest.mark.parametrize("nx", [16, 32, 48, 96])
def test_chkdt_rows_shorter_than_a_warp(B, nx, path):
    """nx / 2 < 32 or not a multiple of 32: a warp of the chkdt kernels holds several rows (or a row and a part), so a row
    starts and ends in the middle of a warp.  The value beyond a lane's pair must then come from the boundary rule of the
    lane's own row, not from the neighbouring lane (which holds another row).  The maximum is planted at the first and last
    cells of rows that start inside a warp, with periodic x (the wrapped value) and with walls in x, next to periodic and
    non-periodic y; both the planned kernel and the plan-free one (cans_chkdt_static) are checked against the oracle."""
    ny, nz = 16, 5
    hx = nx // 2
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    rows = [j for j in range(ny) if (j * hx) % 32 != 0][:3] + [j for j in range(ny) if (j * hx) % 32 != 0][-2:]
    rows = sorted(set(rows + [0, ny - 1]))
    spots = [(i, j, k) for i in (0, 1, nx - 2, nx - 1) for j in rows for k in (0, 2, nz - 1)]
    for bcs in ("PP/PP/PP", "PP/NN/DD", "PP/DN/NN", "NN/PP/PP", "DN/ND/ND"):
        px, py, pz = bcs.split("/")
        bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
        rng = np.random.default_rng(nx + len(bcs))
        faces = _faces(rng, bc, (nz, ny, nx), inflow=tuple(d for d in range(3) if bc[d][0] == "N"))
        for f in faces.values():
            f *= 1e-3
        fd = {d: torch.from_numpy(f.copy()).cuda() for d, f in faces.items()}
        plan = None
        if path == "planned":
            plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
            for d, t in fd.items():
                plan.set_lower_face(d, t)
        dzc_d, dzf_d = dzc_t.cuda(), dzf_t.cuda()
        dti = torch.zeros((1,), dtype=torch.float64, device="cuda")
        base = [1e-3 * rng.standard_normal((nz, ny, nx)) for _ in range(3)]
        for (i, j, k) in spots:
            fields = [b.copy() for b in base]
            for f in fields:         # O(1) values in the cell and its neighbours along x, wrapped where x is periodic
                for di in (-1, 0, 1):
                    ii = i + di
                    if bc[0][0] == "P":
                        ii %= nx
                    if 0 <= ii < nx:
                        f[k, j, ii] = rng.uniform(0.5, 1.5) * rng.choice((-1.0, 1.0))
            u, v, w = fields
            ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
            if plan is not None:
                plan.chkdt(ud, vd, wd, dti)
            else:
                B.chkdt_static(ud, vd, wd, dti, lx, ly, lz, bc, dzc_d, dzf_d, fd)
            torch.cuda.synchronize()
            want = orc.chkdt(u, v, w, lx, ly, lz, bc, dzc, dzf, faces)
            assert abs(float(dti[0]) - want) <= 1e-13 * want, (bcs, (i, j, k), float(dti[0]), want)
        if plan is not None:
            plan.close()


def test_chkdt_special_values_and_errors(B):
    nx, ny, nz = 32, 16, 8
    bc = (("P", "P"), ("P", "P"), ("N", "N"))
    plan = B.PoissonPlan(nx, ny, nz, 1.0, 1.0, 1.0, bc)
    z = torch.zeros((nz, ny, nx), dtype=torch.float64, device="cuda")
    dti = torch.full((1,), 7.0, dtype=torch.float64, device="cuda")
    plan.chkdt(z, z, z, dti)
    assert float(dti[0]) == 0.0                                           # field at rest: "dti = 0."
    # uniform flow: |a|/dx + |b|/dy (w = 0), reached on the interior faces
    a, b = 1.5, -0.25
    plan.chkdt(z + a, z + b, z, dti)
    assert abs(float(dti[0]) - (abs(a) * nx + abs(b) * ny)) < 1e-12
    plan.close()
    pland = B.PoissonPlan(nx, ny, nz, 1.0, 1.0, 1.0, (("D", "N"), ("P", "P"), ("N", "N")))
    with pytest.raises(B.CansError) as ei:
        pland.chkdt(z, z, z, dti)
    assert ei.value.status == B.CANS_ERR_NEEDS_FACE
    pland.close()


def test_projection_rejects_aliased_fields(B):
    """p is overwritten with the divergence while u, v, w are still being read, and p_acc is updated next to them: any two
    of the arrays being the same memory would silently corrupt the step."""
    nx, ny, nz = 32, 16, 8
    plan = B.PoissonPlan(nx, ny, nz, 1.0, 1.0, 1.0, (("P", "P"), ("P", "P"), ("N", "N")))
    u, v, w, p, pa = (torch.zeros((nz, ny, nx), dtype=torch.float64, device="cuda") for _ in range(5))
    for args, kw in (((u, v, w, u), {}), ((u, v, w, w), {}), ((u, u, w, p), {}), ((u, v, w, p), {"p_acc": v}), ((u, v, w, p), {"p_acc": p})):
        with pytest.raises(B.CansError) as ei:
            plan.projection_step(*args, 1e-3, **kw)
        assert ei.value.status == B.CANS_ERR_INVALID_ARG
    plan.projection_step(u, v, w, p, 1e-3, p_acc=pa)          # five distinct arrays are accepted
    torch.cuda.synchronize()
    plan.close()


@pytest.mark.parametrize("nx,ny,nz,bcs", [(96, 64, 40, ("PP", "PP", "NN")), (512, 32, 9, ("NN", "DN", "ND")),
                                          (48, 768, 6, ("ND", "PP", "PP")), (1024, 32, 4, ("PP", "NN", "DD"))])
def test_projection_step_fuses_eq_2d_and_returns_chkdt(B, nx, ny, nz, bcs):
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, 1.6)
    dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    bc = tuple((p[0], p[1]) for p in bcs)
    rng = np.random.default_rng(nx + nz)
    u, v, w, pacc = (rng.standard_normal((nz, ny, nx)) for _ in range(4))
    pacc *= 100.0
    faces = _faces(rng, bc, (nz, ny, nx))
    dt = 1e-3
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    # plain projection first: the step variant must return the same bits for u, v, w, Phi and the planes
    ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
    fd = {d: torch.from_numpy(f).cuda() for d, f in faces.items()}
    for d, t in fd.items():
        plan.set_lower_face(d, t)
    pd = torch.empty_like(ud)
    plan.projection(ud, vd, wd, pd, dt)
    us, vs, ws = (torch.from_numpy(a).cuda() for a in (u, v, w))
    fs = {d: torch.from_numpy(f).cuda() for d, f in faces.items()}
    for d, t in fs.items():
        plan.set_lower_face(d, t)
    ps = torch.empty_like(us)
    pa = torch.from_numpy(pacc).cuda()
    dti = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    plan.projection_step(us, vs, ws, ps, dt, p_acc=pa, dti=dti)
    torch.cuda.synchronize()
    for a, b in ((ud, us), (vd, vs), (wd, ws), (pd, ps)):
        assert torch.equal(a, b)
    for d in fd:
        assert torch.equal(fd[d], fs[d])
    # eq. 2d against the oracle; |Phi| ~ 1/dt, so the absolute bar applies to dt * p (reading S12)
    un, vn, wn, phi, fn = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf, faces)
    want = orc.pressure_update(pacc, phi)
    got = pa.cpu().numpy()
    assert np.linalg.norm(got - want) <= 1e-11 * np.linalg.norm(want)
    assert np.max(np.abs(got - want)) * dt <= 1e-10
    assert np.array_equal(got, pacc + ps.cpu().numpy())                   # exactly one rounding: the sum of the two fields
    # chkdt of the corrected velocities (Listing 1) against the oracle on the oracle's corrected fields
    want_dti = orc.chkdt(un, vn, wn, lx, ly, lz, bc, dzc, dzf, fn)
    assert abs(float(dti[0]) - want_dti) <= 1e-10 * want_dti
    # p_acc must not alias p
    with pytest.raises(B.CansError) as ei:
        plan.projection_step(us, vs, ws, ps, dt, p_acc=ps)
    assert ei.value.status == B.CANS_ERR_INVALID_ARG
    plan.close()


def _implicit_case(B, nx, ny, nz, bc, coef, seed, stretch=1.6):
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    if bc[2][0] == "P":
        dzc = dzf = None                                  # periodic z: uniform (single-valued wrap spacing)
    else:
        dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, stretch)
        dzc, dzf = dzc_t.numpy(), dzf_t.numpy()
    rng = np.random.default_rng(seed)
    u, v, w, pacc = (rng.standard_normal((nz, ny, nx)) for _ in range(4))
    pacc *= 100.0
    faces = _faces(rng, bc, (nz, ny, nx))
    dt = 1e-3
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    ud, vd, wd, pa = (torch.from_numpy(a).cuda() for a in (u, v, w, pacc))
    fd = {d: torch.from_numpy(f).cuda() for d, f in faces.items()}
    for d, t in fd.items():
        plan.set_lower_face(d, t)
    pd = torch.empty_like(ud)
    plan.projection_step(ud, vd, wd, pd, dt, p_acc=pa, nu_dt_half=coef)
    torch.cuda.synchronize()
    plan.close()
    un, vn, wn, phi, _ = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf, faces)
    want = orc.pressure_update_implicit(pacc, phi, coef, lx, ly, lz, bc, dzc, dzf)
    got = pa.cpu().numpy()
    # the Laplacian term must matter in this test, or a wrong stencil would pass unnoticed
    plain = orc.pressure_update(pacc, phi)
    assert np.linalg.norm(want - plain) >= 0.05 * np.linalg.norm(phi), "test too weak: coef * L Phi is negligible"
    assert np.linalg.norm(got - want) <= 1e-11 * np.linalg.norm(want), bc
    assert np.max(np.abs(got - want)) * dt <= 1e-10, bc
    for g, r in ((ud, un), (vd, vn), (wd, wn)):            # the velocities are those of the plain step
        assert np.linalg.norm(g.cpu().numpy() - r) <= 1e-11 * np.linalg.norm(r)


def test_eq_3e_every_boundary_combination(B):
    """cans_projection_step_implicit: p_acc += Phi - (gamma nu dt / 2) L Phi (eq. 3e) for all 125 combinations of
    boundary pairs, against the oracle's apply_laplacian of the oracle's Phi.  The grid is two chunks of planes tall
    (GRAD_KC = 32), so the carried plane below is exercised across a chunk boundary."""
    n = 0
    for px, py, pz in itertools.product(ALL_PAIRS, ALL_PAIRS, ALL_PAIRS):
        bc = ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))
        _implicit_case(B, 32, 16, 36, bc, 4e-3, seed=n)
        n += 1


@pytest.mark.parametrize("nx,ny,nz,bcs,coef", [(512, 64, 40, ("PP", "PP", "NN"), 2e-5), (96, 768, 9, ("ND", "DD", "DN"), 2e-5),
                                               (1024, 32, 70, ("NN", "PP", "PP"), 4e-6)])
def test_eq_3e_on_the_fast_kernel_sizes(B, nx, ny, nz, bcs, coef):
    _implicit_case(B, nx, ny, nz, tuple((p[0], p[1]) for p in bcs), coef, seed=nx + nz)


def test_eq_3e_argument_checks(B):
    nx, ny, nz = 32, 16, 8
    plan = B.PoissonPlan(nx, ny, nz, 1.0, 1.0, 1.0, (("P", "P"), ("P", "P"), ("N", "N")))
    u, v, w, p, pa = (torch.zeros((nz, ny, nx), dtype=torch.float64, device="cuda") for _ in range(5))
    for kw in ({"nu_dt_half": -1.0, "p_acc": pa}, {"nu_dt_half": 1e-3}):        # negative coefficient; eq. 3e without p_acc
        with pytest.raises(B.CansError) as ei:
            plan.projection_step(u, v, w, p, 1e-3, **kw)
        assert ei.value.status == B.CANS_ERR_INVALID_ARG
    plan.close()
