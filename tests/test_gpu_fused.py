"""GPU tests of the fused launch sequence (persistent pass-A / pass-C kernels, fused_pass.cuh).

The fused sequence runs the 3-pass phase functions of xy_pass.cuh.  Where the unfused sequence runs the same
functions (neither nx nor ny in {512, 768, 1024}) the two results must be BIT-identical; for the long lines the unfused
sequence uses the warp-level kernels (xw_pass.cuh / yw_pass.cuh, another factorisation) and the two must agree to rounding
(relative L2 <= 1e-13).  The fused sequence is additionally compared with the CPU oracle (bar of test_gpu_parity.py).
Small nz values exercise the ramp-up / ramp-down of the ticket order (planes fewer than the lag).
"""
import itertools

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


def same(a, b, nx, ny=0):
    """fused vs unfused: identical bits when both run the same phase functions, else equal to rounding"""
    if nx not in (512, 768, 1024) and ny not in (512, 768, 1024):
        return torch.equal(a, b)
    den = float(b.norm())
    return float((a - b).norm()) <= 1e-13 * den if den > 0 else float((a - b).abs().max()) <= 1e-13


def make_bc(px, py, pz):
    return ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))


def grid(nz, lz, stretch):
    if stretch is None:
        return None, None
    dzc_t, dzf_t, _ = wl.tanh_grid(nz, lz, stretch)
    return dzc_t.numpy(), dzf_t.numpy()


def rhs(nx, ny, nz, bc, dzf, seed):
    rng = np.random.default_rng(seed)
    f = rng.uniform(-1, 1, (nz, ny, nx))
    if orc.is_singular(bc):
        wz = dzf if dzf is not None else np.ones(nz)
        f -= np.sum(f * wz[:, None, None]) / (np.sum(wz) * nx * ny)
    return f


def check(got, ref, scale=1.0, what=""):
    diff = got - ref
    nrm = np.linalg.norm(ref.ravel())
    if nrm > 0:
        rel = np.linalg.norm(diff.ravel()) / nrm
        assert rel <= REL_L2, f"{what}: rel-L2 {rel:.3e}"
    mabs = np.max(np.abs(diff)) * scale
    assert mabs <= MAX_ABS, f"{what}: max-abs {mabs:.3e}"


@pytest.mark.parametrize("nx,ny,nz,stretch", [(256, 256, 5, None), (384, 768, 19, 1.6), (1024, 256, 2, None),
                                               (512, 384, 1 + 16, 2.0), (768, 1024, 3, None), (256, 512, 33, 1.5)])
def test_fused_equals_unfused_bitwise_poisson(B, nx, ny, nz, stretch):
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = grid(nz, lz, stretch)
    seed = 500
    for px, py, pz in [("PP", "PP", "NN"), ("NN", "DD", "DN"), ("DD", "PP", "ND"), ("PP", "NN", "DD")]:
        bc = make_bc(px, py, pz)
        seed += 1
        f = torch.from_numpy(rhs(nx, ny, nz, bc, dzf, seed)).cuda()
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        assert plan.set_fusion(True) is True          # these sizes have fused kernels
        assert plan.launches_per_solve == 3
        p1 = f.clone()
        plan.poisson_solve(p1)
        p1b = f.clone()
        plan.poisson_solve(p1b)                       # second call: scheduler state is reset per call
        assert plan.set_fusion(False) is False
        assert plan.launches_per_solve == 5
        p0 = f.clone()
        plan.poisson_solve(p0)
        torch.cuda.synchronize()
        plan.close()
        assert same(p1, p0, nx, ny), f"{px}/{py}/{pz} {nx}x{ny}x{nz}"
        assert torch.equal(p1b, p1)


@pytest.mark.parametrize("nx,ny,nz", [(256, 256, 6), (512, 768, 9), (1024, 384, 2), (384, 256, 1 + 32)])
def test_fused_equals_unfused_bitwise_projection(B, nx, ny, nz):
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = grid(nz, lz, 1.6)
    rng = np.random.default_rng(nx + ny + nz)
    for px, py, pz in [("PP", "PP", "NN"), ("NN", "PP", "NN"), ("PP", "NN", "ND")]:
        bc = make_bc(px, py, pz)
        u, v, w = (torch.from_numpy(rng.standard_normal((nz, ny, nx))).cuda() for _ in range(3))
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        out = []
        for fused in (True, False):
            assert plan.set_fusion(fused) is fused
            assert plan.launches_per_projection == (3 if fused else 6)
            uu, vv, ww = u.clone(), v.clone(), w.clone()
            p = torch.full_like(u, float("nan"))
            plan.projection(uu, vv, ww, p, 1e-3)
            torch.cuda.synchronize()
            out.append((uu, vv, ww, p))
        plan.close()
        for a, b, nm in zip(out[0], out[1], "uvwp"):
            assert same(a, b, nx, ny), f"{nm}: {px}/{py}/{pz} {nx}x{ny}x{nz}"


def test_fused_poisson_against_oracle(B):
    nx, ny, nz = 256, 384, 20
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = grid(nz, lz, 1.6)
    for s, (px, py, pz) in enumerate(itertools.product(["PP", "NN", "DD"], ["PP", "DD"], ["NN", "DN"])):
        bc = make_bc(px, py, pz)
        f = rhs(nx, ny, nz, bc, dzf, 900 + s)
        plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        assert plan.set_fusion(True)
        p = torch.from_numpy(f).cuda()
        plan.poisson_solve(p)
        torch.cuda.synchronize()
        plan.close()
        ref = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        check(p.cpu().numpy(), ref, what=f"{px}/{py}/{pz}")


def test_fused_projection_against_oracle(B):
    nx, ny, nz = 384, 256, 12
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = grid(nz, lz, 1.6)
    bc = make_bc("PP", "PP", "NN")
    rng = np.random.default_rng(11)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    w[-1] = 0
    dt = 1e-3
    plan = B.PoissonPlan(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    assert plan.set_fusion(True)
    ud, vd, wd = (torch.from_numpy(a).cuda() for a in (u, v, w))
    pd = torch.full((nz, ny, nx), float("nan"), dtype=torch.float64, device="cuda")
    plan.projection(ud, vd, wd, pd, dt)
    torch.cuda.synchronize()
    plan.close()
    un, vn, wn, phi, _ = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf)
    check(ud.cpu().numpy(), un, what="u")
    check(vd.cpu().numpy(), vn, what="v")
    check(wd.cpu().numpy(), wn, what="w")
    check(pd.cpu().numpy(), phi, scale=dt, what="dt*Phi")
    assert np.array_equal(wd.cpu().numpy()[-1], w[-1])


def test_unfused_only_sizes_report_it(B):
    bc = make_bc("PP", "PP", "NN")
    plan = B.PoissonPlan(256, 128, 4, 1.0, 1.0, 1.0, bc)        # ny = 128 has no fused kernels
    assert plan.set_fusion(True) is False
    assert plan.launches_per_solve == 5
    plan.close()
