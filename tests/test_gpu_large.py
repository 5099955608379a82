"""GPU parity at BASELINE.json's full sizes (C3, C4, C5), in the launch configuration bench.py times.

C3 is compared element by element with the full oracle.  For C4 / C5 the naive oracle would need
~1e12 multiply-adds, so:
  * element-by-element oracle parity on the same nx, ny, boundary conditions and stretching recipe with
    fewer z planes, and
  * at FULL size, on sampled z-planes, everything the oracle can compute plane by plane from the GPU
    output: the divergence f = D u*/dt, the residual L Phi - f (normwise backward error <= 1e-12), the
    correction u - dt G Phi, the discrete divergence of the corrected velocity; plus the zero
    dzf-weighted mean of Phi and (C4) the closed-form answer of the 64 planted eigenmodes.
"""
import os

import numpy as np
import pytest
import scipy.linalg
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


def rel_l2(a, b):
    nb = np.linalg.norm(b.ravel())
    d = np.linalg.norm((a - b).ravel())
    return d / nb if nb > 0 else d        # absolute form when the reference vanishes (e.g. the wall plane of w)


def op_norm_inf(w):
    nx, ny, nz = w.n
    lx, ly, lz = w.lengths
    dzc = w.dzc.numpy() if w.dzc is not None else np.full(nz + 1, lz / nz)
    dzf = w.dzf.numpy() if w.dzf is not None else np.full(nz, lz / nz)
    a, c = orc.z_coefficients(dzc, dzf)
    return 4.0 / (lx / nx) ** 2 + 4.0 / (ly / ny) ** 2 + 2.0 * np.max(a + c), dzc, dzf


def laplacian_on_plane(phi_dev, k, w, dzc, dzf):
    """(L Phi) on plane k from the oracle's operator applied to the 3-plane slab around it."""
    nx, ny, nz = w.n
    k0, k1 = max(k - 1, 0), min(k + 1, nz - 1)
    slab = phi_dev[k0:k1 + 1].cpu().numpy()
    bcz = (w.bc[2][0] if k0 == 0 else "N", w.bc[2][1] if k1 == nz - 1 else "N")
    if k0 == 0 and k1 == nz - 1:
        bcz = w.bc[2]
    bc = (w.bc[0], w.bc[1], bcz)
    out = orc.apply_laplacian(slab, *w.lengths, bc, dzc[k0:k1 + 2], dzf[k0:k1 + 1])
    return out[k - k0]


def test_c3_full_parity(B):
    w = wl.make_workload("C3", device="cuda")
    f = w.fields["f"]
    plan = B.plan_for(w)
    p = f.clone()
    plan.poisson_solve(p)
    torch.cuda.synchronize()
    plan.close()
    ref = orc.poisson_solve(f.cpu().numpy(), *w.lengths, w.bc)
    got = p.cpu().numpy()
    assert rel_l2(got, ref) <= REL_L2
    assert np.max(np.abs(got - ref)) <= MAX_ABS
    # white-noise RHS: plain relative residual below 1e-12 (reading S13), on sampled planes
    for k in (0, 1, 100, 254, 255):
        res = laplacian_on_plane(p, k, w, *orc.uniform_spacing(w.n[2], w.lengths[2])) - f[k].cpu().numpy()
        assert np.linalg.norm(res) / np.linalg.norm(f[k].cpu().numpy()) < 1e-12


def _c4_modes(w, nmodes=64, seed=20010523404):
    """64 seeded discrete eigenmodes X_q (x) Y_r (x) Z_s of the C4 operator with amplitudes U[-1,1];
    X, Y from the oracle's tables, Z from LAPACK on the symmetrised stretched z stencil."""
    nx, ny, nz = w.n
    lx, ly, lz = w.lengths
    dzc, dzf = w.dzc.numpy(), w.dzf.numpy()
    Bx, lamx, _ = orc.basis("PP", nx)
    By, lamy, _ = orc.basis("DD", ny)
    a, b, c = orc.z_matrix_rows("NN", dzc, dzf)
    T = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
    D = np.diag(dzf)
    mu, Z = scipy.linalg.eigh(D @ T, D)
    Z = Z / np.max(np.abs(Z), axis=0, keepdims=True)
    rng = np.random.default_rng(seed)
    picks = set()
    while len(picks) < nmodes:
        picks.add((int(rng.integers(nx)), int(rng.integers(ny)), int(rng.integers(nz))))
    picks = sorted(picks)
    amps = rng.uniform(-1, 1, len(picks))
    # the outer products are accumulated with torch on the device only to build the 2 GB arrays quickly;
    # every vector, eigenvalue and amplitude comes from the lines above
    f = torch.zeros((nz, ny, nx), dtype=torch.float64, device="cuda")
    sol = torch.zeros_like(f)
    for (q, r, s), A in zip(picks, amps):
        lam = lamx[q] / (lx / nx) ** 2 + lamy[r] / (ly / ny) ** 2 + mu[s]
        zx = torch.from_numpy(np.ascontiguousarray(Z[:, s])).cuda()
        yx = torch.from_numpy(np.ascontiguousarray(By[r])).cuda()
        xx = torch.from_numpy(np.ascontiguousarray(Bx[q])).cuda()
        mode = zx[:, None, None] * (yx[:, None] * xx[None, :])[None]
        f.add_(mode, alpha=float(A))
        sol.add_(mode, alpha=float(A / lam))
    return f, sol


def test_c4_full_size_eigenmodes_and_backward_error(B):
    w = wl.make_workload("C4", device="cuda")
    nx, ny, nz = w.n
    f_modes, sol_modes = _c4_modes(w)
    plan = B.plan_for(w)
    # (a) noise-free part: closed form  sum A_m / lam_m * mode_m
    p = f_modes.clone()
    plan.poisson_solve(p)
    torch.cuda.synchronize()
    got, ref = p.cpu().numpy(), sol_modes.cpu().numpy()
    assert rel_l2(got, ref) <= REL_L2
    assert np.max(np.abs(got - ref)) <= MAX_ABS          # |Phi| = O(1e-1) here: the bar applies to Phi directly
    del got, ref
    # (b) full C4 right-hand side (modes + 1e-3 Gaussian noise): backward error on sampled planes
    f = f_modes + w.fields["f"]
    p = f.clone()
    plan.poisson_solve(p)
    torch.cuda.synchronize()
    plan.close()
    lnorm, dzc, dzf = op_norm_inf(w)
    for k in (0, 1, 7, 200, 256, 510, 511):
        fk = f[k].cpu().numpy()
        res = laplacian_on_plane(p, k, w, dzc, dzf) - fk
        pk = p[max(k - 1, 0):k + 2].cpu().numpy()
        assert np.linalg.norm(res) / (lnorm * np.linalg.norm(pk) + np.linalg.norm(fk)) < 1e-12


def test_c4_reduced_nz_oracle_parity(B):
    w = wl.make_workload("C4", device="cuda", n_override=(1024, 512, 48))
    f = w.fields["f"] * 1e3          # unit-amplitude Gaussian noise
    plan = B.plan_for(w)
    p = f.clone()
    plan.poisson_solve(p)
    torch.cuda.synchronize()
    plan.close()
    ref = orc.poisson_solve(f.cpu().numpy(), *w.lengths, w.bc, w.dzc.numpy(), w.dzf.numpy())
    got = p.cpu().numpy()
    assert rel_l2(got, ref) <= REL_L2 and np.max(np.abs(got - ref)) <= MAX_ABS


def test_c5_reduced_nz_oracle_parity(B):
    w = wl.make_workload("C5", device="cuda", n_override=(1024, 768, 32))
    plan = B.plan_for(w)
    u, v, ww = (w.fields[c].clone() for c in "uvw")
    p = torch.empty_like(u)
    plan.projection(u, v, ww, p, w.dt)
    torch.cuda.synchronize()
    plan.close()
    dzc, dzf = w.dzc.numpy(), w.dzf.numpy()
    un, vn, wn, phi, _ = orc.projection(*(w.fields[c].cpu().numpy() for c in "uvw"), w.dt, *w.lengths, w.bc, dzc, dzf)
    for got, ref, scale in ((u, un, 1.0), (v, vn, 1.0), (ww, wn, 1.0), (p, phi, w.dt)):
        g = got.cpu().numpy()
        assert rel_l2(g, ref) <= REL_L2
        assert np.max(np.abs(g - ref)) * scale <= MAX_ABS


def test_c5_full_size_projection_sampled_planes(B):
    w = wl.make_workload("C5", device="cuda")
    nx, ny, nz = w.n
    lx, ly, lz = w.lengths
    dt = w.dt
    plan = B.plan_for(w)
    u0, v0, w0 = (w.fields[c] for c in "uvw")
    u, v, ww = u0.clone(), v0.clone(), w0.clone()
    p = torch.full_like(u0, float("nan"))
    plan.projection(u, v, ww, p, dt)
    torch.cuda.synchronize()
    plan.close()
    lnorm, dzc, dzf = op_norm_inf(w)
    hmin = min(lx / nx, ly / ny, float(dzf.min()))
    assert bool(torch.isfinite(p).all()) and bool(torch.isfinite(u).all())
    # zero volume-weighted mean of Phi (reading S3)
    wz = w.dzf.cuda()
    mean = float((p.mean(dim=(1, 2)) * wz).sum() / wz.sum())
    assert abs(mean) <= 1e-12 * float(p.abs().max())
    # upper wall face untouched, bit for bit
    assert torch.equal(ww[nz - 1], w0[nz - 1])
    for k in (0, 1, 2, 255, 256, 509, 510, 511):
        k0 = max(k - 1, 0)
        k1 = min(k + 1, nz - 1)
        bcz_lo = (w.bc[2][0] if k0 == 0 else "N")
        # divergence of u* on plane k (slab k-1..k; for k = 0 the true lower wall face)
        sl = slice(k0, k + 1)
        bc_lo = (w.bc[0], w.bc[1], (bcz_lo, "N"))
        f_k = orc.divergence(u0[sl].cpu().numpy(), v0[sl].cpu().numpy(), w0[sl].cpu().numpy(),
                             lx, ly, lz, bc_lo, dzc[k0:k + 2], dzf[k0:k + 1])[k - k0] / dt
        # Phi solves the system: normwise backward error of the residual on this plane
        res = laplacian_on_plane(p, k, w, dzc, dzf) - f_k
        pk = p[k0:k1 + 1].cpu().numpy()
        assert np.linalg.norm(res) / (lnorm * np.linalg.norm(pk) + np.linalg.norm(f_k)) < 1e-12, k
        # correction on plane k from the GPU's Phi, element by element (slab k..k+1; top plane: ghost rule)
        su = slice(k, k1 + 1)
        bc_up = (w.bc[0], w.bc[1], ("N", w.bc[2][1] if k1 == nz - 1 else "N"))
        un, vn, wn, _ = orc.correct_velocity(u0[su].cpu().numpy(), v0[su].cpu().numpy(), w0[su].cpu().numpy(),
                                             p[su].cpu().numpy(), dt, lx, ly, lz, bc_up, dzc[k:k1 + 2], dzf[k:k1 + 1])
        for got, ref in ((u[k], un[0]), (v[k], vn[0]), (ww[k], wn[0])):
            g = got.cpu().numpy()
            assert np.max(np.abs(g - ref)) <= MAX_ABS and rel_l2(g, ref) <= REL_L2, k
        # corrected velocity is discretely solenoidal on this plane
        div = orc.divergence(u[sl].cpu().numpy(), v[sl].cpu().numpy(), ww[sl].cpu().numpy(),
                             lx, ly, lz, bc_lo, dzc[k0:k + 2], dzf[k0:k + 1])[k - k0]
        assert np.max(np.abs(div)) <= 1e-10 * float(u0.abs().max()) / hmin, k


def _host_ram_gb():
    import psutil
    return psutil.virtual_memory().available / 2**30


def test_c5_full_size_oracle_parity(B):
    """The whole C5 step (1024x768x512, the configuration and launch sequence bench.py times) against the oracle on the
    same buffers: u, v, w and dt*Phi element by element at the BASELINE.json bar (rel-L2 <= 1e-11 on the raw fields,
    max-abs <= 1e-10 on u, v, w and dt*Phi -- reading S12)."""
    if _host_ram_gb() < 96:
        pytest.skip("the full-size oracle needs ~60 GB of host memory")
    w = wl.make_workload("C5", device="cuda")
    plan = B.plan_for(w)
    u, v, ww = (w.fields[c].clone() for c in "uvw")
    p = torch.empty_like(u)
    plan.projection(u, v, ww, p, w.dt)
    torch.cuda.synchronize()
    plan.close()
    got = [t.cpu().numpy() for t in (u, v, ww, p)]
    del u, v, ww, p
    host = [w.fields[c].cpu().numpy() for c in "uvw"]
    w.fields.clear()
    torch.cuda.empty_cache()
    un, vn, wn, phi, _ = orc.projection(*host, w.dt, *w.lengths, w.bc, w.dzc.numpy(), w.dzf.numpy())
    del host
    for g, ref, scale, name in ((got[0], un, 1.0, "u"), (got[1], vn, 1.0, "v"), (got[2], wn, 1.0, "w"), (got[3], phi, w.dt, "dt*Phi")):
        assert rel_l2(g, ref) <= REL_L2, name
        assert np.max(np.abs(g - ref)) * scale <= MAX_ABS, name


def test_c4_full_size_oracle_parity(B):
    """Full C4 (1024x512x512, PP/DD/NN, tanh a = 2): 64 planted eigenmodes + 1e-3 Gaussian noise against orc.poisson_solve,
    element by element."""
    if _host_ram_gb() < 64:
        pytest.skip("the full-size oracle needs ~40 GB of host memory")
    w = wl.make_workload("C4", device="cuda")
    f_modes, _ = _c4_modes(w)
    f = f_modes + w.fields["f"]
    del f_modes
    plan = B.plan_for(w)
    p = f.clone()
    plan.poisson_solve(p)
    torch.cuda.synchronize()
    plan.close()
    got = p.cpu().numpy()
    fh = f.cpu().numpy()
    del p, f
    torch.cuda.empty_cache()
    ref = orc.poisson_solve(fh, *w.lengths, w.bc, w.dzc.numpy(), w.dzf.numpy())
    assert rel_l2(got, ref) <= REL_L2
    assert np.max(np.abs(got - ref)) <= MAX_ABS
