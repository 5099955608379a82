"""Pins for the CPU oracle (oracle/cans_oracle.py): everything here checks the oracle against
something OTHER than itself -- matrices assembled in this file from the 7-point stencil of eq. 5
 and the ghost-cell rules, scipy/LAPACK routines, closed forms and invariants of
eqs. 2b-2c.  No GPU needed."""
import itertools

import numpy as np
import pytest
import scipy.fft
import scipy.linalg

from oracle import cans_oracle as orc

PAIRS_XY = ["PP", "NN", "DD", "ND", "DN"]
PAIRS_Z = ["NN", "DD", "ND", "DN", "PP"]


# ----------------------------------------------------------------------------------------------
# independent assembly of the operator from the stencil + ghost rules (written out here, not
# imported): neighbour outside the range -> wrap (P), +self (N), -self (D)
# ----------------------------------------------------------------------------------------------
def second_difference_1d(n, pair, lo_coef=None, up_coef=None):
    """n x n matrix of  lo_k*(phi_{k-1}-phi_k) + up_k*(phi_{k+1}-phi_k)  with ghost rules."""
    lo_coef = np.ones(n) if lo_coef is None else lo_coef
    up_coef = np.ones(n) if up_coef is None else up_coef
    M = np.zeros((n, n))
    for k in range(n):
        for off, coef, side in ((-1, lo_coef[k], 0), (+1, up_coef[k], 1)):
            M[k, k] -= coef
            kk = k + off
            if 0 <= kk < n:
                M[k, kk] += coef
            elif pair == "PP":
                M[k, kk % n] += coef
            elif pair[side] == "N":
                M[k, k] += coef
            elif pair[side] == "D":
                M[k, k] -= coef
            else:
                raise AssertionError
    return M


def stretched(nz, lz, a):
    """Independent tanh grid for the tests (faces mapped, centres = midpoints)."""
    Z = np.arange(nz + 1) / nz
    zf = 0.5 * (1 + np.tanh(a * (Z - 0.5)) / np.tanh(a / 2)) * lz
    dzf = np.diff(zf)
    zc = 0.5 * (zf[1:] + zf[:-1])
    dzc = np.empty(nz + 1)
    dzc[1:nz] = np.diff(zc)
    dzc[0] = dzf[0]
    dzc[nz] = dzf[-1]
    return dzc, dzf


def laplacian_matrix(nx, ny, nz, lx, ly, lz, bc, dzc, dzf):
    """Dense (N x N) matrix of eq. 5 on the x-fastest ordering, from Kronecker sums of the 1-D
    stencil matrices above (z: lo = 1/(dzf dzc_k), up = 1/(dzf dzc_{k+1}))."""
    px, py, pz = (b[0] + b[1] for b in bc)
    Lx = second_difference_1d(nx, px) / (lx / nx) ** 2
    Ly = second_difference_1d(ny, py) / (ly / ny) ** 2
    Lz = second_difference_1d(nz, pz, 1.0 / (dzf * dzc[:nz]), 1.0 / (dzf * dzc[1:]))
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    return (np.kron(Iz, np.kron(Iy, Lx)) + np.kron(Iz, np.kron(Ly, Ix)) + np.kron(Lz, np.kron(Iy, Ix)))


def bc_of(px, py, pz):
    return ((px[0], px[1]), (py[0], py[1]), (pz[0], pz[1]))


# ----------------------------------------------------------------------------------------------
# 1-D tables (O2)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("pair", PAIRS_XY)
@pytest.mark.parametrize("n", [2, 5, 8, 12, 33])
def test_basis_diagonalises_stencil(pair, n):
    B, lam, w = orc.basis(pair, n)
    L = second_difference_1d(n, pair)
    assert np.max(np.abs(L @ B.T - B.T * lam[None, :])) < 5e-14
    assert np.max(np.abs((B.T * w[None, :]) @ B - np.eye(n))) < 5e-15 * n
    assert np.all(lam <= 0)


@pytest.mark.parametrize("n", [8, 12, 768, 1024])
def test_basis_matches_scipy_transforms(n):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n)
    scale = np.sqrt(n)
    B, _, _ = orc.basis("NN", n)
    assert np.max(np.abs(2 * B @ x - scipy.fft.dct(x, type=2))) < 2e-14 * scale * 2
    B, _, _ = orc.basis("DD", n)
    assert np.max(np.abs(2 * B @ x - scipy.fft.dst(x, type=2))) < 2e-14 * scale * 2
    B, _, _ = orc.basis("ND", n)
    assert np.max(np.abs(2 * B @ x - scipy.fft.dct(x, type=4))) < 2e-14 * scale * 2
    B, _, _ = orc.basis("DN", n)
    assert np.max(np.abs(2 * B @ x - scipy.fft.dst(x, type=4))) < 2e-14 * scale * 2
    B, _, _ = orc.basis("PP", n)
    X = np.fft.rfft(x)
    got = B @ x
    nc = n // 2 + 1
    assert np.max(np.abs(got[:nc] - X.real)) < 2e-14 * scale
    assert np.max(np.abs(got[nc:] + X.imag[1:(n + 1) // 2])) < 2e-14 * scale


def test_inverse_weights_roundtrip_odd_even():
    for pair, n in itertools.product(PAIRS_XY, [7, 16]):
        B, _, w = orc.basis(pair, n)
        x = np.random.default_rng(1).standard_normal(n)
        assert np.max(np.abs((B.T * w) @ (B @ x) - x)) < 1e-13


# ----------------------------------------------------------------------------------------------
# Thomas (O3) against LAPACK
# ----------------------------------------------------------------------------------------------
def test_thomas_vs_banded_random_dominant():
    rng = np.random.default_rng(3)
    nz = 200
    a = rng.uniform(0.5, 2.0, nz)
    c = rng.uniform(0.5, 2.0, nz)
    b = -(a + c) - rng.uniform(0.01, 3.0, nz)
    d = rng.standard_normal((nz, 4, 3))
    x = orc.thomas(a, b[:, None, None] * np.ones((1, 4, 3)), c, d)
    ab = np.zeros((3, nz))
    ab[0, 1:] = c[:-1]
    ab[1] = b
    ab[2, :-1] = a[1:]
    ref = scipy.linalg.solve_banded((1, 1), ab, d.reshape(nz, -1)).reshape(d.shape)
    assert np.max(np.abs(x - ref)) / np.max(np.abs(ref)) < 1e-13


def test_thomas_near_singular_low_mode():
    # stretched 512-point grid, small shift: cond ~ 3e6.  Thomas (no pivoting) and LAPACK's pivoted
    # banded LU are two correct algorithms; both sit ~1e-12 from a long-double solve, so the bound is
    # a small multiple of cond*eps: 3e-18*cond (1e-11 at cond 3e6, 1e-15 floor).
    nz = 512
    dzc, dzf = stretched(nz, 2.0, 2.0)
    a, b, c = orc.z_matrix_rows("NN", dzc, dzf)
    rng = np.random.default_rng(5)
    d = rng.standard_normal((nz, 1))
    for lam in (-0.25, -1.0, -2.7e4):
        x = orc.thomas(a, (b + lam)[:, None], c, d)
        ab = np.zeros((3, nz))
        ab[0, 1:] = c[:-1]
        ab[1] = b + lam
        ab[2, :-1] = a[1:]
        ref = scipy.linalg.solve_banded((1, 1), ab, d)
        M = np.diag(b + lam) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
        tol = max(1e-15, 3e-18 * np.linalg.cond(M))
        assert np.linalg.norm(x - ref) / np.linalg.norm(ref) < tol


def test_z_rows_match_stencil_matrix():
    nz = 9
    dzc, dzf = stretched(nz, 1.3, 1.7)
    for pz in ("NN", "DD", "ND", "DN"):
        a, b, c = orc.z_matrix_rows(pz, dzc, dzf)
        M = np.diag(b) + np.diag(a[1:], -1) + np.diag(c[:-1], 1)
        ref = second_difference_1d(nz, pz, 1.0 / (dzf * dzc[:nz]), 1.0 / (dzf * dzc[1:]))
        assert np.max(np.abs(M - ref)) < 1e-12 * np.max(np.abs(ref))


# ----------------------------------------------------------------------------------------------
# the operator (O1) and the whole solve (O2-O5) against dense LU, every boundary combination
# ----------------------------------------------------------------------------------------------
def _dense_reference(M, f, singular, dzf, shape):
    nz, ny, nx = shape
    if not singular:
        return np.linalg.solve(M, f.ravel()).reshape(shape)
    # bordered system [L 1; wT 0][phi; mu] = [f; 0] with w = cell volumes (dzf weights)
    wvec = np.repeat(dzf, ny * nx)
    N = M.shape[0]
    A = np.zeros((N + 1, N + 1))
    A[:N, :N] = M
    A[:N, N] = 1.0
    A[N, :N] = wvec
    rhs = np.concatenate([f.ravel(), [0.0]])
    sol = np.linalg.solve(A, rhs)
    return sol[:N].reshape(shape)


@pytest.mark.parametrize("grid", ["uniform", "stretched"])
def test_solve_vs_dense_lu_all_boundary_combinations(grid):
    nx, ny, nz = 8, 8, 8
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    if grid == "uniform":
        dzc, dzf = orc.uniform_spacing(nz, lz)
    else:
        dzc, dzf = stretched(nz, lz, 1.6)
    rng = np.random.default_rng(11)
    worst = 0.0
    for px, py, pz in itertools.product(PAIRS_XY, PAIRS_XY, PAIRS_Z):
        bc = bc_of(px, py, pz)
        M = laplacian_matrix(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        f = rng.uniform(-1, 1, (nz, ny, nx))
        singular = orc.is_singular(bc)
        assert singular == all(p in ("PP", "NN") for p in (px, py, pz))
        if singular:
            f -= np.sum(f * dzf[:, None, None]) / (np.sum(dzf) * nx * ny)   # compatibility (S3)
        # pin O1: the oracle's operator equals the independently assembled matrix
        phi_r = rng.standard_normal((nz, ny, nx))
        lap = orc.apply_laplacian(phi_r, lx, ly, lz, bc, dzc, dzf)
        assert np.max(np.abs(lap.ravel() - M @ phi_r.ravel())) < 1e-11
        # pin O2-O5
        phi = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        ref = _dense_reference(M, f, singular, dzf, (nz, ny, nx))
        err = np.max(np.abs(phi - ref)) / max(np.max(np.abs(ref)), 1e-300)
        worst = max(worst, err)
        assert err < 2e-12, (px, py, pz, err)
        if singular:
            assert abs(np.sum(phi * dzf[:, None, None])) < 1e-12
    assert worst < 2e-12


def test_solve_vs_dense_lu_ragged_sizes():
    # non-power-of-two, all different extents: catches transposed operands / swapped axes
    nx, ny, nz = 6, 5, 7
    lx, ly, lz = 1.0, 2.5, 0.7
    dzc, dzf = stretched(nz, lz, 2.0)
    rng = np.random.default_rng(12)
    for px, py, pz in [("PP", "NN", "DN"), ("DD", "PP", "NN"), ("ND", "DN", "DD"), ("NN", "NN", "NN"),
                       ("PP", "PP", "PP")]:
        bc = bc_of(px, py, pz)
        M = laplacian_matrix(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
        f = rng.uniform(-1, 1, (nz, ny, nx))
        singular = orc.is_singular(bc)
        if singular:
            f -= np.sum(f * dzf[:, None, None]) / (np.sum(dzf) * nx * ny)
        phi = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        ref = _dense_reference(M, f, singular, dzf, (nz, ny, nx))
        assert np.max(np.abs(phi - ref)) / np.max(np.abs(ref)) < 2e-12


# ----------------------------------------------------------------------------------------------
# eigenmodes: f = X_q (x) Y_r (x) Z_s  =>  Phi = f / (lam_q/dx^2 + lam_r/dy^2 + mu_s)   (eq. 6)
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("px,py,pz,a", [("PP", "PP", "NN", 1.6), ("NN", "NN", "DN", None),
                                        ("PP", "DD", "NN", 2.0), ("DD", "NN", "DD", None)])
def test_eigenmode_solution_is_f_over_lambda(px, py, pz, a):
    nx, ny, nz = 24, 18, 20
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = orc.uniform_spacing(nz, lz) if a is None else stretched(nz, lz, a)
    # z eigenpairs from LAPACK on the symmetrised stencil matrix (independent of the oracle's tables)
    Tz = second_difference_1d(nz, pz, 1.0 / (dzf * dzc[:nz]), 1.0 / (dzf * dzc[1:]))
    D = np.diag(dzf)
    mu, Zs = scipy.linalg.eigh(D @ Tz, D)
    Lx = second_difference_1d(nx, px)
    Ly = second_difference_1d(ny, py)
    lamx, Xs = np.linalg.eigh(Lx)
    lamy, Ys = np.linalg.eigh(Ly)
    rng = np.random.default_rng(17)
    bc = bc_of(px, py, pz)
    for _ in range(6):
        q, r, s = rng.integers(nx), rng.integers(ny), rng.integers(nz)
        lam = lamx[q] / (lx / nx) ** 2 + lamy[r] / (ly / ny) ** 2 + mu[s]
        if abs(lam) < 1e-9:
            continue
        f = Zs[:, s][:, None, None] * Ys[:, r][None, :, None] * Xs[:, q][None, None, :]
        f /= np.max(np.abs(f))
        phi = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
        assert np.max(np.abs(phi - f / lam)) < 1e-11 * np.max(np.abs(f / lam))


# ----------------------------------------------------------------------------------------------
# residual / backward error at a size with several hundred modes per direction
# ----------------------------------------------------------------------------------------------
@pytest.mark.parametrize("px,py,pz,a", [("PP", "PP", "NN", 1.5), ("NN", "NN", "DN", None),
                                        ("PP", "DD", "NN", 2.0), ("DN", "ND", "ND", 1.2)])
def test_residual_below_1e12(px, py, pz, a):
    nx, ny, nz = 96, 80, 64
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = orc.uniform_spacing(nz, lz) if a is None else stretched(nz, lz, a)
    bc = bc_of(px, py, pz)
    rng = np.random.default_rng(23)
    f = rng.uniform(-1, 1, (nz, ny, nx))
    if orc.is_singular(bc):
        f -= np.sum(f * dzf[:, None, None]) / (np.sum(dzf) * nx * ny)
    phi = orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
    res = orc.apply_laplacian(phi, lx, ly, lz, bc, dzc, dzf) - f
    assert np.linalg.norm(res) / np.linalg.norm(f) < 1e-12          # white-noise RHS (S13)
    # normwise backward error with |L||phi| from the independently assembled 1-D matrices
    Lx = np.abs(second_difference_1d(nx, px)) / (lx / nx) ** 2
    Ly = np.abs(second_difference_1d(ny, py)) / (ly / ny) ** 2
    Lz = np.abs(second_difference_1d(nz, pz, 1.0 / (dzf * dzc[:nz]), 1.0 / (dzf * dzc[1:])))
    ap = np.abs(phi)
    absl = ap @ Lx.T + np.einsum("rj,kjq->krq", Ly, ap) + np.einsum("sk,kjq->sjq", Lz, ap)
    assert np.linalg.norm(res) / (np.linalg.norm(absl) + np.linalg.norm(f)) < 1e-12


def test_uniform_z_matches_full_3d_spectral_closed_form():
    # on a uniform grid the z direction diagonalises too: Phi^ = f^ / (lx+ly+lz), a closed form that
    # never touches the Thomas recurrence
    nx, ny, nz = 20, 12, 16
    lx, ly, lz = 1.0, 2.0, 3.0
    rng = np.random.default_rng(29)
    for px, py, pz in [("PP", "NN", "DD"), ("DD", "PP", "ND"), ("NN", "DN", "DN")]:
        bc = bc_of(px, py, pz)
        f = rng.standard_normal((nz, ny, nx))
        Lx = second_difference_1d(nx, px) / (lx / nx) ** 2
        Ly = second_difference_1d(ny, py) / (ly / ny) ** 2
        Lz = second_difference_1d(nz, pz) / (lz / nz) ** 2
        ex, Vx = np.linalg.eigh(Lx)
        ey, Vy = np.linalg.eigh(Ly)
        ez, Vz = np.linalg.eigh(Lz)
        fh = np.einsum("kjq,qa->kja", f, Vx)
        fh = np.einsum("kja,jb->kba", fh, Vy)
        fh = np.einsum("kba,kc->cba", fh, Vz)
        fh /= ez[:, None, None] + ey[None, :, None] + ex[None, None, :]
        ref = np.einsum("cba,kc->kba", fh, Vz)
        ref = np.einsum("kba,jb->kja", ref, Vy)
        ref = np.einsum("kja,qa->kjq", ref, Vx)
        phi = orc.poisson_solve(f, lx, ly, lz, bc)
        assert np.max(np.abs(phi - ref)) < 1e-12 * np.max(np.abs(ref))


# ----------------------------------------------------------------------------------------------
# divergence / gradient (O6): D G = L, and the projection invariants of eqs. 2b-2c
# ----------------------------------------------------------------------------------------------
def _gradient_via_correction(phi, lx, ly, lz, bc, dzc, dzf, faces):
    nz, ny, nx = phi.shape
    z = np.zeros_like(phi)
    un, vn, wn, fn = orc.correct_velocity(z, z, z, phi, -1.0, lx, ly, lz, bc, dzc, dzf, faces)
    return un, vn, wn, fn


@pytest.mark.parametrize("px,py,pz", list(itertools.product(["PP", "NN", "DD", "ND", "DN"],
                                                             ["PP", "DN"], ["NN", "DD", "ND", "DN", "PP"])))
def test_div_of_grad_is_the_laplacian(px, py, pz):
    nx, ny, nz = 6, 4, 5
    lx, ly, lz = 1.1, 0.9, 1.7
    dzc, dzf = stretched(nz, lz, 1.4)
    bc = bc_of(px, py, pz)
    rng = np.random.default_rng(31)
    phi = rng.standard_normal((nz, ny, nx))
    faces = {}
    shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    for d, p in enumerate((px, py, pz)):
        if p[0] == "D":
            faces[d] = np.zeros(shapes[d])
    gu, gv, gw, gf = _gradient_via_correction(phi, lx, ly, lz, bc, dzc, dzf, faces)
    div = orc.divergence(gu, gv, gw, lx, ly, lz, bc, dzc, dzf, gf)
    M = laplacian_matrix(nx, ny, nz, lx, ly, lz, bc, dzc, dzf)
    assert np.max(np.abs(div.ravel() - M @ phi.ravel())) < 1e-11


@pytest.mark.parametrize("px,py,pz", [("PP", "PP", "NN"), ("PP", "NN", "NN"), ("NN", "NN", "NN"),
                                      ("PP", "PP", "ND"), ("PP", "DD", "NN"), ("NN", "NN", "DN")])
def test_projection_invariants(px, py, pz):
    nx, ny, nz = 24, 16, 20
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = stretched(nz, lz, 1.6)
    bc = bc_of(px, py, pz)
    rng = np.random.default_rng(37)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    faces = {}
    shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    pairs = (px, py, pz)
    for d, p in enumerate(pairs):
        if p[0] == "D":
            faces[d] = rng.standard_normal(shapes[d])
    # closed (upper 'N') boundary faces carry no flow so that the singular problems are compatible
    if px[1] == "N":
        u[:, :, -1] = 0
    if py[1] == "N":
        v[:, -1, :] = 0
    if pz[1] == "N":
        w[-1] = 0
    dt = 1e-2
    un, vn, wn, phi, fn = orc.projection(u, v, w, dt, lx, ly, lz, bc, dzc, dzf, faces)
    # (i) discretely divergence free
    div = orc.divergence(un, vn, wn, lx, ly, lz, bc, dzc, dzf, fn)
    assert np.max(np.abs(div)) < 1e-11 * np.max(np.abs(u)) / min(lx / nx, ly / ny, dzf.min())
    # (ii) idempotent
    u2, v2, w2, phi2, _ = orc.projection(un, vn, wn, dt, lx, ly, lz, bc, dzc, dzf, fn)
    assert np.max(np.abs(dt * phi2)) < 1e-11
    assert np.max(np.abs(u2 - un)) < 1e-11
    # (v) upper 'N' boundary faces unchanged exactly
    if px[1] == "N":
        assert np.array_equal(un[:, :, -1], u[:, :, -1])
    if py[1] == "N":
        assert np.array_equal(vn[:, -1, :], v[:, -1, :])
    if pz[1] == "N":
        assert np.array_equal(wn[-1], w[-1])


def test_projection_annihilates_pure_gradient_and_keeps_poiseuille():
    nx, ny, nz = 16, 12, 24
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = stretched(nz, lz, 1.6)
    bc = bc_of("PP", "PP", "NN")
    rng = np.random.default_rng(41)
    psi = rng.standard_normal((nz, ny, nx))
    dt = 1e-3
    z = np.zeros_like(psi)
    gu, gv, gw, _ = orc.correct_velocity(z, z, z, psi, -dt, lx, ly, lz, bc, dzc, dzf)   # u* = dt G psi
    un, vn, wn, phi, _ = orc.projection(gu, gv, gw, dt, lx, ly, lz, bc, dzc, dzf)
    scale = np.max(np.abs(gu))
    assert max(np.max(np.abs(un)), np.max(np.abs(vn)), np.max(np.abs(wn))) < 1e-11 * scale
    wmean = np.sum(psi * dzf[:, None, None]) / (np.sum(dzf) * nx * ny)
    assert np.max(np.abs(phi - (psi - wmean))) < 1e-10 * np.max(np.abs(psi))
    # (iv) a Poiseuille profile u(z) is already solenoidal: returned unchanged with Phi ~ 0
    zc = np.cumsum(dzf) - 0.5 * dzf
    up = np.broadcast_to((6 * (zc / lz) * (1 - zc / lz))[:, None, None], (nz, ny, nx)).copy()
    un, vn, wn, phi, _ = orc.projection(up, z, z, dt, lx, ly, lz, bc, dzc, dzf)
    assert np.max(np.abs(un - up)) < 1e-14 and np.max(np.abs(dt * phi)) < 1e-13


# ----------------------------------------------------------------------------------------------
# divergence (eq. 2b) and correction (eq. 2c) pinned INDIVIDUALLY on linear fields, whose staggered differences
# are known in closed form (the pair test above fixes only the product D.G)
# ----------------------------------------------------------------------------------------------
def _linear_setup(nx=6, ny=5, nz=7, a=1.7):
    lx, ly, lz = 1.5, 2.5, 2.0
    dzc, dzf = stretched(nz, lz, a)
    zf = np.concatenate([[0.0], np.cumsum(dzf)])            # face heights, zf[k+1] = upper face of cell k
    zc = 0.5 * (zf[1:] + zf[:-1])
    xf = (np.arange(nx) + 1) * lx / nx                      # +x face of cell i
    yf = (np.arange(ny) + 1) * ly / ny
    xc = (np.arange(nx) + 0.5) * lx / nx
    yc = (np.arange(ny) + 0.5) * ly / ny
    return (nx, ny, nz), (lx, ly, lz), dzc, dzf, (xf, yf, zf[1:]), (xc, yc, zc)


def test_divergence_of_linear_fields_is_their_slope():
    """u = cu*x_face, v = cv*y_face, w = cw*z_face  =>  D u = cu + cv + cw exactly (sign, scale, spacing and
    staggering of every term of eq. 2b; stretched z uses dzf).  Non-periodic sides: the lower face of an
    'N' side is the wall at coordinate 0 (value 0 = the linear field there), of a 'D' side the registered plane."""
    (nx, ny, nz), (lx, ly, lz), dzc, dzf, (xf, yf, zfu), _ = _linear_setup()
    cu, cv, cw = 0.75, -1.25, 2.5
    u = np.broadcast_to(cu * xf[None, None, :], (nz, ny, nx)).copy()
    v = np.broadcast_to(cv * yf[None, :, None], (nz, ny, nx)).copy()
    w = np.broadcast_to(cw * zfu[:, None, None], (nz, ny, nx)).copy()
    bc = (("N", "N"), ("N", "N"), ("N", "N"))
    d = orc.divergence(u, v, w, lx, ly, lz, bc, dzc, dzf)
    assert np.max(np.abs(d - (cu + cv + cw))) < 1e-13
    # each term alone: only one component non-zero
    z = np.zeros_like(u)
    assert np.max(np.abs(orc.divergence(u, z, z, lx, ly, lz, bc, dzc, dzf) - cu)) < 1e-13
    assert np.max(np.abs(orc.divergence(z, v, z, lx, ly, lz, bc, dzc, dzf) - cv)) < 1e-13
    assert np.max(np.abs(orc.divergence(z, z, w, lx, ly, lz, bc, dzc, dzf) - cw)) < 1e-13
    # lower 'D' sides with registered planes holding the linear field's value there (0), and a shifted plane:
    # a constant offset c0 on the lower plane changes only the first cell, by -c0/h
    bcd = (("D", "D"), ("D", "N"), ("D", "D"))
    faces = {0: np.zeros((nz, ny, 1)), 1: np.zeros((nz, 1, nx)), 2: np.zeros((1, ny, nx))}
    d = orc.divergence(u, v, w, lx, ly, lz, bcd, dzc, dzf, faces)
    assert np.max(np.abs(d - (cu + cv + cw))) < 1e-13
    faces[2] = np.full((1, ny, nx), 0.5)
    d2 = orc.divergence(u, v, w, lx, ly, lz, bcd, dzc, dzf, faces)
    assert np.max(np.abs(d2[0] - (cu + cv + cw - 0.5 / dzf[0]))) < 1e-13 and np.array_equal(d2[1:], d[1:])
    # prescribed inflow on a lower 'N' side is read the same way
    d3 = orc.divergence(u, v, w, lx, ly, lz, bc, dzc, dzf, {0: np.full((nz, ny, 1), -2.0)})
    assert np.max(np.abs(d3[:, :, 0] - (cu + cv + cw + 2.0 / (lx / nx)))) < 1e-13
    # periodic: the lower face is the wrapped last value
    bcp = (("P", "P"), ("N", "N"), ("N", "N"))
    d4 = orc.divergence(u, z, z, lx, ly, lz, bcp, dzc, dzf)
    assert np.max(np.abs(d4[:, :, 1:] - cu)) < 1e-13
    assert np.max(np.abs(d4[:, :, 0] - (cu * xf[0] - cu * xf[-1]) / (lx / nx))) < 1e-13


def test_gradient_of_linear_phi_is_constant():
    """phi = gx*x_c + gy*y_c + gz*z_c  =>  eq. 2c subtracts dt*(gx, gy, gz) on every interior face
    (stretched z: centre distances dzc); on the upper faces the ghost rule decides: 'N' leaves the value
    bit-identical, 'D' subtracts dt*(-phi_last - phi_last)/h.  Lower 'D' planes: -= dt*2*phi_first/h."""
    (nx, ny, nz), (lx, ly, lz), dzc, dzf, _, (xc, yc, zc) = _linear_setup()
    gx, gy, gz = 1.5, -0.5, 2.0
    phi = gx * xc[None, None, :] + gy * yc[None, :, None] + gz * zc[:, None, None]
    rng = np.random.default_rng(3)
    u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
    dt = 0.125
    bc = (("N", "N"), ("D", "D"), ("D", "N"))
    faces = {1: rng.standard_normal((nz, 1, nx)), 2: rng.standard_normal((1, ny, nx))}
    un, vn, wn, fn = orc.correct_velocity(u, v, w, phi, dt, lx, ly, lz, bc, dzc, dzf, faces)
    assert np.max(np.abs(un[:, :, :-1] - (u[:, :, :-1] - dt * gx))) < 1e-13
    assert np.max(np.abs(vn[:, :-1, :] - (v[:, :-1, :] - dt * gy))) < 1e-13
    assert np.max(np.abs(wn[:-1] - (w[:-1] - dt * gz))) < 1e-13
    assert np.array_equal(un[:, :, -1], u[:, :, -1])                      # upper 'N' in x
    assert np.array_equal(wn[-1], w[-1])                                  # upper 'N' in z
    dy = ly / ny
    assert np.max(np.abs(vn[:, -1, :] - (v[:, -1, :] - dt * (-2.0 * phi[:, -1, :]) / dy))) < 1e-13   # upper 'D' in y
    assert np.max(np.abs(fn[1] - (faces[1] - dt * 2.0 * phi[:, :1, :] / dy))) < 1e-13               # lower 'D' in y
    assert np.max(np.abs(fn[2] - (faces[2] - dt * 2.0 * phi[:1] / dzc[0]))) < 1e-13                 # lower 'D' in z
    # periodic x: the last face sees the wrapped phi
    bcp = (("P", "P"), ("N", "N"), ("N", "N"))
    un, _, _, _ = orc.correct_velocity(u, v, w, phi, dt, lx, ly, lz, bcp, dzc, dzf)
    assert np.max(np.abs(un[:, :, -1] - (u[:, :, -1] - dt * (phi[:, :, 0] - phi[:, :, -1]) / (lx / nx)))) < 1e-13


# ----------------------------------------------------------------------------------------------
# NEXT row f3: eq. 2d and the chkdt reduction of Listing 1, pinned on inputs whose per-face sums are
# known by hand from the printed lines and their symmetric counterparts (reading S15)
# ----------------------------------------------------------------------------------------------
def test_pressure_update_is_a_plain_sum():
    rng = np.random.default_rng(5)
    p, phi = rng.standard_normal((3, 4, 5)), rng.standard_normal((3, 4, 5))
    out = orc.pressure_update(p, phi)
    assert np.array_equal(out, p + phi) and out is not p
    # by hand (eq. 2d): constant fields 2.5 and -0.75 give 1.75 everywhere; a single cell 3 + 4 = 7
    a, b = np.full((2, 3, 4), 2.5), np.full((2, 3, 4), -0.75)
    assert np.all(orc.pressure_update(a, b) == 1.75)
    a[1, 2, 3], b[1, 2, 3] = 3.0, 4.0
    out = orc.pressure_update(a, b)
    assert out[1, 2, 3] == 7.0 and out[0, 0, 0] == 1.75 and a[1, 2, 3] == 3.0


def test_pressure_update_implicit_closed_forms():
    """eq. 3e: p + Phi - c L Phi, on fields whose Laplacian is known by hand."""
    nz, ny, nx = 6, 8, 12
    lx, ly, lz = 3.0, 2.0, 1.5
    c = 0.37
    rng = np.random.default_rng(8)
    p = rng.standard_normal((nz, ny, nx))
    x = (np.arange(nx) + 0.5) * lx / nx
    # (1) a discrete eigenmode of the periodic second difference: L Phi = -(4/dx^2) sin^2(pi m / nx) Phi, nothing from y, z
    #     (Neumann there: a field constant along y and z has zero second differences, ghosts included)
    m = 2
    phi = np.broadcast_to(np.cos(2 * np.pi * m * x / lx), (nz, ny, nx)).copy()
    lam = -4.0 * np.sin(np.pi * m / nx) ** 2 / (lx / nx) ** 2
    bc = (("P", "P"), ("N", "N"), ("N", "N"))
    out = orc.pressure_update_implicit(p, phi, c, lx, ly, lz, bc)
    assert np.allclose(out, p + (1.0 - c * lam) * phi, rtol=0, atol=1e-12)
    # (2) Phi linear in z on a stretched grid: the flux (Phi_{k+1} - Phi_k) / dzc_{k+1} is the same through every face, so
    #     L Phi = 0 in the interior; next to a Neumann wall only the inner flux is left: L Phi = -+ slope / dzf
    dzc, dzf = stretched(nz, lz, 1.7)
    zc = np.cumsum(dzf) - 0.5 * dzf
    slope = 1.3
    phi = np.broadcast_to((slope * zc)[:, None, None], (nz, ny, nx)).copy()
    out = orc.pressure_update_implicit(p, phi, c, lx, ly, lz, bc, dzc, dzf)
    want = p + phi
    want[0] -= c * slope / dzf[0]
    want[-1] += c * slope / dzf[-1]
    assert np.allclose(out, want, rtol=0, atol=1e-12)
    # (3) Dirichlet walls in y, Phi = 1: the anti-mirrored ghost is -1, so L Phi = -2/dy^2 in the two rows next to the walls
    bcd = (("P", "P"), ("D", "D"), ("N", "N"))
    out = orc.pressure_update_implicit(p, np.ones_like(p), c, lx, ly, lz, bcd)
    want = p + 1.0
    want[:, 0, :] += 2.0 * c / (ly / ny) ** 2
    want[:, -1, :] += 2.0 * c / (ly / ny) ** 2
    assert np.allclose(out, want, rtol=0, atol=1e-12)
    # (4) c = 0 is eq. 2d
    assert np.array_equal(orc.pressure_update_implicit(p, phi, 0.0, lx, ly, lz, bc, dzc, dzf), orc.pressure_update(p, phi))


def test_chkdt_of_uniform_flow():
    """u = a, v = b, w = c everywhere on a triperiodic grid: every face sum is |a|/dx + |b|/dy + |c|/dz."""
    nz, ny, nx = 5, 6, 8
    lx, ly, lz = 4.0, 1.5, 2.5
    bc = (("P", "P"), ("P", "P"), ("P", "P"))
    a, b, c = 2.0, -3.0, 0.5
    u, v, w = (np.full((nz, ny, nx), t) for t in (a, b, c))
    want = abs(a) * nx / lx + abs(b) * ny / ly + abs(c) * nz / lz
    fx, fy, fz = orc.chkdt_fields(u, v, w, lx, ly, lz, bc)
    for f in (fx, fy, fz):
        assert np.max(np.abs(f - want)) < 1e-13
    assert abs(orc.chkdt(u, v, w, lx, ly, lz, bc) - want) < 1e-13
    # stretched z: dtix, dtiy weigh w with 1/dzf(k), dtiz with 1/dzc(k+1) (dzci(k) of the face k+1/2)
    dzc, dzf = stretched(nz, lz, 1.7)
    dzc[0] = dzc[-1] = 0.5 * (dzf[0] + dzf[-1])          # single-valued wrap spacing
    fx, fy, fz = orc.chkdt_fields(u, v, w, lx, ly, lz, bc, dzc, dzf)
    base = abs(a) * nx / lx + abs(b) * ny / ly
    assert np.max(np.abs(fx - (base + abs(c) / dzf)[:, None, None])) < 1e-13
    assert np.max(np.abs(fy - (base + abs(c) / dzf)[:, None, None])) < 1e-13
    assert np.max(np.abs(fz - (base + abs(c) / dzc[1:])[:, None, None])) < 1e-13
    assert orc.chkdt(np.zeros_like(u), np.zeros_like(u), np.zeros_like(u), lx, ly, lz, bc) == 0.0


def test_chkdt_stencils_from_unit_impulses():
    """One non-zero velocity value: the faces that see it and with which weight, written out from Listing 1
    (vx, wx: P:L183-185 as printed; the lost uy, wy, uz, vz lines by the same pattern rotated)."""
    nz, ny, nx = 6, 7, 8
    lx, ly, lz = 4.0, 3.5, 3.0
    dx, dy = lx / nx, ly / ny
    dzc, dzf = stretched(nz, lz, 1.4)
    bc = (("N", "N"), ("N", "N"), ("N", "N"))
    i0, j0, k0 = 3, 2, 3
    z = np.zeros((nz, ny, nx))

    def support(f):
        return {(int(k), int(j), int(i)): f[k, j, i] for k, j, i in zip(*np.nonzero(f))}

    # impulse in v
    v = z.copy(); v[k0, j0, i0] = 2.0
    fx, fy, fz = orc.chkdt_fields(z, v, z, lx, ly, lz, bc, dzc, dzf)
    q = 0.25 * 2.0 / dy
    assert support(fx) == {(k0, j0, i0): q, (k0, j0 + 1, i0): q, (k0, j0, i0 - 1): q, (k0, j0 + 1, i0 - 1): q}
    assert support(fy) == {(k0, j0, i0): 2.0 / dy}
    assert support(fz) == {(k0, j0, i0): q, (k0, j0 + 1, i0): q, (k0 - 1, j0, i0): q, (k0 - 1, j0 + 1, i0): q}
    # impulse in w: 1/dzf of the face's own cell for dtix, dtiy; 1/dzc(k+1) for dtiz
    w = z.copy(); w[k0, j0, i0] = -2.0
    fx, fy, fz = orc.chkdt_fields(z, z, w, lx, ly, lz, bc, dzc, dzf)
    qa, qb = 0.5 / dzf[k0], 0.5 / dzf[k0 + 1]
    assert support(fx) == pytest.approx({(k0, j0, i0): qa, (k0, j0, i0 - 1): qa, (k0 + 1, j0, i0): qb, (k0 + 1, j0, i0 - 1): qb})
    assert support(fy) == pytest.approx({(k0, j0, i0): qa, (k0, j0 - 1, i0): qa, (k0 + 1, j0, i0): qb, (k0 + 1, j0 - 1, i0): qb})
    assert support(fz) == pytest.approx({(k0, j0, i0): 2.0 / dzc[k0 + 1]})
    # impulse in u
    u = z.copy(); u[k0, j0, i0] = 2.0
    fx, fy, fz = orc.chkdt_fields(u, z, z, lx, ly, lz, bc, dzc, dzf)
    q = 0.5 / dx
    assert support(fx) == {(k0, j0, i0): 2.0 / dx}
    assert support(fy) == {(k0, j0, i0): q, (k0, j0 - 1, i0): q, (k0, j0, i0 + 1): q, (k0, j0 - 1, i0 + 1): q}
    assert support(fz) == {(k0, j0, i0): q, (k0, j0, i0 + 1): q, (k0 - 1, j0, i0): q, (k0 - 1, j0, i0 + 1): q}
    # the magnitude is taken of the 4-point SUM ("0.25*abs(v+v+v+v)"): opposite neighbours cancel
    v = z.copy(); v[k0, j0, i0] = 1.0; v[k0, j0, i0 + 1] = -1.0
    fx, _, _ = orc.chkdt_fields(z, v, z, lx, ly, lz, bc, dzc, dzf)
    assert fx[k0, j0, i0] == 0.0 and fx[k0, j0, i0 - 1] == 0.25 / dy and fx[k0, j0, i0 + 1] == 0.25 / dy


def test_chkdt_boundaries():
    """Reading S17: periodic directions wrap; in a non-periodic direction the layer below index 0 is the lower boundary
    face for the normal component (registered plane, else 0) and 0 for the tangential ones; the layer above is 0."""
    nz, ny, nx = 4, 5, 6
    lx, ly, lz = 3.0, 2.5, 2.0
    dx, dy, dz = lx / nx, ly / ny, lz / nz
    z = np.zeros((nz, ny, nx))
    # periodic x: u(nx-1) is the face below cell 0
    bc = (("P", "P"), ("N", "N"), ("N", "N"))
    u = z.copy(); u[1, 2, nx - 1] = 4.0
    _, fy, fz = orc.chkdt_fields(u, z, z, lx, ly, lz, bc)
    assert fy[1, 2, 0] == 1.0 / dx and fy[1, 1, 0] == 1.0 / dx and fz[1, 2, 0] == 1.0 / dx and fz[0, 2, 0] == 1.0 / dx
    # non-periodic x without a plane: nothing wraps
    bcn = (("N", "N"), ("N", "N"), ("N", "N"))
    _, fy, fz = orc.chkdt_fields(u, z, z, lx, ly, lz, bcn)
    assert fy[1, 2, 0] == 0.0 and fz[1, 2, 0] == 0.0
    # a registered lower plane in z enters the w averages of the first layer of cells
    plane = np.zeros((1, ny, nx)); plane[0, 2, 3] = 4.0
    fx, fy, fz = orc.chkdt_fields(z, z, z, lx, ly, lz, (("N", "N"), ("N", "N"), ("D", "N")), lower_face={2: plane})
    assert fx[0, 2, 3] == 1.0 / dz and fx[0, 2, 2] == 1.0 / dz and fy[0, 2, 3] == 1.0 / dz and fy[0, 1, 3] == 1.0 / dz
    assert np.count_nonzero(fx) == 2 and np.count_nonzero(fy) == 2 and np.count_nonzero(fz) == 0
    # tangential components beyond the upper end are 0: the last u-face sees only its two interior v values
    v = np.ones((nz, ny, nx))
    fx, _, _ = orc.chkdt_fields(z, v, z, lx, ly, lz, bcn)
    assert fx[1, 2, nx - 1] == 0.5 / dy and fx[1, 2, 0] == 1.0 / dy and fx[1, 0, 0] == 0.5 / dy


def test_chkdt_is_invariant_under_shifts_along_periodic_directions():
    """A periodic direction has no origin: rolling every field AND every registered lower-face plane along it rolls the
    three per-face sums and leaves the maximum unchanged.  This holds whatever the other directions are, so it pins how
    a lower-face plane of a wall direction is continued along a periodic one (reading S18: wrapped) -- a plane padded
    with zeros there breaks the invariance at the cells next to the wrap."""
    nz, ny, nx = 5, 6, 8
    lx, ly, lz = 3.0, 2.5, 2.0
    rng = np.random.default_rng(17)
    cases = [((("P", "P"), ("D", "N"), ("N", "D")), (2,)),            # x periodic; planes in y ('D') and z (inflow on 'N')
             ((("P", "P"), ("P", "P"), ("D", "D")), (2, 1)),          # x, y periodic; plane in z
             ((("N", "N"), ("P", "P"), ("D", "N")), (1,)),            # y periodic; planes in x (inflow) and z
             ((("D", "D"), ("N", "D"), ("P", "P")), (0,))]            # z periodic (uniform grid); planes in x and y
    shapes = {0: (nz, ny, 1), 1: (nz, 1, nx), 2: (1, ny, nx)}
    for bc, axes in cases:
        u, v, w = (rng.standard_normal((nz, ny, nx)) for _ in range(3))
        faces = {d: rng.standard_normal(shapes[d]) for d in range(3) if bc[d][0] != "P"}
        ref_fields = orc.chkdt_fields(u, v, w, lx, ly, lz, bc, None, None, faces)
        ref = orc.chkdt(u, v, w, lx, ly, lz, bc, None, None, faces)
        for axis in axes:                       # numpy axis: 2 = x, 1 = y, 0 = z
            for s in (1, 3):
                ur, vr, wr = (np.roll(a, s, axis=axis) for a in (u, v, w))
                fr = {d: np.roll(f, s, axis=axis) for d, f in faces.items()}       # (extent 1 along its own direction)
                got_fields = orc.chkdt_fields(ur, vr, wr, lx, ly, lz, bc, None, None, fr)
                for g, r in zip(got_fields, ref_fields):
                    assert np.array_equal(g, np.roll(r, s, axis=axis)), (bc, axis, s)
                assert orc.chkdt(ur, vr, wr, lx, ly, lz, bc, None, None, fr) == ref


# ----------------------------------------------------------------------------------------------
# NEXT row f4: the Helmholtz solve of eq. 3b, cell-centred and with the unknown on the z faces
# ----------------------------------------------------------------------------------------------
def face_second_difference_1d(nz, dzc, dzf, periodic, upper_neumann=False):
    """nz x nz matrix of the second difference of a FACE-located quantity, written from the geometry alone: face k at
    height zf_{k+1}, neighbours dzf_k below and dzf_{k+1} above, control volume dzc_{k+1}.  Non-periodic: wall nodes below
    face 0 and at face nz-1 (value 0), so row nz-1 is left empty -- unless upper_neumann: then face nz-1 (the upper
    boundary) is an unknown whose upper neighbour is the mirror image of face nz-2, a ghost cell of width dzf_{nz-1} away."""
    M = np.zeros((nz, nz))
    rows = nz if periodic else nz - 1
    if upper_neumann:
        k = nz - 1
        lo = 1.0 / (dzc[k + 1] * dzf[k])
        up = 1.0 / (dzc[k + 1] * dzf[k])          # mirrored cell
        M[k, k] = -(lo + up)
        M[k, k - 1] = lo + up                     # w_{k+1} := w_{k-1}
    for k in range(rows):
        lo = 1.0 / (dzc[k + 1] * dzf[k])
        up = 1.0 / (dzc[k + 1] * dzf[(k + 1) % nz])
        M[k, k] = -(lo + up)
        if periodic:
            M[k, (k - 1) % nz] += lo
            M[k, (k + 1) % nz] += up
        else:
            if k - 1 >= 0:
                M[k, k - 1] += lo
            if k + 1 <= nz - 2 or (upper_neumann and k + 1 <= nz - 1):
                M[k, k + 1] += up
    return M


@pytest.mark.parametrize("grid", ["uniform", "stretched"])
def test_helmholtz_vs_dense_lu(grid):
    nx, ny, nz = 6, 8, 7
    lx, ly, lz = 2 * np.pi, np.pi, 2.0
    dzc, dzf = orc.uniform_spacing(nz, lz) if grid == "uniform" else stretched(nz, lz, 1.6)
    rng = np.random.default_rng(23)
    Ix, Iy, Iz = np.eye(nx), np.eye(ny), np.eye(nz)
    # cell-centred unknown: every boundary combination, two shifts
    for px, py, pz in itertools.product(PAIRS_XY, PAIRS_XY, PAIRS_Z):
        bc = bc_of(px, py, pz)
        if pz == "PP":
            dzc_u = dzc.copy(); dzc_u[0] = dzc_u[-1] = 0.5 * (dzf[0] + dzf[-1])
        else:
            dzc_u = dzc
        M = laplacian_matrix(nx, ny, nz, lx, ly, lz, bc, dzc_u, dzf)
        f = rng.uniform(-1, 1, (nz, ny, nx))
        for alpha in (-0.37, -2.0e4):
            ref = np.linalg.solve(M + alpha * np.eye(M.shape[0]), f.ravel()).reshape(f.shape)
            got = orc.helmholtz_solve(f, alpha, lx, ly, lz, bc, dzc_u, dzf)
            assert np.max(np.abs(got - ref)) < 2e-12 * np.max(np.abs(ref)), (px, py, pz, alpha)
    # unknown on the z faces (w): walls (DD) and periodic, x / y any pair
    for px, py, pz in itertools.product(["PP", "DD", "ND"], ["PP", "NN"], ["DD", "PP", "DN"]):
        bc = bc_of(px, py, pz)
        dzc_u = dzc.copy()
        if pz == "PP":
            dzc_u[0] = dzc_u[-1] = 0.5 * (dzf[0] + dzf[-1])
        Lx = second_difference_1d(nx, px) / (lx / nx) ** 2
        Ly = second_difference_1d(ny, py) / (ly / ny) ** 2
        Lz = face_second_difference_1d(nz, dzc_u, dzf, pz == "PP", upper_neumann=(pz == "DN"))
        f = rng.uniform(-1, 1, (nz, ny, nx))
        alpha = -3.5
        rows = np.ones(nz) if pz in ("PP", "DN") else np.concatenate([np.ones(nz - 1), [0.0]])     # row nz-1 of DD: identity
        R = np.diag(rows)
        M = (np.kron(R, np.kron(Iy, Lx)) + np.kron(R, np.kron(Ly, Ix)) + np.kron(Lz, np.kron(Iy, Ix))
             + np.kron(alpha * R + (Iz - R), np.kron(Iy, Ix)))
        ref = np.linalg.solve(M, f.ravel()).reshape(f.shape)
        got = orc.helmholtz_solve(f, alpha, lx, ly, lz, bc, dzc_u, dzf, stagger=2)
        assert np.max(np.abs(got - ref)) < 2e-12 * np.max(np.abs(ref)), (px, py, pz)
        if pz == "DD":
            assert np.max(np.abs(got[-1] - f[-1])) < 1e-13                # the wall slot comes back as it went in
    # staggered along a periodic x or y: same operator as for centres
    bc = bc_of("PP", "PP", "DD")
    f = rng.uniform(-1, 1, (nz, ny, nx))
    assert np.array_equal(orc.helmholtz_solve(f, -1.0, lx, ly, lz, bc, dzc, dzf, stagger=0),
                          orc.helmholtz_solve(f, -1.0, lx, ly, lz, bc, dzc, dzf))
    with pytest.raises(NotImplementedError):
        orc.helmholtz_solve(f, -1.0, lx, ly, lz, bc_of("NN", "PP", "DD"), dzc, dzf, stagger=0)
    with pytest.raises(NotImplementedError):
        orc.helmholtz_solve(f, -1.0, lx, ly, lz, bc_of("PP", "PP", "NN"), dzc, dzf, stagger=2)


def test_helmholtz_face_unknown_with_outflow_top_eigenmodes():
    """Textbook pin of the 'DN' face-located case on a uniform grid: nodes k = 0..n-1 at heights (k+1) dz, zero value at
    height 0, zero slope at the last node.  The eigenvectors of that second difference are sin((q + 1/2) pi (k+1) / n) with
    eigenvalues -(4/dz^2) sin^2((q + 1/2) pi / (2n)) (the DST-III family), so for a right-hand side that is one of them,
    constant in x and y, Phi = f / (lambda + alpha)."""
    nx, ny, nz = 4, 4, 9
    lx, ly, lz = 1.0, 1.0, 1.8
    dz = lz / nz
    k = np.arange(nz)
    for q in (0, 3, nz - 1):
        vec = np.sin((q + 0.5) * np.pi * (k + 1) / nz)
        lam = -4.0 / dz**2 * np.sin((q + 0.5) * np.pi / (2 * nz)) ** 2
        f = np.broadcast_to(vec[:, None, None], (nz, ny, nx)).copy()
        alpha = -2.5
        got = orc.helmholtz_solve(f, alpha, lx, ly, lz, bc_of("PP", "PP", "DN"), stagger=2)
        assert np.max(np.abs(got - f / (lam + alpha))) < 1e-12 * np.max(np.abs(f / (lam + alpha))), q


def test_helmholtz_closed_forms():
    """(i) a constant right-hand side under all-Neumann / periodic conditions: L c = 0, so Phi = f / alpha exactly;
    (ii) alpha -> 0 on a non-singular boundary set reproduces the Poisson solve; (iii) eq. 3b itself: with
    alpha = -2/(gamma nu dt) and f = -rhs * 2/(gamma nu dt), u* - (gamma nu dt/2) L u* = rhs to rounding."""
    nx, ny, nz = 8, 6, 9
    lx, ly, lz = 1.0, 2.0, 1.5
    dzc, dzf = stretched(nz, lz, 1.3)
    f = np.full((nz, ny, nx), 2.5)
    got = orc.helmholtz_solve(f, -4.0, lx, ly, lz, bc_of("PP", "NN", "NN"), dzc, dzf)
    assert np.max(np.abs(got - 2.5 / -4.0)) < 1e-14
    rng = np.random.default_rng(2)
    f = rng.standard_normal((nz, ny, nx))
    bc = bc_of("PP", "DD", "DN")
    assert np.max(np.abs(orc.helmholtz_solve(f, 0.0, lx, ly, lz, bc, dzc, dzf) - orc.poisson_solve(f, lx, ly, lz, bc, dzc, dzf))) < 1e-15
    gamma, nu, dt = 8.0 / 15.0, 1e-3, 2e-2
    cdiff = gamma * nu * dt / 2
    rhs = rng.standard_normal((nz, ny, nx))
    ustar = orc.helmholtz_solve(-rhs / cdiff, -1.0 / cdiff, lx, ly, lz, bc, dzc, dzf)
    back = ustar - cdiff * orc.apply_laplacian(ustar, lx, ly, lz, bc, dzc, dzf)
    assert np.max(np.abs(back - rhs)) < 1e-12
