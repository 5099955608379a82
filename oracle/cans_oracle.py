"""CPU oracle for the CaNS pressure-projection hot path  --  TEST INFRASTRUCTURE ONLY.

This module is the plain, slow, obviously-correct FP64 definition of what the CUDA
library in ``paper_2001_05234_b200/csrc`` must compute.  It is *not* part of the
product: only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import it.  It shares no code,
tables or helpers with the CUDA path and never imports it.

Source: /root/reference/PAPER.md ("P:L<n>" = line n of that file).

  * eq. 2b  P:L59   L Phi = D u* / (gamma_k dt)            -> ``divergence``
  * eq. 2c  P:L62   u^{k+1} = u* - gamma_k dt G Phi        -> ``correct_velocity``
  * eq. 5   P:L95   7-point second-order Laplacian         -> ``apply_laplacian``
  * eq. 6   P:L102  (lam_i/dx^2+lam_j/dy^2) Phi^ + d_zz Phi^ = f^, "Gauss elimination"
                    P:L98-100                              -> ``poisson_solve``
  * P:L104  "the grid in z can be non-uniform"             -> ``z_coefficients``
  * eq. 2d  P:L64   p^{k+1/2} = p^{k-1/2} + Phi             -> ``pressure_update``
  * eq. 3e  P:L80   ... + Phi - (gamma nu dt / 2) L Phi     -> ``pressure_update_implicit``
  * eq. 4   P:L87 and Listing 1 P:L142-205 (``chkdt``)     -> ``chkdt_fields``, ``chkdt``
  * eq. 3b  P:L73, P:L106 (implicit diffusion: "solved with the same type of direct solver")
                                                           -> ``z_face_coefficients``, ``helmholtz_solve``

The paper delegates the eigenfunction tables to its refs [11,17], which are
not available; the tables below are the DESIGN.md reading S1 and are *pinned* in
``tests/test_oracle_pins.py`` against matrices assembled from the stencil and the
ghost-cell rules alone (no eigenvalue formula involved), against scipy's DCT/DST/FFT,
against dense LU on tiny grids for every boundary combination, and against discrete
eigenmodes.  Pin status of every public function: **pinned** (see that test file).

Conventions:
  * fields are numpy float64 arrays of shape (nz, ny, nx): x fastest, no halo;
  * ``bc`` is a 3x2 nested sequence of 'P' | 'N' | 'D' -- the *pressure* boundary
    condition on the (lower, upper) face of direction x, y, z;
  * u[k,j,i] lives on the +x face of cell (i,j,k), v on the +y face, w on the +z face;
  * dzf[k] (k=0..nz-1) is the width of cell k, dzc[k] (k=0..nz) the distance between the
    centres of cells k-1 and k (mirror ghost centres at both ends).
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "pair_of", "basis", "z_coefficients", "z_matrix_rows", "thomas",
    "apply_laplacian", "poisson_solve", "divergence", "correct_velocity",
    "projection", "is_singular", "uniform_spacing", "pressure_update", "pressure_update_implicit", "chkdt_fields", "chkdt",
    "z_face_coefficients", "helmholtz_solve",
]


# --------------------------------------------------------------------------------------
# helpers
# --------------------------------------------------------------------------------------
def pair_of(bc_dir) -> str:
    """'PP', 'NN', 'DD', 'ND' or 'DN' from a (lower, upper) boundary pair."""
    lo, up = str(bc_dir[0]).upper(), str(bc_dir[1]).upper()
    pair = lo + up
    if pair not in ("PP", "NN", "DD", "ND", "DN"):
        raise ValueError(f"invalid boundary pair {pair!r} (periodic must be two-sided)")
    return pair


def uniform_spacing(nz: int, lz: float):
    """dzc (nz+1), dzf (nz) of a uniform grid: the dzc=dzf=NULL case of the ABI."""
    h = lz / nz
    return np.full(nz + 1, h), np.full(nz, h)


def _cos_pi_frac(t, d):
    """cos(pi*t/d) for integer arrays t and integer d, reduced in integers first."""
    t = np.asarray(t, dtype=np.int64) % (2 * d)
    return np.cos(np.pi * t.astype(np.float64) / d)


def _sin_pi_frac(t, d):
    """sin(pi*t/d) for integer arrays t and integer d, reduced in integers first."""
    t = np.asarray(t, dtype=np.int64) % (2 * d)
    return np.sin(np.pi * t.astype(np.float64) / d)


# --------------------------------------------------------------------------------------
# O2: one-dimensional eigenfunction tables (reading S1 of P:L102-104)
# --------------------------------------------------------------------------------------
def basis(pair: str, n: int):
    """Eigenfunctions of the undivided 1-D second difference with the ghost rule of `pair`.

    Returns (B, lam, w): B[q, j] = b_q(j) (n x n), lam[q] the eigenvalue of
    (phi_{j-1} - 2 phi_j + phi_{j+1}) on b_q, and w[q] = 1 / sum_j b_q(j)^2 the weight of
    the inverse expansion phi_j = sum_q w_q b_q(j) phi^_q   (eq. 6 operators F, F^-1,
    P:L100-104; "different scaling factors" P:L114).
    """
    j = np.arange(n, dtype=np.int64)[None, :]
    if pair == "PP":
        # real Fourier pair: cos(2 pi m j/n), m = 0..floor(n/2); sin(2 pi m j/n), m = 1..ceil(n/2)-1
        mc = np.arange(0, n // 2 + 1, dtype=np.int64)
        ms = np.arange(1, (n + 1) // 2, dtype=np.int64)
        Bc = _cos_pi_frac(2 * mc[:, None] * j, n)
        Bs = _sin_pi_frac(2 * ms[:, None] * j, n)
        B = np.concatenate([Bc, Bs], axis=0)
        m = np.concatenate([mc, ms])
        lam = -4.0 * _sin_pi_frac(m, n) ** 2
    elif pair == "NN":
        q = np.arange(n, dtype=np.int64)
        B = _cos_pi_frac(q[:, None] * (2 * j + 1), 2 * n)
        lam = -4.0 * _sin_pi_frac(q, 2 * n) ** 2
    elif pair == "DD":
        q = np.arange(n, dtype=np.int64)
        B = _sin_pi_frac((q[:, None] + 1) * (2 * j + 1), 2 * n)
        lam = -4.0 * _sin_pi_frac(q + 1, 2 * n) ** 2
    elif pair == "ND":
        q = np.arange(n, dtype=np.int64)
        B = _cos_pi_frac((2 * q[:, None] + 1) * (2 * j + 1), 4 * n)
        lam = -4.0 * _sin_pi_frac(2 * q + 1, 4 * n) ** 2
    elif pair == "DN":
        q = np.arange(n, dtype=np.int64)
        B = _sin_pi_frac((2 * q[:, None] + 1) * (2 * j + 1), 4 * n)
        lam = -4.0 * _sin_pi_frac(2 * q + 1, 4 * n) ** 2
    else:
        raise ValueError(pair)
    w = 1.0 / np.sum(B * B, axis=1)
    return B, lam, w


# --------------------------------------------------------------------------------------
# O1 / O3: z operator on a possibly stretched grid (reading S2 of P:L104)
# --------------------------------------------------------------------------------------
def z_coefficients(dzc, dzf):
    """a_k = 1/(dzf_k dzc_k), c_k = 1/(dzf_k dzc_{k+1}): the composition D.G of the staggered
    divergence and gradient in z, which reduces to 1/dz^2 of eq. 5 on a uniform grid."""
    dzc = np.asarray(dzc, dtype=np.float64)
    dzf = np.asarray(dzf, dtype=np.float64)
    nz = dzf.shape[0]
    assert dzc.shape[0] == nz + 1
    a = 1.0 / (dzf * dzc[:nz])
    c = 1.0 / (dzf * dzc[1:])
    return a, c


def z_matrix_rows(pair_z: str, dzc, dzf):
    """Tridiagonal rows (sub a, diag b, super c) of the z operator with boundary rows folded in
    (O3): ghost = +interior for 'N', -interior for 'D'.  z-periodic is handled by the caller."""
    a, c = z_coefficients(dzc, dzf)
    b = -(a + c)
    lo, up = pair_z[0], pair_z[1]
    if lo == "N":
        b[0] += a[0]
    elif lo == "D":
        b[0] -= a[0]
    if up == "N":
        b[-1] += c[-1]
    elif up == "D":
        b[-1] -= c[-1]
    return a, b, c


def thomas(a, b, c, d):
    """Thomas algorithm without pivoting along axis 0 ("Gauss elimination").

    a, c: (nz,) sub/super diagonals (a[0], c[-1] unused); b: (nz, ...) diagonal, may carry the
    per-mode shift; d: (nz, ...) right-hand sides.  Returns x with the shape of d.
    """
    nz = d.shape[0]
    cp = np.empty_like(d)
    dp = np.empty_like(d)
    denom = b[0]
    cp[0] = c[0] / denom
    dp[0] = d[0] / denom
    for k in range(1, nz):
        denom = b[k] - a[k] * cp[k - 1]
        cp[k] = c[k] / denom
        dp[k] = (d[k] - a[k] * dp[k - 1]) / denom
    x = np.empty_like(d)
    x[nz - 1] = dp[nz - 1]
    for k in range(nz - 2, -1, -1):
        x[k] = dp[k] - cp[k] * x[k + 1]
    return x


def _thomas_singular(a, b, c, d, dzf):
    """O4 (reading S3): the lambda = 0 column of an all-periodic/Neumann problem.  Forward sweep on
    rows 0..nz-2, x[nz-1] = 0, back-substitute, then remove the dzf-weighted mean."""
    nz = d.shape[0]
    x = np.zeros(nz)
    if nz > 1:
        x[: nz - 1] = thomas(a[: nz - 1], b[: nz - 1], c[: nz - 1], d[: nz - 1])
        # x[nz-1] = 0 so the dropped super-diagonal coupling of row nz-2 contributes nothing
    x -= np.sum(x * dzf) / np.sum(dzf)
    return x


def _cyclic_thomas(a, b, c, d):
    """z-periodic column solve (NEXT row f1): Sherman-Morrison on top of ``thomas``."""
    nz = d.shape[0]
    gamma = -b[0]
    bb = np.array(b, dtype=np.float64, copy=True)
    bb[0] = b[0] - gamma
    bb[-1] = b[-1] - c[-1] * a[0] / gamma
    uvec = np.zeros_like(d)
    uvec[0] = gamma
    uvec[-1] = c[-1]
    y = thomas(a, bb, c, d)
    q = thomas(a, bb, c, uvec)
    fact = (y[0] + a[0] * y[-1] / gamma) / (1.0 + q[0] + a[0] * q[-1] / gamma)
    return y - q * fact


def is_singular(bc) -> bool:
    """True if every direction is periodic or Neumann-Neumann (constant null vector)."""
    return all(pair_of(bc[d]) in ("PP", "NN") for d in range(3))


# --------------------------------------------------------------------------------------
# O1: the operator itself, straight from eq. 5 and the ghost rules
# --------------------------------------------------------------------------------------
def _pad_ghost(phi, axis, pair):
    lo = np.take(phi, [0], axis=axis)
    hi = np.take(phi, [-1], axis=axis)
    if pair == "PP":
        glo, ghi = hi, lo
    else:
        glo = lo if pair[0] == "N" else -lo
        ghi = hi if pair[1] == "N" else -hi
    return np.concatenate([glo, phi, ghi], axis=axis)


def apply_laplacian(phi, lx, ly, lz, bc, dzc=None, dzf=None):
    """(L phi)_{ijk} of eq. 5 with ghost cells: P wrap, N mirror, D anti-mirror.
    Stretched z uses a_k, c_k of ``z_coefficients`` (reading S2)."""
    phi = np.asarray(phi, dtype=np.float64)
    nz, ny, nx = phi.shape
    if dzc is None or dzf is None:
        dzc, dzf = uniform_spacing(nz, lz)
    dx, dy = lx / nx, ly / ny
    a, c = z_coefficients(dzc, dzf)
    px = _pad_ghost(phi, 2, pair_of(bc[0]))
    py = _pad_ghost(phi, 1, pair_of(bc[1]))
    pz = _pad_ghost(phi, 0, pair_of(bc[2]))
    out = (px[:, :, :-2] - 2.0 * phi + px[:, :, 2:]) / dx**2
    out += (py[:, :-2, :] - 2.0 * phi + py[:, 2:, :]) / dy**2
    out += a[:, None, None] * (pz[:-2] - phi) + c[:, None, None] * (pz[2:] - phi)
    return out


# --------------------------------------------------------------------------------------
# O2-O5: the eigenfunction-expansion solve, step by step in the paper's order
# --------------------------------------------------------------------------------------
def poisson_solve(f, lx, ly, lz, bc, dzc=None, dzf=None):
    """Solve L Phi = f (eq. 5) by eq. 6: F^x, F^y, tridiagonal solve in z, inverse transforms.

    Naive O(n^2) transforms (matrix products with the tables of ``basis``), Thomas per (q, r)
    mode, singular mode pinned to zero dzf-weighted mean (O4).  Returns Phi, shape (nz, ny, nx).
    """
    f = np.asarray(f, dtype=np.float64)
    nz, ny, nx = f.shape
    if dzc is None or dzf is None:
        dzc, dzf = uniform_spacing(nz, lz)
    dzc = np.asarray(dzc, dtype=np.float64)
    dzf = np.asarray(dzf, dtype=np.float64)
    dx, dy = lx / nx, ly / ny
    px, py, pz = pair_of(bc[0]), pair_of(bc[1]), pair_of(bc[2])

    Bx, lamx, wx = basis(px, nx)
    By, lamy, wy = basis(py, ny)

    # O2: f^(q, r, k) = sum_j Y_r(j) sum_i X_q(i) f(i, j, k)
    fh = np.matmul(f, Bx.T)            # (nz, ny, q)
    fh = np.matmul(By, fh)             # (nz, r, q)

    # O3: (T_z + lam_qr I) Phi^ = f^ for every (q, r)
    lam = lamy[:, None] / dy**2 + lamx[None, :] / dx**2      # (r, q)
    if pz == "PP":
        a, c = z_coefficients(dzc, dzf)
        b = -(a + c)
        solver = _cyclic_thomas
    else:
        a, b, c = z_matrix_rows(pz, dzc, dzf)
        solver = thomas
    bfull = b[:, None, None] + lam[None, :, :]
    singular = is_singular(bc)
    if singular:
        # O4: the exactly-zero eigenvalue sits at q = r = 0 for both PP and NN tables
        assert lam[0, 0] == 0.0
        d00 = fh[:, 0, 0].copy()
        bfull[:, 0, 0] = b - 1.0       # placeholder (non-singular, result discarded) so the vectorised sweep stays finite
    ph = solver(a, bfull, c, fh)
    if singular:
        if pz == "PP":
            # drop the last row of the cyclic system: x[nz-1] = 0 leaves an open tridiagonal system
            x = np.zeros(nz)
            if nz > 1:
                x[: nz - 1] = thomas(a[: nz - 1], b[: nz - 1], c[: nz - 1], d00[: nz - 1])
            x -= np.sum(x * dzf) / np.sum(dzf)
            ph[:, 0, 0] = x
        else:
            ph[:, 0, 0] = _thomas_singular(a, b, c, d00, dzf)

    # O5: Phi(i, j, k) = sum_q w_q X_q(i) sum_r w_r Y_r(j) Phi^(q, r, k)
    ph = np.matmul(By.T * wy[None, :], ph)                 # (nz, j, q)
    ph = np.matmul(ph, wx[:, None] * Bx)                   # (nz, j, i)
    return ph


# --------------------------------------------------------------------------------------
# O6: divergence (eq. 2b) and correction (eq. 2c) on the compact staggered layout
# --------------------------------------------------------------------------------------
def _lower_face(vel, axis, pair, face):
    """Velocity on the lower boundary face of `axis`: wrapped (P), prescribed plane or 0 (N),
    registered plane (D, required)."""
    shape = list(vel.shape)
    shape[axis] = 1
    if pair == "PP":
        return np.take(vel, [-1], axis=axis)
    if face is None:
        if pair[0] == "D":
            raise ValueError("a lower 'D' side needs a registered lower-face plane")
        return np.zeros(shape)
    return np.asarray(face, dtype=np.float64).reshape(shape)


def divergence(u, v, w, lx, ly, lz, bc, dzc=None, dzf=None, lower_face=None):
    """(D u)_{ijk} = (u_i - u_{i-1})/dx + (v_j - v_{j-1})/dy + (w_k - w_{k-1})/dzf_k (eq. 2b,
    staggered arrangement P:L53).  ``lower_face`` maps a direction index to its boundary plane."""
    nz, ny, nx = u.shape
    if dzc is None or dzf is None:
        dzc, dzf = uniform_spacing(nz, lz)
    lower_face = lower_face or {}
    dx, dy = lx / nx, ly / ny
    ul = np.concatenate([_lower_face(u, 2, pair_of(bc[0]), lower_face.get(0)), u], axis=2)
    vl = np.concatenate([_lower_face(v, 1, pair_of(bc[1]), lower_face.get(1)), v], axis=1)
    wl = np.concatenate([_lower_face(w, 0, pair_of(bc[2]), lower_face.get(2)), w], axis=0)
    return ((ul[:, :, 1:] - ul[:, :, :-1]) / dx
            + (vl[:, 1:, :] - vl[:, :-1, :]) / dy
            + (wl[1:] - wl[:-1]) / np.asarray(dzf)[:, None, None])


def correct_velocity(u, v, w, phi, dt, lx, ly, lz, bc, dzc=None, dzf=None, lower_face=None):
    """u -= dt G phi (eq. 2c): u_i -= dt (phi_{i+1}-phi_i)/dx, v_j likewise,
    w_k -= dt (phi_{k+1}-phi_k)/dzc_{k+1}; the phi beyond the upper face follows the ghost rule.
    Returns (u, v, w, lower_face_new) as new arrays."""
    nz, ny, nx = u.shape
    if dzc is None or dzf is None:
        dzc, dzf = uniform_spacing(nz, lz)
    dzc = np.asarray(dzc, dtype=np.float64)
    lower_face = lower_face or {}
    dx, dy = lx / nx, ly / ny
    px = _pad_ghost(phi, 2, pair_of(bc[0]))
    py = _pad_ghost(phi, 1, pair_of(bc[1]))
    pz = _pad_ghost(phi, 0, pair_of(bc[2]))
    un = u - dt * (px[:, :, 2:] - px[:, :, 1:-1]) / dx
    vn = v - dt * (py[:, 2:, :] - py[:, 1:-1, :]) / dy
    wn = w - dt * (pz[2:] - pz[1:-1]) / dzc[1:, None, None]
    new_faces = {}
    for d, (pad, h, ax) in enumerate(((px, dx, 2), (py, dy, 1), (pz, None, 0))):
        if d in lower_face and lower_face[d] is not None:
            pair = pair_of(bc[d])
            face = np.asarray(lower_face[d], dtype=np.float64)
            if pair[0] == "D":
                first = np.take(pad, 1, axis=ax)
                ghost = np.take(pad, 0, axis=ax)
                hh = h if h is not None else dzc[0]
                new_faces[d] = face - dt * (first - ghost).reshape(face.shape) / hh
            else:
                new_faces[d] = face.copy()   # prescribed inflow on an 'N' side is not modified
    return un, vn, wn, new_faces


def projection(u, v, w, dt, lx, ly, lz, bc, dzc=None, dzf=None, lower_face=None):
    """One pressure-projection step (eqs. 2b-2c): f = D u*/dt, L Phi = f, u -= dt G Phi.
    `dt` is the whole factor gamma_k*Delta t.  Returns (u, v, w, Phi, lower_face_new)."""
    f = divergence(u, v, w, lx, ly, lz, bc, dzc, dzf, lower_face) / dt
    phi = poisson_solve(f, lx, ly, lz, bc, dzc, dzf)
    un, vn, wn, faces = correct_velocity(u, v, w, phi, dt, lx, ly, lz, bc, dzc, dzf, lower_face)
    return un, vn, wn, phi, faces


# --------------------------------------------------------------------------------------
# NEXT row f3: pressure update (eq. 2d) and the stable-time-step reduction of Listing 1 (``chkdt``)
# --------------------------------------------------------------------------------------
def pressure_update(p, phi):
    """p^{k+1/2} = p^{k-1/2} + Phi (eq. 2d, explicit diffusion)."""
    return np.asarray(p, dtype=np.float64) + np.asarray(phi, dtype=np.float64)


def pressure_update_implicit(p, phi, coeff, lx, ly, lz, bc, dzc=None, dzf=None):
    """p^{k+1/2} = p^{k-1/2} + Phi - coeff * L Phi with coeff = gamma_k nu dt / 2 (eq. 3e, implicit diffusion);
    L is the Laplacian of eq. 5 with the ghost rules of Phi (``apply_laplacian``)."""
    phi = np.asarray(phi, dtype=np.float64)
    return np.asarray(p, dtype=np.float64) + phi - coeff * apply_laplacian(phi, lx, ly, lz, bc, dzc, dzf)


def _pad_velocity(vel, axis, pair, normal, face):
    """One layer below and above `vel` along `axis` for the face averages of Listing 1 (reading S17): periodic ->
    wrapped; non-periodic -> below: the lower boundary face (registered plane or 0) for the component normal to the
    axis, 0 for a tangential one; above: 0."""
    shape = list(vel.shape)
    shape[axis] = 1
    if pair == "PP":
        lo, hi = np.take(vel, [-1], axis=axis), np.take(vel, [0], axis=axis)
    else:
        lo = _lower_face(vel, axis, pair, face) if normal else np.zeros(shape)
        hi = np.zeros(shape)
    return np.concatenate([lo, vel, hi], axis=axis)


def chkdt_fields(u, v, w, lx, ly, lz, bc, dzc=None, dzf=None, lower_face=None):
    """The three per-face sums of Listing 1, 0-based on the compact layout:

      dtix(i,j,k) = |u(i,j,k)|/dx + 0.25|v(i,j,k)+v(i,j-1,k)+v(i+1,j,k)+v(i+1,j-1,k)|/dy
                                  + 0.25|w(i,j,k)+w(i,j,k-1)+w(i+1,j,k)+w(i+1,j,k-1)|/dzf(k)        (printed)
      dtiy(i,j,k) = 0.25|u(i,j,k)+u(i,j+1,k)+u(i-1,j+1,k)+u(i-1,j,k)|/dx + |v(i,j,k)|/dy
                                  + 0.25|w(i,j,k)+w(i,j+1,k)+w(i,j+1,k-1)+w(i,j,k-1)|/dzf(k)        (lines lost: by symmetry, S15)
      dtiz(i,j,k) = 0.25|u(i,j,k)+u(i-1,j,k)+u(i-1,j,k+1)+u(i,j,k+1)|/dx
                  + 0.25|v(i,j,k)+v(i,j-1,k)+v(i,j-1,k+1)+v(i,j,k+1)|/dy + |w(i,j,k)|/dzc(k+1)      (dzci(k) of the face k+1/2)

    i.e. at the face a component lives on: its own magnitude plus the 4-point averages of the other two."""
    u, v, w = (np.asarray(a, dtype=np.float64) for a in (u, v, w))
    nz, ny, nx = u.shape
    if dzc is None or dzf is None:
        dzc, dzf = uniform_spacing(nz, lz)
    dzc = np.asarray(dzc, dtype=np.float64)
    dzf = np.asarray(dzf, dtype=np.float64)
    lower_face = lower_face or {}
    dxi, dyi = nx / lx, ny / ly
    px, py, pz = pair_of(bc[0]), pair_of(bc[1]), pair_of(bc[2])

    def pad3(a, comp):
        a = _pad_velocity(a, 2, px, comp == 0, lower_face.get(0))
        # the planes registered for y and z have the extent of the unpadded field: they get the same layers along the
        # directions already padded -- wrapped where that direction is periodic (the plane is a layer of the same periodic
        # field, reading S18 "wrapped when periodic"), 0 otherwise (a tangential value beyond a wall)
        wrap_x, wrap_y = ("wrap" if px == "PP" else "constant"), ("wrap" if py == "PP" else "constant")
        fy, fz = lower_face.get(1), lower_face.get(2)
        if fy is not None:
            fy = np.pad(np.asarray(fy, dtype=np.float64).reshape(nz, 1, nx), ((0, 0), (0, 0), (1, 1)), mode=wrap_x)
        a = _pad_velocity(a, 1, py, comp == 1, fy if comp == 1 else None)
        if fz is not None:
            fz = np.pad(np.asarray(fz, dtype=np.float64).reshape(1, ny, nx), ((0, 0), (0, 0), (1, 1)), mode=wrap_x)
            fz = np.pad(fz, ((0, 0), (1, 1), (0, 0)), mode=wrap_y)
        a = _pad_velocity(a, 0, pz, comp == 2, fz if comp == 2 else None)
        return a                                    # index [k+1, j+1, i+1] = cell (i, j, k)

    U, V, W = pad3(u, 0), pad3(v, 1), pad3(w, 2)
    c = slice(1, -1)          # the cell itself
    m = slice(0, -2)          # index - 1
    q = slice(2, None)        # index + 1
    dzfi = (1.0 / dzf)[:, None, None]
    dzci = (1.0 / dzc[1:])[:, None, None]
    dtix = (np.abs(U[c, c, c]) * dxi
            + 0.25 * np.abs(V[c, c, c] + V[c, m, c] + V[c, c, q] + V[c, m, q]) * dyi
            + 0.25 * np.abs(W[c, c, c] + W[m, c, c] + W[c, c, q] + W[m, c, q]) * dzfi)
    dtiy = (0.25 * np.abs(U[c, c, c] + U[c, q, c] + U[c, q, m] + U[c, c, m]) * dxi
            + np.abs(V[c, c, c]) * dyi
            + 0.25 * np.abs(W[c, c, c] + W[c, q, c] + W[m, q, c] + W[m, c, c]) * dzfi)
    dtiz = (0.25 * np.abs(U[c, c, c] + U[c, c, m] + U[q, c, m] + U[q, c, c]) * dxi
            + 0.25 * np.abs(V[c, c, c] + V[c, m, c] + V[q, m, c] + V[q, c, c]) * dyi
            + np.abs(W[c, c, c]) * dzci)
    return dtix, dtiy, dtiz


def chkdt(u, v, w, lx, ly, lz, bc, dzc=None, dzf=None, lower_face=None):
    """dti = max(0, max_ijk(dtix, dtiy, dtiz)) of Listing 1; the stable step of eq. 4 follows
    on the host as min(1.65 dl^2 / nu, sqrt(3) / dti)."""
    dtix, dtiy, dtiz = chkdt_fields(u, v, w, lx, ly, lz, bc, dzc, dzf, lower_face)
    return float(max(0.0, dtix.max(), dtiy.max(), dtiz.max()))


# --------------------------------------------------------------------------------------
# NEXT row f4: the Helmholtz solve of the implicit-diffusion step (eq. 3b; "solved with the same type of
# direct solver"):  (L + alpha I) Phi = f,  alpha = -2/(gamma_k nu dt) < 0 after dividing eq. 3b by -gamma nu dt/2
# --------------------------------------------------------------------------------------
def z_face_coefficients(dzc, dzf, periodic):
    """Second difference in z of a quantity living on the +z FACES (the wall-normal velocity w, staggered arrangement
    P:L53): face k sits between centres k and k+1, at distance dzf_k from the face below and dzf_{k+1} from the one
    above, and its control volume has height dzc_{k+1}:
        (d_zz w)_k = [ (w_{k+1} - w_k)/dzf_{k+1} - (w_k - w_{k-1})/dzf_k ] / dzc_{k+1}
    => a_k = 1/(dzc_{k+1} dzf_k), c_k = 1/(dzc_{k+1} dzf_{k+1}) (dzf wrapped if periodic).  Non-periodic: the unknowns are
    the interior faces k = 0..nz-2 (the face nz-1 is the upper wall); the last returned entry is unused."""
    dzc = np.asarray(dzc, dtype=np.float64)
    dzf = np.asarray(dzf, dtype=np.float64)
    nz = dzf.shape[0]
    up = np.roll(dzf, -1) if periodic else np.concatenate([dzf[1:], [np.inf]])
    a = 1.0 / (dzc[1:] * dzf)
    c = 1.0 / (dzc[1:] * up)
    return a, c


def helmholtz_solve(f, alpha, lx, ly, lz, bc, dzc=None, dzf=None, stagger=None):
    """(L + alpha I) Phi = f with the eigenfunction expansion of eq. 6: the same transforms in x and y, the
    tridiagonal systems shifted by lam_qr + alpha.  alpha < 0 (eq. 3b); with alpha = 0 this is ``poisson_solve`` for a
    non-singular boundary set.  ``bc`` is the ghost rule of the unknown itself ('D': zero on the boundary face, e.g. a
    no-slip wall for a tangential velocity; 'N': zero normal derivative; 'P').

    ``stagger`` = None for a cell-centred unknown, or the direction (0, 1, 2) along which the unknown lives on the
    faces (u: 0, v: 1, w: 2 -- "face-located unknowns in the wall-normal direction").  Along a periodic direction the
    operator is the same as for centres (x, y uniform).  Along z: rows of ``z_face_coefficients``; 'PP' cyclic, 'DD' = walls
    at the lower boundary and at face nz-1 (homogeneous: the wall values do not enter the right-hand side), slot nz-1 is
    returned as it came; 'DN' = wall below, zero normal derivative at the upper boundary face nz-1 (an outflow / free-slip
    top: that face is an unknown, mirrored neighbour above).  Other staggered cases are not implemented: face-located along
    a non-periodic x or y (the node-based DST-I / DCT-I family), and z pairs with a lower 'N' (the lower boundary face
    would be an unknown, and the compact layout has no slot for it): NotImplementedError."""
    f = np.asarray(f, dtype=np.float64)
    nz, ny, nx = f.shape
    if dzc is None or dzf is None:
        dzc, dzf = uniform_spacing(nz, lz)
    dzc = np.asarray(dzc, dtype=np.float64)
    dzf = np.asarray(dzf, dtype=np.float64)
    dx, dy = lx / nx, ly / ny
    px, py, pz = pair_of(bc[0]), pair_of(bc[1]), pair_of(bc[2])
    if stagger in (0, 1) and (px, py)[stagger] != "PP":
        raise NotImplementedError("face-located unknowns along a non-periodic x or y")
    if stagger == 2 and pz not in ("PP", "DD", "DN"):
        raise NotImplementedError("face-located unknowns along z need PP, DD or DN")
    Bx, lamx, wx = basis(px, nx)
    By, lamy, wy = basis(py, ny)
    fh = np.matmul(By, np.matmul(f, Bx.T))
    lam = lamy[:, None] / dy**2 + lamx[None, :] / dx**2 + alpha
    n_solve = nz
    if stagger == 2:
        a, c = z_face_coefficients(dzc, dzf, pz == "PP")
        b = -(a + c)
        if pz == "DD":
            n_solve = nz - 1                   # wall nodes below face 0 and at face nz-1: their couplings drop out
            a, b, c = a[:n_solve], b[:n_solve], c[:n_solve]
        elif pz == "DN":
            # zero normal derivative AT the upper boundary face: face nz-1 is an unknown, the face above it is the mirror
            # image of face nz-2 (ghost cell of width dzf_{nz-1}), so its coupling 1/(dzc_nz dzf_{nz-1}) adds to a_{nz-1}
            a, c = a.copy(), c.copy()
            ghost = 1.0 / (dzc[nz] * dzf[nz - 1])
            b[nz - 1] = -(a[nz - 1] + ghost)
            a[nz - 1] += ghost
            c[nz - 1] = 0.0
        solver = _cyclic_thomas if pz == "PP" else thomas
    elif pz == "PP":
        a, c = z_coefficients(dzc, dzf)
        b = -(a + c)
        solver = _cyclic_thomas
    else:
        a, b, c = z_matrix_rows(pz, dzc, dzf)
        solver = thomas
    ph = np.array(fh, copy=True)
    ph[:n_solve] = solver(a, b[:, None, None] + lam[None, :, :], c, fh[:n_solve])
    ph = np.matmul(By.T * wy[None, :], ph)
    return np.matmul(ph, wx[:, None] * Bx)
