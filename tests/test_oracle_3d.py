"""Pins of the 3-D extension of the oracle (no GPU): the 7-point
and the 13-point 4th-order cross Laplacian with the per-axis boundary rule of the 2-D path, and the
same integrators on top of them.  Nothing here compares the oracle with itself: polynomial
exactness, closed-form eigenvalues and amplification factors, the conserved trapezoid integral, a
dense-matrix brute force on a tiny grid, and the reduction of a z-independent state to the (already
pinned) 2-D problem.
Cites: PAPER.md:108-114 (stencil, boundary), :116-118 (integrators), :208 (3-D); Q3, Q4, f4.
"""
import itertools

import numpy as np
import pytest

import oracle as O

FHN, KARMA, BOCF = 0, 1, 2
LAP5, LAP9X4, BOX9 = 0, 1, 2          # in 3-D: 7-point, 13-point cross, (none)
EULER, HEUN, RK4 = 0, 1, 2


def sch(stencil, integrator, boundary=0):
    return O.scheme_bits(stencil, integrator, boundary, 0)


def karma_as_pure_diffusion(D):
    p = O.default_params(KARMA)
    p[0], p[1], p[2] = D, 1e300, 1e300
    return p


def lam1d(theta, stencil):
    if stencil == LAP9X4:
        return 2 * (4 / 3) * (np.cos(theta) - 1) - 2 * (1 / 12) * (np.cos(2 * theta) - 1)
    return 2 * (np.cos(theta) - 1)


@pytest.mark.parametrize("stencil,order", [(LAP5, 3), (LAP9X4, 5)])
def test_exact_on_polynomials_interior(stencil, order):
    """Every monomial x^p y^q z^r of total degree <= 3 (7-point) / <= 5 (13-point) is differentiated
    exactly at the interior nodes; the first inexact one has the textbook error term."""
    n, h = 11, 0.1
    r = 2 if stencil == LAP9X4 else 1
    k, j, i = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    x, y, z = (i - 5) * h, (j - 5) * h, (k - 5) * h
    inner = (slice(r, n - r),) * 3
    for p, q, s in itertools.product(range(order + 1), repeat=3):
        if p + q + s > order:
            continue
        U = x ** p * y ** q * z ** s
        exact = (p * (p - 1) * x ** max(p - 2, 0) * y ** q * z ** s
                 + q * (q - 1) * x ** p * y ** max(q - 2, 0) * z ** s
                 + s * (s - 1) * x ** p * y ** q * z ** max(s - 2, 0))
        L = O.laplacian3d(U, h, stencil)
        assert np.max(np.abs(L[inner] - exact[inner])) < 2e-10, (p, q, s)
    if stencil == LAP5:        # t^4: error (h^2/12) d^4/dt^4 = 2 h^2, the same along every axis
        for t in (x, y, z):
            L = O.laplacian3d(t ** 4, h, stencil)
            assert np.allclose(L[inner] - 12 * t[inner] ** 2, 2 * h * h, atol=1e-10)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
def test_cosine_modes_are_eigenvectors_with_mirror_boundary(stencil):
    """Index reflection about the boundary nodes (Q3) is an even extension in every axis:
    cos x cos y cos modes are exact eigenvectors, boundary nodes included, with eigenvalue
    [lam(tx) + lam(ty) + lam(tz)] / dx^2."""
    nx, ny, nz, h = 13, 9, 7, 0.03
    kx, ky, kz = 3, 2, 1
    tx, ty, tz = np.pi * kx / (nx - 1), np.pi * ky / (ny - 1), np.pi * kz / (nz - 1)
    K, J, I = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    mode = np.cos(tx * I) * np.cos(ty * J) * np.cos(tz * K)
    lam = (lam1d(tx, stencil) + lam1d(ty, stencil) + lam1d(tz, stencil)) / h ** 2
    L = O.laplacian3d(mode, h, stencil)
    assert np.max(np.abs(L - lam * mode)) < 1e-9 * abs(lam)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
def test_periodic_fourier_modes(stencil):
    nx, ny, nz, h = 8, 6, 5, 0.05
    K, J, I = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    tx, ty, tz = 2 * np.pi * 1 / nx, 2 * np.pi * 2 / ny, 2 * np.pi * 1 / nz
    mode = np.cos(tx * I + 0.3) * np.sin(ty * J) * np.cos(tz * K - 1.0)
    lam = (lam1d(tx, stencil) + lam1d(ty, stencil) + lam1d(tz, stencil)) / h ** 2
    L = O.laplacian3d(mode, h, stencil, boundary=1)
    assert np.max(np.abs(L - lam * mode)) < 1e-9 * abs(lam)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
def test_dense_matrix_brute_force_tiny_grid(stencil):
    """5 x 6 x 5: the operator assembled as Kronecker sums of explicitly written 1-D matrices
    (rows typed from the weights (1,-2,1) and (-1,16,-30,16,-1)/12 with reflected indices)."""
    nx, ny, nz, h = 5, 6, 5, 0.2
    def one_d(n):
        A = np.zeros((n, n))
        w = {LAP5: {0: -2.0, 1: 1.0}, LAP9X4: {0: -30 / 12, 1: 16 / 12, 2: -1 / 12}}[stencil]
        for i in range(n):
            for m, c in w.items():
                for sgn in ((0,) if m == 0 else (-1, 1)):
                    t = i + sgn * m
                    t = -t if t < 0 else (2 * (n - 1) - t if t > n - 1 else t)
                    A[i, t] += c
        return A / h ** 2
    Ax, Ay, Az = one_d(nx), one_d(ny), one_d(nz)
    rng = np.random.default_rng(3)
    U = rng.standard_normal((nz, ny, nx))
    ref = (np.einsum("ab,kjb->kja", Ax, U) + np.einsum("ab,kbi->kai", Ay, U) + np.einsum("ab,bji->aji", Az, U))
    assert np.max(np.abs(O.laplacian3d(U, h, stencil) - ref)) < 1e-11 / h ** 2 * 1e-1
    assert np.all(O.laplacian3d(np.full((nz, ny, nx), 3.7), h, stencil) == 0.0)      # difference form


def test_rejects_box_stencil_and_thin_grids():
    with pytest.raises(ValueError):
        O.laplacian3d(np.zeros((5, 5, 5)), 0.1, BOX9)
    with pytest.raises(ValueError):
        O.laplacian3d(np.zeros((4, 9, 9)), 0.1, LAP9X4)
    with pytest.raises(ValueError):
        O.step3d(FHN, np.zeros((2, 5, 5, 5)), 0.1, 1e-3, sch(BOX9, RK4), 1)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
@pytest.mark.parametrize("integrator", [EULER, HEUN, RK4])
def test_amplification_factor_on_eigenmode(stencil, integrator):
    """Pure diffusion of a 3-D cosine mode: amplitude R(dt D lambda)^n after n steps."""
    Rf = {EULER: lambda z: 1 + z, HEUN: lambda z: 1 + z + z ** 2 / 2,
          RK4: lambda z: 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24}[integrator]
    nx, ny, nz, h, D = 11, 8, 6, 0.0262, 0.0011
    dt = 0.5 * h * h / (6 * D)                   # half the 3-D explicit limit dx^2 / (6 D)
    tx, ty, tz = np.pi * 2 / (nx - 1), np.pi * 3 / (ny - 1), np.pi * 1 / (nz - 1)
    K, J, I = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    mode = np.cos(tx * I) * np.cos(ty * J) * np.cos(tz * K)
    Z = np.stack([0.7 * mode, np.full_like(mode, 0.25)])
    n = 20
    out = O.step3d(KARMA, Z, h, dt, sch(stencil, integrator), n, params=karma_as_pure_diffusion(D))
    z = dt * D * (lam1d(tx, stencil) + lam1d(ty, stencil) + lam1d(tz, stencil)) / h ** 2
    assert np.max(np.abs(out[0] - 0.7 * Rf(z) ** n * mode)) < 5e-14
    assert np.all(out[1] == 0.25)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
def test_trapezoid_integral_conserved(stencil):
    """No-flux walls: the trapezoid-weighted sum (1/2 on boundary nodes per axis) is conserved under
    pure diffusion (per axis)."""
    rng = np.random.default_rng(8)
    nx, ny, nz, h, D = 9, 8, 7, 0.0262, 0.0011
    Z = np.stack([rng.uniform(0, 3, (nz, ny, nx)), np.zeros((nz, ny, nx))])
    w = lambda n: np.r_[0.5, np.ones(n - 2), 0.5]
    Wt = w(nz)[:, None, None] * w(ny)[None, :, None] * w(nx)[None, None, :]
    out = O.step3d(KARMA, Z, h, 0.5 * h * h / (6 * D), sch(stencil, RK4), 30, params=karma_as_pure_diffusion(D))
    assert abs(np.sum(Wt * out[0]) - np.sum(Wt * Z[0])) < 1e-11 * np.sum(Wt * Z[0])
    assert np.max(np.abs(out[0] - Z[0])) > 1e-2


@pytest.mark.parametrize("model", [FHN, KARMA, BOCF])
@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
def test_z_independent_state_is_the_2d_problem(model, stencil):
    """Planes identical in z: the z-differences vanish exactly, so every plane follows the pinned
    2-D oracle bitwise; and a uniform state follows the scalar ODE (nothing diffuses)."""
    rng = np.random.default_rng(model)
    nv = O.num_fields(model)
    plane = rng.uniform(0.05, 0.9, (nv, 9, 11))
    Z = np.repeat(plane[:, None], 6, axis=1)
    h = {FHN: 0.04, KARMA: 0.0262, BOCF: 0.03}[model]
    D = {FHN: 1.5, KARMA: 0.0011, BOCF: 1.171e-3}[model]
    dt = 0.5 * h * h / (6 * D)
    out3 = O.step3d(model, Z, h, dt, sch(stencil, RK4), 12)
    out2 = O.step(model, plane, h, dt, sch(stencil, RK4), 12)
    for k in range(6):
        assert np.array_equal(out3[:, k], out2)
