"""Pins of the oracle's Laplacian + boundary rule against what mathematics fixes (no GPU).

Every expected value here is a closed form, a polynomial identity, a dense-matrix brute force or a
convergence rate — none comes from the oracle itself or from the CUDA path.
Cites: PAPER.md:106-114 (Eq. 6, boundary), Q1-Q4; SURVEY.md §8(c) "Pins".
"""
import numpy as np
import pytest

import oracle as O

LAP5, LAP9X4, BOX9 = 0, 1, 2
NOFLUX, PERIODIC = 0, 1


def _grid(nx, ny, h, x0=0.3, y0=-0.2):
    x = x0 + h * np.arange(nx)
    y = y0 + h * np.arange(ny)
    return np.meshgrid(x, y)  # X[j,i], Y[j,i]


def _interior(a, r):
    return a[r:-r, r:-r]


@pytest.mark.parametrize("stencil,r,maxdeg", [(LAP5, 1, 3), (BOX9, 1, 3), (LAP9X4, 2, 5)])
def test_exact_on_polynomials(stencil, r, maxdeg):
    """Interior exactness on all monomials x^p y^q with p+q <= order+1."""
    h = 0.125  # power of two: products are exact-ish, errors stay at roundoff
    X, Y = _grid(13, 11, h)
    for p in range(maxdeg + 1):
        for q in range(maxdeg + 1 - p):
            U = X ** p * Y ** q
            exact = (p * (p - 1) * X ** max(p - 2, 0) * Y ** q if p >= 2 else 0 * X) + \
                    (q * (q - 1) * X ** p * Y ** max(q - 2, 0) if q >= 2 else 0 * X)
            L = O.laplacian(U, h, stencil)
            err = np.max(np.abs(_interior(L - exact, r)))
            scale = max(1.0, np.max(np.abs(U))) / h ** 2
            assert err < 64 * np.finfo(float).eps * scale, (p, q, err)


def test_leading_error_terms():
    """LAP5: x^4 -> 12x^2 + 2h^2.  BOX9: x^4 -> 12x^2 + 2h^2 and x^2y^2 -> 2(x^2+y^2) + 2h^2/3
    (error (h^2/12) lap^2, the isotropic member, Q1).  LAP9X4: x^6 -> 30x^4 - 8h^4."""
    h = 0.25
    X, Y = _grid(12, 12, h)
    e = lambda L, ref, r: np.max(np.abs(_interior(L - ref, r)))
    assert e(O.laplacian(X ** 4, h, LAP5), 12 * X ** 2 + 2 * h ** 2, 1) < 1e-10
    assert e(O.laplacian(X ** 4, h, BOX9), 12 * X ** 2 + 2 * h ** 2, 1) < 1e-10
    assert e(O.laplacian(X ** 2 * Y ** 2, h, BOX9), 2 * (X ** 2 + Y ** 2) + 2 * h ** 2 / 3, 1) < 1e-10
    assert e(O.laplacian(X ** 2 * Y ** 2, h, LAP5), 2 * (X ** 2 + Y ** 2), 1) < 1e-10
    # 4th-order cross: (-1/12)(f(2h)+f(-2h)) + (4/3)(f(h)+f(-h)) - (5/2) f(0) on x^6:
    # f'' + (2/6!)( (4/3) - (64/12) ) h^4 f^(6) = 30x^4 + (2/720)(-4)(720) h^4 = 30 x^4 - 8 h^4
    assert e(O.laplacian(X ** 6, h, LAP9X4), 30 * X ** 4 - 8 * h ** 4, 2) < 1e-8


def _lam(theta, stencil):
    """Symbol of the 1-D second difference, times dx^2."""
    if stencil == LAP9X4:
        return 2 * (4.0 / 3.0) * (np.cos(theta) - 1) + 2 * (-1.0 / 12.0) * (np.cos(2 * theta) - 1)
    return 2 * (np.cos(theta) - 1)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4, BOX9])
@pytest.mark.parametrize("nx,ny,kx,ky", [(17, 12, 3, 2), (9, 9, 0, 4), (24, 31, 23, 1), (5, 5, 4, 4)])
def test_cosine_modes_are_eigenvectors_noflux(stencil, nx, ny, kx, ky):
    """With index reflection about the boundary nodes, cos(pi kx i/(nx-1)) cos(pi ky j/(ny-1)) is an
    exact eigenvector, boundary rows included (Q3)."""
    h = 0.04
    tx, ty = np.pi * kx / (nx - 1), np.pi * ky / (ny - 1)
    I, J = np.meshgrid(np.arange(nx), np.arange(ny))
    U = np.cos(tx * I) * np.cos(ty * J)
    if stencil == BOX9:
        # axial 2/3, diagonal 1/6: symbol (2/3)(lx + ly) + (1/6)(4 cx cy - 4)
        lam = (2 / 3) * (_lam(tx, 0) + _lam(ty, 0)) + (1 / 6) * (4 * np.cos(tx) * np.cos(ty) - 4)
    else:
        lam = _lam(tx, stencil) + _lam(ty, stencil)
    L = O.laplacian(U, h, stencil)
    assert np.max(np.abs(L - lam / h ** 2 * U)) < 2e-12 / h ** 2 * 1e-1


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4, BOX9])
def test_fourier_modes_periodic(stencil):
    nx, ny, kx, ky, h = 16, 10, 3, 2, 0.03
    tx, ty = 2 * np.pi * kx / nx, 2 * np.pi * ky / ny
    I, J = np.meshgrid(np.arange(nx), np.arange(ny))
    U = np.cos(tx * I + 0.3) * np.sin(ty * J - 0.1)
    if stencil == BOX9:
        lam = (2 / 3) * (_lam(tx, 0) + _lam(ty, 0)) + (1 / 6) * (4 * np.cos(tx) * np.cos(ty) - 4)
    else:
        lam = _lam(tx, stencil) + _lam(ty, stencil)
    L = O.laplacian(U, h, stencil, PERIODIC)
    assert np.max(np.abs(L - lam / h ** 2 * U)) < 1e-10


def _op1d(n, stencil, boundary):
    """Dense 1-D second-difference matrix (times dx^2), built entry by entry."""
    taps = {1: 1.0} if stencil != LAP9X4 else {1: 4.0 / 3.0, 2: -1.0 / 12.0}
    A = np.zeros((n, n))
    for i in range(n):
        for m, c in taps.items():
            for s in (+1, -1):
                t = i + s * m
                if boundary == PERIODIC:
                    t %= n
                elif t < 0:
                    t = -t
                elif t > n - 1:
                    t = 2 * (n - 1) - t
                A[i, t] += c
                A[i, i] -= c
    return A


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
@pytest.mark.parametrize("boundary", [NOFLUX, PERIODIC])
@pytest.mark.parametrize("nx,ny", [(5, 5), (7, 6), (6, 9)])
def test_tiny_grid_dense_matrix(stencil, boundary, nx, ny):
    """Brute force: lap = I (x) Ax + Ay (x) I as explicit (nx ny)^2 matrices."""
    rng = np.random.default_rng(7)
    U = rng.standard_normal((ny, nx))
    h = 0.5
    Ax, Ay = _op1d(nx, stencil, boundary), _op1d(ny, stencil, boundary)
    big = np.kron(np.eye(ny), Ax) + np.kron(Ay, np.eye(nx))
    ref = (big @ U.reshape(-1)).reshape(ny, nx) / h ** 2
    assert np.max(np.abs(O.laplacian(U, h, stencil, boundary) - ref)) < 1e-12


def test_box9_tiny_grid_dense():
    rng = np.random.default_rng(8)
    nx, ny, h = 6, 5, 0.25
    U = rng.standard_normal((ny, nx))
    refl = lambda t, n: -t if t < 0 else (2 * (n - 1) - t if t > n - 1 else t)
    ref = np.zeros_like(U)
    for j in range(ny):
        for i in range(nx):
            acc = -(10.0 / 3.0) * U[j, i]
            for dj in (-1, 0, 1):
                for di in (-1, 0, 1):
                    if di == 0 and dj == 0:
                        continue
                    wgt = 2.0 / 3.0 if (di == 0 or dj == 0) else 1.0 / 6.0
                    acc += wgt * U[refl(j + dj, ny), refl(i + di, nx)]
            ref[j, i] = acc / h ** 2
    assert np.max(np.abs(O.laplacian(U, h, BOX9) - ref)) < 1e-12


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4, BOX9])
def test_uniform_field_gives_exact_zero(stencil):
    U = np.full((9, 11), 0.7312345678912345)
    assert np.all(O.laplacian(U, 0.04, stencil) == 0.0)
    assert np.all(O.laplacian(U, 0.04, stencil, PERIODIC) == 0.0)


@pytest.mark.parametrize("stencil", [LAP5, LAP9X4])
def test_trapezoid_sum_conserved(stencil):
    """sum_ij w_i w_j lap(U)_ij = 0 with w = 1/2 on boundary nodes (index reflection conserves the
    trapezoid-rule integral, not the plain sum)."""
    rng = np.random.default_rng(3)
    ny, nx = 14, 19
    U = rng.standard_normal((ny, nx))
    wx, wy = np.ones(nx), np.ones(ny)
    wx[[0, -1]] = 0.5
    wy[[0, -1]] = 0.5
    L = O.laplacian(U, 1.0, stencil)
    assert abs(np.sum(wy[:, None] * wx[None, :] * L)) < 1e-12
    assert abs(np.sum(L)) > 1e-3  # the plain sum is NOT conserved: it would be under edge replication
    assert abs(np.sum(O.laplacian(U, 1.0, stencil, PERIODIC))) < 1e-12


@pytest.mark.parametrize("stencil,order", [(LAP5, 2), (BOX9, 2), (LAP9X4, 4)])
def test_spatial_order_including_boundary(stencil, order):
    """Smooth Neumann-compatible function on [0,1]^2: max error over ALL nodes (boundary included)
    falls as h^order, because index reflection is an even extension."""
    errs = []
    for n in (17, 33, 65):
        h = 1.0 / (n - 1)
        x = h * np.arange(n)
        X, Y = np.meshgrid(x, x)
        U = np.cos(np.pi * X) * np.cos(2 * np.pi * Y)
        exact = -(np.pi ** 2 + 4 * np.pi ** 2) * U
        errs.append(np.max(np.abs(O.laplacian(U, h, stencil) - exact)))
    r1, r2 = np.log2(errs[0] / errs[1]), np.log2(errs[1] / errs[2])
    assert abs(r1 - order) < 0.15 and abs(r2 - order) < 0.1, (errs, r1, r2)


def test_literal_displacement_flip_is_not_what_we_do():
    """DESIGN.md Q3: at node 1 the offset -2 must reach node 1 (index reflection), not node 3."""
    n, h = 9, 1.0
    U = np.zeros((n, n))
    U[4, 3] = 1.0  # a spike at i = 3, row 4
    L = O.laplacian(U, h, LAP9X4)
    # the row-4 stencil at i = 1 sees i+2 = 3 once (weight -1/12) and nothing through the mirror
    assert L[4, 1] == pytest.approx(-1.0 / 12.0, abs=1e-15)
    U[:] = 0.0
    U[4, 1] = 1.0
    L = O.laplacian(U, h, LAP9X4)
    # at i = 1: centre -5/2 (x) -5/2 (y) and the reflected offset -2 -> node 1 itself: -1/12
    assert L[4, 1] == pytest.approx(-5.0 - 1.0 / 12.0, abs=1e-14)
    # at i = 0: both +-1 neighbours are node 1: 2 * 4/3
    assert L[4, 0] == pytest.approx(8.0 / 3.0, abs=1e-14)


def test_rejects_too_small_grids():
    with pytest.raises(ValueError):
        O.laplacian(np.zeros((4, 9)), 1.0, LAP9X4)
    with pytest.raises(ValueError):
        O.laplacian(np.zeros((9, 2)), 1.0, LAP5)
