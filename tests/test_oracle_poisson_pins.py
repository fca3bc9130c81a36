"""Pins for the oracle's free-space Poisson solve and field (reading R19; "the Poisson equation is solved in
the bunch rest frame").  Independent of the oracle's code: Coulomb's law, 3-D quadrature of 1/r over a cell in
multi-precision arithmetic, linearity / translation, the analytic potential and field of a Gaussian bunch with second-order
convergence, exactness of the difference stencils on polynomials."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle as O

K = 1.0 / (4.0 * math.pi * O.EPS0)


@pytest.mark.parametrize("box", [(1.0, 1.0, 1.0), (1e-3, 2e-3, 0.5e-3), (1.0, 1.0, 7.0)])
def test_self_term_is_the_cell_average_of_one_over_r(box):
    """G(0) = (1/V) int_cell 1/r dV by nested tanh-sinh quadrature over one octant (the integrand is singular at the corner)."""
    mp.mp.dps = 20
    a, b, c = [mp.mpf(v) / 2 for v in box]
    inner = lambda x, y: mp.quad(lambda z: 1 / mp.sqrt(x * x + y * y + z * z), [0, c])
    # int_0^c dz / sqrt(s^2 + z^2) = asinh(c / s): use it to keep the quadrature two-dimensional and accurate
    f = lambda x, y: mp.asinh(c / mp.sqrt(x * x + y * y))
    assert abs(inner(mp.mpf("0.3") * a, mp.mpf("0.7") * b) - f(mp.mpf("0.3") * a, mp.mpf("0.7") * b)) < mp.mpf(10) ** -12
    octant = mp.quad(f, [0, a], [0, b])
    ref = 8 * octant / (8 * a * b * c)
    got = O.green_self(*box)
    assert abs(got - ref) <= 1e-9 * ref
    if box == (1.0, 1.0, 1.0):
        assert abs(got - 2.38007736) < 1e-7


def test_point_charge_gives_coulomb_potential_on_an_anisotropic_stretched_grid():
    d, gz = (1e-3, 2e-3, 0.5e-3), 3.0
    rho = np.zeros((7, 6, 9))
    rho[2, 4, 5] = 2e-10
    phi = O.poisson(rho, d, gz)
    for (k, j, i) in [(2, 4, 6), (0, 0, 0), (6, 5, 8), (2, 1, 5), (5, 4, 5)]:
        r = math.sqrt(((i - 5) * d[0]) ** 2 + ((j - 4) * d[1]) ** 2 + ((k - 2) * gz * d[2]) ** 2)
        assert abs(phi[k, j, i] - K * 2e-10 / r) <= 4e-16 * K * 2e-10 / r
    assert abs(phi[2, 4, 5] - K * 2e-10 * O.green_self(d[0], d[1], gz * d[2])) <= 4e-16 * phi[2, 4, 5]


def test_linearity_and_translation_invariance():
    rng = np.random.default_rng(2)
    d = (1.0, 1.5, 0.8)
    a = np.zeros((8, 8, 8))
    b = np.zeros((8, 8, 8))
    a[1:5, 2:6, 1:4] = rng.uniform(0, 1e-9, (4, 4, 3))
    b[3:7, 1:3, 4:8] = rng.uniform(-1e-9, 1e-9, (4, 2, 4))
    pa, pb, pab = O.poisson(a, d), O.poisson(b, d), O.poisson(2.0 * a - 3.0 * b, d)
    assert np.max(np.abs(pab - (2.0 * pa - 3.0 * pb))) <= 1e-14 * np.max(np.abs(pab))
    shifted = np.roll(a, (2, 1, 3), axis=(0, 1, 2))           # content stays inside the grid
    ps = O.poisson(shifted, d)
    assert np.max(np.abs(ps[3:7, 3:7, 4:7] - pa[1:5, 2:6, 1:4])) <= 1e-14 * np.max(np.abs(pa))


def gaussian_node_charges(n, sigma, half_width, Q):
    ax = np.linspace(-half_width, half_width, n)
    d = ax[1] - ax[0]
    Z, Y, X = np.meshgrid(ax, ax, ax, indexing="ij")
    dens = np.exp(-(X * X + Y * Y + Z * Z) / (2 * sigma * sigma)) / ((2 * math.pi) ** 1.5 * sigma ** 3)
    return Q * dens * d ** 3, ax, d, (X, Y, Z)


def test_gaussian_bunch_potential_and_field_converge_to_the_analytic_solution():
    """phi(r) = Q erf(r / (sqrt2 sigma)) / (4 pi eps0 r), phi(0) = Q sqrt(2/pi) / (4 pi eps0 sigma); second order in d."""
    sigma, Q = 1e-3, 1e-9
    errs = []
    for n in (13, 25):
        rho, ax, d, (X, Y, Z) = gaussian_node_charges(n, sigma, 4e-3, Q)
        phi = O.poisson(rho, (d, d, d))
        R = np.sqrt(X * X + Y * Y + Z * Z)
        with np.errstate(invalid="ignore", divide="ignore"):
            ref = K * Q * np.vectorize(math.erf)(R / (math.sqrt(2) * sigma)) / R
        ref[R == 0] = K * Q * math.sqrt(2 / math.pi) / sigma
        errs.append(np.max(np.abs(phi - ref)) / ref.max())
    assert errs[1] < 5e-3 and errs[0] / errs[1] > 3.0            # ~ d^2
    # field on the finer grid against the analytic radial field, away from the faces
    Ex, Ey, Ez = O.efield(phi, (d, d, d))
    with np.errstate(invalid="ignore", divide="ignore"):
        Er = K * Q / R ** 2 * (np.vectorize(math.erf)(R / (math.sqrt(2) * sigma))
                               - math.sqrt(2 / math.pi) * R / sigma * np.exp(-R * R / (2 * sigma * sigma)))
        refx = np.where(R > 0, Er * X / R, 0.0)
        refz = np.where(R > 0, Er * Z / R, 0.0)
    inner = (slice(2, -2),) * 3
    scale = np.nanmax(np.abs(refx))
    assert np.max(np.abs(Ex[inner] - refx[inner])) <= 5e-2 * scale          # d = sigma/3: O(d^2) truncation of phi and of the stencil
    assert np.max(np.abs(Ez[inner] - refz[inner])) <= 5e-2 * scale
    assert np.max(np.abs(Ex[inner] + Ex[inner][:, :, ::-1])) <= 1e-9 * scale      # odd in x


def test_field_stencils_are_exact_on_polynomials_and_use_the_stretched_spacing():
    d, gz = (0.5, 0.25, 2.0), 1.5
    nx, ny, nz = 6, 5, 7
    x = d[0] * np.arange(nx)[None, None, :]
    y = d[1] * np.arange(ny)[None, :, None]
    z = gz * d[2] * np.arange(nz)[:, None, None]
    phi = 3.0 * x + x * x - 2.0 * y * y + 0.5 * z * z + x * y + 0 * (x + y + z)
    Ex, Ey, Ez = O.efield(phi, d, gz)
    X, Y, Zz = np.broadcast_arrays(x, y, z)
    # centred differences are exact on quadratics
    assert np.allclose(Ex[:, :, 1:-1], -(3.0 + 2.0 * X + Y)[:, :, 1:-1], rtol=0, atol=1e-12)
    assert np.allclose(Ey[:, 1:-1, :], -(-4.0 * Y + X)[:, 1:-1, :], rtol=0, atol=1e-12)
    assert np.allclose(Ez[1:-1], -(Zz)[1:-1], rtol=0, atol=1e-12)
    # one-sided first-order differences at the faces: exact derivative at the half point
    assert np.allclose(Ex[:, :, 0], -(3.0 + 2.0 * (X[:, :, 0] + d[0] / 2) + Y[:, :, 0]), atol=1e-12)
    assert np.allclose(Ez[-1], -(Zz[-1] - gz * d[2] / 2), atol=1e-12)


def test_invalid_arguments():
    with pytest.raises(ValueError):
        O.poisson(np.zeros((1, 4, 4)), (1, 1, 1))
    with pytest.raises(ValueError):
        O.poisson(np.zeros((4, 4, 4)), (1, 1, 1), gz=0.0)


def test_sampled_sum_equals_the_full_sum():
    rng = np.random.default_rng(4)
    rho = rng.uniform(0, 1e-12, (6, 7, 5))
    d, gz = (1e-3, 1.2e-3, 0.7e-3), 2.0
    full = O.poisson(rho, d, gz).reshape(-1)
    idx = np.array([0, 17, 209, 100, 3])
    assert np.array_equal(O.poisson_sample(rho, d, gz, idx), full[idx])
