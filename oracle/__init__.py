"""ctypes loader for the CPU oracle (oracle/bt_oracle.c).

TEST INFRASTRUCTURE.  May be imported only by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Imports nothing from paper_2208_02382_b200.

All functions work in place on contiguous float64 numpy arrays, argument meaning as in
bt_oracle.c (readings R1-R13, SURVEY.md 8(c) / DESIGN.md).
"""
import ctypes as C

import numpy as np

from . import build as _build

DRIFT, QUAD, SBEND, DIPEDGE, MULTIPOLE, SHORTRF, DRIFT_EXACT, SHORTRF_SIN, QUAD_CHROMATIC = range(9)
_TYPE_BY_NAME = {"drift": DRIFT, "quad": QUAD, "sbend": SBEND, "dipedge": DIPEDGE,
                 "multipole": MULTIPOLE, "shortrf": SHORTRF, "drift_exact": DRIFT_EXACT, "shortrf_sin": SHORTRF_SIN, "quad_chromatic": QUAD_CHROMATIC}

ELEMENT_DTYPE = np.dtype([("type", "<i4"), ("nslice", "<i4"), ("ds", "<f8"), ("p", "<f8", (6,))])
assert ELEMENT_DTYPE.itemsize == 64

_lib = None
_dp = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        L.orc_ref_from_kinetic.argtypes = [C.c_double, C.c_double, _dp, _dp, _dp]
        L.orc_ref_from_kinetic.restype = None
        L.orc_num_threads.restype = C.c_int
        L.orc_set_num_threads.argtypes = [C.c_int]
        L.orc_track.argtypes = [C.c_int64] + [_dp] * 6 + [C.c_void_p, C.c_int32, C.c_int32, _dp, _dp]
        L.orc_track.restype = C.c_int
        L.orc_deposit_cic.argtypes = [C.c_int64, _dp, _dp, _dp, C.c_int32, C.c_int32, C.c_int32,
                                      _dp, _dp, C.c_double, C.c_double, _dp, C.c_int]
        L.orc_deposit_cic.restype = C.c_int64
        L.orc_gather_kick.argtypes = [C.c_int64] + [_dp] * 6 + [C.c_int32] * 3 + [_dp, _dp] + [_dp] * 3 + [_dp, C.c_double]
        L.orc_gather_kick.restype = C.c_int64
        L.orc_gather_field.argtypes = [C.c_int64] + [_dp] * 3 + [C.c_int32] * 3 + [_dp, _dp] + [_dp] * 3 + [C.c_double] + [_dp] * 3
        L.orc_gather_field.restype = C.c_int64
        L.orc_deposit_tsc.argtypes = L.orc_deposit_cic.argtypes
        L.orc_deposit_tsc.restype = C.c_int64
        L.orc_gather_kick_tsc.argtypes = L.orc_gather_kick.argtypes
        L.orc_gather_kick_tsc.restype = C.c_int64
        L.orc_green_self.argtypes = [C.c_double] * 3
        L.orc_green_self.restype = C.c_double
        L.orc_poisson.argtypes = [C.c_int32] * 3 + [_dp, C.c_double, _dp, _dp]
        L.orc_poisson.restype = C.c_int
        L.orc_poisson_sample.argtypes = [C.c_int32] * 3 + [_dp, C.c_double, _dp, C.c_int64, C.POINTER(C.c_int64), _dp]
        L.orc_poisson_sample.restype = C.c_int
        L.orc_efield.argtypes = [C.c_int32] * 3 + [_dp, C.c_double, _dp, _dp, _dp, _dp]
        L.orc_efield.restype = C.c_int
        L.orc_moments.argtypes = [C.c_int64, C.POINTER(_dp), _dp, _dp]
        L.orc_moments.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous, "need contiguous float64"
    return a.ctypes.data_as(_dp)


def _v3(v):
    a = np.ascontiguousarray(np.asarray(v, dtype=np.float64))
    assert a.shape == (3,)
    return a


def num_threads():
    return int(lib().orc_num_threads())


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))


def ref_from_kinetic(kin_MeV, mass_MeV):
    """R2 -> (gamma0, beta0*gamma0, beta0)."""
    g, bg, b = C.c_double(), C.c_double(), C.c_double()
    lib().orc_ref_from_kinetic(kin_MeV, mass_MeV, C.byref(g), C.byref(bg), C.byref(b))
    return g.value, bg.value, b.value


def pack_lattice(lattice):
    """lattice: iterable of (kind, ds, nslice, params...) tuples (workloads format) -> struct array."""
    lattice = list(lattice)
    arr = np.zeros(len(lattice), dtype=ELEMENT_DTYPE)
    for i, el in enumerate(lattice):
        kind, ds, nslice = el[0], el[1], el[2]
        params = list(el[3:])
        arr[i]["type"] = _TYPE_BY_NAME[kind] if isinstance(kind, str) else int(kind)
        arr[i]["nslice"] = nslice
        arr[i]["ds"] = ds
        arr[i]["p"][: len(params)] = params
    return arr


def track(coords, lattice, nturns, gamma, s=0.0):
    """In place on coords = [x, px, y, py, t, pt]; returns (gamma_after, s_after)."""
    elems = lattice if isinstance(lattice, np.ndarray) else pack_lattice(lattice)
    assert elems.dtype == ELEMENT_DTYPE and elems.flags.c_contiguous
    n = coords[0].shape[0]
    assert all(c.shape == (n,) for c in coords)
    g, ss = C.c_double(gamma), C.c_double(s)
    rc = lib().orc_track(n, *[_p(c) for c in coords], elems.ctypes.data, len(elems), nturns,
                         C.byref(g), C.byref(ss))
    if rc != 0:
        raise ValueError("oracle: invalid lattice / arguments")
    return g.value, ss.value


def deposit_cic(x, y, t, shape, lo, d, q_weight, zscale=1.0, rho=None, order=1):
    """Returns (rho[nz,ny,nx] charge per node, n_inside). rho given => accumulate onto it.
    order = 1: CIC (R11); order = 2: quadratic B-spline (R16, PAPER.md l.60 set_particle_shape(2))."""
    nx, ny, nz = shape
    zero_first = rho is None
    if rho is None:
        rho = np.zeros((nz, ny, nx), dtype=np.float64)
    lo, d = _v3(lo), _v3(d)
    fn = {1: lib().orc_deposit_cic, 2: lib().orc_deposit_tsc}[order]
    inside = fn(x.shape[0], _p(x), _p(y), _p(t), nx, ny, nz, _p(lo), _p(d),
                q_weight, zscale, _p(rho.reshape(-1)), int(zero_first))
    if inside < 0:
        raise ValueError("oracle: invalid grid")
    return rho, int(inside)


def gather_kick(coords, shape, lo, d, E, coef, zscale=1.0, order=1):
    """In place px,py,pt += coef * interp(E) ; E = (Ex,Ey,Ez) node arrays, x fastest; order 1 trilinear, 2 quadratic B-spline."""
    nx, ny, nz = shape
    lo, d, coef = _v3(lo), _v3(d), _v3(coef)
    x, px, y, py, t, pt = coords
    Ex, Ey, Ez = [np.ascontiguousarray(e, dtype=np.float64).reshape(-1) for e in E]
    assert Ex.size == nx * ny * nz
    fn = {1: lib().orc_gather_kick, 2: lib().orc_gather_kick_tsc}[order]
    inside = fn(x.shape[0], _p(x), _p(px), _p(y), _p(py), _p(t), _p(pt), nx, ny, nz,
                _p(lo), _p(d), _p(Ex), _p(Ey), _p(Ez), _p(coef), zscale)
    if inside < 0:
        raise ValueError("oracle: invalid grid")
    return int(inside)


def gather_field(x, y, t, shape, lo, d, E, zscale=1.0, order=1):
    if order == 2:
        out = [np.zeros_like(x) for _ in range(3)]
        gather_kick([x, out[0], y, out[1], t, out[2]], shape, lo, d, E, (1.0, 1.0, 1.0), zscale, order=2)
        return out
    nx, ny, nz = shape
    lo, d = _v3(lo), _v3(d)
    Ex, Ey, Ez = [np.ascontiguousarray(e, dtype=np.float64).reshape(-1) for e in E]
    out = [np.zeros_like(x) for _ in range(3)]
    lib().orc_gather_field(x.shape[0], _p(x), _p(y), _p(t), nx, ny, nz, _p(lo), _p(d),
                           _p(Ex), _p(Ey), _p(Ez), zscale, *[_p(o) for o in out])
    return out


def moments(coords):
    """Beam statistics: returns (mean[6], cov[6,6]) of coords = [x, px, y, py, t, pt],
    population second moments about the mean."""
    n = coords[0].shape[0]
    ptrs = (_dp * 6)(*[_p(c) for c in coords])
    mean, cov = np.zeros(6), np.zeros(36)
    if lib().orc_moments(n, ptrs, _p(mean), _p(cov)) != 0:
        raise ValueError("oracle: moments of an empty set")
    return mean, cov.reshape(6, 6)


def rms_emittances(cov):
    """Unnormalised rms emittances of the three planes from the 6x6 second moments:
    eps = sqrt(<q q><p p> - <q p>^2) for (x,px), (y,py), (t,pt)."""
    return tuple(float(np.sqrt(cov[a, a] * cov[a + 1, a + 1] - cov[a, a + 1] ** 2)) for a in (0, 2, 4))


EPS0 = 8.8541878128e-12


def green_self(dx, dy, dz):
    """(1/V) * integral of 1/r over one cell dx*dy*dz centred on the origin (R19 self term)."""
    return float(lib().orc_green_self(dx, dy, dz))


def poisson(rho, d, gz=1.0):
    """R19: free-space potential [V] at the nodes from rho[nz,ny,nx] (charge per node [C]); third axis spacing gz*d[2]."""
    nz, ny, nx = rho.shape
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    phi = np.zeros_like(rho)
    if lib().orc_poisson(nx, ny, nz, _p(_v3(d)), gz, _p(rho.reshape(-1)), _p(phi.reshape(-1))) != 0:
        raise ValueError("oracle: invalid grid")
    return phi


def efield(phi, d, gz=1.0):
    """E = -grad phi (rest frame): centred differences inside, one-sided at the faces.  Returns (Ex, Ey, Ez)."""
    nz, ny, nx = phi.shape
    phi = np.ascontiguousarray(phi, dtype=np.float64)
    E = [np.zeros_like(phi) for _ in range(3)]
    if lib().orc_efield(nx, ny, nz, _p(_v3(d)), gz, _p(phi.reshape(-1)), *[_p(e.reshape(-1)) for e in E]) != 0:
        raise ValueError("oracle: invalid grid")
    return E


def poisson_sample(rho, d, gz, targets):
    """R19 potential at the listed linear node indices only (same sum as poisson())."""
    nz, ny, nx = rho.shape
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    t = np.ascontiguousarray(targets, dtype=np.int64)
    out = np.zeros(t.size)
    if lib().orc_poisson_sample(nx, ny, nz, _p(_v3(d)), gz, _p(rho.reshape(-1)), t.size,
                                t.ctypes.data_as(C.POINTER(C.c_int64)), _p(out)) != 0:
        raise ValueError("oracle: invalid grid")
    return out
