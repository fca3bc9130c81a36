"""paper_2208_02382_b200 -- thin Python binding of libbt.so (include/bt.h).

Argument marshalling only: every step of the hot path (fused lattice walk, CIC deposit, gather+kick)
runs in the CUDA kernels of csrc/.  PyTorch is used for device memory and streams, nothing else.
There is NO CPU fallback: importing works without a GPU (so the symbols can be checked), but every
device call raises BtError, and a missing libbt.so raises ImportError.

Function names and arguments mirror the C-ABI one to one (bt_beam_create, bt_lattice_set, bt_track,
bt_deposit_cic, bt_gather_kick, ...); `Beam` and `Grid` are small RAII conveniences on top.
"""
import ctypes as C
import os

import numpy as np

from . import _build

__all__ = ["lib", "BtError", "Beam", "Grid", "pack_lattice", "ELEMENT_DTYPE", "EXPORTS",
           "calib_fp64", "calib_rw6", "launch_count", "debug_knob", "version", "moments_static",
           "MOMENTS_STATIC_MAX_PARTICLES"]

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libbt.so")

BT_OK, BT_ERR_INVALID, BT_ERR_CUDA, BT_ERR_OOM, BT_ERR_STATE, BT_ERR_UNSUPPORTED = 0, -1, -2, -3, -4, -5
BT_DRIFT, BT_QUAD, BT_SBEND, BT_DIPEDGE, BT_MULTIPOLE, BT_SHORTRF, BT_DRIFT_EXACT, BT_SHORTRF_SIN, BT_QUAD_CHROMATIC = range(9)
_KIND = {"drift": BT_DRIFT, "quad": BT_QUAD, "sbend": BT_SBEND, "dipedge": BT_DIPEDGE,
         "multipole": BT_MULTIPOLE, "shortrf": BT_SHORTRF, "drift_exact": BT_DRIFT_EXACT, "shortrf_sin": BT_SHORTRF_SIN, "quad_chromatic": BT_QUAD_CHROMATIC}

# bt_element: 64 bytes
ELEMENT_DTYPE = np.dtype([("type", "<i4"), ("nslice", "<i4"), ("ds", "<f8"), ("p", "<f8", (6,))])
assert ELEMENT_DTYPE.itemsize == 64

_dp = C.POINTER(C.c_double)
_vp = C.c_void_p

# every symbol include/bt.h declares: name -> (restype, argtypes)
EXPORTS = {
    "bt_beam_create": (C.c_int, [C.POINTER(_vp), C.c_int64, C.POINTER(_vp), _vp]),
    "bt_beam_destroy": (None, [_vp]),
    "bt_beam_set_ref": (C.c_int, [_vp, C.c_double, C.c_double, C.c_double]),
    "bt_beam_get_ref": (C.c_int, [_vp, _dp, _dp, C.POINTER(C.c_int64)]),
    "bt_beam_upload": (C.c_int, [_vp, C.POINTER(_vp)]),
    "bt_beam_download": (C.c_int, [_vp, C.POINTER(_vp)]),
    "bt_beam_ptrs": (C.c_int, [_vp, C.POINTER(_vp)]),
    "bt_beam_size": (C.c_int64, [_vp]),
    "bt_beam_sort_by_cell": (C.c_int, [_vp, _vp, C.c_double]),
    "bt_beam_ids": (C.c_int, [_vp, C.POINTER(_vp)]),
    "bt_beam_set_sort_pingpong": (C.c_int, [_vp, C.c_int]),
    "bt_beam_rehome": (C.c_int, [_vp]),
    "bt_beam_storage": (C.c_int, [_vp, C.POINTER(C.c_int32), C.POINTER(C.c_int64)]),
    "bt_beam_set_resort_interval": (C.c_int, [_vp, C.c_int32]),
    "bt_lattice_set": (C.c_int, [_vp, _vp, C.c_int32]),
    "bt_track": (C.c_int, [_vp, C.c_int32]),
    "bt_track_host": (C.c_int, [_vp, C.POINTER(_vp), C.POINTER(_vp), C.c_int32, C.c_int32]),
    "bt_grid_create": (C.c_int, [C.POINTER(_vp), C.c_int32, C.c_int32, C.c_int32, _dp, _dp]),
    "bt_grid_destroy": (None, [_vp]),
    "bt_grid_set_field": (C.c_int, [_vp, _vp, _vp, _vp, C.c_int]),
    "bt_grid_set_particle_shape": (C.c_int, [_vp, C.c_int32]),
    "bt_grid_rho": (C.c_int, [_vp, C.POINTER(_vp)]),
    "bt_grid_solve_poisson": (C.c_int, [_vp, C.c_double, _vp]),
    "bt_grid_download_phi": (C.c_int, [_vp, _vp]),
    "bt_grid_download_field": (C.c_int, [_vp, _vp, _vp, _vp]),
    "bt_grid_download_rho": (C.c_int, [_vp, _vp]),
    "bt_deposit_cic": (C.c_int, [_vp, _vp, C.c_double, C.c_double, C.c_int]),
    "bt_gather_kick": (C.c_int, [_vp, _vp, _dp, C.c_double, C.c_double, C.c_double]),
    "bt_beam_moments": (C.c_int, [_vp, _dp, _dp]),
    "bt_beam_moments_device": (C.c_int, [_vp, _vp]),
    "bt_moments_static": (C.c_int, [C.POINTER(_vp), C.c_int64, _vp, _vp]),
    "bt_track_diagnostics": (C.c_int, [_vp, C.c_int32, C.c_int32, _dp]),
    "bt_track_diagnostics_records": (C.c_int, [_vp, C.c_int32, C.c_int32, C.POINTER(C.c_int64)]),
    "bt_track_diagnostics_n": (C.c_int, [_vp, C.c_int32, C.c_int32, _dp, C.c_int64]),
    "bt_beam_release_scratch": (C.c_int, [_vp]),
    "bt_sync": (C.c_int, [_vp]),
    "bt_last_error": (C.c_char_p, []),
    "bt_version": (C.c_int, []),
    "bt_launch_count": (C.c_int64, []),
    "bt_debug_knob": (C.c_int, [C.c_char_p, C.c_int32]),
    "bt_track_last_launch": (C.c_int, [_vp] + [C.POINTER(C.c_int32)] * 4),
    "bt_calib_fp64": (C.c_int, [_vp, C.c_double, _dp]),
    "bt_calib_rw6": (C.c_int, [_vp, C.c_int64, C.c_int32, _dp]),
}


class BtError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib.bt_last_error()
        super().__init__("%s failed (%d): %s" % (where, code, msg.decode() if msg else ""))


def _load():
    if _build.needs_build():
        # (re)build on demand where nvcc exists; never fall back to anything else
        try:
            _build.build()
        except Exception as exc:  # pragma: no cover
            if os.path.exists(LIB_PATH):
                raise ImportError("libbt.so is stale (sources changed) and nvcc failed: %r" % (exc,))
            raise ImportError("libbt.so is missing and could not be built with nvcc: %r. "
                              "There is no CPU fallback." % (exc,))
    L = C.CDLL(LIB_PATH)
    for name, (res, args) in EXPORTS.items():
        fn = getattr(L, name)      # AttributeError => the library does not export what bt.h declares
        fn.restype = res
        fn.argtypes = args
    return L


lib = _load()


def _check(rc, where):
    if rc != BT_OK:
        raise BtError(rc, where)


def version():
    return lib.bt_version()


def launch_count():
    return int(lib.bt_launch_count())


def debug_knob(name, value):
    """bt_debug_knob: force a kernel variant (tests, A/B measurements); value -1 restores the measured default."""
    _check(lib.bt_debug_knob(name.encode(), int(value)), "bt_debug_knob")


MOMENTS_STATIC_MAX_PARTICLES = 67108864   # BT_MOMENTS_STATIC_MAX_PARTICLES of include/bt.h


def moments_static(dev_ptrs, n, out_ptr, stream=0):
    """bt_moments_static: beam statistics of six caller-owned device arrays without any device allocation by the
    library, for hosts that cannot let a library call cudaMalloc: an application whose arena already holds all of HBM,
    a multi-stream step loop that an allocation would stall (cudaMalloc synchronises the device), a process under an
    allocation checker.  dev_ptrs: six device addresses (x, px, y, py, t, pt; n doubles each, on the current device);
    out_ptr: device address of 42 doubles (mean[6], cov[36]); stream: a cudaStream_t handle (0 = default stream).
    Only enqueues work.  n above MOMENTS_STATIC_MAX_PARTICLES raises BtError(BT_ERR_INVALID).  All calls on one GPU share
    one fixed scratch array inside libbt.so: never let two of them overlap on the GPU (see include/bt.h)."""
    _check(lib.bt_moments_static(_ptr6(dev_ptrs), int(n), _vp(int(out_ptr)), _vp(int(stream))), "bt_moments_static")


def pack_lattice(lattice):
    """[(kind, ds, nslice, *params)] (workloads format) or a ready ELEMENT_DTYPE array -> bt_element array."""
    if isinstance(lattice, np.ndarray):
        assert lattice.dtype == ELEMENT_DTYPE
        return np.ascontiguousarray(lattice)
    lattice = list(lattice)
    arr = np.zeros(len(lattice), dtype=ELEMENT_DTYPE)
    for i, el in enumerate(lattice):
        arr[i]["type"] = _KIND[el[0]] if isinstance(el[0], str) else int(el[0])
        arr[i]["ds"] = el[1]
        arr[i]["nslice"] = el[2]
        params = list(el[3:])
        arr[i]["p"][:len(params)] = params
    return arr


def _ptr6(ptrs):
    return (_vp * 6)(*[int(p) for p in ptrs])


def _host_ptrs(arrays):
    """6 contiguous float64 host arrays (numpy, or CPU torch tensors e.g. pinned) -> pointer array."""
    ptrs = []
    for a in arrays:
        if isinstance(a, np.ndarray):
            assert a.dtype == np.float64 and a.flags.c_contiguous
            ptrs.append(a.ctypes.data)
        else:  # torch CPU tensor
            assert a.device.type == "cpu" and a.is_contiguous() and a.element_size() == 8
            ptrs.append(a.data_ptr())
    return _ptr6(ptrs)


def _current_stream_ptr():
    import torch
    return int(torch.cuda.current_stream().cuda_stream)


class Beam:
    """bt_beam handle.  `storage`: None -> six torch.float64 CUDA tensors are allocated here and lent to
    the library (PyTorch owns device memory); "library" -> bt_beam_create allocates; or a list of six
    CUDA tensors to borrow.  `pingpong` (bt_beam_set_sort_pingpong): None = the safe default -- tensors passed in by the
    caller always hold the bunch (a sort copies its result back into them); tensors allocated here and library storage
    ping-pong (use .tensors / ptrs() after anything that may sort)."""

    def __init__(self, n, storage=None, stream=None, pingpong=None):
        self._h = _vp()
        self.n = int(n)
        self._tensors = None
        storage_was_none = False
        if storage == "library":
            dev = None
        else:
            import torch
            storage_was_none = storage is None
            if storage is None:
                storage = [torch.empty(self.n, dtype=torch.float64, device="cuda") for _ in range(6)]
            assert len(storage) == 6 and all(t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == self.n for t in storage)
            self._tensors = list(storage)
            dev = _ptr6([t.data_ptr() for t in self._tensors])
        self.stream = _current_stream_ptr() if stream is None else int(stream)
        _check(lib.bt_beam_create(C.byref(self._h), self.n, dev, _vp(self.stream)), "bt_beam_create")
        # Tensors this object allocated itself are reachable only through .tensors, which follows the bunch: ping-pong sorts
        # (no copy back) are safe.  Tensors the caller passed in keep holding the bunch unless the caller says pingpong=True.
        if pingpong is None and storage_was_none:
            pingpong = True
        if pingpong is not None:
            self.set_sort_pingpong(pingpong)

    def close(self):
        if getattr(self, "_h", None) is not None and self._h and lib is not None:   # lib is None at interpreter shutdown
            lib.bt_beam_destroy(self._h)
            self._h = None

    __del__ = close

    @property
    def tensors(self):
        """Six CUDA tensors over the arrays the particles live in NOW (storage order): the tensors lent at construction,
        or -- after bt_beam_sort_by_cell moved the bunch into the library's partner arrays (ping-pong) -- zero-copy views
        of those (valid until the next sort / upload / close).  None for library-owned storage that was never lent."""
        import torch
        cur = self.ptrs()
        if self._tensors is not None and all(t.data_ptr() == p for t, p in zip(self._tensors, cur)):
            return self._tensors
        if self._tensors is None:
            return None
        n = self.n

        def view(ptr):
            class _V:
                __cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 3, "strides": None}
            return torch.as_tensor(_V(), device="cuda")
        return [view(p) for p in cur]

    def set_ref(self, kin_energy_MeV, mass_MeV, charge_qe=1.0):
        _check(lib.bt_beam_set_ref(self._h, kin_energy_MeV, mass_MeV, charge_qe), "bt_beam_set_ref")

    def get_ref(self):
        g, s, t = C.c_double(), C.c_double(), C.c_int64()
        _check(lib.bt_beam_get_ref(self._h, C.byref(g), C.byref(s), C.byref(t)), "bt_beam_get_ref")
        return g.value, s.value, t.value

    def upload(self, host_arrays):
        _check(lib.bt_beam_upload(self._h, _host_ptrs(host_arrays)), "bt_beam_upload")

    def track_host(self, host_in, host_out=None, nturns=1, nchunks=8):
        """bt_track_host: host arrays in, host arrays out (in place when host_out is None), copies overlapped with the walk."""
        if host_out is None:
            host_out = host_in
        _check(lib.bt_track_host(self._h, _host_ptrs(host_in), _host_ptrs(host_out), int(nturns), int(nchunks)), "bt_track_host")
        return host_out

    def download(self, out=None):
        if out is None:
            out = [np.empty(self.n, dtype=np.float64) for _ in range(6)]
        _check(lib.bt_beam_download(self._h, _host_ptrs(out)), "bt_beam_download")
        return out

    def ptrs(self):
        p = (_vp * 6)()
        _check(lib.bt_beam_ptrs(self._h, p), "bt_beam_ptrs")
        return [int(v) for v in p]

    def lattice_set(self, lattice):
        arr = pack_lattice(lattice)
        _check(lib.bt_lattice_set(self._h, arr.ctypes.data, len(arr)), "bt_lattice_set")

    def track(self, nturns=1):
        _check(lib.bt_track(self._h, nturns), "bt_track")

    def last_launch(self):
        v = [C.c_int32() for _ in range(4)]
        _check(lib.bt_track_last_launch(self._h, *[C.byref(x) for x in v]), "bt_track_last_launch")
        return dict(zip(("grid", "block", "particles_per_thread", "smem_bytes"), [x.value for x in v]))

    def deposit_cic(self, grid, q_weight, zscale=1.0, zero_first=True):
        _check(lib.bt_deposit_cic(self._h, grid._h, q_weight, zscale, int(zero_first)), "bt_deposit_cic")

    def gather_kick(self, grid, coef, zscale=1.0, half_drift_before=0.0, half_drift_after=0.0):
        c = (C.c_double * 3)(*coef)
        _check(lib.bt_gather_kick(self._h, grid._h, c, zscale, half_drift_before, half_drift_after), "bt_gather_kick")

    def track_diagnostics(self, nturns, n_boundaries=None, granularity="element"):
        """bt_track(nturns) with the beam statistics taken inside the walk after every element ("element") or every slice
        ("slice"): returns (mean[nturns, B, 6], cov[nturns, B, 6, 6]) with B = boundaries per turn = number of elements,
        resp. the sum of their nslice.  The output is sized from the library's own count (bt_track_diagnostics_records) and
        passed with its capacity; n_boundaries, when given, is only checked against B."""
        gran = {"element": 0, "slice": 1}[granularity]
        nturns = int(nturns)
        per_turn = C.c_int64()
        _check(lib.bt_track_diagnostics_records(self._h, 1, gran, C.byref(per_turn)), "bt_track_diagnostics_records")
        nb = int(per_turn.value)
        if n_boundaries is not None and int(n_boundaries) != nb:
            raise ValueError("track_diagnostics: the lattice has %d boundaries per turn at %s granularity, not %d" % (nb, granularity, int(n_boundaries)))
        out = np.zeros((nturns, nb, 42))
        _check(lib.bt_track_diagnostics_n(self._h, nturns, gran, out.ctypes.data_as(_dp), nturns * nb), "bt_track_diagnostics_n")
        return out[:, :, :6].copy(), out[:, :, 6:].reshape(nturns, nb, 6, 6).copy()

    def release_scratch(self):
        _check(lib.bt_beam_release_scratch(self._h), "bt_beam_release_scratch")

    def moments(self):
        """(mean[6], cov[6, 6]) of x, px, y, py, t, pt -- computed on the device, returned as numpy arrays."""
        mean, cov = np.zeros(6), np.zeros(36)
        _check(lib.bt_beam_moments(self._h, mean.ctypes.data_as(_dp), cov.ctypes.data_as(_dp)), "bt_beam_moments")
        return mean, cov.reshape(6, 6)

    def moments_device(self, out):
        """bt_beam_moments_device: the 42 statistics (mean[6], cov[36]) into a CUDA float64 tensor of >= 42 elements, enqueued
        on the beam's stream without synchronisation."""
        assert out.is_cuda and out.is_contiguous() and out.element_size() == 8 and out.numel() >= 42
        _check(lib.bt_beam_moments_device(self._h, _vp(out.data_ptr())), "bt_beam_moments_device")
        return out

    def set_sort_pingpong(self, enable):
        _check(lib.bt_beam_set_sort_pingpong(self._h, int(bool(enable))), "bt_beam_set_sort_pingpong")

    def rehome(self):
        _check(lib.bt_beam_rehome(self._h), "bt_beam_rehome")

    def storage(self):
        """(in_home, epoch): whether the bunch is in the arrays of bt_beam_create, and the count of storage changes so far."""
        h, e = C.c_int32(), C.c_int64()
        _check(lib.bt_beam_storage(self._h, C.byref(h), C.byref(e)), "bt_beam_storage")
        return bool(h.value), int(e.value)

    def set_resort_interval(self, every_n_deposits):
        _check(lib.bt_beam_set_resort_interval(self._h, int(every_n_deposits)), "bt_beam_set_resort_interval")

    def sort_by_cell(self, grid, zscale=1.0):
        _check(lib.bt_beam_sort_by_cell(self._h, grid._h, zscale), "bt_beam_sort_by_cell")

    def ids_ptr(self):
        p = _vp()
        _check(lib.bt_beam_ids(self._h, C.byref(p)), "bt_beam_ids")
        return int(p.value) if p.value else 0

    def sync(self):
        _check(lib.bt_sync(self._h), "bt_sync")


class Grid:
    def __init__(self, shape, lo, d):
        self._h = _vp()
        self.shape = tuple(int(s) for s in shape)
        lo_a, d_a = (C.c_double * 3)(*lo), (C.c_double * 3)(*d)
        _check(lib.bt_grid_create(C.byref(self._h), self.shape[0], self.shape[1], self.shape[2], lo_a, d_a), "bt_grid_create")

    def close(self):
        if getattr(self, "_h", None) is not None and self._h and lib is not None:
            lib.bt_grid_destroy(self._h)
            self._h = None

    __del__ = close

    def set_particle_shape(self, order):
        """1 = CIC (default), 2 = quadratic B-spline."""
        _check(lib.bt_grid_set_particle_shape(self._h, int(order)), "bt_grid_set_particle_shape")

    def solve_poisson(self, gz=1.0, stream=None):
        """rho -> phi -> E (rest frame, third axis stretched by gz) on the current torch stream; see bt_grid_solve_poisson."""
        sp = _current_stream_ptr() if stream is None else stream
        _check(lib.bt_grid_solve_poisson(self._h, float(gz), sp), "bt_grid_solve_poisson")

    def download_phi(self):
        out = np.empty((self.shape[2], self.shape[1], self.shape[0]), dtype=np.float64)
        _check(lib.bt_grid_download_phi(self._h, out.ctypes.data), "bt_grid_download_phi")
        return out

    def download_field(self):
        out = [np.empty((self.shape[2], self.shape[1], self.shape[0]), dtype=np.float64) for _ in range(3)]
        _check(lib.bt_grid_download_field(self._h, *[o.ctypes.data for o in out]), "bt_grid_download_field")
        return out

    def set_field(self, Ex, Ey, Ez):
        """Host numpy arrays (any shape with nx*ny*nz elements, x fastest) or CUDA torch tensors."""
        arrs = [Ex, Ey, Ez]
        if isinstance(Ex, np.ndarray):
            arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in arrs]
            ptrs, on_dev = [a.ctypes.data for a in arrs], 0
        else:
            assert all(a.is_cuda and a.is_contiguous() for a in arrs)
            ptrs, on_dev = [a.data_ptr() for a in arrs], 1
        n = self.shape[0] * self.shape[1] * self.shape[2]
        assert all((a.size if isinstance(a, np.ndarray) else a.numel()) == n for a in arrs)
        _check(lib.bt_grid_set_field(self._h, ptrs[0], ptrs[1], ptrs[2], on_dev), "bt_grid_set_field")

    def rho_ptr(self):
        p = _vp()
        _check(lib.bt_grid_rho(self._h, C.byref(p)), "bt_grid_rho")
        return int(p.value)

    def rho_tensor(self):
        """Zero-copy torch view [nz, ny, nx] of the library-owned rho (valid until close())."""
        import torch
        nx, ny, nz = self.shape

        class _View:  # CUDA Array Interface v3 over the raw device pointer
            __cuda_array_interface__ = {"shape": (nz, ny, nx), "typestr": "<f8", "data": (self.rho_ptr(), False),
                                        "version": 3, "strides": None}
        return torch.as_tensor(_View(), device="cuda")

    def download_rho(self):
        nx, ny, nz = self.shape
        out = np.empty((nz, ny, nx), dtype=np.float64)
        _check(lib.bt_grid_download_rho(self._h, out.ctypes.data), "bt_grid_download_rho")
        return out


def calib_fp64(min_ms=200.0, stream=None):
    v = C.c_double()
    s = _current_stream_ptr() if stream is None else int(stream)
    _check(lib.bt_calib_fp64(_vp(s), min_ms, C.byref(v)), "bt_calib_fp64")
    return v.value


def calib_rw6(n=64_000_000, reps=5, stream=None):
    v = C.c_double()
    s = _current_stream_ptr() if stream is None else int(stream)
    _check(lib.bt_calib_rw6(_vp(s), n, reps, C.byref(v)), "bt_calib_rw6")
    return v.value
