"""Thin ctypes binding of the C-ABI library declared in include/streams.h.

Argument marshalling only: every step of the path runs in the CUDA kernels of
libstreams_b200.so.  PyTorch is used for device memory and the CUDA stream, nothing else.
There is no CPU fallback: if the library is missing or no GPU is present, calls raise.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libstreams_b200.so")

STREAMS_OK, STREAMS_EINVAL, STREAMS_ECUDA, STREAMS_ENOMEM, STREAMS_ENONFINITE, STREAMS_ESTATE = 0, -1, -2, -3, -4, -5

EXPORTS = ["streams_workspace_bytes", "streams_create", "streams_set_state", "streams_set_state_host",
           "streams_get_state", "streams_get_state_host", "streams_rhs", "streams_sensor", "streams_step",
           "streams_diagnostics", "streams_step_begin", "streams_stage_rhs", "streams_stage_mid", "streams_stage_end", "streams_reduce_ptr",
           "streams_halo_bytes", "streams_halo_pack", "streams_halo_unpack", "streams_flag_halo_bytes", "streams_flag_halo_pack",
           "streams_flag_halo_unpack", "streams_stats_accumulate", "streams_stats_read", "streams_stats_reset", "streams_profile", "streams_profile_read", "streams_fp64_peak", "streams_max_speed_static",
           "streams_launch_count", "streams_last_error", "streams_destroy"]


class StreamsGrid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("pad_", C.c_int), ("len", C.c_double * 3)]


class StreamsParams(C.Structure):
    _fields_ = [("gamma", C.c_double), ("Pr", C.c_double), ("Rgas", C.c_double), ("mu_ref", C.c_double),
                ("T_ref", C.c_double), ("visc_exp", C.c_double), ("suth_S", C.c_double),
                ("sensor_threshold", C.c_double), ("sensor_eps", C.c_double),
                ("T_wall", C.c_double * 2), ("y_wall", C.c_double * 2), ("fs", C.c_double * 5),
                ("shock_angle_deg", C.c_double), ("x_shock", C.c_double), ("cfl", C.c_double),
                ("dt_fixed", C.c_double),
                ("visc_model", C.c_int), ("order", C.c_int), ("weno_enable", C.c_int), ("forcing", C.c_int),
                ("viscous_enable", C.c_int), ("bc", C.c_int * 6), ("weno_order", C.c_int)]


class StreamsDiag(C.Structure):
    _fields_ = [("step", C.c_longlong), ("time", C.c_double), ("dt", C.c_double), ("forcing", C.c_double),
                ("mass", C.c_double), ("mom", C.c_double * 3), ("energy", C.c_double), ("kinetic", C.c_double),
                ("volume", C.c_double), ("bulk_rhou", C.c_double),
                ("min_rho", C.c_double), ("min_p", C.c_double), ("max_mach", C.c_double), ("max_theta", C.c_double),
                ("max_speed", C.c_double * 3),
                ("weno_ifaces", C.c_longlong * 3), ("total_ifaces", C.c_longlong * 3),
                ("nonfinite", C.c_int), ("pad_", C.c_int)]


class StreamsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"streams error {code}: {msg}")
        self.code = code


_lib = None
_DBL = C.POINTER(C.c_double)


def lib():
    """Load libstreams_b200.so (built by paper_2004_02276_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2004_02276_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.streams_workspace_bytes.argtypes = [C.POINTER(StreamsGrid), C.POINTER(StreamsParams)]
        L.streams_workspace_bytes.restype = C.c_size_t
        L.streams_create.argtypes = [C.POINTER(StreamsGrid), _DBL, _DBL, _DBL, C.POINTER(StreamsParams),
                                     C.c_void_p, C.c_size_t, C.c_void_p, C.POINTER(C.c_void_p)]
        for name in ("streams_set_state", "streams_set_state_host", "streams_get_state", "streams_get_state_host",
                     "streams_rhs"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        L.streams_sensor.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.streams_step.argtypes = [C.c_void_p, C.c_int]
        L.streams_diagnostics.argtypes = [C.c_void_p, C.POINTER(StreamsDiag)]
        L.streams_step_begin.argtypes = [C.c_void_p]
        L.streams_stage_rhs.argtypes = [C.c_void_p, C.c_int, C.c_int]
        L.streams_stage_end.argtypes = [C.c_void_p, C.c_int]
        L.streams_stage_mid.argtypes = [C.c_void_p, C.c_int]
        L.streams_reduce_ptr.argtypes = [C.c_void_p]
        L.streams_reduce_ptr.restype = C.c_void_p
        L.streams_halo_bytes.argtypes = [C.c_void_p]
        L.streams_halo_bytes.restype = C.c_size_t
        L.streams_halo_pack.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.streams_halo_unpack.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.streams_flag_halo_bytes.argtypes = [C.c_void_p]
        L.streams_flag_halo_bytes.restype = C.c_size_t
        L.streams_flag_halo_pack.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.streams_flag_halo_unpack.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.streams_stats_accumulate.argtypes = [C.c_void_p]
        L.streams_stats_read.argtypes = [C.c_void_p, _DBL, C.POINTER(C.c_longlong)]
        L.streams_stats_reset.argtypes = [C.c_void_p]
        L.streams_profile.argtypes = [C.c_void_p, C.c_int]
        L.streams_profile_read.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        L.streams_fp64_peak.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
        L.streams_max_speed_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.streams_launch_count.argtypes = [C.c_void_p]
        L.streams_launch_count.restype = C.c_longlong
        L.streams_last_error.argtypes = [C.c_void_p]
        L.streams_last_error.restype = C.c_char_p
        L.streams_destroy.argtypes = [C.c_void_p]
        L.streams_destroy.restype = None
        _lib = L
    return _lib


def fp64_peak(stream=None) -> float:
    """Measured fp64 lane-instruction rate of the device in 1e12/s (include/streams.h: streams_fp64_peak)."""
    v = C.c_double(0.0)
    rc = lib().streams_fp64_peak(C.c_void_p(stream or 0), C.byref(v))
    if rc != 0:
        raise StreamsError(rc, lib().streams_last_error(None).decode())
    return v.value


def make_params(params: dict) -> StreamsParams:
    p = StreamsParams()
    for name, _t in StreamsParams._fields_:
        if name == "pad_":
            continue
        v = params.get("weno_order", 5) if name == "weno_order" else params[name]
        if isinstance(v, (list, tuple, np.ndarray)):
            arr = getattr(p, name)
            for i, x in enumerate(v):
                arr[i] = x
        else:
            setattr(p, name, v)
    return p


def make_grid(grid: dict) -> StreamsGrid:
    g = StreamsGrid()
    g.nx, g.ny, g.nz = int(grid["nx"]), int(grid["ny"]), int(grid["nz"])
    for i in range(3):
        g.len[i] = grid["len"][i]
    return g


def workspace_bytes(grid: dict, params: dict) -> int:
    g, p = make_grid(grid), make_params(params)
    return lib().streams_workspace_bytes(C.byref(g), C.byref(p))


class Streams:
    """One context of the CUDA library.  Device buffers are torch tensors owned by this object."""

    def __init__(self, grid: dict, x, y, z, params: dict, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2004_02276_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device)
        self.n = (int(grid["nx"]), int(grid["ny"]), int(grid["nz"]))
        self.shape = (5, self.n[2], self.n[1], self.n[0])
        self._g, self._p = make_grid(grid), make_params(params)
        self._h = None
        nbytes = lib().streams_workspace_bytes(C.byref(self._g), C.byref(self._p))
        if nbytes == 0:
            raise StreamsError(STREAMS_EINVAL, "invalid grid/params")
        with torch.cuda.device(self.device):
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            # a private (non-blocking) stream per context: the library's launches do not serialise with the legacy
            # default stream, and streams_step may capture its kernels into CUDA graphs (include/streams.h).  A
            # caller-supplied torch stream is used as given (the legacy default stream disables the graphs).
            self._stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            xs = [np.ascontiguousarray(a, dtype=np.float64) for a in (x, y, z)]
            h = C.c_void_p()
            rc = lib().streams_create(C.byref(self._g), xs[0].ctypes.data_as(_DBL), xs[1].ctypes.data_as(_DBL),
                                      xs[2].ctypes.data_as(_DBL), C.byref(self._p), C.c_void_p(self._ws.data_ptr()),
                                      nbytes, C.c_void_p(self._stream.cuda_stream), C.byref(h))
        if rc != 0:
            raise StreamsError(rc, lib().streams_last_error(None).decode())
        self._h = h
        self.workspace_bytes = nbytes
        self._red = None

    def close(self):
        if self._h:
            lib().streams_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def stream(self):
        """The torch.cuda.Stream all kernels of this context are enqueued on."""
        return self._stream

    def _pre(self, t=None):
        """The context stream waits for what the caller's current stream has enqueued (producer of `t`)."""
        cur = self._torch.cuda.current_stream(self.device)
        if cur != self._stream:
            self._stream.wait_stream(cur)
            if t is not None:
                t.record_stream(self._stream)

    def _post(self, t=None):
        """The caller's current stream waits for the context stream (consumer of `t`)."""
        cur = self._torch.cuda.current_stream(self.device)
        if cur != self._stream:
            cur.wait_stream(self._stream)
            if t is not None:
                t.record_stream(self._stream)

    def _chk(self, rc, allow=()):
        if rc != 0 and rc not in allow:
            raise StreamsError(rc, lib().streams_last_error(self._h).decode())
        return rc

    def _dev(self, t, shape=None, dtype=None):
        torch = self._torch
        dtype = dtype or torch.float64
        assert t.is_cuda and t.dtype == dtype and t.is_contiguous(), "need a contiguous CUDA tensor"
        if shape is not None:
            assert tuple(t.shape) == tuple(shape), (tuple(t.shape), shape)
        return C.c_void_p(t.data_ptr())

    # --- state --------------------------------------------------------------------------------
    def set_state(self, w):
        """w: torch CUDA tensor [5][nz][ny][nx] (device path) or NumPy array (host path)."""
        if isinstance(w, np.ndarray):
            w = np.ascontiguousarray(w, dtype=np.float64)
            assert w.shape == self.shape
            self._chk(lib().streams_set_state_host(self._h, C.c_void_p(w.ctypes.data)))
        else:
            self._pre(w)
            self._chk(lib().streams_set_state(self._h, self._dev(w, self.shape)))

    def set_state_host_ptr(self, ptr):
        self._chk(lib().streams_set_state_host(self._h, C.c_void_p(ptr)))

    def get_state_host_ptr(self, ptr):
        self._chk(lib().streams_get_state_host(self._h, C.c_void_p(ptr)))

    def get_state(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._pre()
        self._chk(lib().streams_get_state(self._h, self._dev(out, self.shape)))
        self._post(out)
        return out

    def get_state_host(self):
        out = np.empty(self.shape)
        self._chk(lib().streams_get_state_host(self._h, C.c_void_p(out.ctypes.data)))
        return out

    # --- hot path -------------------------------------------------------------------------------
    def rhs(self, out=None):
        torch = self._torch
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._pre()
        self._chk(lib().streams_rhs(self._h, self._dev(out, self.shape)))
        self._post(out)
        return out

    def sensor(self):
        torch = self._torch
        th = torch.empty(self.shape[1:], dtype=torch.float64, device=self.device)
        fl = torch.empty((3,) + self.shape[1:], dtype=torch.uint8, device=self.device)
        self._pre()
        self._chk(lib().streams_sensor(self._h, C.c_void_p(th.data_ptr()), C.c_void_p(fl.data_ptr())))
        self._post(th)
        self._post(fl)
        return th, fl

    def step(self, n=1):
        self._chk(lib().streams_step(self._h, int(n)))

    # --- staged stepping and z-slab halos (include/streams.h) ------------
    PART_ALL, PART_INTERIOR, PART_BOUNDARY = 0, 1, 2
    FACE_ZMIN, FACE_ZMAX = 4, 5
    STATIC_MAX_NODES = 33554432          # streams_max_speed_static (include/streams.h)

    def step_begin(self):
        self._chk(lib().streams_step_begin(self._h))

    def stage_rhs(self, stage, part=0):
        self._chk(lib().streams_stage_rhs(self._h, int(stage), int(part)))

    def stage_mid(self, stage):
        """forcing with the hybrid switch: WENO correction of R and its sums -> red[0..1] (after the flag-word swap)."""
        self._chk(lib().streams_stage_mid(self._h, int(stage)))

    def stage_end(self, stage):
        self._chk(lib().streams_stage_end(self._h, int(stage)))

    @property
    def red(self):
        """torch view (4 fp64, device) of the partial reductions the caller combines across slabs."""
        if self._red is None:
            ptr = lib().streams_reduce_ptr(self._h)
            off = ptr - self._ws.data_ptr()
            assert 0 <= off <= self.workspace_bytes - 32 and off % 8 == 0
            self._red = self._ws[off:off + 32].view(self._torch.float64)
        return self._red

    def halo_shape(self):
        return (7, 3, self.n[1], self.n[0])

    def new_buffer(self):
        """An uninitialised halo message buffer on the context's device."""
        return self._torch.empty(self.halo_shape(), dtype=self._torch.float64, device=self.device)

    def halo_pack(self, face, out=None, stream=None):
        """Message [7][3][ny][nx] of the interior planes next to z face `face` (4 = zmin, 5 = zmax)."""
        torch = self._torch
        if out is None:
            out = torch.empty(self.halo_shape(), dtype=torch.float64, device=self.device)
        st = stream.cuda_stream if stream is not None else 0
        self._chk(lib().streams_halo_pack(self._h, int(face), self._dev(out, self.halo_shape()), C.c_void_p(st)))
        return out

    def halo_unpack(self, face, buf, stream=None):
        st = stream.cuda_stream if stream is not None else 0
        self._chk(lib().streams_halo_unpack(self._h, int(face), self._dev(buf, self.halo_shape()), C.c_void_p(st)))

    def flag_shape(self):
        return (3, self.n[1], (self.n[0] + 31) // 32)

    def new_flag_buffer(self):
        return self._torch.empty(self.flag_shape(), dtype=self._torch.int32, device=self.device)

    def flag_halo_pack(self, face, out, stream=None):
        st = stream.cuda_stream if stream is not None else 0
        self._chk(lib().streams_flag_halo_pack(self._h, int(face), self._dev(out, self.flag_shape(), self._torch.int32), C.c_void_p(st)))
        return out

    def flag_halo_unpack(self, face, buf, stream=None):
        st = stream.cuda_stream if stream is not None else 0
        self._chk(lib().streams_flag_halo_unpack(self._h, int(face), self._dev(buf, self.flag_shape(), self._torch.int32), C.c_void_p(st)))

    def diagnostics(self, check=True):
        d = StreamsDiag()
        rc = lib().streams_diagnostics(self._h, C.byref(d))
        self._chk(rc, allow=() if check else (STREAMS_ENONFINITE,))
        return d

    def max_speed_static(self, w, out):
        """S10 maxima of the conservative state `w` ([5][nz][ny][nx], device) into `out` (3 doubles, device), asynchronous
        on the context stream; the library call allocates nothing (its scratch is a static device array; grids of at most
        STATIC_MAX_NODES nodes).  Both tensors are the caller's: nothing is allocated here either."""
        self._pre(w)
        self._chk(lib().streams_max_speed_static(self._h, self._dev(w, self.shape), self._dev(out, (3,))))
        self._post(out)
        return out

    # --- statistics --------------------------------------------------------------
    def stats_accumulate(self):
        self._chk(lib().streams_stats_accumulate(self._h))

    def stats_read(self):
        """(time-averaged x-z plane means [16][ny] as a NumPy array, number of samples)"""
        out = np.empty((16, self.n[1]))
        n = C.c_longlong(0)
        self._chk(lib().streams_stats_read(self._h, out.ctypes.data_as(_DBL), C.byref(n)))
        return out, n.value

    def stats_reset(self):
        self._chk(lib().streams_stats_reset(self._h))

    def profile(self, enable=True):
        self._chk(lib().streams_profile(self._h, 1 if enable else 0))

    def profile_read(self):
        """(summed k_rhs device time in ms, number of k_rhs launches recorded)"""
        ms, n = C.c_double(0.0), C.c_longlong(0)
        self._chk(lib().streams_profile_read(self._h, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def launch_count(self):
        return lib().streams_launch_count(self._h)
