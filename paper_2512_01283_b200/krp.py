"""Thin ctypes binding of libkrp.so (include/krp.h): same names, argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  torch is used for device buffers
and streams.  There is no CPU fallback: a missing library raises.
"""
import ctypes as C
import os

import numpy as np

from . import _build

OK, ERR_ARG, ERR_CUDA, ERR_OOM, ERR_STATE, ERR_EVENT_FULL = 0, -1, -2, -3, -4, -5
MEM_DEVICE, MEM_HOST = 0, 1
NOALLOC_MAX_EVENTS = 262144      # KRP_NOALLOC_MAX_EVENTS of include/krp.h

SYMBOLS = [
    "krp_last_error", "krp_version", "krp_grid_create", "krp_grid_destroy", "krp_grid_update", "krp_grid_stage", "krp_grid_update_staged", "krp_source_set",
    "krp_events_reserve", "krp_transport", "krp_packet_id_set", "krp_image", "krp_image_get",
    "krp_image_reset", "krp_stats_get", "krp_stats_reset", "krp_events_get", "krp_events_select", "krp_events_clear",
    "krp_tune", "krp_tune_schedule", "krp_tune_fused", "krp_timing_enable", "krp_timing_get", "krp_launch_count",
    "krp_sgrid_begin", "krp_sgrid_get", "krp_sgrid_reset", "krp_sgrid_end", "krp_image_rays", "krp_freq_define", "krp_freq_select", "krp_zmatrix_set",
    "krp_image_events_noalloc",
]
T_FLIGHT, T_SCATTER, T_ORDER, T_IMAGE, T_EMIT, T_DEPOSIT, T_RAYS, T_COUNT = 0, 1, 2, 3, 4, 5, 6, 7
T_NAMES = ("flight", "scatter", "order", "image", "emit", "deposit", "rays")


class KrpError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("krp error %d: %s" % (code, msg))
        self.code = code


class Tables(C.Structure):
    _fields_ = [("n_ang", C.c_int), ("mueller", C.c_void_p), ("n_inc", C.c_int), ("opacity", C.c_void_p),
                ("w_min", C.c_float), ("max_scatter", C.c_int), ("periodic", C.c_int)]


class Source(C.Structure):
    _fields_ = [("kind", C.c_int), ("pos", C.c_double * 3), ("dir", C.c_double * 3),
                ("cell_weight", C.c_void_p), ("emit_records", C.c_int)]


class Observer(C.Structure):
    _fields_ = [("theta", C.c_double), ("phi", C.c_double), ("center", C.c_double * 3),
                ("half_w", C.c_double), ("half_h", C.c_double)]


class Stats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("packets", "events", "records", "steps_transport", "steps_image",
                                          "contributions", "dropped", "overflow", "segments")] + \
               [(n, C.c_double) for n in ("w_emitted", "w_escaped", "w_absorbed", "w_cut")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


_lib = None


def library_path():
    return _build.LIB


def lib():
    """Load libkrp.so, rebuilding it first when it was not compiled from the sources beside it (the build id is a
    hash of the sources).  A library that is stale and cannot be rebuilt is an error: nothing runs on old kernels."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    override = os.environ.get("KRP_LIBRARY")          # development: a library built with other compile-time options (A/B runs)
    if override:
        path = override
    elif _build.stale():
        try:
            _build.build()
        except Exception as exc:
            raise ImportError("libkrp.so is missing or was built from other sources (want build id %s) and could not be "
                              "rebuilt (%s); run `python -m paper_2512_01283_b200._build`" % (_build.source_id(), exc)) from exc
    L = C.CDLL(path)
    L.krp_version.restype = C.c_char_p
    if not override and _build.source_id().encode() not in L.krp_version():
        raise ImportError("libkrp.so reports %r, the sources beside it have build id %s" % (L.krp_version(), _build.source_id()))
    vp, u64, i32 = C.c_void_p, C.c_uint64, C.c_int
    sig = {
        "krp_last_error": (C.c_char_p, []),
        "krp_version": (C.c_char_p, []),
        "krp_grid_create": (i32, [C.POINTER(vp), i32, i32, i32, C.POINTER(C.c_double), vp, vp, i32,
                                  C.POINTER(Tables), vp]),
        "krp_grid_destroy": (i32, [vp]),
        "krp_grid_update": (i32, [vp, vp, vp, i32, vp]),
        "krp_grid_stage": (i32, [vp, vp, vp, vp]),
        "krp_grid_update_staged": (i32, [vp, vp]),
        "krp_source_set": (i32, [vp, C.POINTER(Source), vp]),
        "krp_events_reserve": (i32, [vp, u64]),
        "krp_transport": (i32, [vp, u64, u64, vp]),
        "krp_packet_id_set": (i32, [vp, u64]),
        "krp_image": (i32, [vp, C.POINTER(Observer), i32, i32, i32, i32, vp]),
        "krp_image_get": (i32, [vp, vp, i32, vp]),
        "krp_image_reset": (i32, [vp, vp]),
        "krp_stats_get": (i32, [vp, C.POINTER(Stats)]),
        "krp_stats_reset": (i32, [vp, vp]),
        "krp_events_get": (i32, [vp, u64, C.POINTER(u64), vp, vp, vp, vp, vp, vp]),
        "krp_events_select": (i32, [vp, u64, u64, u64, C.POINTER(u64), vp, vp, vp, vp, vp, vp]),
        "krp_events_clear": (i32, [vp, vp]),
        "krp_tune": (i32, [vp, i32, i32, i32, i32]),
        "krp_timing_enable": (i32, [vp, i32]),
        "krp_timing_get": (i32, [vp, vp, vp]),
        "krp_tune_schedule": (i32, [vp, i32, i32, i32]),
        "krp_tune_fused": (i32, [vp, C.c_longlong]),
        "krp_launch_count": (u64, [vp]),
        "krp_zmatrix_set": (i32, [vp, i32, i32, i32, vp, vp]),
        "krp_freq_define": (i32, [vp, i32, C.POINTER(Tables), vp, vp]),
        "krp_freq_select": (i32, [vp, i32, vp]),
        "krp_sgrid_begin": (i32, [vp, C.POINTER(Observer), i32, vp]),
        "krp_sgrid_get": (i32, [vp, vp, i32, vp]),
        "krp_sgrid_reset": (i32, [vp, vp]),
        "krp_sgrid_end": (i32, [vp]),
        "krp_image_rays": (i32, [vp, C.POINTER(Observer), i32, i32, i32, vp, i32, vp]),
        "krp_image_events_noalloc": (i32, [vp, u64, vp, vp, vp, vp, vp, C.POINTER(Observer), i32, i32, i32, vp,
                                           C.POINTER(u64), vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def _check(rc):
    if rc != OK:
        raise KrpError(rc, lib().krp_last_error().decode())


def _stream(stream):
    if stream is None:
        import torch
        return C.c_void_p(torch.cuda.current_stream().cuda_stream)
    if hasattr(stream, "cuda_stream"):
        return C.c_void_p(stream.cuda_stream)
    return C.c_void_p(int(stream))


def _ptr_mem(a):
    """(pointer, mem, keep-alive) of a torch CUDA tensor, a torch CPU tensor or a numpy array (float32)."""
    if a is None:
        return None, None, None
    if isinstance(a, np.ndarray):
        a = np.ascontiguousarray(a, np.float32)
        return C.c_void_p(a.ctypes.data), MEM_HOST, a
    import torch
    if not isinstance(a, torch.Tensor):
        raise TypeError("expected a torch tensor or numpy array")
    if a.dtype != torch.float32:
        raise TypeError("expected float32")
    a = a.contiguous()
    return C.c_void_p(a.data_ptr()), (MEM_DEVICE if a.is_cuda else MEM_HOST), a


def make_observer(theta, phi, center, half_w, half_h=None):
    o = Observer()
    o.theta, o.phi = float(theta), float(phi)
    o.center[:] = [float(c) for c in center]
    o.half_w = float(half_w)
    o.half_h = float(half_w if half_h is None else half_h)
    return o


class Grid:
    """Owner of one krp_grid handle.  Methods mirror the C entry points one to one."""

    def __init__(self, nx, ny, nz, bounds, density, bfield, mueller, opacity, w_min=1e-4, max_scatter=64,
                 stream=None, periodic=0):
        L = lib()
        self._h = C.c_void_p()
        dptr, dmem, dkeep = _ptr_mem(density)
        bptr, bmem, bkeep = _ptr_mem(bfield)
        if bptr is not None and bmem != dmem:
            raise ValueError("density and bfield must live in the same memory space")
        mu = np.ascontiguousarray(np.asarray(mueller, np.float32).reshape(-1, 4))
        op = np.ascontiguousarray(np.asarray(opacity, np.float32).reshape(-1, 4))
        t = Tables(mu.shape[0], mu.ctypes.data, op.shape[0], op.ctypes.data, float(w_min), int(max_scatter), int(periodic))
        b = (C.c_double * 6)(*[float(x) for x in bounds])
        self.shape = (int(nx), int(ny), int(nz))
        self.bounds = [float(x) for x in bounds]
        _check(L.krp_grid_create(C.byref(self._h), int(nx), int(ny), int(nz), b, dptr, bptr, dmem, C.byref(t),
                                 _stream(stream)))
        self.n_obs = self.npx = self.npy = 0
        self._weights = None

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            lib().krp_grid_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def update(self, density, bfield=None, stream=None):
        """New density (and field) for the same grid: arrays as for the constructor."""
        dptr, dmem, dkeep = _ptr_mem(density)
        bptr, bmem, bkeep = _ptr_mem(bfield)
        if bptr is not None and bmem != dmem:
            raise ValueError("density and bfield must live in the same memory space")
        _check(lib().krp_grid_update(self._h, dptr, bptr, dmem, _stream(stream)))

    def stage(self, density, bfield=None, copy_stream=None):
        """Start the host-to-device copy of the next snapshot (host arrays, pinned for an asynchronous copy) on copy_stream."""
        dptr, dmem, dkeep = _ptr_mem(density)
        bptr, bmem, bkeep = _ptr_mem(bfield)
        if dmem != MEM_HOST or (bptr is not None and bmem != MEM_HOST):
            raise ValueError("krp_grid_stage takes host arrays")
        _check(lib().krp_grid_stage(self._h, dptr, bptr, _stream(copy_stream)))

    def update_staged(self, stream=None):
        """Re-pack the cells from the staged snapshot once its copy has arrived."""
        _check(lib().krp_grid_update_staged(self._h, _stream(stream)))

    def source_set(self, kind=0, pos=None, direction=(0, 0, 1), cell_weight=None, emit_records=0, stream=None):
        s = Source()
        s.kind = int(kind)
        if pos is None:
            pos = [(self.bounds[0] + self.bounds[1]) / 2, (self.bounds[2] + self.bounds[3]) / 2,
                   (self.bounds[4] + self.bounds[5]) / 2]
        s.pos[:] = [float(x) for x in pos]
        s.dir[:] = [float(x) for x in direction]
        s.emit_records = int(emit_records)
        if cell_weight is not None:
            if not cell_weight.is_cuda:
                raise ValueError("cell_weight must be a CUDA tensor")
            ptr, _, self._weights = _ptr_mem(cell_weight)
            s.cell_weight = ptr
        _check(lib().krp_source_set(self._h, C.byref(s), _stream(stream)))

    def events_reserve(self, max_events):
        _check(lib().krp_events_reserve(self._h, int(max_events)))

    def transport(self, n_packets, seed, stream=None):
        _check(lib().krp_transport(self._h, int(n_packets), int(seed), _stream(stream)))

    def packet_id_set(self, next_id):
        _check(lib().krp_packet_id_set(self._h, int(next_id)))

    def image(self, observers, npix_x, npix_y, flags=0, stream=None):
        n = len(observers)
        arr = (Observer * n)(*observers)
        _check(lib().krp_image(self._h, arr, n, int(npix_x), int(npix_y), int(flags), _stream(stream)))
        self.n_obs, self.npx, self.npy = n, int(npix_x), int(npix_y)

    def image_get(self, out=None, stream=None):
        """Returns the maps [n_obs,4,npy,npx] fp64: a numpy array (host copy) unless `out` is a CUDA tensor."""
        shape = (self.n_obs, 4, self.npy, self.npx)
        if out is None:
            out = np.empty(shape, np.float64)
        if isinstance(out, np.ndarray):
            assert out.dtype == np.float64 and out.flags.c_contiguous and out.size == int(np.prod(shape))
            _check(lib().krp_image_get(self._h, C.c_void_p(out.ctypes.data), MEM_HOST, _stream(stream)))
            return out.reshape(shape)
        assert out.is_contiguous() and out.numel() == int(np.prod(shape))
        _check(lib().krp_image_get(self._h, C.c_void_p(out.data_ptr()), MEM_DEVICE if out.is_cuda else MEM_HOST,
                                   _stream(stream)))
        return out

    def image_reset(self, stream=None):
        _check(lib().krp_image_reset(self._h, _stream(stream)))

    def stats_get(self):
        s = Stats()
        _check(lib().krp_stats_get(self._h, C.byref(s)))
        return s.as_dict()

    def stats_reset(self, stream=None):
        _check(lib().krp_stats_reset(self._h, _stream(stream)))

    def events_get(self, cap=None, id_first=None, id_count=None):
        """Buffered events as host arrays; with id_first/id_count only those of that packet id range (krp_events_select)."""
        L = lib()
        if id_first is None:
            call = lambda *a: L.krp_events_get(self._h, *a)
        else:
            call = lambda *a: L.krp_events_select(self._h, int(id_first), int(id_count), *a)
        n = C.c_uint64(0)
        _check(call(0, C.byref(n), None, None, None, None, None, None))
        m = n.value if cap is None else min(int(cap), n.value)
        ev = dict(id=np.zeros(m, np.uint64), k=np.zeros(m, np.int32), cell=np.zeros(m, np.int64),
                  pos=np.zeros((m, 3), np.float32), dir=np.zeros((m, 3), np.float32),
                  stokes=np.zeros((m, 4), np.float32))
        if m:
            _check(call(m, C.byref(n), ev["id"].ctypes.data, ev["k"].ctypes.data, ev["cell"].ctypes.data,
                        ev["pos"].ctypes.data, ev["dir"].ctypes.data, ev["stokes"].ctypes.data))
        return ev

    def events_clear(self, stream=None):
        _check(lib().krp_events_clear(self._h, _stream(stream)))

    # --- full scattering matrix of aligned grains ---
    def zmatrix_set(self, Z, stream=None):
        """Z[n_ti, n_to, n_dp, 4, 4] (fp32) in the grain frame, or None to return to the F(Theta) table."""
        if Z is None:
            _check(lib().krp_zmatrix_set(self._h, 0, 0, 0, None, _stream(stream)))
            return
        Z = np.ascontiguousarray(np.asarray(Z, np.float32))
        assert Z.ndim == 5 and Z.shape[3:] == (4, 4)
        _check(lib().krp_zmatrix_set(self._h, Z.shape[0], Z.shape[1], Z.shape[2], C.c_void_p(Z.ctypes.data), _stream(stream)))

    # --- frequency bins ---
    def freq_define(self, tables, kappa_scale, stream=None):
        """tables: list of (mueller [n_ang,4], opacity [n_inc,4], w_min, max_scatter) per bin; kappa_scale: density factor per bin."""
        n = len(tables)
        keep = []
        arr = (Tables * n)()
        for b, (mu, op, w_min, max_scatter) in enumerate(tables):
            mu = np.ascontiguousarray(np.asarray(mu, np.float32).reshape(-1, 4)); op = np.ascontiguousarray(np.asarray(op, np.float32).reshape(-1, 4))
            keep += [mu, op]
            arr[b] = Tables(mu.shape[0], mu.ctypes.data, op.shape[0], op.ctypes.data, float(w_min), int(max_scatter), 0)
        ks = np.ascontiguousarray(np.asarray(kappa_scale, np.float32))
        assert ks.size == n
        _check(lib().krp_freq_define(self._h, n, arr, C.c_void_p(ks.ctypes.data), _stream(stream)))

    def freq_select(self, b, stream=None):
        _check(lib().krp_freq_select(self._h, int(b), _stream(stream)))

    # --- the paper's two-step form ---
    def sgrid_begin(self, observers, stream=None):
        n = len(observers)
        arr = (Observer * n)(*observers)
        _check(lib().krp_sgrid_begin(self._h, arr, n, _stream(stream)))
        self._sg_n_obs = n

    def sgrid_get(self, stream=None):
        """Source grid as a numpy array [nz, ny, nx, n_obs, 4] (fp32)."""
        nx, ny, nz = self.shape
        out = np.empty((nz, ny, nx, max(1, getattr(self, "_sg_n_obs", 0)), 4), np.float32)      # no open grid: the library says so
        _check(lib().krp_sgrid_get(self._h, C.c_void_p(out.ctypes.data), MEM_HOST, _stream(stream)))
        return out

    def sgrid_reset(self, stream=None):
        _check(lib().krp_sgrid_reset(self._h, _stream(stream)))

    def sgrid_end(self):
        _check(lib().krp_sgrid_end(self._h))

    def image_rays(self, observers, npix_x, npix_y, emis=None, stream=None):
        n = len(observers)
        arr = (Observer * n)(*observers)
        eptr, emem, keep = _ptr_mem(emis)
        _check(lib().krp_image_rays(self._h, arr, n, int(npix_x), int(npix_y), eptr, MEM_DEVICE if emem is None else emem,
                                    _stream(stream)))
        self.n_obs, self.npx, self.npy = n, int(npix_x), int(npix_y)

    def image_events_noalloc(self, k, cell, pos, dir, stokes, observer, npix_x, npix_y, img, flags=0, want_rejected=False,
                             stream=None):
        """krp_image_events_noalloc: torch CUDA tensors k int32 [n], cell int64 [n], pos, dir float32 [n,3], stokes float32
        [n,4], img float64 [4,npix_y,npix_x] (added to).  Pointers and sizes only: nothing is copied or allocated here."""
        import torch
        n = int(k.shape[0])
        want = ((k, torch.int32, (n,)), (cell, torch.int64, (n,)), (pos, torch.float32, (n, 3)), (dir, torch.float32, (n, 3)),
                (stokes, torch.float32, (n, 4)), (img, torch.float64, (4, int(npix_y), int(npix_x))))
        for t, dt, shape in want:
            if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dt and tuple(t.shape) == shape and t.is_contiguous()):
                raise TypeError("expected a contiguous CUDA tensor of dtype %s and shape %s" % (dt, shape))
        rej = C.c_uint64(0)
        _check(lib().krp_image_events_noalloc(self._h, n, k.data_ptr(), cell.data_ptr(), pos.data_ptr(), dir.data_ptr(),
                                              stokes.data_ptr(), C.byref(observer), int(npix_x), int(npix_y), int(flags),
                                              img.data_ptr(), C.byref(rej) if want_rejected else None, _stream(stream)))
        return int(rej.value) if want_rejected else None

    def tune(self, transport_block=0, image_block=0, blocks_per_sm=0, flight_burst=0):
        _check(lib().krp_tune(self._h, int(transport_block), int(image_block), int(blocks_per_sm), int(flight_burst)))

    def tune_schedule(self, dir_sort=-1, obs_cells=-1, order_policy=-1):
        _check(lib().krp_tune_schedule(self._h, int(dir_sort), int(obs_cells), int(order_policy)))

    def tune_fused(self, max_packets):
        _check(lib().krp_tune_fused(self._h, int(max_packets)))

    def version(self):
        return lib().krp_version().decode()

    def timing_enable(self, on=True):
        _check(lib().krp_timing_enable(self._h, int(bool(on))))

    def timing_get(self):
        """{class: (milliseconds, launches)} since the last call; synchronises."""
        ms = (C.c_double * T_COUNT)()
        cnt = (C.c_uint64 * T_COUNT)()
        _check(lib().krp_timing_get(self._h, ms, cnt))
        return {T_NAMES[c]: (float(ms[c]), int(cnt[c])) for c in range(T_COUNT)}

    def launch_count(self):
        return int(lib().krp_launch_count(self._h))
