"""ctypes wrapper of oracle/krp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Argument marshalling only; all arithmetic is in krp_oracle.c.  Shares nothing
with paper_2512_01283_b200 (neither imports the other).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "krp_oracle.c")
# Two builds of the same source (R12): "fp32state" is the oracle proper (the state between steps is
# defined in fp32 where the 48-byte record and the queue store it); "pure" is the control build with those
# roundings off (-DORA_STATE_FP32=0).  KRP_ORACLE_VARIANT picks the default (the pins are run on both).
VARIANTS = {"fp32state": ("libkrp_oracle.so", []), "pure": ("libkrp_oracle_pure.so", ["-DORA_STATE_FP32=0"])}
_libs = {}


def default_variant():
    v = os.environ.get("KRP_ORACLE_VARIANT", "fp32state")
    if v not in VARIANTS:
        raise ValueError("KRP_ORACLE_VARIANT must be one of %s" % sorted(VARIANTS))
    return v


def build(force=False, variant=None):
    """Compile krp_oracle.c with gcc (no fast-math: fp64 IEEE as written).  variant=None builds every variant
    and returns the path of the default one."""
    if variant is None:
        for v in VARIANTS:
            build(force, v)
        return os.path.join(_HERE, VARIANTS[default_variant()][0])
    so = os.path.join(_HERE, VARIANTS[variant][0])
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(_SRC):
        tmp = so + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off"] + VARIANTS[variant][1] +
                              ["-o", tmp, _SRC, "-lm"])
        os.replace(tmp, so)
    return so


class OracleStats(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in ("packets", "events", "records", "steps_transport", "steps_image",
                                          "contributions", "dropped", "overflow")] + \
               [(n, C.c_double) for n in ("w_emitted", "w_escaped", "w_absorbed", "w_cut")]

    def as_dict(self):
        return {n: getattr(self, n) for n, _ in self._fields_}


class _Events(C.Structure):
    _fields_ = [("cap", C.c_int64), ("n", C.c_int64), ("cell", C.c_void_p), ("p", C.c_void_p),
                ("n_in", C.c_void_p), ("S", C.c_void_p), ("id", C.c_void_p), ("k", C.c_void_p)]


class Observer(C.Structure):
    _fields_ = [("theta", C.c_double), ("phi", C.c_double), ("center", C.c_double * 3),
                ("half_w", C.c_double), ("half_h", C.c_double)]

    @staticmethod
    def make(theta, phi, center, half_w, half_h=None):
        o = Observer()
        o.theta, o.phi = float(theta), float(phi)
        o.center[:] = [float(c) for c in center]
        o.half_w = float(half_w)
        o.half_h = float(half_w if half_h is None else half_h)
        return o


class OracleEvents:
    """Caller-allocated SoA event list (capacity cap)."""

    def __init__(self, cap):
        self.cap = int(cap)
        self.cell = np.zeros(cap, np.int64)
        self.p = np.zeros((cap, 3), np.float64)
        self.n_in = np.zeros((cap, 3), np.float64)
        self.S = np.zeros((cap, 4), np.float64)
        self.id = np.zeros(cap, np.uint64)
        self.k = np.zeros(cap, np.int32)
        self.c = _Events(self.cap, 0, self.cell.ctypes.data, self.p.ctypes.data, self.n_in.ctypes.data,
                         self.S.ctypes.data, self.id.ctypes.data, self.k.ctypes.data)

    @property
    def n(self):
        return int(self.c.n)

    def clear(self):
        self.c.n = 0


_D = C.POINTER(C.c_double)
_dp = np.ctypeslib.ndpointer(np.float64, flags="C_CONTIGUOUS")
_fp = np.ctypeslib.ndpointer(np.float32, flags="C_CONTIGUOUS")
_ip = np.ctypeslib.ndpointer(np.int32, flags="C_CONTIGUOUS")
_up = np.ctypeslib.ndpointer(np.uint32, flags="C_CONTIGUOUS")


def lib(variant=None):
    variant = variant or default_variant()
    if variant in _libs:
        return _libs[variant]
    L = C.CDLL(build(variant=variant))
    sig = {
        "ora_state_is_fp32": (C.c_int, []),
        "ora_emit": (None, [C.c_void_p, C.c_uint64, C.c_uint64, _ip, _dp, _dp, _D]),
        "ora_emit_full": (None, [C.c_void_p, C.c_uint64, C.c_uint64, _ip, _dp, _dp, _D, _dp]),
        "ora_philox": (None, [_up, _up, _up]),
        "ora_u01": (C.c_double, [C.c_uint32]),
        "ora_u53": (C.c_double, [C.c_uint32, C.c_uint32]),
        "ora_quat_mul": (None, [_dp, _dp, _dp]),
        "ora_quat_from_B": (None, [_dp, _dp]),
        "ora_rot_to_gf": (None, [_dp, _dp, _dp]),
        "ora_rot_to_lab": (None, [_dp, _dp, _dp]),
        "ora_basis": (None, [_dp, _dp, _dp]),
        "ora_eta_gf": (None, [_dp, _dp, _D, _D]),
        "ora_rotate_qu": (None, [_dp, C.c_double, C.c_double]),
        "ora_appA": (None, [_dp, C.c_double, C.c_double, C.c_double, C.c_double]),
        "ora_event_solve": (C.c_double, [C.c_double] * 5),
        "ora_model_create": (C.c_void_p, [C.c_int, C.c_int, C.c_int, _dp, C.c_void_p, C.c_void_p,
                                          C.c_int, _fp, C.c_int, _fp, C.c_double, C.c_int]),
        "ora_model_free": (None, [C.c_void_p]),
        "ora_model_set_periodic": (None, [C.c_void_p, C.c_int]),
        "ora_source_set": (None, [C.c_void_p, C.c_int, _dp, _dp, C.c_void_p, C.c_int]),
        "ora_mueller_at": (None, [C.c_void_p, C.c_double, _dp]),
        "ora_opac_at": (None, [C.c_void_p, C.c_double, _dp]),
        "ora_dda_exit": (C.c_double, [C.c_void_p, _dp, _dp, C.POINTER(C.c_int)]),
        "ora_cell_step": (None, [C.c_void_p, _dp, _dp, _dp, C.c_double]),
        "ora_march": (C.c_int64, [C.c_void_p, _ip, _dp, _dp, _dp, C.c_int64, C.c_void_p, C.c_void_p]),
        "ora_sample_theta": (C.c_double, [C.c_void_p, C.c_double]),
        "ora_phi_accept": (C.c_int, [C.c_double] * 5),
        "ora_scatter_angles": (None, [C.c_void_p, _dp, _dp, _dp, C.c_double, C.c_double, _dp, _dp]),
        "ora_scatter": (C.c_int, [C.c_void_p, _dp, _dp, _dp, C.c_uint64, C.c_uint64, C.c_uint32, _dp, _dp, _D]),
        "ora_transport": (C.c_int64, [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(_Events),
                                      C.POINTER(OracleStats), C.c_int64, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.c_void_p]),
        "ora_peel": (None, [C.c_void_p, _dp, _dp, _dp, _dp]),
        "ora_appA_src": (None, [_dp, C.c_double, C.c_double, C.c_double, _dp, C.c_double]),
        "ora_segment_integral": (None, [_dp, C.c_double, C.c_double, C.c_double, C.c_double, _dp]),
        "ora_transport_deposit": (None, [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint64, C.POINTER(_Events),
                                         C.POINTER(OracleStats), C.POINTER(Observer), C.c_int, C.c_void_p, C.c_void_p,
                                         C.POINTER(C.c_uint64)]),
        "ora_image_rays": (None, [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(Observer), C.c_int, C.c_int, C.c_int, _dp,
                                  C.POINTER(OracleStats)]),
        "ora_ztable_create": (C.c_void_p, [C.c_int, C.c_int, C.c_int, _fp]),
        "ora_ztable_free": (None, [C.c_void_p]),
        "ora_ztable_at": (None, [C.c_void_p, C.c_double, C.c_double, C.c_double, _dp]),
        "ora_ztable_norm": (C.c_double, [C.c_void_p, C.c_double, _dp]),
        "ora_peel_z": (None, [C.c_void_p, _dp, _dp, _dp, _dp, _dp]),
        "ora_scatter_z": (C.c_int, [C.c_void_p, _dp, _dp, _dp, C.c_uint64, C.c_uint64, C.c_uint32, _dp, _dp, _D]),
        "ora_model_set_ztable": (None, [C.c_void_p, C.c_void_p]),
        "ora_image": (None, [C.c_void_p, C.POINTER(_Events), C.POINTER(Observer), C.c_int, C.c_int, C.c_int,
                             C.c_int, _dp, C.c_void_p, C.POINTER(OracleStats)]),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    assert L.ora_state_is_fp32() == (0 if variant == "pure" else 1)
    _libs[variant] = L
    return L


def _v(x, n):
    a = np.ascontiguousarray(np.asarray(x, np.float64).reshape(n))
    return a


class OracleModel:
    """Grid + tables + source.  density [nz,ny,nx] f32 (kappa*rho per unit length),
    bfield [nz,ny,nx,3] f32 or None, mueller [n_ang,4] f32 (S11,S12,S33,S34 on
    Theta_j = j*180/(n_ang-1) deg), opac [n_inc,4] f32 (a1,a2,a3,albedo on
    mu_m = m/(n_inc-1), mu = |cos(angle(n,B))|)."""

    def __init__(self, nx, ny, nz, bounds, density, bfield, mueller, opac, w_min=1e-4, max_scatter=64, variant=None):
        L = self.L = lib(variant)
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.bounds = _v(bounds, 6)
        self.density = np.ascontiguousarray(np.asarray(density, np.float32).reshape(nz, ny, nx))
        self.bfield = None if bfield is None else np.ascontiguousarray(
            np.asarray(bfield, np.float32).reshape(nz, ny, nx, 3))
        self.mueller = np.ascontiguousarray(np.asarray(mueller, np.float32).reshape(-1, 4))
        self.opac = np.ascontiguousarray(np.asarray(opac, np.float32).reshape(-1, 4))
        self._w = None
        self.h = L.ora_model_create(self.nx, self.ny, self.nz, self.bounds, self.density.ctypes.data,
                                    None if self.bfield is None else self.bfield.ctypes.data,
                                    self.mueller.shape[0], self.mueller, self.opac.shape[0], self.opac,
                                    float(w_min), int(max_scatter))
        ctr = [(self.bounds[0] + self.bounds[1]) / 2, (self.bounds[2] + self.bounds[3]) / 2,
               (self.bounds[4] + self.bounds[5]) / 2]
        self.source_set(0, ctr, [0, 0, 1], None, 0)

    def __del__(self):
        if getattr(self, "h", None):
            self.L.ora_model_free(self.h)
            self.h = None

    def set_ztable(self, ztab):
        """Scatter and peel with the full Z (OracleZTable) instead of the F(Theta) table; None switches back."""
        self._ztab = ztab
        self.L.ora_model_set_ztable(self.h, None if ztab is None else ztab.h)

    def set_periodic(self, mask):
        """bit a of mask: axis a (0 x, 1 y, 2 z) is periodic (reading R20)."""
        self.L.ora_model_set_periodic(self.h, int(mask))

    def source_set(self, kind, pos, direction, cell_weight=None, emit_records=0):
        """kind bit0: volume (else point at pos); bit1: collimated along direction (else isotropic)."""
        self._w = None if cell_weight is None else np.ascontiguousarray(np.asarray(cell_weight, np.float32).ravel())
        self.L.ora_source_set(self.h, int(kind), _v(pos, 3), _v(direction, 3),
                             None if self._w is None else self._w.ctypes.data, int(emit_records))

    # --- per-step functions (pins) ---
    def mueller_at(self, theta_deg):
        F = np.zeros(4); self.L.ora_mueller_at(self.h, float(theta_deg), F); return F

    def opac_at(self, mu):
        a = np.zeros(4); self.L.ora_opac_at(self.h, float(mu), a); return a

    def dda_exit(self, p, n):
        ax = C.c_int(-1)
        t = self.L.ora_dda_exit(self.h, _v(p, 3), _v(n, 3), C.byref(ax))
        return t, ax.value

    def cell_step(self, b, n, S, dtau):
        S = _v(S, 4).copy(); self.L.ora_cell_step(self.h, _v(b, 3), _v(n, 3), S, float(dtau)); return S

    def march(self, idx, p, n, S, log_cap=0):
        S = _v(S, 4).copy()
        lc = np.zeros(max(log_cap, 1), np.int64); ld = np.zeros(max(log_cap, 1), np.float64)
        steps = self.L.ora_march(self.h, np.ascontiguousarray(np.asarray(idx, np.int32)), _v(p, 3), _v(n, 3), S,
                                int(log_cap), lc.ctypes.data, ld.ctypes.data)
        m = min(int(steps), log_cap)
        return S, int(steps), lc[:m], ld[:m]

    def emit(self, seed, pid):
        """(cell index triple, cell-local position, direction, tau*) of packet pid (S1, schedule R11)."""
        idx = np.zeros(3, np.int32); p = np.zeros(3); n = np.zeros(3); t = C.c_double(0)
        self.L.ora_emit(self.h, int(seed), int(pid), idx, p, n, C.byref(t))
        return idx, p, n, t.value

    def emit_full(self, seed, pid):
        """emit() plus the Stokes vector (1, q, u, v) the packet starts with (thermal emission of aligned grains: R22)."""
        idx = np.zeros(3, np.int32); p = np.zeros(3); n = np.zeros(3); t = C.c_double(0); S = np.zeros(4)
        self.L.ora_emit_full(self.h, int(seed), int(pid), idx, p, n, C.byref(t), S)
        return idx, p, n, t.value, S

    def sample_theta(self, u):
        return self.L.ora_sample_theta(self.h, float(u))

    def scatter_angles(self, b, n_in, S_in, theta_deg, phi):
        no = np.zeros(3); So = np.zeros(4)
        self.L.ora_scatter_angles(self.h, _v(b, 3), _v(n_in, 3), _v(S_in, 4), float(theta_deg), float(phi), no, So)
        return no, So

    def scatter(self, b, n_in, S_in, seed, pid, k):
        no = np.zeros(3); So = np.zeros(4); tn = C.c_double(0)
        r = self.L.ora_scatter(self.h, _v(b, 3), _v(n_in, 3), _v(S_in, 4), int(seed), int(pid), int(k), no, So,
                              C.byref(tn))
        return no, So, tn.value, r

    def peel(self, n_in, S_in, n_obs):
        So = np.zeros(4); self.L.ora_peel(self.h, _v(n_in, 3), _v(S_in, 4), _v(n_obs, 3), So); return So

    # --- whole-path functions ---
    def transport(self, id0, n_packets, seed, events, stats=None, esc_cap=0):
        st = stats if stats is not None else OracleStats()
        esc = None
        if esc_cap > 0:
            esc = dict(n=np.zeros((esc_cap, 3)), S=np.zeros((esc_cap, 4)), id=np.zeros(esc_cap, np.uint64),
                       k=np.zeros(esc_cap, np.int32))
            ne = self.L.ora_transport(self.h, int(id0), int(n_packets), int(seed), C.byref(events.c), C.byref(st),
                                     int(esc_cap), esc["n"].ctypes.data, esc["S"].ctypes.data,
                                     esc["id"].ctypes.data, esc["k"].ctypes.data)
            esc = {k: v[:ne] for k, v in esc.items()}
        else:
            self.L.ora_transport(self.h, int(id0), int(n_packets), int(seed), C.byref(events.c), C.byref(st),
                                0, None, None, None, None)
        return st, esc

    def image(self, events, observers, npx, npy, flags=0, stats=None, second_moment=True):
        st = stats if stats is not None else OracleStats()
        n_obs = len(observers)
        arr = (Observer * n_obs)(*observers)
        img = np.zeros((n_obs, 4, npy, npx)); img2 = np.zeros_like(img) if second_moment else None
        self.L.ora_image(self.h, C.byref(events.c), arr, n_obs, int(npx), int(npy), int(flags), img,
                        None if img2 is None else img2.ctypes.data, C.byref(st))
        return img, img2, st

    # --- the paper's two-step form (NEXT-1) and thermal emission in the ray step (NEXT-3) ---
    def transport_deposit(self, id0, n_packets, seed, events, observers, stats=None, collisions=False):
        """Transport as usual and deposit every path segment: returns (sgrid [ncell, n_obs, 4], coll [ncell] or None, segments)."""
        st = stats if stats is not None else OracleStats()
        n_obs = len(observers)
        arr = (Observer * n_obs)(*observers)
        ncell = self.nx * self.ny * self.nz
        sgrid = np.zeros((ncell, n_obs, 4))
        coll = np.zeros(ncell) if collisions else None
        nseg = C.c_uint64(0)
        self.L.ora_transport_deposit(self.h, int(id0), int(n_packets), int(seed), C.byref(events.c), C.byref(st), arr, n_obs,
                                     sgrid.ctypes.data, None if coll is None else coll.ctypes.data, C.byref(nseg))
        return sgrid, coll, nseg.value

    def image_rays(self, sgrid, observers, npx, npy, emis=None, stats=None):
        """One ray per pixel with App. A and source terms (scattering source sgrid and/or thermal emission emis [ncell] f32)."""
        st = stats if stats is not None else OracleStats()
        n_obs = len(observers)
        arr = (Observer * n_obs)(*observers)
        img = np.zeros((n_obs, 4, npy, npx))
        if sgrid is not None:
            sgrid = np.ascontiguousarray(sgrid, np.float64)
            assert sgrid.size == self.nx * self.ny * self.nz * n_obs * 4
        if emis is not None:
            emis = np.ascontiguousarray(np.asarray(emis, np.float32).ravel())
            assert emis.size == self.nx * self.ny * self.nz
        self.L.ora_image_rays(self.h, None if sgrid is None else sgrid.ctypes.data, None if emis is None else emis.ctypes.data,
                              arr, n_obs, int(npx), int(npy), img, C.byref(st))
        return img, st


class OracleZTable:
    """Full scattering matrix of aligned grains in the grain frame, Z[n_ti, n_to, n_dp, 4, 4] (fp32), reading R21."""

    def __init__(self, Z, variant=None):
        self.L = lib(variant)
        self.Z = np.ascontiguousarray(np.asarray(Z, np.float32))
        assert self.Z.ndim == 5 and self.Z.shape[3:] == (4, 4)
        self.h = self.L.ora_ztable_create(self.Z.shape[0], self.Z.shape[1], self.Z.shape[2], self.Z.reshape(-1))

    def __del__(self):
        if getattr(self, "h", None):
            self.L.ora_ztable_free(self.h); self.h = None

    def at(self, ti_deg, to_deg, dphi_deg):
        M = np.zeros(16); self.L.ora_ztable_at(self.h, float(ti_deg), float(to_deg), float(dphi_deg), M); return M.reshape(4, 4)

    def norm(self, ti_deg, Sg):
        return self.L.ora_ztable_norm(self.h, float(ti_deg), _v(Sg, 4))

    def peel(self, b, n_in, S_in, n_obs):
        So = np.zeros(4); self.L.ora_peel_z(self.h, _v(b, 3), _v(n_in, 3), _v(S_in, 4), _v(n_obs, 3), So); return So

    def scatter(self, b, n_in, S_in, seed, pid, k):
        no = np.zeros(3); So = np.zeros(4); tn = C.c_double(0)
        r = self.L.ora_scatter_z(self.h, _v(b, 3), _v(n_in, 3), _v(S_in, 4), int(seed), int(pid), int(k), no, So, C.byref(tn))
        return no, So, tn.value, r
