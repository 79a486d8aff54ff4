"""Pins of the oracle (oracle/krp_oracle.c) to things other than itself.

Every expected value here comes from a closed form the paper prints
(/root/reference/PAPER.md, cited as PAPER.md:<line>), from plain mathematics
written out with numpy (rotation matrices, E-vector optics, matrix
exponential), from a library routine (scipy.linalg.expm, cuRAND's host
Philox), or from brute force.  Nothing here calls the CUDA path.
"""
import ctypes as C
import math
import os

import numpy as np
import pytest
import scipy.linalg

from oracle import lib, OracleModel, OracleEvents, OracleStats, Observer

L = lib()
FP32_STATE = bool(L.ora_state_is_fp32())       # False in the pure-fp64 control build (KRP_ORACLE_VARIANT=pure, R12)
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


# ----------------------------------------------------------------------------
# plain-numpy helpers (independent restatements, not oracle calls)
# ----------------------------------------------------------------------------
def Ry(t):
    return np.array([[math.cos(t), 0, math.sin(t)], [0, 1, 0], [-math.sin(t), 0, math.cos(t)]])


def Rz(p):
    return np.array([[math.cos(p), -math.sin(p), 0], [math.sin(p), math.cos(p), 0], [0, 0, 1]])


def sph_basis(n):
    """eq. 4-5 for a unit propagation direction n."""
    n = np.asarray(n, float) / np.linalg.norm(n)
    th = math.acos(max(-1.0, min(1.0, n[2])))
    ph = math.atan2(n[1], n[0]) if (n[0] ** 2 + n[1] ** 2) >= 1e-24 else 0.0
    tv = np.array([math.cos(th) * math.cos(ph), math.cos(th) * math.sin(ph), -math.sin(th)])
    pv = np.array([-math.sin(ph), math.cos(ph), 0.0])
    return tv, pv


def stokes_of_E(e, a, b):
    """Fully linearly polarised light with E along e, in the reference (a, b):
    +Q along a, +U at 45 deg from a toward b (PAPER.md:80 and reading R5)."""
    ea, eb = float(np.dot(e, a)), float(np.dot(e, b))
    I = ea * ea + eb * eb
    return np.array([I, ea * ea - eb * eb, 2 * ea * eb, 0.0])


def rand_unit(rng):
    v = rng.normal(size=3)
    return v / np.linalg.norm(v)


def rayleigh_table(n_ang=181):
    th = np.linspace(0, math.pi, n_ang)
    c = np.cos(th)
    return np.stack([0.75 * (1 + c * c), -0.75 * (1 - c * c), 1.5 * c, np.zeros_like(c)], 1).astype(np.float32)


def const_opac(a1=1.0, a2=0.0, a3=0.0, om=0.5, n_inc=2):
    return np.tile(np.array([a1, a2, a3, om], np.float32), (n_inc, 1))


def box_model(n=(4, 4, 4), kr=1.0, bvec=None, mueller=None, opac=None, bounds=(0, 1, 0, 1, 0, 1), **kw):
    nx, ny, nz = n
    dens = np.full((nz, ny, nx), kr, np.float32) if np.isscalar(kr) else kr
    bf = None
    if bvec is not None:
        bf = np.broadcast_to(np.asarray(bvec, np.float32), (nz, ny, nx, 3)).copy()
    return OracleModel(nx, ny, nz, bounds, dens, bf, rayleigh_table() if mueller is None else mueller,
                       const_opac() if opac is None else opac, **kw)


# ----------------------------------------------------------------------------
# P11  Philox4x32-10 against cuRAND's host generator (library routine)
# ----------------------------------------------------------------------------
def _curand():
    for p in ("libcurand.so", "/usr/local/cuda/lib64/libcurand.so", "libcurand.so.10"):
        try:
            return C.CDLL(p)
        except OSError:
            continue
    return None


def _curand_words(cur, seed, block, nblocks):
    gen = C.c_void_p()
    assert cur.curandCreateGeneratorHost(C.byref(gen), 161) == 0          # CURAND_RNG_PHILOX4_32_10
    assert cur.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    assert cur.curandSetGeneratorOffset(gen, C.c_ulonglong(4 * block)) == 0
    out = np.zeros(4 * nblocks, np.uint32)
    assert cur.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(out.size)) == 0
    cur.curandDestroyGenerator(gen)
    return out.reshape(nblocks, 4)


def _philox(seed, ctr):
    key = np.array([seed & 0xFFFFFFFF, seed >> 32], np.uint32)
    o = np.zeros(4, np.uint32)
    L.ora_philox(key, np.array(ctr, np.uint32), o)
    return o


def test_philox_matches_curand_host():
    """cuRAND's host Philox4_32_10 emits, as its block b, the Philox output for
    key = seed and counter (c_lo, c_hi, b mod 65536, 0), c = b div 65536
    (mapping found by probing the library, not taken from the oracle)."""
    cur = _curand()
    if cur is None:
        pytest.skip("libcurand not found")
    for seed in (1, 0xDEADBEEF12345678, 2 ** 64 - 1):
        for b0 in (0, 65535, 65536 * 12345 + 77, 65536 * (2 ** 33 + 5) + 9):
            w = _curand_words(cur, seed, b0, 3)
            for j in range(3):
                b = b0 + j
                c = b // 65536
                assert (_philox(seed, (c & 0xFFFFFFFF, c >> 32, b % 65536, 0)) == w[j]).all()


def test_philox_counter_word3_and_uniforms():
    # word 3 of the counter (the draw-block index) is not reachable through
    # cuRAND's host API; check that it enters the bijection (all outputs distinct)
    seen = {tuple(_philox(7, (5, 6, 7, b))) for b in range(64)}
    assert len(seen) == 64
    # u01: ((x>>9)+0.5)/2^23, exact in fp32, never 0 or 1 (reading R11)
    for x in (0, 511, 512, 0xFFFFFFFF, 0x80000000):
        u = L.ora_u01(x)
        assert u == ((x >> 9) + 0.5) / 2 ** 23 and 0 < u < 1 and float(np.float32(u)) == u
    assert 0 < L.ora_u53(0, 0) < L.ora_u53(0xFFFFFFFF, 0xFFFFFFFF) < 1


# ----------------------------------------------------------------------------
# P1  quaternions: eq. 1-3
# ----------------------------------------------------------------------------
def qmul(a, b):
    o = np.zeros(4); L.ora_quat_mul(np.asarray(a, float), np.asarray(b, float), o); return o


def test_hamilton_relations_eq1():
    one, i, j, k = np.eye(4)
    for u in (i, j, k):
        assert np.array_equal(qmul(u, u), -one)
    assert np.array_equal(qmul(qmul(i, j), k), -one)
    assert np.array_equal(qmul(i, j), k) and np.array_equal(qmul(j, i), -k)


def test_qB_is_RzRy_and_maps_B_to_z_eq2_eq3():
    rng = np.random.default_rng(1)
    for _ in range(200):
        thB, phB = math.acos(rng.uniform(-1, 1)), rng.uniform(-math.pi, math.pi)
        b = np.array([math.sin(thB) * math.cos(phB), math.sin(thB) * math.sin(phB), math.cos(thB)])
        q = np.zeros(4); L.ora_quat_from_B(b, q)
        # eq. 2 literally
        want = np.array([math.cos(phB / 2) * math.cos(thB / 2), -math.sin(phB / 2) * math.sin(thB / 2),
                         math.cos(phB / 2) * math.sin(thB / 2), math.sin(phB / 2) * math.cos(thB / 2)])
        assert np.allclose(q, want, atol=1e-14)
        assert abs(np.dot(q, q) - 1) < 1e-14                           # unit norm (north_star)
        R = Rz(phB) @ Ry(thB)                                           # rotation taking z to B
        v = rng.normal(size=3)
        g = np.zeros(3); L.ora_rot_to_gf(q, v, g)
        assert np.allclose(g, R.T @ v, atol=1e-13)                      # eq. 3 is the inverse rotation
        l = np.zeros(3); L.ora_rot_to_lab(q, g, l)
        assert np.allclose(l, v, atol=1e-13)                            # round trip
        z = np.zeros(3); L.ora_rot_to_gf(q, b, z)
        assert np.allclose(z, [0, 0, 1], atol=1e-13)                    # B^ -> z_GF


def test_basis_eq4_eq5_right_handed():
    rng = np.random.default_rng(2)
    for _ in range(100):
        n = rand_unit(rng)
        th = np.zeros(3); ph = np.zeros(3); L.ora_basis(n, th, ph)
        tv, pv = sph_basis(n)
        assert np.allclose(th, tv, atol=1e-13) and np.allclose(ph, pv, atol=1e-13)
        assert np.allclose(np.cross(th, ph), n, atol=1e-13)
    th = np.zeros(3); ph = np.zeros(3)
    L.ora_basis(np.array([0, 0, -1.0]), th, ph)                         # pole rule R10: phi = 0
    assert np.allclose(th, [-1, 0, 0]) and np.allclose(ph, [0, 1, 0])


# ----------------------------------------------------------------------------
# P2  reference-frame rotation eq. 6-7 against E-vector optics
# ----------------------------------------------------------------------------
def test_eta_rotation_matches_E_vector_projection():
    rng = np.random.default_rng(3)
    for _ in range(300):
        n, b = rand_unit(rng), rand_unit(rng)
        thB, phB = math.acos(b[2]), math.atan2(b[1], b[0])
        R = Rz(phB) @ Ry(thB)
        tv, pv = sph_basis(n)
        psi = rng.uniform(0, math.pi)
        e = math.cos(psi) * tv + math.sin(psi) * pv                     # E direction, lab
        S = stokes_of_E(e, tv, pv)
        assert np.allclose(S[:3], [1, math.cos(2 * psi), math.sin(2 * psi)])
        # grain-frame reference: basis of n_GF = R^T n, carried back to the lab
        ng = R.T @ n
        tg, pg = sph_basis(ng)
        want = stokes_of_E(e, R @ tg, R @ pg)
        q = np.zeros(4); L.ora_quat_from_B(b, q)
        ce, se = C.c_double(), C.c_double()
        L.ora_eta_gf(q, n, C.byref(ce), C.byref(se))
        assert abs(ce.value ** 2 + se.value ** 2 - 1) < 1e-12
        got = S.copy(); got[3] = 0.3
        L.ora_rotate_qu(got, ce.value, se.value)
        assert np.allclose(got[:3], want[:3], atol=1e-12) and got[0] == S[0] and got[3] == 0.3   # I, V invariant
        # reading R2: same angle, mod pi, from the lab projection theta'_lab = ((n.B)n - B)/sin
        c = float(np.dot(n, b)); tp = (c * n - b) / math.sqrt(1 - c * c)
        c2 = np.dot(tv, tp) ** 2 - np.dot(pv, tp) ** 2; s2 = 2 * np.dot(tv, tp) * np.dot(pv, tp)
        assert abs(c2 - (ce.value ** 2 - se.value ** 2)) < 1e-12 and abs(s2 - 2 * ce.value * se.value) < 1e-12
        L.ora_rotate_qu(got, ce.value, -se.value)                       # and back
        assert np.allclose(got[:3], S[:3], atol=1e-12)


# ----------------------------------------------------------------------------
# P3  App. A with reading R1 for the garbled matrix
# ----------------------------------------------------------------------------
def Kmat(a1, a2, a3):
    return np.array([[a1, a2, 0, 0], [a2, a1, 0, 0], [0, 0, a1, a3], [0, 0, -a3, a1]], float)


def test_appA_equals_matrix_exponential():
    rng = np.random.default_rng(4)
    for _ in range(200):
        a1 = rng.uniform(0.5, 2); a2 = rng.uniform(-0.4, 0.4) * a1; a3 = rng.uniform(-0.5, 0.5)
        dt = 10 ** rng.uniform(-3, 1.3)
        S0 = rng.normal(size=4)
        want = scipy.linalg.expm(-Kmat(a1, a2, a3) * dt) @ S0
        got = S0.copy(); L.ora_appA(got, a1, a2, a3, dt)
        assert np.allclose(got, want, rtol=1e-10, atol=1e-13 * np.abs(S0).max())


def test_appA_printed_solution_source_free():
    """The solution as printed at PAPER.md:302-316 with S_i = 0."""
    a1, a2, a3, dt = 1.3, 0.2, -0.15, 0.7
    I0, Q0, U0, V0 = 1.0, 0.3, -0.2, 0.1
    e = math.exp(-a1 * dt)
    want = [I0 * e * math.cosh(-a2 * dt) + Q0 * e * math.sinh(-a2 * dt),
            I0 * e * math.sinh(-a2 * dt) + Q0 * e * math.cosh(-a2 * dt),
            U0 * e * math.cos(-a3 * dt) + V0 * e * math.sin(-a3 * dt),
            -U0 * e * math.sin(-a3 * dt) + V0 * e * math.cos(-a3 * dt)]
    got = np.array([I0, Q0, U0, V0]); L.ora_appA(got, a1, a2, a3, dt)
    assert np.allclose(got, want, rtol=1e-13)


def test_appA_scalar_limit_semigroup_minkowski_thick():
    S = np.array([1.0, 0.4, -0.3, 0.2])
    a = S.copy(); L.ora_appA(a, 1.5, 0.0, 0.0, 2.0)
    assert np.allclose(a, S * math.exp(-3.0), rtol=1e-14)               # alpha2 = alpha3 = 0
    a = S.copy(); L.ora_appA(a, 1.1, 0.05, 0.02, 0.4); L.ora_appA(a, 1.1, 0.05, 0.02, 1.7)
    b = S.copy(); L.ora_appA(b, 1.1, 0.05, 0.02, 2.1)
    assert np.allclose(a, b, rtol=1e-13)                                # why thick cells are exact
    m0 = S[0] ** 2 - S[1] ** 2 - S[2] ** 2 - S[3] ** 2
    assert abs((b[0] ** 2 - b[1] ** 2 - b[2] ** 2 - b[3] ** 2) / (m0 * math.exp(-2 * 1.1 * 2.1)) - 1) < 1e-12
    t = S.copy(); L.ora_appA(t, 1.05, 0.05, 0.02, 1.0e3)                # delta tau = 1e3: no overflow, no NaN
    assert np.all(np.isfinite(t)) and t[0] >= 0 and t[0] ** 2 >= t[1] ** 2 + t[2] ** 2 + t[3] ** 2


def test_event_solve_root_and_closed_form():
    rng = np.random.default_rng(5)
    for _ in range(200):
        a1 = rng.uniform(0.5, 2); a2 = rng.uniform(-0.3, 0.3) * a1
        Ie = rng.uniform(0.1, 1); q = rng.uniform(-0.9, 0.9)
        t_true = 10 ** rng.uniform(-4, 1.5)
        S = np.array([Ie, q * Ie, 0.0, 0.0]); L.ora_appA(S, a1, a2, 0.0, t_true)
        t = L.ora_event_solve(Ie, q, a1, a2, S[0])
        assert abs(t - t_true) <= 1e-9 * t_true
    assert abs(L.ora_event_solve(0.8, 0.3, 1.25, 0.0, 0.2) - math.log(4.0) / 1.25) < 1e-14


# ----------------------------------------------------------------------------
# P10  DDA ("from cell interface to cell interface", reading R11b)
# ----------------------------------------------------------------------------
def test_dda_chord_and_brute_force():
    rng = np.random.default_rng(6)
    n_ = (4, 5, 3)
    bounds = (0.0, 2.0, -1.0, 1.5, 3.0, 4.5)
    kr = rng.uniform(0.2, 3.0, size=(n_[2], n_[1], n_[0])).astype(np.float32)
    m = box_model(n_, kr, bounds=bounds, opac=const_opac(1, 0, 0, 0.5))
    lo = np.array(bounds[0::2]); hi = np.array(bounds[1::2]); d = (hi - lo) / np.array(n_)
    for _ in range(40):
        idx = np.array([rng.integers(0, n_[a]) for a in range(3)], np.int32)
        p = rng.uniform(0.05, 0.95, 3)
        n = rand_unit(rng)
        x0 = lo + (idx + p) * d
        S, steps, cells, ds = m.march(idx, p, n, [1, 0, 0, 0], log_cap=64)
        # chord to the box edge
        tt = [((hi[a] - x0[a]) / n[a]) if n[a] > 0 else ((lo[a] - x0[a]) / n[a]) for a in range(3)]
        chord = min(tt)
        assert steps == len(cells) and abs(ds.sum() - chord) < 1e-12
        # brute force: fine stepping, which cell is the midpoint of each sub-step in
        N = 200000
        s = (np.arange(N) + 0.5) * chord / N
        X = x0[None, :] + s[:, None] * n[None, :]
        ci = np.minimum(np.floor((X - lo) / d).astype(np.int64), np.array(n_) - 1)
        lin = (ci[:, 2] * n_[1] + ci[:, 1]) * n_[0] + ci[:, 0]
        tau_bf = kr.ravel()[lin].sum() * chord / N
        tau = float((kr.ravel()[cells] * ds).sum())
        assert abs(tau - tau_bf) < 5e-4 * max(tau, 1)
        assert abs(S[0] - math.exp(-tau)) < 1e-13
        # visited cells are those the fine steps see, in order
        seq = lin[np.r_[True, lin[1:] != lin[:-1]]]
        big = ds > 2 * chord / N
        assert list(cells[big]) == [c for c in seq if c in set(cells[big])][:big.sum()] or \
            set(cells[big]) <= set(seq)


def test_dda_tie_order_and_zero_components():
    m = box_model((4, 4, 4))
    t, ax = m.dda_exit([0.5, 0.5, 0.5], [1 / math.sqrt(3)] * 3)
    assert ax == 0 and abs(t - 0.125 * math.sqrt(3)) < 1e-15           # x before y before z
    t, ax = m.dda_exit([0.5, 0.5, 0.5], [0.0, -1.0, 0.0])
    assert ax == 1 and abs(t - 0.125) < 1e-15                           # zero components never exit
    S, steps, cells, ds = m.march(np.array([1, 2, 3], np.int32), [0.5, 0.25, 0.5], [0, 0, -1.0], [1, 0, 0, 0], 16)
    assert steps == 4 and list(cells) == [(z * 4 + 2) * 4 + 1 for z in (3, 2, 1, 0)]
    assert np.allclose(ds, [0.125, 0.25, 0.25, 0.25])


# ----------------------------------------------------------------------------
# P4  uniform aligned slab: source-free corollary of eq. 15
# ----------------------------------------------------------------------------
def test_aligned_slab_cosh_sinh():
    a1, a2, a3 = (float(np.float32(x)) for x in (1.05, 0.05, 0.02))      # the tables are fp32 (R13)
    for bvec, sign in (((1, 0, 0), -1.0), ((0, 1, 0), +1.0)):
        # n = +z: theta^ = x, phi^ = y (pole rule).  B along x: grains remove E || x, Q -> -tanh.
        # B along y: they remove E || y, the light becomes polarised along x = theta^: Q -> +tanh.
        for tau in (0.125, 1.0, 7.0, 30.0, 300.0):        # exact in fp32 (the density array is fp32)
            m = box_model((2, 2, 16), tau, bvec=bvec, opac=const_opac(a1, a2, a3, 0.5))
            S, steps, _, _ = m.march(np.array([0, 1, 0], np.int32), [0.3, 0.6, 0.0], [0, 0, 1.0], [1, 0, 0, 0])
            assert steps == 16
            assert abs(S[0] / (math.exp(-a1 * tau) * math.cosh(a2 * tau)) - 1) < 1e-11 or tau > 100
            assert abs(S[1] / S[0] - sign * math.tanh(a2 * tau)) < 1e-11
            assert abs(S[2]) < 1e-13 * S[0] and S[3] == 0 or tau > 100


def test_aligned_slab_oblique_field_uses_table_and_projection():
    # B at 45 deg to the line of sight in the x-z plane (BASELINE config 3): the
    # opacity table is read at mu = cos 45; polarisation is in the n-B plane, i.e. along x
    n_inc = 91
    mu = np.linspace(0, 1, n_inc); s2 = 1 - mu * mu
    R, c = 1.1, 0.02
    opac = np.stack([1 + 0.5 * (R - 1) * s2, 0.5 * (R - 1) * s2, c * s2, np.full(n_inc, 0.5)], 1).astype(np.float32)
    b = (math.sin(math.pi / 4), 0, math.cos(math.pi / 4))
    m = box_model((2, 2, 8), 3.0, bvec=b, opac=opac)
    a = m.opac_at(math.cos(math.pi / 4))
    s2_45 = 0.5
    assert np.allclose(a, [1 + 0.05 * s2_45, 0.05 * s2_45, 0.02 * s2_45, 0.5], atol=2e-6)   # (dmu)^2 f''/8
    x = math.cos(math.pi / 4) * (n_inc - 1); j = int(x)                 # linear interpolation written out (R13)
    assert np.allclose(a, (1 - (x - j)) * opac[j].astype(float) + (x - j) * opac[j + 1].astype(float), atol=1e-15)
    assert np.allclose(m.opac_at(-0.3), m.opac_at(0.3)) and np.allclose(m.opac_at(1.0), opac[-1])
    S, _, _, _ = m.march(np.array([0, 0, 0], np.int32), [0.5, 0.5, 0.0], [0, 0, 1.0], [1, 0, 0, 0])
    assert abs(S[1] / S[0] + math.tanh(a[1] * 3.0)) < 1e-12 and abs(S[2]) < 1e-15


# ----------------------------------------------------------------------------
# P5  twisted-field slab, eq. 13-14 with reading R6
# ----------------------------------------------------------------------------
def test_twisted_slab_eq14():
    p0 = -0.01                          # R6: p0 = -alpha2/alpha1 and alpha3 = -alpha2
    a2 = -p0
    N = 2000
    z = (np.arange(N) + 0.5) / N        # depth tau grows with +z, total tau = 1
    bf = np.zeros((N, 1, 1, 3), np.float32)
    bf[:, 0, 0, 0] = np.cos(2 * math.pi * z); bf[:, 0, 0, 1] = np.sin(2 * math.pi * z)   # eq. 13
    m = OracleModel(1, 1, N, (0, 1, 0, 1, 0, 1), np.ones((N, 1, 1), np.float32), bf, rayleigh_table(),
                    const_opac(1.0, a2, -a2, 0.5))
    k = p0 / (4 * math.pi)
    for tau in (0.1, 0.25, 0.4, 0.6, 0.85, 1.0):
        iz = int(round(tau * N)) - 1
        # born at depth tau, travels -z to tau = 0 (R6); reference of n = -z is theta^ = -x, phi^ = +y
        S, steps, _, _ = m.march(np.array([0, 0, iz], np.int32), [0.5, 0.5, 1.0], [0, 0, -1.0], [1, 0, 0, 0])
        assert steps == iz + 1
        x = 4 * math.pi * tau
        want = np.array([k * math.sin(x), -k * (1 - math.cos(x)), k * k * (math.sin(x) - x)])
        got = S[1:] / S[0]
        assert abs(got[0] - want[0]) < 3e-6 and abs(got[1] - want[1]) < 3e-6      # O(p0^2 tau) + O(1/N^2)
        assert abs(got[2] - want[2]) < 2e-8


# ----------------------------------------------------------------------------
# P6  peel-off: Rayleigh single scattering, dipole E-vector optics, eq. 12
# ----------------------------------------------------------------------------
def test_peel_rayleigh_degree_and_orientation():
    m = box_model()
    rng = np.random.default_rng(7)
    for _ in range(300):
        n_in, n_obs = rand_unit(rng), rand_unit(rng)
        mu = float(np.dot(n_in, n_obs))
        S = m.peel(n_in, [1, 0, 0, 0], n_obs)
        assert abs(S[0] * 4 * math.pi - 0.75 * (1 + mu * mu)) < 2e-4            # table interpolation
        P = math.hypot(S[1], S[2]) / S[0]
        assert abs(P - (1 - mu * mu) / (1 + mu * mu)) < 2e-4 and abs(S[3]) < 1e-15
        s = np.cross(n_in, n_obs); s /= np.linalg.norm(s)                       # E is normal to the plane
        to, po = sph_basis(n_obs)
        want = stokes_of_E(s, to, po)
        assert np.allclose(np.array([S[1], S[2]]) / (P * S[0]), want[1:3], atol=1e-9)


def test_peel_fully_polarised_dipole():
    """Rayleigh = dipole: E_out is E_in projected on the plane normal to n_obs,
    phase function 3/(8 pi) (1 - (e.n_obs)^2) per unit incident flux."""
    m = box_model()
    rng = np.random.default_rng(8)
    for _ in range(300):
        n_in, n_obs = rand_unit(rng), rand_unit(rng)
        ti, pi_ = sph_basis(n_in)
        psi = rng.uniform(0, math.pi)
        e = math.cos(psi) * ti + math.sin(psi) * pi_
        S = m.peel(n_in, stokes_of_E(e, ti, pi_), n_obs)
        eo = e - np.dot(e, n_obs) * n_obs
        to, po = sph_basis(n_obs)
        want = 3 / (8 * math.pi) * stokes_of_E(eo, to, po)
        assert np.allclose(S, want, atol=1e-4 * 3 / (8 * math.pi))           # 1-degree table: (dT)^2 f"/8


def test_peel_inclined_disk_eq12():
    """PAPER.md:135 eq. 12: in-plane isotropic illumination of a thin disk seen at
    inclination i gives p = sin^2 i / (2 + sin^2 i), along the minor axis, U = 0.
    Values also stored in tests/golden/eq12_inclined_disk.txt."""
    m = box_model()
    gold = np.loadtxt(os.path.join(GOLD, "eq12_inclined_disk.txt"))
    for inc_deg, p_gold in gold:
        inc = math.radians(inc_deg)
        assert abs(p_gold - math.sin(inc) ** 2 / (2 + math.sin(inc) ** 2)) < 5e-7
        n_obs = np.array([math.sin(inc), 0, math.cos(inc)])
        tot = np.zeros(4)
        for a in np.linspace(0, 2 * math.pi, 720, endpoint=False) + 0.001:
            tot += m.peel([math.cos(a), math.sin(a), 0.0], [1, 0, 0, 0], n_obs)
        # minor axis of the projected disk = projection of z = -theta^_obs: +Q (reading R14)
        assert abs(tot[1] / tot[0] - p_gold) < 1e-4 and abs(tot[2] / tot[0]) < 1e-6


# ----------------------------------------------------------------------------
# P7  scattering: sampler distributions and the rotation chain of S5
# ----------------------------------------------------------------------------
def hg_table(g, n_ang=181, pmax=0.4):
    th = np.linspace(0, math.pi, n_ang); c = np.cos(th)
    s11 = (1 - g * g) / (1 + g * g - 2 * g * c) ** 1.5
    s11 /= 0.5 * np.trapezoid(s11 * np.sin(th), th)
    pol = (1 - c * c) / (1 + c * c)
    return np.stack([s11, -pmax * s11 * pol, s11 * 2 * c / (1 + c * c), -0.2 * s11 * pol], 1).astype(np.float32)


def test_theta_sampler_moments():
    u = (np.arange(200000) + 0.5) / 200000                     # stratified: a quadrature of the inverse CDF
    m = box_model()
    th = np.array([m.sample_theta(x) for x in u[::10]])
    c = np.cos(np.radians(th))
    assert abs(c.mean()) < 2e-4 and abs((c * c).mean() - 0.4) < 3e-4          # Rayleigh: <mu^2> = 2/5
    g = 0.5
    m = box_model(mueller=hg_table(g))
    th = np.array([m.sample_theta(x) for x in u[::10]])
    assert abs(np.cos(np.radians(th)).mean() - g) < 1.5e-3                    # HG: <mu> = g
    assert m.sample_theta(1e-9) < 1.0 and m.sample_theta(1 - 1e-9) > 179.0
    # piecewise-linear CDF: histogram against S11 sin(Theta) on the nodes
    h, _ = np.histogram(th, bins=18, range=(0, 180))
    T = np.radians(np.linspace(0, 180, 181)); w = hg_table(g)[:, 0].astype(float) * np.sin(T)
    cdf = np.r_[0, np.cumsum(0.5 * (w[1:] + w[:-1]))]; cdf /= cdf[-1]
    assert np.allclose(h / h.sum(), np.diff(cdf[::10]), atol=2e-4)


def test_phi_accept_distribution():
    rng = np.random.default_rng(9)
    p12, q, u_ = -0.8, 0.6, -0.3
    phi = rng.uniform(0, 2 * math.pi, 400000); ua = rng.uniform(0, 1, 400000)
    acc = np.array([L.ora_phi_accept(p12, q, u_, a, b) for a, b in zip(phi, ua)], bool)
    bound = 1 + abs(p12) * math.hypot(q, u_)
    assert abs(acc.mean() - 1 / bound) < 4e-3                                  # mean of the pdf is 1
    f = phi[acc]
    c2 = np.cos(2 * f).mean(); s2 = np.sin(2 * f).mean()                       # pdf ~ 1 + p12(q cos2f + u sin2f)
    assert abs(c2 - 0.5 * p12 * q) < 6e-3 and abs(s2 - 0.5 * p12 * u_) < 6e-3


def test_scatter_angles_geometry_and_dipole_optics():
    rng = np.random.default_rng(10)
    m = box_model()
    for _ in range(300):
        b, n_in = rand_unit(rng), rand_unit(rng)
        b = b.astype(np.float32).astype(float); n_in = n_in.astype(np.float32).astype(float)
        Theta = rng.uniform(1, 179); phi = rng.uniform(0, 2 * math.pi)
        ti, pi_ = sph_basis(n_in)
        psi = rng.uniform(0, math.pi)
        e = math.cos(psi) * ti + math.sin(psi) * pi_
        n_out, S = m.scatter_angles(b, n_in, stokes_of_E(e, ti, pi_), Theta, phi)
        # geometry in the grain frame (R = Rz Ry takes z_GF to B^)
        bn = b / np.linalg.norm(b)
        R = Rz(math.atan2(bn[1], bn[0])) @ Ry(math.acos(bn[2]))
        ng = R.T @ (n_in / np.linalg.norm(n_in))
        tg, pg = sph_basis(ng)
        T = math.radians(Theta)
        want_g = math.cos(T) * ng + math.sin(T) * (math.cos(phi) * tg + math.sin(phi) * pg)
        assert np.allclose(n_out, R @ want_g, atol=2e-7)                        # fp32-rounded state (R12)
        assert abs(np.linalg.norm(n_out) - 1) < 2e-7
        # optics: dipole projection of E on the plane normal to n_out
        no = n_out / np.linalg.norm(n_out)
        eo = e - np.dot(e, no) * no
        to, po = sph_basis(no)
        want = stokes_of_E(eo, to, po); want /= want[0]
        assert abs(S[0] - 1) < 1e-14
        if np.dot(eo, eo) > 1e-3:
            # 1-degree table: absolute error ~1e-4 in F S, amplified by 1/I_out = 1/|eo|^2
            assert np.allclose(S[1:3], want[1:3], atol=2e-4 / np.dot(eo, eo))
    # I^2 >= Q^2+U^2+V^2 after scattering (north_star invariant), on a table strictly inside the
    # physical cone S11^2 >= S12^2+S33^2+S34^2 (Rayleigh sits on its boundary, up to fp32 rounding)
    mh = box_model(mueller=hg_table(0.5))
    for _ in range(300):
        S_in = np.r_[1.0, rand_unit(rng) * rng.uniform(0, 1)]
        _, S = mh.scatter_angles(rand_unit(rng), rand_unit(rng), S_in, rng.uniform(0, 180), rng.uniform(0, 6.28))
        assert S[0] == 1.0 and S[1] ** 2 + S[2] ** 2 + S[3] ** 2 <= 1 + 1e-12
    # unpolarised in: degree (1-mu^2)/(1+mu^2) (north_star pin), any B
    n_out, S = m.scatter_angles([0.3, -0.2, 0.9], [0, 0, 1.0], [1, 0, 0, 0], 60.0, 1.0)
    assert abs(math.hypot(S[1], S[2]) - (1 - 0.25) / (1 + 0.25)) < 1e-4


# ----------------------------------------------------------------------------
# S5 draws: the schedule of reading R11 (block 0: Theta, phi, accept, next tau*)
# ----------------------------------------------------------------------------
def test_scatter_draw_schedule():
    m = box_model(mueller=hg_table(0.5))
    rng = np.random.default_rng(11)
    seen_retry = 0
    for t in range(400):
        b, n_in = rand_unit(rng), rand_unit(rng).astype(np.float32).astype(float)
        S_in = np.r_[1.0, rand_unit(rng) * 0.9]
        seed, pid, k = 12345 + t, 2 ** 33 + 17 * t, 1 + t % 7
        n_out, S, tau_next, rounds = m.scatter(b, n_in, S_in, seed, pid, k)
        w = _philox(seed, (pid & 0xFFFFFFFF, pid >> 32, k, 0))
        u = [L.ora_u01(int(x)) for x in w]
        Theta = m.sample_theta(u[0])
        assert abs(tau_next + math.log(u[3])) < 1e-15
        # replay the rejection loop with the documented words
        F = m.mueller_at(Theta); p12 = F[1] / F[0]
        q4 = np.zeros(4); L.ora_quat_from_B(b, q4)
        ce, se = C.c_double(), C.c_double(); L.ora_eta_gf(q4, n_in, C.byref(ce), C.byref(se))
        Sg = S_in.copy(); L.ora_rotate_qu(Sg, ce.value, se.value)
        cands = [(u[1], u[2])]
        blk = 1
        while len(cands) < 64:
            w = _philox(seed, (pid & 0xFFFFFFFF, pid >> 32, k, blk)); blk += 1
            uu = [L.ora_u01(int(x)) for x in w]
            cands += [(uu[0], uu[1]), (uu[2], uu[3])]
        for r, (up, ua) in enumerate(cands, 1):
            phi = 2 * math.pi * up
            if ua * (1 + abs(p12) * math.hypot(Sg[1], Sg[2])) < 1 + p12 * (Sg[1] * math.cos(2 * phi) + Sg[2] * math.sin(2 * phi)):
                break
        assert r == rounds
        seen_retry += rounds > 1
        n2, S2 = m.scatter_angles(b, n_in, S_in, Theta, phi)
        assert np.array_equal(n2, n_out) and np.array_equal(S2, S)
    assert seen_retry > 20


# ----------------------------------------------------------------------------
# P8  transport: exp(-tau) escape, dichroic survival, energy conservation
# ----------------------------------------------------------------------------
def run_transport(m, n, seed, cap=None, esc=False):
    ev = OracleEvents(cap or 40 * n)
    st, e = m.transport(0, n, seed, ev, esc_cap=n if esc else 0)
    assert st.overflow == 0
    return ev, st, e


def test_collimated_beam_pure_absorber_escape_fraction():
    tau, N, seed = 2.0, 200000, 3
    m = box_model((8, 8, 8), tau, opac=const_opac(1, 0, 0, 0.0))
    m.source_set(2, [0.4, 0.6, 0.0], [0, 0, 1.0], None, 0)
    ev, st, esc = run_transport(m, N, seed, esc=True)
    p = math.exp(-tau)
    assert abs(st.w_escaped / N - p) < 4 * math.sqrt(p * (1 - p) / N)
    # exactly the packets whose tau* = -ln u_2 exceeds tau (u_2 = word 2 of block 0, R11)
    ids = np.arange(2000)
    u = np.array([L.ora_u01(int(_philox(seed, (i, 0, 0, 0))[2])) for i in ids])
    assert set(esc["id"][esc["id"] < 2000]) == set(ids[-np.log(u) > tau])
    # pure absorber: every interacting packet has exactly one event, weight 0, all absorbed
    assert st.events == N - len(esc["id"]) and abs(st.w_absorbed - st.events) < 1e-9 and st.w_cut == 0
    # depth of the first event ~ truncated exponential: mean of tau' given tau' < tau
    z = ev.p[:ev.n, 2] / 8 + (ev.cell[:ev.n] // 64) / 8
    want = (1 - (1 + tau) * math.exp(-tau)) / (1 - math.exp(-tau)) / tau
    assert abs(z.mean() - want) < 4 * 0.28 / math.sqrt(ev.n)


def test_collimated_direction_is_normalised():
    """Reading R23: the `dir` of a collimated source need not be normalised (include/krp.h) -- the packet direction is the unit
    vector along it, so the optical depth along the beam does not scale with |dir|.  A beam along (0,0,3) through a pure
    absorber of depth tau: escape fraction e^{-tau} (it would be e^{-tau/3} if the march took |dir| as path length per unit
    parameter), the same packets escape as with (0,0,1), events at the same places with unit directions; and an oblique
    beam along k*(1,2,2)/3 for k = 0.2, 1, 7 gives identical records."""
    tau, N, seed = 2.0, 100000, 3
    out = []
    for k in (1.0, 3.0):
        m = box_model((8, 8, 8), tau, opac=const_opac(1, 0, 0, 0.0))
        m.source_set(2, [0.4, 0.6, 0.0], [0, 0, k], None, 0)
        ev, st, esc = run_transport(m, N, seed, esc=True)
        p = math.exp(-tau)
        assert abs(st.w_escaped / N - p) < 4 * math.sqrt(p * (1 - p) / N), (k, st.w_escaped / N, p)
        assert np.array_equal(ev.n_in[:ev.n], np.broadcast_to([0.0, 0.0, 1.0], (ev.n, 3)))
        out.append((set(esc["id"]), ev.cell[:ev.n].copy(), ev.p[:ev.n].copy()))
    assert out[0][0] == out[1][0] and np.array_equal(out[0][1], out[1][1]) and np.array_equal(out[0][2], out[1][2])
    recs = []
    for k in (0.2, 1.0, 7.0):
        m = box_model((6, 6, 6), 3.0, opac=const_opac(1, 0, 0, 0.6))
        m.source_set(2, [0.1, 0.2, 0.0], [k / 3, 2 * k / 3, 2 * k / 3], None, 0)
        ev, st, esc = run_transport(m, 4000, 11, esc=True)
        recs.append((ev.n, ev.cell[:ev.n].copy(), ev.p[:ev.n].copy(), ev.n_in[:ev.n].copy(), st.w_escaped))
    for r in recs[1:]:
        assert r[0] == recs[0][0] and np.array_equal(r[1], recs[0][1]) and r[4] == recs[0][4]
        assert np.allclose(r[2], recs[0][2], atol=2e-7) and np.allclose(r[3], recs[0][3], atol=2e-7)     # dir/|dir| to fp64 rounding, then fp32
    d0 = recs[0][3][0]
    assert abs(float(np.dot(d0.astype(np.float64), d0.astype(np.float64))) - 1.0) < 3e-7


def test_source_outside_the_box_starts_on_its_surface():
    """Reading R24: a source position outside the box is moved to the nearest point of the box, coordinate by coordinate --
    the records equal those of a source placed at that point."""
    recs = []
    for pos in ([1.4, 0.6, -0.2], [1.0, 0.6, 0.0]):          # box [0,1]^3
        m = box_model((6, 6, 6), 3.0, opac=const_opac(1, 0, 0, 0.6))
        m.source_set(0, pos, [0, 0, 1.0], None, 0)
        ev, st, esc = run_transport(m, 3000, 9, esc=True)
        recs.append((ev.n, ev.cell[:ev.n].copy(), ev.p[:ev.n].copy(), ev.n_in[:ev.n].copy(), st.w_escaped))
    a, b = recs
    assert a[0] == b[0] and a[0] > 500 and a[4] == b[4]
    for k in (1, 2, 3):
        assert np.array_equal(a[k], b[k])
    assert np.all((a[2] >= 0.0) & (a[2] <= 1.0))


def test_dichroic_survival_sampling():
    """Reading R7: the survival probability of a flight is I(s)/I(0) of App. A.
    Unpolarised beam, n perpendicular to B: escape fraction e^{-a1 tau} cosh(a2 tau) (P4)."""
    a1, a2, tau, N = 1.0, 0.5, 1.5, 200000
    m = box_model((4, 4, 12), tau, bvec=(1, 0, 0), opac=const_opac(a1, a2, 0.1, 0.0))
    m.source_set(2, [0.5, 0.5, 0.0], [0, 0, 1.0], None, 0)
    ev, st, esc = run_transport(m, N, 5, esc=True)
    p = math.exp(-a1 * tau) * math.cosh(a2 * tau)
    assert abs(st.w_escaped / N - p) < 4 * math.sqrt(p * (1 - p) / N)
    # escaped packets carry the normalised App. A state: q = -tanh(a2 tau) (B along x = theta^ of +z)
    assert np.allclose(esc["S"][:, 1], -math.tanh(a2 * tau), atol=1e-12) and np.allclose(esc["S"][:, 0], 1.0)
    # event depths: CDF 1 - e^{-a1 t} cosh(a2 t); compare the fraction of events before tau/2
    t = (ev.p[:ev.n, 2] + ev.cell[:ev.n] // 16) / 12 * tau
    F = lambda x: 1 - math.exp(-a1 * x) * math.cosh(a2 * x)
    frac = (t < tau / 2).mean(); want = F(tau / 2) / F(tau)
    assert abs(frac - want) < 4 * math.sqrt(want * (1 - want) / ev.n)
    # Stokes at the event: q = -tanh(a2 t), normalised to I = 1, weight omega W = 0 here -> S stored is 0
    assert np.all(ev.S[:ev.n] == 0)


def test_event_stokes_in_dichroic_medium_and_invariants():
    a1, a2, a3, om = 1.0, 0.3, 0.1, 0.7
    m = box_model((6, 6, 6), 3.0, bvec=(1, 0, 0), mueller=hg_table(0.3), opac=const_opac(a1, a2, a3, om))
    m.source_set(2, [0.5, 0.5, 0.0], [0, 0, 1.0], None, 0)
    N = 20000
    ev, st, esc = run_transport(m, N, 9, esc=True)
    n = ev.n
    S = ev.S[:n]
    # first events: omega (1, -tanh(a2 t), 0, 0) with t the depth in tau units
    first = ev.k[:n] == 1
    t = (ev.p[:n, 2] + ev.cell[:n] // 36) / 6 * 3.0
    assert np.allclose(S[first, 0], om, rtol=1e-7)                           # omega is an fp32 table entry
    assert np.allclose(S[first, 1] / S[first, 0], -np.tanh(a2 * t[first]), atol=1e-9)
    # invariants on every event and every escaping packet (north_star)
    assert np.all(S[:, 0] ** 2 >= (S[:, 1:] ** 2).sum(1) * (1 - 1e-12))
    E = esc["S"]; assert np.all(E[:, 0] ** 2 >= (E[:, 1:] ** 2).sum(1) * (1 - 1e-12))
    assert np.allclose(np.linalg.norm(ev.n_in[:n], axis=1), 1, atol=2e-7)
    assert np.array_equal(ev.n_in[:n].astype(np.float32).astype(float), ev.n_in[:n])     # fp32 state (R12)
    if FP32_STATE:
        assert np.array_equal(ev.p[:n].astype(np.float32).astype(float), ev.p[:n])       # fp32 positions (R12)
    assert np.all((ev.p[:n] >= 0) & (ev.p[:n] <= 1))
    # weights: k-th event carries omega^k
    assert np.allclose(S[:, 0], float(np.float32(om)) ** ev.k[:n], rtol=1e-12)
    # energy conservation against albedo
    assert st.packets == N and st.w_emitted == N and st.events == n
    assert abs(st.w_emitted - (st.w_escaped + st.w_absorbed + st.w_cut)) < 1e-9 * N
    assert abs(esc["S"][:, 0].sum() - st.w_escaped) < 1e-9 * N
    # termination (R12): W < w_min = 1e-4 first happens at k = 26 for omega = 0.7
    assert ev.k[:n].max() <= 26
    m = box_model((4, 4, 4), 80.0, opac=const_opac(1, 0, 0, 0.5))           # deep box: 0.5^14 < 1e-4 <= 0.5^13
    ev, st, _ = run_transport(m, 300, 2)
    assert ev.k[:ev.n].max() == 14 and abs(st.w_cut / 0.5 ** 14 - round(st.w_cut / 0.5 ** 14)) < 1e-9
    assert st.w_cut > 0 and abs(st.w_emitted - (st.w_escaped + st.w_absorbed + st.w_cut)) < 1e-9


def test_max_scatter_cut():
    m = box_model((4, 4, 4), 50.0, opac=const_opac(1, 0, 0, 1.0), max_scatter=5)
    ev, st, _ = run_transport(m, 500, 1)
    assert ev.k[:ev.n].max() == 5 and st.w_absorbed == 0
    assert abs(st.w_emitted - st.w_escaped - st.w_cut) < 1e-9


def test_voxelised_sphere_escape_fraction():
    """BASELINE config 1 geometry: 32^3, kappa rho constant inside r < L/2 (cell centres),
    radial tau = 1, centred isotropic point source, pure absorber: the escape fraction is
    the direction average of exp(-tau_vox(n)), within the staircase error of exp(-1)."""
    n = 32; tau = 1.0
    c = (np.arange(n) + 0.5) / n - 0.5
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    kr = np.where(X * X + Y * Y + Z * Z < 0.25, tau / 0.5, 0.0).astype(np.float32)
    m = box_model((n, n, n), kr, opac=const_opac(1, 0, 0, 0.0))
    N = 100000
    ev, st, _ = run_transport(m, N, 1)
    frac = st.w_escaped / N
    # brute force: fine stepping along 3000 random directions from the centre
    rng = np.random.default_rng(12)
    d = rng.normal(size=(3000, 3)); d /= np.linalg.norm(d, axis=1)[:, None]
    s = (np.arange(4000) + 0.5) / 4000 * 0.6
    P = 0.5 + d[:, None, :] * s[None, :, None]
    ok = np.all((P >= 0) & (P < 1), axis=2)
    I = np.clip(np.floor(P * n).astype(int), 0, n - 1)
    tv = (kr[I[..., 2], I[..., 1], I[..., 0]] * ok).sum(1) * 0.6 / 4000
    want = np.exp(-tv).mean(); sig_dir = np.exp(-tv).std() / math.sqrt(3000)
    assert abs(frac - want) < 4 * (math.sqrt(want * (1 - want) / N) + sig_dir)
    assert abs(frac - math.exp(-1)) < 0.03                                    # staircase error ~ dx/R


def test_volume_source_positions():
    n = (4, 3, 2)
    m = box_model(n, 0.0)
    m.source_set(1, [0, 0, 0], [0, 0, 1], None, 1)                           # uniform in volume, emission records on
    N = 48000
    ev, st, _ = run_transport(m, N, 4)
    assert ev.n == N and st.records == N and st.events == 0 and np.all(ev.k[:N] == 0)
    cnt = np.bincount(ev.cell[:N], minlength=24)
    assert np.all(np.abs(cnt - N / 24) < 5 * math.sqrt(N / 24))
    assert np.allclose(ev.p[:N].mean(0), 0.5, atol=5 * 0.29 / math.sqrt(N))
    assert abs(ev.n_in[:N, 2].mean()) < 5 * 0.58 / math.sqrt(N)              # isotropic
    w = np.arange(24, dtype=np.float32)                                      # weighted: P(cell) ~ w
    m.source_set(1, [0, 0, 0], [0, 0, 1], w, 1)
    ev, st, _ = run_transport(m, N, 4)
    cnt = np.bincount(ev.cell[:N], minlength=24)
    want = N * w / w.sum()
    assert cnt[0] == 0 and np.all(np.abs(cnt - want) < 5 * np.sqrt(want + 1))


# ----------------------------------------------------------------------------
# P9  imaging against the paper's naive estimator
# ----------------------------------------------------------------------------
def test_image_matches_naive_cone_estimator():
    """Collimated beam along +z into a small cube, Rayleigh, albedo 0.9.  The image summed
    over pixels is the radiant intensity toward the observer [weight/sr]; the naive
    estimator bins escaping packets in a cone about the observer direction and divides by
    its solid angle.  Four observers at 90 deg (phi = 0,90,180,270) are equivalent by symmetry."""
    m = box_model((8, 8, 8), 1.5, opac=const_opac(1, 0, 0, 0.9))
    m.source_set(2, [0.5, 0.5, 0.0], [0, 0, 1.0], None, 0)
    N = 400000
    ev, st, esc = run_transport(m, N, 21, esc=True)
    obs = [Observer.make(math.pi / 2, k * math.pi / 2, [0.5, 0.5, 0.5], 0.9) for k in range(4)]
    img, img2, st2 = m.image(ev, obs, 16, 16, 0)
    assert st2.dropped == 0 and st2.contributions == 4 * ev.n
    tot = img.sum(axis=(2, 3)) / N                                           # [obs, 4]
    half = math.radians(12.0); dom = 2 * math.pi * (1 - math.cos(half))
    naive = np.zeros((4, 4)); cnt = np.zeros(4)
    for k in range(4):
        no = np.array([math.cos(k * math.pi / 2), math.sin(k * math.pi / 2), 0.0])
        sel = esc["n"] @ no > math.cos(half)
        naive[k] = esc["S"][sel].sum(0) / dom / N; cnt[k] = sel.sum()
    a, b = tot.mean(0), naive.mean(0)
    rel = 1 / math.sqrt(cnt.sum())
    assert cnt.sum() > 8000
    assert abs(a[0] / b[0] - 1) < 4 * rel + 0.02                             # normalisation incl. 1/(4 pi)
    # strongly polarised (near 90-degree Rayleigh scattering), normal to the scattering plane:
    # E along the horizontal = phi^_obs, so Q < 0 in the theta^ reference (R14)
    assert a[1] / a[0] < -0.5 and abs(a[1] / a[0] - b[1] / b[0]) < 0.03
    assert abs(a[2] / a[0]) < 0.01 and abs(b[2] / b[0]) < 0.03
    for k in range(4):                                                       # the four views agree
        assert abs(tot[k, 0] / a[0] - 1) < 0.02 and abs(tot[k, 1] / a[1] - 1) < 0.03
    # second moments are the sums of squares of the same contributions
    assert np.all(img2 >= 0) and np.all(img2[:, 0].sum() >= (img[:, 0] ** 2).sum() / ev.n)


def test_image_direct_light_and_projection():
    """One emission record at a known place: pixel position (R14: x along phi^_obs, y along
    -theta^_obs) and value W/(4 pi) exp(-tau to the edge)."""
    m = box_model((8, 8, 8), 2.0, opac=const_opac(1, 0, 0, 0.5), bounds=(-1, 1, -1, 1, -1, 1))
    m.source_set(0, [0.3, -0.2, 0.5], [0, 0, 1], None, 1)
    ev = OracleEvents(4)
    st, _ = m.transport(0, 1, 1, ev)
    assert ev.k[0] == 0 and np.allclose(ev.S[0], [1, 0, 0, 0])
    ev.c.n = 1                                                               # keep the emission record only
    th, ph = math.radians(60), math.radians(30)
    o = Observer.make(th, ph, [0, 0, 0], 1.5, 1.0)
    img, _, st2 = m.image(ev, [o], 30, 20, 1)
    n_obs = np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), math.cos(th)])
    tv, pv = sph_basis(n_obs)
    # the record holds the cell index and the fp32 cell-local position (reading R12): rebuild x from them
    cl = (np.array([0.3, -0.2, 0.5]) + 1) / 0.25
    frac = cl - np.floor(cl)
    x = -1 + (np.floor(cl) + (frac.astype(np.float32).astype(float) if FP32_STATE else frac)) * 0.25
    ix = int(math.floor((np.dot(x, pv) / 1.5 + 1) * 15)); iy = int(math.floor((-np.dot(x, tv) / 1.0 + 1) * 10))
    tt = min(((1 - x[a]) / n_obs[a]) if n_obs[a] > 0 else ((-1 - x[a]) / n_obs[a]) for a in range(3))
    assert st2.contributions == 1 and np.count_nonzero(img[0, 0]) == 1
    assert abs(img[0, 0, iy, ix] - math.exp(-2.0 * tt) / (4 * math.pi)) < 1e-14
    img, _, st2 = m.image(ev, [o], 30, 20, 0)                                # flag off: not imaged
    assert st2.contributions == 0 and not img.any()
    o2 = Observer.make(th, ph, [5, 5, 5], 0.1)                               # out of frame: dropped, counted
    img, _, st2 = m.image(ev, [o2], 8, 8, 1)
    assert st2.dropped == 1 and not img.any()


# ----------------------------------------------------------------------------
# second-moment map: the sigma of every "3 sigma per pixel" parity assertion
# ----------------------------------------------------------------------------
def _manual_events(m, recs):
    """Event list written by hand: recs = [(idx triple, cell-local p, n_in, S, k)]."""
    ev = OracleEvents(len(recs))
    for i, (idx, p, n_in, S, k) in enumerate(recs):
        ev.cell[i] = (idx[2] * m.ny + idx[1]) * m.nx + idx[0]
        ev.p[i] = p; ev.n_in[i] = n_in; ev.S[i] = S; ev.id[i] = i; ev.k[i] = k
    ev.c.n = len(recs)
    return ev


def test_image_second_moment_is_the_sum_of_squares():
    """img2 accumulates the SQUARE of every contribution: one record gives img2 == img^2 exactly, two
    records in one pixel give s1^2 + s2^2 (not (s1+s2)^2, not |s1|+|s2|, not s1+s2)."""
    m = box_model((6, 6, 6), 1.3, bvec=(0.2, 0.5, 0.8), mueller=hg_table(0.4), opac=const_opac(1.0, 0.2, 0.1, 0.5))
    o = [Observer.make(1.0, 0.7, [0.5, 0.5, 0.5], 0.9), Observer.make(2.2, 4.0, [0.5, 0.5, 0.5], 0.9)]
    r1 = ((2, 3, 1), [0.3, 0.6, 0.2], [0.6, 0.0, 0.8], [0.7, 0.21, -0.14, 0.35], 1)
    r2 = ((2, 3, 1), [0.3, 0.6, 0.2], [0.0, -0.6, 0.8], [0.4, -0.1, 0.2, -0.12], 2)     # same place, other state
    imgs = []
    for recs in ([r1], [r2], [r1, r2]):
        img, img2, st = m.image(_manual_events(m, recs), o, 8, 8, 0)
        assert st.contributions == 2 * len(recs) and st.dropped == 0
        imgs.append((img, img2))
    for img, img2 in imgs[:2]:
        assert np.count_nonzero(img[:, 0]) == 2                                # one pixel per observer
        assert np.all(img[:, 1:].reshape(2, 3, -1).any(axis=2))               # Q, U, V all exercised
        assert np.array_equal(img2, img * img)                                 # one record: exactly the square
    (i1, q1), (i2, q2), (i12, q12) = imgs
    assert np.allclose(i12, i1 + i2, rtol=1e-15, atol=0)
    assert np.allclose(q12, q1 + q2, rtol=1e-15, atol=0)                       # sum of squares ...
    nz = i12 != 0
    assert np.all(np.abs(q12[nz] - i12[nz] ** 2) > 1e-3 * q12[nz])             # ... which is not the square of the sum
    img, img2, _ = m.image(_manual_events(m, [r1]), o, 8, 8, 0, second_moment=False)
    assert img2 is None and np.array_equal(img, i1)


# ----------------------------------------------------------------------------
# the (U,V) block and the S34 terms of F(Theta), in the sampler and in the peel-off
# ----------------------------------------------------------------------------
def _F_printed(F):
    """F(Theta) as SURVEY.md 8(c) S5 prints it (spherical-form scattering matrix; reading R6 fixes the sign of S34)."""
    s11, s12, s33, s34 = F
    return np.array([[s11, s12, 0, 0], [s12, s11, 0, 0], [0, 0, s33, s34], [0, 0, -s34, s33]])


def test_circular_light_through_rayleigh_scattering():
    """Circular input has no linear part, so no frame rotation touches it: after one Rayleigh scattering
    V'/I' = S33/S11 = 2 cos(Theta)/(1 + cos^2 Theta), Q'/I' = -(1-cos^2)/(1+cos^2) in the scattering plane's
    reference, for any B and any azimuth -- in the sampler's chain and in the peel-off."""
    m = box_model()
    rng = np.random.default_rng(31)
    for hel in (1.0, -1.0):
        for _ in range(200):
            b, n_in = rand_unit(rng), rand_unit(rng)
            Theta = rng.uniform(2, 178); c = math.cos(math.radians(Theta))
            n_out, S = m.scatter_angles(b, n_in, [1, 0, 0, hel], Theta, rng.uniform(0, 2 * math.pi))
            assert abs(S[3] - hel * 2 * c / (1 + c * c)) < 2e-4 and S[0] == 1.0
            assert abs(math.hypot(S[1], S[2]) - (1 - c * c) / (1 + c * c)) < 2e-4
            n_obs = rand_unit(rng); mu = float(np.dot(n_in, n_obs))
            P = m.peel(n_in, [1, 0, 0, hel], n_obs)
            assert abs(P[3] / P[0] - hel * 2 * mu / (1 + mu * mu)) < 2e-4
            assert abs(P[0] * 4 * math.pi - 0.75 * (1 + mu * mu)) < 2e-4


def test_F_entry_by_entry_in_the_xz_plane():
    """A scattering inside the x-z plane with B = z^ (q_B = 1) and azimuth 0 needs no frame rotation at all:
    theta^ of n_in is e_par and theta^ of n_out is e_par,out.  The oracle's output must then be the printed
    F(Theta) times the input, entry by entry, on a table with S34 != 0 -- rows U and V included."""
    tab = hg_table(0.4)
    m = box_model(bvec=(0, 0, 1), mueller=tab)
    rng = np.random.default_rng(32)
    seen = np.zeros((4, 4), bool)
    for _ in range(200):
        a = math.radians(rng.uniform(5, 60)); Theta = float(rng.integers(10, 110))       # a table node: no interpolation
        n_in = np.array([math.sin(a), 0.0, math.cos(a)])
        S_in = np.r_[1.0, rand_unit(rng) * rng.uniform(0.2, 0.95)]
        F = _F_printed(tab[int(Theta)].astype(float))
        want = F @ S_in
        n_out, S = m.scatter_angles([0, 0, 1], n_in, S_in, Theta, 0.0)
        b = a + math.radians(Theta)
        assert np.allclose(n_out, [math.sin(b), 0, math.cos(b)], atol=1e-7)
        assert np.allclose(S, want / want[0], atol=1e-12)
        P = m.peel(n_in, S_in, [math.sin(b), 0.0, math.cos(b)])
        assert np.allclose(P * 4 * math.pi, want, atol=1e-6 * want[0])              # acos(mu) -> Theta: 1e-8 degrees off the node
        seen |= F != 0
    assert seen[2, 3] and seen[3, 2]
    # each entry alone: unit inputs (the rows of F read off one by one from differences)
    Theta = 70.0; F = _F_printed(tab[70].astype(float)); a = 0.4
    n_in = [math.sin(a), 0.0, math.cos(a)]; n_o = [math.sin(a + math.radians(Theta)), 0.0, math.cos(a + math.radians(Theta))]
    base = m.peel(n_in, [1, 0, 0, 0], n_o) * 4 * math.pi
    assert np.allclose(base, F[:, 0], atol=1e-6)
    for j in (1, 2, 3):
        e = np.zeros(4); e[0] = 1; e[j] = 0.5
        col = (m.peel(n_in, e, n_o) * 4 * math.pi - base) / 0.5
        assert np.allclose(col, F[:, j], atol=2e-6), (j, col, F[:, j])
    assert F[2, 3] == -F[3, 2] and F[2, 3] != 0


# ----------------------------------------------------------------------------
# S1 emission: the exact map from the Philox words, and isotropy
# ----------------------------------------------------------------------------
def test_emission_map_and_isotropy():
    """PAPER.md:107 (emission) with the schedule R11: block 0 of event 0 gives cos(theta) = 1 - 2 u0, phi = 2 pi u1,
    tau* = -ln u2.  Three ids exactly; then moments an isotropic direction must have (theta uniform instead of
    cos(theta) uniform gives <n_z^2> = 1/2, phi = pi u gives <n_y> > 0)."""
    m = box_model((4, 4, 4), 1.0)
    m.source_set(0, [0.3, 0.55, 0.8], [0, 0, 1], None, 0)
    seed = 77
    for pid in (0, 12345, 2 ** 35 + 9):
        w = _philox(seed, (pid & 0xFFFFFFFF, pid >> 32, 0, 0))
        u = [((int(x) >> 9) + 0.5) / 8388608.0 for x in w]
        ct = 1 - 2 * u[0]; st = math.sqrt(1 - ct * ct); ph = 2 * math.pi * u[1]
        idx, p, n, tau = m.emit(seed, pid)
        want = np.array([st * math.cos(ph), st * math.sin(ph), ct])
        assert np.array_equal(n, want.astype(np.float32).astype(float))           # fp32 direction (first-commit state)
        assert abs(tau + math.log(u[2])) < 1e-15
        assert list(idx) == [1, 2, 3]
        pw = np.array([0.3, 0.55, 0.8]) * 4 - np.array([1, 2, 3])
        assert np.allclose(p, pw, atol=1e-7 if FP32_STATE else 1e-15)
    N = 200000
    nn = np.array([m.emit(5, i)[2] for i in range(N)])
    assert np.all(np.abs(nn.mean(0)) < 5 * 0.577 / math.sqrt(N))                     # <n> = 0
    assert np.all(np.abs((nn * nn).mean(0) - 1 / 3) < 5 * 0.298 / math.sqrt(N))       # <n_i^2> = 1/3 (var 4/45)
    assert abs((nn[:, 0] * nn[:, 1]).mean()) < 5 * 0.26 / math.sqrt(N)
    h, _ = np.histogram(nn[:, 2], bins=20, range=(-1, 1))                            # cos(theta) uniform
    assert np.all(np.abs(h - N / 20) < 5 * math.sqrt(N / 20))
    h, _ = np.histogram(np.arctan2(nn[:, 1], nn[:, 0]), bins=24, range=(-math.pi, math.pi))     # phi uniform
    assert np.all(np.abs(h - N / 24) < 5 * math.sqrt(N / 24))
    # collimated source: the direction is the given one, tau* still from word 2
    m.source_set(2, [0.5, 0.5, 0.0], [0, 0.6, 0.8], None, 0)
    idx, p, n, tau = m.emit(seed, 3)
    assert np.allclose(n, [0, 0.6, 0.8], atol=1e-7)
    assert abs(tau + math.log(((int(_philox(seed, (3, 0, 0, 0))[2]) >> 9) + 0.5) / 8388608.0)) < 1e-15
