"""Pins of the oracle's statement of the paper's own two-step form (eq. 11)
and of the in-cell solution with source terms (App. A; thermal emission, NEXT-3).

Expected values: scipy.linalg.expm of the augmented system, the printed eq. 15, closed forms of the
segment integral derived in DESIGN.md section 12, scipy.integrate.quad of a numpy restatement, flux conservation,
and -- for the track-length deposit -- equality in expectation with the per-event estimator that is already pinned.
Nothing here calls the CUDA path.
"""
import math

import numpy as np
import scipy.integrate
import scipy.linalg

from oracle import lib, OracleModel, OracleEvents, OracleStats, Observer
from test_oracle_pins import Kmat, box_model, const_opac, hg_table, rand_unit, sph_basis

L = lib()


def _appA_src(S, a1, a2, a3, src, dtau):
    S = np.array(S, float)
    L.ora_appA_src(S, a1, a2, a3, np.array(src, float), dtau)
    return S


# ----------------------------------------------------------------------------
# App. A with source terms
# ----------------------------------------------------------------------------
def test_appA_with_sources_equals_augmented_matrix_exponential():
    """dS/dtau = -K S + src with K of reading R1: the solution over dtau is the top block of expm([[-K, src],[0, 0]] dtau)."""
    rng = np.random.default_rng(41)
    for _ in range(200):
        a1 = rng.uniform(0.5, 2.0); a2 = rng.uniform(-0.9, 0.9) * a1; a3 = rng.uniform(-1.5, 1.5)
        src = rng.normal(size=4); S0 = rng.normal(size=4); dtau = math.exp(rng.uniform(math.log(1e-4), math.log(8.0)))
        M = np.zeros((5, 5)); M[:4, :4] = -Kmat(a1, a2, a3); M[:4, 4] = src
        want = (scipy.linalg.expm(M * dtau) @ np.r_[S0, 1.0])[:4]
        got = _appA_src(S0, a1, a2, a3, src, dtau)
        assert np.allclose(got, want, rtol=1e-10, atol=1e-12 * np.abs(want).max())
    # no source: the source-free solution; thick cell: the stationary vector of eq. A3, K S_s = src
    S = _appA_src([1, .3, -.2, .1], 1.0, 0.4, 0.2, [0, 0, 0, 0], 0.7)
    S2 = np.array([1, .3, -.2, .1]); L.ora_appA(S2, 1.0, 0.4, 0.2, 0.7)
    assert np.array_equal(S, S2)
    src = np.array([0.7, -0.2, 0.4, 0.1])
    Ss = _appA_src([5, 1, 2, 3], 1.0, 0.4, 0.2, src, 1e3)
    assert np.allclose(Kmat(1.0, 0.4, 0.2) @ Ss, src, atol=1e-13)


def test_printed_solution_with_sources():
    """PAPER.md:302-328 typed in as printed (A2 with the auxiliary quantities A3)."""
    rng = np.random.default_rng(42)
    for _ in range(50):
        a1, a2, a3, dt = rng.uniform(0.5, 2), rng.uniform(-0.4, 0.4), rng.uniform(-1, 1), rng.uniform(0.01, 5)
        I0, Q0, U0, V0 = rng.normal(size=4); S1, S2, S3, S4 = rng.normal(size=4)
        Is = (a1 * S1 - a2 * S2) / (a1 ** 2 - a2 ** 2); Qs = (a1 * S2 - a2 * S1) / (a1 ** 2 - a2 ** 2)
        Us = (a1 * S3 - a3 * S4) / (a1 ** 2 + a3 ** 2); Vs = (a1 * S4 + a3 * S3) / (a1 ** 2 + a3 ** 2)
        e = math.exp(-a1 * dt)
        I = Is + (I0 - Is) * e * math.cosh(-a2 * dt) + (Q0 - Qs) * e * math.sinh(-a2 * dt)
        Q = Qs + (I0 - Is) * e * math.sinh(-a2 * dt) + (Q0 - Qs) * e * math.cosh(-a2 * dt)
        U = Us + (U0 - Us) * e * math.cos(-a3 * dt) + (V0 - Vs) * e * math.sin(-a3 * dt)
        V = Vs - (U0 - Us) * e * math.sin(-a3 * dt) + (V0 - Vs) * e * math.cos(-a3 * dt)
        got = _appA_src([I0, Q0, U0, V0], a1, a2, a3, [S1, S2, S3, S4], dt)
        assert np.allclose(got, [I, Q, U, V], rtol=1e-12, atol=1e-13)


def _slab_model(n, tau_total, a1, a2, om, bvec):
    """n x 1 x 1 cells along x, total kappa*rho*length = tau_total, uniform field bvec."""
    opac = const_opac(a1, a2, 0.0, om)
    return box_model((n, 1, 1), tau_total, bvec=bvec, opac=opac, bounds=(0, 1, 0, 1, 0, 1))


def test_eq15_thermal_emission_of_an_aligned_slab():
    """PAPER.md:198 eq. 15: uniform isothermal aligned slab without scattering, P = e^{-tau} sinh(p0 tau) / (1 - e^{-tau} cosh(p0 tau))
    with tau = alpha1 x (extinction depth) and p0 = alpha2/alpha1 -- through the pixel-ray march (App. A with the thermal source
    (1 - omega)(alpha1, alpha2, 0, 0) B in every cell), for one cell and for many, up to tau = 30."""
    a1, a2 = 1.0, float(np.float32(0.12))                           # tables and densities reach the oracle as fp32
    p0 = a2 / a1
    for tau in (0.01, 0.3, 1.0, 3.0, 10.0, 30.0):
        tau = float(np.float32(tau))
        for n in (1, 7, 64):
            m = _slab_model(n, tau, a1, a2, 0.0, (0, 0, 1))               # B along z, line of sight along +x: vartheta = 90 deg
            o = Observer.make(math.pi / 2, 0.0, [0.5, 0.5, 0.5], 0.5)
            img, st = m.image_rays(None, [o], 1, 1, emis=np.full(n, 2.5, np.float32))
            I, Q, U, V = img[0, :, 0, 0]
            P = math.exp(-tau) * math.sinh(p0 * tau) / (1 - math.exp(-tau) * math.cosh(p0 * tau))
            assert abs(I - 2.5 * (1 - math.exp(-tau) * math.cosh(p0 * tau))) < 1e-12 * 2.5      # pixel area 1
            # theta^_obs of the +x view is -z, i.e. along B: the grain frame's +Q (E in the n-B plane, R8) is the image's +Q
            assert abs(Q / I - P) < 1e-11 and abs(U) < 1e-14 and abs(V) < 1e-14
            assert st.steps_image == n
    # albedo: only the absorbed fraction emits (alpha_abs = (1 - omega) alpha, reading R19)
    m = _slab_model(5, 2.0, a1, a2, 0.75, (0, 0, 1))
    o = Observer.make(math.pi / 2, 0.0, [0.5, 0.5, 0.5], 0.5)
    img, _ = m.image_rays(None, [o], 1, 1, emis=np.ones(5, np.float32))
    assert abs(img[0, 0, 0, 0] - 0.25 * (1 - math.exp(-2.0) * math.cosh(p0 * 2.0))) < 1e-12


# ----------------------------------------------------------------------------
# step 1: the segment integral J = int_0^T r s^ dtau and the deposit
# ----------------------------------------------------------------------------
def _J(Sg, a1, a2, a3, T):
    J = np.zeros(4)
    L.ora_segment_integral(np.array(Sg, float), a1, a2, a3, T, J)
    return J


def test_segment_integral_closed_forms_and_quadrature():
    """With q0 the grain-frame Q/I at the start and g(T) = cosh(a2 T) - q0 sinh(a2 T) (so that I~(T) = e^{-a1 T} g(T)):
      J_I  = int r dtau       = -ln I~(T)                       = a1 T - ln g(T)
      J_Q  = int r q^ dtau    = q^(T) - q0 + a2 T + a1 int q^   , int_0^T q^ dtau = -ln g(T) / a2
    (from r s^ = s^' + K s^); U and V against scipy.integrate.quad of expm(-K tau) s0, normalised."""
    rng = np.random.default_rng(43)
    for _ in range(120):
        a1 = rng.uniform(0.5, 2.0); a2 = rng.uniform(-0.8, 0.8) * a1; a3 = rng.uniform(-1.5, 1.5)
        T = math.exp(rng.uniform(math.log(1e-3), math.log(12.0)))
        pol = rand_unit(rng) * rng.uniform(0, 0.95); scale = rng.uniform(0.1, 3.0)          # any normalisation of the state
        S0 = scale * np.r_[1.0, pol]
        J = _J(S0, a1, a2, a3, T)
        q0 = pol[0]
        g = math.cosh(a2 * T) - q0 * math.sinh(a2 * T)
        assert abs(J[0] - (a1 * T - math.log(g))) < 1e-12 * max(1.0, a1 * T)
        qT = (q0 * math.cosh(a2 * T) - math.sinh(a2 * T)) / g
        if abs(a2) > 1e-3:
            want_q = qT - q0 + a2 * T + a1 * (-math.log(g) / a2)
            assert abs(J[1] - want_q) < 1e-11 * max(1.0, a1 * T)
        K = Kmat(a1, a2, a3)

        def f(tau, k):
            s = scipy.linalg.expm(-K * tau) @ np.r_[1.0, pol]
            return (a1 + a2 * s[1] / s[0]) * s[k] / s[0]
        for k in (2, 3):
            want, _ = scipy.integrate.quad(f, 0, T, args=(k,), epsabs=1e-12, epsrel=1e-12, limit=200)
            assert abs(J[k] - want) < 2e-10 * max(1.0, a1 * T)
    # scalar medium: the state does not change, J = a1 T s^
    assert np.allclose(_J([2, 0.4, -0.6, 0.2], 1.5, 0, 0, 0.8), 1.5 * 0.8 * np.array([1, 0.2, -0.3, 0.1]), rtol=1e-14)
    assert np.all(_J([1, 0, 0, 0], 1, 0.2, 0.1, 0.0) == 0)


def _events_by_cell(ev, ncell):
    n = ev.n
    w = ev.S[:n, 0]
    return np.bincount(ev.cell[:n], weights=w, minlength=ncell)


def test_deposit_equals_the_event_estimator_in_expectation():
    """The track-length deposit and the scattering events estimate the same collision density: per block of cells the
    expected number of collisions (coll, weight W before the albedo) against the weights of the events that did happen
    (omega W stored, so divided by omega), and the summed, unattenuated output toward two cameras against the summed
    peel-off of the events -- same packets, so the noise of the difference is that of the collision estimator alone."""
    om = 0.7
    n = 12
    rng = np.random.default_rng(44)
    dens = (3.0 * np.exp(0.5 * rng.normal(size=(n, n, n)))).astype(np.float32)
    mu = np.linspace(0, 1, 5)
    opac = np.stack([1 + 0.3 * (1 - mu * mu), 0.3 * (1 - mu * mu), 0.2 * (1 - mu * mu), np.full(5, om)], 1).astype(np.float32)
    bf = np.broadcast_to(np.array([0.6, 0.0, 0.8], np.float32), (n, n, n, 3)).copy()
    m = OracleModel(n, n, n, [0, 1, 0, 1, 0, 1], dens, bf, hg_table(0.4), opac)
    m.source_set(0, [0.5, 0.5, 0.5], [0, 0, 1], None, 0)
    obs = [Observer.make(1.0, 0.5, [0.5, 0.5, 0.5], 0.9), Observer.make(2.4, 3.0, [0.5, 0.5, 0.5], 0.9)]
    N, nb = 24000, 8
    tot_dep = np.zeros((nb, 2, 4)); tot_ev = np.zeros((nb, 2, 4)); coll = np.zeros(n ** 3); evw = np.zeros(n ** 3)
    for b in range(nb):                                                       # batches: for the noise estimate
        ev = OracleEvents(40 * N // nb); st = OracleStats()
        sg, cl, nseg = m.transport_deposit(b * (N // nb), N // nb, 9, ev, obs, stats=st, collisions=True)
        assert nseg == st.steps_transport                                     # one deposit per cell step with kappa rho > 0
        tot_dep[b] = sg.sum(0)
        k = ev.n
        for e in range(k):
            for o, ob in enumerate(obs):
                no = [math.sin(ob.theta) * math.cos(ob.phi), math.sin(ob.theta) * math.sin(ob.phi), math.cos(ob.theta)]
                tot_ev[b, o] += m.peel(ev.n_in[e], ev.S[e], no)
        coll += cl; evw += _events_by_cell(ev, n ** 3) / float(np.float32(om))
    # (1) collision density in 3^3 blocks of 4^3 cells
    blk = lambda a: a.reshape(3, 4, 3, 4, 3, 4).sum(axis=(1, 3, 5)).ravel()
    cb, eb = blk(coll), blk(evw)
    assert abs(coll.sum() / evw.sum() - 1) < 0.01
    assert np.all(np.abs(cb - eb) < 5 * np.sqrt(eb) + 5)                       # Poisson-like noise of the event counts
    # (2) polarised output toward the cameras, summed over the grid
    d = tot_dep - tot_ev
    mean, err = d.mean(0), d.std(0, ddof=1) / math.sqrt(nb)
    ref = tot_ev.mean(0)[:, :1]
    assert np.all(np.abs(mean) < 4.5 * err + 2e-4 * ref), (mean, err)
    assert np.all(err[:, 0] < 0.02 * ref[:, 0])                                # and the test has the power to see 2 %
    assert np.abs(tot_dep.mean(0)[:, 1:3]).max() > 10 * err[:, 1:3].max()             # a polarised signal, resolved above the noise


# ----------------------------------------------------------------------------
# step 2: one ray per pixel
# ----------------------------------------------------------------------------
def test_pixel_rays_conserve_the_deposited_flux():
    """A source grid written by hand, almost no extinction: the image summed over fine pixels returns the deposited
    totals (checks the 1/V_cell, the pixel area and the source per extinction depth), from any direction; with extinction
    the emission of one cell seen along an axis is attenuated by the closed form (1 - e^{-t})/t e^{-tau_front}."""
    n = 6
    kr = 1e-6
    m = box_model((n, n, n), kr, opac=const_opac(1.0, 0.0, 0.0, 0.5))
    rng = np.random.default_rng(45)
    obs = [Observer.make(0.0, 0.0, [0.5, 0.5, 0.5], 0.9), Observer.make(1.1, 0.7, [0.5, 0.5, 0.5], 0.9),
           Observer.make(math.pi / 2, math.pi / 2, [0.5, 0.5, 0.5], 0.9)]
    sg = np.zeros((n ** 3, 3, 4))
    cells = rng.integers(0, n ** 3, 5)
    for c in cells:
        sg[c] = rng.normal(size=(3, 4))
    img, st = m.image_rays(sg, obs, 240, 240)
    # pixel centres sample the projected cell: an oblique view averages the cell's outline over many pixel rows (1e-4 here), an
    # axis-aligned view counts whole pixel rows per cell edge (1 in 22 pixels per cell)
    tot = img.sum(axis=(2, 3))
    assert np.allclose(tot[1], sg.sum(0)[1], rtol=2e-4, atol=2e-4)
    assert np.allclose(tot, sg.sum(0), rtol=0.1, atol=0.1)
    # axis-aligned view, pixels that divide the cells exactly: exact
    img, _ = m.image_rays(sg[:, :1], obs[:1], 6 * 9, 6 * 9)                        # 0.9/27 per pixel: not commensurate ...
    o = Observer.make(0.0, 0.0, [0.5, 0.5, 0.5], 0.5)
    img, _ = m.image_rays(sg[:, :1].copy(), [o], 12, 12)                              # ... this one is: 2 x 2 pixels per cell
    assert np.allclose(img.sum(axis=(2, 3)), sg[:, 0].sum(0), rtol=1e-5)
    # optically thick: the +z view of a uniformly emitting column
    kr = 4.0
    m = box_model((1, 1, 5), kr, opac=const_opac(1.0, 0.0, 0.0, 0.5))
    sg = np.zeros((5, 1, 4)); sg[1, 0, 0] = 3.0                                       # second cell from the bottom emits
    o = Observer.make(0.0, 0.0, [0.5, 0.5, 0.5], 0.5)
    img, _ = m.image_rays(sg, [o], 1, 1)
    t = kr * 0.2
    want = 3.0 / (1 * 1 * 0.2) / kr * (1 - math.exp(-t)) * math.exp(-3 * t) * 1.0     # src (1 - e^-t), three cells in front, area 1
    assert abs(img[0, 0, 0, 0] - want) < 1e-6 * want          # kappa rho is fp32
    o = Observer.make(math.pi, 0.0, [0.5, 0.5, 0.5], 0.5)                              # from below: one cell in front
    img, _ = m.image_rays(sg, [o], 1, 1)
    assert abs(img[0, 0, 0, 0] - 3.0 / 0.2 / kr * (1 - math.exp(-t)) * math.exp(-1 * t)) < 1e-6 * want * 100
    # a ray that misses the box gives nothing
    o = Observer.make(0.3, 0.2, [5.0, 5.0, 0.5], 0.2)
    img, st = m.image_rays(sg, [o], 4, 4)
    assert not img.any()


def test_two_step_image_equals_event_image_in_expectation():
    """The paper's form (deposit on every segment, one ray per pixel with source terms) against the per-event form on a
    16^3 grid of optically thin cells (the grid form spreads a cell's collisions evenly over the cell and samples the
    pixel centre, which differs from the per-event attenuation at second order in the cell's depth): image-integrated
    I, Q, U, V per observer within the noise of the collision estimator plus 1.5 %, and coarse 4 x 4 maps of I."""
    n = 16
    c = (np.arange(n) + 0.5) / n - 0.5
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    dens = (6.0 * np.exp(-(X * X + Y * Y + Z * Z) / (2 * 0.25 ** 2))).astype(np.float32)       # tau ~ 1.9 centre to edge, <= 0.38 per cell
    mu = np.linspace(0, 1, 5)
    opac = np.stack([1 + 0.2 * (1 - mu * mu), 0.2 * (1 - mu * mu), 0.1 * (1 - mu * mu), np.full(5, 0.8)], 1).astype(np.float32)
    bf = np.broadcast_to(np.array([0.0, 0.6, 0.8], np.float32), (n, n, n, 3)).copy()
    m = OracleModel(n, n, n, [-.5, .5, -.5, .5, -.5, .5], dens, bf, hg_table(0.3), opac)
    m.source_set(0, [0.02, -0.03, 0.01], [0, 0, 1], None, 0)
    # the axis-aligned view frames the grid exactly (4 x 4 pixel rays per cell: no aliasing of pixel centres against cell edges)
    obs = [Observer.make(1.0, 0.5, [0, 0, 0], 0.9), Observer.make(math.pi / 2, 0.0, [0, 0, 0], 0.5)]
    N, nb, npix = 32000, 8, 64
    tot_g = np.zeros((nb, 2, 4)); tot_e = np.zeros((nb, 2, 4)); map_g = 0; map_e = 0
    for b in range(nb):
        ev = OracleEvents(40 * N // nb); st = OracleStats()
        sg, _, _ = m.transport_deposit(b * (N // nb), N // nb, 3, ev, obs, stats=st)
        ig, _ = m.image_rays(sg, obs, npix, npix)
        ie, _, _ = m.image(ev, obs, npix, npix, second_moment=False)
        tot_g[b] = ig.sum(axis=(2, 3)); tot_e[b] = ie.sum(axis=(2, 3))
        map_g = map_g + ig[:, 0].reshape(2, 4, 16, 4, 16).sum(axis=(2, 4)); map_e = map_e + ie[:, 0].reshape(2, 4, 16, 4, 16).sum(axis=(2, 4))
    d = tot_g - tot_e
    mean, err = d.mean(0), d.std(0, ddof=1) / math.sqrt(nb)
    ref = tot_e.mean(0)[:, :1]
    assert np.all(np.abs(mean) < 4.5 * err + 0.015 * ref), (mean / ref, err / ref)
    assert np.all(err < 0.02 * ref)
    assert np.abs(tot_g.mean(0)[:, 1:3]).max() > 0.05 * ref[:, 0].max()                        # a polarised case
    assert np.all(np.abs(map_g - map_e) < 0.06 * map_e + 0.01 * map_e.max())


# ----------------------------------------------------------------------------
# NEXT-3: periodic boundaries, reading R20
# ----------------------------------------------------------------------------
def test_periodic_box_is_an_infinite_slab():
    """Periodic in x and y, open in z: an isotropic point source in the mid-plane of a uniform pure absorber of half
    depth tau escapes with probability int_0^1 e^{-tau/mu} dmu = E_2(tau) (scipy.special.expn); the open box loses
    packets through its sides and gives more.  A source moved by a fraction of the box gives the same events up to the shift."""
    import scipy.special
    tau, N = 1.5, 100000
    m = box_model((8, 8, 8), 2 * tau, opac=const_opac(1, 0, 0, 0.0))      # kappa rho = 2 tau per unit length, half height 1/2
    m.source_set(0, [0.5, 0.5, 0.5], [0, 0, 1], None, 0)
    ev = OracleEvents(2 * N)
    st_open, _ = m.transport(0, N, 6, ev)
    m.set_periodic(3)
    ev = OracleEvents(2 * N)
    st_per, _ = m.transport(0, N, 6, ev)
    want = float(scipy.special.expn(2, tau))
    assert abs(st_per.w_escaped / N - want) < 4 * math.sqrt(want * (1 - want) / N)
    assert st_open.w_escaped / N > want + 0.05
    # translation by (3/8, -2/8, 0) of the source in the periodic box: same packets, same depths, cells shifted modulo the box
    m.source_set(0, [0.5 + 3 / 8, 0.5 - 2 / 8, 0.5], [0, 0, 1], None, 0)
    ev2 = OracleEvents(2 * N)
    st2, _ = m.transport(0, N, 6, ev2)
    assert ev2.n == ev.n and st2.w_escaped == st_per.w_escaped and st2.steps_transport == st_per.steps_transport
    c1, c2 = ev.cell[:ev.n], ev2.cell[:ev.n]
    x1, y1, z1 = c1 % 8, (c1 // 8) % 8, c1 // 64
    assert np.array_equal((x1 + 3) % 8, c2 % 8) and np.array_equal((y1 - 2) % 8, (c2 // 8) % 8) and np.array_equal(z1, c2 // 64)
    assert np.allclose(ev.p[:ev.n], ev2.p[:ev.n], atol=1e-6)


def test_periodic_march_wraps_and_ends_at_the_open_faces():
    """An oblique ray in a box periodic in x only: the logged cells wrap in x, the segments add up to the chord to the
    nearest open face (y or z), the optical depth is kappa rho times that chord; fully periodic and parallel to every open
    face it ends after ORA_MAX_WRAPS crossings."""
    kr = float(np.float32(0.7))                                              # densities reach the oracle as fp32
    m = box_model((5, 4, 6), kr, opac=const_opac(1, 0, 0, 0.5), bounds=(0, 5, 0, 4, 0, 6))
    m.set_periodic(1)
    n = np.array([0.9, 0.1, 0.42]); n /= np.linalg.norm(n)
    S, steps, cells, ds = m.march([1, 1, 0], [0.3, 0.4, 0.0], n, [1, 0, 0, 0], log_cap=400)
    chord = min((4 - 1.4) / n[1], 6.0 / n[2])
    assert abs(ds.sum() - chord) < 1e-12 and abs(S[0] - math.exp(-kr * chord)) < 1e-15
    xs = cells % 5
    assert steps == len(cells) and np.all(np.diff(xs) % 5 <= 1) and (np.diff(xs) == -4).sum() == int((1.3 + n[0] * chord) // 5)
    m.set_periodic(0)
    S0, steps0, _, ds0 = m.march([1, 1, 0], [0.3, 0.4, 0.0], n, [1, 0, 0, 0], log_cap=400)
    assert abs(ds0.sum() - (5 - 1.3) / n[0]) < 1e-12                       # open box: leaves through the x face first
    m.set_periodic(7)
    S, steps, cells, ds = m.march([1, 1, 0], [0.3, 0.4, 0.5], [1.0, 0.0, 0.0], [1, 0, 0, 0], log_cap=10)
    assert steps == 4 + 4096 * 5                                            # 4 cells to the face, 4096 wraps of 5 cells, the next wrap refused
    # imaging ray of one emission record through the periodic box: W/(4 pi) e^{-tau of the wrapped path}
    m.set_periodic(1)
    m.source_set(0, [1.3, 1.4, 0.0], [0, 0, 1], None, 1)
    ev = OracleEvents(4)
    m.transport(0, 1, 1, ev); ev.c.n = 1
    th, ph = math.acos(n[2]), math.atan2(n[1], n[0])
    img, _, st = m.image(ev, [Observer.make(th, ph, [2.5, 2, 3], 30.0)], 1, 1, 1)
    assert abs(img[0, 0, 0, 0] - math.exp(-kr * chord) / (4 * math.pi)) < 1e-15


def test_pixel_rays_in_a_periodic_slab():
    """Thermal emission of a uniform slab periodic in x and y, seen at inclination mu: every pixel ray crosses the same depth
    tau/mu wherever it enters, so every pixel holds B (1 - e^{-tau/mu}) times its area -- also pixels whose line misses the
    box of one period; open in x and y the oblique rays are cut short."""
    tau = 0.8
    m = box_model((6, 6, 3), tau, opac=const_opac(1, 0, 0, 0.0), bounds=(0, 2, 0, 2, 0, 1))
    o = Observer.make(math.radians(50), math.radians(20), [1, 1, 0.5], 3.0)
    mu = math.cos(math.radians(50))
    emis = np.full((3, 6, 6), 1.7, np.float32)
    m.set_periodic(3)
    img, st = m.image_rays(None, [o], 8, 8, emis=emis)
    apix = (6.0 / 8) ** 2
    assert np.allclose(img[0, 0], float(np.float32(1.7)) * (1 - math.exp(-float(np.float32(tau)) / mu)) * apix, rtol=1e-12)
    m.set_periodic(0)
    img0, _ = m.image_rays(None, [o], 8, 8, emis=emis)
    assert (img0[0, 0] == 0).sum() > 20 and img0[0, 0].max() < img[0, 0].max() * (1 + 1e-12)


# ----------------------------------------------------------------------------
# NEXT-3: thermal emission of aligned grains as the packet source of the Monte-Carlo step (reading R22)
# ----------------------------------------------------------------------------
def _aligned_table(n_inc=9, R=1.6, c3=0.1, om=0.3):
    mu = np.linspace(0, 1, n_inc); s2 = 1 - mu * mu
    return np.stack([1 + 0.5 * (R - 1) * s2, 0.5 * (R - 1) * s2, c3 * s2, om + 0.2 * mu], 1).astype(np.float32)


def test_thermal_packets_follow_the_emissivity():
    """kind = 5 (volume source, thermal): directions are distributed as (1 - omega(mu)) alpha1(mu), mu = |n . B^|, and the
    packet carries (1, alpha2/alpha1, 0, 0) in the grain-frame reference: rotated back there (eq. 6-7) Q/I = alpha2/alpha1 at
    the packet's own mu, U = V = 0.  Draws replayed from the Philox words for the first candidates."""
    from test_oracle_pins import _philox
    tab = _aligned_table()
    b = np.array([0.48, -0.6, 0.64], np.float32).astype(float)
    m = box_model((3, 3, 3), 1.0, bvec=b, opac=tab)
    m.source_set(5, [0, 0, 0], [0, 0, 1], None, 0)
    mu_n = np.linspace(0, 1, 9)
    emis = (1 - tab[:, 3].astype(float)) * tab[:, 0].astype(float)
    emax = emis.max()
    N = 60000
    mus = np.zeros(N); first = 0
    q4 = np.zeros(4); L.ora_quat_from_B(b, q4)
    import ctypes as C
    for pid in range(N):
        idx, p, n, tau, S = m.emit_full(11, pid)
        mu = abs(float(np.dot(n, b))) / np.linalg.norm(n) / np.linalg.norm(b)
        mus[pid] = mu
        if pid < 2000:
            a = m.opac_at(mu)
            ce, se = C.c_double(), C.c_double(); L.ora_eta_gf(q4, n, C.byref(ce), C.byref(se))
            Sg = S.copy(); L.ora_rotate_qu(Sg, ce.value, se.value)
            assert abs(Sg[1] - a[1] / a[0]) < 2e-7 and abs(Sg[2]) < 2e-7 and Sg[3] == 0 and S[0] == 1      # fp32 (q,u,v) state (R12)
            # the first candidate (block 0: cos theta, phi, -, accept = word 3) is taken exactly when its test passes
            w = _philox(11, (pid, 0, 0, 0)); u = [((int(x) >> 9) + 0.5) / 8388608.0 for x in w]
            ct = 1 - 2 * u[0]; st = math.sqrt(1 - ct * ct); ph = 2 * math.pi * u[1]
            n0 = np.array([st * math.cos(ph), st * math.sin(ph), ct]).astype(np.float32).astype(float)
            a0 = m.opac_at(abs(float(np.dot(n0, b))) / np.linalg.norm(n0) / np.linalg.norm(b))
            took_first = np.array_equal(n, n0)
            assert took_first == (u[3] * emax < (1 - a0[3]) * a0[0])
            first += took_first
            assert abs(tau + math.log(u[2])) < 1e-15
    assert 0.5 * 2000 < first < 2000                                       # rejections happen
    h, edges = np.histogram(mus, bins=8, range=(0, 1))
    # isotropic candidates are uniform in mu; accepted density ~ emissivity(mu), piecewise linear on the nodes
    fine = np.linspace(0, 1, 8001); dens = np.interp(fine, mu_n, emis)
    want = np.array([dens[(fine >= a_) & (fine < b_)].sum() for a_, b_ in zip(edges[:-1], edges[1:])]); want /= want.sum()
    assert np.all(np.abs(h / N - want) < 5 * np.sqrt(want / N)), (h / N, want)


def test_thermal_packets_and_thermal_rays_agree():
    """The two halves of NEXT-3 describe the same radiation: in an optically thin, non-scattering aligned cube the packets that
    leave toward a direction (naive cone estimator) carry, per steradian, L_tot/N times their count, with
    L_tot = 4 pi <(1 - omega) alpha1>_mu sum(kappa rho B V); the ray step's image toward that direction integrates to the same
    radiant intensity, with the same Q/I = alpha2/alpha1 in the reference theta^_obs."""
    tab = _aligned_table(om=0.0); tab[:, 3] = 0.0                                   # pure absorber / emitter
    b = np.array([0.0, 0.0, 1.0])
    kr, Bv, n = 0.02, 1.7, 4
    m = box_model((n, n, n), kr, bvec=b, opac=tab, bounds=(-.5, .5, -.5, .5, -.5, .5))
    m.source_set(5, [0, 0, 0], [0, 0, 1], None, 0)
    N = 400000
    ev = OracleEvents(4 * N)
    st, esc = m.transport(0, N, 3, ev, esc_cap=N)
    mu_n = np.linspace(0, 1, 9)
    mean_emis = np.trapezoid(tab[:, 0].astype(float), mu_n)
    L_tot = 4 * math.pi * mean_emis * float(np.float32(kr)) * Bv * 1.0
    for th_deg in (90.0, 50.0):
        th = math.radians(th_deg); no = np.array([math.sin(th), 0.0, math.cos(th)])
        half = math.radians(15.0); dom = 2 * math.pi * (1 - math.cos(half))
        sel = esc["n"] @ no > math.cos(half)
        naive = esc["S"][sel].sum(0) / dom * L_tot / N                               # radiant intensity, lab reference of each packet
        o = Observer.make(th, 0.0, [0, 0, 0], 0.9)
        img, _ = m.image_rays(None, [o], 96, 96, emis=np.full(n ** 3, Bv, np.float32))
        tot = img[0].sum(axis=(1, 2))
        cnt = sel.sum()
        assert cnt > 5000
        assert abs(naive[0] / tot[0] - 1) < 4 / math.sqrt(cnt) + 0.02               # cone average of a smooth pattern, thin-limit e^{-tau}
        # polarisation: B along z, observer in the x-z plane: the grain frame's +Q (E in the n-B plane) is +Q of theta^_obs
        a = m.opac_at(abs(no[2]))
        assert abs(tot[1] / tot[0] - a[1] / a[0]) < 5e-3 and abs(tot[2]) < 1e-12 * tot[0]      # thin limit: O(tau = 0.02) self-absorption
        # packets inside the cone: their Q in their own lab reference is the same grain-frame Q (B = z: theta^' = theta^)
        assert abs(naive[1] / naive[0] - a[1] / a[0]) < 0.03
