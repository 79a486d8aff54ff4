"""Pins of the oracle's full aligned-grain scattering matrix Z(Omega; Omega') path (PAPER.md:103-109,
:129; reading R21): interpolation, reduction to the pinned F(Theta) path for isotropic dipoles, conservation of the scattered
flux, the rejection sampler against the table's own density.  Nothing here calls the CUDA path."""
import math

import numpy as np

from oracle import lib, OracleZTable
from paper_2512_01283_b200 import inputs
from test_oracle_pins import box_model, rand_unit, sph_basis, stokes_of_E, _philox, Ry, Rz

L = lib()


def test_ztable_interpolation():
    rng = np.random.default_rng(51)
    Z = rng.normal(size=(7, 5, 8, 4, 4)).astype(np.float32)
    zt = OracleZTable(Z)
    for _ in range(50):
        i, o, d = rng.integers(0, 7), rng.integers(0, 5), rng.integers(0, 8)
        assert np.array_equal(zt.at(i * 30.0, o * 45.0, d * 45.0), Z[i, o, d].astype(float))          # nodes
        assert np.allclose(zt.at(i * 30.0, o * 45.0, d * 45.0 - 720.0), Z[i, o, d], atol=1e-12)       # periodic in dphi
    a = zt.at(47.0, 100.0, 350.0)                                                                      # trilinear, wrapping d = 7 -> 0
    wi, wo, wd = 47 / 30 - 1, 100 / 45 - 2, 350 / 45 - 7
    want = 0
    for A, wa in ((1, 1 - wi), (2, wi)):
        for B, wb in ((2, 1 - wo), (3, wo)):
            for Cc, wc in ((7, 1 - wd), (0, wd)):
                want = want + wa * wb * wc * Z[A, B, Cc].astype(float)
    assert np.allclose(a, want, atol=1e-12)


def test_isotropic_dipole_reduces_to_the_rayleigh_path():
    """a_par = a_perp: Z is the Rayleigh matrix between meridional references, so the peel-off through Z must equal the
    pinned peel-off through F(Theta) for any field direction, and the phase function needs no normalisation (N = 1)."""
    zt = OracleZTable(inputs.dipole_ztable(73, 73, 144))                     # 2.5-degree nodes
    m = box_model()                                                          # Rayleigh F table, 1-degree nodes
    rng = np.random.default_rng(52)
    worst = 0.0
    for _ in range(300):
        b, n_in, n_obs = rand_unit(rng), rand_unit(rng), rand_unit(rng)
        S_in = 0.8 * np.r_[1.0, rand_unit(rng) * rng.uniform(0, 0.9)]
        a = zt.peel(b, n_in, S_in, n_obs)
        w = m.peel(n_in, S_in, n_obs)
        worst = max(worst, np.abs(a - w).max() / w[0])
    assert worst < 1e-2, worst            # trilinear interpolation on 2.5-degree nodes (largest near the poles, where the meridional reference turns with dphi)
    for ti in (0.0, 33.0, 90.0, 161.0):
        assert abs(zt.norm(ti, [1, 0, 0, 0]) - 1) < 2e-3 and abs(zt.norm(ti, [0, 1, 0, 0])) < 2e-3
        assert abs(zt.norm(ti, [0, 0, 1, 0])) < 1e-6 and abs(zt.norm(ti, [0, 0, 0, 1])) < 1e-6


def _sphere_quadrature(n_mu=48, n_phi=96):
    x, w = np.polynomial.legendre.leggauss(n_mu)
    ph = (np.arange(n_phi) + 0.5) * 2 * math.pi / n_phi
    dirs, wts = [], []
    for mu, wm in zip(x, w):
        s = math.sqrt(1 - mu * mu)
        for p in ph:
            dirs.append([s * math.cos(p), s * math.sin(p), mu]); wts.append(wm * 2 * math.pi / n_phi)
    return np.array(dirs), np.array(wts)


def test_scattered_flux_is_conserved():
    """The peel-off is the phase function times the event's weight: integrated over all observer directions its I component
    returns the weight, for an anisotropic absorbing dipole and polarised input (this pins the normalisation N)."""
    zt = OracleZTable(inputs.dipole_ztable(37, 37, 72, a_par=0.6 + 0.2j, a_perp=1.0 + 0.05j))
    dirs, wts = _sphere_quadrature()
    rng = np.random.default_rng(53)
    for _ in range(6):
        b, n_in = rand_unit(rng), rand_unit(rng)
        S_in = 0.37 * np.r_[1.0, rand_unit(rng) * rng.uniform(0.2, 0.9)]
        tot = sum(wt * zt.peel(b, n_in, S_in, d)[0] for d, wt in zip(dirs, wts))
        assert abs(tot / S_in[0] - 1) < 6e-3, tot / S_in[0]


def test_rejection_sampler_follows_the_table():
    """Outgoing directions of ora_scatter_z are distributed as row 1 of Z . s: the draws are replayed from the Philox words
    (schedule R11 / R21), and the sampled density is compared with the table's in bins of the grain frame's polar angle."""
    Zt = inputs.dipole_ztable(37, 37, 72, a_par=0.5 + 0.1j, a_perp=1.0)
    zt = OracleZTable(Zt)
    b = np.array([0.0, 0.0, 1.0])                                           # grain frame = lab frame: q_B = 1
    n_in = np.array([math.sin(0.7), 0.0, math.cos(0.7)]).astype(np.float32).astype(float)
    S_in = np.array([1.0, 0.5, -0.3, 0.2])
    ti = math.degrees(math.acos(n_in[2] / np.linalg.norm(n_in)))
    N = 40000
    ct = np.zeros(N); rounds = np.zeros(N, int)
    for pid in range(N):
        n_out, S_out, tau, r = zt.scatter(b, n_in, S_in, 77, pid, 3)
        ct[pid] = n_out[2]; rounds[pid] = r
        if pid < 300:                                                       # replay: candidates from the documented words
            for blk in range(r):
                w = _philox(77, (pid, 0, 3, blk)); u = [((int(x) >> 9) + 0.5) / 8388608.0 for x in w]
            to = math.degrees(math.acos(1 - 2 * u[0])); dp = 360.0 * u[1]
            want_n = [math.sin(math.radians(to)) * math.cos(math.radians(dp)), math.sin(math.radians(to)) * math.sin(math.radians(dp)),
                      math.cos(math.radians(to))]                       # phi_in = 0: phi_out = dphi
            assert np.allclose(n_out, want_n, atol=2e-7)
            M = zt.at(ti, to, dp)
            s = M @ S_in
            # reference: theta^ of n_out in the grain frame = lab here; S_out is referenced to theta^ of the fp32-rounded n_out
            assert np.allclose(S_out, s / s[0], atol=3e-6)
            if blk == 0:
                assert abs(tau + math.log(u[3])) < 1e-15
    # density in cos(theta_out): integrate the interpolated table over dphi on a fine grid
    edges = np.linspace(-1, 1, 11)
    mu = np.linspace(-1, 1, 801); mu_c = 0.5 * (mu[1:] + mu[:-1])
    dps = (np.arange(72) + 0.5) * 5.0
    dens = np.array([np.mean([(zt.at(ti, math.degrees(math.acos(c)), d) @ S_in)[0] for d in dps]) for c in mu_c])
    want = np.array([dens[(mu_c >= a) & (mu_c < bb)].sum() for a, bb in zip(edges[:-1], edges[1:])]); want /= want.sum()
    got, _ = np.histogram(ct, bins=edges); got = got / N
    assert np.all(np.abs(got - want) < 5 * np.sqrt(want / N) + 2e-3), (got, want)
    assert rounds.mean() > 1.2 and rounds.max() < 60                         # rejections do happen, the bound holds


def test_scatter_z_geometry_for_any_field_direction():
    """Isotropic dipoles, any B: the scattering is Rayleigh whatever the grain frame, so for unpolarised input the sampled
    angle between n_in and n_out has <cos^2> = 2/5 and the outgoing light is polarised normal to the plane of n_in and n_out
    with degree (1 - mu^2)/(1 + mu^2) -- which fails if direction and Stokes vector are not taken at the same (theta_out, dphi)."""
    zt = OracleZTable(inputs.dipole_ztable(73, 73, 144))
    rng = np.random.default_rng(54)
    c2 = []
    for t in range(3000):
        b = rand_unit(rng); n_in = rand_unit(rng).astype(np.float32).astype(float)
        n_out, S, tau, r = zt.scatter(b, n_in, [1, 0, 0, 0], 5, t, 1)
        mu = float(np.dot(n_in, n_out) / np.linalg.norm(n_in) / np.linalg.norm(n_out))
        c2.append(mu * mu)
        if t < 400 and abs(mu) < 0.95:
            sperp = np.cross(n_in, n_out); sperp /= np.linalg.norm(sperp)
            to, po = sph_basis(n_out)
            want = stokes_of_E(sperp, to, po)
            P = (1 - mu * mu) / (1 + mu * mu)
            assert np.allclose(S[1:3], P * want[1:3], atol=2e-2), (S, P * want)
            assert abs(S[3]) < 1e-3
    assert abs(np.mean(c2) - 0.4) < 4 * 0.27 / math.sqrt(3000)
